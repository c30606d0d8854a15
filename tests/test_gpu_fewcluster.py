"""The few-cluster variant (second half; reading 21) through the C-ABI
(sw_fewcluster_step: k_scan -> k_seam -> k_few_seeds -> k_final<MODE_FEW>) against the oracle's plain statement of it
(orc_fewcluster_step: decompose, select the clusters that hold a seed point, flip each with probability p_flip): spins, canonical
labels and the number of flipped sites bit for bit after every step."""
import numpy as np
import pytest

import oracle
from paper_1105_5804_b200 import binding

pytestmark = pytest.mark.gpu

BETA_C = oracle.beta_c(2)


@pytest.mark.parametrize("L,beta,seed,n_seeds,p_flip", [
    (4, BETA_C, 1, 3, 0.7), (8, BETA_C, 2, 1, 0.999), (64, BETA_C, 3, 16, 0.5), (100, 0.40, 4, 25, 0.7),
    (132, BETA_C, 5, 300, 0.3), (260, 0.50, 6, 8, 0.9), (512, BETA_C, 7, 1024, 0.6), (1024, BETA_C, 0xDEADBEEF12345, 64, 0.7)])
def test_fewcluster_steps_match_the_oracle(L, beta, seed, n_seeds, p_flip):
    lat = binding.Lattice(L, 2, beta, seed)
    T, Tf = lat.get_threshold(), oracle.threshold_from_p(p_flip)
    lat.init_spins(1)
    lat.sweep(3)                                                      # a few sweeps towards equilibrium first
    s = lat.spins_host().copy()
    t = lat.get_counter()
    total = 0
    for k in range(6):
        got = lat.fewcluster_step(1, n_seeds, Tf)
        f, nfc, lab = oracle.fewcluster_step(L, T, seed, t + k, n_seeds, Tf, s)
        assert got == [f], (k, got, f)
        assert np.array_equal(lat.labels_host(), lab), k
        assert np.array_equal(lat.spins_host(), s), k
        total += f
    # a batch without reading the counts back in between, then the counts of all of them at once
    got = lat.fewcluster_step(5, n_seeds, Tf)
    want = [oracle.fewcluster_step(L, T, seed, t + 6 + k, n_seeds, Tf, s)[0] for k in range(5)]
    assert got == want and np.array_equal(lat.spins_host(), s)
    assert lat.get_counter() == t + 11
    o = lat.observables()
    w = oracle.observables(L, 2, s)
    assert o["energy"] == w["energy"] and o["magnetisation"] == w["magnetisation"]
    if L >= 64:
        assert total + sum(want) > 0                                  # something was flipped along the way
    lat.close()


def test_fewcluster_special_cases():
    L, seed = 128, 9
    lat = binding.Lattice(L, 2, BETA_C, seed)
    T = lat.get_threshold()
    lat.init_spins(1)
    s = lat.spins_host().copy()
    before = s.copy()
    # no seeds, or p_flip = 0: nothing moves, the counter still advances and the labels are those of the decomposition
    assert lat.fewcluster_step(1, 0, 0xFFFFFFFF) == [0]
    assert lat.fewcluster_step(1, 50, 0) == [0]
    assert np.array_equal(lat.spins_host(), before) and lat.get_counter() == 2
    codes, _ = oracle.bonds(L, T, seed, 1, before)
    assert np.array_equal(lat.labels_host(), oracle.label(L, codes)[0])
    # one seed and p_flip = 1 - 2^-32: the Wolff step of the same counter
    twin = binding.Lattice(L, 2, BETA_C, seed)
    twin.init_spins(1)
    twin.set_counter(2)
    for k in range(10):
        assert lat.fewcluster_step(1, 1, 0xFFFFFFFF) == twin.wolff_step(1)
    assert np.array_equal(lat.spins_host(), twin.spins_host())
    twin.close()
    # cold start at low temperature: one cluster holds (almost) every seed; it is flipped once, not once per seed
    lat.init_spins(0)
    lat.set_counter(0)
    lat.set_threshold(0xFFFFFFFF)
    s = lat.spins_host().copy()
    got = lat.fewcluster_step(1, 4096, 0xFFFFFFFF)
    f, nfc, _ = oracle.fewcluster_step(L, 0xFFFFFFFF, seed, 0, 4096, 0xFFFFFFFF, s)
    assert got == [f] and nfc == 1 and f == L * L and np.array_equal(lat.spins_host(), s)
    lat.close()


def test_fewcluster_argument_checks():
    lib = binding.lib()
    lat = binding.Lattice(64, 2, BETA_C, 1)
    assert lib.sw_fewcluster_step(lat._h, -1, 4, 1, None, None) == binding.SW_EINVAL
    assert lib.sw_fewcluster_step(lat._h, 1, -1, 1, None, None) == binding.SW_EINVAL
    assert lib.sw_fewcluster_step(lat._h, 1, 65537, 1, None, None) == binding.SW_EINVAL
    assert lib.sw_fewcluster_step(lat._h, 1, 4096, 1, None, None) == binding.SW_EINVAL       # table of 8192 slots > N = 4096
    assert lib.sw_fewcluster_step(lat._h, 0, 4, 1, None, None) == binding.SW_OK
    lat.close()
    potts = binding.Lattice(64, 3, 0.5, 1)
    assert lib.sw_fewcluster_step(potts._h, 1, 4, 1, None, None) == binding.SW_EINVAL         # q = 2 only
    potts.close()
    cubic = binding.Lattice(8, 2, 0.2, 1, dim=3)
    assert lib.sw_fewcluster_step(cubic._h, 1, 4, 1, None, None) == binding.SW_EINVAL
    cubic.close()


def test_fewcluster_L4096_critical():
    """The size and temperature of BASELINE.json configs[4]'s Wolff half: 64 seeds, p_flip = 0.7, equilibrated lattice."""
    L, seed = 4096, 1
    lat = binding.Lattice(L, 2, BETA_C, seed)
    T, Tf = lat.get_threshold(), oracle.threshold_from_p(0.7)
    lat.init_spins(1)
    lat.sweep(40)
    s = lat.spins_host().copy()
    t = lat.get_counter()
    got = lat.fewcluster_step(4, 64, Tf)
    want = []
    for k in range(4):
        f, nfc, lab = oracle.fewcluster_step(L, T, seed, t + k, 64, Tf, s)
        want.append(f)
    assert got == want and np.array_equal(lat.spins_host(), s) and np.array_equal(lat.labels_host(), lab)
    lat.close()
