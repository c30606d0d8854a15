"""Multi-GPU row bands (include/swb200.h "MULTI-GPU ROW BANDS") run as G bands on ONE GPU, band after
band (-m gpu): the stitched spins and labels, the summed counters and the energy / magnetisation of every configuration must
equal the oracle's single-lattice sweep bit for bit -- the same bar as sw_sweep."""
import numpy as np
import pytest

import oracle
from paper_1105_5804_b200 import bands, binding

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

BETA_C = oracle.beta_c(2)


@pytest.fixture(scope="module", autouse=True)
def _need_gpu():
    if not torch.cuda.is_available():
        pytest.fail("these tests need a CUDA device (the product has no CPU path)")
    binding.lib()


def band_parity(L, q, beta, seed, G, mode, nsweeps, T=None):
    grp = bands.BandGroup(L, q, beta, seed, G)
    if T is not None:
        for lat in grp.lats:
            lat.set_threshold(T)
    T = grp.lats[0].get_threshold()
    grp.init_spins(mode)
    s = oracle.init_spins(L, q, seed, mode)
    N = L * L
    for t in range(nsweeps):
        before = oracle.observables(L, q, s)
        grp.sweep(1)
        lab, codes, nc, nb = oracle.sweep(L, q, T, seed, t, s)
        got_l, got_s = grp.labels_host(), grp.spins_host()
        assert np.array_equal(got_l, lab), f"G={G} L={L}: labels differ at sweep {t} ({int((got_l != lab).sum())} sites)"
        assert np.array_equal(got_s, s), f"G={G} L={L}: spins differ at sweep {t}"
        c = grp.counters()
        assert c["n_clusters"] == nc and c["n_active_bonds"] == nb
        assert c["sat_before"] == before["sat_bonds"]
        if q == 2:
            assert N - 2 * c["minus_before"] == before["magnetisation"]
        assert all(lat.get_counter() == t + 1 for lat in grp.lats)
    grp.close()


@pytest.mark.parametrize("L,G", [(64, 2), (128, 2), (128, 4), (256, 8), (512, 2), (512, 16), (1024, 4)])
def test_ising_bands_every_sweep(L, G):
    band_parity(L, 2, BETA_C, 100 + L + G, G, 1, 6)


def test_potts_and_off_critical_bands():
    band_parity(256, 3, oracle.beta_c(3), 5, 4, 1, 5)
    band_parity(256, 4, oracle.beta_c(4), 6, 2, 1, 5)
    band_parity(512, 2, 0.40, 7, 4, 1, 4)
    band_parity(512, 2, 0.50, 8, 4, 1, 4)


def test_cold_start_giant_cluster_across_all_bands():
    band_parity(512, 2, 0.6, 9, 8, 0, 3)                 # one cluster through every band and both wraps
    band_parity(256, 2, BETA_C, 10, 4, 0, 4)
    band_parity(128, 2, 0.3, 11, 4, 0, 2, T=2 ** 32 - 1)  # all bonds
    band_parity(128, 2, 0.3, 12, 2, 1, 2, T=0)            # no bonds


def test_bands_equal_single_gpu_chain_L4096():
    """A longer chain at L=4096: 4 bands against sw_sweep on one handle (itself checked against the oracle elsewhere), every
    sweep; then one sweep from that equilibrated state against the oracle."""
    L, q, seed, G = 4096, 2, 3, 4
    grp = bands.BandGroup(L, q, BETA_C, seed, G)
    ref = binding.Lattice(L, q, BETA_C, seed)
    grp.init_spins(1); ref.init_spins(1)
    for t in range(40):
        grp.sweep(1); ref.sweep(1)
        if t % 8 == 7:
            assert np.array_equal(grp.spins_host(), ref.spins_host()) and np.array_equal(grp.labels_host(), ref.labels_host())
    s = grp.spins_host().copy()
    T = ref.get_threshold()
    grp.sweep(1)
    lab, _, nc, nb = oracle.sweep(L, q, T, seed, 40, s)
    assert np.array_equal(grp.labels_host(), lab) and np.array_equal(grp.spins_host(), s)
    c = grp.counters()
    assert c["n_clusters"] == nc and c["n_active_bonds"] == nb
    grp.close(); ref.close()


def test_band_arguments_and_states():
    lat = binding.Lattice(256, 2, 0.4, 1)
    lib = binding.lib()
    assert lib.sw_set_band(lat._h, 0, 3) == binding.SW_EINVAL       # 8 strip rows do not split into 3 bands
    assert lib.sw_set_band(lat._h, 2, 2) == binding.SW_EINVAL
    assert lib.sw_sweep_band_begin(lat._h, None) == binding.SW_ESTATE   # not banded
    lat.set_band(1, 2)
    assert lib.sw_sweep(lat._h, 1, None) == binding.SW_ESTATE
    assert lib.sw_sweep_band_end(lat._h, None) == binding.SW_ESTATE     # begin has not run
    with pytest.raises(binding.SwError):
        lat.observables()                                            # a banded handle holds its band's rows only
    with pytest.raises(binding.SwError):
        lat.wolff_step(1)
    lay = lat.band_layout(1)
    assert lay["y_first"] == 128 and lay["n_rows"] == 128 and lay["y_halo"] == 0
    lat.set_band(0, 1)                                               # back to the whole lattice
    lat.init_spins(1); lat.sweep(1)
    lat.close()
    l2 = binding.Lattice(100, 2, 0.4, 1)
    assert lib.sw_set_band(l2._h, 0, 2) == binding.SW_EINVAL           # L must be a multiple of the strip height
    l2.close()


def test_L16384_four_bands_equilibrated_vs_single_gpu_and_oracle():
    """Full size: the equilibrated critical L=16384 state (giant cluster through every band) handed to 4 bands; 3 sweeps must
    equal the single-GPU chain bit for bit, the last one is also checked against the oracle from the same state."""
    L, q, seed, G = 16384, 2, 1, 4
    ref = binding.Lattice(L, q, BETA_C, seed)
    ref.init_spins(1)
    ref.sweep(60)
    grp = bands.BandGroup(L, q, BETA_C, seed, G)
    for lat in grp.lats:
        lat.spins.copy_(ref.spins)
        lat.set_counter(ref.get_counter())
    grp.sweep(2); ref.sweep(2)
    assert np.array_equal(grp.spins_host(), ref.spins_host())
    s = ref.spins_host().copy()
    t = ref.get_counter()
    grp.sweep(1); ref.sweep(1)
    got_s, got_l = grp.spins_host(), grp.labels_host()
    assert np.array_equal(got_s, ref.spins_host()) and np.array_equal(got_l, ref.labels_host())
    lab, _, nc, nb = oracle.sweep(L, q, ref.get_threshold(), seed, t, s)
    assert np.array_equal(got_l, lab) and np.array_equal(got_s, s)
    c = grp.counters()
    assert c["n_clusters"] == nc and c["n_active_bonds"] == nb
    grp.close(); ref.close()
