"""GPU-vs-oracle parity at BASELINE.json's FULL sizes (-m gpu), in the launch configuration bench.py times.

The serial oracle needs ~15 s per sweep at L=16384, so the chain is not followed sweep by sweep: the state of the
method is (spins, step counter t) -- every draw is a pure function of (seed, t, site, direction) (reading 5)
-- so the GPU state after a few sweeps is handed to the oracle, which performs ONE sweep from it; spins, labels,
cluster and bond counts, energy and magnetisation of that sweep must agree bit for bit (SURVEY.md 8(d) "parity at
L=16384").  Properties that hold at any size (canonical labels, bond ends in one cluster) are checked on the device.
"""
import math

import numpy as np
import pytest

import oracle
from paper_1105_5804_b200 import binding, inputs

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

BETA_C = oracle.beta_c(2)


@pytest.fixture(scope="module", autouse=True)
def _need_gpu():
    if not torch.cuda.is_available():
        pytest.fail("these tests need a CUDA device (the product has no CPU path)")
    binding.lib()


def check_label_properties(L, labels, bonds_packed=None):
    """Invariants of canonical labels at any size, on the device: label[i] <= i, label[label[i]] == label[i], and (if
    the packed bonds are given) both ends of every active bond carry the same label."""
    N = L * L
    idx = torch.arange(N, dtype=torch.int32, device=labels.device)
    assert bool((labels <= idx).all()) and bool((labels >= 0).all())
    assert bool((labels[labels.long()] == labels).all())
    if bonds_packed is not None:
        lab2 = labels.view(L, L)
        b = bonds_packed.view(L, L // 4)
        for j in range(4):
            east = ((b >> (2 * j)) & 1).bool()
            north = ((b >> (2 * j + 1)) & 1).bool()
            here = lab2[:, j::4]
            e_nb = torch.roll(lab2, -1, dims=1)[:, j::4]
            n_nb = torch.roll(lab2, -1, dims=0)[:, j::4]
            assert bool((here[east] == e_nb[east]).all())
            assert bool((here[north] == n_nb[north]).all())
    return int((labels == idx).sum())


def one_oracle_sweep_from_gpu_state(lat, L, q, seed, t):
    """GPU: one more sweep from its current state; oracle: the same sweep from a copy of that state."""
    T = lat.get_threshold()
    assert lat.get_counter() == t
    s = lat.spins_host().copy()
    lat.sweep(1)
    lab, _, nc, nb = oracle.sweep(L, q, T, seed, t, s)
    got_lab = lat.labels_host()
    assert np.array_equal(got_lab, lab), "labels differ at L=%d, t=%d" % (L, t)
    del got_lab
    assert np.array_equal(lat.spins_host(), s), "spins differ at L=%d, t=%d" % (L, t)
    o = lat.observables()
    w = oracle.observables(L, q, s)
    assert o["energy"] == w["energy"] and o["magnetisation"] == w["magnetisation"]
    assert o["n_clusters"] == nc and o["n_active_bonds"] == nb and o["counter"] == t + 1
    return o


def sweep_with_bond_end_check(lat, L):
    """One GPU sweep whose labels are checked against the bonds of that very step: sw_activate materialises the bond
    set of step t (same draws as the sweep's own, reading 16), the sweep labels it, and both ends of every
    active bond must carry one label -- a union lost to a race cannot pass this (the invariants alone could)."""
    lat.activate()
    lat.sweep(1)
    o = lat.observables()
    assert check_label_properties(L, lat.labels, lat.bonds) == o["n_clusters"]
    assert int(popcount_bytes(lat.bonds)) == o["n_active_bonds"]
    return o


def popcount_bytes(t):
    x = t.to(torch.int32)
    x = (x & 0x55) + ((x >> 1) & 0x55)
    x = (x & 0x33) + ((x >> 2) & 0x33)
    x = (x & 0x0F) + (x >> 4)
    return x.sum(dtype=torch.int64)


def test_config3_L16384_beta_c_sampled_sweeps_vs_oracle():
    """BASELINE.json configs[2] at beta_c, the workload bench.py times: the sampled sweeps {0, 1, 2, 50, 199} of
    SURVEY.md 8(d) "parity at L=16384", each one oracle sweep from the GPU state.  By sweep 199 the largest cluster holds
    a quarter of the lattice and spans thousands of strips: the contention of the timed state."""
    L, seed = 16384, 1
    lat = binding.Lattice(L, 2, BETA_C, seed, with_bonds=True)
    assert lat.get_threshold() == oracle.threshold(2, BETA_C) == 2515933592
    lat.init_spins(1)
    assert oracle.fnv1a64(lat.spins_host()) == oracle.fnv1a64(oracle.init_spins(L, 2, seed, 1))
    for t in (0, 1, 2):
        one_oracle_sweep_from_gpu_state(lat, L, 2, seed, t)
    lat.sweep(47)
    o = one_oracle_sweep_from_gpu_state(lat, L, 2, seed, 50)
    assert check_label_properties(L, lat.labels) == o["n_clusters"]
    lat.sweep(147)
    sweep_with_bond_end_check(lat, L)                                  # sweep 198, on the device
    o = one_oracle_sweep_from_gpu_state(lat, L, 2, seed, 199)
    st = lat.cluster_stats()
    assert st["max_cluster"] == o["max_cluster"] > 0.1 * L * L         # the giant critical cluster is there
    lat.close()


def test_config3_L16384_beta_c_cold_start_giant_cluster():
    """Cold start at beta_c: p = 0.586 is above the bond-percolation threshold, so sweep 0 builds one cluster through
    ~90 % of the lattice and every wrap -- the heaviest root contention the seam pass can see."""
    L, seed = 16384, 5
    lat = binding.Lattice(L, 2, BETA_C, seed, with_bonds=True)
    lat.init_spins(0)
    o = one_oracle_sweep_from_gpu_state(lat, L, 2, seed, 0)
    assert o["max_cluster"] > 0.8 * L * L
    sweep_with_bond_end_check(lat, L)
    lat.close()


@pytest.mark.parametrize("beta", [0.40, 0.50])
def test_config3_L16384_off_critical_vs_oracle(beta):
    """The other temperatures of configs[2]: sweep 50 from the GPU state against the oracle bit for bit, and the
    bond-end check on the device for the sweep before it."""
    L, seed = 16384, 1
    lat = binding.Lattice(L, 2, beta, seed, with_bonds=True)
    assert lat.get_threshold() == oracle.threshold(2, beta)
    lat.init_spins(1)
    lat.sweep(49)
    sweep_with_bond_end_check(lat, L)
    o = one_oracle_sweep_from_gpu_state(lat, L, 2, seed, 50)
    assert check_label_properties(L, lat.labels) == o["n_clusters"]
    st = lat.cluster_stats()
    assert st["n_clusters"] == o["n_clusters"] and sum(st["hist32"]) == o["n_clusters"]
    if beta == 0.50:
        assert o["max_cluster"] > 0.5 * L * L                          # ordered phase: one spanning cluster
    lat.close()


@pytest.mark.parametrize("what", ["p=0.5", "p=0.7", "sw beta=0.5"])
def test_L16384_labelling_repeats_bit_for_bit(what):
    """compute-sanitizer is closed on this GPU pool, so races are hunted by repetition at the size and contention of
    the bench: the same packed bonds are labelled 30 times; every result must equal the first (the canonical labelling
    is unique, reading 7) and the first must equal the oracle's labelling of the same bonds."""
    L = 16384
    lat = binding.Lattice(L, 2, 0.5, 3, with_bonds=True)
    if what.startswith("p="):
        lat.init_spins(0)
        lat.set_threshold(oracle.threshold_from_p(float(what[2:])))
    else:
        lat.init_spins(1)
        lat.sweep(30)                                                  # ordered phase: a spanning cluster
    lat.activate()
    first = torch.empty(L * L, dtype=torch.int32, device="cuda")
    lat.label(lat.bonds, first)
    check_label_properties(L, first, lat.bonds)
    want, _ = oracle.label(L, oracle.unpack_bonds(lat.bonds.cpu().numpy(), L * L))   # the first against the oracle, once
    assert np.array_equal(first.cpu().numpy(), want), what
    del want
    out = torch.empty_like(first)
    for rep in range(30):
        out.fill_(-7)
        lat.label(lat.bonds, out)
        assert torch.equal(out, first), "labelling %d of %s differs from the first" % (rep, what)
    lat.close()


def test_L16388_ragged_above_2_28_sites_vs_oracle():
    """The smallest lattice with N > 2^28: k_final keeps the new state in ONE bit above the label (Params::sbit = 30)
    and every strip row / column has a ragged last strip.  A few sweeps, then one oracle sweep from the GPU state."""
    L, seed = 16388, 2
    lat = binding.Lattice(L, 2, BETA_C, seed, with_bonds=True)
    lat.init_spins(1)
    one_oracle_sweep_from_gpu_state(lat, L, 2, seed, 0)
    lat.sweep(5)
    sweep_with_bond_end_check(lat, L)
    o = one_oracle_sweep_from_gpu_state(lat, L, 2, seed, 7)
    assert check_label_properties(L, lat.labels) == o["n_clusters"]
    lat.close()


def test_L32768_largest_lattice_properties():
    """The largest lattice the library accepts (N = 2^30, q = 2): init, a few sweeps, canonical-label invariants and the
    bond-end check on the device, energy moving towards the critical value, cluster statistics consistent."""
    L = 32768
    N = L * L
    lat = binding.Lattice(L, 2, BETA_C, 4, with_bonds=True)
    lat.init_spins(1)
    o0 = lat.observables()
    assert abs(o0["energy"]) < 20 * math.sqrt(2 * N) and abs(o0["magnetisation"]) < 20 * math.sqrt(N)
    lat.sweep(3)
    o = sweep_with_bond_end_check(lat, L)
    assert o["counter"] == 4 and -1.3 * N < o["energy"] < -0.9 * N
    st = lat.cluster_stats()
    assert st["n_clusters"] == o["n_clusters"] and sum(st["hist32"]) == o["n_clusters"]
    assert sum(o["state_count"]) == N
    # cold start: one cluster through most of the lattice (indices up to 2^30 - 1 on the seam pass)
    lat.init_spins(0)
    lat.set_counter(0)
    o = sweep_with_bond_end_check(lat, L)
    assert o["max_cluster"] > 0.8 * N
    lat.close()


def test_config4_L16384_percolation_labels_and_densities():
    """BASELINE.json configs[3]: i.i.d. bonds at p in {0.3, 0.5, 0.7}; bonds and labels of all three against the oracle
    bit for bit and against the invariants; cluster densities against the pins of SURVEY.md 8(c) (square-lattice bond percolation:
    n_c(1/2) = (3 sqrt 3 - 5)/2 per site; Euler duality n_c(0.3) - n_c(0.7) = 1 - 2*0.3)."""
    L, N = 16384, 16384 * 16384
    lat = binding.Lattice(L, 2, 0.1, 1, with_bonds=True)
    lat.init_spins(0)
    dens = {}
    for p in (0.3, 0.5, 0.7):
        lat.set_threshold(oracle.threshold_from_p(p))
        lat.set_counter(0)
        lat.activate()
        lat.label()
        nroots = check_label_properties(L, lat.labels, lat.bonds)
        st = lat.cluster_stats()
        assert st["n_clusters"] == nroots and sum(st["hist32"]) == nroots
        dens[p] = nroots / N
        # every p against the oracle bit for bit (the invariants above cannot see two clusters sharing one label)
        codes = oracle.unpack_bonds(lat.bonds.cpu().numpy(), N)
        want_codes, _ = oracle.bonds(L, oracle.threshold_from_p(p), 1, 0, oracle.init_spins(L, 2, 1, 0))
        assert np.array_equal(codes, want_codes), p
        del want_codes
        want, nc = oracle.label(L, codes)
        assert nc == nroots and np.array_equal(lat.labels_host(), want), p
        del want, codes
    sigma = math.sqrt(0.15 / N)                                       # per-sample sigma of clusters/N
    assert abs(dens[0.5] - ((3 * math.sqrt(3) - 5) / 2 + 0.8835 / N)) < 5 * sigma
    assert abs((dens[0.3] - dens[0.7]) - 0.4) < 5 * math.sqrt(2) * sigma
    lat.close()


def test_config5_potts_q4_L4096():
    """BASELINE.json configs[4], first half: q=4 at beta_c = ln 3 (T = 0xAAAAAAAA), L=4096: the first sweeps one by one,
    then one oracle sweep from the GPU state after 40 sweeps; satisfied-bond fraction near 3/4 (loose duality pin)."""
    L, q, seed = 4096, 4, 1
    lat = binding.Lattice(L, q, math.log(3.0), seed)
    assert lat.get_threshold() == 0xAAAAAAAA
    lat.init_spins(1)
    for t in range(3):
        one_oracle_sweep_from_gpu_state(lat, L, q, seed, t)
    lat.sweep(37)
    o = one_oracle_sweep_from_gpu_state(lat, L, q, seed, 40)
    assert check_label_properties(L, lat.labels) == o["n_clusters"]
    lat.close()


def test_config5_wolff_L4096():
    """BASELINE.json configs[4], second half: Wolff steps on L=4096 Ising at beta_c after SW equilibration; every step of
    the first 30 and a batch of 200 against the oracle's serial cluster growth from the same state."""
    L, seed = 4096, 1
    lat = binding.Lattice(L, 2, BETA_C, seed)
    T = lat.get_threshold()
    lat.init_spins(1)
    lat.sweep(60)
    s = lat.spins_host().copy()
    t = lat.get_counter()
    for k in range(30):
        sizes = lat.wolff_step(1)
        sz, i0, root = oracle.wolff_step(L, T, seed, t + k, s)
        assert sizes == [sz], k
    assert np.array_equal(lat.spins_host(), s)
    sizes = lat.wolff_step(200)
    want = [oracle.wolff_step(L, T, seed, t + 30 + k, s)[0] for k in range(200)]
    assert sizes == want and np.array_equal(lat.spins_host(), s)
    assert lat.get_counter() == t + 230
    lat.close()
