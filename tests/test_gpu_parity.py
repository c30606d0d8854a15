"""GPU-vs-oracle parity, through the C-ABI (-m gpu).  Everything here is integer / byte work: the bar is BIT-EXACT
equality of spins, labels, bonds, cluster counts, energy and magnetisation (BASELINE.json north_star)."""
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


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


# ------------------------------------------------------------------------------------------------ init / bonds
@pytest.mark.parametrize("L,q", [(4, 2), (64, 2), (100, 3), (256, 4), (132, 8)])
def test_init_spins(L, q):
    lat = binding.Lattice(L, q, 0.4, 1234)
    for mode in (0, 1):
        lat.init_spins(mode)
        assert np.array_equal(lat.spins_host(), oracle.init_spins(L, q, 1234, mode))
    lat.close()


@pytest.mark.parametrize("L,q,beta,seed", [(4, 2, BETA_C, 1234), (64, 2, BETA_C, 1), (100, 2, 0.5, 2),
                                           (260, 3, oracle.beta_c(3), 3), (512, 4, math.log(3), 0xDEADBEEFCAFEF00D)])
def test_activate_matches_oracle_bonds(L, q, beta, seed):
    lat = binding.Lattice(L, q, beta, seed, with_bonds=True)
    assert lat.get_threshold() == oracle.threshold(q, beta)
    lat.init_spins(1)
    s = lat.spins_host()
    for t in (0, 1, (3 << 32) + 7):
        lat.set_counter(t)
        lat.activate()
        codes, _ = oracle.bonds(L, lat.get_threshold(), seed, t, s)
        assert np.array_equal(lat.bonds.cpu().numpy(), oracle.pack_bonds(codes)), t
        assert lat.get_counter() == t
    lat.close()


# ------------------------------------------------------------------------------------------------ sw_label
def label_case(L, codes):
    lat = binding.Lattice(L, 2, 0.1, 0)
    out = torch.empty(L * L, dtype=torch.int32, device="cuda")
    lat.label(dev(inputs.pack_codes(codes)), out)
    want, nc = oracle.label(L, codes)
    got = out.cpu().numpy()
    if not np.array_equal(got, want):
        bad = np.flatnonzero(got != want)
        raise AssertionError(f"L={L}: {bad.size} labels differ, first at site {bad[0]}: {got[bad[0]]} != {want[bad[0]]}")
    st = lat.cluster_stats(out)
    assert st == oracle.cluster_stats(want)
    assert st["n_clusters"] == nc
    lat.close()


@pytest.mark.parametrize("L,levels,seed", [(64, 2, 1), (132, 3, 2), (516, 4, 3), (1024, 2, 4), (1024, 6, 5)])
def test_label_image_segments(L, levels, seed):
    """A generic CCL input ("image segmentation"): sw_label on the 4-connected equal-value pixel graph of a
    synthetic grey-level image (no periodic bonds, blobs of all sizes) against the oracle, with cluster statistics."""
    label_case(L, inputs.image_bond_codes(inputs.blob_image(L, levels, seed)))


@pytest.mark.parametrize("L", [4, 8, 12, 64, 100, 128, 132, 192, 256, 260, 516, 1024])
@pytest.mark.parametrize("p", [0.3, 0.5, 0.7])
def test_label_random_bonds(L, p):
    label_case(L, inputs.random_bond_codes(L, p, p, 1000 + L))


@pytest.mark.parametrize("L", [4, 64, 132, 256, 320])
def test_label_special_patterns(L):
    N = L * L
    label_case(L, np.zeros(N, np.uint8))                  # no bonds
    label_case(L, np.full(N, 3, np.uint8))                # every bond (all wrap bonds too)
    label_case(L, np.full(N, 1, np.uint8))                # rows
    label_case(L, np.full(N, 2, np.uint8))                # columns
    label_case(L, inputs.snake_codes(L))                  # one boustrophedon path: the longest chain
    label_case(L, inputs.spiral_codes(L))                 # comb
    c = np.zeros(N, np.uint8); c[L - 1] = 1; c[(L - 1) * L + 3] = 2
    label_case(L, c)                                      # single wrap bonds
    label_case(L, inputs.random_bond_codes(L, 0.9, 0.1, 5))
    label_case(L, inputs.random_bond_codes(L, 0.1, 0.9, 6))


def test_label_is_deterministic_across_runs():
    L = 512
    codes = inputs.random_bond_codes(L, 0.5, 0.5, 77)
    lat = binding.Lattice(L, 2, 0.1, 0)
    b = dev(inputs.pack_codes(codes))
    outs = []
    for _ in range(5):
        out = torch.empty(L * L, dtype=torch.int32, device="cuda")
        lat.label(b, out)
        outs.append(out.cpu().numpy())
    for o in outs[1:]:
        assert np.array_equal(o, outs[0])
    lat.close()


# ------------------------------------------------------------------------------------------------ full sweeps
def sweep_parity(L, q, beta, seed, mode, nsweeps, check_every=1, T=None):
    lat = binding.Lattice(L, q, beta, seed)
    if T is not None:
        lat.set_threshold(T)
    T = lat.get_threshold()
    lat.init_spins(mode)
    s = oracle.init_spins(L, q, seed, mode)
    for t in range(nsweeps):
        lat.sweep(1)
        lab, codes, nc, nb = oracle.sweep(L, q, T, seed, t, s)
        if t % check_every and t != nsweeps - 1:
            continue
        assert np.array_equal(lat.labels_host(), lab), f"labels differ at sweep {t}"
        assert np.array_equal(lat.spins_host(), s), f"spins differ at sweep {t}"
        o = lat.observables()
        want = oracle.observables(L, q, s)
        cs = oracle.cluster_stats(lab)
        assert o["energy"] == want["energy"] and o["magnetisation"] == want["magnetisation"]
        assert o["sat_bonds"] == want["sat_bonds"] and o["state_count"] == want["state_count"]
        assert o["n_clusters"] == nc and o["n_active_bonds"] == nb
        assert o["max_cluster"] == cs["max_cluster"] and o["sum_sq_cluster"] == cs["sum_sq_cluster"]
        assert o["counter"] == t + 1
    lat.close()


def test_config1_L64_100_sweeps_every_sweep():
    sweep_parity(64, 2, BETA_C, 1234, 1, 100)


@pytest.mark.parametrize("L", [4, 8, 36, 132, 200])
def test_small_and_ragged_lattices(L):
    sweep_parity(L, 2, BETA_C, 7, 1, 20)


def test_config2_L1024_cold_start():
    sweep_parity(1024, 2, BETA_C, 1, 0, 30)


@pytest.mark.parametrize("beta", [0.40, 0.50])
def test_L512_off_critical(beta):
    sweep_parity(512, 2, beta, 3, 1, 15)


@pytest.mark.parametrize("q,L", [(3, 96), (4, 256), (8, 64)])
def test_potts(q, L):
    sweep_parity(L, q, oracle.beta_c(q), 11, 1, 25)


def test_degenerate_thresholds():
    sweep_parity(64, 2, 0.0, 5, 1, 3)                          # T = 0: no bonds, every site its own cluster
    sweep_parity(128, 2, 50.0, 5, 0, 3)                        # T = 2^32-1, cold: one cluster through every wrap
    sweep_parity(128, 4, 50.0, 5, 1, 3)


def test_chained_sweeps_equal_single_sweeps_and_counter_resume():
    L, seed = 256, 9
    a = binding.Lattice(L, 2, BETA_C, seed)
    b = binding.Lattice(L, 2, BETA_C, seed)
    a.init_spins(1)
    b.init_spins(1)
    a.sweep(12)
    for _ in range(12):
        b.sweep(1)
    assert np.array_equal(a.spins_host(), b.spins_host()) and np.array_equal(a.labels_host(), b.labels_host())
    # resume: (spins, t) is the whole state
    c = binding.Lattice(L, 2, BETA_C, seed)
    c.set_spins(a.spins_host())
    c.set_counter(a.get_counter())
    a.sweep(3)
    c.sweep(3)
    assert np.array_equal(a.spins_host(), c.spins_host())
    for lat in (a, b, c):
        lat.close()


def test_golden_vector_L64():
    from conftest import read_golden
    g = read_golden("survey_pipeline.txt")
    lat = binding.Lattice(64, 2, BETA_C, 1234)
    lat.init_spins(1)
    marks = {1: "L64_sweep1", 2: "L64_sweep2", 10: "L64_sweep10", 100: "L64_sweep100"}
    for t in range(1, 101):
        lat.sweep(1)
        if t in marks:
            o = lat.observables()
            assert [o["n_clusters"], o["n_active_bonds"], o["energy"], o["magnetisation"]] == \
                [int(x) for x in g[marks[t]].split()]
    lat.close()


# ------------------------------------------------------------------------------------------------ Wolff
@pytest.mark.parametrize("L,beta,nsteps", [(64, BETA_C, 60), (256, BETA_C, 40), (132, 0.5, 20), (4, BETA_C, 50)])
def test_wolff_steps(L, beta, nsteps):
    seed = 1234
    lat = binding.Lattice(L, 2, beta, seed)
    T = lat.get_threshold()
    lat.init_spins(1)
    s = oracle.init_spins(L, 2, seed, 1)
    for t in range(nsteps):
        sizes = lat.wolff_step(1)
        sz, i0, root = oracle.wolff_step(L, T, seed, t, s)
        assert sizes == [sz], t
        assert np.array_equal(lat.spins_host(), s), t
        assert lat.labels_host()[i0] == root
    # a batch call equals single calls
    sizes = lat.wolff_step(7)
    want = [oracle.wolff_step(L, T, seed, nsteps + k, s)[0] for k in range(7)]
    assert sizes == want and np.array_equal(lat.spins_host(), s)
    assert lat.get_counter() == nsteps + 7
    lat.close()


# ------------------------------------------------------------------------------------------------ observables
@pytest.mark.parametrize("q,L", [(2, 64), (2, 260), (3, 128), (5, 100), (8, 32)])
def test_observables_on_arbitrary_spins(q, L):
    lat = binding.Lattice(L, q, 0.3, 1)
    for seed in range(3):
        s = inputs.random_spins(L, q, seed)
        lat.set_spins(s)
        o = lat.observables()
        w = oracle.observables(L, q, s)
        for k in ("sat_bonds", "energy", "magnetisation", "state_count"):
            assert o[k] == w[k], k
        assert o["n_clusters"] == 0 and o["max_cluster"] == 0      # no labelling yet on this handle
    lat.set_spins(inputs.striped_spins(L, q, 4))
    assert lat.observables()["energy"] == oracle.observables(L, q, inputs.striped_spins(L, q, 4))["energy"]
    lat.close()


def test_sweep_host_end_to_end():
    L, seed = 256, 5
    lat = binding.Lattice(L, 2, BETA_C, seed)
    s = oracle.init_spins(L, 2, seed, 1)
    h_in = torch.from_numpy(s.copy()).pin_memory()
    h_out = torch.empty(L * L, dtype=torch.int8).pin_memory()
    h_lab = torch.empty(L * L, dtype=torch.int32).pin_memory()
    o = lat.sweep_host(h_in, 3, h_out, h_lab)
    lab = None
    for t in range(3):
        lab, _, nc, nb = oracle.sweep(L, 2, lat.get_threshold(), seed, t, s)
    assert np.array_equal(h_out.numpy(), s) and np.array_equal(h_lab.numpy(), lab)
    assert o["energy"] == oracle.observables(L, 2, s)["energy"] and o["n_clusters"] == nc
    assert o["max_cluster"] == oracle.cluster_stats(lab)["max_cluster"]
    # the cheap variant: spin part and the labelling's own counters, no cluster-size pass
    h_in.copy_(h_out)
    o2 = lat.sweep_host(h_in, 1, h_out, None, obs_flags=binding.OBS_SPINS)
    lab, _, nc, nb = oracle.sweep(L, 2, lat.get_threshold(), seed, 3, s)
    w = oracle.observables(L, 2, s)
    assert np.array_equal(h_out.numpy(), s)
    assert o2["energy"] == w["energy"] and o2["magnetisation"] == w["magnetisation"]
    assert o2["n_clusters"] == nc and o2["n_active_bonds"] == nb and o2["max_cluster"] == 0
    lat.close()


# ------------------------------------------------------------------------------------------------ fused E / M series
@pytest.mark.parametrize("L,q,beta,mode", [(64, 2, BETA_C, 1), (132, 2, 0.5, 0), (260, 2, 0.4, 1), (96, 3, oracle.beta_c(3), 1)])
def test_series_of_a_chain_matches_the_oracle(L, q, beta, mode):
    """sw_series_read: E (and M for q=2) of the configuration every sweep started from, counted by the sweep's own scan
    kernel, against the oracle's observables of the same chain -- bit for bit, including ragged strips (L=132, 260)."""
    seed, n = 21, 37
    lat = binding.Lattice(L, q, beta, seed)
    lat.init_spins(mode)
    s = oracle.init_spins(L, q, seed, mode)
    T = lat.get_threshold()
    want_E, want_M = [], []
    for t in range(n):
        w = oracle.observables(L, q, s)
        want_E.append(w["energy"]); want_M.append(w["magnetisation"])
        oracle.sweep(L, q, T, seed, t, s)
    lat.sweep(10)
    lat.sweep(n - 10)                                      # two batched calls: the series is contiguous across calls
    E, M = lat.series(0, n, magnetisation=(q == 2))
    assert E == want_E
    if q == 2:
        assert M == want_M
    else:
        with pytest.raises(binding.SwError):
            lat.series(0, n, magnetisation=True)
    assert lat.series(n - 5, 5, magnetisation=False)[0] == want_E[-5:]
    with pytest.raises(binding.SwError):
        lat.series(0, n + 1, magnetisation=False)          # the current configuration has not been scanned yet
    # the state is untouched: spins equal the oracle's
    assert np.array_equal(lat.spins_host(), s)
    lat.close()


def test_series_ring_wraps_and_follows_wolff_steps():
    L, seed = 8, 5
    lat = binding.Lattice(L, 2, BETA_C, seed)
    lat.init_spins(1)
    s = oracle.init_spins(L, 2, seed, 1)
    T = lat.get_threshold()
    n = 4096 + 300                                         # more sweeps than the ring holds
    ser = oracle.run_chain(L, 2, T, seed, 0, n, s)         # (E, M, ...) AFTER every sweep = configuration at counter t+1
    lat.sweep(n)
    E, M = lat.series(n - 4096, 4096)
    assert E == [int(x) for x in ser[n - 4097:n - 1, 0]] and M == [int(x) for x in ser[n - 4097:n - 1, 1]]
    with pytest.raises(binding.SwError):
        lat.series(n - 4097, 4)                            # overwritten
    # Wolff steps are filed under their counters too
    w = oracle.wolff_chain(L, T, seed, n, 6, s)
    lat.wolff_step(6)
    E, M = lat.series(n, 6)
    assert E == [int(ser[n - 1, 0])] + [int(x) for x in w[:5, 0]]
    assert M == [int(ser[n - 1, 1])] + [int(x) for x in w[:5, 1]]
    lat.close()


# ------------------------------------------------------------------------------------------------ frontier Wolff
@pytest.mark.parametrize("L,beta,levels,nsteps", [(64, BETA_C, 1000, 60), (64, BETA_C, 2, 60), (256, 0.40, 40, 80),
                                                  (132, 0.30, 1000, 50), (4, BETA_C, 5, 50), (256, 0.5, 3, 25)])
def test_wolff_frontier_growth_matches_the_oracle(L, beta, levels, nsteps):
    """sw_wolff_frontier: the cluster grown from the seed site (bonds drawn on demand) must be the oracle's cluster --
    sizes and spins after every step -- whether the growth finishes (large `levels`) or gives up and hands the step to the
    labelling path (small `levels`: clusters deeper than that take the fallback, spins restored first)."""
    seed = 77
    lat = binding.Lattice(L, 2, beta, seed)
    T = lat.get_threshold()
    lat.init_spins(1)
    lat.sweep(5)
    s = lat.spins_host().copy()
    t0 = lat.get_counter()
    lat.wolff_frontier(levels)
    for k in range(nsteps):
        sizes = lat.wolff_step(1)
        sz, i0, root = oracle.wolff_step(L, T, seed, t0 + k, s)
        assert sizes == [sz], k
        assert np.array_equal(lat.spins_host(), s), k
    sizes = lat.wolff_step(9)                              # a batch call equals single calls
    want = [oracle.wolff_step(L, T, seed, t0 + nsteps + k, s)[0] for k in range(9)]
    assert sizes == want and np.array_equal(lat.spins_host(), s)
    o = lat.observables()
    assert o["n_clusters"] == 0 and o["counter"] == t0 + nsteps + 9      # no labelling is maintained in this mode
    # back to the labelling path: labels and series are maintained again
    lat.wolff_frontier(0)
    sizes = lat.wolff_step(1)
    sz, i0, root = oracle.wolff_step(L, T, seed, t0 + nsteps + 9, s)
    assert sizes == [sz] and lat.labels_host()[i0] == root and np.array_equal(lat.spins_host(), s)
    lat.close()


def test_sweeps_on_a_side_stream_and_two_handles_interleaved():
    """The kernels of a sweep are chained by programmatic dependent launch: the chain must hold on a non-default stream and
    when the launches of two handles alternate on one stream."""
    L, q = 260, 2
    side = torch.cuda.Stream()
    with torch.cuda.stream(side):
        a = binding.Lattice(L, q, BETA_C, 11)
        b = binding.Lattice(L, q, 0.5, 12)
        a.init_spins(1); b.init_spins(1)
        for _ in range(4):
            a.sweep(1); b.sweep(1); a.sweep(1)
        side.synchronize()
        for lat, seed, n in ((a, 11, 8), (b, 12, 4)):
            s = oracle.init_spins(L, q, seed, 1)
            lab = None
            for t in range(n):
                lab, _, nc, nb = oracle.sweep(L, q, lat.get_threshold(), seed, t, s)
            assert np.array_equal(lat.spins_host(), s) and np.array_equal(lat.labels_host(), lab)
            o = lat.observables(spins=False, clusters=False)
            assert o["n_clusters"] == nc and o["n_active_bonds"] == nb
        a.close(); b.close()
