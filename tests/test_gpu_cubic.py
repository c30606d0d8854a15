"""Simple cubic lattice through the C-ABI against the oracle's orc3_* functions (-m gpu): spins, labels,
bond bytes, cluster counts, energy and magnetisation BIT-EXACT after every sweep; ragged tiles (L not a multiple of 32 / 8),
lattices smaller than one tile, giant clusters through every wrap, degenerate thresholds, the fused E / M series."""
import numpy as np
import pytest

import oracle
from paper_1105_5804_b200 import binding

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

BETA_C3 = 0.2216546          # 3D Ising critical coupling (literature value; only used to choose a workload)


@pytest.fixture(scope="module", autouse=True)
def _need_gpu():
    if not torch.cuda.is_available():
        pytest.fail("these tests need a CUDA device (the product has no CPU path)")
    binding.lib()


def sweep_parity3(L, q, beta, seed, mode, nsweeps, T=None, t0=0):
    lat = binding.Lattice(L, q, beta, seed, with_bonds=True, dim=3)
    if T is not None:
        lat.set_threshold(T)
    else:
        assert lat.get_threshold() == oracle.threshold(q, beta)
    T = lat.get_threshold()
    lat.init_spins(mode)
    s = oracle.init_spins3(L, q, seed, mode)
    assert np.array_equal(lat.spins_host(), s)
    lat.set_counter(t0)
    N = L ** 3
    for t in range(t0, t0 + nsweeps):
        lat.activate()
        want_codes, _ = oracle.bonds3(L, T, seed, t, s)
        assert np.array_equal(lat.bonds.cpu().numpy(), want_codes), f"bond bytes differ at sweep {t}"
        e_before = oracle.observables3(L, q, s)
        lat.sweep(1)
        lab, codes, nc, nb = oracle.sweep3(L, q, T, seed, t, s)
        assert np.array_equal(lat.labels_host(), lab), f"labels differ at sweep {t}"
        assert np.array_equal(lat.spins_host(), s), f"spins differ at sweep {t}"
        o = lat.observables()
        want = oracle.observables3(L, q, s)
        cs = oracle.cluster_stats(lab)
        assert o["energy"] == want["energy"] and o["magnetisation"] == want["magnetisation"]
        assert o["sat_bonds"] == want["sat_bonds"] and o["state_count"] == want["state_count"]
        assert o["n_clusters"] == nc and o["n_active_bonds"] == nb
        assert o["max_cluster"] == cs["max_cluster"] and o["sum_sq_cluster"] == cs["sum_sq_cluster"]
        assert o["counter"] == t + 1
        assert lat.cluster_stats() == cs
        # fused series: E (and M for q = 2) of the configuration the sweep STARTED from
        en, mg = lat.series(t, 1, magnetisation=(q == 2))
        assert en[0] == e_before["energy"]
        if q == 2:
            assert mg[0] == e_before["magnetisation"]
    lat.close()


@pytest.mark.parametrize("L", [4, 8, 12, 20, 32, 36, 64])
def test_ising_cubic_every_sweep(L):
    sweep_parity3(L, 2, BETA_C3, 1000 + L, 1, 6)


@pytest.mark.parametrize("L,q,beta", [(8, 3, 0.55), (24, 3, 0.5506), (40, 4, 0.63), (16, 8, 0.8)])
def test_potts_cubic_every_sweep(L, q, beta):
    sweep_parity3(L, q, beta, 7, 1, 5)


def test_cold_start_giant_cluster_through_every_wrap():
    sweep_parity3(36, 2, 0.6, 3, 0, 3)                   # p = 0.70: one cluster spans the lattice in all three directions
    sweep_parity3(64, 2, 0.3, 4, 0, 3)


def test_degenerate_thresholds_and_counter_high_word():
    sweep_parity3(12, 2, 0.2, 5, 1, 2, T=0)              # no bonds: every site its own cluster
    sweep_parity3(12, 2, 0.2, 5, 0, 2, T=2 ** 32 - 1)    # cold + all bonds: one cluster
    sweep_parity3(20, 2, BETA_C3, 6, 1, 3, t0=(5 << 32) + 1)


def test_L128_equilibrated_from_gpu_state():
    L, q, seed = 128, 2, 9
    lat = binding.Lattice(L, q, BETA_C3, seed, dim=3)
    lat.init_spins(1)
    lat.sweep(60)
    T = lat.get_threshold()
    for _ in range(2):
        t = lat.get_counter()
        s = lat.spins_host().copy()
        lat.sweep(1)
        lab, codes, nc, nb = oracle.sweep3(L, q, T, seed, t, s)
        assert np.array_equal(lat.labels_host(), lab) and np.array_equal(lat.spins_host(), s)
        o = lat.observables()
        assert o["n_clusters"] == nc and o["n_active_bonds"] == nb
        assert o["energy"] == oracle.observables3(L, q, s)["energy"]
    lat.close()


@pytest.mark.parametrize("L", [8, 20, 36, 64, 96])
def test_label_bond_percolation_cubic(L):
    """sw_label on a cubic handle: i.i.d. bond bytes (below, at and above the bond-percolation threshold 0.2488 of the simple
    cubic lattice) and structured sets -> canonical labels, cluster count and statistics of the oracle."""
    N = L ** 3
    lat = binding.Lattice(L, 2, 0.1, 0, dim=3)
    out = torch.empty(N, dtype=torch.int32, device="cuda")
    rng = np.random.default_rng(L)
    cases = []
    for p in (0.15, 0.2488, 0.35):
        c = np.zeros(N, dtype=np.uint8)
        for d in range(3):
            c |= (rng.random(N) < p).astype(np.uint8) << d
        cases.append(c)
    cases += [np.zeros(N, np.uint8), np.full(N, 7, np.uint8), np.full(N, 1, np.uint8), np.full(N, 2, np.uint8), np.full(N, 4, np.uint8)]
    wrap = np.zeros(N, np.uint8)
    wrap[L - 1] = 1; wrap[(L - 1) * L] |= 2; wrap[(L - 1) * L * L] |= 4            # one wrap bond per direction
    cases.append(wrap)
    for c in cases:
        lat.label(torch.from_numpy(c).cuda(), out)
        want, nc = oracle.label3(L, c)
        got = out.cpu().numpy()
        assert np.array_equal(got, want), f"L={L}: {int((got != want).sum())} labels differ"
        assert lat.cluster_stats(out) == oracle.cluster_stats(want)
        assert lat.observables(spins=False, clusters=False)["n_clusters"] == nc
    lat.close()


def test_unsupported_calls_and_shapes():
    lib = binding.lib()
    assert lib.sw_workspace_bytes3d(6, 2) == 0 and lib.sw_workspace_bytes3d(1028, 2) == 0 and lib.sw_workspace_bytes3d(64, 9) == 0
    lat = binding.Lattice(8, 2, 0.2, 1, with_bonds=True, dim=3)
    with pytest.raises(binding.SwError):
        lat.wolff_step(1)
    with pytest.raises(binding.SwError):
        lat.label_paper(0, 8)
    assert lib.sw_wolff_frontier(lat._h, 8) == binding.SW_EINVAL
    lat.close()
