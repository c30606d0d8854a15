"""Pins for the oracle's labelling, flip bookkeeping, observables and cluster statistics (CPU only).

The labeller is pinned to an independent definition -- the transitive closure of the bond graph, computed with
boolean matrix squaring in numpy -- on ALL 2^18 bond configurations of the 3x3 torus, to special patterns with
known answers and to the invariants of a canonical labelling (SURVEY.md 8(c) "Labelling").
"""
import math

import numpy as np
import pytest

import oracle
from paper_1105_5804_b200 import inputs


def closure_labels(L, codes_batch):
    """Independent labeller: label[i] = min{ j : j ~ i } via reflexive-transitive closure of the adjacency matrix.
    codes_batch: uint8[B, N].  Returns int32[B, N]."""
    N = L * L
    B = codes_batch.shape[0]
    idx = np.arange(N)
    east = (idx // L) * L + (idx % L + 1) % L
    north = ((idx // L + 1) % L) * L + idx % L
    A = np.zeros((B, N, N), dtype=bool)
    A[:, idx, idx] = True
    e = (codes_batch & 1).astype(bool)
    n = ((codes_batch >> 1) & 1).astype(bool)
    for i in range(N):
        A[:, i, east[i]] |= e[:, i]
        A[:, east[i], i] |= e[:, i]
        A[:, i, north[i]] |= n[:, i]
        A[:, north[i], i] |= n[:, i]
    for _ in range(int(math.ceil(math.log2(N))) + 1):
        A = np.matmul(A.astype(np.uint8), A.astype(np.uint8)) > 0
    return np.argmax(A, axis=2).astype(np.int32)            # first True column = minimum reachable index


def test_all_bond_configurations_of_the_3x3_torus():
    L, N = 3, 9
    total = 1 << (2 * N)
    chunk = 1 << 13
    for start in range(0, total, chunk):
        ids = np.arange(start, start + chunk, dtype=np.int64)
        codes = np.stack([((ids >> (2 * i)) & 3).astype(np.uint8) for i in range(N)], axis=1)
        want = closure_labels(L, codes)
        for b in range(chunk):
            got, nc = oracle.label(L, codes[b])
            if not np.array_equal(got, want[b]):
                raise AssertionError((int(ids[b]), got, want[b]))
            assert nc == int((want[b] == np.arange(N)).sum())


@pytest.mark.parametrize("L,p,seed", [(4, 0.5, 1), (4, 0.3, 2), (5, 0.6, 3), (6, 0.45, 4), (7, 0.5, 5)])
def test_random_subsets_against_closure(L, p, seed):
    codes = np.stack([inputs.random_bond_codes(L, p, p, seed * 1000 + k) for k in range(64)])
    want = closure_labels(L, codes)
    for b in range(codes.shape[0]):
        got, _ = oracle.label(L, codes[b])
        assert np.array_equal(got, want[b])


def test_special_patterns():
    L = 8
    N = L * L
    i = np.arange(N)
    lab, nc = oracle.label(L, np.zeros(N, np.uint8))
    assert np.array_equal(lab, i) and nc == N                              # no bonds
    lab, nc = oracle.label(L, np.full(N, 3, np.uint8))
    assert not lab.any() and nc == 1                                       # all bonds
    lab, nc = oracle.label(L, np.full(N, 1, np.uint8))
    assert np.array_equal(lab, (i // L) * L) and nc == L                   # all east bonds: one cluster per row
    lab, nc = oracle.label(L, np.full(N, 2, np.uint8))
    assert np.array_equal(lab, i % L) and nc == L                          # all north bonds: one per column
    codes = np.zeros(N, np.uint8)
    codes[L - 1] = 1                                                       # east wrap bond (7,0)-(0,0)
    lab, nc = oracle.label(L, codes)
    assert lab[L - 1] == 0 and nc == N - 1 and np.array_equal(np.delete(lab, L - 1), np.delete(i, L - 1))
    codes = np.zeros(N, np.uint8)
    codes[(L - 1) * L + 3] = 2                                             # north wrap bond (3,7)-(3,0)
    lab, nc = oracle.label(L, codes)
    assert lab[(L - 1) * L + 3] == 3 and nc == N - 1
    lab, nc = oracle.label(L, inputs.snake_codes(L))
    assert not lab.any() and nc == 1


def check_canonical(L, codes, lab, nc):
    N = L * L
    i = np.arange(N)
    assert np.all(lab <= i) and np.all(lab >= 0)
    assert np.array_equal(lab[lab], lab)
    east = (i // L) * L + (i % L + 1) % L
    north = ((i // L + 1) % L) * L + i % L
    e = (codes & 1).astype(bool)
    n = ((codes >> 1) & 1).astype(bool)
    assert np.array_equal(lab[i[e]], lab[east[e]])
    assert np.array_equal(lab[i[n]], lab[north[n]])
    assert nc == int((lab == i).sum())
    nbonds = int(e.sum() + n.sum())
    assert nc >= N - nbonds


@pytest.mark.parametrize("L,p", [(16, 0.3), (64, 0.5), (100, 0.5), (128, 0.7), (257, 0.45)])
def test_invariants_and_scipy_components(L, p):
    from scipy.sparse import coo_matrix
    from scipy.sparse.csgraph import connected_components
    codes = inputs.random_bond_codes(L, p, p, 17 + L)
    lab, nc = oracle.label(L, codes)
    check_canonical(L, codes, lab, nc)
    # third opinion: scipy's connected components on the same graph (a library routine, different algorithm)
    N = L * L
    i = np.arange(N)
    east = (i // L) * L + (i % L + 1) % L
    north = ((i // L + 1) % L) * L + i % L
    e = (codes & 1).astype(bool)
    n = ((codes >> 1) & 1).astype(bool)
    rows = np.concatenate([i[e], i[n]])
    cols = np.concatenate([east[e], north[n]])
    g = coo_matrix((np.ones(rows.size, np.int8), (rows, cols)), shape=(N, N))
    ncomp, comp = connected_components(g, directed=False)
    assert ncomp == nc
    mins = np.full(ncomp, N, dtype=np.int64)
    np.minimum.at(mins, comp, i)
    assert np.array_equal(mins[comp].astype(np.int32), lab)


def test_forest_equality_case():
    # n_clusters = N - n_bonds iff the bond graph is a forest: a snake path is a tree
    L = 12
    codes = inputs.snake_codes(L)
    lab, nc = oracle.label(L, codes)
    nb = int((codes & 1).sum() + ((codes >> 1) & 1).sum())
    assert nc == 1 == L * L - nb


@pytest.mark.parametrize("q", [2, 3, 5])
def test_observables_against_numpy_definition(q):
    L = 24
    for seed in range(3):
        s = inputs.random_spins(L, q, seed)
        sq = s.reshape(L, L).astype(np.int64)
        o = oracle.observables(L, q, s)
        sat = int((sq == np.roll(sq, -1, 1)).sum() + (sq == np.roll(sq, -1, 0)).sum())
        assert o["sat_bonds"] == sat
        if q == 2:
            assert o["energy"] == -int((sq * np.roll(sq, -1, 1)).sum() + (sq * np.roll(sq, -1, 0)).sum())   # P:32 Eq. 1, Ising form
            assert o["magnetisation"] == int(sq.sum())
            assert o["state_count"][:2] == [int((sq == 1).sum()), int((sq == -1).sum())]
        else:
            assert o["energy"] == -sat
            cnt = np.bincount(sq.reshape(-1), minlength=q)
            assert o["state_count"][:q] == [int(c) for c in cnt]
            assert o["magnetisation"] == q * int(cnt.max()) - L * L
    # closed forms: cold, checkerboard, stripes
    N = L * L
    assert oracle.observables(L, 2, np.ones(N, np.int8))["energy"] == -2 * N
    cb = (1 - 2 * ((np.arange(N) // L + np.arange(N) % L) % 2)).astype(np.int8)
    o = oracle.observables(L, 2, cb)
    assert o["energy"] == 2 * N and o["magnetisation"] == 0 and o["sat_bonds"] == 0
    st = inputs.striped_spins(L, 2, 1)                       # alternating columns: all east bonds broken
    o = oracle.observables(L, 2, st)
    assert o["energy"] == 0 and o["sat_bonds"] == N


def test_cluster_stats_against_bincount():
    L = 96
    codes = inputs.random_bond_codes(L, 0.5, 0.5, 5)
    lab, nc = oracle.label(L, codes)
    c = oracle.cluster_stats(lab)
    sizes = np.bincount(lab, minlength=L * L)
    sizes = sizes[sizes > 0]
    assert c["n_clusters"] == nc == sizes.size
    assert c["max_cluster"] == int(sizes.max())
    assert c["sum_sq_cluster"] == int((sizes.astype(np.int64) ** 2).sum())
    assert sum(c["hist32"]) == nc
    want = np.bincount(np.floor(np.log2(sizes)).astype(int), minlength=32)
    assert c["hist32"] == [int(x) for x in want]
    assert int(sizes.sum()) == L * L


def test_flip_is_constant_on_clusters_and_keyed_by_root():
    L, q, seed, t = 32, 4, 77, 9
    codes = inputs.random_bond_codes(L, 0.5, 0.5, 1)
    lab, _ = oracle.label(L, codes)
    s = oracle.flip(L, q, seed, t, lab)
    assert np.array_equal(s, s[lab])                          # every site carries its root's new state
    assert s.min() >= 0 and s.max() < q
    # k_r = (PHILOX(seed; r, t_lo, t_hi, FLIP=2)[0] * q) >> 32, through the KAT-pinned primitive
    key = [seed & 0xFFFFFFFF, seed >> 32]
    for r in np.unique(lab)[:200]:
        w = oracle.philox([int(r), t, 0, 2], key)
        assert s[r] == (int(w[0]) * q) >> 32
    # a relabelled copy of the same partition with a different sweep counter gives a different assignment
    assert not np.array_equal(s, oracle.flip(L, q, seed, t + 1, lab))
    # Ising storage: k=0 -> +1, k=1 -> -1
    s2 = oracle.flip(L, 2, seed, t, lab)
    assert set(np.unique(s2)) <= {-1, 1}
    for r in np.unique(lab)[:200]:
        w = oracle.philox([int(r), t, 0, 2], key)
        assert s2[r] == (1 if (int(w[0]) >> 31) == 0 else -1)


def test_percolation_cluster_density_and_duality():
    # literature pins (not in the paper), statistical: clusters per site of bond percolation at p = 1/2 on the
    # square lattice -> (3 sqrt 3 - 5)/2 (Temperley-Lieb), torus correction +0.8835/N (Ziff-Finch-Adamchik);
    # Euler duality on the self-dual lattice: n(p) - n(1-p) = 1 - 2p per site.
    L = 512
    N = L * L
    dens = {}
    for p in (0.3, 0.5, 0.7):
        T = oracle.threshold_from_p(p)
        cold = oracle.init_spins(L, 2, 1, 0)
        vals = []
        for seed in (1, 2, 3):
            codes, _ = oracle.bonds(L, T, seed, 0, cold)
            _, nc = oracle.label(L, codes)
            vals.append(nc / N)
        dens[p] = float(np.mean(vals))
    sigma = math.sqrt(0.15 / N / 3)
    assert abs(dens[0.5] - ((3 * math.sqrt(3) - 5) / 2 + 0.8835 / N)) < 5 * sigma
    assert abs((dens[0.3] - dens[0.7]) - 0.4) < 5 * math.sqrt(2) * sigma


def test_label_of_an_image_adjacency_graph_matches_ndimage_segments():
    """Generic CCL input ("image segmentation"): the oracle's labelling of the 4-connected equal-value
    pixel graph of a synthetic image against scipy.ndimage.label run grey level by grey level (an independent labeller with
    its own numbering: compared as partitions, and the oracle's label must be the smallest pixel index of its segment)."""
    from scipy import ndimage
    for L, levels, seed in ((64, 2, 1), (100, 3, 2), (132, 5, 3)):
        img = inputs.blob_image(L, levels, seed)
        assert len(np.unique(img)) == levels
        codes = inputs.image_bond_codes(img)
        assert not (codes.reshape(L, L)[:, L - 1] & 1).any() and not (codes.reshape(L, L)[L - 1, :] & 2).any()   # no wrap
        lab, nc = oracle.label(L, codes)
        seg = np.zeros((L, L), dtype=np.int64)
        total = 0
        for v in range(levels):
            s, n = ndimage.label(img == v)                      # default structure: 4-connectivity
            seg[s > 0] = s[s > 0] + total
            total += n
        assert nc == total
        seg = seg.reshape(-1)
        first = np.full(total + 1, L * L, dtype=np.int64)
        np.minimum.at(first, seg, np.arange(L * L))
        assert np.array_equal(lab, first[seg].astype(np.int32))
