"""Pins of the oracle's simple-cubic functions (oracle/sw_oracle.c orc3_*), none of them the oracle itself:
an independent transitive closure and scipy's connected components for the labelling, single-spin patterns for the
direction -> neighbour map, the pinned Philox for the keying, numpy definitions and closed forms for the observables, and the
exact partition sum of the 3 x 3 x 3 Ising model (all 2^27 states, summed plane by plane) for the whole chain."""
import math

import numpy as np
import pytest

import oracle


def nbr(L, i, d):
    x, y, z = i % L, (i // L) % L, i // (L * L)
    if d == 0:
        x = (x + 1) % L
    elif d == 1:
        y = (y + 1) % L
    else:
        z = (z + 1) % L
    return z * L * L + y * L + x


def closure_labels(L, codes):
    """minimum reachable index by repeated squaring of the boolean adjacency matrix"""
    N = L ** 3
    A = np.eye(N, dtype=bool)
    for i in range(N):
        for d in range(3):
            if (codes[i] >> d) & 1:
                j = nbr(L, i, d)
                A[i, j] = A[j, i] = True
    while True:
        B = (A.astype(np.uint8) @ A.astype(np.uint8)) > 0
        if (B == A).all():
            break
        A = B
    return A.argmax(axis=1).astype(np.int32)


def test_label3_against_transitive_closure_L3():
    rng = np.random.default_rng(5)
    for k in range(120):
        p = rng.uniform(0.05, 0.6)
        codes = (rng.random((27, 3)) < p).astype(np.uint8)
        codes = (codes[:, 0] | (codes[:, 1] << 1) | (codes[:, 2] << 2)).astype(np.uint8)
        lab, nc = oracle.label3(3, codes)
        ref = closure_labels(3, codes)
        assert (lab == ref).all()
        assert nc == int((ref == np.arange(27)).sum())


def test_label3_against_scipy_and_structured_cases():
    from scipy.sparse import coo_matrix
    from scipy.sparse.csgraph import connected_components
    rng = np.random.default_rng(6)
    for L in (4, 5, 6, 9):
        N = L ** 3
        for p in (0.1, 0.2488, 0.4):                       # 0.2488: bond percolation threshold of the cubic lattice
            codes = np.zeros(N, dtype=np.uint8)
            for d in range(3):
                codes |= ((rng.random(N) < p).astype(np.uint8) << d)
            lab, nc = oracle.label3(L, codes)
            rows, cols = [], []
            for d in range(3):
                src = np.nonzero((codes >> d) & 1)[0]
                rows.append(src)
                cols.append(np.array([nbr(L, int(i), d) for i in src], dtype=np.int64))
            rows, cols = np.concatenate(rows), np.concatenate(cols)
            g = coo_matrix((np.ones(rows.size), (rows, cols)), shape=(N, N))
            ncc, comp = connected_components(g, directed=False)
            first = np.full(ncc, N, dtype=np.int64)
            np.minimum.at(first, comp, np.arange(N))
            assert nc == ncc and (lab == first[comp]).all()
        idx = np.arange(N)
        assert (oracle.label3(L, np.zeros(N, np.uint8))[0] == idx).all()
        assert (oracle.label3(L, np.full(N, 7, np.uint8))[0] == 0).all()
        assert (oracle.label3(L, np.full(N, 1, np.uint8))[0] == idx - idx % L).all()              # east only: rows
        assert (oracle.label3(L, np.full(N, 2, np.uint8))[0] == idx - ((idx // L) % L) * L).all()  # north only: columns of a plane
        assert (oracle.label3(L, np.full(N, 4, np.uint8))[0] == idx % (L * L)).all()               # up only: lines along z
        for d, site, other in ((0, L - 1, 0), (1, (L - 1) * L, 0), (2, (L - 1) * L * L, 0)):      # one wrap bond per direction
            c = np.zeros(N, np.uint8)
            c[site] = 1 << d
            lab, nc = oracle.label3(L, c)
            assert nc == N - 1 and lab[site] == other and (np.delete(lab, site) == np.delete(idx, site)).all()


def test_bonds3_special_cases_directions_and_keying():
    L, seed, t = 5, 0xDEADBEEFCAFEF00D, (7 << 32) | 3
    N = L ** 3
    cold = np.ones(N, dtype=np.int8)
    codes, n = oracle.bonds3(L, 0, seed, t, cold)
    assert n == 0 and not codes.any()
    codes, n = oracle.bonds3(L, 2 ** 32 - 1, seed, t, cold)
    assert n == 3 * N and (codes == 7).all()
    # one flipped spin: exactly its own three bonds and the bond of the neighbour behind it in each direction are missing
    for j in (0, 62, N - 1):
        s = cold.copy()
        s[j] = -1
        codes, n = oracle.bonds3(L, 2 ** 32 - 1, seed, t, s)
        assert n == 3 * N - 6 and codes[j] == 0
        x, y, z = j % L, (j // L) % L, j // (L * L)
        west = z * L * L + y * L + (x - 1) % L
        south = z * L * L + ((y - 1) % L) * L + x
        down = ((z - 1) % L) * L * L + y * L + x
        assert codes[west] == 7 & ~1 and codes[south] == 7 & ~2 and codes[down] == 7 & ~4
        rest = np.ones(N, bool)
        rest[[j, west, south, down]] = False
        assert (codes[rest] == 7).all()
    # keying (reading 19) through the pinned Philox: u3(i,d,t) = PHILOX(seed; i, t_lo, t_hi, 4)[d] < T
    T = oracle.threshold(2, 0.2216546)
    spins = oracle.init_spins3(L, 2, seed, 1)
    codes, n = oracle.bonds3(L, T, seed, t, spins)
    key = [seed & 0xFFFFFFFF, seed >> 32]
    tot = 0
    for i in range(N):
        w = oracle.philox([i, t & 0xFFFFFFFF, t >> 32, 4], key)
        for d in range(3):
            want = int(spins[i] == spins[nbr(L, i, d)] and int(w[d]) < T)
            assert (codes[i] >> d) & 1 == want
            tot += want
    assert tot == n
    # random spins never bond unequal neighbours; density p * sat / 3N within 5 sigma on a larger lattice
    L2 = 24
    s2 = oracle.init_spins3(L2, 3, 11, 1)
    T3 = oracle.threshold(3, 0.55)
    c2, n2 = oracle.bonds3(L2, T3, 11, 9, s2)
    sat = oracle.observables3(L2, 3, s2)["sat_bonds"]
    p = T3 / 2.0 ** 32
    assert abs(n2 - p * sat) < 5 * math.sqrt(sat * p * (1 - p))


def test_observables3_numpy_definition_and_closed_forms():
    L = 6
    N = L ** 3
    for q in (2, 3, 5):
        s = oracle.init_spins3(L, q, 3, 1)
        a = s.reshape(L, L, L)                             # [z, y, x]
        sat = int((a == np.roll(a, -1, 2)).sum() + (a == np.roll(a, -1, 1)).sum() + (a == np.roll(a, -1, 0)).sum())
        o = oracle.observables3(L, q, s)
        assert o["sat_bonds"] == sat
        if q == 2:
            assert o["energy"] == -(2 * sat - 3 * N) and o["magnetisation"] == int(s.astype(np.int64).sum())
            e = -int((a * np.roll(a, -1, 2)).astype(np.int64).sum() + (a * np.roll(a, -1, 1)).astype(np.int64).sum()
                     + (a * np.roll(a, -1, 0)).astype(np.int64).sum())
            assert o["energy"] == e
        else:
            cnt = np.bincount(s.astype(np.uint8), minlength=8)
            assert o["state_count"] == cnt.tolist() and o["energy"] == -sat and o["magnetisation"] == q * cnt.max() - N
    cold = np.ones(N, dtype=np.int8)
    assert oracle.observables3(L, 2, cold)["energy"] == -3 * N
    layers = np.repeat(np.where(np.arange(L) % 2 == 0, 1, -1).astype(np.int8), L * L)     # planes alternate along z
    o = oracle.observables3(L, 2, layers)
    assert o["sat_bonds"] == 2 * N and o["energy"] == -N and o["magnetisation"] == 0


def exact_3x3x3(beta):
    """<E>/N, <|m|>, <m^2> of the periodic 3 x 3 x 3 Ising model: sum over all 2^27 states, one 3 x 3 plane at a time."""
    st = np.arange(512)
    s = 1 - 2 * ((st[:, None] >> np.arange(9)[None, :]) & 1)          # [512, 9] spins +-1, k = 3 y + x
    g = s.reshape(512, 3, 3)
    e_in = -((g * np.roll(g, -1, 2)).sum(axis=(1, 2)) + (g * np.roll(g, -1, 1)).sum(axis=(1, 2)))
    e_x = -(s @ s.T)                                                   # [512, 512] coupling of two stacked planes
    m = s.sum(axis=1)
    Z = E = Mabs = M2 = 0.0
    for a in range(512):
        e = e_in[a] + e_in[:, None] + e_in[None, :] + e_x[a][:, None] + e_x + e_x[:, a][None, :]
        w = np.exp(-beta * (e + 81.0))                                 # shifted by the ground-state energy
        mm = (m[a] + m[:, None] + m[None, :]).astype(np.float64)
        Z += w.sum(); E += (w * e).sum(); Mabs += (w * np.abs(mm)).sum(); M2 += (w * mm * mm).sum()
    return E / Z / 27.0, Mabs / Z / 27.0, M2 / Z / 27.0 ** 2


def blocked_error(x, nblocks=50):
    b = np.asarray(x, dtype=np.float64)[: len(x) // nblocks * nblocks].reshape(nblocks, -1).mean(axis=1)
    return b.std(ddof=1) / math.sqrt(nblocks)


@pytest.mark.parametrize("beta", [0.2216546, 0.30])
def test_chain3_against_exact_3x3x3(beta):
    e_ex, mabs_ex, m2_ex = exact_3x3x3(beta)
    L, N = 3, 27
    T = oracle.threshold(2, beta)
    spins = oracle.init_spins3(L, 2, 77, 1)
    oracle.run_chain3(L, 2, T, 77, 0, 2000, spins)
    n = 300000
    ser = oracle.run_chain3(L, 2, T, 77, 2000, n, spins)
    e, mm = ser[:, 0] / N, ser[:, 1] / N
    for got, want in ((e, e_ex), (np.abs(mm), mabs_ex), (mm * mm, m2_ex), (ser[:, 3] / float(N * N), m2_ex)):   # last: FK identity
        assert abs(got.mean() - want) < 4.5 * blocked_error(got) + 1e-12


def test_init_spins3_is_the_2d_definition_over_N_sites_keyed_by_quad():
    """orc3_init_spins (S:8c.8 over N = L^3 sites, reading 19): k_i = (PHILOX(seed; i>>2, 0, 0, INIT=0)[i&3] q) >> 32.
    Pinned (a) to the 2D function at equal N (its own pin is the survey's golden L4_init_k) and (b) to the keying rebuilt from
    the KAT-pinned Philox primitive; a slip in the counter word (i>>1 for i>>2), the word index or the domain fails both."""
    for q, seed in ((2, 11), (3, 2 ** 40 + 7), (8, 5)):
        key = [seed & 0xFFFFFFFF, seed >> 32]
        s3 = oracle.init_spins3(4, q, seed, 1)                          # N = 64
        s2 = oracle.init_spins(8, q, seed, 1)                           # N = 64
        assert s3.shape == (64,) and np.array_equal(s3, s2)
        k3 = (1 - s3.astype(np.int64)) // 2 if q == 2 else s3.astype(np.int64)
        want = [(int(oracle.philox([i >> 2, 0, 0, 0], key)[i & 3]) * q) >> 32 for i in range(64)]
        assert k3.tolist() == want
        assert len(set(want)) > 1
        # a larger, non-power-of-two lattice through the primitive only
        s3 = oracle.init_spins3(6, q, seed, 1)
        k3 = (1 - s3.astype(np.int64)) // 2 if q == 2 else s3.astype(np.int64)
        assert k3.tolist() == [(int(oracle.philox([i >> 2, 0, 0, 0], key)[i & 3]) * q) >> 32 for i in range(216)]
        cold = oracle.init_spins3(5, q, seed, 0)
        assert (cold == (1 if q == 2 else 0)).all()


def test_flip3_is_constant_on_clusters_and_keyed_by_root():
    """orc3_flip (P:55 step 3; S:8c.6): every site takes k_r = (PHILOX(seed; r, t_lo, t_hi, FLIP=2)[0] q) >> 32 of its root r.
    The 3D twin of test_flip_is_constant_on_clusters_and_keyed_by_root, with the step counter's high word in use."""
    L, q, seed = 6, 4, 77 + (3 << 32)
    t = (5 << 32) + 9
    rng = np.random.default_rng(12)
    codes = (rng.random((L ** 3, 3)) < 0.22)
    codes = (codes[:, 0] | (codes[:, 1] << 1) | (codes[:, 2] << 2)).astype(np.uint8)
    lab, nc = oracle.label3(L, codes)
    assert 1 < nc < L ** 3
    key = [seed & 0xFFFFFFFF, seed >> 32]
    s = oracle.flip3(q, seed, t, lab)
    assert np.array_equal(s, s[lab]) and s.min() >= 0 and s.max() < q
    roots = np.unique(lab)
    for r in roots:
        w = oracle.philox([int(r), t & 0xFFFFFFFF, t >> 32, 2], key)
        assert s[r] == (int(w[0]) * q) >> 32
    assert not np.array_equal(s, oracle.flip3(q, seed, t + 1, lab))
    assert not np.array_equal(s, oracle.flip3(q, seed, t + (1 << 32), lab))      # the high word of t is part of the counter
    s2 = oracle.flip3(2, seed, t, lab)                                  # Ising storage: k=0 -> +1, k=1 -> -1
    assert set(np.unique(s2)) <= {-1, 1}
    for r in roots:
        w = oracle.philox([int(r), t & 0xFFFFFFFF, t >> 32, 2], key)
        assert s2[r] == (1 if (int(w[0]) >> 31) == 0 else -1)
