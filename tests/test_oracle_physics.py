"""Statistical-physics pins of the oracle's whole SW chain and Wolff step (CPU only).

What fixes the answers (none of it comes from the oracle):
  * brute-force enumeration of all 2^16 states of the 4x4 periodic Ising model, done here in numpy
    (BASELINE.json north_star; SURVEY.md 8(c) "Flip rule / whole SW chain");
  * Kaufman's exact partition function of the finite periodic lattice (the paper's own check, ref. [40]),
    implemented here from the closed form and validated against the enumeration at L=4;
  * the Fortuin-Kasteleyn identity <sum_clusters size^2> = N^2 <m^2> (the FK clusters carry the spin
    correlations), which links the oracle's LABELS to its SPINS;
  * brute-force enumeration of the q=3 and q=4 Potts models on the 3x3 torus;
  * the survey's independently computed golden vectors (tests/golden/survey_pipeline.txt).
"""
import math

import numpy as np
import pytest

import oracle
from conftest import read_golden


# ---------------------------------------------------------------- exact references ---------------------------
def enumerate_ising(L):
    """E = -sum s_i s_j and M = sum s_i of every state of the L x L torus (L=4: 65536 states)."""
    N = L * L
    states = np.arange(1 << N, dtype=np.int64)
    s = (1 - 2 * ((states[:, None] >> np.arange(N)[None, :]) & 1)).astype(np.int8).reshape(-1, L, L)
    E = -(s * np.roll(s, -1, 2)).sum(axis=(1, 2), dtype=np.int64) - (s * np.roll(s, -1, 1)).sum(axis=(1, 2), dtype=np.int64)
    M = s.sum(axis=(1, 2), dtype=np.int64)
    return E, M


def boltzmann_averages(E, M, beta, N):
    w = np.exp(-beta * (E - E.min()))
    Z = w.sum()
    e = (w * E).sum() / Z / N
    am = (w * np.abs(M)).sum() / Z / N
    m2 = (w * M.astype(float) ** 2).sum() / Z / N ** 2
    return e, am, m2, w / Z


def kaufman_lnZ(L, K):
    """ln Z of the L x L periodic Ising model, Kaufman 1949 (Phys. Rev. 76, 1232), Eq. for an n x m torus."""
    n = m = L
    r = np.arange(2 * n)
    cg = math.cosh(2 * K) / math.tanh(2 * K) - np.cos(math.pi * r / n)
    gamma = np.arccosh(np.maximum(cg, 1.0))
    gamma[0] = 2 * K + math.log(math.tanh(K))                # gamma_0 keeps its sign
    odd, even = gamma[1::2], gamma[0::2]

    def lnprod_cosh(g):
        x = m * g / 2
        return float(np.sum(np.abs(x) + np.log1p(np.exp(-2 * np.abs(x)))))      # ln prod 2 cosh x

    def lnprod_sinh(g):
        x = m * g / 2
        sign = float(np.prod(np.sign(x)))
        return float(np.sum(np.abs(x) + np.log1p(-np.exp(-2 * np.abs(x))))), sign  # ln |prod 2 sinh x|

    t1 = lnprod_cosh(odd)
    t2, s2 = lnprod_sinh(odd)
    t3 = lnprod_cosh(even)
    t4, s4 = lnprod_sinh(even)
    top = max(t1, t2, t3, t4)
    tot = math.exp(t1 - top) + s2 * math.exp(t2 - top) + math.exp(t3 - top) + s4 * math.exp(t4 - top)
    return -math.log(2) + 0.5 * n * m * math.log(2 * math.sinh(2 * K)) + top + math.log(tot)


def kaufman_energy_per_site(L, beta, h=1e-5):
    return -(kaufman_lnZ(L, beta + h) - kaufman_lnZ(L, beta - h)) / (2 * h) / (L * L)


def blocked_error(x, nblocks=50):
    x = np.asarray(x, dtype=float)
    nb = len(x) // nblocks
    means = x[: nb * nblocks].reshape(nblocks, nb).mean(axis=1)
    return means.std(ddof=1) / math.sqrt(nblocks)


BETA_C = 0.5 * math.log(1 + math.sqrt(2))


def test_kaufman_matches_enumeration_at_L4_and_onsager_limit():
    E, M = enumerate_ising(4)
    for beta in (0.3, 0.4, BETA_C, 0.5):
        e, _, _, _ = boltzmann_averages(E, M, beta, 16)
        assert abs(kaufman_energy_per_site(4, beta) - e) < 1e-8
    # values the survey quotes (SURVEY.md 8(c) "Energy at large L"), and Onsager's e(beta_c) = -sqrt 2 for L -> inf
    assert abs(kaufman_energy_per_site(64, BETA_C) - (-1.4239383898)) < 2e-8
    assert abs(kaufman_energy_per_site(1024, BETA_C) - (-1.4148214132)) < 2e-7
    assert abs(kaufman_energy_per_site(1024, BETA_C) + math.sqrt(2)) < 1e-3


# ---------------------------------------------------------------- SW chain on 4x4 -----------------------------
@pytest.mark.slow
@pytest.mark.parametrize("beta", [0.30, BETA_C, 0.50])
def test_sw_4x4_reproduces_exact_enumeration(beta):
    L, N, nsweeps = 4, 16, 2_000_000
    E, M = enumerate_ising(L)
    e_x, am_x, m2_x, prob = boltzmann_averages(E, M, beta, N)
    T = oracle.threshold(2, beta)
    s = oracle.init_spins(L, 2, 42, 1)
    ser = oracle.run_chain(L, 2, T, 42, 0, nsweeps, s)[1000:]
    e, m, ssq = ser[:, 0] / N, ser[:, 1] / N, ser[:, 3]
    assert abs(e.mean() - e_x) < 4.5 * blocked_error(e)
    assert abs(np.abs(m).mean() - am_x) < 4.5 * blocked_error(np.abs(m))
    assert abs((m ** 2).mean() - m2_x) < 4.5 * blocked_error(m ** 2)
    # FK identity: sum of squared cluster sizes of the labelling inside sweep s, averaged, equals N^2 <m^2>
    fk = ssq / N ** 2
    assert abs(fk.mean() - m2_x) < 4.5 * blocked_error(fk)
    # energy histogram against g(E) exp(-beta E)/Z: chi^2 on a thinned series (tau_int ~ 1-2 sweeps on 4x4)
    thin = ser[::10, 0]
    levels = np.unique(E)
    p_exact = np.array([prob[E == lv].sum() for lv in levels])
    obs = np.array([(thin == lv).sum() for lv in levels], dtype=float)
    exp = p_exact * thin.size
    keep = exp > 5
    chi2 = float(((obs[keep] - exp[keep]) ** 2 / exp[keep]).sum())
    dof = int(keep.sum()) - 1
    assert chi2 < dof + 6 * math.sqrt(2 * dof), (chi2, dof)
    # E=+-28 is impossible on the 4x4 torus (density of states g(28) = 0): never visited
    assert not np.any(np.abs(ser[:, 0]) == 28)


@pytest.mark.slow
def test_sw_L64_energy_matches_kaufman():
    L, nsweeps = 64, 40000
    T = oracle.threshold(2, BETA_C)
    s = oracle.init_spins(L, 2, 3, 0)                         # cold start (config 2's protocol at smaller L)
    ser = oracle.run_chain(L, 2, T, 3, 0, nsweeps, s)[500:]
    e = ser[:, 0] / (L * L)
    exact = kaufman_energy_per_site(L, BETA_C)
    err = blocked_error(e, 25)
    assert err < 1.5e-3
    assert abs(e.mean() - exact) < 4.5 * err, (e.mean(), exact, err)
    assert abs(e.mean() + math.sqrt(2)) > 3 * err            # finite-size shift is visible: compare to finite-L value


# ---------------------------------------------------------------- Potts q=3, q=4 on 3x3 -----------------------
def enumerate_potts_sat(L, q):
    N = L * L
    ids = np.arange(q ** N, dtype=np.int64)
    s = np.stack([(ids // q ** i) % q for i in range(N)], axis=1).astype(np.int8).reshape(-1, L, L)
    sat = (s == np.roll(s, -1, 2)).sum(axis=(1, 2)) + (s == np.roll(s, -1, 1)).sum(axis=(1, 2))
    return sat.astype(np.int64)


@pytest.mark.slow
@pytest.mark.parametrize("q,want", [(3, -1.742122215), (4, -1.716879642)])
def test_potts_3x3_energy_matches_enumeration(q, want):
    L, N = 3, 9
    beta = math.log(1 + math.sqrt(q))
    sat = enumerate_potts_sat(L, q)
    w = np.exp(beta * (sat - sat.max()))
    e_x = -(w * sat).sum() / w.sum() / N
    assert abs(e_x - want) < 1e-8                             # the survey's transfer-matrix value, SURVEY 8(c)
    T = oracle.threshold(q, beta)
    s = oracle.init_spins(L, q, 5, 1)
    ser = oracle.run_chain(L, q, T, 5, 0, 1_000_000, s)[1000:]
    e = ser[:, 0] / N
    assert abs(e.mean() - e_x) < 4.5 * blocked_error(e)
    assert s.min() >= 0 and s.max() < q


# ---------------------------------------------------------------- Wolff ---------------------------------------
@pytest.mark.slow
def test_wolff_4x4_reproduces_exact_enumeration():
    L, N = 4, 16
    E, M = enumerate_ising(L)
    e_x, am_x, m2_x, _ = boltzmann_averages(E, M, BETA_C, N)
    T = oracle.threshold(2, BETA_C)
    s = oracle.init_spins(L, 2, 9, 1)
    ser = oracle.wolff_chain(L, T, 9, 0, 2_000_000, s)[1000:]
    e, m, sz = ser[:, 0] / N, ser[:, 1] / N, ser[:, 2]
    assert abs(e.mean() - e_x) < 4.5 * blocked_error(e)
    assert abs(np.abs(m).mean() - am_x) < 4.5 * blocked_error(np.abs(m))
    # improved estimator: <|C|> / N = <m^2> (the FK identity for the single-cluster algorithm)
    assert abs((sz / N).mean() - m2_x) < 4.5 * blocked_error(sz / N)


def test_wolff_equals_label_then_flip_one_cluster():
    # P:330/P:334 option (a): a Wolff step is "SW-decompose, pick a site, flip its cluster"
    L, seed = 48, 21
    T = oracle.threshold(2, BETA_C)
    s = oracle.init_spins(L, 2, seed, 1)
    for t in range(40):
        before = s.copy()
        codes, _ = oracle.bonds(L, T, seed, t, before)
        lab, _ = oracle.label(L, codes)
        size, i0, root = oracle.wolff_step(L, T, seed, t, s)
        members = lab == lab[i0]
        assert root == lab[i0] and size == int(members.sum())
        want = before.copy()
        want[members] = -want[members]
        assert np.array_equal(s, want)
        assert 0 <= i0 < L * L


# ---------------------------------------------------------------- few-cluster variant -------------
def test_fewcluster_equals_decompose_select_flip():
    """The paper's own statement of the variant: full SW decomposition, select points, flip the distinct clusters
    they belong to -- each with probability p_flip.  Restated in numpy from the pinned pieces (bonds, labels, the KAT-pinned
    Philox) with the keying of DESIGN.md reading 21: seeds (k, t, WSEED)[0], flip decision (root, t, FLIP)[1] < T_flip."""
    L, seed = 24, 77 + (1 << 35)
    N = L * L
    T = oracle.threshold(2, BETA_C)
    key = [seed & 0xFFFFFFFF, seed >> 32]
    s = oracle.init_spins(L, 2, seed, 1)
    seen_partial = False
    for t, n_seeds, T_flip in [(0, 1, 0xFFFFFFFF), (1, 5, 0x80000000), (2, 40, 0xB3333333), ((7 << 32) + 3, 17, 0x40000000),
                               (4, 9, 0), (5, 0, 0xFFFFFFFF)]:
        before = s.copy()
        codes, _ = oracle.bonds(L, T, seed, t, before)
        lab, _ = oracle.label(L, codes)
        tl, th = t & 0xFFFFFFFF, t >> 32
        roots = {int(lab[(int(oracle.philox([k, tl, th, 3], key)[0]) * N) >> 32]) for k in range(n_seeds)}
        flip_roots = [r for r in sorted(roots) if int(oracle.philox([r, tl, th, 2], key)[1]) < T_flip]
        want = before.copy()
        m = np.isin(lab, flip_roots)
        want[m] = -want[m]
        f, nfc, lab_o = oracle.fewcluster_step(L, T, seed, t, n_seeds, T_flip, s)
        assert np.array_equal(lab_o, lab) and np.array_equal(s, want)
        assert f == int(m.sum()) and nfc == len(flip_roots)
        seen_partial = seen_partial or (0 < len(flip_roots) < len(roots))
    assert seen_partial                                          # some selected cluster was NOT flipped: p_flip < 1 is exercised


def test_fewcluster_with_one_seed_and_pflip_one_is_the_wolff_step():
    """n_seeds = 1, T_flip = 2^32 - 1: the seed (0, t, WSEED)[0] is the Wolff seed and its cluster is flipped (unless the one
    draw equals 2^32 - 1): the same configuration as orc_wolff_step, whose keying the survey's golden vectors pin."""
    L, seed = 32, 1234
    T = oracle.threshold(2, BETA_C)
    a = oracle.init_spins(L, 2, seed, 1)
    b = a.copy()
    for t in range(60):
        sz, i0, root = oracle.wolff_step(L, T, seed, t, a)
        f, nfc, lab = oracle.fewcluster_step(L, T, seed, t, 1, 0xFFFFFFFF, b)
        assert (f, nfc) == (sz, 1) and lab[i0] == root and np.array_equal(a, b), t


@pytest.mark.slow
def test_fewcluster_4x4_reproduces_exact_enumeration():
    """Flipping any subset of FK clusters chosen independently of the spins, each with a probability that depends on the bond
    configuration only, keeps the Boltzmann weight stationary: <E> and <|m|> of the 4 x 4 model, 3 seeds, p_flip = 0.7."""
    L, N = 4, 16
    E, M = enumerate_ising(L)
    e_x, am_x, m2_x, _ = boltzmann_averages(E, M, BETA_C, N)
    T = oracle.threshold(2, BETA_C)
    s = oracle.init_spins(L, 2, 5, 1)
    ser = oracle.fewcluster_chain(L, T, 5, 0, 1_500_000, 3, oracle.threshold_from_p(0.7), s)[1000:]
    e, m = ser[:, 0] / N, ser[:, 1] / N
    assert abs(e.mean() - e_x) < 4.5 * blocked_error(e)
    assert abs(np.abs(m).mean() - am_x) < 4.5 * blocked_error(np.abs(m))
    assert abs((m * m).mean() - m2_x) < 4.5 * blocked_error(m * m)
    assert 0 < ser[:, 2].mean() < N


def test_wolff_seed_sites_are_uniform():
    L, N = 16, 256
    T = oracle.threshold(2, 0.2)
    s = oracle.init_spins(L, 2, 4, 1)
    hits = np.zeros(N, dtype=np.int64)
    n = 20000
    for t in range(n):
        _, i0, _ = oracle.wolff_step(L, T, 4, t, s)
        hits[i0] += 1
    chi2 = float(((hits - n / N) ** 2 / (n / N)).sum())
    assert chi2 < (N - 1) + 6 * math.sqrt(2 * (N - 1))


# ---------------------------------------------------------------- golden vectors ------------------------------
def _ints(v):
    return [int(x) for x in v.split()]


def test_survey_golden_vectors_L4():
    g = read_golden("survey_pipeline.txt")
    L, T, seed = 4, 2515933592, 1234
    s = oracle.init_spins(L, 2, seed, 1)
    assert [int(x) for x in (1 - s) // 2] == _ints(g["L4_init_k"])
    for t in (0, 1):
        lab, codes, nc, nb = oracle.sweep(L, 2, T, seed, t, s)
        assert [int(x) for x in codes] == _ints(g[f"L4_t{t}_codes"])
        assert [int(x) for x in lab] == _ints(g[f"L4_t{t}_labels"])
        assert nc == int(g[f"L4_t{t}_nclusters"])
        assert [int(x) for x in (1 - s) // 2] == _ints(g[f"L4_t{t}_new_k"])
        o = oracle.observables(L, 2, s)
        assert [o["energy"], o["magnetisation"]] == _ints(g[f"L4_t{t}_E_M"])


def test_survey_golden_vectors_L64_and_wolff():
    g = read_golden("survey_pipeline.txt")
    L, T, seed = 64, 2515933592, 1234
    s = oracle.init_spins(L, 2, seed, 1)
    o = oracle.observables(L, 2, s)
    assert [o["energy"], o["magnetisation"]] == _ints(g["L64_init_E_M"])
    marks = {1: "L64_sweep1", 2: "L64_sweep2", 10: "L64_sweep10", 100: "L64_sweep100"}
    lab = None
    for t in range(100):
        lab, codes, nc, nb = oracle.sweep(L, 2, T, seed, t, s)
        if t + 1 in marks:
            o = oracle.observables(L, 2, s)
            assert [nc, nb, o["energy"], o["magnetisation"]] == _ints(g[marks[t + 1]]), t + 1
    assert oracle.fnv1a64(((1 - s) // 2).astype(np.uint8)) == int(g["L64_fnv_k_after100"], 16)
    assert oracle.fnv1a64(lab.astype("<i4")) == int(g["L64_fnv_labels_sweep99"], 16)
    s = oracle.init_spins(L, 2, seed, 1)
    seeds, roots, sizes, Es, Ms = [], [], [], [], []
    for t in range(5):
        sz, i0, r = oracle.wolff_step(L, T, seed, t, s)
        o = oracle.observables(L, 2, s)
        seeds.append(i0), roots.append(r), sizes.append(sz), Es.append(o["energy"]), Ms.append(o["magnetisation"])
    assert seeds == _ints(g["wolff_seed_sites"]) and roots == _ints(g["wolff_roots"])
    assert sizes == _ints(g["wolff_sizes"]) and Es == _ints(g["wolff_E"]) and Ms == _ints(g["wolff_M"])
