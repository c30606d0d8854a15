"""Pins for the oracle's Philox, thresholds, initialisation and bond rule (all CPU, -m "not gpu").

Nothing here retypes the oracle's formulae: Philox is pinned to the published Random123 known answers and to a
second implementation's keying examples (tests/golden/philox_kat.txt); thresholds to closed forms evaluated in
50-digit decimal arithmetic; the bond rule to its special cases and to the binomial law of the draws.
"""
from decimal import Decimal, getcontext
import math

import numpy as np
import pytest

import oracle
from conftest import read_golden
from paper_1105_5804_b200 import inputs


def test_philox_known_answers():
    for name, line in read_golden("philox_kat.txt").items():
        ctr, key, want = [[int(w, 16) for w in part.split()] for part in line.split("|")]
        got = oracle.philox(ctr, key)
        assert [int(x) for x in got] == want, name


def test_philox_is_a_bijection_of_the_counter_lowbits():
    # distinct counters -> distinct outputs (Philox is a permutation of the 128-bit counter for a fixed key)
    outs = {tuple(int(x) for x in oracle.philox([c, 0, 0, 1], [7, 9])) for c in range(4096)}
    assert len(outs) == 4096


def _floor_p_2_32(p: Decimal) -> int:
    return int((p * Decimal(2 ** 32)).to_integral_value(rounding="ROUND_FLOOR"))


def test_thresholds_closed_forms():
    getcontext().prec = 60
    g = {k: int(v) for k, v in read_golden("thresholds.txt").items()}
    sqrt2, sqrt3 = Decimal(2).sqrt(), Decimal(3).sqrt()
    # Ising +-1 convention: p = 1 - exp(-2 beta); at beta_c = ln(1+sqrt2)/2, exp(-2 beta_c) = 1/(1+sqrt2) = sqrt2-1
    assert _floor_p_2_32(2 - sqrt2) == g["ising_beta_c"] == oracle.threshold(2, oracle.beta_c(2))
    assert _floor_p_2_32(1 - (Decimal(-2) * Decimal("0.40")).exp()) == g["ising_0.40"] == oracle.threshold(2, 0.40)
    assert _floor_p_2_32(1 - (Decimal(-2) * Decimal("0.50")).exp()) == g["ising_0.50"] == oracle.threshold(2, 0.50)
    # Potts delta convention: p = 1 - exp(-beta); beta_c = ln(1+sqrt q)
    assert _floor_p_2_32(Decimal(2) / Decimal(3)) == g["potts4_beta_c"] == oracle.threshold(4, math.log(3.0))
    assert _floor_p_2_32(sqrt3 / (1 + sqrt3)) == g["potts3_beta_c"] == oracle.threshold(3, oracle.beta_c(3))
    for name, p in (("perc_0.3", "0.3"), ("perc_0.5", "0.5"), ("perc_0.7", "0.7")):
        # the double nearest to 0.3 / 0.7 is what a caller passes; floor of that times 2^32
        assert _floor_p_2_32(Decimal(float(p))) == g[name] == oracle.threshold_from_p(float(p)), name
    assert oracle.threshold(2, 0.0) == 0
    assert oracle.threshold(2, 1e9) == 2 ** 32 - 1       # clamped: p -> 1


def test_init_cold_and_random_statistics():
    for q in (2, 3, 4, 8):
        cold = oracle.init_spins(16, q, 5, 0)
        assert np.all(cold == (1 if q == 2 else 0))
        s = oracle.init_spins(256, q, 99, 1)
        k = ((1 - s) // 2) if q == 2 else s
        cnt = np.bincount(k.astype(np.int64), minlength=q)
        assert cnt.sum() == 256 * 256 and len(cnt) == q
        n = 256 * 256
        sigma = math.sqrt(n * (1 / q) * (1 - 1 / q))
        assert np.all(np.abs(cnt - n / q) < 5 * sigma), (q, cnt)
    # different seeds give different configurations, same seed the same
    a, b, c = oracle.init_spins(64, 2, 1, 1), oracle.init_spins(64, 2, 1, 1), oracle.init_spins(64, 2, 2, 1)
    assert np.array_equal(a, b) and not np.array_equal(a, c)


@pytest.mark.parametrize("q", [2, 3, 4])
def test_bond_rule_special_cases(q):
    L = 32
    s = inputs.random_spins(L, q, 11)
    sq = s.reshape(L, L)
    eq_e = (sq == np.roll(sq, -1, axis=1)).reshape(-1)      # east neighbour  (x+1 mod L, y)
    eq_n = (sq == np.roll(sq, -1, axis=0)).reshape(-1)      # north neighbour (x, y+1 mod L)
    codes, n = oracle.bonds(L, 0, 3, 0, s)                  # T = 0: no bond ever
    assert n == 0 and not codes.any()
    codes, n = oracle.bonds(L, 2 ** 32 - 1, 3, 0, s)        # T = max: every satisfied bond (up to 2^-32 each)
    assert np.array_equal(codes & 1, eq_e.astype(np.uint8))
    assert np.array_equal((codes >> 1) & 1, eq_n.astype(np.uint8))
    assert n == int(eq_e.sum() + eq_n.sum())
    for t in range(3):                                      # never joins unequal spins, for any T, t
        codes, n = oracle.bonds(L, 2515933592, 3, t, s)
        assert not np.any((codes & 1).astype(bool) & ~eq_e)
        assert not np.any(((codes >> 1) & 1).astype(bool) & ~eq_n)
        assert n == int((codes & 1).sum() + ((codes >> 1) & 1).sum())


def test_bond_density_is_p_times_satisfied_fraction():
    L, T = 256, 2515933592                                   # p = 2 - sqrt 2
    p = T / 2.0 ** 32
    s = oracle.init_spins(L, 2, 7, 0)                        # cold: all 2N bonds satisfied
    tot = 0
    for t in range(4):
        codes, n = oracle.bonds(L, T, 7, t, s)
        tot += n
    nb = 4 * 2 * L * L
    assert abs(tot - p * nb) < 5 * math.sqrt(nb * p * (1 - p))
    # east and north separately, and the draws of different sweeps / seeds differ
    c0, _ = oracle.bonds(L, T, 7, 0, s)
    c1, _ = oracle.bonds(L, T, 7, 1, s)
    c2, _ = oracle.bonds(L, T, 8, 0, s)
    assert not np.array_equal(c0, c1) and not np.array_equal(c0, c2)
    for bit in (0, 1):
        k = int(((c0 >> bit) & 1).sum())
        assert abs(k - p * L * L) < 5 * math.sqrt(L * L * p * (1 - p))
    # no correlation between the east and north draws of a site: P(both) = p^2
    both = int((c0 == 3).sum())
    assert abs(both - p * p * L * L) < 5 * math.sqrt(L * L * p * p * (1 - p * p))


def test_bond_draw_keying_uses_pair_counter_and_word_index():
    # u(i,d,t) = PHILOX(seed; i>>1, t_lo, t_hi, BOND=1)[2 (i&1) + d].  Rebuild the codes of a cold
    # lattice from raw Philox calls made through the (KAT-pinned) primitive and compare.
    L, T, seed, t = 8, 1288490188, 0xDEADBEEFCAFEF00D, (5 << 32) | 17
    s = oracle.init_spins(L, 2, seed, 0)
    codes, _ = oracle.bonds(L, T, seed, t, s)
    key = [seed & 0xFFFFFFFF, seed >> 32]
    for i in range(L * L):
        w = oracle.philox([i >> 1, t & 0xFFFFFFFF, t >> 32, 1], key)
        e = int(w[2 * (i & 1)] < T)
        n = int(w[2 * (i & 1) + 1] < T)
        assert codes[i] == e | (n << 1), i


def test_pack_unpack_roundtrip_matches_boundary_layout():
    codes = inputs.random_bond_codes(16, 0.5, 0.5, 3)
    packed = oracle.pack_bonds(codes)
    assert np.array_equal(packed, inputs.pack_codes(codes))
    assert np.array_equal(oracle.unpack_bonds(packed, codes.size), codes)
    assert np.array_equal(inputs.unpack_codes(packed), codes)
