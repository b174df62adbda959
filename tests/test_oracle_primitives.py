"""Pins for the oracle's primitives: Philox, threshold, site draw, indexing, start lattice, observables.

Every expected value here comes from outside the oracle: published known-answer vectors, exact integer
arithmetic, closed forms, or brute force written independently in numpy.
"""
import math
import os

import numpy as np
import pytest

import oracle
from paper_1110_0899_b200 import workloads as wl


# ------------------------------------------------------------------ Philox4x32-10 (reading R11)

def test_philox_known_answers(golden_dir):
    rows = []
    with open(os.path.join(golden_dir, "philox4x32_10_kat.txt")) as f:
        for line in f:
            if line.startswith("#") or not line.strip():
                continue
            rows.append([int(x, 16) for x in line.split()])
    assert len(rows) == 3
    for r in rows:
        assert oracle.philox4x32_10(r[0:4], r[4:6]) == tuple(r[6:10])


def test_philox_bit_balance_and_avalanche():
    # Property pin: flipping one counter bit changes about half of the 128 output bits.
    rng = np.random.default_rng(7)
    flips = []
    for _ in range(200):
        ctr = [int(x) for x in rng.integers(0, 2**32, size=4)]
        key = [int(x) for x in rng.integers(0, 2**32, size=2)]
        a = oracle.philox4x32_10(ctr, key)
        w, b = int(rng.integers(0, 4)), int(rng.integers(0, 32))
        ctr2 = list(ctr)
        ctr2[w] ^= 1 << b
        c = oracle.philox4x32_10(ctr2, key)
        flips.append(sum(bin(x ^ y).count("1") for x, y in zip(a, c)))
    assert 60 < np.mean(flips) < 68


# ------------------------------------------------------------------ threshold (readings R1, R7, R14)

def test_threshold_closed_form_2d_tc():
    # p = 1 - exp(-2/T_c) = 1 - 1/(1+sqrt2)^... ; with T_c = 2/ln(1+sqrt2): exp(-2/T_c) = 1/(1+sqrt2) = sqrt2 - 1,
    # so p = 2 - sqrt2 exactly and floor(p * 2^32) = 2^33 - ceil(sqrt2 * 2^32) in exact integer arithmetic.
    ceil_sqrt2_scaled = math.isqrt(2 << 64) + 1          # sqrt2 * 2^32 is irrational -> ceil = floor + 1
    exact = (1 << 33) - ceil_sqrt2_scaled
    assert exact == 0x95F61998
    assert oracle.threshold(1.0, wl.TC_2D) == exact


def test_threshold_limits_and_monotone():
    assert oracle.threshold(0.0, 1.0) == 0                     # J = 0 -> p = 0
    assert oracle.threshold(1.0, 0.04) == 1 << 32              # 2J/T = 50 -> p rounds to 1.0 -> always active
    ts = np.linspace(0.5, 10.0, 200)
    thr = [oracle.threshold(1.0, float(t)) for t in ts]
    assert all(a >= b for a, b in zip(thr, thr[1:]))           # p decreases with T
    for t, v in zip(ts, thr):
        p = 1.0 - math.exp(-2.0 / t)
        assert abs(v / 2**32 - p) < 1e-9


def test_threshold_values_quoted_in_design():
    # Exact big-rational check of floor(p * 2^32) for the other BASELINE temperatures, using Python's
    # fractions on a 60-digit Taylor series of exp (independent of libm's expm1).
    from fractions import Fraction

    def exact_thr(two_beta: Fraction) -> int:
        term, total = Fraction(1), Fraction(1)
        for k in range(1, 80):
            term = term * (-two_beta) / k
            total += term
        p = 1 - total
        return int(p * (1 << 32))       # floor for positive p

    assert oracle.threshold(1.0, wl.TC_3D) == exact_thr(Fraction(2) / Fraction("4.511528")) == 0x5BABDAA8
    assert oracle.threshold(1.0, 5.0) == exact_thr(Fraction(2, 5)) == 0x5465E7CC
    assert oracle.threshold(1.0, 2.269185) == exact_thr(Fraction(2) / Fraction("2.269185")) == 0x95F61A71


# ------------------------------------------------------------------ site draw (reading R8)

def test_site_draw_range_and_pow2_exactness():
    seed = 12345
    for N in (2, 7, 16, 4096, 1000003, 2**24, 2**31):
        for u in range(50):
            i0 = oracle.site_draw(seed, u, N)
            assert 0 <= i0 < N
    # For N = 2^k the draw must equal the top k bits of r = x0 | x1 << 32 of the SITE-domain Philox block.
    for u in (0, 1, 2, 99, 2**33 + 5):
        x = oracle.philox4x32_10([0, 1 << 30, u & 0xFFFFFFFF, u >> 32], [seed & 0xFFFFFFFF, seed >> 32])
        r = x[0] | (x[1] << 32)
        for k in (1, 4, 12, 24, 31):
            assert oracle.site_draw(seed, u, 1 << k) == r >> (64 - k)
        assert oracle.site_draw(seed, u, 1000003) == (r * 1000003) >> 64


def test_site_draw_uniform_chi2():
    N, n = 64, 200_000
    counts = np.zeros(N)
    for u in range(n):
        counts[oracle.site_draw(1, u, N)] += 1
    chi2 = ((counts - n / N) ** 2 / (n / N)).sum()
    # 63 degrees of freedom: mean 63, sd 11.2; 5 sd band
    assert 63 - 56 < chi2 < 63 + 56


# ------------------------------------------------------------------ neighbours / edges (readings R5, R6)

@pytest.mark.parametrize("dim,L", [(2, 2), (2, 3), (2, 5), (2, 8), (3, 2), (3, 3), (3, 4), (3, 6)])
def test_neighbours_brute_force(dim, L):
    N = L ** dim
    coords = np.stack(np.unravel_index(np.arange(N), (L,) * dim)[::-1], axis=1)   # columns x, y, (z); x fastest
    weights = np.array([L ** k for k in range(dim)])
    edge_cover = {}
    for i in range(N):
        assert (coords[i] * weights).sum() == i
        for d in range(dim):
            for sign in (+1, -1):
                c = coords[i].copy()
                c[d] = (c[d] + sign) % L
                expect = int((c * weights).sum())
                j = oracle.nbr(dim, L, i, d, sign)
                assert j == expect
                assert oracle.nbr(dim, L, j, d, -sign) == i
                owner = i if sign > 0 else j
                edge_cover[(owner, d)] = edge_cover.get((owner, d), 0) + 1
    # every one of the dim*N undirected edges is looked at exactly twice (once from each end)
    assert len(edge_cover) == dim * N
    assert set(edge_cover.values()) == {2}


# ------------------------------------------------------------------ bond variable layout (readings R6, R10)

def test_bond_layout_recomputed_from_the_philox_block():
    """oracle.bond_active is word d of Philox(key = seed, ctr = (owner_lo, BOND << 30 | owner_hi, u_lo, u_hi)) < thr: the block
    is recomputed here from the documented layout (R10) with the known-answer-pinned Philox, for seeds with a high
    word, update indices beyond 2^32 and owners up to 2^31 - 1.  A bond stream that ignored u, the seed's high word, the
    direction or the domain tag fails here."""
    rng = np.random.default_rng(20260611)
    for _ in range(400):
        seed = int(rng.integers(0, 1 << 63)) * 2 + int(rng.integers(0, 2))
        u = int(rng.integers(0, 1 << 40)) + (int(rng.integers(0, 2)) << 45)
        owner = int(rng.integers(0, 1 << 31))
        d = int(rng.integers(0, 3))
        thr = int(rng.integers(0, (1 << 32) + 1))
        x = oracle.philox4x32_10([owner & 0xFFFFFFFF, (0 << 30) | (owner >> 32), u & 0xFFFFFFFF, u >> 32],
                                 [seed & 0xFFFFFFFF, seed >> 32])
        assert oracle.bond_active(seed, u, owner, d, thr) == (x[d] < thr)
        # the same counter in the SITE / INIT domains is another block: the three streams are disjoint
        assert x != oracle.philox4x32_10([owner & 0xFFFFFFFF, 1 << 30, u & 0xFFFFFFFF, u >> 32], [seed & 0xFFFFFFFF, seed >> 32])
    # thr = 0: no bond; thr = 2^32: every bond
    assert not any(oracle.bond_active(5, 9, o, d, 0) for o in range(200) for d in range(3))
    assert all(oracle.bond_active(5, 9, o, d, 1 << 32) for o in range(200) for d in range(3))


def test_bond_stream_depends_on_update_seed_and_direction_and_has_the_right_density():
    thr = oracle.threshold(1.0, wl.TC_2D)
    p = thr / 2.0 ** 32
    n = 10_000
    base = np.array([oracle.bond_active(77, 3, o, 0, thr) for o in range(n)])
    sd_diff = (n * 2 * p * (1 - p) * (1 - 2 * p * (1 - p))) ** 0.5      # two independent streams differ with prob. 2 p (1 - p)
    for other in (np.array([oracle.bond_active(77, 4, o, 0, thr) for o in range(n)]),                    # next update
                  np.array([oracle.bond_active(77, 3 + (1 << 32), o, 0, thr) for o in range(n)]),        # high word of u
                  np.array([oracle.bond_active(77 + (1 << 32), 3, o, 0, thr) for o in range(n)]),        # high word of the seed
                  np.array([oracle.bond_active(77, 3, o, 1, thr) for o in range(n)])):                   # other direction
        assert abs(int((base != other).sum()) - n * 2 * p * (1 - p)) < 5 * sd_diff
    # active fraction over 10^5 edges = thr / 2^32 within 4 sigma (p = 1 - exp(-2 J / T))
    m = 100_000
    act = sum(oracle.bond_active(123456789, 11, o % 50_000, o // 50_000, thr) for o in range(m))
    assert abs(act - m * p) < 4 * (m * p * (1 - p)) ** 0.5
    assert abs(p - (1 - np.exp(-2 / wl.TC_2D))) < 1e-9


# ------------------------------------------------------------------ start lattice (reading R9)

def test_start_lattice_bits_and_balance():
    seed = 1
    o = oracle.OracleWolff(2, 64, 1.0, wl.TC_2D, seed)
    s = o.get_spins()
    assert set(np.unique(s)) == {-1, 1}
    for i in (0, 1, 31, 32, 127, 128, 4095):
        b = i >> 7
        x = oracle.philox4x32_10([b, 2 << 30, 0, 0], [seed, 0])
        bit = (x[(i >> 5) & 3] >> (i & 31)) & 1
        assert s[i] == (1 if bit else -1) == oracle.init_spin(seed, i)
    assert abs(int(s.sum())) < 5 * 64          # 5 sigma of a fair coin on 4096 sites
    # different seeds give different lattices; same seed the same
    assert np.array_equal(s, oracle.OracleWolff(2, 64, 1.0, wl.TC_2D, seed).get_spins())
    assert not np.array_equal(s, oracle.OracleWolff(2, 64, 1.0, wl.TC_2D, seed + 1).get_spins())


def test_create_rejects_bad_arguments():
    for args in [(1, 8, 1.0, 1.0, 0), (4, 8, 1.0, 1.0, 0), (2, 1, 1.0, 1.0, 0), (2, 8, -1.0, 1.0, 0),
                 (2, 8, 1.0, 0.0, 0), (2, 8, 1.0, float("nan"), 0), (3, 2048, 1.0, 1.0, 0)]:
        with pytest.raises(ValueError):
            oracle.OracleWolff(*args)


# ------------------------------------------------------------------ observables (reading R13)

@pytest.mark.parametrize("dim,L", [(2, 2), (2, 4), (2, 6), (3, 2), (3, 4), (3, 6)])
def test_observables_closed_forms(dim, L):
    N = L ** dim
    o = oracle.OracleWolff(dim, L, 1.0, 2.0, 3)
    o.set_spins(wl.cold(N, +1))
    assert o.observables() == (-dim * N, N)
    o.set_spins(wl.cold(N, -1))
    assert o.observables() == (-dim * N, -N)
    o.set_spins(wl.checkerboard(dim, L))            # L even: every bond frustrated
    assert o.observables() == (+dim * N, 0)
    o.set_spins(wl.stripes(dim, L, 1, axis=0))      # x-bonds frustrated, the other dim-1 directions satisfied
    assert o.observables() == (N - (dim - 1) * N, 0)


def test_observables_vs_numpy_roll():
    for dim, L in [(2, 7), (3, 5), (2, 16)]:
        N = L ** dim
        s = wl.random_pm1(N, seed=11)
        o = oracle.OracleWolff(dim, L, 1.0, 2.0, 3)
        o.set_spins(s)
        g = s.reshape((L,) * dim).astype(np.int64)
        E = -sum(int((g * np.roll(g, -1, axis=ax)).sum()) for ax in range(dim))
        assert o.observables() == (E, int(g.sum()))
