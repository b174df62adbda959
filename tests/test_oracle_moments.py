"""Pins for the oracle's moment accumulators and Binder ratio (PAPER.md:126 measurement; Eq. 3).

What fixes them, none of it the oracle itself: a series small enough to sum by hand; Python's arbitrary-precision
integers for sums that pass 2^64 and 2^96 (the reason the accumulators are 128 bits wide); the closed forms
U = 2/3 for |M| = const and U -> 0 for Gaussian M; and the exact Boltzmann value of U from brute-force enumeration
of the 4x4 and 3x3x3 lattices (0.61719932 at the 2D T_c), which a long Wolff chain's accumulated
moments must reproduce within 3 jackknife standard errors.
"""
import math
from fractions import Fraction

import numpy as np
import pytest

import oracle
from paper_1110_0899_b200 import workloads as wl
from test_oracle_sampler import binder_jackknife, exact_averages


def test_moments_of_a_series_summed_by_hand():
    E = [-8, 0, 4]
    M = [4, -2, 0]
    m = oracle.moments_dict(oracle.moments_raw(E, M))
    # by hand: n = 3; sum E = -4; sum |M| = 6; sum E^2 = 64 + 0 + 16; sum M^2 = 16 + 4 + 0; sum M^4 = 256 + 16 + 0
    assert m == {"n": 3, "sum_E": -4, "sum_absM": 6, "sum_E2": 80, "sum_M2": 20, "sum_M4": 272}
    # Eq. 3: U = 1 - (272/3) / (3 (20/3)^2) = 1 - 272*3/(3*400) = 1 - 0.68
    assert oracle.binder(oracle.moments_raw(E, M)) == pytest.approx(0.32, abs=1e-15)


def test_moments_past_64_and_96_bits_against_python_integers():
    rng = np.random.default_rng(5)
    N = 1 << 24                                   # the largest BASELINE lattice: |M| <= 2^24, |E| <= 3 * 2^24
    M = rng.integers(-N, N + 1, size=5000, dtype=np.int64)
    E = rng.integers(-3 * N, 3 * N + 1, size=5000, dtype=np.int64)
    M[:64] = N                                    # 64 * 2^96 = 2^102: the fourth moment is past 2^96 at once
    M[64:128] = -N
    m = oracle.moments_dict(oracle.moments_raw(E, M))
    Ml, El = [int(x) for x in M], [int(x) for x in E]
    assert m["n"] == 5000
    assert m["sum_E"] == sum(El) and m["sum_absM"] == sum(abs(x) for x in Ml)
    assert m["sum_E2"] == sum(x * x for x in El)
    assert m["sum_M2"] == sum(x * x for x in Ml) and m["sum_M2"] > 1 << 48
    assert m["sum_M4"] == sum(x ** 4 for x in Ml) and m["sum_M4"] > 1 << 102
    U_exact = 1 - Fraction(m["n"] * m["sum_M4"], 3 * m["sum_M2"] ** 2)
    assert oracle.binder(oracle.moments_raw(E, M)) == pytest.approx(float(U_exact), rel=1e-13)


def test_moments_continue_an_earlier_accumulation():
    rng = np.random.default_rng(6)
    M = rng.integers(-4096, 4097, size=300, dtype=np.int64)
    E = rng.integers(-8192, 8193, size=300, dtype=np.int64)
    whole = oracle.moments_raw(E, M)
    part = oracle.moments_raw(E[:100], M[:100])
    part = oracle.moments_raw(E[100:], M[100:], acc=part)
    assert np.array_equal(whole, part)
    assert oracle.moments_dict(oracle.moments_raw([], []))["n"] == 0
    assert math.isnan(oracle.binder(oracle.moments_raw([], [])))


def test_binder_closed_forms():
    # |M| = N in every sample (T -> 0): <M^4> = <M^2>^2, U = 2/3
    M = np.array([4096, -4096] * 50, dtype=np.int64)
    assert oracle.binder(oracle.moments_raw(np.zeros(100, dtype=np.int64), M)) == pytest.approx(2.0 / 3.0, abs=1e-15)
    # Gaussian M (T -> infinity, i.i.d. spins): <M^4> = 3 <M^2>^2, U -> 0 like 1/sqrt(samples)
    rng = np.random.default_rng(7)
    M = np.rint(rng.normal(0.0, 1000.0, size=400000)).astype(np.int64)
    assert abs(oracle.binder(oracle.moments_raw(np.zeros(M.size, dtype=np.int64), M))) < 0.01


@pytest.mark.parametrize("dim,L,T,seed", [(2, 4, wl.TC_2D, 111), (3, 3, wl.TC_3D, 112)])
def test_binder_of_a_long_chain_matches_exact_enumeration(dim, L, T, seed):
    o = oracle.OracleWolff(dim, L, 1.0, T, seed)
    o.run(2000)
    _, E, M = o.run_logged(400_000)
    raw = oracle.moments_raw(E, M)
    U = oracle.binder(raw)
    U_np, seU = binder_jackknife(M)                       # numpy restatement + jackknife error
    assert U == pytest.approx(U_np, abs=1e-12)
    ex = exact_averages(dim, L, T)
    assert abs(U - ex["U"]) < 3 * seU, (U, ex["U"], seU)
    assert seU < 2e-3                                     # the pin has teeth
    if dim == 2:
        assert abs(ex["U"] - 0.61719932) < 1e-7           # SURVEY.md 8(c), exact 4x4 value at T_c
    N = L ** dim
    m = oracle.moments_dict(raw)
    assert abs(m["sum_M2"] / m["n"] / N ** 2 - ex["m2"]) < 0.01
    assert abs(m["sum_E"] / m["n"] / N - ex["e"]) < 0.01
