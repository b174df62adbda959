"""Pins for the oracle as a SAMPLER: long Wolff chains must reproduce exact Boltzmann averages.

Exact values come from (a) brute-force enumeration of all states of the 4x4 (2^16) and 3x3x3 (2^27) periodic
lattices (oracle/ising_enum.c, independent of the Wolff code) and (b) Kaufman's closed-form partition function of
the finite m x n torus, itself checked against the enumeration below.  Criterion: 3 binned standard errors
(north_star: 'must agree with long Wolff runs within 3 standard errors').  Seeds are fixed, so outcomes are
deterministic.
"""
import math

import numpy as np
import pytest

import oracle
from paper_1110_0899_b200 import workloads as wl


# ------------------------------------------------------------------ exact averages from the joint density of states

_dos_cache = {}


def dos(dim, L):
    if (dim, L) not in _dos_cache:
        _dos_cache[(dim, L)] = oracle.joint_density_of_states(dim, L)
    return _dos_cache[(dim, L)]


def exact_averages(dim, L, T, J=1.0):
    g = dos(dim, L).astype(np.float64)
    N = L ** dim
    E = np.arange(-dim * N, dim * N + 1, dtype=np.float64)[:, None]
    M = np.arange(-N, N + 1, dtype=np.float64)[None, :]
    w = g * np.exp(-(J / T) * (E - E.min()))
    Z = w.sum()
    avg = lambda f: float((w * f).sum() / Z)
    m2, m4 = avg(M ** 2), avg(M ** 4)
    return {"e": avg(E) / N, "absm": avg(np.abs(M)) / N, "m2": m2 / N ** 2, "U": 1 - m4 / (3 * m2 ** 2),
            "C": m2 / N}


def test_enumeration_4x4_density_of_states():
    # g(E) of the 4x4 torus; values restated from SURVEY.md 8(c) and checked against total count and symmetry.
    g = dos(2, 4)
    assert int(g.sum()) == 2 ** 16
    gE = {int(E): int(c) for E, c in zip(range(-32, 33), g.sum(axis=1)) if c}
    assert gE == {-32: 2, -24: 32, -20: 64, -16: 424, -12: 1728, -8: 6688, -4: 13568, 0: 20524,
                  4: 13568, 8: 6688, 12: 1728, 16: 424, 20: 64, 24: 32, 32: 2}
    assert np.array_equal(g, g[:, ::-1])               # M -> -M symmetry
    ex = exact_averages(2, 4, wl.TC_2D)
    assert abs(ex["e"] - (-1.56562379)) < 1e-7 and abs(ex["absm"] - 0.84386044) < 1e-7


def test_enumeration_3x3x3_density_of_states():
    g = dos(3, 3)
    assert int(g.sum()) == 2 ** 27
    gE = g.sum(axis=1)
    first = [(int(E), int(c)) for E, c in zip(range(-81, 82), gE) if c][:6]
    assert first == [(-81, 2), (-69, 54), (-61, 162), (-57, 594), (-53, 648), (-49, 3402)]
    assert np.array_equal(g, g[:, ::-1])
    # independent cross-check of the enumerator: high-temperature moments.  At T = infinity spins are i.i.d.:
    # <E> = 0, <E^2> = number of bonds = 81, <M^2> = N = 27.
    E = np.arange(-81, 82, dtype=np.float64)
    M = np.arange(-27, 28, dtype=np.float64)
    gf = g.astype(np.float64) / 2.0 ** 27
    assert abs((gf.sum(axis=1) * E).sum()) < 1e-9
    assert abs((gf.sum(axis=1) * E ** 2).sum() - 81) < 1e-9
    assert abs((gf.sum(axis=0) * M ** 2).sum() - 27) < 1e-9


# ------------------------------------------------------------------ Wolff chains vs exact

def binned(x, nbins=200):
    x = np.asarray(x, dtype=np.float64)
    n = (len(x) // nbins) * nbins
    b = x[:n].reshape(nbins, -1).mean(axis=1)
    return b.mean(), b.std(ddof=1) / math.sqrt(nbins), b


def binder_jackknife(M, nbins=200):
    M = np.asarray(M, dtype=np.float64)
    n = (len(M) // nbins) * nbins
    m2 = (M[:n] ** 2).reshape(nbins, -1).mean(axis=1)
    m4 = (M[:n] ** 4).reshape(nbins, -1).mean(axis=1)
    U = 1 - m4.mean() / (3 * m2.mean() ** 2)
    jk = np.array([1 - np.delete(m4, k).mean() / (3 * np.delete(m2, k).mean() ** 2) for k in range(nbins)])
    return U, math.sqrt((nbins - 1) * ((jk - jk.mean()) ** 2).mean())


CASES = [
    (2, 4, wl.TC_2D, 101), (2, 4, 2.0, 102), (2, 4, 3.0, 103),
    (3, 3, wl.TC_3D, 104), (3, 3, 4.0, 105), (3, 3, 5.0, 106),
]


@pytest.mark.parametrize("dim,L,T,seed", CASES)
def test_wolff_chain_matches_exact_enumeration(dim, L, T, seed):
    N = L ** dim
    o = oracle.OracleWolff(dim, L, 1.0, T, seed)
    o.run(2000)                                        # equilibrate
    sizes, E, M = o.run_logged(1_000_000)
    ex = exact_averages(dim, L, T)
    for name, series, scale in [("e", E, 1.0 / N), ("absm", np.abs(M), 1.0 / N), ("m2", M.astype(np.float64) ** 2, 1.0 / N ** 2)]:
        mean, se, _ = binned(np.asarray(series, dtype=np.float64) * scale)
        assert abs(mean - ex[name]) < 3 * se, (name, mean, ex[name], se)
        assert se < 0.01 * max(abs(ex[name]), 0.05)    # the test has teeth: errors are at the 1e-3 level or below
    U, seU = binder_jackknife(M)
    assert abs(U - ex["U"]) < 3 * seU, (U, ex["U"], seU)
    # Wolff improved estimator: <|C|> = <M^2>/N ties the size log to the magnetisation.
    # sizes[k] is the cluster grown from the state BEFORE update k, M[k] is measured after; both are stationary.
    meanC, seC, _ = binned(sizes)
    assert abs(meanC - ex["C"]) < 3 * seC, (meanC, ex["C"], seC)


def test_survey_quoted_exact_values():
    ex = exact_averages(2, 4, wl.TC_2D)
    assert abs(ex["m2"] - 0.76135891) < 1e-7 and abs(ex["U"] - 0.61719932) < 1e-7 and abs(ex["C"] - 12.18174254) < 1e-6
    assert abs(exact_averages(2, 4, 2.0)["e"] + 1.75538029) < 1e-7
    assert abs(exact_averages(2, 4, 3.0)["absm"] - 0.60129133) < 1e-7
    ex3 = exact_averages(3, 3, wl.TC_3D)
    assert abs(ex3["e"] + 1.43444029) < 1e-7 and abs(ex3["absm"] - 0.59082488) < 1e-7
    assert abs(ex3["m2"] - 0.42300072) < 1e-7 and abs(ex3["C"] - 11.42101954) < 1e-6 and abs(ex3["U"] - 0.50132209) < 1e-7


# ------------------------------------------------------------------ Kaufman's finite-torus solution (2D, larger L)

def kaufman_log_Z(n, m, K):
    """ln Z of the n x m periodic square lattice, B. Kaufman, Phys. Rev. 76, 1232 (1949), in mpmath precision."""
    import mpmath as mp
    K = mp.mpf(K)
    gam = []
    for l in range(2 * n):
        if l == 0:
            gam.append(2 * K + mp.log(mp.tanh(K)))
        else:
            c = mp.cosh(2 * K) * mp.coth(2 * K) - mp.cos(mp.pi * l / n)
            gam.append(mp.acosh(c))
    P1 = mp.fprod(2 * mp.cosh(m * gam[2 * r + 1] / 2) for r in range(n))
    P2 = mp.fprod(2 * mp.sinh(m * gam[2 * r + 1] / 2) for r in range(n))
    P3 = mp.fprod(2 * mp.cosh(m * gam[2 * r] / 2) for r in range(n))
    P4 = mp.fprod(2 * mp.sinh(m * gam[2 * r] / 2) for r in range(n))
    return mp.log(mp.mpf(1) / 2) + (mp.mpf(n * m) / 2) * mp.log(2 * mp.sinh(2 * K)) + mp.log(P1 + P2 + P3 + P4)


def kaufman_energy_per_site(L, T):
    import mpmath as mp
    mp.mp.dps = 60
    K = mp.mpf(1) / mp.mpf(T)
    return float(-mp.diff(lambda k: kaufman_log_Z(L, L, k), K) / (L * L))


def test_kaufman_formula_against_enumeration():
    import mpmath as mp
    mp.mp.dps = 60
    for L in (3, 4):
        g = dos(2, L).sum(axis=1)
        N = L * L
        for T in (1.5, wl.TC_2D, 2.5, 4.0):
            K = mp.mpf(1) / mp.mpf(T)
            Z = mp.fsum(int(c) * mp.exp(-K * E) for E, c in zip(range(-2 * N, 2 * N + 1), g) if c)
            assert abs(kaufman_log_Z(L, L, K) - mp.log(Z)) < mp.mpf(10) ** -40
        assert abs(kaufman_energy_per_site(L, 2.0) - exact_averages(2, L, 2.0)["e"]) < 1e-10


@pytest.mark.parametrize("L,T,seed,n", [(16, wl.TC_2D, 201, 60000), (32, wl.TC_2D, 202, 30000), (24, 2.6, 203, 60000)])
def test_wolff_chain_matches_kaufman_energy(L, T, seed, n):
    o = oracle.OracleWolff(2, L, 1.0, T, seed)
    o.set_spins(wl.cold(L * L))
    o.run(500)
    _, E, _ = o.run_logged(n)
    mean, se, _ = binned(E / float(L * L), nbins=100)
    exact = kaufman_energy_per_site(L, T)
    assert abs(mean - exact) < 3 * se, (mean, exact, se)
    assert se < 2e-3


def test_onsager_band_large_L():
    # north_star: at T_c the 2D energy per spin approaches Onsager's -sqrt 2 for large L (loose band 1/L).
    L = 64
    o = oracle.OracleWolff(2, L, 1.0, wl.TC_2D, 301)
    o.set_spins(wl.cold(L * L))
    o.run(300)
    _, E, _ = o.run_logged(6000)
    mean, se, _ = binned(E / float(L * L), nbins=50)
    assert abs(mean + math.sqrt(2)) < 1.0 / L
    assert mean < -math.sqrt(2)                        # approached from below on a torus
    assert abs(mean - kaufman_energy_per_site(L, wl.TC_2D)) < 3 * se
