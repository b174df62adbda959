"""Pins for the oracle's update: the flipped set IS the connected component (SURVEY.md 8(c) 'Definition').

The checker is a different algorithm from the oracle's stack walk: enumerate all dim*N bonds, keep the active
ones between two spins equal to s0, union-find, and compare component(i0) with the set of sites that changed.
Neighbour arithmetic here is numpy's, not oracle.nbr.
"""
import numpy as np
import pytest

import oracle
from paper_1110_0899_b200 import workloads as wl


def forward_neighbour_table(dim, L):
    N = L ** dim
    grid = np.arange(N).reshape((L,) * dim)          # numpy axis dim-1 is x (fastest)
    return [np.roll(grid, -1, axis=dim - 1 - d).reshape(-1) for d in range(dim)]


class UnionFind:
    def __init__(self, n):
        self.p = list(range(n))

    def find(self, a):
        while self.p[a] != a:
            self.p[a] = self.p[self.p[a]]
            a = self.p[a]
        return a

    def union(self, a, b):
        ra, rb = self.find(a), self.find(b)
        if ra != rb:
            self.p[ra] = rb


def component_by_union_find(dim, L, seed, u, thr, before):
    N = L ** dim
    i0 = oracle.site_draw(seed, u, N)
    s0 = before[i0]
    fwd = forward_neighbour_table(dim, L)
    uf = UnionFind(N)
    for d in range(dim):
        for i in range(N):
            j = int(fwd[d][i])
            if before[i] == s0 and before[j] == s0 and oracle.bond_active(seed, u, i, d, thr):
                uf.union(i, j)
    root = uf.find(i0)
    return i0, s0, {i for i in range(N) if uf.find(i) == root}


@pytest.mark.parametrize("dim,L,T,seed,n", [
    (2, 2, 2.0, 5, 40), (2, 3, 2.0, 6, 40), (2, 4, wl.TC_2D, 1, 60), (2, 6, 1.8, 2, 40), (2, 16, wl.TC_2D, 3, 40),
    (3, 2, 4.0, 7, 40), (3, 3, wl.TC_3D, 8, 40), (3, 4, wl.TC_3D, 1, 40), (3, 6, 4.0, 9, 25),
    (2, 48, wl.TC_2D, 4, 12),
])
def test_cluster_is_connected_component(dim, L, T, seed, n):
    o = oracle.OracleWolff(dim, L, 1.0, T, seed)
    if L >= 16:
        o.set_spins(wl.cold(L ** dim))          # big clusters right away
    for _ in range(n):
        u = o.update_index
        before = o.get_spins()
        size = int(o.run(1)[0])
        after = o.get_spins()
        changed = set(np.nonzero(before != after)[0].tolist())
        i0, s0, comp = component_by_union_find(dim, L, seed, u, o.threshold, before)
        assert changed == comp
        assert size == len(comp)
        assert all(before[i] == s0 and after[i] == -s0 for i in comp)     # single-signed, all flipped
        assert i0 in comp
        assert o.update_index == u + 1


def test_cluster_closed_under_active_bonds():
    # north_star invariant: no active bond joins a member to a same-sign non-member.
    dim, L, seed = 2, 12, 21
    o = oracle.OracleWolff(dim, L, 1.0, 2.0, seed)
    fwd = forward_neighbour_table(dim, L)
    for _ in range(30):
        u = o.update_index
        before = o.get_spins()
        o.run(1)
        after = o.get_spins()
        member = before != after
        s0 = before[oracle.site_draw(seed, u, L ** dim)]
        for d in range(dim):
            for i in range(L ** dim):
                j = int(fwd[d][i])
                if member[i] != member[j] and before[i] == s0 and before[j] == s0:
                    assert not oracle.bond_active(seed, u, i, d, o.threshold)


@pytest.mark.parametrize("dim,L", [(2, 8), (3, 4), (2, 2)])
def test_p_zero_flips_only_the_seed_site(dim, L):
    o = oracle.OracleWolff(dim, L, 0.0, 1.0, 3)       # J = 0 -> thr = 0
    assert o.threshold == 0
    for _ in range(50):
        u = o.update_index
        before = o.get_spins()
        assert int(o.run(1)[0]) == 1
        diff = np.nonzero(before != o.get_spins())[0]
        assert diff.tolist() == [oracle.site_draw(3, u, L ** dim)]


def flood_fill(dim, L, spins, start):
    N = L ** dim
    grid = np.arange(N).reshape((L,) * dim)
    nbrs = [np.roll(grid, sh, axis=ax).reshape(-1) for ax in range(dim) for sh in (-1, 1)]
    seen, todo = {start}, [start]
    while todo:
        i = todo.pop()
        for t in nbrs:
            j = int(t[i])
            if j not in seen and spins[j] == spins[start]:
                seen.add(j)
                todo.append(j)
    return seen


@pytest.mark.parametrize("dim,L,maker", [
    (2, 16, lambda: wl.random_pm1(256, 5)), (2, 24, lambda: wl.blobs(2, 24, 3)), (3, 8, lambda: wl.random_pm1(512, 6)),
    (3, 10, lambda: wl.blobs(3, 10, 4)), (2, 2, lambda: wl.random_pm1(4, 1)), (2, 9, lambda: wl.random_pm1(81, 2, 0.7)),
])
def test_p_one_gives_full_same_sign_component(dim, L, maker):
    o = oracle.OracleWolff(dim, L, 1.0, 0.04, 17)     # thr = 2^32: every bond active
    assert o.threshold == 1 << 32
    o.set_spins(maker())
    for _ in range(10):
        u = o.update_index
        before = o.get_spins()
        size = int(o.run(1)[0])
        comp = flood_fill(dim, L, before, oracle.site_draw(17, u, L ** dim))
        assert set(np.nonzero(before != o.get_spins())[0].tolist()) == comp
        assert size == len(comp)


def test_p_one_cold_start_flips_everything():
    for dim, L in [(2, 32), (3, 8)]:
        o = oracle.OracleWolff(dim, L, 1.0, 0.04, 1)
        o.set_spins(wl.cold(L ** dim))
        assert int(o.run(1)[0]) == L ** dim
        assert np.all(o.get_spins() == -1)
        assert o.observables() == (-dim * L ** dim, -(L ** dim))


def test_split_run_equivalence_and_resume():
    # reading R12: the update index never resets, so run(a); run(b) == run(a+b); and (lattice, u) is the whole state.
    a = oracle.OracleWolff(2, 16, 1.0, wl.TC_2D, 9)
    b = oracle.OracleWolff(2, 16, 1.0, wl.TC_2D, 9)
    sa = np.concatenate([a.run(7), a.run(13), a.run(1)])
    sb = b.run(21)
    assert np.array_equal(sa, sb) and np.array_equal(a.get_spins(), b.get_spins())
    c = oracle.OracleWolff(2, 16, 1.0, wl.TC_2D, 9)
    c.set_spins(a.get_spins())
    c.update_index = a.update_index
    assert np.array_equal(a.run(10), c.run(10)) and np.array_equal(a.get_spins(), c.get_spins())
