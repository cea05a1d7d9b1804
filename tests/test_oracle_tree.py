"""Pins for oracle.Tree (O3 tree, O4 moments): PAPER.md:147-151 (octree, Eq. 14), :173 (bounding box)."""
import math

import numpy as np
import pytest

import ffgen
import oracle
from helpers import brute_tree, canonical_from_oracle, morton_keys_numpy


def _check_invariants(tree, pos):
    nd = tree.nodes()
    key, perm = tree.keys()
    N = len(pos)
    assert sorted(perm.tolist()) == list(range(N))                       # a permutation
    assert (np.diff(key.astype(np.int64)) >= 0).all()                    # keys non-decreasing
    ties = np.diff(key.astype(np.int64)) == 0
    assert (np.diff(perm)[ties] > 0).all()                               # stable: ties keep caller order
    assert nd["first"][0] == 0 and nd["count"][0] == N and nd["level"][0] == 0
    covered = np.zeros(N, int)
    for i in range(tree.n_nodes):
        f, c, l, p = int(nd["first"][i]), int(nd["count"][i]), int(nd["level"][i]), int(nd["prefix"][i])
        assert c >= 1
        assert ((key[f:f + c].astype(np.int64) >> (3 * (10 - l))) == p).all()   # every particle has its cell's prefix
        if f > 0:
            assert (int(key[f - 1]) >> (3 * (10 - l))) != p              # the range is the WHOLE cell
        if f + c < N:
            assert (int(key[f + c]) >> (3 * (10 - l))) != p
        if nd["is_leaf"][i]:
            assert c <= tree.nleaf or l == 10
            covered[f:f + c] += 1
        else:
            assert c > tree.nleaf and l < 10
            ch = nd["child"][i][nd["child"][i] >= 0]
            assert nd["count"][ch].sum() == c                            # children partition the parent
            assert nd["first"][ch][0] == f
            assert (nd["first"][ch][1:] == nd["first"][ch][:-1] + nd["count"][ch][:-1]).all()
            assert (nd["level"][ch] == l + 1).all()
            for o in range(8):
                if nd["child"][i][o] >= 0:
                    assert nd["prefix"][nd["child"][i][o]] == (p << 3 | o)
    assert (covered == 1).all()                                          # leaves partition [0, N)


@pytest.mark.parametrize("N,nleaf,seed", [(1, 1, 0), (2, 1, 0), (7, 1, 1), (64, 1, 2), (64, 4, 3), (33, 1, 4), (50, 8, 5)])
def test_matches_brute_force_prefix_grouping(N, nleaf, seed):
    pos = ffgen.uniform_points(N, 5.0, seed)
    t = oracle.Tree(pos, nleaf)
    nodes, sk, perm, lo, S = brute_tree(pos, nleaf)
    assert canonical_from_oracle(t) == nodes
    key, operm = t.keys()
    assert np.array_equal(key, sk) and np.array_equal(operm, perm)
    olo, oS = t.bbox()
    assert np.array_equal(olo, lo) and oS == S
    _check_invariants(t, pos)


def test_invariants_on_config1(cfg1):
    t = oracle.Tree(cfg1["pos"])
    _check_invariants(t, cfg1["pos"])
    assert canonical_from_oracle(t) == brute_tree(cfg1["pos"])[0]
    # hard spheres (d = 1) never reach the depth cap: finest cell diagonal < 1
    assert t.nodes()["level"].max() < 10


def test_eight_corners_and_same_octant():
    corners = np.array([[x, y, z] for x in (0, 1) for y in (0, 1) for z in (0, 1)], np.float32)
    t = oracle.Tree(corners)
    nd = t.nodes()
    assert t.n_nodes == 9 and nd["is_leaf"].tolist() == [0] + [1] * 8
    assert nd["prefix"][1:].tolist() == list(range(8))                   # octant digit = 4x + 2y + z
    key, perm = t.keys()
    assert perm.tolist() == list(range(8))
    # q = 1023 for a coordinate on the far face, 0 on the near face: every digit equals the octant
    assert key.tolist() == [o * ((2**30 - 1) // 7) for o in range(8)]
    assert key[4] == int("100" * 10, 2)
    # two particles in the same deep octant -> single-child chain kept, one node per level
    pos = np.array([[0, 0, 0], [1, 1, 1], [0.99, 0.99, 0.99]], np.float32)
    t = oracle.Tree(pos)
    nd = t.nodes()
    chain = [i for i in range(t.n_nodes) if nd["count"][i] == 2]
    assert len(chain) >= 5 and nd["level"][chain].tolist() == list(range(1, len(chain) + 1))


def test_coincident_points_and_depth_cap():
    pos = np.zeros((5, 3), np.float32)                                   # S = 0 -> S := 1, all keys 0
    t = oracle.Tree(pos)
    lo, S = t.bbox()
    assert S == 1.0
    nd = t.nodes()
    assert t.n_nodes == 11 and nd["level"].tolist() == list(range(11))   # chain to the 10-level cap
    assert nd["is_leaf"].tolist() == [0] * 10 + [1] and nd["count"][-1] == 5
    key, perm = t.keys()
    assert perm.tolist() == [0, 1, 2, 3, 4]


def test_quantisation_is_fp32_in_the_stated_order():
    rng = np.random.default_rng(11)
    pos = (rng.random((2000, 3)) * 37.3).astype(np.float32)
    key, _, _ = morton_keys_numpy(pos)
    t = oracle.Tree(pos)
    okey, perm = t.keys()
    assert np.array_equal(okey, key[perm])


def test_moments_eq14(cfg1):
    pos, mom = cfg1["pos"], cfg1["mom"]
    t = oracle.Tree(pos)
    m = t.moments(mom)
    nd = t.nodes()
    _, perm = t.keys()
    sp, sm = pos[perm].astype(np.float64), mom[perm].astype(np.float64)
    # root: u' = sum u, rho' = mean rho, against a correctly rounded sum
    for a in range(3):
        assert abs(m["sum_u"][0, a] - math.fsum(sm[:, a])) <= 1e-12 * np.abs(sm[:, a]).sum()
        assert abs(m["sum_p"][0, a] - math.fsum(sp[:, a])) <= 1e-12 * np.abs(sp[:, a]).sum()
    assert np.array_equal(m["cen"][0], (m["sum_p"][0] / len(pos)).astype(np.float32))
    assert np.array_equal(m["mu"][0], m["sum_u"][0].astype(np.float32))
    # every node against the plain definition over its particle range
    rng = np.random.default_rng(0)
    for i in rng.choice(t.n_nodes, 300, replace=False):
        f, c = int(nd["first"][i]), int(nd["count"][i])
        assert np.allclose(m["sum_u"][i], sm[f:f + c].sum(0), rtol=0, atol=1e-12 * c)
        assert np.allclose(m["sum_p"][i] / c, sp[f:f + c].mean(0), rtol=1e-13)
        assert np.abs(m["cen"][i] - sp[f:f + c].mean(0)).max() <= np.spacing(np.float32(np.abs(m["cen"][i]).max()))
    # a single-particle node reproduces the particle exactly
    for i in np.nonzero(nd["count"] == 1)[0][:200]:
        f = int(nd["first"][i])
        assert np.array_equal(m["cen"][i], pos[perm[f]]) and np.array_equal(m["mu"][i], mom[perm[f]])


def test_moments_fixed_recursion_order():
    # internal sum = ((c0 + c1) + c2) + ... over children in octant order; leaf = left to right
    pos = ffgen.uniform_points(40, 3.0, 9)
    mom = ffgen.moments_isotropic(40, 9)
    for nleaf in (1, 3):
        t = oracle.Tree(pos, nleaf)
        m = t.moments(mom)
        nd = t.nodes()
        _, perm = t.keys()
        sp, sm = pos[perm].astype(np.float64), mom[perm].astype(np.float64)
        for i in range(t.n_nodes):
            f, c = int(nd["first"][i]), int(nd["count"][i])
            if nd["is_leaf"][i]:
                su, spp = sm[f].copy(), sp[f].copy()
                for s in range(f + 1, f + c):
                    su += sm[s]
                    spp += sp[s]
            else:
                ch = [int(x) for x in nd["child"][i] if x >= 0]
                su, spp = m["sum_u"][ch[0]].copy(), m["sum_p"][ch[0]].copy()
                for x in ch[1:]:
                    su += m["sum_u"][x]
                    spp += m["sum_p"][x]
            assert np.array_equal(su, m["sum_u"][i]) and np.array_equal(spp, m["sum_p"][i])
