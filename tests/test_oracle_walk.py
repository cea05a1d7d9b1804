"""Pins for the oracle's Barnes-Hut evaluation (O5): PAPER.md:153 traversal with the
opening rule of DESIGN.md (s/d < theta, group rule, fp32 test in a fixed operation order)."""
import math

import numpy as np
import pytest

import ffgen
import oracle
from helpers import build_lists as _build_lists, eval_lists as _eval_lists, pair_terms, rel_err


@pytest.mark.parametrize("N,W,nleaf,theta,seed", [
    (64, 32, 1, 0.5, 0), (64, 1, 1, 0.5, 1), (50, 8, 1, 0.7, 2), (64, 32, 4, 0.6, 3), (37, 32, 1, 1.0, 4), (60, 4, 2, 0.3, 5),
])
def test_against_independent_list_builder(N, W, nleaf, theta, seed):
    pos = ffgen.uniform_points(N, 4.0, seed)
    mom = ffgen.moments_isotropic(N, seed)
    lists, info, sp, sm, perm = _build_lists(pos, mom, theta, W, nleaf)
    H_ref, F_ref = _eval_lists(lists, info, sp, sm, perm)
    H, F, cnt, t = oracle.barnes_hut(pos, mom, theta, W, nleaf)
    assert np.allclose(H, H_ref, rtol=1e-11, atol=1e-13)
    assert np.allclose(F, F_ref, rtol=1e-11, atol=1e-13)
    nd = t.nodes()
    n_cell = n_part = 0
    for g, (g0, g1, cells, parts) in enumerate(lists):
        oc, op = t.group_lists(theta, W, g)
        assert sorted((int(nd["level"][i]), int(nd["prefix"][i])) for i in oc) == sorted(cells)
        assert sorted(op.tolist()) == sorted(parts)
        n_cell += len(cells) * (g1 - g0)
        n_part += sum(1 for k in range(g0, g1) for j in parts if j != k)
    assert cnt[0] == n_cell and cnt[1] == n_part
    assert theta < 0.9 or any(len(c) for _, _, c, _ in lists)   # the test exercises accepted cells


def test_theta_zero_is_all_pairs(cfg1):
    pos, mom = cfg1["pos"][:1500], cfg1["mom"][:1500]
    H, F = oracle.allpairs(pos, mom)
    for W in (1, 32):
        Hb, Fb, cnt, _ = oracle.barnes_hut(pos, mom, 0.0, W)
        assert cnt[0] == 0 and cnt[1] == 1500 * 1499
        assert np.allclose(Hb, H, rtol=1e-11, atol=1e-13) and np.allclose(Fb, F, rtol=1e-11, atol=1e-13)


def test_single_leaf_is_all_pairs():
    pos = ffgen.uniform_points(20, 3.0, 1)
    mom = ffgen.moments_isotropic(20, 1)
    H, F = oracle.allpairs(pos, mom)
    Hb, Fb, cnt, t = oracle.barnes_hut(pos, mom, 0.5, 32, nleaf=32)     # N <= N_leaf: the root is a leaf
    assert t.n_nodes == 1 and cnt == (0, 20 * 19, 0)
    assert np.allclose(Hb, H, rtol=1e-12, atol=1e-14) and np.allclose(Fb, F, rtol=1e-12, atol=1e-14)


def test_self_cell_is_never_accepted():
    # theta > 1/sqrt(3): a cell holding the target could pass s/d < theta (Q3); it must be opened instead
    pos, mom = ffgen.uniform_points(64, 4.0, 6), ffgen.moments_isotropic(64, 6)
    for W in (1, 32):
        t = oracle.Tree(pos)
        t.moments(mom)
        nd = t.nodes()
        for g in range((64 + W - 1) // W):
            cells, parts = t.group_lists(2.0, W, g)
            g0, g1 = g * W, min(64, g * W + W)
            for i in cells:
                assert nd["first"][i] >= g1 or nd["first"][i] + nd["count"][i] <= g0
            assert set(range(g0, g1)) <= set(parts.tolist())


def test_far_cluster_becomes_one_dipole():
    # two clusters far apart: the far cluster acts as ONE pseudo-particle (sum u at mean rho, Eq. 14),
    # and the error of that replacement shrinks as s/d shrinks
    rng = np.random.default_rng(5)
    near = rng.random((16, 3)).astype(np.float32)
    mom = ffgen.moments_vmf(32, 3.0, 2)
    errs = []
    for dist in (20.0, 80.0, 320.0):
        far = (rng.random((16, 3)) + [dist, dist, dist]).astype(np.float32)
        pos = np.vstack([near, far])
        t = oracle.Tree(pos)
        m = t.moments(mom)
        nd = t.nodes()
        _, perm = t.keys()
        far_slots = set(np.nonzero(perm >= 16)[0].tolist())
        cen = pos[16:].astype(np.float64).mean(0)
        mu = mom[16:].astype(np.float64).sum(0)
        for slot in np.nonzero(perm < 16)[0]:
            cells, parts = t.group_lists(0.5, 1, int(slot))
            big = [i for i in cells if set(range(nd["first"][i], nd["first"][i] + nd["count"][i])) == far_slots]
            assert len(big) == 1 and not (far_slots & set(parts.tolist()))
            assert np.allclose(m["cen"][big[0]], cen, rtol=1e-6) and np.allclose(m["mu"][big[0]], mu, rtol=1e-6, atol=1e-7)
        Hap, _ = oracle.allpairs(pos, mom)
        Hnn, _ = oracle.allpairs(near, mom[:16])
        far_exact = Hap[:16] - Hnn                      # what the far cluster really does to the near one
        one, _ = pair_terms(pos[:16].astype(np.float64), mom[:16].astype(np.float64), cen, mu)
        errs.append(np.linalg.norm(one - far_exact) / np.linalg.norm(far_exact))
    assert errs[0] > errs[1] > errs[2] and errs[2] < errs[0] / 8 and errs[0] < 0.1


def test_bulk_interaction_count_per_level():
    # per octree level a target in the bulk accepts about (28 pi / 3) theta^-3 cells: the cells of side s
    # in the shell s/theta < d < 2s/theta (continuum estimate; averaged over targets to wash out the lattice)
    N = 262144
    pos = ffgen.uniform_points(N, 1.0, 3)
    mom = ffgen.moments_isotropic(N, 3)
    t = oracle.Tree(pos)
    t.moments(mom)
    nd = t.nodes()
    key, perm = t.keys()
    near_centre = np.nonzero(np.abs(pos[perm] - 0.5).max(1) < 0.08)[0][::20][:40]
    for theta in (0.4, 0.5):
        lv = np.zeros(11)
        for slot in near_centre:
            cells, _ = t.group_lists(theta, 1, int(slot))
            lv += np.bincount(nd["level"][cells], minlength=11)
        lv /= len(near_centre)
        expect = 28 * math.pi / 3 / theta**3
        for level in (4, 5):        # shells inside the unit cube, cells still hold several particles
            assert 0.85 * expect < lv[level] < 1.15 * expect, (theta, level, lv, expect)


def test_error_shrinks_with_theta_and_group_rule_is_tighter(cfg1):
    pos, mom = cfg1["pos"], cfg1["mom"]
    H, F = oracle.allpairs(pos, mom)
    prev = None
    for theta in (0.7, 0.5, 0.3):
        H1, F1, c1, _ = oracle.barnes_hut(pos, mom, theta, 1)
        H32, F32, c32, _ = oracle.barnes_hut(pos, mom, theta, 32)
        e1, e32 = rel_err(H1, H)[3], rel_err(H32, H)[3]
        assert e32 < e1 < 0.2                                   # every-member rule opens more cells
        assert c32[0] + c32[1] > c1[0] + c1[1]
        assert prev is None or e1 < prev
        prev = e1


# ---- the opening test itself, on its threshold (reading O5 / Q1 of PAPER.md:153: "strict; equality opens", and the
# fp32 operation order d2 = fma(dz,dz, fma(dy,dy, fl(dx dx))), fl(s^2) < fl(fl(theta^2) d2)) -------------------------
from helpers import fma_sensitive_targets, opening_case, opening_d2


def _pair_cell_decision(t):
    """Does the oracle's group 0 accept the level-2 cell of the pair (helpers.opening_case)?  Also checks that the
    whole interaction list equals the independently written list builder's."""
    pos, mom, ia, ib = opening_case(t)
    tree = oracle.Tree(pos)
    tree.moments(mom)
    _, perm = tree.keys()
    slot = {int(c): s for s, c in enumerate(perm)}
    sa, sb = sorted((slot[ia], slot[ib]))
    assert (sa, sb) == (32, 33)                              # group 0 = the 32 particles of octant 0
    nd = tree.nodes()
    om = tree.moments(mom)
    cell = [i for i in range(tree.n_nodes) if nd["level"][i] == 2 and nd["first"][i] == 32 and nd["count"][i] == 2]
    assert len(cell) == 1 and not nd["is_leaf"][cell[0]]
    assert np.array_equal(om["cen"][cell[0]], np.array([5, 1, 1], np.float32))     # the centre is exact
    cells, parts = tree.group_lists(0.5, 32, 0)
    accepted = cell[0] in set(int(c) for c in cells)
    assert accepted != ({32, 33} <= set(int(p) for p in parts))                    # either the cell or its two particles
    lists, *_ = _build_lists(pos, mom, 0.5, 32, 1)
    g0, g1, bcells, bparts = lists[0]
    assert sorted((int(nd["level"][c]), int(nd["prefix"][c])) for c in cells) == sorted(bcells)
    assert sorted(int(p) for p in parts) == sorted(bparts)
    # the counters of the evaluation agree with the lists (32 members per accepted cell, self term excluded)
    _, _, cnt = tree.eval(0.5, 32, groups=[0])
    assert cnt[0] == 32 * len(cells) and cnt[1] == 32 * len(parts) - 32
    return accepted


def test_opening_test_equality_opens():
    """t = (1, 1, 1): d = 4 = 2 s_2 exactly, fl(s^2) = 4 = fl(theta^2 d2).  The test is STRICT: equality opens."""
    assert float(opening_d2([1, 1, 1])) == 16.0
    assert _pair_cell_decision([1.0, 1.0, 1.0]) is False


def test_opening_test_one_ulp_beyond_accepts():
    """The neighbouring target whose dx is one fp32 step longer (4 + 2^-21): d2 = 16 + 2^-18, rhs = 4 + 2^-20 > 4."""
    t = [1.0 - 2.0 ** -21, 1.0, 1.0]
    assert float(opening_d2(t)) == 16.0 + 2.0 ** -18
    assert _pair_cell_decision(t) is True
    # and one step short of the threshold (dx = 4 - 2^-22, d2 < 16) opens
    t = [1.0 + 2.0 ** -22, 1.0, 1.0]
    assert float(opening_d2(t)) < 16.0
    assert _pair_cell_decision(t) is False


def test_opening_test_uses_the_fused_order():
    """Two targets (seeded search, helpers.fma_sensitive_targets) on which d2 in the order of reading O5 and d2 as
    three rounded squares added left to right fall on different sides of the threshold: the oracle must decide as the
    fused order does, in both directions."""
    found = fma_sensitive_targets()
    for fused_accepts, t in found.items():
        assert bool(opening_d2(t, True) > 16.0) == fused_accepts
        assert bool(opening_d2(t, False) > 16.0) != fused_accepts
        assert _pair_cell_decision(t) is fused_accepts
