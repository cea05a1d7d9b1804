"""Pins for the oracle's first-order cell term (oracle/ff_oracle.c O1b, O4b).

Not in the paper: Eq. 14 keeps the lowest-order term of a cell only, which leaves an error of first
order in (cell size / distance).  The correction is the next term of the Taylor expansion of Eq. 11-12 about the cell
centre rho' with the cell tensor D = sum_i (rho_i - rho') (x) u_i.  Pinned against: numerical derivatives of the
independently written pair terms (helpers.pair_terms), an independently derived contracted closed form
(helpers.first_order_terms), the order of the remaining error, numpy for D, and theta = 0."""
import numpy as np
import pytest

import ffgen
import oracle
from helpers import brute_tree, build_lists, eval_lists, first_order_terms, pair_terms


def test_first_order_term_is_the_derivative_of_the_pair_terms_in_the_source_position():
    """d/d(eps) of Eq. 11-12 for a source u at rc + eps * dhat, at eps = 0, by central differences, equals the
    first-order term with D = dhat (x) u -- component by component, for h and f.  A wrong sign, a dropped term or a
    transposed index in the rank-3 / rank-4 tensors fails this."""
    rng = np.random.default_rng(3)
    for trial in range(20):
        rk, rc = rng.normal(size=3) * 3, rng.normal(size=3) * 3
        if np.linalg.norm(rk - rc) < 1.0:
            rk = rk + 3.0
        uk, u, dhat = rng.normal(size=3), rng.normal(size=3), rng.normal(size=3)
        eps = 1e-4
        hp, fp = pair_terms(rk, uk, rc + eps * dhat, u)
        hm, fm = pair_terms(rk, uk, rc - eps * dhat, u)
        dh_num, df_num = (hp - hm) / (2 * eps), (fp - fm) / (2 * eps)
        dh, df = oracle.first_order(rk, uk, rc, np.outer(dhat, u))
        assert np.allclose(dh, dh_num, rtol=1e-6, atol=1e-7 * np.abs(dh_num).max())
        assert np.allclose(df, df_num, rtol=1e-6, atol=1e-7 * np.abs(df_num).max())


def test_matches_contracted_closed_form_and_ignores_the_antisymmetric_part():
    rng = np.random.default_rng(4)
    for trial in range(20):
        rk, rc, uk = rng.normal(size=3) * 4, rng.normal(size=3), rng.normal(size=3)
        D = rng.normal(size=(3, 3))
        dh, df = oracle.first_order(rk, uk, rc, D)
        dh2, df2 = first_order_terms(rk, uk, rc, D)
        assert np.allclose(dh, dh2, rtol=1e-12, atol=1e-14) and np.allclose(df, df2, rtol=1e-12, atol=1e-14)
        dh3, df3 = oracle.first_order(rk, uk, rc, 0.5 * (D + D.T))
        assert np.allclose(dh, dh3, rtol=1e-12, atol=1e-14) and np.allclose(df, df3, rtol=1e-12, atol=1e-14)
        # linear in D
        dh4, df4 = oracle.first_order(rk, uk, rc, 3.0 * D)
        assert np.allclose(3 * dh, dh4, rtol=1e-12) and np.allclose(3 * df, df4, rtol=1e-12)


def test_two_particle_cell_is_reproduced_to_second_order():
    """Exact sum of two dipoles against pseudo-particle (+ first-order term): halving the cell halves the error of the
    paper's cell and quarters the corrected one."""
    rk, uk = np.array([6.0, 2.0, -1.0]), np.array([0.3, -0.5, 0.8])
    u1, u2 = np.array([1.0, 0.2, 0.0]), np.array([-0.3, 0.9, 0.4])
    c, d = np.array([0.5, -0.2, 0.1]), np.array([0.35, -0.2, 0.3])
    e0, e1 = [], []
    for scale in (1.0, 0.5, 0.25):
        p1, p2 = c + scale * d, c - scale * d                 # centre (unweighted mean, Eq. 14) stays at c
        h_ex = sum(pair_terms(rk, uk, p, u)[0] for p, u in ((p1, u1), (p2, u2)))
        f_ex = sum(pair_terms(rk, uk, p, u)[1] for p, u in ((p1, u1), (p2, u2)))
        h0, f0 = pair_terms(rk, uk, c, u1 + u2)
        D = np.outer(p1 - c, u1) + np.outer(p2 - c, u2)
        dh, df = oracle.first_order(rk, uk, c, D)
        e0.append((np.linalg.norm(h0 - h_ex), np.linalg.norm(f0 - f_ex)))
        e1.append((np.linalg.norm(h0 + dh - h_ex), np.linalg.norm(f0 + df - f_ex)))
    for k in (0, 1):
        assert 1.8 < e0[0][k] / e0[1][k] < 2.2 and 1.8 < e0[1][k] / e0[2][k] < 2.2          # first-order error
        assert 3.6 < e1[0][k] / e1[1][k] < 4.4 and 3.6 < e1[1][k] / e1[2][k] < 4.4          # second-order error
        assert e1[0][k] < 0.2 * e0[0][k]


def test_cell_tensor_against_numpy_and_single_particles():
    c = ffgen.config(2, N=700, seed=4)
    pos, mom = c["pos"], c["mom"]
    t = oracle.Tree(pos)
    m = t.moments(mom)
    nd = t.nodes()
    _, perm = t.keys()
    sp, su = pos[perm].astype(np.float64), mom[perm].astype(np.float64)
    for i in range(t.n_nodes):
        f, cnt = int(nd["first"][i]), int(nd["count"][i])
        d = sp[f:f + cnt] - sp[f:f + cnt].mean(0)
        D = d.T @ su[f:f + cnt]
        Ds = 0.5 * (D + D.T)
        ref = np.array([Ds[0, 0], Ds[1, 1], Ds[2, 2], Ds[0, 1], Ds[0, 2], Ds[1, 2]])
        tol = 4e-7 * max(1.0, np.abs(ref).max()) + 1e-9 * cnt * np.abs(sp[f:f + cnt]).max()
        assert np.abs(m["dsym"][i] - ref).max() <= tol, (i, cnt, m["dsym"][i], ref)
        if cnt == 1:
            assert np.all(m["dsym"][i] == 0)
    assert np.abs(m["dsym"]).max() > 1.0                       # the test sees non-trivial tensors


def test_theta_zero_is_unchanged_and_counters_do_not_depend_on_the_order(cfg1):
    pos, mom = cfg1["pos"][:1200], cfg1["mom"][:1200]
    H0, F0, c0, _ = oracle.barnes_hut(pos, mom, 0.0, 32)
    H1, F1, c1, _ = oracle.barnes_hut(pos, mom, 0.0, 32, order=1)
    assert np.array_equal(H0, H1) and np.array_equal(F0, F1) and c0 == c1
    # the order changes what an accepted cell contributes, not which cells are accepted
    _, _, a0, _ = oracle.barnes_hut(pos, mom, 0.6, 32)
    Hb, _, a1, _ = oracle.barnes_hut(pos, mom, 0.6, 32, order=1)
    assert a0 == a1 and a0[0] > 0 and not np.array_equal(Hb, H0)


@pytest.mark.parametrize("N,W,nleaf,theta,seed", [(64, 32, 1, 0.5, 0), (64, 1, 1, 0.7, 1), (60, 8, 2, 0.6, 2)])
def test_against_independent_list_builder_with_contracted_terms(N, W, nleaf, theta, seed):
    """Brute force on N <= 64: the independently written list builder, cell tensors from numpy on the builder's own
    cells, contracted closed form for the terms."""
    pos = ffgen.uniform_points(N, 4.0, seed)
    mom = ffgen.moments_vmf(N, 2.0, seed)
    lists, info, sp, sm, perm = build_lists(pos, mom, theta, W, nleaf)
    H_ref, F_ref = eval_lists(lists, info, sp, sm, perm)
    n_cells = 0
    for g0, g1, cells, parts in lists:
        for (l, p) in cells:
            f, c, leaf, cen, mu = info[(l, p)]
            mean = sp[f:f + c].astype(np.float64).sum(0) / c
            D = (sp[f:f + c].astype(np.float64) - mean).T @ sm[f:f + c].astype(np.float64)
            for k in range(g0, g1):
                dh, df = first_order_terms(sp[k], sm[k], cen, D)
                H_ref[perm[k]] += dh
                F_ref[perm[k]] += df
            n_cells += 1
    assert n_cells > 0
    H, F, cnt, t = oracle.barnes_hut(pos, mom, theta, W, nleaf, order=1)
    # D is rounded to fp32 in the tree (relative 6e-8 of a term that is itself a fraction of the total)
    assert np.allclose(H, H_ref, rtol=1e-6, atol=1e-8) and np.allclose(F, F_ref, rtol=1e-6, atol=1e-8)


def test_far_cluster_error_becomes_second_order():
    """The far-cluster pin of the walk, with the correction: for every near target the walk accepts the far cluster
    as ONE cell; replacing the cluster by that cell's pseudo-particle leaves an error that falls as s/d, adding the
    first-order term with the TREE's tensor D one that falls as (s/d)^2 (distances 20, 80, 320: factors of ~4 / ~16)."""
    rng = np.random.default_rng(5)
    near = rng.random((16, 3)).astype(np.float32)
    mom = ffgen.moments_vmf(32, 3.0, 2)
    shape = rng.random((16, 3))                                # the same far cluster, moved away
    e0, e1 = [], []
    for dist in (20.0, 80.0, 320.0):
        far = (shape + [dist, dist, dist]).astype(np.float32)
        pos = np.vstack([near, far])
        t = oracle.Tree(pos)
        m = t.moments(mom)
        nd = t.nodes()
        _, perm = t.keys()
        far_slots = set(np.nonzero(perm >= 16)[0].tolist())
        d0 = d1 = ref = 0.0
        for slot in np.nonzero(perm < 16)[0]:
            k = int(perm[slot])
            cells, parts = t.group_lists(0.5, 1, int(slot))
            big = [i for i in cells if set(range(nd["first"][i], nd["first"][i] + nd["count"][i])) == far_slots]
            assert len(big) == 1
            ds = m["dsym"][big[0]].astype(np.float64)
            D = np.array([[ds[0], ds[3], ds[4]], [ds[3], ds[1], ds[5]], [ds[4], ds[5], ds[2]]])
            cen, mu = m["cen"][big[0]].astype(np.float64), m["mu"][big[0]].astype(np.float64)
            h0, f0 = pair_terms(pos[k].astype(np.float64), mom[k].astype(np.float64), cen, mu)
            dh, df = oracle.first_order(pos[k].astype(np.float64), mom[k].astype(np.float64), cen, D)
            # what the far cluster really does to this target: the plain sum over its particles
            hx, fx = pair_terms(pos[k].astype(np.float64), mom[k].astype(np.float64), far.astype(np.float64),
                                mom[16:].astype(np.float64))
            ex = np.concatenate([hx.sum(0), fx.sum(0) * dist])
            d0 += np.sum((np.concatenate([h0, f0 * dist]) - ex) ** 2)
            d1 += np.sum((np.concatenate([h0 + dh, (f0 + df) * dist]) - ex) ** 2)
            ref += np.sum(ex ** 2)
        e0.append(np.sqrt(d0 / ref))
        e1.append(np.sqrt(d1 / ref))
    assert 3.0 < e0[0] / e0[1] < 5.5 and 3.0 < e0[1] / e0[2] < 5.5
    assert 11.0 < e1[0] / e1[1] < 22.0 and 11.0 < e1[1] / e1[2] < 22.0
    assert e1[0] < 0.1 * e0[0]
