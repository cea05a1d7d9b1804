"""Pins for the oracle's Q output (scale=True): Q_k = sqrt(sum_j |t_kj|^2), the root-sum-square of the terms of
particle k's own sum (Eq. 11 terms for H, Eq. 12 terms for F).  Q_k / kappa is the floor of the
denominator of the GPU parity metric, so a Q that is too large by any factor would silently
loosen every tolerance: these tests fail if Q is off by a factor (1 + 1e-10)."""
from fractions import Fraction
import math

import numpy as np
import pytest

import ffgen
import oracle
from golden_io import golden
from helpers import build_lists, eval_lists, pair_terms


def _q_numpy(pos, mom):
    """Independent numpy statement: per target the squared norms of the pair terms, summed over j != k."""
    p, u = np.asarray(pos, np.float64), np.asarray(mom, np.float64)
    N = len(p)
    Q = np.zeros((N, 2))
    for k in range(N):
        m = np.arange(N) != k
        h, f = pair_terms(p[k], u[k], p[m], u[m])
        Q[k] = np.sqrt((h * h).sum()), np.sqrt((f * f).sum())
    return Q


def test_allpairs_scale_matches_independent_numpy():
    c = ffgen.config(1, N=300)
    pos, mom = c["pos"], c["mom"]
    H, F, Q = oracle.allpairs(pos, mom, scale=True)
    Qn = _q_numpy(pos, mom)
    assert Q.shape == (300, 2) and np.allclose(Q, Qn, rtol=1e-11, atol=0)
    # a factor-2 (or any other) mistake in Q fails the line above; make that explicit
    assert not np.allclose(2 * Q, Qn, rtol=0.5) and not np.allclose(Q * Q, Qn, rtol=1e-3)
    # asking for the scale does not change the sums, and a target subset returns the matching rows
    H0, F0 = oracle.allpairs(pos, mom)
    assert np.array_equal(H, H0) and np.array_equal(F, F0)
    idx = np.array([7, 0, 299])
    _, _, Qs = oracle.allpairs(pos, mom, targets=idx, scale=True, nthreads=1)
    assert np.array_equal(Qs, Q[idx])
    # Q bounds the sum: |sum_j t_kj| <= sqrt(N-1) Q_k (Cauchy-Schwarz) and Q_k <= sum_j |t_kj|
    assert (np.linalg.norm(H, axis=1) <= math.sqrt(299) * Q[:, 0]).all()
    assert (np.linalg.norm(F, axis=1) <= math.sqrt(299) * Q[:, 1]).all()


@pytest.mark.parametrize("N,W,nleaf,theta,seed", [(64, 32, 1, 0.5, 0), (64, 1, 1, 0.5, 1), (50, 8, 1, 0.7, 2),
                                                  (64, 32, 4, 0.6, 3), (37, 32, 1, 1.0, 4)])
def test_barnes_hut_scale_matches_independent_list_builder(N, W, nleaf, theta, seed):
    """Barnes-Hut: the terms are those of the group's interaction list (accepted cells with (u', rho') + particles
    reached through leaves); the list and the terms come from the independently written python builder."""
    pos = ffgen.uniform_points(N, 4.0, seed)
    mom = ffgen.moments_isotropic(N, seed)
    lists, info, sp, sm, perm = build_lists(pos, mom, theta, W, nleaf)
    H_ref, F_ref, Q_ref = eval_lists(lists, info, sp, sm, perm, scale=True)
    H, F, cnt, t, Q = oracle.barnes_hut(pos, mom, theta, W, nleaf, scale=True)
    assert np.allclose(Q, Q_ref, rtol=1e-11, atol=0)
    assert np.allclose(H, H_ref, rtol=1e-11, atol=1e-13) and np.allclose(F, F_ref, rtol=1e-11, atol=1e-13)
    H0, F0, _, _ = oracle.barnes_hut(pos, mom, theta, W, nleaf)
    assert np.array_equal(H, H0) and np.array_equal(F, F0)
    # sampled groups: rows outside the sample stay NaN, rows inside equal the full evaluation
    if W < N:
        _, _, _, Qg = t.eval(theta, W, groups=np.array([1]), scale=True)
        _, operm = t.keys()
        rows = operm[W:min(N, 2 * W)]
        other = np.setdiff1d(np.arange(N), rows)
        assert np.array_equal(Qg[rows], Q[rows]) and np.isnan(Qg[other]).all()


def test_theta_zero_scale_equals_allpairs_scale():
    c = ffgen.config(1, N=500, seed=2)
    _, _, Qa = oracle.allpairs(c["pos"], c["mom"], scale=True)
    _, _, _, _, Qb = oracle.barnes_hut(c["pos"], c["mom"], 0.0, 32, scale=True)
    assert np.allclose(Qa, Qb, rtol=1e-12, atol=0)        # same terms, different order of the sum of squares


def test_straight_chain_scale_closed_form():
    """Straight chain of 32 touching dipoles, all u = z: every term is along z, h_kj = 2/|i-j|^3 and
    f_kj = -+6/|i-j|^4 (Eq. 11-12 on the axis), so Q_h(i)^2 = sum 4/|i-j|^6 and Q_f(i)^2 = sum 36/|i-j|^8, exactly."""
    n = 32
    pos = np.zeros((n, 3), np.float32)
    pos[:, 2] = np.arange(n)
    mom = np.zeros((n, 3), np.float32)
    mom[:, 2] = 1
    _, _, Q = oracle.allpairs(pos, mom, scale=True)
    qh = [math.sqrt(sum(Fraction(4, abs(i - j) ** 6) for j in range(n) if j != i)) for i in range(n)]
    qf = [math.sqrt(sum(Fraction(36, abs(i - j) ** 8) for j in range(n) if j != i)) for i in range(n)]
    assert np.allclose(Q[:, 0], qh, rtol=1e-13) and np.allclose(Q[:, 1], qf, rtol=1e-13)
    assert Q[0, 0] == pytest.approx(golden("chain32_qh_end"), abs=1e-6)
    assert Q[15, 0] == pytest.approx(golden("chain32_qh_mid"), abs=1e-6)
    assert Q[16, 0] == pytest.approx(golden("chain32_qh_mid"), abs=1e-6)
    assert Q[31, 1] == pytest.approx(golden("chain32_qf_end"), abs=1e-6)
    assert Q[15, 1] == pytest.approx(golden("chain32_qf_mid"), abs=1e-6)
    # the cancellation the floor exists for: in the chain interior the two neighbour forces cancel, |f| << Q_f
    _, F = oracle.allpairs(pos, mom)
    assert abs(F[15, 2]) < 1e-2 * Q[15, 1] and abs(F[0, 2]) > Q[0, 1]
