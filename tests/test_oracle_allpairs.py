"""Pins for oracle.allpairs (O2): Eq. 10 without h_ext and Eq. 12 summed over j != k."""
from fractions import Fraction

import numpy as np
import pytest

import ffgen
import oracle
from golden_io import golden
from helpers import allpairs_numpy


@pytest.fixture(scope="module")
def small():
    c = ffgen.config(1, N=300)
    return c["pos"], c["mom"]


def test_matches_independent_numpy(small):
    pos, mom = small
    H, F = oracle.allpairs(pos, mom)
    H2, F2 = allpairs_numpy(pos, mom)
    assert np.allclose(H, H2, rtol=1e-11, atol=1e-13)
    assert np.allclose(F, F2, rtol=1e-11, atol=1e-13)


def test_targets_subset_and_threads(small):
    pos, mom = small
    H, F = oracle.allpairs(pos, mom)
    idx = np.array([5, 0, 299, 17])
    Hs, Fs = oracle.allpairs(pos, mom, targets=idx, nthreads=1)
    assert np.array_equal(Hs, H[idx]) and np.array_equal(Fs, F[idx])


def test_newton_third_law_and_torque_balance(cfg1):
    pos, mom = cfg1["pos"], cfg1["mom"]
    H, F = oracle.allpairs(pos, mom)
    fs = np.abs(F).sum(0)
    assert np.abs(F.sum(0)).max() < 1e-12 * fs.max()           # sum_k f_k = 0
    p, u = pos.astype(np.float64), mom.astype(np.float64)
    tau = np.cross(p, F) + np.cross(u, H)                      # orbital + spin torque
    assert np.abs(tau.sum(0)).max() < 1e-11 * np.abs(tau).sum(0).max()


def test_rotation_translation_covariance(small):
    pos, mom = small
    rng = np.random.default_rng(7)
    Q, _ = np.linalg.qr(rng.normal(size=(3, 3)))
    if np.linalg.det(Q) < 0:
        Q[:, 0] = -Q[:, 0]
    t = np.array([3.0, -2.0, 5.0])
    # fp32 inputs cannot be rotated exactly: rotate in fp64 and evaluate the rotated copy with the
    # independent fp64 formula; the oracle's result must map onto it
    H, F = oracle.allpairs(pos, mom)
    p2 = pos.astype(np.float64) @ Q.T + t
    u2 = mom.astype(np.float64) @ Q.T
    H2, F2 = allpairs_numpy(p2, u2)
    assert np.allclose(H @ Q.T, H2, rtol=1e-9, atol=1e-11)
    assert np.allclose(F @ Q.T, F2, rtol=1e-9, atol=1e-11)
    U1 = -0.5 * (mom.astype(np.float64) * H).sum()
    U2 = -0.5 * (u2 * H2).sum()
    assert abs(U1 - U2) < 1e-10 * abs(U1)


def test_straight_chain_closed_form():
    n = 32
    pos = np.zeros((n, 3), np.float32)
    pos[:, 2] = np.arange(n)
    mom = np.zeros((n, 3), np.float32)
    mom[:, 2] = 1
    H, F = oracle.allpairs(pos, mom)
    h_exact = [float(sum(Fraction(2, abs(i - j) ** 3) for j in range(n) if j != i)) for i in range(n)]
    f_exact = [float(sum(Fraction(-6 if i > j else 6, abs(i - j) ** 4) for j in range(n) if j != i)) for i in range(n)]
    assert np.allclose(H[:, 2], h_exact, rtol=1e-13) and np.abs(H[:, :2]).max() == 0
    assert np.allclose(F[:, 2], f_exact, rtol=1e-12, atol=1e-13) and np.abs(F[:, :2]).max() == 0
    assert H[0, 2] == pytest.approx(golden("chain32_h_end"), abs=1e-6)
    assert H[15, 2] == pytest.approx(golden("chain32_h_mid"), abs=1e-6)
    assert H[16, 2] == pytest.approx(golden("chain32_h_mid"), abs=1e-6)
    assert F[0, 2] == pytest.approx(golden("chain32_f_end"), abs=1e-6)      # attracted towards the chain
    assert F[31, 2] == pytest.approx(-golden("chain32_f_end"), abs=1e-6)
    zeta3 = sum(1.0 / k**3 for k in range(1, 200000))
    assert 4 * zeta3 == pytest.approx(golden("chain_inf_h"), abs=1e-6)
    assert H[15, 2] < 4 * zeta3
