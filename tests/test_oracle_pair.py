"""Pins for oracle.pair (O1): Eq. 11 and Eq. 12."""
from fractions import Fraction

import numpy as np
import pytest

import oracle
from golden_io import golden
from helpers import pair_terms

X, Y, Z, O = np.eye(3)[0], np.eye(3)[1], np.eye(3)[2], np.zeros(3)


def test_single_dipole_closed_forms():
    # dipole m at the origin: on-axis h = 2m/r^3 (parallel to m); equatorial h = -m/r^3
    for r in (1.0, 2.0, 3.7):
        h, _ = oracle.pair(r * Z, X, O, Z)
        assert np.allclose(h, 2 * Z / r**3, rtol=1e-14, atol=0)
        h, _ = oracle.pair(r * X, X, O, Z)
        assert np.allclose(h, -Z / r**3, rtol=1e-14, atol=1e-17)
        h, _ = oracle.pair(-r * Y, X, O, Z)
        assert np.allclose(h, -Z / r**3, rtol=1e-14, atol=1e-17)
    assert oracle.pair(2 * Z, X, O, Z)[0][2] == pytest.approx(golden("dipole_axial_hz"), abs=1e-12)
    assert oracle.pair(2 * X, X, O, Z)[0][2] == pytest.approx(golden("dipole_equatorial_hz"), abs=1e-12)


def test_two_dipole_force_closed_forms():
    d = 2.0
    _, f = oracle.pair(d * Z, Z, O, Z)                       # head to tail: attractive
    assert np.allclose(f, [0, 0, float(Fraction(-6) / Fraction(d) ** 4)], atol=1e-15)
    assert f[2] == pytest.approx(golden("pair_head_to_tail_fz"), abs=1e-12)
    _, f = oracle.pair(d * X, Z, O, Z)                       # side by side parallel: repulsive
    assert np.allclose(f, [3 / d**4, 0, 0], atol=1e-15)
    assert f[0] == pytest.approx(golden("pair_side_parallel_fx"), abs=1e-12)
    _, f = oracle.pair(d * X, Z, O, -Z)                      # side by side antiparallel: attractive
    assert np.allclose(f, [-3 / d**4, 0, 0], atol=1e-15)
    assert f[0] == pytest.approx(golden("pair_side_antiparallel_fx"), abs=1e-12)
    _, f = oracle.pair(d * X, Z, O, X)                       # crossed
    assert np.allclose(f, [0, 0, 3 / d**4], atol=1e-15)
    assert f[2] == pytest.approx(golden("pair_crossed_fz"), abs=1e-12)


def test_matches_independent_numpy_formula():
    rng = np.random.default_rng(1)
    for _ in range(50):
        rk, rj = rng.normal(size=3) * 3, rng.normal(size=3) * 3
        uk, uj = rng.normal(size=3), rng.normal(size=3)      # need not be unit: both forms are bilinear
        h, f = oracle.pair(rk, uk, rj, uj)
        h2, f2 = pair_terms(rk, uk, rj, uj)
        assert np.allclose(h, h2, rtol=1e-13, atol=1e-15)
        assert np.allclose(f, f2, rtol=1e-13, atol=1e-15)


def test_force_is_gradient_of_u_dot_h():
    # f_k = grad_{rho_k} (u_k . h_kj): ties Eq. 12 to Eq. 11 (Eq. 3: mu0 (m_k . grad_k) H_k with curl H = 0)
    rng = np.random.default_rng(2)
    for _ in range(20):
        rk, rj = rng.normal(size=3) * 2 + 4, rng.normal(size=3)
        uk, uj = rng.normal(size=3), rng.normal(size=3)
        _, f = oracle.pair(rk, uk, rj, uj)
        g = np.zeros(3)
        eps = 1e-5
        for a in range(3):
            e = np.zeros(3)
            e[a] = eps
            hp, _ = oracle.pair(rk + e, uk, rj, uj)
            hm, _ = oracle.pair(rk - e, uk, rj, uj)
            g[a] = (uk @ hp - uk @ hm) / (2 * eps)
        assert np.allclose(f, g, rtol=1e-7, atol=1e-10)


def test_pair_force_antisymmetric_and_field_divergence_free():
    rng = np.random.default_rng(3)
    rk, rj = rng.normal(size=3) + 3, rng.normal(size=3)
    uk, uj = rng.normal(size=3), rng.normal(size=3)
    _, fkj = oracle.pair(rk, uk, rj, uj)
    _, fjk = oracle.pair(rj, uj, rk, uk)
    assert np.allclose(fkj, -fjk, rtol=1e-13)
    # div h = 0 and curl h = 0 away from the source (central differences)
    eps = 1e-4
    J = np.zeros((3, 3))
    for a in range(3):
        e = np.zeros(3)
        e[a] = eps
        J[:, a] = (oracle.pair(rk + e, uk, rj, uj)[0] - oracle.pair(rk - e, uk, rj, uj)[0]) / (2 * eps)
    scale = np.abs(J).max()
    assert abs(np.trace(J)) < 1e-6 * scale
    assert np.abs(J - J.T).max() < 1e-6 * scale
