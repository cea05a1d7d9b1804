"""Pins for the input generators (ffgen): Eq. 16 box side, hard-core separation, Eq. 17 mean."""
import math

import numpy as np
import pytest

import ffgen
from golden_io import golden


def _min_pair_distance(pos):
    from scipy.spatial import cKDTree
    d, _ = cKDTree(pos.astype(np.float64)).query(pos.astype(np.float64), k=2)
    return d[:, 1].min()


def test_box_side_eq16():
    # phi = N (4/3 pi R^3) / V_f (Eq. 16) with R = 1/2
    for N, phi, L in [(4096, 0.05, 35.005), (65536, 0.1, 70.010), (1048576, 0.1, 176.414), (16777216, 0.2, 352.828)]:
        assert abs(ffgen.box_side(N, phi) - L) < 1e-3
        assert abs(N * (4.0 / 3.0) * math.pi * 0.5**3 / ffgen.box_side(N, phi) ** 3 - phi) < 1e-12


def test_config1_shape_and_separation(cfg1):
    pos, mom = cfg1["pos"], cfg1["mom"]
    assert pos.shape == (4096, 3) and pos.dtype == np.float32
    assert mom.shape == (4096, 3) and mom.dtype == np.float32
    assert pos.min() >= 0 and pos.max() < cfg1["L"]
    assert _min_pair_distance(pos) >= 1.0
    assert np.allclose(np.linalg.norm(mom, axis=1), 1.0, atol=1e-6)
    # isotropic: mean of each component ~ 0 within 5 sigma (sigma = 1/sqrt(3N))
    assert np.abs(mom.mean(0)).max() < 5 / math.sqrt(3 * 4096)


def test_deterministic_and_seeded():
    a = ffgen.config(1, N=512)
    b = ffgen.config(1, N=512)
    c = ffgen.config(1, N=512, seed=1)
    assert np.array_equal(a["pos"], b["pos"]) and np.array_equal(a["mom"], b["mom"])
    assert not np.array_equal(a["pos"], c["pos"])


def test_vmf_mean_is_langevin():
    c = ffgen.config(2)
    L5 = 1 / math.tanh(5.0) - 1 / 5.0
    assert abs(L5 - golden("langevin_5")) < 1e-6
    # sigma of u_z for kappa=5 is < 0.2; N = 65536 -> 5 sigma < 0.004
    assert abs(c["mom"][:, 2].mean() - L5) < 4e-3
    assert _min_pair_distance(c["pos"]) >= 1.0


def test_chains_geometry():
    c = ffgen.config(4, N=32 * 256)
    pos, mom = c["pos"].astype(np.float64), c["mom"].astype(np.float64)
    assert pos.shape == (8192, 3)
    P = pos.reshape(256, 32, 3)
    step = np.diff(P, axis=1)
    assert np.allclose(np.linalg.norm(step, axis=2), 1.0, atol=1e-4)          # touching spheres
    ax = mom.reshape(256, 32, 3)[:, 0]
    assert np.allclose(step, ax[:, None, :], atol=1e-4)                         # moments along the axis
    assert (ax[:, 2] >= math.cos(math.radians(15.0)) - 1e-6).all()              # 15 degree cap about z
    assert _min_pair_distance(c["pos"]) >= 1.0 - 1e-4
