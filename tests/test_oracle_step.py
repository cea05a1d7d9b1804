"""Pins of oracle/md_step.py: Eq. 13 and the Euler-Maruyama step against closed forms.

None of these re-types the oracle's formula: the Lennard-Jones force is checked against the gradient of
its potential, its zero, its symmetries and the cut-off; the integrator against analytic solutions of the
equations of motion it discretises (error O(dtau)).
"""
import numpy as np

from oracle.md_step import lj_force, md_step, wall_force


# ------------------------------------------------------------------ Eq. 13 ----
def _potential(pos, eps, sigma):
    # U = sum_{k<j} 2 eps (s/r)^12 - 4 eps (s/r)^6 : the potential whose gradient Eq. 13 is
    d = pos[:, None, :] - pos[None, :, :]
    r = np.sqrt((d * d).sum(-1))
    iu = np.triu_indices(len(pos), 1)
    sr6 = (sigma / r[iu]) ** 6
    return float((2.0 * eps * sr6 * sr6 - 4.0 * eps * sr6).sum())


def test_lj_vanishes_at_sigma_and_changes_sign():
    for sigma in (1.0, 2.0):                      # contact at rho = 2 in the paper's radius units
        for r, sign in ((0.95 * sigma, +1), (sigma, 0), (1.2 * sigma, -1)):
            pos = np.array([[0.0, 0.0, 0.0], [r, 0.0, 0.0]])
            f = lj_force(pos, 0.7, sigma, 10.0)
            # particle 1 sits at +x of particle 0: repulsion pushes it further along +x
            assert np.sign(round(f[1, 0], 12)) == sign
            assert np.allclose(f[0], -f[1]) and np.allclose(f[:, 1:], 0.0)


def test_lj_is_minus_gradient_of_the_potential():
    rng = np.random.default_rng(3)
    g3 = np.stack(np.meshgrid(*[np.arange(3)] * 3, indexing="ij"), -1).reshape(-1, 3)[:12]
    pos = 1.3 * g3 + rng.uniform(-0.15, 0.15, (12, 3))        # jittered lattice: no pair deep inside the steep core
    eps, sigma = 0.8, 1.1
    f = lj_force(pos, eps, sigma, 1e9)
    h = 1e-6
    for k in (0, 5, 11):
        for a in range(3):
            pp, pm = pos.copy(), pos.copy()
            pp[k, a] += h
            pm[k, a] -= h
            g = (_potential(pp, eps, sigma) - _potential(pm, eps, sigma)) / (2 * h)
            assert abs(f[k, a] + g) <= 1e-6 * max(1.0, abs(g))


def test_lj_newton_third_law_cutoff_and_invariance():
    rng = np.random.default_rng(4)
    pos = rng.uniform(0, 8.0, (300, 3))
    f = lj_force(pos, 1.0, 1.0, 2.5)
    assert np.abs(f.sum(0)).max() <= 1e-9 * np.abs(f).max()
    # translation and rotation
    c, s = np.cos(0.7), np.sin(0.7)
    R = np.array([[c, -s, 0], [s, c, 0], [0, 0, 1.0]])
    f2 = lj_force(pos @ R.T + np.array([3.0, -2.0, 5.0]), 1.0, 1.0, 2.5)
    assert np.allclose(f2, f @ R.T, rtol=1e-9, atol=1e-9 * np.abs(f).max())
    # a particle further than the cut-off from everything feels nothing and exerts nothing
    far = np.vstack([pos, [[100.0, 100.0, 100.0]]])
    f3 = lj_force(far, 1.0, 1.0, 2.5)
    assert np.all(f3[-1] == 0.0) and np.allclose(f3[:-1], f)
    # brute-force double loop on a few particles
    sub = pos[:20]
    ref = np.zeros((20, 3))
    for k in range(20):
        for j in range(20):
            if j == k:
                continue
            d = sub[k] - sub[j]
            r = np.sqrt(d @ d)
            if r < 2.5:
                ref[k] += 24.0 * d / r ** 2 * (r ** -12 - r ** -6)
    assert np.allclose(lj_force(sub, 1.0, 1.0, 2.5), ref, rtol=1e-12, atol=1e-12)


# ------------------------------------------------------------------- walls ----
def test_wall_force_zero_at_sigma_repulsive_inside_and_gradient():
    lo, hi = np.zeros(3), np.array([10.0, 10.0, 10.0])
    eps, sg = 0.9, 0.5
    # one particle near the x = 0 wall only (every other wall beyond the cut-off)
    for d, sign in ((0.45, +1), (0.5, 0), (0.7, -1)):
        f = wall_force(np.array([[d, 5.0, 5.0]]), lo, hi, eps, sg, 2.0)
        assert np.sign(round(f[0, 0], 12)) == sign and f[0, 1] == 0.0 and f[0, 2] == 0.0
    # mirror image at the opposite wall, and beyond the cut-off nothing
    f1 = wall_force(np.array([[0.45, 5.0, 5.0], [9.55, 5.0, 5.0], [5.0, 5.0, 5.0]]), lo, hi, eps, sg, 2.0)
    assert np.isclose(f1[0, 0], -f1[1, 0]) and np.all(f1[2] == 0.0)
    # minus the gradient of the wall potential U(d) = 2 eps (s/d)^12 - 4 eps (s/d)^6 summed over the six walls
    def U(x):
        d = np.concatenate([x - lo, hi - x])
        return float((2 * eps * (sg / d) ** 12 - 4 * eps * (sg / d) ** 6).sum())
    x = np.array([0.62, 9.2, 4.0])
    f = wall_force(x[None, :], lo, hi, eps, sg, 1e9)[0]
    for a in range(3):
        e = np.zeros(3)
        e[a] = 1e-6
        g = (U(x + e) - U(x - e)) / 2e-6
        assert abs(f[a] + g) <= 1e-6 * max(1.0, abs(g))


def test_wall_force_monolayer_box_centres_the_layer():
    # the 2.1 R high box of PAPER.md:204 in diameter units: height 1.05, sigma_w = 0.5 (sphere touching a wall)
    lo, hi = np.array([0.0, 0.0, 0.0]), np.array([50.0, 50.0, 1.05])
    mid = wall_force(np.array([[25.0, 25.0, 0.525]]), lo, hi, 1.0, 0.5, 2.5)
    assert abs(mid[0, 2]) <= 1e-12                                  # the two walls cancel at mid height
    up = wall_force(np.array([[25.0, 25.0, 0.56]]), lo, hi, 1.0, 0.5, 2.5)
    down = wall_force(np.array([[25.0, 25.0, 0.49]]), lo, hi, 1.0, 0.5, 2.5)
    assert up[0, 2] < 0.0 < down[0, 2]                              # restoring towards the mid plane


# ------------------------------------------------------- Euler-Maruyama step ----
def _run(n_steps, dtau, x, v, u, w, h, f, **kw):
    z = np.zeros_like(x)
    for _ in range(n_steps):
        x, v, u, w = md_step(x, v, u, w, z + h, z + f, dtau, **kw)
    return x, v, u, w


def test_translation_drag_decay_and_terminal_velocity():
    one = np.zeros((1, 3))
    dtau, G = 1e-3, 2.0
    x, v, u, w = _run(1000, dtau, one.copy(), one + [1.0, 0, 0], one + [0, 0, 1.0], one.copy(), 0.0, 0.0, gamma_d=G)
    assert abs(v[0, 0] - np.exp(-G)) <= 3e-3 * np.exp(-G)                 # v = v0 exp(-Gamma tau), Euler error n (G dtau)^2 / 2
    assert abs(x[0, 0] - (1 - np.exp(-G)) / G) <= 2e-3
    # constant force: v -> f / Gamma, x ~ (f / Gamma) tau at late times
    x, v, u, w = _run(8000, dtau, one.copy(), one.copy(), one + [0, 0, 1.0], one.copy(), 0.0, np.array([0, 3.0, 0]),
                      gamma_d=G)
    assert abs(v[0, 1] - 1.5) <= 1e-5
    # no drag: uniform acceleration, x = f tau^2 / 2 (explicit Euler: f tau (tau - dtau) / 2)
    x, v, u, w = _run(1000, dtau, one.copy(), one.copy(), one + [0, 0, 1.0], one.copy(), 0.0, np.array([2.0, 0, 0]))
    assert abs(v[0, 0] - 2.0) <= 1e-12 and abs(x[0, 0] - 1.0) <= 2e-3


def test_rotation_small_angle_oscillation_in_a_field():
    # (2/5) theta'' = -h sin(theta)  =>  theta(tau) = theta0 cos(sqrt(5 h / 2) tau) for small theta0
    one = np.zeros((1, 3))
    th0, hz, dtau = 0.02, 1.6, 1e-3
    u0 = one + [np.sin(th0), 0.0, np.cos(th0)]
    om = np.sqrt(2.5 * hz)
    for n in (500, 1571, 3000):
        x, v, u, w = _run(n, dtau, one.copy(), one.copy(), u0.copy(), one.copy(), 0.0, 0.0, h_ext=(0, 0, hz))
        th = np.arctan2(u[0, 0], u[0, 2])
        assert abs(th - th0 * np.cos(om * n * dtau)) <= 0.02 * th0
        assert abs(np.linalg.norm(u[0]) - 1.0) <= 1e-12 and abs(u[0, 1]) <= 1e-15
    # the moment turns TOWARDS the field (reading Q12: literal Eq. 7-8 would leave theta'' = 0)
    x, v, u, w = _run(200, dtau, one.copy(), one.copy(), one + [1.0, 0, 0], one.copy(), 0.0, 0.0, h_ext=(0, 0, 1.0))
    assert u[0, 2] > 0.0


def test_rotation_overdamped_alignment_and_free_spin():
    one = np.zeros((1, 3))
    # strong drag: omega ~ (u x h) / Gamma_r, d(theta)/dtau = -(h / Gamma_r) sin(theta)
    # => tan(theta/2) = tan(theta0/2) exp(-h tau / Gamma_r)
    G, hz, th0, dtau, n = 50.0, 2.0, 2.0, 1e-3, 20000
    u0 = one + [np.sin(th0), 0.0, np.cos(th0)]
    x, v, u, w = _run(n, dtau, one.copy(), one.copy(), u0, one.copy(), 0.0, 0.0, gamma_r=G, h_ext=(0, 0, hz))
    th = np.arctan2(u[0, 0], u[0, 2])
    expect = 2 * np.arctan(np.tan(th0 / 2) * np.exp(-hz * n * dtau / G))
    assert abs(th - expect) <= 0.02 * expect
    # no field, no drag: omega is constant and u turns about it at the rate |omega|
    x, v, u, w = _run(1000, dtau, one.copy(), one.copy(), one + [1.0, 0, 0], one + [0, 0, 0.5], 0.0, 0.0)
    assert np.allclose(w[0], [0, 0, 0.5])
    assert abs(np.arctan2(u[0, 1], u[0, 0]) - 0.5) <= 1e-3


def test_noise_enters_as_amplitude_times_sqrt_dtau():
    one = np.zeros((2, 3))
    xi_d = np.array([[1.0, -2.0, 0.5], [0.0, 1.0, 3.0]])
    xi_r = -xi_d
    x, v, u, w = md_step(one, one, one + [0, 0, 1.0], one, one, one, 0.01, noise_d=0.3, noise_r=0.2, xi_d=xi_d, xi_r=xi_r)
    assert np.allclose(v, 0.3 * 0.1 * xi_d) and np.allclose(w, 0.2 * 0.1 * xi_r)
