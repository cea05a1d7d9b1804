"""oracle.md_step -- plain fp64 numpy statement of the steps either side of the hot path.

TEST INFRASTRUCTURE ONLY (same rule as oracle/__init__.py): imported by tests/ and by bench.py's
reference leg, never by the CUDA package, and it imports nothing of it.

What is computed, in the paper's notation (all citations are lines of /root/reference/PAPER.md):

* lj_force      Eq. 13: f_k^sr = 24 eps sum_{j != k} rho_kj / rho_kj^2 [ (sigma/rho_kj)^12 - (sigma/rho_kj)^6 ],
                taken literally (no factor 2 on the r^-12 term: the force vanishes at rho = sigma, PAPER.md:52;
                DESIGN.md reading Q14), restricted to pairs with rho_kj < cutoff (reading Q16).
* wall_force    PAPER.md:52: "The interaction between a particle and container walls is also modeled with a
                Lennard-Jones potential of the same type" (containers: PAPER.md:204, a cube and a 2.1 R high
                monolayer box).  Reading Q20: each of the six planes of an axis-aligned box acts on a
                particle inside it with the pair term of Eq. 13 evaluated at the distance vector from the plane to
                the particle centre, f = 24 eps_w n / d [ (sigma_w/d)^12 - (sigma_w/d)^6 ], n = inward normal,
                for d < cutoff; sigma_w is the centre-to-wall distance at which the force vanishes.
* md_step       one Euler-Maruyama step of size dtau of Eq. 9 and of the rotational
                equations in the vector form of DESIGN.md reading Q12 (Eq. 7-8, attach the torque
                components to the wrong angles; 2/5 = I/(M R^2)):
                    d(rho)/dtau   = v
                    d(v)/dtau     = f^dip + f^sr - Gamma_d v            (+ noise_d xi_d / sqrt(dtau))
                    d(omega)/dtau = 5/2 (u x h - Gamma_r omega)         (+ noise_r xi_r / sqrt(dtau))
                    d(u)/dtau     = omega x u,   then u <- u / |u|
                with h = h^dip + h^ext (Eq. 10).  Explicit: every right-hand side uses the values at
                the START of the step.  The unit Gaussians xi are INPUTS (reading Q15: the thermal amplitudes of
                PAPER.md:52, 78 are garbled, so the two dimensionless amplitudes are parameters; 0 = deterministic).

Pinned in tests/test_oracle_step.py against closed forms (potential gradient, zero at sigma, Newton's third law,
exponential velocity decay, terminal velocity, small-angle oscillation of a dipole in a field, free rotation).
No blocking, no neighbour lists: the pair sum is the plain double loop written with numpy broadcasting in
row chunks.
"""
from __future__ import annotations

import numpy as np


def lj_force(pos, eps: float, sigma: float, cutoff: float, chunk: int = 512, targets=None):
    """Eq. 13 summed over all j != k with |rho_kj| < cutoff.  pos [N][3] -> f^sr [N][3], fp64.
    targets: optional index array -> only those k are evaluated (still against ALL j) and row t belongs to targets[t]."""
    p = np.asarray(pos, dtype=np.float64)
    n = len(p)
    tk = np.arange(n) if targets is None else np.asarray(targets, dtype=np.int64)
    f = np.zeros((len(tk), 3))
    for a in range(0, len(tk), chunk):
        k = tk[a:a + chunk]
        rho = p[k, None, :] - p[None, :, :]                       # rho_kj = rho_k - rho_j
        r2 = np.einsum("kja,kja->kj", rho, rho)
        r2[np.arange(len(k)), k] = np.inf                         # j != k, by index
        inside = r2 < cutoff * cutoff
        r2 = np.where(inside, r2, np.inf)
        sr6 = (sigma * sigma / r2) ** 3
        w = 24.0 * eps * (sr6 * sr6 - sr6) / r2                   # [ (s/r)^12 - (s/r)^6 ] / r^2
        f[a:a + chunk] = np.einsum("kj,kja->ka", w, rho)
    return f


def wall_force(pos, lo, hi, eps: float, sigma: float, cutoff: float):
    """Force of the six walls of the box [lo, hi] on particles inside it.  pos [N][3] -> [N][3], fp64."""
    p = np.asarray(pos, dtype=np.float64)
    lo = np.asarray(lo, dtype=np.float64)
    hi = np.asarray(hi, dtype=np.float64)
    f = np.zeros_like(p)
    for a in range(3):
        for d, sign in ((p[:, a] - lo[a], +1.0), (hi[a] - p[:, a], -1.0)):     # distance to the wall, inward normal
            d = np.where(d < cutoff, d, np.inf)
            sr6 = (sigma / d) ** 6
            f[:, a] += sign * 24.0 * eps * (sr6 * sr6 - sr6) / d
    return f


def md_step(pos, vel, mom, angvel, h_dip, f_dip, dtau: float, gamma_d: float = 0.0, gamma_r: float = 0.0,
            h_ext=(0.0, 0.0, 0.0), f_sr=None, noise_d: float = 0.0, noise_r: float = 0.0, xi_d=None, xi_r=None):
    """One explicit Euler-Maruyama step.  Returns (pos, vel, mom, angvel) after the step, fp64."""
    x = np.asarray(pos, dtype=np.float64)
    v = np.asarray(vel, dtype=np.float64)
    u = np.asarray(mom, dtype=np.float64)
    w = np.asarray(angvel, dtype=np.float64)
    h = np.asarray(h_dip, dtype=np.float64) + np.asarray(h_ext, dtype=np.float64)[None, :]   # Eq. 10
    f = np.asarray(f_dip, dtype=np.float64).copy()
    if f_sr is not None:
        f += np.asarray(f_sr, dtype=np.float64)
    sq = np.sqrt(dtau)
    kick_d = noise_d * sq * np.asarray(xi_d, dtype=np.float64) if noise_d != 0.0 else 0.0
    kick_r = noise_r * sq * np.asarray(xi_r, dtype=np.float64) if noise_r != 0.0 else 0.0
    x_new = x + dtau * v
    v_new = v + dtau * (f - gamma_d * v) + kick_d                                 # Eq. 9
    w_new = w + dtau * 2.5 * (np.cross(u, h) - gamma_r * w) + kick_r              # Eq. 7-8, vector form
    u_new = u + dtau * np.cross(w, u)
    u_new /= np.linalg.norm(u_new, axis=1, keepdims=True)
    return x_new, v_new, u_new, w_new
