"""Physics validation at reduced scale: the paper's own accuracy benchmark.

PAPER.md:206-233 (Eq. 15-18, Fig. 3): for a dilute ferrofluid with weak coupling the reduced magnetisation
<u_z> follows the Langevin function L(alpha) = coth(alpha) - 1/alpha.  Here ff_step runs N = 4096 dipoles at
volume fraction 1 % with thermal noise; the expected values are analytic, nothing comes from the CUDA path.

Reduced units of the step (reading Q15): the energy of a moment is -u.h and the moment of inertia is
2/5, so with a bath of reduced temperature T the fluctuation-dissipation theorem fixes the two amplitudes,
    noise_r = 5/2 sqrt(2 Gamma_r T),   noise_d = sqrt(2 Gamma_d T),
alpha = h_ext / T, and equipartition gives <omega_a^2> = 5 T / 2 and <v_a^2> = T per component.
"""
import numpy as np
import pytest

import ffgen

pytestmark = pytest.mark.gpu


def _langevin(a):
    return 1.0 / np.tanh(a) - 1.0 / a


@pytest.mark.parametrize("alpha", [1.0, 3.0])
def test_magnetisation_follows_the_langevin_function(alpha):
    import torch
    import paper_1212_2934_b200 as ff
    assert torch.cuda.is_available()
    N, T, G = 4096, 4.0, 2.0                     # coupling lambda ~ 1/T < 1 (lambda < 1, phi = 1 %)
    pos, mom, L = ffgen.ensemble(N, 0.01, "isotropic", 5.0, 11)
    p = ff.ff_step_params()
    p.dtau, p.gamma_d, p.gamma_r = 2e-3, G, G
    p.h_ext[0], p.h_ext[1], p.h_ext[2] = 0.0, 0.0, alpha * T
    p.lj_epsilon, p.lj_sigma, p.lj_cutoff = 1.0, 1.0, 2.5
    p.noise_r = 2.5 * np.sqrt(2 * G * T)
    p.noise_d = np.sqrt(2 * G * T)
    p.seed = 5
    x, u = torch.from_numpy(pos).cuda(), torch.from_numpy(mom).cuda()
    v, w = torch.zeros_like(x), torch.zeros_like(x)
    ctx = ff.FFContext(N, 0.5)
    uz, w2, v2 = [], [], []
    for s in range(3000):
        ctx.step(x, v, u, w, p, s)
        if s >= 1500 and s % 25 == 0:
            uz.append(float(u[:, 2].double().mean()))
            w2.append(float((w.double() ** 2).mean()))
            v2.append(float((v.double() ** 2).mean()))
    assert torch.isfinite(x).all() and torch.isfinite(u).all()
    assert abs(float(u.double().norm(dim=1).mean()) - 1.0) < 1e-6
    m = float(np.mean(uz))
    # 3 %: statistical error ~ 0.5 %, O(dtau) bias of Euler-Maruyama and the weak dipolar coupling the rest
    assert abs(m - _langevin(alpha)) <= 0.03 * _langevin(alpha), (m, _langevin(alpha))
    assert abs(np.mean(w2) - 2.5 * T) <= 0.05 * 2.5 * T, np.mean(w2)          # equipartition, rotation
    assert abs(np.mean(v2) - T) <= 0.05 * T, np.mean(v2)                      # equipartition, translation


def test_average_dipole_field_barnes_hut_vs_all_pairs():
    """PAPER.md:239-243 (Fig. 4): the average dipole field <h_z^dip> from the Barnes-Hut and the All-Pairs
    algorithms "almost identical".  Here: N = 8192 at phi = 5 %, moments partially aligned by a field (the state
    after 400 thermal steps at alpha = 3), theta = 0.5; both averages over the same configuration."""
    import torch
    import paper_1212_2934_b200 as ff
    N, T, G, alpha = 8192, 4.0, 2.0, 3.0
    pos, mom, L = ffgen.ensemble(N, 0.05, "isotropic", 5.0, 21)
    p = ff.ff_step_params()
    p.dtau, p.gamma_d, p.gamma_r = 2e-3, G, G
    p.h_ext[2] = alpha * T
    p.lj_epsilon, p.lj_sigma, p.lj_cutoff = 1.0, 1.0, 2.5
    p.noise_r, p.noise_d, p.seed = 2.5 * np.sqrt(2 * G * T), np.sqrt(2 * G * T), 9
    x, u = torch.from_numpy(pos).cuda(), torch.from_numpy(mom).cuda()
    v, w = torch.zeros_like(x), torch.zeros_like(x)
    ctx = ff.FFContext(N, 0.5)
    for s in range(400):
        ctx.step(x, v, u, w, p, s)
    ctx.build_tree(x)
    Hb, _ = ctx.eval_bh(x, u)
    Hd, _ = ctx.eval_direct(x, u)
    hb, hd = float(Hb[:, 2].double().mean()), float(Hd[:, 2].double().mean())
    assert float(u[:, 2].mean()) > 0.5                       # the sample is magnetised, <h_z^dip> is not noise
    assert abs(hd) > 1e-3
    assert abs(hb - hd) <= 0.03 * abs(hd), (hb, hd)
    # third leg: the fp64 oracle's all-pairs sum on the SAME configuration (the two GPU kernels share their pair
    # arithmetic, so agreeing with each other proves less than agreeing with the oracle) -- <h_z> and every row
    import oracle
    xs, us = x.cpu().numpy(), u.cpu().numpy()
    Ho, _, Qo = oracle.allpairs(xs, us, scale=True)
    ho = float(Ho[:, 2].mean())
    assert abs(hd - ho) <= 1e-5 * abs(ho), (hd, ho)
    assert abs(hb - ho) <= 0.03 * abs(ho), (hb, ho)
    e = np.linalg.norm(Hd.cpu().numpy() - Ho, axis=1) / np.maximum(np.linalg.norm(Ho, axis=1), Qo[:, 0] / 8.0)
    assert e.max() <= 1e-5, e.max()
    # ... and the oracle's Barnes-Hut <h_z> at the same theta and group width equals the GPU's
    Hob, _, _, _ = oracle.barnes_hut(xs, us, 0.5, 32)
    assert abs(hb - float(Hob[:, 2].mean())) <= 1e-5 * abs(ho)
    # the per-particle fields differ by the percent-level error of Eq. 14's lowest-order cell
    rel = float((Hb - Hd).double().norm() / Hd.double().norm())
    assert rel < 0.06


def test_magnetisation_all_pairs_and_barnes_hut_agree():
    """PAPER.md:233, Fig. 3(b): the magnetisation of N = 10^3 particles from the All-Pairs and the Barnes-Hut
    algorithm, "almost identical".  Same initial state and noise stream for both; each must follow L(alpha)."""
    import torch
    import paper_1212_2934_b200 as ff
    N, T, G, alpha = 1024, 4.0, 2.0, 2.0
    pos, mom, L = ffgen.ensemble(N, 0.01, "isotropic", 5.0, 31)
    res = {}
    for name, flag in (("bh", 0), ("ap", 1)):
        p = ff.ff_step_params()
        p.dtau, p.gamma_d, p.gamma_r = 2e-3, G, G
        p.h_ext[2] = alpha * T
        p.lj_epsilon, p.lj_sigma, p.lj_cutoff = 1.0, 1.0, 2.5
        p.noise_r, p.noise_d, p.seed = 2.5 * np.sqrt(2 * G * T), np.sqrt(2 * G * T), 3
        p.all_pairs = flag
        x, u = torch.from_numpy(pos).cuda(), torch.from_numpy(mom).cuda()
        v, w = torch.zeros_like(x), torch.zeros_like(x)
        ctx = ff.FFContext(N, 0.5)
        uz = []
        for s in range(6000):
            ctx.step(x, v, u, w, p, s)
            if s >= 1000 and s % 20 == 0:
                uz.append(float(u[:, 2].double().mean()))
        res[name] = float(np.mean(uz))
    lang = _langevin(alpha)
    assert abs(res["ap"] - lang) <= 0.04 * lang and abs(res["bh"] - lang) <= 0.04 * lang, (res, lang)
    assert abs(res["ap"] - res["bh"]) <= 0.03 * lang, res
