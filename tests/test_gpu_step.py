"""GPU parity of ff_step against oracle/md_step.py + the Barnes-Hut oracle.

One step from a given state is deterministic (noise amplitudes 0): the GPU's new state is compared with the
oracle's step from the SAME state, with h^dip, f^dip from the oracle's Barnes-Hut at the same theta and group
width and f^sr from the plain pair sum of Eq. 13.  For a multi-step run the oracle is re-evaluated on the
GPU's own states (trajectories of a chaotic many-body system are not compared), SURVEY.md 8(d).
"""
import numpy as np
import pytest

import ffgen
import oracle
from oracle.md_step import lj_force, md_step, wall_force

pytestmark = pytest.mark.gpu

# north_star's Barnes-Hut tolerance, applied to the increments of the step (the increments are sums
# of the Barnes-Hut force / torque, the pair force of Eq. 13 and the drag term, each carrying its own fp32 rounding)
TOL_STEP = 1e-4


@pytest.fixture(scope="module")
def ff():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    import paper_1212_2934_b200 as ff
    ff.lib()
    return ff


def _dev(a):
    import torch
    return torch.from_numpy(np.ascontiguousarray(a, dtype=np.float32)).cuda()


def _params(ff, **kw):
    p = ff.ff_step_params()
    p.dtau = kw.get("dtau", 1e-3)
    p.gamma_d = kw.get("gamma_d", 0.0)
    p.gamma_r = kw.get("gamma_r", 0.0)
    for a in range(3):
        p.h_ext[a] = kw.get("h_ext", (0.0, 0.0, 0.0))[a]
    p.lj_epsilon = kw.get("eps", 0.0)
    p.lj_sigma = kw.get("sigma", 1.0)
    p.lj_cutoff = kw.get("cutoff", 2.5)
    p.noise_d = kw.get("noise_d", 0.0)
    p.noise_r = kw.get("noise_r", 0.0)
    p.seed = kw.get("seed", 0)
    for a in range(3):
        p.wall_lo[a] = kw.get("wall_lo", (0.0, 0.0, 0.0))[a]
        p.wall_hi[a] = kw.get("wall_hi", (0.0, 0.0, 0.0))[a]
    p.wall_epsilon = kw.get("wall_eps", 0.0)
    p.wall_sigma = kw.get("wall_sigma", 0.5)
    p.all_pairs = 1 if kw.get("all_pairs", False) else 0
    return p


def _oracle_step(x, v, u, w, theta, kw):
    """fp64 step from the fp32 state (x, v, u, w) the GPU started from."""
    if kw.get("all_pairs", False):
        H, F, Q = oracle.allpairs(x, u, scale=True)
    else:
        H, F, _, _, Q = oracle.barnes_hut(x, u, theta, 32, scale=True)
    fsr = lj_force(x, kw["eps"], kw["sigma"], kw["cutoff"]) if kw.get("eps", 0.0) != 0.0 else None
    if kw.get("wall_eps", 0.0) != 0.0:
        fw = wall_force(x, kw["wall_lo"], kw["wall_hi"], kw["wall_eps"], kw["wall_sigma"], kw.get("cutoff", 2.5))
        fsr = fw if fsr is None else fsr + fw
    out = md_step(x, v, u, w, H, F, kw.get("dtau", 1e-3), kw.get("gamma_d", 0.0), kw.get("gamma_r", 0.0),
                  kw.get("h_ext", (0.0, 0.0, 0.0)), fsr)
    return out, (H, F, Q, fsr)


def _check_step(before, after, ref, aux, kw, subtract_rep=True):
    """Compare through the increments, which is where the arithmetic of the step sits.

    subtract_rep=False gates the RAW error (nothing taken off): for states that start at rest, where the representation
    term below vanishes and the tolerance applies to the arithmetic of the step alone.  Returns, for the record, the raw
    maximum errors and the largest share of the gate the subtraction absorbed."""
    x0, v0, u0, w0 = [a.astype(np.float64) for a in before]
    x1, v1, u1, w1 = [a.astype(np.float64) for a in after]
    xr, vr, ur, wr = ref
    H, F, Q, fsr = aux
    dt = kw.get("dtau", 1e-3)
    ulp = 2.0 ** -24
    # positions: x + dtau v, one fp32 rounding of the result and of the product
    assert np.abs(x1 - xr).max() <= 4 * ulp * max(1.0, np.abs(xr).max())
    # velocity increment / dtau = total force - drag.  Two things are kept apart:
    #  (1) the REPRESENTATION error of the fp32 state the increment is recovered from: v1 is stored with a relative
    #      rounding of at most 2^-24 per component, i.e. an absolute 2^-24 |v1| / dtau in the increment, whatever the
    #      forces are (it dominates for an isolated, slowly accelerating particle) -- subtracted before the gate;
    #  (2) the error of the arithmetic of the step, gated at north_star's 1e-4 relative to the scale of the force
    #      terms: max(|total|, Q_f / 8, |f_sr| / 8), as for the Barnes-Hut force itself.
    acc_gpu, acc_ref = (v1 - v0) / dt, (vr - v0) / dt
    scale = np.maximum(np.linalg.norm(acc_ref, axis=1), Q[:, 1] / 8.0)
    if fsr is not None:
        scale = np.maximum(scale, np.linalg.norm(fsr, axis=1) / 8.0)
    rep = ulp * np.linalg.norm(v1, axis=1) / dt if subtract_rep else np.zeros(len(v1))
    raw = np.linalg.norm(acc_gpu - acc_ref, axis=1)
    err = np.maximum(raw - rep, 0.0) / scale
    assert err.max() <= TOL_STEP, err.max()
    # the same gate written on the raw error, row by row, so that what the subtraction absorbs is visible: the raw
    # error may exceed the tolerance only by that row's own representation term
    assert (raw <= rep + TOL_STEP * scale).all()
    # angular-velocity increment / dtau = 5/2 (u x h - Gamma_r omega)
    t_gpu, t_ref = (w1 - w0) / dt, (wr - w0) / dt
    tscale = np.maximum(np.linalg.norm(t_ref, axis=1), 2.5 * Q[:, 0] / 8.0)
    trep = ulp * np.linalg.norm(w1, axis=1) / dt if subtract_rep else np.zeros(len(w1))
    traw = np.linalg.norm(t_gpu - t_ref, axis=1)
    terr = np.maximum(traw - trep, 0.0) / tscale
    assert terr.max() <= TOL_STEP, terr.max()
    assert (traw <= trep + TOL_STEP * tscale).all()
    # moments: unit length, and the same direction as the oracle's
    assert np.abs(np.linalg.norm(u1, axis=1) - 1.0).max() <= 4 * ulp
    assert np.abs(u1 - ur).max() <= 8 * ulp
    # how much the subtraction absorbed is reported, not hidden (pytest -s / -rP shows it); the from-rest test below is
    # the one where it absorbs nothing
    stats = dict(raw_acc=float((raw / scale).max()), raw_torque=float((traw / tscale).max()),
                 gated_acc=float(err.max()), gated_torque=float(terr.max()),
                 rep_share_acc=float((rep / scale).max() / TOL_STEP), rep_share_torque=float((trep / tscale).max() / TOL_STEP))
    print("step parity:", stats)
    return stats


KW = dict(dtau=1e-3, gamma_d=0.7, gamma_r=1.3, h_ext=(0.0, 0.1, 0.4), eps=0.5, sigma=1.0, cutoff=2.5)


def _state(cfg_id, N, seed):
    c = ffgen.config(cfg_id, N=N, seed=seed)
    rng = np.random.default_rng(seed + 100)
    v = (0.05 * rng.standard_normal((N, 3))).astype(np.float32)
    w = (0.2 * rng.standard_normal((N, 3))).astype(np.float32)
    return c["pos"], v, c["mom"], w


@pytest.mark.parametrize("cfg_id,N", [(1, 4096), (1, 1531), (2, 6000)])
def test_one_step_matches_oracle(ff, cfg_id, N):
    x, v, u, w = _state(cfg_id, N, 0)
    ctx = ff.FFContext(N, 0.5)
    dx, dv, du, dw = _dev(x), _dev(v), _dev(u), _dev(w)
    ctx.step(dx, dv, du, dw, _params(ff, **KW), 0)
    after = [t.cpu().numpy() for t in (dx, dv, du, dw)]
    ref, aux = _oracle_step(x, v, u, w, 0.5, KW)
    _check_step((x, v, u, w), after, ref, aux, KW)
    # the short-range force is not trivially zero in this test
    assert np.linalg.norm(aux[3], axis=1).max() > 0.1


@pytest.mark.parametrize("all_pairs", [False, True])
def test_step_from_rest_gates_the_arithmetic_alone(ff, all_pairs):
    """v = omega = 0 at the start: the new velocities are dtau x (force), stored with a relative 2^-24, so the
    representation term of _check_step is ~6e-8 of the force and nothing is subtracted: the 1e-4 gate applies to the raw
    error of the step's arithmetic (Barnes-Hut or all-pairs field and force, Eq. 13, the update)."""
    N = 3000
    x, _, u, _ = _state(1, N, 5)
    v, w = np.zeros_like(x), np.zeros_like(x)
    kw = dict(KW, all_pairs=all_pairs)
    ctx = ff.FFContext(N, 0.5)
    dx, dv, du, dw = _dev(x), _dev(v), _dev(u), _dev(w)
    ctx.step(dx, dv, du, dw, _params(ff, **kw), 0)
    after = [t.cpu().numpy() for t in (dx, dv, du, dw)]
    ref, aux = _oracle_step(x, v, u, w, 0.5, kw)
    stats = _check_step((x, v, u, w), after, ref, aux, kw, subtract_rep=False)
    assert stats["rep_share_acc"] == 0.0 and stats["gated_acc"] == stats["raw_acc"]


def test_refused_parameters_enqueue_nothing(ff):
    """Every parameter check of ff_step runs before its first launch (tree path and all-pairs path): a refused call
    leaves the state arrays and the context's launch count as they were."""
    import torch
    N = 512
    x, v, u, w = _state(1, N, 9)
    ctx = ff.FFContext(N, 0.5)
    for bad in (dict(wall_eps=1.0, wall_sigma=0.0, wall_lo=(0, 0, 0), wall_hi=(90, 90, 90)),
                dict(wall_eps=1.0, wall_sigma=0.5, cutoff=0.0, eps=0.0, wall_lo=(0, 0, 0), wall_hi=(90, 90, 90)),
                dict(eps=0.5, sigma=0.0), dict(eps=0.5, cutoff=-1.0), dict(dtau=0.0)):
        for all_pairs in (False, True):
            kw = dict(KW, **bad, all_pairs=all_pairs)
            dx, dv, du, dw = _dev(x), _dev(v), _dev(u), _dev(w)
            before = ctx.launch_count()
            with pytest.raises(ff.FFError) as err:
                ctx.step(dx, dv, du, dw, _params(ff, **kw), 0)
            assert err.value.code == ff.FF_ERR_INVALID_ARG
            assert ctx.launch_count() == before, (bad, all_pairs)
            torch.cuda.synchronize()
            assert np.array_equal(dx.cpu().numpy(), x) and np.array_equal(dv.cpu().numpy(), v)
    # and the context still works
    dx, dv, du, dw = _dev(x), _dev(v), _dev(u), _dev(w)
    ctx.step(dx, dv, du, dw, _params(ff, **KW), 0)
    assert ctx.launch_count() > before


def test_step_without_short_range_force_and_drag(ff):
    kw = dict(dtau=2e-3)
    x, v, u, w = _state(1, 2048, 3)
    ctx = ff.FFContext(2048, 0.4)
    dx, dv, du, dw = _dev(x), _dev(v), _dev(u), _dev(w)
    ctx.step(dx, dv, du, dw, _params(ff, **kw), 0)
    after = [t.cpu().numpy() for t in (dx, dv, du, dw)]
    ref, aux = _oracle_step(x, v, u, w, 0.4, kw)
    _check_step((x, v, u, w), after, ref, aux, kw)


def test_twenty_steps_checked_on_the_gpu_states(ff):
    N = 4096
    x, v, u, w = _state(1, N, 1)
    ctx = ff.FFContext(N, 0.5)
    dx, dv, du, dw = _dev(x), _dev(v), _dev(u), _dev(w)
    p = _params(ff, **KW)
    for s in range(20):
        before = [t.cpu().numpy().copy() for t in (dx, dv, du, dw)]
        ctx.step(dx, dv, du, dw, p, s)
        if s in (0, 10, 19):
            after = [t.cpu().numpy() for t in (dx, dv, du, dw)]
            ref, aux = _oracle_step(*before, 0.5, KW)
            _check_step(before, after, ref, aux, KW)
    # hard spheres at contact with sigma = 1 stay apart over 20 short steps
    xs = dx.cpu().numpy().astype(np.float64)
    assert np.isfinite(xs).all()


def test_thermal_noise_statistics_and_reproducibility(ff):
    """xi are unit Gaussians keyed by (seed, step, particle, component): mean 0, variance 1, independent
    of the launch; the kick is amplitude * sqrt(dtau) * xi (reading Q15)."""
    import torch
    N = 1 << 16
    c = ffgen.config(1, N=4096)
    x = np.tile(c["pos"], (16, 1)) + np.repeat(np.arange(16), 4096)[:, None].astype(np.float32) * np.float32(100.0)
    u = np.tile(c["mom"], (16, 1))
    z = np.zeros((N, 3), np.float32)
    p = _params(ff, dtau=1e-2, noise_d=0.5, noise_r=0.25, seed=7)
    q = _params(ff, dtau=1e-2)
    ctx = ff.FFContext(N, 0.5)
    outs = []
    for prm in (p, p, q):
        dx, dv, du, dw = _dev(x), _dev(z), _dev(u), _dev(z)
        ctx.step(dx, dv, du, dw, prm, 5)
        outs.append((dv.cpu().numpy().astype(np.float64), dw.cpu().numpy().astype(np.float64)))
    assert np.array_equal(outs[0][0], outs[1][0]) and np.array_equal(outs[0][1], outs[1][1])   # counter-based
    xi_d = (outs[0][0] - outs[2][0]) / (0.5 * 0.1)
    xi_r = (outs[0][1] - outs[2][1]) / (0.25 * 0.1)
    for xi in (xi_d, xi_r):
        assert abs(xi.mean()) <= 0.01 and abs(xi.var() - 1.0) <= 0.02
        assert abs(np.mean(xi ** 4) - 3.0) <= 0.15                                   # Gaussian kurtosis
        cc = np.corrcoef(xi.T)
        assert np.abs(cc - np.eye(3)).max() <= 0.02
    assert abs(np.corrcoef(xi_d[:, 0], xi_r[:, 0])[0, 1]) <= 0.02
    # another step index gives other numbers
    dx, dv, du, dw = _dev(x), _dev(z), _dev(u), _dev(z)
    ctx.step(dx, dv, du, dw, p, 6)
    assert not np.array_equal(dv.cpu().numpy(), outs[0][0].astype(np.float32))


def test_monolayer_between_walls(ff):
    """The paper's second container: a 2.1 R = 1.05 d high box holding one layer of particles.
    Quasi-2D input: the octree degenerates to a quadtree, and the wall forces are large and nearly cancel."""
    rng = np.random.default_rng(8)
    n1 = 64
    g = np.stack(np.meshgrid(np.arange(n1), np.arange(n1), indexing="ij"), -1).reshape(-1, 2).astype(np.float64)
    xy = 1.3 * g + rng.uniform(-0.12, 0.12, g.shape)                      # centres >= 1.06 apart
    z = 0.525 + rng.uniform(-0.03, 0.03, len(g))
    x = np.column_stack([xy, z]).astype(np.float32)
    N = len(x)
    u = ffgen.moments_isotropic(N, 2)
    v = (0.02 * rng.standard_normal((N, 3))).astype(np.float32)
    w = (0.1 * rng.standard_normal((N, 3))).astype(np.float32)
    L = float(1.3 * n1)
    kw = dict(KW, wall_lo=(-1.0, -1.0, 0.0), wall_hi=(L + 1.0, L + 1.0, 1.05), wall_eps=1.0, wall_sigma=0.5)
    ctx = ff.FFContext(N, 0.5, counters=True)
    dx, dv, du, dw = _dev(x), _dev(v), _dev(u), _dev(w)
    ctx.step(dx, dv, du, dw, _params(ff, **kw), 0)
    after = [t.cpu().numpy() for t in (dx, dv, du, dw)]
    ref, aux = _oracle_step(x, v, u, w, 0.5, kw)
    _check_step((x, v, u, w), after, ref, aux, kw)
    fw = wall_force(x, kw["wall_lo"], kw["wall_hi"], 1.0, 0.5, 2.5)
    assert np.abs(fw[:, 2]).max() > 1.0                                   # the walls do act
    # same interaction sets as the oracle on the flat tree
    cnt = oracle.barnes_hut(x, u, 0.5, 32)[2]
    assert ctx.counters() == cnt


@pytest.mark.parametrize("N", [1000, 3001])
def test_all_pairs_step_matches_oracle(ff, N):
    """The paper's All-Pairs step (Algorithm 1): h^dip, f^dip and f^sr from one exact pair loop,
    no tree; against the oracle's all-pairs sums + Eq. 13 + the same update."""
    kw = dict(KW, all_pairs=True, wall_lo=(-5.0, -5.0, -5.0), wall_hi=(60.0, 60.0, 60.0), wall_eps=0.3, wall_sigma=0.5)
    x, v, u, w = _state(1, N, 4)
    ctx = ff.FFContext(N, 0.5)
    dx, dv, du, dw = _dev(x), _dev(v), _dev(u), _dev(w)
    ctx.step(dx, dv, du, dw, _params(ff, **kw), 0)
    after = [t.cpu().numpy() for t in (dx, dv, du, dw)]
    ref, aux = _oracle_step(x, v, u, w, 0.5, kw)
    _check_step((x, v, u, w), after, ref, aux, kw)
    # and the Barnes-Hut step from the same state differs from it only by the approximation error of the tree
    dx2, dv2, du2, dw2 = _dev(x), _dev(v), _dev(u), _dev(w)
    ctx.step(dx2, dv2, du2, dw2, _params(ff, **dict(kw, all_pairs=False)), 0)
    dvel = (dv2 - dv).double().norm() / (dv - _dev(v)).double().norm()
    assert 0.0 < float(dvel) < 0.05
