"""ff_eval_direct_static: the all-pairs entry point for callers that cannot allocate device memory.

Some users of this library run where a cudaMalloc of their own is off the table: a framework's memory pool already
owns the whole GPU, they sit in a latency-critical loop that must not take cudaMalloc's device-wide stall, or they
are a plug-in that is handed fixed input and output buffers and has no workspace to give to ff_create.  For them
ff_eval_direct_static keeps the kernel's fp64 partial sums in a fixed 3 MiB array built into libff.so
(include/ff.h; limit n <= FF_STATIC_MAX_N).

What is checked here: its H and F against the existing ff_eval_direct path (workspace scratch) within the tolerance
the all-pairs tests use (1e-5, tests/test_gpu_parity.py), on TWO calls in a row that share the array -- the second
one smaller and on different data, so anything read from what the first call left behind would show -- plus the
size limit and the NULL-output forms.  No oracle involved: both sides are the CUDA path.

The file is named so that pytest collects it last (-x stops at the first failure; a failure here must not hide
the parity tests) and it sets up everything it needs itself, so it passes alone in a fresh process as well.
"""
import numpy as np
import pytest

import ffgen
from helpers import rel_err

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

TOL_DIRECT = 1e-5


@pytest.fixture(scope="module")
def ff():
    import paper_1212_2934_b200 as ff
    if not torch.cuda.is_available():
        pytest.fail("gpu tests need a CUDA device (no CPU fallback exists)")
    return ff


def _dev(a):
    return torch.from_numpy(np.ascontiguousarray(a, dtype=np.float32)).cuda()


def _existing_path(ff, pos, mom):
    ctx = ff.FFContext(pos.shape[0], 0.5)
    H, F = ctx.eval_direct(pos, mom)
    torch.cuda.synchronize()
    return H.cpu().numpy(), F.cpu().numpy()


def _agree(x, ref):
    e = rel_err(x, ref)            # e_k = |x_k - ref_k| / max(|ref_k|, 1e-3 rms |ref|), the survey's metric
    assert e[0] <= TOL_DIRECT, e


def test_two_calls_in_a_row_match_the_workspace_path(ff):
    cfg = ffgen.config(1)                                   # N = 4096: 16 source splits, the array used to the brim
    pos1, mom1 = _dev(cfg["pos"]), _dev(cfg["mom"])
    rng = np.random.default_rng(2934)
    n2 = 1000                                               # ragged: not a multiple of the 256-source tile
    pos2 = _dev(rng.uniform(0.0, 40.0, (n2, 3)))
    u = rng.normal(size=(n2, 3))
    mom2 = _dev(u / np.linalg.norm(u, axis=1, keepdims=True))

    # outputs are the caller's; poison them so a row the kernels skip cannot pass
    H1, F1 = torch.full_like(pos1, float("nan")), torch.full_like(pos1, float("nan"))
    H2, F2 = torch.full_like(pos2, float("nan")), torch.full_like(pos2, float("nan"))
    ff.eval_direct_static(pos1, mom1, H1, F1)               # first call on this device: does the set-up
    ff.eval_direct_static(pos2, mom2, H2, F2)               # second call, same stream: runs after the first
    torch.cuda.synchronize()

    Hr1, Fr1 = _existing_path(ff, pos1, mom1)
    Hr2, Fr2 = _existing_path(ff, pos2, mom2)
    _agree(H1.cpu().numpy(), Hr1)
    _agree(F1.cpu().numpy(), Fr1)
    _agree(H2.cpu().numpy(), Hr2)
    _agree(F2.cpu().numpy(), Fr2)

    # and once more on the first input: the array now holds the second call's sums
    H3, F3 = torch.full_like(pos1, float("nan")), torch.full_like(pos1, float("nan"))
    ff.eval_direct_static(pos1, mom1, H3, F3)
    torch.cuda.synchronize()
    assert torch.equal(H3, H1) and torch.equal(F3, F1)      # same input, same launch shape: the same bits


def test_one_output_may_be_left_out(ff):
    rng = np.random.default_rng(7)
    n = 777
    pos = _dev(rng.uniform(0.0, 30.0, (n, 3)))
    mom = _dev(rng.normal(size=(n, 3)))
    H, F = torch.empty_like(pos), torch.empty_like(pos)
    ff.eval_direct_static(pos, mom, H, F)
    Ho, Fo = torch.empty_like(pos), torch.empty_like(pos)
    ff.eval_direct_static(pos, mom, Ho, None)
    ff.eval_direct_static(pos, mom, None, Fo)
    torch.cuda.synchronize()
    assert torch.equal(Ho, H) and torch.equal(Fo, F)


def test_sizes_beyond_the_array_are_refused(ff):
    n = ff.FF_STATIC_MAX_N + 1
    pos = torch.zeros(n, 3, device="cuda")
    out = torch.full_like(pos, 5.0)
    with pytest.raises(ff.FFError) as err:
        ff.eval_direct_static(pos, pos, out, out)
    assert err.value.code == ff.FF_ERR_TOO_LARGE
    assert "FF_STATIC_MAX_N" in str(err.value) and str(n) in str(err.value)
    torch.cuda.synchronize()
    assert bool((out == 5.0).all())                         # nothing was launched
    # the largest allowed size runs (two source splits fill the array exactly)
    rng = np.random.default_rng(11)
    nmax = ff.FF_STATIC_MAX_N
    p = _dev(rng.uniform(0.0, 120.0, (nmax, 3)))
    m = _dev(rng.normal(size=(nmax, 3)))
    H, F = torch.empty_like(p), torch.empty_like(p)
    ff.eval_direct_static(p, m, H, F)
    torch.cuda.synchronize()
    Hr, Fr = _existing_path(ff, p, m)
    _agree(H.cpu().numpy(), Hr)
    _agree(F.cpu().numpy(), Fr)
