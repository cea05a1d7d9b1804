"""Negative control of the checked build (FF_CHECKED=1, libff_checked.so): a deliberately corrupted tree must raise
FF_ERR_CHECK.  One entry of the sorted-to-caller permutation is overwritten with an out-of-range row (through the
caller-owned workspace tensor); the walk's epilogue then scatters one result row out of range.  The output tensors are
views of larger allocations, so that stray row lands in memory this script owns.  Run by
tests/test_gpu_parity.py::test_checked_build_catches_a_corrupted_tree; exits 0 iff the check fired."""
import ctypes
import os
import sys

sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.abspath(__file__))))

import torch

import ffgen
import paper_1212_2934_b200 as ff


def main():
    assert os.environ.get("FF_CHECKED") == "1", "run with FF_CHECKED=1"
    N = 3000
    c = ffgen.config(1, N=N)
    pos, mom = torch.from_numpy(c["pos"]).cuda(), torch.from_numpy(c["mom"]).cuda()
    Hbig, Fbig = torch.zeros((N + 64, 3), device="cuda"), torch.zeros((N + 64, 3), device="cuda")
    H, F = Hbig[:N], Fbig[:N]
    ctx = ff.FFContext(N, 0.5, timing=True)
    ctx.build_tree(pos)
    ctx.eval_bh(pos, mom, H, F)
    ctx.timings()                                          # clean tree: no error
    v = ff.ff_tree_view()
    assert ctx._L.ff_get_tree(ctx._h, ctypes.byref(v)) == ff.FF_OK
    off = v.perm - ctx.workspace.data_ptr()
    perm = ctx.workspace[off:off + 4 * N].view(torch.int32)
    perm[17] = N + 5                                       # out of range, but inside Hbig / Fbig
    ctx.eval_bh(pos, mom, H, F)
    torch.cuda.synchronize()
    try:
        ctx.timings()
    except ff.FFError as e:
        assert e.code == ff.FF_ERR_CHECK, e
        print("checked build caught the corrupted permutation:", e)
        return 0
    print("the corrupted permutation was NOT caught")
    return 1


if __name__ == "__main__":
    sys.exit(main())
