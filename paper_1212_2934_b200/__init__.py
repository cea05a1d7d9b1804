"""paper_1212_2934_b200 -- thin Python binding of the C-ABI library declared in include/ff.h.

Barnes-Hut dipole field + force for ferrofluid molecular dynamics (arxiv 1212.2934) on one
B200.  Every step of the path runs in the hand-written CUDA kernels of csrc/ (libff.so);
this module only marshals arguments (torch tensors -> device pointers) and owns nothing but
the workspace tensor.  There is NO CPU fallback: without a CUDA device or without libff.so
every call raises.

    ctx = FFContext(N, theta=0.5)
    ctx.build_tree(pos)                     # ff_build_tree
    H, F = ctx.eval_bh(pos, mom)            # ff_eval_bh
    H, F = ctx.eval_direct(pos, mom)        # ff_eval_direct
"""
from __future__ import annotations

import ctypes
import os

from . import build as _build

_lib = None

FF_OK = 0
FF_ERR_INVALID_ARG, FF_ERR_WORKSPACE, FF_ERR_NO_TREE, FF_ERR_CAPACITY, FF_ERR_CUDA, FF_ERR_CHECK = -1, -2, -3, -4, -5, -6
FF_ERR_TOO_LARGE = -7
FF_STATIC_MAX_N = 32768
FF_OPT_THETA, FF_OPT_NLEAF, FF_OPT_COUNTERS, FF_OPT_TIMING, FF_OPT_GROUP, FF_OPT_CELL_ORDER = 1, 2, 3, 4, 5, 6
FF_N_PHASES = 7
PHASES = ("bbox_keys", "sort", "build", "moments", "walk", "direct", "step")
FF_PROBE_FFMA, FF_PROBE_FFMA2_PAIRS, FF_PROBE_FFMA2_REUSE, FF_PROBE_FFMA2_SCALAR, FF_PROBE_EVAL = 0, 1, 2, 3, 4
FF_PROBE_EVAL_SCALAR, FF_PROBE_EVAL_HYBRID = 5, 6
FF_CHILD_EMPTY = -1
FF_CHILD_LEAF1, FF_CHILD_MULTI, FF_CHILD_SLOT = 0x80000000, 0x40000000, 0x3FFFFFFF

# every symbol include/ff.h declares (checked by tests/test_abi.py)
SYMBOLS = (
    "ff_workspace_bytes", "ff_create", "ff_destroy", "ff_set_stream", "ff_set_option", "ff_build_tree",
    "ff_eval_bh", "ff_eval_bh_range", "ff_eval_direct", "ff_eval_bh_host", "ff_eval_direct_host", "ff_step", "ff_get_tree",
    "ff_get_timings", "ff_eval_bh_host_async", "ff_host_sync", "ff_get_counters", "ff_get_prefilter_count", "ff_get_launch_count", "ff_measure_fp32_peak", "ff_measure_probe", "ff_error_string",
    "ff_last_error", "ff_eval_direct_static", "ff_static_last_error",
)


class ff_step_params(ctypes.Structure):
    _fields_ = [("dtau", ctypes.c_float), ("gamma_d", ctypes.c_float), ("gamma_r", ctypes.c_float),
                ("h_ext", ctypes.c_float * 3), ("lj_epsilon", ctypes.c_float), ("lj_sigma", ctypes.c_float),
                ("lj_cutoff", ctypes.c_float), ("noise_d", ctypes.c_float), ("noise_r", ctypes.c_float),
                ("seed", ctypes.c_uint64), ("wall_lo", ctypes.c_float * 3), ("wall_hi", ctypes.c_float * 3),
                ("wall_epsilon", ctypes.c_float), ("wall_sigma", ctypes.c_float),
                ("all_pairs", ctypes.c_int32), ("reserved", ctypes.c_int32)]


class ff_tree_view(ctypes.Structure):
    _fields_ = [("n", ctypes.c_int64), ("n_cells", ctypes.c_int64), ("nleaf", ctypes.c_int32),
                ("lo", ctypes.c_float * 3), ("S", ctypes.c_float),
                ("key", ctypes.c_void_p), ("perm", ctypes.c_void_p), ("pos_sorted", ctypes.c_void_p),
                ("mom_sorted", ctypes.c_void_p), ("cell_first", ctypes.c_void_p), ("cell_end", ctypes.c_void_p),
                ("cell_level", ctypes.c_void_p), ("child", ctypes.c_void_p), ("leaf_count", ctypes.c_void_p),
                ("cell_centre", ctypes.c_void_p), ("cell_moment", ctypes.c_void_p), ("cell_quad", ctypes.c_void_p)]


def shard_groups(n: int, world: int, rank: int, group: int = 32):
    """Target sharding of SURVEY.md 8(e): the walk groups (`group` consecutive sorted targets, FF_OPT_GROUP) of an
    n-particle ensemble split into `world` Morton-contiguous slices of equal size (+-1); returns
    (group_begin, group_end) of `rank`."""
    groups = (n + group - 1) // group
    base, rem = divmod(groups, world)
    begin = rank * base + min(rank, rem)
    return begin, begin + base + (1 if rank < rem else 0)


class FFError(RuntimeError):
    def __init__(self, code, where, detail=""):
        self.code = code
        msg = "%s failed: %s (%d)" % (where, lib().ff_error_string(code).decode(), code)
        super().__init__(msg + (": " + detail if detail else ""))


def lib():
    """Load libff.so (building it in-tree with nvcc if it is missing or stale).  Raises if that fails."""
    global _lib
    if _lib is None:
        so = _build.build(checked=os.environ.get("FF_CHECKED", "0") == "1")
        L = ctypes.CDLL(so)
        vp, i64, i32, f32, f64, u64 = (ctypes.c_void_p, ctypes.c_int64, ctypes.c_int, ctypes.c_float,
                                       ctypes.c_double, ctypes.c_uint64)
        L.ff_workspace_bytes.restype = ctypes.c_size_t
        L.ff_workspace_bytes.argtypes = [i64]
        L.ff_create.restype = i32
        L.ff_create.argtypes = [ctypes.POINTER(vp), i64, f32, vp, ctypes.c_size_t]
        L.ff_destroy.restype = i32
        L.ff_destroy.argtypes = [vp]
        L.ff_set_stream.restype = i32
        L.ff_set_stream.argtypes = [vp, vp]
        L.ff_set_option.restype = i32
        L.ff_set_option.argtypes = [vp, i32, f64]
        L.ff_build_tree.restype = i32
        L.ff_build_tree.argtypes = [vp, vp, i64]
        L.ff_eval_bh.restype = i32
        L.ff_eval_bh.argtypes = [vp, vp, vp, vp, vp]
        L.ff_eval_direct.restype = i32
        L.ff_eval_direct.argtypes = [vp, vp, vp, i64, vp, vp]
        L.ff_eval_bh_range.restype = i32
        L.ff_eval_bh_range.argtypes = [vp, vp, vp, vp, vp, i64, i64]
        L.ff_eval_bh_host.restype = i32
        L.ff_eval_bh_host.argtypes = [vp, vp, vp, i64, vp, vp]
        L.ff_eval_bh_host_async.restype = i32
        L.ff_eval_bh_host_async.argtypes = [vp, vp, vp, i64, vp, vp]
        L.ff_host_sync.restype = i32
        L.ff_host_sync.argtypes = [vp]
        L.ff_eval_direct_host.restype = i32
        L.ff_eval_direct_host.argtypes = [vp, vp, vp, i64, vp, vp]
        L.ff_step.restype = i32
        L.ff_step.argtypes = [vp, vp, vp, vp, vp, i64, ctypes.POINTER(ff_step_params), u64]
        L.ff_get_tree.restype = i32
        L.ff_get_tree.argtypes = [vp, ctypes.POINTER(ff_tree_view)]
        L.ff_get_timings.restype = i32
        L.ff_get_timings.argtypes = [vp, ctypes.POINTER(f32 * FF_N_PHASES)]
        L.ff_get_counters.restype = i32
        L.ff_get_counters.argtypes = [vp, ctypes.POINTER(u64), ctypes.POINTER(u64), ctypes.POINTER(u64)]
        L.ff_get_prefilter_count.restype = i32
        L.ff_get_prefilter_count.argtypes = [vp, ctypes.POINTER(u64)]
        L.ff_get_launch_count.restype = i32
        L.ff_get_launch_count.argtypes = [vp, ctypes.POINTER(u64)]
        L.ff_measure_fp32_peak.restype = i32
        L.ff_measure_fp32_peak.argtypes = [vp, i32, ctypes.POINTER(f64)]
        L.ff_measure_probe.restype = i32
        L.ff_measure_probe.argtypes = [vp, i32, i32, ctypes.POINTER(f64)]
        L.ff_error_string.restype = ctypes.c_char_p
        L.ff_error_string.argtypes = [i32]
        L.ff_last_error.restype = ctypes.c_char_p
        L.ff_last_error.argtypes = [vp]
        L.ff_eval_direct_static.restype = i32
        L.ff_eval_direct_static.argtypes = [vp, vp, i64, vp, vp, vp]
        L.ff_static_last_error.restype = ctypes.c_char_p
        L.ff_static_last_error.argtypes = []
        _lib = L
    return _lib


def ff_workspace_bytes(N: int) -> int:
    return int(lib().ff_workspace_bytes(int(N)))


def _dev_f32(t, n=None, name="tensor"):
    import torch
    if not (isinstance(t, torch.Tensor) and t.is_cuda and t.dtype == torch.float32 and t.is_contiguous()
            and t.dim() == 2 and t.shape[1] == 3):
        raise ValueError("%s must be a contiguous CUDA float32 tensor of shape (n, 3)" % name)
    if n is not None and t.shape[0] != n:
        raise ValueError("%s has %d rows, expected %d" % (name, t.shape[0], n))
    return t.data_ptr()


def eval_direct_static(pos, mom, H, F, stream=None):
    """ff_eval_direct_static: exact all-pairs field and force for n <= FF_STATIC_MAX_N particles without a context,
    a workspace or any device allocation -- the partial sums live in an array built into libff.so.  Meant for code
    that may not call cudaMalloc where it runs (a memory pool owns the whole GPU, a latency-critical loop, a plug-in
    that only gets fixed buffers).  The caller passes the outputs too (H or F may be None to skip one); nothing is
    allocated here either.  `stream`: a raw cudaStream_t, default torch's current stream of pos.device.  Calls that
    can overlap on the GPU share the array and race; see include/ff.h."""
    import torch
    if not torch.cuda.is_available():
        raise RuntimeError("paper_1212_2934_b200 needs a CUDA device: there is no CPU fallback")
    n = pos.shape[0]
    p, m = _dev_f32(pos, n, "pos"), _dev_f32(mom, n, "mom")
    hp = _dev_f32(H, n, "H") if H is not None else None
    fp = _dev_f32(F, n, "F") if F is not None else None
    L = lib()
    with torch.cuda.device(pos.device):
        if stream is None:
            stream = torch.cuda.current_stream(pos.device).cuda_stream
        rc = L.ff_eval_direct_static(p, m, n, hp, fp, ctypes.c_void_p(stream))
    if rc != FF_OK:
        raise FFError(rc, "ff_eval_direct_static", L.ff_static_last_error().decode())
    return H, F


class FFContext:
    """One ff_ctx plus the workspace tensor it lives in (torch owns the device memory)."""

    def __init__(self, N: int, theta: float = 0.5, device="cuda:0", nleaf: int = 1, timing: bool = False,
                 counters: bool = False):
        import torch
        if not torch.cuda.is_available():
            raise RuntimeError("paper_1212_2934_b200 needs a CUDA device: there is no CPU fallback")
        self._L = lib()
        self.N = int(N)
        self.device = torch.device(device)
        nbytes = ff_workspace_bytes(self.N)
        if nbytes == 0:
            raise FFError(FF_ERR_INVALID_ARG, "ff_workspace_bytes")
        with torch.cuda.device(self.device):
            self.workspace = torch.empty(nbytes, dtype=torch.uint8, device=self.device)
            h = ctypes.c_void_p()
            self._check(self._L.ff_create(ctypes.byref(h), self.N, float(theta), self.workspace.data_ptr(), nbytes),
                        "ff_create")
        self._h = h
        self.theta = float(theta)
        self.n = 0
        self.set_stream(torch.cuda.current_stream(self.device).cuda_stream)
        if nleaf != 1:
            self.set_option(FF_OPT_NLEAF, nleaf)
        if timing:
            self.set_option(FF_OPT_TIMING, 1)
        if counters:
            self.set_option(FF_OPT_COUNTERS, 1)

    # -- plumbing ---------------------------------------------------------------
    def _check(self, rc, where):
        if rc != FF_OK:
            detail = ""
            if rc in (FF_ERR_CUDA, FF_ERR_CHECK) and getattr(self, "_h", None):
                detail = self._L.ff_last_error(self._h).decode()
            raise FFError(rc, where, detail)

    def close(self):
        if getattr(self, "_h", None):
            self._L.ff_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def set_stream(self, cuda_stream: int):
        self._check(self._L.ff_set_stream(self._h, ctypes.c_void_p(cuda_stream)), "ff_set_stream")

    def set_option(self, key: int, value: float):
        self._check(self._L.ff_set_option(self._h, int(key), float(value)), "ff_set_option")
        if key == FF_OPT_THETA:
            self.theta = float(value)

    # -- the hot path -------------------------------------------------------------
    def build_tree(self, pos):
        n = pos.shape[0]
        self._check(self._L.ff_build_tree(self._h, _dev_f32(pos, name="pos"), n), "ff_build_tree")
        self.n = n

    def eval_bh(self, pos, mom, H=None, F=None, want_H=True, want_F=True):
        import torch
        n = self.n
        p, m = _dev_f32(pos, n, "pos"), _dev_f32(mom, n, "mom")
        if H is None and want_H:
            H = torch.empty_like(pos)
        if F is None and want_F:
            F = torch.empty_like(pos)
        hp = _dev_f32(H, n, "H") if H is not None else None
        fp = _dev_f32(F, n, "F") if F is not None else None
        self._check(self._L.ff_eval_bh(self._h, p, m, hp, fp), "ff_eval_bh")
        return H, F

    def eval_bh_range(self, pos, mom, H, F, group_begin: int, group_end: int = -1):
        """ff_eval_bh_range: only the walk groups [group_begin, group_end) of the sorted order; only their rows of
        H and F (caller order) are written."""
        n = self.n
        self._check(self._L.ff_eval_bh_range(self._h, _dev_f32(pos, n, "pos"), _dev_f32(mom, n, "mom"),
                                             _dev_f32(H, n, "H") if H is not None else None,
                                             _dev_f32(F, n, "F") if F is not None else None,
                                             int(group_begin), int(group_end)), "ff_eval_bh_range")
        return H, F

    def eval_direct(self, pos, mom, H=None, F=None):
        import torch
        n = pos.shape[0]
        p, m = _dev_f32(pos, n, "pos"), _dev_f32(mom, n, "mom")
        H = torch.empty_like(pos) if H is None else H
        F = torch.empty_like(pos) if F is None else F
        self._check(self._L.ff_eval_direct(self._h, p, m, n, _dev_f32(H, n, "H"), _dev_f32(F, n, "F")),
                    "ff_eval_direct")
        return H, F

    def _host(self, fn, name, pos, mom, H, F):
        import numpy as np
        import torch
        def ptr(x):
            if isinstance(x, torch.Tensor):
                assert not x.is_cuda and x.dtype == torch.float32 and x.is_contiguous()
                return x.data_ptr()
            assert isinstance(x, np.ndarray) and x.dtype == np.float32 and x.flags.c_contiguous
            return x.ctypes.data
        n = pos.shape[0]
        self._check(fn(self._h, ptr(pos), ptr(mom), n, ptr(H), ptr(F)), name)
        self.n = n
        return H, F

    def eval_bh_host(self, pos, mom, H, F):
        """End to end with HOST buffers (numpy or CPU torch, ideally pinned): H2D, build, eval, D2H."""
        return self._host(self._L.ff_eval_bh_host, "ff_eval_bh_host", pos, mom, H, F)

    def eval_bh_host_async(self, pos, mom, H, F):
        """eval_bh_host without the final synchronise: successive calls overlap their copies with each other's
        compute.  Use pinned buffers, keep them alive and untouched until host_sync()."""
        return self._host(self._L.ff_eval_bh_host_async, "ff_eval_bh_host_async", pos, mom, H, F)

    def host_sync(self):
        self._check(self._L.ff_host_sync(self._h), "ff_host_sync")

    def eval_direct_host(self, pos, mom, H, F):
        return self._host(self._L.ff_eval_direct_host, "ff_eval_direct_host", pos, mom, H, F)

    def step(self, pos, vel, mom, angvel, params: ff_step_params, step_index: int):
        n = pos.shape[0]
        self._check(self._L.ff_step(self._h, _dev_f32(pos, n, "pos"), _dev_f32(vel, n, "vel"), _dev_f32(mom, n, "mom"),
                                    _dev_f32(angvel, n, "angvel"), n, ctypes.byref(params), int(step_index)), "ff_step")
        self.n = n

    # -- introspection ---------------------------------------------------------------
    def get_tree(self) -> dict:
        """Copy of the device tree (numpy arrays) in the layout of ff_tree_view."""
        import numpy as np
        import torch
        v = ff_tree_view()
        self._check(self._L.ff_get_tree(self._h, ctypes.byref(v)), "ff_get_tree")
        base = self.workspace.data_ptr()

        def arr(ptr, count, dtype):
            nbytes = count * torch.empty((), dtype=dtype).element_size()
            off = ptr - base
            return self.workspace[off:off + nbytes].view(dtype).cpu().numpy()

        n, m = int(v.n), int(v.n_cells)
        extra = {}
        if v.cell_quad:
            extra["cell_quad"] = arr(v.cell_quad, 8 * m, torch.float32).reshape(m, 8)
        return dict(
            **extra,
            n=n, n_cells=m, nleaf=int(v.nleaf), lo=np.array(list(v.lo), np.float32), S=np.float32(v.S),
            key=arr(v.key, n, torch.int32).view(np.uint32), perm=arr(v.perm, n, torch.int32).view(np.uint32),
            pos_sorted=arr(v.pos_sorted, 4 * n, torch.float32).reshape(n, 4),
            mom_sorted=arr(v.mom_sorted, 4 * n, torch.float32).reshape(n, 4),
            cell_first=arr(v.cell_first, m, torch.int32), cell_end=arr(v.cell_end, m, torch.int32),
            cell_level=arr(v.cell_level, m, torch.int32), child=arr(v.child, 8 * m, torch.int32).reshape(m, 8),
            leaf_count=arr(v.leaf_count, n, torch.int32),
            cell_centre=arr(v.cell_centre, 4 * m, torch.float32).reshape(m, 4),
            cell_moment=arr(v.cell_moment, 4 * m, torch.float32).reshape(m, 4),
        )

    def timings(self) -> dict:
        ms = (ctypes.c_float * FF_N_PHASES)()
        self._check(self._L.ff_get_timings(self._h, ctypes.byref(ms)), "ff_get_timings")
        return {PHASES[i]: float(ms[i]) for i in range(FF_N_PHASES)}

    def counters(self):
        a, b, c = ctypes.c_uint64(), ctypes.c_uint64(), ctypes.c_uint64()
        self._check(self._L.ff_get_counters(self._h, ctypes.byref(a), ctypes.byref(b), ctypes.byref(c)),
                    "ff_get_counters")
        return int(a.value), int(b.value), int(c.value)

    def prefilter_count(self) -> int:
        a = ctypes.c_uint64()
        self._check(self._L.ff_get_prefilter_count(self._h, ctypes.byref(a)), "ff_get_prefilter_count")
        return int(a.value)

    def launch_count(self) -> int:
        a = ctypes.c_uint64()
        self._check(self._L.ff_get_launch_count(self._h, ctypes.byref(a)), "ff_get_launch_count")
        return int(a.value)

    def measure_fp32_peak(self, iters: int = 4096) -> float:
        t = ctypes.c_double()
        self._check(self._L.ff_measure_fp32_peak(self._h, int(iters), ctypes.byref(t)), "ff_measure_fp32_peak")
        return float(t.value)

    def measure_probe(self, kind: int, iters: int = 4096) -> float:
        """ff_measure_probe: TFLOP/s of one of the FP32-pipe probes (FF_PROBE_*)."""
        t = ctypes.c_double()
        self._check(self._L.ff_measure_probe(self._h, int(kind), int(iters), ctypes.byref(t)), "ff_measure_probe")
        return float(t.value)
