"""oracle -- ctypes front end of oracle/ff_oracle.c (fp64 CPU all-pairs and Barnes-Hut).

TEST INFRASTRUCTURE ONLY.  Importers allowed: tests/, __graft_entry__.smoke(),
bench.py's cpu_baseline and `--impl reference` legs.  The CUDA package
(paper_1212_2934_b200) never imports this module and this module never imports
it; there is no CPU fallback in the product.

Every function is a thin marshalling layer; the arithmetic and its citations
(Eq. 11, 12, 14) live in ff_oracle.c.
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "ff_oracle.c")
_SO = os.path.join(_HERE, "libff_oracle.so")
_lib = None

CFLAGS = ["-O2", "-std=c11", "-ffp-contract=off", "-fno-fast-math", "-fopenmp", "-shared", "-fPIC"]


def build(force: bool = False) -> str:
    """Compile ff_oracle.c into libff_oracle.so (gcc, in-tree)."""
    if force or not os.path.exists(_SO) or os.path.getmtime(_SO) < os.path.getmtime(_SRC):
        tmp = _SO + ".tmp.%d" % os.getpid()
        subprocess.check_call(["gcc", *CFLAGS, "-o", tmp, _SRC, "-lm"])
        os.replace(tmp, _SO)
    return _SO


def _load():
    global _lib
    if _lib is None:
        lib = ctypes.CDLL(build())
        vp, i64, i32, f32 = ctypes.c_void_p, ctypes.c_int64, ctypes.c_int, ctypes.c_float
        lib.ffo_pair.restype = None
        lib.ffo_pair.argtypes = [vp] * 6
        lib.ffo_max_threads.restype = i32
        lib.ffo_allpairs.restype = i32
        lib.ffo_allpairs.argtypes = [i64, vp, vp, i64, vp, vp, vp, vp, i32]
        lib.ffo_tree_build.restype = vp
        lib.ffo_tree_build.argtypes = [i64, vp, i32]
        lib.ffo_tree_free.restype = None
        lib.ffo_tree_free.argtypes = [vp]
        lib.ffo_tree_num_nodes.restype = i64
        lib.ffo_tree_num_nodes.argtypes = [vp]
        lib.ffo_tree_bbox.restype = None
        lib.ffo_tree_bbox.argtypes = [vp, vp, vp]
        lib.ffo_tree_keys.restype = None
        lib.ffo_tree_keys.argtypes = [vp, vp, vp]
        lib.ffo_tree_nodes.restype = None
        lib.ffo_tree_nodes.argtypes = [vp] * 7
        lib.ffo_tree_moments.restype = i32
        lib.ffo_tree_moments.argtypes = [vp, vp]
        lib.ffo_tree_node_moments.restype = None
        lib.ffo_tree_node_moments.argtypes = [vp] * 5
        lib.ffo_bh_eval.restype = i32
        lib.ffo_bh_eval.argtypes = [vp, f32, i32, i64, vp, vp, vp, vp, vp, i32]
        lib.ffo_bh_eval_order.restype = i32
        lib.ffo_bh_eval_order.argtypes = [vp, f32, i32, i32, i64, vp, vp, vp, vp, vp, i32]
        lib.ffo_first_order.restype = None
        lib.ffo_first_order.argtypes = [vp] * 6
        lib.ffo_tree_node_dsym.restype = None
        lib.ffo_tree_node_dsym.argtypes = [vp, vp]
        lib.ffo_bh_group_lists.restype = i32
        lib.ffo_bh_group_lists.argtypes = [vp, f32, i32, i64, vp, i64, vp, vp, i64, vp]
        _lib = lib
    return _lib


def max_threads() -> int:
    return int(_load().ffo_max_threads())


def _f32(a, shape_last=3):
    a = np.ascontiguousarray(a, dtype=np.float32)
    assert a.ndim == 2 and a.shape[1] == shape_last
    return a


def pair(rk, uk, rj, uj):
    """(h_kj, f_kj) of Eq. 11 / Eq. 12 for one ordered pair, fp64."""
    args = [np.ascontiguousarray(x, dtype=np.float64) for x in (rk, uk, rj, uj)]
    h = np.zeros(3)
    f = np.zeros(3)
    _load().ffo_pair(*[a.ctypes.data for a in args], h.ctypes.data, f.ctypes.data)
    return h, f


def first_order(rk, uk, rc, D):
    """(dh, df): the first-order terms of a cell at rc with tensor D = sum_i (rho_i - rc) (x) u_i (3x3) acting on a
    target at rk with moment uk (derivation in ff_oracle.c, O1b), fp64."""
    args = [np.ascontiguousarray(x, dtype=np.float64) for x in (rk, uk, rc, np.asarray(D, np.float64).reshape(9))]
    h = np.zeros(3)
    f = np.zeros(3)
    _load().ffo_first_order(*[a.ctypes.data for a in args], h.ctypes.data, f.ctypes.data)
    return h, f


def allpairs(pos, mom, targets=None, nthreads: int = 0, scale: bool = False):
    """All-pairs H, F (fp64).  targets: optional int64 index array -> rows follow it.
    scale=True also returns Q (nt, 2): sqrt(sum_j |h_kj|^2), sqrt(sum_j |f_kj|^2), the error-metric scale."""
    pos, mom = _f32(pos), _f32(mom)
    N = pos.shape[0]
    if targets is None:
        nt, tp = N, None
    else:
        targets = np.ascontiguousarray(targets, dtype=np.int64)
        nt, tp = targets.shape[0], targets.ctypes.data
    H = np.zeros((nt, 3))
    F = np.zeros((nt, 3))
    Q = np.zeros((nt, 2)) if scale else None
    rc = _load().ffo_allpairs(N, pos.ctypes.data, mom.ctypes.data, nt, tp, H.ctypes.data, F.ctypes.data,
                              Q.ctypes.data if scale else None, nthreads)
    if rc != 0:
        raise RuntimeError("ffo_allpairs failed")
    return (H, F, Q) if scale else (H, F)


class Tree:
    """Octree of SURVEY.md 8(c) O3 built by recursive subdivision."""

    def __init__(self, pos, nleaf: int = 1):
        self.pos = _f32(pos)
        self.N = self.pos.shape[0]
        self.nleaf = nleaf
        self._lib = _load()
        self._t = self._lib.ffo_tree_build(self.N, self.pos.ctypes.data, nleaf)
        if not self._t:
            raise RuntimeError("ffo_tree_build failed")
        self.n_nodes = int(self._lib.ffo_tree_num_nodes(self._t))
        self._mom = None

    def __del__(self):
        if getattr(self, "_t", None):
            self._lib.ffo_tree_free(self._t)
            self._t = None

    def bbox(self):
        lo = np.zeros(3, dtype=np.float32)
        S = np.zeros(1, dtype=np.float32)
        self._lib.ffo_tree_bbox(self._t, lo.ctypes.data, S.ctypes.data)
        return lo, np.float32(S[0])

    def keys(self):
        key = np.zeros(self.N, dtype=np.uint32)
        perm = np.zeros(self.N, dtype=np.int64)
        self._lib.ffo_tree_keys(self._t, key.ctypes.data, perm.ctypes.data)
        return key, perm

    def nodes(self):
        n = self.n_nodes
        out = dict(first=np.zeros(n, np.int64), count=np.zeros(n, np.int64), level=np.zeros(n, np.int32),
                   prefix=np.zeros(n, np.uint32), is_leaf=np.zeros(n, np.int32), child=np.zeros((n, 8), np.int64))
        self._lib.ffo_tree_nodes(self._t, *[out[k].ctypes.data for k in
                                            ("first", "count", "level", "prefix", "is_leaf", "child")])
        return out

    def moments(self, mom):
        self._mom = _f32(mom)
        if self._lib.ffo_tree_moments(self._t, self._mom.ctypes.data) != 0:
            raise RuntimeError("ffo_tree_moments failed")
        n = self.n_nodes
        out = dict(sum_u=np.zeros((n, 3)), sum_p=np.zeros((n, 3)),
                   mu=np.zeros((n, 3), np.float32), cen=np.zeros((n, 3), np.float32))
        self._lib.ffo_tree_node_moments(self._t, *[out[k].ctypes.data for k in ("sum_u", "sum_p", "mu", "cen")])
        out["dsym"] = np.zeros((n, 6), np.float32)          # first-order cell tensor, xx yy zz xy xz yz (8(f4))
        self._lib.ffo_tree_node_dsym(self._t, out["dsym"].ctypes.data)
        return out

    def eval(self, theta: float, W: int = 32, groups=None, nthreads: int = 0, scale: bool = False, order: int = 0):
        """Barnes-Hut H, F (fp64, caller order, (N,3)); rows outside `groups` are NaN.
        Returns (H, F, counters) with counters = (cell terms, particle terms, opening tests);
        scale=True appends Q (N, 2), the per-target root-sum-square of the term magnitudes.
        order=1 adds the first-order term of every accepted cell; 0 is the paper's cell."""
        assert self._mom is not None, "call moments(mom) first"
        H = np.full((self.N, 3), np.nan)
        F = np.full((self.N, 3), np.nan)
        cnt = np.zeros(3, dtype=np.uint64)
        if groups is None:
            ng, gp = 0, None
        else:
            groups = np.ascontiguousarray(groups, dtype=np.int64)
            ng, gp = groups.shape[0], groups.ctypes.data
        Q = np.full((self.N, 2), np.nan) if scale else None
        rc = self._lib.ffo_bh_eval_order(self._t, float(theta), int(W), int(order), ng, gp, H.ctypes.data, F.ctypes.data,
                                         Q.ctypes.data if scale else None, cnt.ctypes.data, nthreads)
        if rc != 0:
            raise RuntimeError("ffo_bh_eval failed")
        cnt = tuple(int(c) for c in cnt)
        return (H, F, cnt, Q) if scale else (H, F, cnt)

    def group_lists(self, theta: float, W: int, g: int):
        """(accepted node indices, sorted slots reached through leaves) of group g."""
        assert self._mom is not None, "call moments(mom) first"
        nc = np.zeros(1, np.int64)
        npart = np.zeros(1, np.int64)
        cells = np.zeros(self.n_nodes, np.int64)
        parts = np.zeros(self.N, np.int64)
        rc = self._lib.ffo_bh_group_lists(self._t, float(theta), int(W), int(g), cells.ctypes.data, cells.size,
                                          nc.ctypes.data, parts.ctypes.data, parts.size, npart.ctypes.data)
        if rc != 0:
            raise RuntimeError("ffo_bh_group_lists failed")
        return cells[: nc[0]].copy(), parts[: npart[0]].copy()


def barnes_hut(pos, mom, theta: float, W: int = 32, nleaf: int = 1, groups=None, nthreads: int = 0,
               scale: bool = False, order: int = 0):
    """Convenience: build, moments, evaluate.  Returns (H, F, counters, tree) [+ (Q,) if scale]."""
    t = Tree(pos, nleaf)
    t.moments(mom)
    out = t.eval(theta, W, groups, nthreads, scale, order)
    return (out[0], out[1], out[2], t) + ((out[3],) if scale else ())
