"""Test-side helpers written independently of oracle/ and of the CUDA path.

Everything here is a restatement, in numpy / exact rational arithmetic, of a
definition in PAPER.md or of a reading in DESIGN.md; it is what the oracle is
pinned against.
"""
from __future__ import annotations

from fractions import Fraction

import numpy as np


# ---- exact fp32 helpers ----------------------------------------------------
def round_f32(x: Fraction) -> np.float32:
    """Round an exact rational to the nearest fp32 (ties to even), no double rounding."""
    if x == 0:
        return np.float32(0.0)
    c = np.float32(float(x))
    cands = {c, np.nextafter(c, np.float32(np.inf)), np.nextafter(c, np.float32(-np.inf))}
    best = None
    for v in cands:
        if not np.isfinite(v):
            continue
        err = abs(Fraction(float(v)) - x)
        even = (int(np.float32(v).view(np.uint32)) & 1) == 0
        key = (err, 0 if even else 1)
        if best is None or key < best[0]:
            best = (key, v)
    return np.float32(best[1])


def fmaf_exact(a, b, c) -> np.float32:
    return round_f32(Fraction(float(a)) * Fraction(float(b)) + Fraction(float(c)))


def member_accepts(p, c, s2, th2) -> bool:
    """fp32 opening test in the exact operation order of DESIGN.md (reading O5)."""
    f = np.float32
    dx, dy, dz = f(p[0]) - f(c[0]), f(p[1]) - f(c[1]), f(p[2]) - f(c[2])
    d2 = fmaf_exact(dz, dz, fmaf_exact(dy, dy, f(dx * dx)))
    return bool(f(s2) < f(f(th2) * d2))


# ---- pair terms, vectorised, written from Eq. 11 / Eq. 12 -------------------
def pair_terms(rk, uk, rj, uj):
    """h_kj (Eq. 11) and f_kj (Eq. 12); broadcasting numpy fp64."""
    rho = np.asarray(rk, float) - np.asarray(rj, float)
    uk = np.asarray(uk, float)
    uj = np.asarray(uj, float)
    r = np.sqrt((rho * rho).sum(-1, keepdims=True))
    a = (uj * rho).sum(-1, keepdims=True)
    b = (uk * rho).sum(-1, keepdims=True)
    c = (uj * uk).sum(-1, keepdims=True)
    h = (3 * rho * a - uj * r**2) / r**5
    f = 3 * (rho * c + uk * a + uj * b) / r**5 - 15 * rho * a * b / r**7
    return h, f


def allpairs_numpy(pos, mom):
    pos = np.asarray(pos, np.float64)
    mom = np.asarray(mom, np.float64)
    N = len(pos)
    H = np.zeros((N, 3))
    F = np.zeros((N, 3))
    for k in range(N):
        m = np.arange(N) != k
        h, f = pair_terms(pos[k], mom[k], pos[m], mom[m])
        H[k] = h.sum(0)
        F[k] = f.sum(0)
    return H, F


# ---- first-order cell term, contracted closed form -------------
def first_order_terms(rk, uk, rc, D):
    """First-order terms (dh, df) of a cell at rc with tensor D = sum_i (rho_i - rc) (x) u_i acting on a target at rk
    with moment uk, from the CONTRACTED form of the Taylor expansion of Eq. 11-12 about the cell centre
    (with R = rk - rc, Ds = (D + D^T) / 2, t = tr D, b = uk.R, q = R.Ds.R):
        dh = -{ 3 [2 Ds R + t R] / R^5 - 15 R q / R^7 }
        df = -{ 3 [2 Ds uk + t uk] / R^5 - 15 [R (2 uk.Ds.R + t b) + uk q + 2 b Ds R] / R^7 + 105 R b q / R^9 }
    Written independently of the oracle, which loops over the components of the rank-3 / rank-4 derivative tensors."""
    R = np.asarray(rk, float) - np.asarray(rc, float)
    u = np.asarray(uk, float)
    D = np.asarray(D, float).reshape(3, 3)
    Ds = 0.5 * (D + D.T)
    t = np.trace(D)
    r = np.sqrt(R @ R)
    DR, Du = Ds @ R, Ds @ u
    q, b, uDR = R @ DR, u @ R, u @ DR
    dh = -(3 * (2 * DR + t * R) / r**5 - 15 * R * q / r**7)
    df = -(3 * (2 * Du + t * u) / r**5 - 15 * (R * (2 * uDR + t * b) + u * q + 2 * b * DR) / r**7 + 105 * R * b * q / r**9)
    return dh, df


# ---- tree by brute-force prefix grouping (reading O3) -----------------------
def morton_keys_numpy(pos):
    """30-bit keys, fp32 arithmetic in the order inv=fl(1024/S); q=floor(fl(fl(p-lo)*inv))."""
    pos = np.asarray(pos, np.float32)
    lo = pos.min(0)
    hi = pos.max(0)
    S = np.float32((hi - lo).astype(np.float32).max())
    if not S > 0:
        S = np.float32(1.0)
    inv = np.float32(np.float32(1024.0) / S)
    d = (pos - lo).astype(np.float32)
    g = (d * inv).astype(np.float32)
    q = np.minimum(np.floor(g).astype(np.int64), 1023)
    key = np.zeros(len(pos), np.int64)
    for b in range(10):
        key |= ((q[:, 0] >> b) & 1) << (3 * b + 2)
        key |= ((q[:, 1] >> b) & 1) << (3 * b + 1)
        key |= ((q[:, 2] >> b) & 1) << (3 * b)
    return key.astype(np.uint32), lo, S


def brute_tree(pos, nleaf=1):
    """Canonical node list [(first, level, prefix, count, is_leaf)] by grouping sorted keys by prefix."""
    key, lo, S = morton_keys_numpy(pos)
    perm = np.argsort(key, kind="stable")
    sk = key[perm].astype(np.int64)
    N = len(sk)
    nodes = []
    internal = {(0, 0)} if N > nleaf else set()
    nodes.append((0, 0, 0, N, 0 if N > nleaf else 1))
    for level in range(1, 11):
        shift = 3 * (10 - level)
        pref = sk >> shift
        vals, first, count = np.unique(pref, return_index=True, return_counts=True)
        new_internal = set()
        for v, f0, c in zip(vals, first, count):
            if (level - 1, int(v) >> 3) not in internal:
                continue
            leaf = not (c > nleaf and level < 10)
            nodes.append((int(f0), level, int(v), int(c), 1 if leaf else 0))
            if not leaf:
                new_internal.add((level, int(v)))
        internal |= new_internal
    nodes.sort(key=lambda t: (t[0], t[1]))
    return nodes, sk.astype(np.uint32), perm, lo, S


def canonical_from_oracle(tree):
    nd = tree.nodes()
    return [(int(a), int(b), int(c), int(d), int(e)) for a, b, c, d, e in
            zip(nd["first"], nd["level"], nd["prefix"], nd["count"], nd["is_leaf"])]


# ---- an independently written list builder (python, exact fp32 emulation) ---
def build_lists(pos, mom, theta, W, nleaf):
    """Per group: (accepted cells as (level, prefix), leaf particles as sorted slots), using only
    brute-force prefix grouping and the plain statement of the rule."""
    nodes, sk, perm, lo, S = brute_tree(pos, nleaf)
    sp = np.asarray(pos, np.float32)[perm]
    sm = np.asarray(mom, np.float32)[perm]
    N = len(sp)
    info = {}
    for (f, l, p, c, leaf) in nodes:
        cen = (np.sum(sp[f:f + c].astype(np.float64), axis=0) / c).astype(np.float32)
        mu = np.sum(sm[f:f + c].astype(np.float64), axis=0).astype(np.float32)
        info[(l, p)] = (f, c, leaf, cen, mu)
    th2 = np.float32(np.float32(theta) * np.float32(theta))
    out = []
    for g0 in range(0, N, W):
        g1 = min(N, g0 + W)
        cells, parts = [], []
        stack = [(0, 0)]
        while stack:
            l, p = stack.pop()
            f, c, leaf, cen, mu = info[(l, p)]
            if leaf:
                parts.extend(range(f, f + c))
                continue
            holds_member = f < g1 and f + c > g0
            if not holds_member:
                s = np.float32(S) * np.float32(2.0 ** -l)
                s2 = np.float32(s * s)
                if all(member_accepts(sp[k], cen, s2, th2) for k in range(g0, g1)):
                    cells.append((l, p))
                    continue
            for o in range(7, -1, -1):
                if (l + 1, p << 3 | o) in info:
                    stack.append((l + 1, p << 3 | o))
        out.append((g0, g1, cells, parts))
    return out, info, sp, sm, perm


def eval_lists(lists, info, sp, sm, perm, scale=False):
    N = len(sp)
    H = np.zeros((N, 3))
    F = np.zeros((N, 3))
    Q = np.zeros((N, 2))
    for g0, g1, cells, parts in lists:
        for k in range(g0, g1):
            h = np.zeros(3)
            f = np.zeros(3)
            q = np.zeros(2)
            for key in cells:
                _, _, _, cen, mu = info[key]
                dh, df = pair_terms(sp[k], sm[k], cen, mu)
                h += dh
                f += df
                q += (dh @ dh, df @ df)
            for j in parts:
                if j == k:
                    continue
                dh, df = pair_terms(sp[k], sm[k], sp[j], sm[j])
                h += dh
                f += df
                q += (dh @ dh, df @ df)
            H[perm[k]] = h
            F[perm[k]] = f
            Q[perm[k]] = np.sqrt(q)      # root-sum-square of the terms of particle k's own sum
    return (H, F, Q) if scale else (H, F)


# ---- canonical form of the GPU tree (ff_tree_view) ----------------------------
_FF_CHILD_EMPTY = -1
_FF_CHILD_MULTI, _FF_CHILD_SLOT = 0x40000000, 0x3FFFFFFF


def canonical_tree(tree: dict):
    """Canonical topology [(first, level, prefix, count, is_leaf)] sorted by (first, level) from the dict of
    FFContext.get_tree() (layout of ff_tree_view, include/ff.h): the internal cells plus the leaf children they point
    to.  A test-side canonicaliser (reading Q7 of DESIGN.md: the GPU may number cells as it likes)."""
    key = tree["key"].astype("int64")
    n, m = tree["n"], tree["n_cells"]
    out = []
    if m == 0:
        return [(0, 0, 0, n, 1)]
    first, end, level, child = tree["cell_first"], tree["cell_end"], tree["cell_level"], tree["child"]
    for i in range(m):
        f, l = int(first[i]), int(level[i])
        out.append((f, l, int(key[f] >> (3 * (10 - l))), int(end[i]) - f, 0))
        for o in range(8):
            e = int(child[i, o])
            if e == _FF_CHILD_EMPTY or e >= 0:
                continue
            u = e & 0xFFFFFFFF
            slot = u & _FF_CHILD_SLOT
            cnt = int(tree["leaf_count"][slot]) if (u & _FF_CHILD_MULTI) else 1
            out.append((slot, l + 1, int(key[slot] >> (3 * (10 - l - 1))), cnt, 1))
    out.sort(key=lambda t: (t[0], t[1]))
    return out


# ---- error metric of DESIGN.md ("error metric", reading Q19) ------------------
KAPPA = 8.0


def rel_err(x, ref, Q=None):
    """Per-particle relative L2 error e_k = |x_k - ref_k| / max(|ref_k|, floor_k).

    floor_k = Q_k / KAPPA with Q_k = sqrt(sum_j |t_kj|^2), the root-sum-square of the terms of
    particle k's own sum (from the oracle): a sum whose terms cancel below 1/KAPPA of their
    natural scale is measured against that scale, because fp32 rounding error is proportional to
    the size of the TERMS, not of their sum.  Without Q: floor = 1e-3 * rms_k |ref|.
    Returns (max, median, p99, global relative L2)."""
    x = np.asarray(x, np.float64)
    ref = np.asarray(ref, np.float64)
    nr = np.linalg.norm(ref, axis=1)
    if Q is None:
        floor = 1e-3 * np.sqrt((nr**2).mean())
    else:
        floor = np.asarray(Q, np.float64) / KAPPA
    e = np.linalg.norm(x - ref, axis=1) / np.maximum(np.maximum(nr, floor), 1e-300)
    glob = np.linalg.norm(x - ref) / max(np.linalg.norm(ref), 1e-300)
    return float(e.max()), float(np.median(e)), float(np.percentile(e, 99)), float(glob)


def check_hf(H, F, Ho, Fo, Q, tol, survey=True):
    """Assert both fields within tol; returns the error tuples.

    Two gates.  (1) the term-scale metric e_k = |dx_k| / max(|ref_k|, Q_k / KAPPA), always.
    (2) survey=True: ALSO the survey's metric (floor 1e-3 rms |ref|, no Q), so that wherever the sums
    do not cancel the result does not depend on the oracle's Q at all.  survey=False is reserved for the inputs whose
    sums cancel by construction (head-to-tail chains: config 4 and the chain cases of the sweep), named in DESIGN.md."""
    eh, ef = rel_err(H, Ho, Q[:, 0]), rel_err(F, Fo, Q[:, 1])
    assert eh[0] <= tol and ef[0] <= tol, ("term-scale metric", eh, ef)
    if survey == "tail":
        # Unsampled runs over ~10^6 rows (third gate): the survey metric of every row is <= tol
        # except for at most 1e-5 of the rows; those are <= 2 tol and are rows whose own sum cancels below 1/KAPPA of
        # its term scale (where the survey's floor is too low by arithmetic, the reason gate (1) exists).
        for x, ref, q in ((H, Ho, Q[:, 0]), (F, Fo, Q[:, 1])):
            x, ref = np.asarray(x, np.float64), np.asarray(ref, np.float64)
            nr = np.linalg.norm(ref, axis=1)
            e = np.linalg.norm(x - ref, axis=1) / np.maximum(np.maximum(nr, 1e-3 * np.sqrt((nr**2).mean())), 1e-300)
            over = e > tol
            assert over.sum() <= max(1, int(1e-5 * len(e))), ("survey metric: rows beyond tol", int(over.sum()), float(e.max()))
            assert e.max() <= 2 * tol, ("survey metric: tail", float(e.max()))
            assert (nr[over] < np.asarray(q, np.float64)[over] / KAPPA).all(), "a non-cancelling row beyond tol"
    elif survey:
        sh, sf = rel_err(H, Ho), rel_err(F, Fo)
        assert sh[0] <= tol and sf[0] <= tol, ("survey metric (no Q)", sh, sf)
    return eh, ef


# ---- crafted inputs that sit ON the opening test's threshold (reading O5 / Q1) ----------------------------
def opening_case(t, seed=0):
    """35 particles around ONE decision: does group 0 (W = 32) accept the level-2 cell of the pair a, b?

    Root cube [0, 8]^3 (a target at the origin, a particle at (8, 8, 8)), so s_2 = 2 and fl(s_2^2) = 4.  The pair
    a = (4.5, 0.5, 1), b = (5.5, 1.5, 1) is alone in the level-2 cell [4,6) x [0,2) x [0,2); its centre (Eq. 14) is
    exactly (5, 1, 1) in fp64 and in fp32.  Group 0 = the 32 particles of octant 0: 30 fillers in [0.05, 0.9]^3 and
    the origin, all at d^2 >= 16.8 from the centre (they accept at theta = 0.5, where the rule reads 4 < d2 / 4),
    and the critical target t, which alone decides.  Returns (pos, mom, slot_a, slot_b): caller-order fp32 arrays
    and the caller indices of a and b."""
    rng = np.random.default_rng(seed)
    fill = rng.uniform(0.05, 0.9, (30, 3)).astype(np.float32)
    pos = np.concatenate([fill, np.zeros((1, 3), np.float32), np.asarray(t, np.float32).reshape(1, 3),
                          np.array([[4.5, 0.5, 1.0], [5.5, 1.5, 1.0], [8.0, 8.0, 8.0]], np.float32)])
    u = rng.normal(size=(len(pos), 3))
    mom = (u / np.linalg.norm(u, axis=1, keepdims=True)).astype(np.float32)
    return pos, mom, 32, 33


OPENING_CENTRE = np.array([5.0, 1.0, 1.0], np.float32)


def opening_d2(t, fused=True):
    """d2 of target t against OPENING_CENTRE in fp32: the order of reading O5 (fused: fma(dz,dz, fma(dy,dy, fl(dx dx))))
    or the plausible mistake (three rounded squares added left to right)."""
    f = np.float32
    dx, dy, dz = (f(t[0]) - OPENING_CENTRE[0], f(t[1]) - OPENING_CENTRE[1], f(t[2]) - OPENING_CENTRE[2])
    xx = f(dx * dx)
    if fused:
        return fmaf_exact(dz, dz, fmaf_exact(dy, dy, xx))
    return f(f(xx + f(dy * dy)) + f(dz * dz))


def fma_sensitive_targets(seed=1212, tries=4000):
    """Seeded search for two critical targets on which the fused and the unfused d2 fall on different sides of the
    threshold d2 > 16 (theta = 0.5, s_2 = 2): one the fused order accepts and the unfused opens, one the other way
    round.  Returns {True: t, False: t} keyed by the FUSED decision."""
    rng = np.random.default_rng(seed)
    found = {}
    f = np.float32
    for _ in range(tries):
        ty, tz = f(rng.uniform(0.3, 1.7)), f(rng.uniform(0.3, 1.7))
        dy, dz = float(ty) - 1.0, float(tz) - 1.0
        tx = f(5.0 - np.sqrt(16.0 - dy * dy - dz * dz))
        for _ in range(6):
            tx = np.nextafter(tx, f(-np.inf))
        for _ in range(13):
            t = np.array([tx, ty, tz], f)
            a, b = bool(opening_d2(t, True) > f(16.0)), bool(opening_d2(t, False) > f(16.0))
            if a != b and a not in found:
                found[a] = t
            tx = np.nextafter(tx, f(np.inf))
        if len(found) == 2:
            return found
    raise AssertionError("no fma-sensitive target found")
