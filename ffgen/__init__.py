"""ffgen -- seeded synthetic dipole ensembles shared by the CUDA path and the oracle.

Input generators only: this package holds none of the method's arithmetic (no
field, force, key or tree code).  The recipes follow BASELINE.json `configs`
and SURVEY.md 8(d); they stand in for the paper's self-generated random
ensembles.  Length unit: sphere diameter d = 1.

    cfg = ffgen.config(1)          # dict: pos (N,3) f32, mom (N,3) f32, theta, L, ...
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "ffgen.c")
_SO = os.path.join(_HERE, "libffgen.so")
_lib = None


def build(force: bool = False) -> str:
    """Compile ffgen.c into libffgen.so (gcc, in-tree)."""
    if force or not os.path.exists(_SO) or os.path.getmtime(_SO) < os.path.getmtime(_SRC):
        tmp = _SO + ".tmp.%d" % os.getpid()
        subprocess.check_call(["gcc", "-O2", "-std=c11", "-shared", "-fPIC", "-o", tmp, _SRC, "-lm"])
        os.replace(tmp, _SO)
    return _SO


def _load():
    global _lib
    if _lib is None:
        lib = ctypes.CDLL(build())
        i64, u64, dbl, fp = ctypes.c_int64, ctypes.c_uint64, ctypes.c_double, ctypes.c_void_p
        lib.ffgen_box_side.restype = dbl
        lib.ffgen_box_side.argtypes = [i64, dbl]
        lib.ffgen_hard_spheres.restype = i64
        lib.ffgen_hard_spheres.argtypes = [i64, dbl, u64, fp]
        lib.ffgen_moments_isotropic.restype = None
        lib.ffgen_moments_isotropic.argtypes = [i64, u64, fp]
        lib.ffgen_moments_vmf.restype = None
        lib.ffgen_moments_vmf.argtypes = [i64, dbl, u64, fp]
        lib.ffgen_chains.restype = i64
        lib.ffgen_chains.argtypes = [i64, ctypes.c_int, dbl, dbl, u64, fp, fp]
        lib.ffgen_uniform_points.restype = None
        lib.ffgen_uniform_points.argtypes = [i64, dbl, u64, fp]
        _lib = lib
    return _lib


def box_side(N: int, phi: float) -> float:
    """L = (N pi d^3 / (6 phi))^(1/3), Eq. 16 with d = 1."""
    return float(_load().ffgen_box_side(int(N), float(phi)))


def hard_spheres(N: int, L: float, seed: int = 0) -> np.ndarray:
    pos = np.empty((N, 3), dtype=np.float32)
    rc = _load().ffgen_hard_spheres(int(N), float(L), int(seed), pos.ctypes.data)
    if rc < 0:
        raise RuntimeError("ffgen_hard_spheres failed (%d)" % rc)
    return pos


def moments_isotropic(N: int, seed: int = 0) -> np.ndarray:
    mom = np.empty((N, 3), dtype=np.float32)
    _load().ffgen_moments_isotropic(int(N), int(seed), mom.ctypes.data)
    return mom


def moments_vmf(N: int, kappa: float, seed: int = 0) -> np.ndarray:
    mom = np.empty((N, 3), dtype=np.float32)
    _load().ffgen_moments_vmf(int(N), float(kappa), int(seed), mom.ctypes.data)
    return mom


def chains(n_chains: int, length: int, L: float, cap_deg: float = 15.0, seed: int = 0):
    N = n_chains * length
    pos = np.empty((N, 3), dtype=np.float32)
    mom = np.empty((N, 3), dtype=np.float32)
    rc = _load().ffgen_chains(int(n_chains), int(length), float(L), float(cap_deg), int(seed),
                              pos.ctypes.data, mom.ctypes.data)
    if rc < 0:
        raise RuntimeError("ffgen_chains failed (%d)" % rc)
    return pos, mom


def uniform_points(N: int, L: float, seed: int = 0) -> np.ndarray:
    pos = np.empty((N, 3), dtype=np.float32)
    _load().ffgen_uniform_points(int(N), float(L), int(seed), pos.ctypes.data)
    return pos


# BASELINE.json `configs`, 1-based as in SURVEY.md 8(d).
CONFIGS = {
    1: dict(N=4096, phi=0.05, moments="isotropic", theta=0.5, kind="uniform"),
    2: dict(N=65536, phi=0.1, moments="vmf", kappa=5.0, theta=0.5, thetas=(0.3, 0.5, 0.7), kind="uniform"),
    3: dict(N=1048576, phi=0.1, moments="isotropic", theta=0.5, kind="uniform"),
    4: dict(N=1048576, phi=0.1, moments="axis", theta=0.5, kind="chains", n_chains=32768, chain_len=32),
    5: dict(N=16777216, phi=0.2, moments="isotropic", theta=0.6, kind="uniform"),
}


def ensemble(N: int, phi: float, moments: str = "isotropic", kappa: float = 5.0, seed: int = 0):
    """Uniform hard-sphere ensemble at volume fraction phi (any N)."""
    L = box_side(N, phi)
    pos = hard_spheres(N, L, seed)
    if moments == "isotropic":
        mom = moments_isotropic(N, seed)
    elif moments == "vmf":
        mom = moments_vmf(N, kappa, seed)
    else:
        raise ValueError(moments)
    return pos, mom, L


def config(idx: int, seed: int = 0, N: int | None = None) -> dict:
    """Config `idx` (1..5) of BASELINE.json; `N` overrides the size (same recipe, same phi)."""
    c = dict(CONFIGS[idx])
    if N is not None:
        if c["kind"] == "chains":
            c["n_chains"] = max(1, N // c["chain_len"])
            N = c["n_chains"] * c["chain_len"]
        c["N"] = int(N)
    c["seed"] = seed
    if c["kind"] == "uniform":
        pos, mom, L = ensemble(c["N"], c["phi"], c["moments"], c.get("kappa", 5.0), seed)
    else:
        # the chain config states no volume fraction: config 3's density
        L = box_side(c["N"], c["phi"])
        pos, mom = chains(c["n_chains"], c["chain_len"], L, 15.0, seed)
    c.update(pos=pos, mom=mom, L=L, config=idx)
    return c
