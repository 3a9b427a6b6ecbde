"""ctypes front-end of the CPU oracle (oracle/z4c_oracle.cpp). TEST INFRASTRUCTURE, NOT PRODUCT.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this. It takes a parameter object with the attribute names of
paper_2409_10383_b200.inputs.Z4cParams (duck-typed; nothing of the CUDA path is imported).
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIB_PATH = os.path.join(_HERE, "liboz4c.so")
NF = 22


class _OParams(C.Structure):
    _fields_ = [("N", C.c_int32 * 3), ("bc", C.c_int32), ("dx", C.c_double), ("cfl", C.c_double),
                ("kappa1", C.c_double), ("kappa2", C.c_double),
                ("lapse_oplog", C.c_double), ("lapse_harmonic", C.c_double), ("lapse_advect", C.c_double),
                ("shift_gamma", C.c_double), ("shift_eta", C.c_double), ("shift_advect", C.c_double),
                ("ko_eps", C.c_double), ("chi_floor", C.c_double), ("ng", C.c_int32)]


def build(force: bool = False) -> str:
    """Compile liboz4c.so with the system g++ (-O2 -ffp-contract=off -fopenmp)."""
    srcs = [os.path.join(_HERE, f) for f in ("z4c_oracle.cpp", "z4c_physics.hpp", "z4c_oracle.hpp", "z4c_amr.hpp")]
    if (not force and os.path.exists(_LIB_PATH)
            and all(os.path.getmtime(_LIB_PATH) >= os.path.getmtime(s) for s in srcs)):
        return _LIB_PATH
    cxx = "/usr/bin/g++" if os.path.exists("/usr/bin/g++") else "g++"
    cmd = [cxx, "-std=c++17", "-O2", "-ffp-contract=off", "-fPIC", "-fopenmp", "-shared",
           "-o", _LIB_PATH, srcs[0]]
    subprocess.run(cmd, check=True, cwd=_HERE)
    return _LIB_PATH


_lib = None


def lib():
    global _lib
    if _lib is None:
        build()
        L = C.CDLL(_LIB_PATH)
        dp = C.POINTER(C.c_double)
        pp = C.POINTER(_OParams)
        L.oz4c_rhs.argtypes = [pp, dp, dp]
        L.oz4c_enforce.argtypes = [pp, dp]
        L.oz4c_enforce.restype = C.c_int
        L.oz4c_step.argtypes = [pp, dp, C.c_int, C.c_int]
        L.oz4c_step.restype = C.c_int
        L.oz4c_step_textbook.argtypes = [pp, dp, C.c_int]
        L.oz4c_inv_cbrt.argtypes = [C.c_double]
        L.oz4c_inv_cbrt.restype = C.c_double
        L.oz4c_constraints.argtypes = [pp, dp, dp, dp]
        L.oz4c_stencil.argtypes = [pp, dp, C.c_int, C.c_int, C.c_int, dp]
        L.oz4c_num_intermediates.restype = C.c_int
        L.oz4c_intermediates.argtypes = [pp, dp, dp]
        L.oz4c_count_flops.argtypes = [pp, dp, C.c_int, C.c_int, C.c_int, C.POINTER(C.c_longlong)]
        L.oz4c_refine_indicators.argtypes = [pp, dp, C.c_int, dp, dp]
        L.oz4c_num_threads.restype = C.c_int
        ip = C.POINTER(C.c_int32)
        L.oz4c_lagrange_weights.argtypes = [C.c_int, dp, C.c_double, dp]
        L.oz4c_restrict_weights.argtypes = [C.c_int, C.c_int, C.c_int, dp]
        L.oz4c_restrict_weights.restype = C.c_int
        L.oz4c_prolong_weights.argtypes = [C.c_int, C.c_int, dp]
        L.oz4c_prolong_weights.restype = C.c_int
        L.oz4c_restrict.argtypes = [C.c_int, C.c_int, ip, dp, dp, C.c_int]
        L.oz4c_prolong.argtypes = [C.c_int, ip, C.c_int, ip, dp, ip, ip, dp, C.c_int]
        L.oz4c_step_two_level.argtypes = [pp, pp, C.c_int, ip, dp, dp, C.c_int]
        L.oz4c_step_two_level.restype = C.c_int
        L.oz4c_set_num_threads.argtypes = [C.c_int]
        _lib = L
    return _lib


def _op(p, N=None) -> _OParams:
    o = _OParams()
    NN = p.N if N is None else N
    for a in range(3):
        o.N[a] = int(NN[a])
    o.bc = int(p.bc)
    o.ng = int(getattr(p, "ng", 3))      # 3 -> 4th-order stencils, 4 -> 6th-order (NEXT-1)
    for name in ("dx", "cfl", "kappa1", "kappa2", "lapse_oplog", "lapse_harmonic", "lapse_advect",
                 "shift_gamma", "shift_eta", "shift_advect", "ko_eps", "chi_floor"):
        setattr(o, name, float(getattr(p, name)))
    return o


def _ptr(a: np.ndarray):
    assert a.dtype == np.float64 and a.flags["C_CONTIGUOUS"]
    return a.ctypes.data_as(C.POINTER(C.c_double))


def _N_of(u):
    return (u.shape[-1], u.shape[-2], u.shape[-3])


def num_threads() -> int:
    return lib().oz4c_num_threads()


def set_num_threads(n: int) -> None:
    lib().oz4c_set_num_threads(int(n))


def rhs(p, u: np.ndarray) -> np.ndarray:
    u = np.ascontiguousarray(u, dtype=np.float64)
    out = np.empty_like(u)
    lib().oz4c_rhs(C.byref(_op(p, _N_of(u))), _ptr(u), _ptr(out))
    return out


def enforce(p, u: np.ndarray):
    u = np.array(u, dtype=np.float64, order="C", copy=True)
    bad = lib().oz4c_enforce(C.byref(_op(p, _N_of(u))), _ptr(u))
    return u, bad


def step(p, u: np.ndarray, nsteps: int, do_enforce: bool = True):
    u = np.array(u, dtype=np.float64, order="C", copy=True)
    bad = lib().oz4c_step(C.byref(_op(p, _N_of(u))), _ptr(u), int(nsteps), int(do_enforce))
    return u, bad


def step_textbook(p, u: np.ndarray, nsteps: int) -> np.ndarray:
    u = np.array(u, dtype=np.float64, order="C", copy=True)
    lib().oz4c_step_textbook(C.byref(_op(p, _N_of(u))), _ptr(u), int(nsteps))
    return u


def inv_cbrt(x: float) -> float:
    return lib().oz4c_inv_cbrt(float(x))


def constraints(p, u: np.ndarray, percell: bool = False):
    u = np.ascontiguousarray(u, dtype=np.float64)
    out = np.zeros(8)
    pc = np.empty((4,) + u.shape[1:]) if percell else None
    lib().oz4c_constraints(C.byref(_op(p, _N_of(u))), _ptr(u), _ptr(out),
                           _ptr(pc) if percell else None)
    return (out, pc) if percell else out


def stencil(p, f: np.ndarray, kind: int, a: int = 0, b: int = 0) -> np.ndarray:
    f = np.ascontiguousarray(f, dtype=np.float64)
    out = np.empty_like(f)
    lib().oz4c_stencil(C.byref(_op(p, _N_of(f))), _ptr(f), kind, a, b, _ptr(out))
    return out


INTERMEDIATE = {"Rt": slice(0, 6), "Rchi": slice(6, 12), "DDalpha": slice(12, 18), "R": 18, "AA": 19,
                "Gd": slice(20, 23), "ginv": slice(23, 29)}


def intermediates(p, u: np.ndarray) -> np.ndarray:
    u = np.ascontiguousarray(u, dtype=np.float64)
    nq = lib().oz4c_num_intermediates()
    out = np.empty((nq,) + u.shape[1:])
    lib().oz4c_intermediates(C.byref(_op(p, _N_of(u))), _ptr(u), _ptr(out))
    return out


def refine_indicators(p, u: np.ndarray, n: int):
    """NEXT-4: per-block (min chi, max |grad chi|), blocks of n^3 cells in lattice order."""
    u = np.ascontiguousarray(u, dtype=np.float64)
    N = _N_of(u)
    nb = (N[0] // n) * (N[1] // n) * (N[2] // n)
    mn, mx = np.empty(nb), np.empty(nb)
    lib().oz4c_refine_indicators(C.byref(_op(p, N)), _ptr(u), int(n), _ptr(mn), _ptr(mx))
    return mn, mx


def count_flops(p, u: np.ndarray, i: int, j: int, k: int):
    u = np.ascontiguousarray(u, dtype=np.float64)
    cnt = (C.c_longlong * 6)()
    lib().oz4c_count_flops(C.byref(_op(p, _N_of(u))), _ptr(u), i, j, k, cnt)
    return {"rhs": {"add": cnt[0], "mul": cnt[1], "div": cnt[2]},
            "constraints": {"add": cnt[3], "mul": cnt[4], "div": cnt[5]}}


# ---- NEXT-3: restriction / prolongation at a factor-2 refinement boundary ----------------
def _i3(v):
    return (C.c_int32 * 3)(int(v[0]), int(v[1]), int(v[2]))


def lagrange_weights(xs, x: float) -> np.ndarray:
    """Eq. (1)."""
    xs = np.ascontiguousarray(xs, dtype=np.float64)
    w = np.empty_like(xs)
    lib().oz4c_lagrange_weights(len(xs), _ptr(xs), float(x), _ptr(w))
    return w


def restrict_weights(Il: int, ng: int, nf: int):
    """(first fine node, weights) of the restriction stencil of local coarse node Il in a fine block of nf cells."""
    w = np.empty(ng + 1)
    s = lib().oz4c_restrict_weights(int(Il), int(ng), int(nf), _ptr(w))
    return s, w


def prolong_weights(i: int, ng: int):
    """(first coarse node, weights) of the prolongation stencil of fine node i (relative to the region corner)."""
    w = np.empty(ng + 1)
    s = lib().oz4c_prolong_weights(int(i), int(ng), _ptr(w))
    return s, w


def restrict(fine: np.ndarray, ng: int, nf: int) -> np.ndarray:
    """fine [F][Nz][Ny][Nx] (active cells of the fine region, blocks of nf^3) -> coarse [F][Nz/2][Ny/2][Nx/2]."""
    fine = np.ascontiguousarray(fine, dtype=np.float64)
    F, Nz, Ny, Nx = fine.shape
    out = np.empty((F, Nz // 2, Ny // 2, Nx // 2))
    lib().oz4c_restrict(int(ng), int(nf), _i3((Nx, Ny, Nz)), _ptr(fine), _ptr(out), F)
    return out


def prolong(coarse: np.ndarray, ng: int, bc: int, origin, lo, hi) -> np.ndarray:
    """coarse [F][Ncz][Ncy][Ncx] -> values on the fine index box [lo, hi) (x, y, z; relative to the corner of the
    fine region, which is the coarse cell `origin`), returned as [F][hz-lz][hy-ly][hx-lx]."""
    coarse = np.ascontiguousarray(coarse, dtype=np.float64)
    F, Nz, Ny, Nx = coarse.shape
    out = np.empty((F, hi[2] - lo[2], hi[1] - lo[1], hi[0] - lo[0]))
    lib().oz4c_prolong(int(ng), _i3((Nx, Ny, Nz)), int(bc), _i3(origin), _ptr(coarse), _i3(lo), _i3(hi), _ptr(out), F)
    return out


def step_two_level(pc, pf, nf: int, origin, uc: np.ndarray, uf: np.ndarray, nsteps: int):
    """Two-level RK4 steps (coarse level everywhere, fine box at coarse cell `origin`); returns (uc, uf, bad)."""
    uc = np.array(uc, dtype=np.float64, order="C", copy=True)
    uf = np.array(uf, dtype=np.float64, order="C", copy=True)
    bad = lib().oz4c_step_two_level(C.byref(_op(pc, _N_of(uc))), C.byref(_op(pf, _N_of(uf))), int(nf), _i3(origin),
                                    _ptr(uc), _ptr(uf), int(nsteps))
    return uc, uf, bad
