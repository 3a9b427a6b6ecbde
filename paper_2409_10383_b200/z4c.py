"""Thin Python binding of the C-ABI library (include/z4c.h): same names, argument marshalling only.

PyTorch is used for device memory and streams and for nothing else: every step of the hot path runs in
the CUDA kernels of `libz4c.so`. There is no CPU fallback: if the library is missing or no CUDA device is
present, the calls raise.
"""
from __future__ import annotations

import ctypes as C
import os
from typing import Optional

import numpy as np

NF = 22
Z4C_OK, Z4C_EINVAL, Z4C_ECUDA, Z4C_ESTATE = 0, -1, -2, -3
_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libz4c.so")            # built with 3 ghost zones (4th-order stencils)
LIB_PATH_NG4 = os.path.join(_HERE, "libz4c_ng4.so")    # built with 4 ghost zones (6th-order stencils)

# every symbol include/z4c.h declares
SYMBOLS = ["z4c_state_bytes", "z4c_workspace_bytes", "z4c_create", "z4c_set_initial_data", "z4c_step",
           "z4c_constraints", "z4c_constraints_static", "z4c_refine_indicators", "z4c_get_interior", "z4c_fill_ghosts", "z4c_eval_rhs", "z4c_enforce", "z4c_sync",
           "z4c_launch_count", "z4c_set_variant", "z4c_use_graph", "z4c_set_fused", "z4c_step_timed",
           "z4c_probe_fp64", "z4c_effective_mode", "z4c_time",
           "z4c_restrict", "z4c_prolongate", "z4c_two_level_step",
           "z4c_enable_peer", "z4c_set_partition", "z4c_set_neighbor", "z4c_state2", "z4c_stage", "z4c_stage_rhs", "z4c_stage_update",
           "z4c_constraints_raw",
           "z4c_last_error", "z4c_destroy"]


class z4c_params(C.Structure):
    """Mirror of `z4c_params` (include/z4c.h)."""
    _fields_ = [("n", C.c_int32), ("ng", C.c_int32), ("nb", C.c_int32 * 3), ("bc", C.c_int32),
                ("xmin", C.c_double * 3), ("dx", C.c_double), ("cfl", C.c_double),
                ("kappa1", C.c_double), ("kappa2", C.c_double),
                ("lapse_oplog", C.c_double), ("lapse_harmonic", C.c_double), ("lapse_advect", C.c_double),
                ("shift_gamma", C.c_double), ("shift_eta", C.c_double), ("shift_advect", C.c_double),
                ("ko_eps", C.c_double), ("chi_floor", C.c_double)]


def make_params(p) -> z4c_params:
    """From any object with the attribute names of `inputs.Z4cParams`."""
    o = z4c_params()
    o.n, o.ng, o.bc = int(p.n), int(p.ng), int(p.bc)
    for a in range(3):
        o.nb[a] = int(p.nb[a])
        o.xmin[a] = float(p.xmin[a])
    for name in ("dx", "cfl", "kappa1", "kappa2", "lapse_oplog", "lapse_harmonic", "lapse_advect",
                 "shift_gamma", "shift_eta", "shift_advect", "ko_eps", "chi_floor"):
        setattr(o, name, float(getattr(p, name)))
    return o


_libs = {}


def load_library(path: Optional[str] = None, ng: int = 3):
    """dlopen the library built for `ng` ghost zones and declare the prototypes. Raises if it is not built."""
    if path is None and ng in _libs:
        return _libs[ng]
    if path is None and ng not in (3, 4):
        raise ValueError("the library is built for ng = 3 (4th order) and ng = 4 (6th order)")
    default = LIB_PATH if ng == 3 else LIB_PATH_NG4
    path = path or default
    if not os.path.exists(path):
        raise RuntimeError(f"{path} is missing: build it with `python -m paper_2409_10383_b200.build` "
                           "(there is no CPU fallback)")
    L = C.CDLL(path)
    pp, vp, dp = C.POINTER(z4c_params), C.c_void_p, C.c_void_p
    L.z4c_state_bytes.argtypes = [pp]
    L.z4c_state_bytes.restype = C.c_size_t
    L.z4c_workspace_bytes.argtypes = [pp]
    L.z4c_workspace_bytes.restype = C.c_size_t
    L.z4c_create.argtypes = [pp, vp, vp, vp, C.POINTER(vp)]
    L.z4c_set_initial_data.argtypes = [vp, dp, C.c_int]
    L.z4c_step.argtypes = [vp, C.c_int]
    L.z4c_constraints.argtypes = [vp, C.POINTER(C.c_double), dp]
    L.z4c_constraints_static.argtypes = [vp, dp]
    L.z4c_refine_indicators.argtypes = [vp, C.c_double, C.c_double, dp, dp, dp]
    L.z4c_get_interior.argtypes = [vp, dp, C.c_int]
    L.z4c_fill_ghosts.argtypes = [vp]
    L.z4c_eval_rhs.argtypes = [vp, dp]
    L.z4c_enforce.argtypes = [vp]
    L.z4c_sync.argtypes = [vp]
    L.z4c_launch_count.argtypes = [vp]
    L.z4c_launch_count.restype = C.c_int64
    L.z4c_set_variant.argtypes = [vp, C.c_int]
    L.z4c_use_graph.argtypes = [vp, C.c_int]
    L.z4c_set_fused.argtypes = [vp, C.c_int]
    L.z4c_step_timed.argtypes = [vp, C.c_int, C.POINTER(C.c_double)]
    L.z4c_probe_fp64.argtypes = [vp, vp, C.c_int, C.POINTER(C.c_double)]
    L.z4c_effective_mode.argtypes = [vp, C.POINTER(C.c_int), C.POINTER(C.c_int)]
    i3 = C.POINTER(C.c_int32)
    L.z4c_restrict.argtypes = [vp, vp, i3]
    L.z4c_prolongate.argtypes = [vp, vp, i3]
    L.z4c_two_level_step.argtypes = [vp, vp, i3, C.c_int]
    L.z4c_set_partition.argtypes = [vp, C.c_int32, C.c_int32]
    L.z4c_set_neighbor.argtypes = [vp, C.c_int32, vp, vp, C.c_int32, C.c_int32]
    L.z4c_state2.argtypes = [vp]
    L.z4c_state2.restype = C.c_void_p
    L.z4c_stage.argtypes = [vp, C.c_int]
    L.z4c_stage_rhs.argtypes = [vp, C.c_int]
    L.z4c_stage_update.argtypes = [vp, C.c_int]
    L.z4c_constraints_raw.argtypes = [vp, C.POINTER(C.c_double)]
    L.z4c_enable_peer.argtypes = [C.c_int32]
    L.z4c_time.argtypes = [vp]
    L.z4c_time.restype = C.c_double
    L.z4c_last_error.argtypes = [vp]
    L.z4c_last_error.restype = C.c_char_p
    L.z4c_destroy.argtypes = [vp]
    L.z4c_destroy.restype = None
    for fn in ("z4c_create", "z4c_set_initial_data", "z4c_step", "z4c_constraints", "z4c_refine_indicators", "z4c_get_interior",
               "z4c_fill_ghosts", "z4c_eval_rhs", "z4c_enforce", "z4c_sync", "z4c_set_variant", "z4c_use_graph",
               "z4c_set_fused", "z4c_step_timed", "z4c_probe_fp64", "z4c_effective_mode", "z4c_restrict", "z4c_prolongate",
               "z4c_two_level_step", "z4c_set_partition", "z4c_set_neighbor", "z4c_stage", "z4c_stage_rhs", "z4c_stage_update",
               "z4c_constraints_raw"):
        getattr(L, fn).restype = C.c_int
    if path == default:
        _libs[ng] = L
    return L


class Z4cError(RuntimeError):
    def __init__(self, code: int, msg: str):
        super().__init__(f"z4c error {code}: {msg}")
        self.code = code


class Z4c:
    """Owns the device buffers (torch tensors) and a library context; methods are 1:1 with the C ABI."""

    def __init__(self, p, device: str = "cuda:0", stream=None):
        import torch
        if not torch.cuda.is_available():
            raise RuntimeError("no CUDA device: the Z4c path has no CPU fallback")
        self.torch = torch
        self.lib = load_library(ng=int(p.ng))
        self.p = p
        self.cp = make_params(p)
        self.device = torch.device(device)
        sb = self.lib.z4c_state_bytes(C.byref(self.cp))
        wb = self.lib.z4c_workspace_bytes(C.byref(self.cp))
        if sb == 0 or wb == 0:
            raise Z4cError(Z4C_EINVAL, "invalid parameters")
        m = p.n + 2 * p.ng
        nblk = p.nb[0] * p.nb[1] * p.nb[2]
        with torch.cuda.device(self.device):
            self.state = torch.empty((NF, nblk, m, m, m), dtype=torch.float64, device=self.device)
            self.work = torch.empty(wb // 8, dtype=torch.float64, device=self.device)
            # a dedicated non-default stream: CUDA-graph capture is not allowed on the legacy default stream
            self.stream = stream if stream is not None else torch.cuda.Stream(self.device)
            torch.cuda.synchronize(self.device)
            assert self.state.numel() * 8 == sb
            h = C.c_void_p()
            rc = self.lib.z4c_create(C.byref(self.cp), self.state.data_ptr(), self.work.data_ptr(),
                                     self.stream.cuda_stream, C.byref(h))
        if rc != 0:
            raise Z4cError(rc, "z4c_create failed")
        self.h = h

    # -- helpers ----------------------------------------------------------------------------
    def _check(self, rc: int):
        if rc != 0:
            raise Z4cError(rc, self.lib.z4c_last_error(self.h).decode())

    def _before(self, *tensors):
        """Order the library's stream after the caller's current stream before a call that reads or writes a
        caller-owned device tensor (stream-ordering contract of include/z4c.h)."""
        cur = self.torch.cuda.current_stream(self.device)
        if cur != self.stream:
            self.stream.wait_stream(cur)
            for t in tensors:
                t.record_stream(self.stream)      # the caching allocator must not reuse it while we still run

    def _after(self):
        """... and the caller's current stream after the library's, so the caller may consume the result."""
        cur = self.torch.cuda.current_stream(self.device)
        if cur != self.stream:
            cur.wait_stream(self.stream)

    @property
    def interior_shape(self):
        N = self.p.N
        return (NF, N[2], N[1], N[0])

    # -- the ABI ----------------------------------------------------------------------------
    def set_initial_data(self, interior):
        """interior: numpy float64 [22][Nz][Ny][Nx] (host) or a CUDA float64 torch tensor of that shape."""
        torch = self.torch
        with torch.cuda.device(self.device):
            if isinstance(interior, np.ndarray):
                a = np.ascontiguousarray(interior, dtype=np.float64)
                assert a.shape == self.interior_shape
                self._check(self.lib.z4c_set_initial_data(self.h, a.ctypes.data, 0))
            else:
                t = interior
                assert t.dtype == torch.float64 and t.is_contiguous() and tuple(t.shape) == self.interior_shape
                if t.is_cuda:
                    self._before(t)
                    self._check(self.lib.z4c_set_initial_data(self.h, t.data_ptr(), 1))
                    self._after()
                else:
                    self._check(self.lib.z4c_set_initial_data(self.h, t.data_ptr(), 0))

    def step(self, nsteps: int = 1):
        with self.torch.cuda.device(self.device):
            self._check(self.lib.z4c_step(self.h, int(nsteps)))

    def constraints(self, percell: bool = False):
        out = (C.c_double * 8)()
        pc = None
        with self.torch.cuda.device(self.device):
            if percell:
                pc = self.torch.empty((4,) + self.interior_shape[1:], dtype=self.torch.float64, device=self.device)
                self._before(pc)
            self._check(self.lib.z4c_constraints(self.h, out, pc.data_ptr() if percell else None))   # synchronises
        res = np.array(list(out))
        return (res, pc.cpu().numpy()) if percell else res

    def constraints_static(self, d_out=None):
        """z4c_constraints_static: the 8 norms into a DEVICE tensor (8 doubles; the caller's, or a new one), computed
        with the library's static scratch: no allocation inside the call, asynchronous on the context's stream."""
        if d_out is None:
            d_out = self.torch.empty(8, dtype=self.torch.float64, device=self.device)
            self._before(d_out)
        with self.torch.cuda.device(self.device):
            self._check(self.lib.z4c_constraints_static(self.h, d_out.data_ptr()))
        return d_out

    def refine_indicators(self, chi_min: float, dchi_max: float):
        """z4c_refine_indicators: (min chi, max |grad chi|, flags) per block as numpy arrays."""
        torch = self.torch
        nblk = self.p.nb[0] * self.p.nb[1] * self.p.nb[2]
        with torch.cuda.device(self.device):
            mn = torch.empty(nblk, dtype=torch.float64, device=self.device)
            mx = torch.empty(nblk, dtype=torch.float64, device=self.device)
            fl = torch.empty(nblk, dtype=torch.int32, device=self.device)
            self._before(mn, mx, fl)
            self._check(self.lib.z4c_refine_indicators(self.h, float(chi_min), float(dchi_max), mn.data_ptr(),
                                                       mx.data_ptr(), fl.data_ptr()))
            self._check(self.lib.z4c_sync(self.h))
        return mn.cpu().numpy(), mx.cpu().numpy(), fl.cpu().numpy()

    def get_interior(self, out=None) -> np.ndarray:
        """Host copy of the interior cells (numpy). If `out` is a CUDA tensor, fills it on the device instead."""
        with self.torch.cuda.device(self.device):
            if out is not None and not isinstance(out, np.ndarray):
                assert out.is_cuda and out.dtype == self.torch.float64 and out.is_contiguous()
                self._before(out)
                self._check(self.lib.z4c_get_interior(self.h, out.data_ptr(), 1))
                self._after()
                return out
            a = out if out is not None else np.empty(self.interior_shape, dtype=np.float64)
            assert a.flags["C_CONTIGUOUS"] and a.dtype == np.float64 and a.shape == self.interior_shape
            self._check(self.lib.z4c_get_interior(self.h, a.ctypes.data, 0))
            return a

    def fill_ghosts(self):
        with self.torch.cuda.device(self.device):
            self._check(self.lib.z4c_fill_ghosts(self.h))

    def eval_rhs(self) -> np.ndarray:
        with self.torch.cuda.device(self.device):
            out = self.torch.empty(self.interior_shape, dtype=self.torch.float64, device=self.device)
            self._before(out)
            self._check(self.lib.z4c_eval_rhs(self.h, out.data_ptr()))
            self._check(self.lib.z4c_sync(self.h))
        return out.cpu().numpy()

    def enforce(self):
        with self.torch.cuda.device(self.device):
            self._check(self.lib.z4c_enforce(self.h))

    def sync(self):
        with self.torch.cuda.device(self.device):
            self._check(self.lib.z4c_sync(self.h))

    def launch_count(self) -> int:
        return int(self.lib.z4c_launch_count(self.h))

    def set_variant(self, v: int):
        self._check(self.lib.z4c_set_variant(self.h, int(v)))

    def effective_mode(self):
        """z4c_effective_mode: (variant, fused) that actually run after fallbacks."""
        v, f = C.c_int(), C.c_int()
        self._check(self.lib.z4c_effective_mode(self.h, C.byref(v), C.byref(f)))
        return int(v.value), int(f.value)

    def use_graph(self, enable: bool):
        self._check(self.lib.z4c_use_graph(self.h, int(bool(enable))))

    def set_fused(self, mode):
        """0: K2, K3, K1 separate; 1 (or True): K2 + K3 with ghost push; 2: one kernel per RK stage (default)."""
        self._check(self.lib.z4c_set_fused(self.h, int(mode)))

    def step_timed(self, nsteps: int = 1):
        """z4c_step_timed: returns {"rhs": ms, "update": ms, "ghost": ms} summed over nsteps."""
        ms = (C.c_double * 3)()
        with self.torch.cuda.device(self.device):
            self._check(self.lib.z4c_step_timed(self.h, int(nsteps), ms))
        return {"rhs": ms[0], "update": ms[1], "ghost": ms[2]}

    def probe_fp64(self, iters: int = 20000) -> float:
        """z4c_probe_fp64: achieved DFMA TFLOP/s on this device."""
        out = C.c_double()
        with self.torch.cuda.device(self.device):
            rc = self.lib.z4c_probe_fp64(self.stream.cuda_stream, self.work.data_ptr(), int(iters), C.byref(out))
        if rc != 0:
            raise Z4cError(rc, "z4c_probe_fp64 failed")
        return float(out.value)

    # -- NEXT-3: two-level static refinement; `self` is the FINE level, `coarse` another Z4c on the same stream --
    def restrict_to(self, coarse: "Z4c", origin):
        """z4c_restrict(fine = self, coarse, origin)."""
        o = (C.c_int32 * 3)(*[int(v) for v in origin])
        with self.torch.cuda.device(self.device):
            self._check(self.lib.z4c_restrict(self.h, coarse.h, o))

    def prolongate_from(self, coarse: "Z4c", origin):
        """z4c_prolongate(coarse, fine = self, origin)."""
        o = (C.c_int32 * 3)(*[int(v) for v in origin])
        with self.torch.cuda.device(self.device):
            self._check(self.lib.z4c_prolongate(coarse.h, self.h, o))

    def two_level_step(self, coarse: "Z4c", origin, nsteps: int = 1):
        """z4c_two_level_step(coarse, fine = self, origin, nsteps)."""
        o = (C.c_int32 * 3)(*[int(v) for v in origin])
        with self.torch.cuda.device(self.device):
            self._check(self.lib.z4c_two_level_step(coarse.h, self.h, o, int(nsteps)))

    # -- NEXT-2: one slab of a partitioned mesh ------------------------------------------------------------
    def enable_peer(self, peer_device: int):
        """z4c_enable_peer with this context's device current: its kernels may then store into `peer_device`'s memory."""
        with self.torch.cuda.device(self.device):
            rc = self.lib.z4c_enable_peer(int(peer_device))
        if rc != 0:
            raise Z4cError(rc, f"z4c_enable_peer({peer_device}) failed: no such device, or no peer path from {self.device}")

    def set_partition(self, nbz_global: int, bz0: int):
        self._check(self.lib.z4c_set_partition(self.h, int(nbz_global), int(bz0)))

    def set_neighbor(self, side: int, d_state: int, d_state2: int, bz0: int, nbz: int):
        """d_state / d_state2: device addresses (ints) of the neighbour's two state buffers, valid in this process."""
        self._check(self.lib.z4c_set_neighbor(self.h, int(side), d_state or None, d_state2 or None, int(bz0), int(nbz)))

    def state2_ptr(self) -> int:
        return int(self.lib.z4c_state2(self.h))

    def stage(self, s: int):
        with self.torch.cuda.device(self.device):
            self._check(self.lib.z4c_stage(self.h, int(s)))

    def stage_rhs(self, s: int):
        with self.torch.cuda.device(self.device):
            self._check(self.lib.z4c_stage_rhs(self.h, int(s)))

    def stage_update(self, s: int):
        with self.torch.cuda.device(self.device):
            self._check(self.lib.z4c_stage_update(self.h, int(s)))

    def constraints_raw(self) -> np.ndarray:
        out = (C.c_double * 8)()
        with self.torch.cuda.device(self.device):
            self._check(self.lib.z4c_constraints_raw(self.h, out))
        return np.array(list(out))

    def time(self) -> float:
        return float(self.lib.z4c_time(self.h))

    def close(self):
        if getattr(self, "h", None) is not None and self.h:
            self.torch.cuda.synchronize(self.device)
            self.lib.z4c_destroy(self.h)
            self.h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass
