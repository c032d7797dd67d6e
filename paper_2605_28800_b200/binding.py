"""ctypes binding of libfe_b200 (include/fe.h).  Argument marshalling only: every step of the hot
path runs in the CUDA kernels of the library.  PyTorch supplies device memory and streams.

There is no CPU fallback: if the shared library is missing or a call fails, an exception is raised.
This module never imports `oracle/`.
"""
from __future__ import annotations

import ctypes
import os
from typing import Optional, Sequence

import numpy as np
import torch

from . import build as _build

FE_OK, FE_EINVAL, FE_ENOMEM, FE_ECUDA, FE_ESTATE, FE_ENONFINITE = range(6)
FE_F64, FE_F32 = 0, 1
FE_TERM_LANDAU, FE_TERM_GRADIENT, FE_TERM_ELEC, FE_TERM_EXT, FE_TERM_ALL = 1, 2, 4, 8, 15
FE_EULER, FE_HEUN, FE_RK4, FE_AB3M2 = 0, 1, 2, 3

SYMBOLS = ["fe_create_grid", "fe_destroy_grid", "fe_workspace_bytes", "fe_bind_workspace", "fe_set_material",
           "fe_set_global", "fe_set_external_field", "fe_set_material_map", "fe_precompute_tensor", "fe_rhs",
           "fe_step", "fe_energy", "fe_get_tensor", "fe_padded_dims", "fe_launch_count", "fe_last_error",
           "fe_version", "fe_profile", "fe_profile_read", "fe_step_rk45", "fe_set_external_wave", "fe_set_time",
           "fe_get_time", "fe_set_option", "fe_get_option", "fe_energy_noalloc"]
KERNEL_KINDS = ["xfwd", "yfwd", "zmul", "yinv", "xinv", "local", "other", "xyfwd", "xyinv"]
FE_OPT_FUSE_XY, FE_OPT_XY_TIMEOUTS, FE_OPT_XY_RING, FE_OPT_XL_SLABS = 0, 1, 2, 3


class fe_rk45_stats(ctypes.Structure):
    _fields_ = [("t", ctypes.c_double), ("dt_last", ctypes.c_double), ("dt_next", ctypes.c_double),
                ("err_last", ctypes.c_double), ("accepted", ctypes.c_int32), ("rejected", ctypes.c_int32),
                ("rhs_evals", ctypes.c_int32)]


class fe_grid_desc(ctypes.Structure):
    _fields_ = [("nx", ctypes.c_int32), ("ny", ctypes.c_int32), ("nz", ctypes.c_int32),
                ("dx", ctypes.c_double), ("dy", ctypes.c_double), ("dz", ctypes.c_double),
                ("periodic", ctypes.c_int32 * 3), ("pbc_images", ctypes.c_int32 * 3),
                ("batch", ctypes.c_int32), ("dtype", ctypes.c_int32), ("n_materials", ctypes.c_int32),
                ("zero_mode", ctypes.c_int32)]


class fe_landau(ctypes.Structure):
    _fields_ = [("a1", ctypes.c_double * 3)] + [(k, ctypes.c_double) for k in
                ("a11", "a12", "a111", "a112", "a123", "a1111", "a1112", "a1122", "a1123")] + \
               [("active", ctypes.c_int32)]


class fe_global(ctypes.Structure):
    _fields_ = [(k, ctypes.c_double) for k in ("G11", "G12", "G44", "G44p", "eps0", "epsB", "L")]


class FeError(RuntimeError):
    def __init__(self, status: int, text: str):
        super().__init__("fe status %d: %s" % (status, text))
        self.status = status


_lib = None


def lib_path() -> str:
    return _build.LIB


def load():
    """Load libfe_b200.so (raises OSError if it has not been built: no fallback)."""
    global _lib
    if _lib is None:
        if not os.path.exists(_build.LIB):
            raise OSError("libfe_b200.so is not built; run `python -m paper_2605_28800_b200.build` "
                          "(the CUDA extension is required, there is no CPU path)")
        L = ctypes.CDLL(_build.LIB)
        vp, i32, u32, dbl = ctypes.c_void_p, ctypes.c_int32, ctypes.c_uint32, ctypes.c_double
        L.fe_create_grid.argtypes = [ctypes.POINTER(fe_grid_desc), ctypes.POINTER(vp)]
        L.fe_destroy_grid.argtypes = [vp]
        L.fe_workspace_bytes.argtypes = [vp]
        L.fe_workspace_bytes.restype = ctypes.c_size_t
        L.fe_bind_workspace.argtypes = [vp, vp, ctypes.c_size_t]
        L.fe_set_material.argtypes = [vp, i32, i32, ctypes.POINTER(fe_landau)]
        L.fe_set_global.argtypes = [vp, i32, ctypes.POINTER(fe_global)]
        L.fe_set_external_field.argtypes = [vp, i32, ctypes.POINTER(dbl)]
        L.fe_set_material_map.argtypes = [vp, vp]
        L.fe_precompute_tensor.argtypes = [vp, vp]
        L.fe_rhs.argtypes = [vp, vp, vp, u32, vp]
        L.fe_step.argtypes = [vp, vp, dbl, i32, i32, u32, vp]
        L.fe_energy.argtypes = [vp, vp, u32, ctypes.POINTER(dbl), vp]
        L.fe_energy_noalloc.argtypes = [vp, vp, u32, vp, vp]
        L.fe_get_tensor.argtypes = [vp, ctypes.POINTER(dbl), vp]
        L.fe_padded_dims.argtypes = [vp, ctypes.POINTER(i32)]
        L.fe_profile.argtypes = [vp, i32]
        L.fe_profile_read.argtypes = [vp, ctypes.POINTER(dbl), ctypes.POINTER(ctypes.c_uint64), vp]
        L.fe_launch_count.argtypes = [vp]
        L.fe_set_external_wave.argtypes = [vp, i32, ctypes.POINTER(dbl), dbl, dbl]
        L.fe_set_time.argtypes = [vp, dbl]
        L.fe_get_time.argtypes = [vp, ctypes.POINTER(dbl)]
        L.fe_step_rk45.argtypes = [vp, vp, dbl, dbl, dbl, i32, u32, ctypes.POINTER(fe_rk45_stats), vp]
        L.fe_set_option.argtypes = [vp, i32, i32]
        L.fe_get_option.argtypes = [vp, i32, ctypes.POINTER(i32)]
        L.fe_launch_count.restype = ctypes.c_uint64
        L.fe_last_error.restype = ctypes.c_char_p
        L.fe_version.restype = ctypes.c_char_p
        for name in ("fe_create_grid", "fe_destroy_grid", "fe_bind_workspace", "fe_set_material", "fe_set_global",
                     "fe_set_external_field", "fe_set_material_map", "fe_precompute_tensor", "fe_rhs", "fe_step",
                     "fe_energy", "fe_get_tensor", "fe_padded_dims", "fe_profile", "fe_profile_read", "fe_set_option",
                     "fe_get_option", "fe_energy_noalloc"):
            getattr(L, name).restype = ctypes.c_int
        _lib = L
    return _lib


def _check(status: int, allow: Sequence[int] = ()):
    if status != FE_OK and status not in allow:
        raise FeError(status, load().fe_last_error().decode())
    return status


def _stream() -> ctypes.c_void_p:
    return ctypes.c_void_p(torch.cuda.current_stream().cuda_stream)


def _landau_struct(m) -> fe_landau:
    c = fe_landau()
    c.a1[0], c.a1[1], c.a1[2] = [float(v) for v in m.a1]
    for k in ("a11", "a12", "a111", "a112", "a123", "a1111", "a1112", "a1122", "a1123"):
        setattr(c, k, float(getattr(m, k)))
    c.active = int(m.active)
    return c


# ---- functions with the names of the C ABI -------------------------------------------------------------
def fe_create_grid(n, d, periodic=(0, 0, 0), pbc_images=(0, 0, 0), batch=1, dtype=FE_F64, n_materials=1,
                   zero_mode=True) -> ctypes.c_void_p:
    desc = fe_grid_desc()
    desc.nx, desc.ny, desc.nz = [int(v) for v in n]
    desc.dx, desc.dy, desc.dz = [float(v) for v in d]
    for a in range(3):
        desc.periodic[a] = int(periodic[a])
        desc.pbc_images[a] = int(pbc_images[a])
    desc.batch, desc.dtype, desc.n_materials, desc.zero_mode = int(batch), int(dtype), int(n_materials), int(bool(zero_mode))
    h = ctypes.c_void_p()
    _check(load().fe_create_grid(ctypes.byref(desc), ctypes.byref(h)))
    return h


def fe_destroy_grid(h):
    _check(load().fe_destroy_grid(h))


def fe_workspace_bytes(h) -> int:
    return int(load().fe_workspace_bytes(h))


def fe_bind_workspace(h, ws: torch.Tensor):
    _check(load().fe_bind_workspace(h, ctypes.c_void_p(ws.data_ptr()), ws.numel() * ws.element_size()))


def fe_set_material(h, member: int, material_id: int, m):
    c = _landau_struct(m)
    _check(load().fe_set_material(h, int(member), int(material_id), ctypes.byref(c)))


def fe_set_global(h, member: int, g):
    c = fe_global(float(g.G11), float(g.G12), float(g.G44), float(g.G44p), float(g.eps0), float(g.epsB), float(g.L))
    _check(load().fe_set_global(h, int(member), ctypes.byref(c)))


def fe_set_external_field(h, member: int, E):
    arr = (ctypes.c_double * 3)(*[float(v) for v in E])
    _check(load().fe_set_external_field(h, int(member), arr))


def fe_set_external_wave(h, member: int, amp, omega: float, phase: float = 0.0):
    a = (ctypes.c_double * 3)(*[float(v) for v in amp])
    _check(load().fe_set_external_wave(h, int(member), a, float(omega), float(phase)))


def fe_set_time(h, t: float):
    _check(load().fe_set_time(h, float(t)))


def fe_get_time(h) -> float:
    t = ctypes.c_double(0.0)
    _check(load().fe_get_time(h, ctypes.byref(t)))
    return t.value


def fe_set_material_map(h, dev_map: Optional[torch.Tensor]):
    _check(load().fe_set_material_map(h, ctypes.c_void_p(dev_map.data_ptr() if dev_map is not None else 0)))


def fe_precompute_tensor(h):
    _check(load().fe_precompute_tensor(h, _stream()))


def fe_rhs(h, P: torch.Tensor, dPdt: torch.Tensor, terms: int = FE_TERM_ALL):
    _check(load().fe_rhs(h, ctypes.c_void_p(P.data_ptr()), ctypes.c_void_p(dPdt.data_ptr()), terms, _stream()))


def fe_step(h, P: torch.Tensor, dt: float, nsteps: int, integrator: int = FE_EULER, terms: int = FE_TERM_ALL):
    _check(load().fe_step(h, ctypes.c_void_p(P.data_ptr()), float(dt), int(nsteps), int(integrator), terms, _stream()))


def fe_step_rk45(h, P: torch.Tensor, t_span: float, dt_init: float, tol: float, max_steps: int = 100000,
                 terms: int = FE_TERM_ALL) -> dict:
    st = fe_rk45_stats()
    _check(load().fe_step_rk45(h, ctypes.c_void_p(P.data_ptr()), float(t_span), float(dt_init), float(tol), int(max_steps),
                               terms, ctypes.byref(st), _stream()))
    return dict(t=st.t, dt_last=st.dt_last, dt_next=st.dt_next, err_last=st.err_last, accepted=st.accepted,
                rejected=st.rejected, rhs_evals=st.rhs_evals)


def fe_energy(h, P: torch.Tensor, batch: int, terms: int = FE_TERM_ALL, allow_nonfinite: bool = False) -> np.ndarray:
    out = np.zeros((batch, 8), dtype=np.float64)
    _check(load().fe_energy(h, ctypes.c_void_p(P.data_ptr()), terms, out.ctypes.data_as(ctypes.POINTER(ctypes.c_double)),
                            _stream()), allow=(FE_ENONFINITE,) if allow_nonfinite else ())
    return out


def fe_energy_noalloc(h, P: torch.Tensor, out: torch.Tensor, terms: int = FE_TERM_ALL) -> torch.Tensor:
    """fe_energy without allocation, host copy or synchronisation: `out` is a DEVICE float64 tensor [B][8] (include/fe.h)."""
    if out.dtype != torch.float64 or not out.is_cuda or not out.is_contiguous() or out.device != P.device:
        raise ValueError("out must be a contiguous float64 CUDA tensor on the state's device")
    _check(load().fe_energy_noalloc(h, ctypes.c_void_p(P.data_ptr()), terms, ctypes.c_void_p(out.data_ptr()), _stream()))
    return out


def fe_padded_dims(h):
    out = (ctypes.c_int32 * 3)()
    _check(load().fe_padded_dims(h, out))
    return tuple(out)


def fe_get_tensor(h) -> np.ndarray:
    mx, my, mz = fe_padded_dims(h)
    out = np.zeros((6, mz, my, mx), dtype=np.float64)
    _check(load().fe_get_tensor(h, out.ctypes.data_as(ctypes.POINTER(ctypes.c_double)), _stream()))
    return out


def fe_profile(h, enable: bool):
    _check(load().fe_profile(h, int(bool(enable))))


def fe_profile_read(h):
    """{kind: (total ms, launches)} since the last read."""
    ms = (ctypes.c_double * len(KERNEL_KINDS))()
    cnt = (ctypes.c_uint64 * len(KERNEL_KINDS))()
    _check(load().fe_profile_read(h, ms, cnt, _stream()))
    return {k: (ms[i], int(cnt[i])) for i, k in enumerate(KERNEL_KINDS)}


def fe_set_option(h, option: int, value: int):
    _check(load().fe_set_option(h, int(option), int(value)))


def fe_get_option(h, option: int) -> int:
    v = ctypes.c_int32(0)
    _check(load().fe_get_option(h, int(option), ctypes.byref(v)))
    return int(v.value)


def fe_launch_count(h) -> int:
    return int(load().fe_launch_count(h))


# ---- convenience wrapper -----------------------------------------------------------------------------------
class Grid:
    """Owns an fe_grid handle plus its torch workspace.  `materials[b][m]` / `globals_[b]` are objects with
    the fields of fe_landau / fe_global (+ E_ext), e.g. fe_inputs.Landau / fe_inputs.Globals."""

    def __init__(self, n, d, periodic=(0, 0, 0), pbc_images=(0, 0, 0), batch=1, dtype="f64", n_materials=1,
                 zero_mode=True, device="cuda:0"):
        if not torch.cuda.is_available():
            raise RuntimeError("paper_2605_28800_b200 needs a CUDA device (no CPU path exists)")
        self.device = torch.device(device)
        torch.cuda.set_device(self.device)
        self.n, self.batch, self.n_materials = tuple(int(v) for v in n), int(batch), int(n_materials)
        self.tdtype = torch.float64 if dtype == "f64" else torch.float32
        self.h = fe_create_grid(n, d, periodic, pbc_images, batch, FE_F64 if dtype == "f64" else FE_F32,
                                n_materials, zero_mode)
        self.ws = torch.empty(fe_workspace_bytes(self.h), dtype=torch.uint8, device=self.device)
        fe_bind_workspace(self.h, self.ws)
        self._map = None

    @classmethod
    def from_workload(cls, w, device="cuda:0", dtype=None) -> "Grid":
        g = cls(w.n, w.d, w.periodic, w.pbc_images, w.batch, dtype or w.dtype, len(w.materials[0]), True, device)
        for b in range(w.batch):
            for m, mat in enumerate(w.materials[b]):
                fe_set_material(g.h, b, m, mat)
            fe_set_global(g.h, b, w.globals_[b])
            fe_set_external_field(g.h, b, w.globals_[b].E_ext)
        if w.matmap is not None:
            g.set_material_map(torch.from_numpy(np.ascontiguousarray(w.matmap)).to(g.device))
        return g

    @property
    def state_shape(self):
        return (self.batch, 3, self.n[2], self.n[1], self.n[0])

    def state(self, P_host: np.ndarray) -> torch.Tensor:
        return torch.from_numpy(np.ascontiguousarray(P_host)).to(self.device, self.tdtype).contiguous()

    def set_material(self, member, material_id, m): fe_set_material(self.h, member, material_id, m)
    def set_global(self, member, g): fe_set_global(self.h, member, g)
    def set_external_field(self, member, E): fe_set_external_field(self.h, member, E)
    def set_external_wave(self, member, amp, omega, phase=0.0): fe_set_external_wave(self.h, member, amp, omega, phase)
    def set_time(self, t): fe_set_time(self.h, t)
    def time(self) -> float: return fe_get_time(self.h)

    def set_material_map(self, dev_map: Optional[torch.Tensor]):
        if dev_map is not None:
            nx, ny, nz = self.n
            if not (dev_map.is_cuda and dev_map.device == self.device and dev_map.dtype == torch.uint8
                    and dev_map.is_contiguous() and tuple(dev_map.shape) == (nz, ny, nx)):
                raise FeError(FE_EINVAL, "material map must be a contiguous uint8 [nz][ny][nx] tensor on %s" % self.device)
            if int(dev_map.max()) >= self.n_materials:
                raise FeError(FE_EINVAL, "material map holds an id >= n_materials = %d" % self.n_materials)
        self._map = dev_map          # keep the borrowed tensor alive
        fe_set_material_map(self.h, dev_map)

    def _state_ok(self, P: torch.Tensor, what: str = "P"):
        """The kernels trust the pointer: refuse anything that is not the ABI's [B][3][nz][ny][nx] array."""
        if not (isinstance(P, torch.Tensor) and P.is_cuda and P.device == self.device and P.dtype == self.tdtype
                and P.is_contiguous() and tuple(P.shape) == self.state_shape):
            raise FeError(FE_EINVAL, "%s must be a contiguous %s tensor of shape %s on %s"
                          % (what, self.tdtype, self.state_shape, self.device))

    def precompute_tensor(self): fe_precompute_tensor(self.h)

    def rhs(self, P: torch.Tensor, terms=FE_TERM_ALL) -> torch.Tensor:
        self._state_ok(P)
        out = torch.empty_like(P)
        fe_rhs(self.h, P, out, terms)
        return out

    def step(self, P: torch.Tensor, dt, nsteps, integrator=FE_EULER, terms=FE_TERM_ALL):
        self._state_ok(P)
        fe_step(self.h, P, dt, nsteps, integrator, terms)
        return P

    def step_rk45(self, P: torch.Tensor, t_span, dt_init, tol, max_steps=100000, terms=FE_TERM_ALL) -> dict:
        self._state_ok(P)
        return fe_step_rk45(self.h, P, t_span, dt_init, tol, max_steps, terms)

    def energy(self, P: torch.Tensor, terms=FE_TERM_ALL, allow_nonfinite=False) -> np.ndarray:
        self._state_ok(P)
        return fe_energy(self.h, P, self.batch, terms, allow_nonfinite)

    def energy_noalloc(self, P: torch.Tensor, out: torch.Tensor, terms=FE_TERM_ALL) -> torch.Tensor:
        self._state_ok(P)
        if tuple(out.shape) != (self.batch, 8):
            raise ValueError("out must have shape (batch, 8)")
        return fe_energy_noalloc(self.h, P, out, terms)

    def get_tensor(self) -> np.ndarray: return fe_get_tensor(self.h)
    def launch_count(self) -> int: return fe_launch_count(self.h)
    def set_option(self, option: int, value: int): fe_set_option(self.h, option, value)
    def get_option(self, option: int) -> int: return fe_get_option(self.h, option)
    def profile(self, enable: bool): fe_profile(self.h, enable)
    def profile_read(self): return fe_profile_read(self.h)

    def close(self):
        if self.h is not None:
            fe_destroy_grid(self.h)
            self.h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass
