"""Thin ctypes binding of libcans_poisson.so (include/cans_poisson.h) -- argument marshalling only.

Every step of the hot path runs in the library's CUDA kernels; torch is used for device memory and
streams.  If the shared library is missing this module raises at import time: there is no fallback.
"""
from __future__ import annotations

import ctypes
import os
from typing import Optional, Sequence

import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libcans_poisson.so")

CANS_OK = 0
CANS_ERR_INVALID_ARG = 1
CANS_ERR_UNSUPPORTED_BC = 2
CANS_ERR_UNSUPPORTED_SIZE = 3
CANS_ERR_ALLOC = 4
CANS_ERR_CUDA = 5
CANS_ERR_NEEDS_FACE = 6
MAX_KERNEL_RECORDS = 16      # CANS_MAX_KERNEL_RECORDS of the header

EXPORTED_SYMBOLS = (
    "cans_poisson_plan_create", "cans_poisson_plan_destroy", "cans_poisson_solve", "cans_projection",
    "cans_projection_step", "cans_projection_step_implicit", "cans_chkdt", "cans_chkdt_static", "cans_helmholtz_plan_create", "cans_helmholtz_solve",
    "cans_probe_fp64_fma", "cans_probe_tile_copy",
    "cans_projection_set_lower_face", "cans_poisson_solve_host", "cans_projection_host",
    "cans_last_error", "cans_last_status", "cans_plan_launches_per_solve",
    "cans_plan_launches_per_projection", "cans_version",
    "cans_plan_set_profiling", "cans_plan_kernel_times", "cans_plan_kernel_name",
)


class CansError(RuntimeError):
    def __init__(self, status: int, message: str):
        super().__init__(f"cans_poisson error {status}: {message}")
        self.status = status


def _load() -> ctypes.CDLL:
    if not os.path.exists(LIB_PATH):
        raise ImportError(
            f"{LIB_PATH} not found: build it with `python -m paper_2001_05234_b200.build` "
            "(nvcc, sm_100a). There is no CPU or library fallback.")
    lib = ctypes.CDLL(LIB_PATH)
    vp, dbl, i32 = ctypes.c_void_p, ctypes.c_double, ctypes.c_int
    lib.cans_poisson_plan_create.restype = vp
    lib.cans_poisson_plan_create.argtypes = [i32, i32, i32, dbl, dbl, dbl, ctypes.c_char_p, vp, vp]
    lib.cans_poisson_plan_destroy.restype = None
    lib.cans_poisson_plan_destroy.argtypes = [vp]
    lib.cans_poisson_solve.restype = i32
    lib.cans_poisson_solve.argtypes = [vp, vp, vp]
    lib.cans_projection.restype = i32
    lib.cans_projection.argtypes = [vp, vp, vp, vp, vp, dbl, vp]
    lib.cans_projection_set_lower_face.restype = i32
    lib.cans_projection_set_lower_face.argtypes = [vp, i32, vp]
    lib.cans_poisson_solve_host.restype = i32
    lib.cans_poisson_solve_host.argtypes = [vp, vp, vp]
    lib.cans_projection_host.restype = i32
    lib.cans_projection_host.argtypes = [vp, vp, vp, vp, vp, dbl, vp]
    lib.cans_last_error.restype = ctypes.c_char_p
    lib.cans_last_error.argtypes = []
    lib.cans_last_status.restype = i32
    lib.cans_last_status.argtypes = []
    lib.cans_plan_launches_per_solve.restype = i32
    lib.cans_plan_launches_per_solve.argtypes = [vp]
    lib.cans_plan_launches_per_projection.restype = i32
    lib.cans_plan_launches_per_projection.argtypes = [vp]
    lib.cans_helmholtz_plan_create.restype = vp
    lib.cans_helmholtz_plan_create.argtypes = lib.cans_poisson_plan_create.argtypes + [i32]
    lib.cans_helmholtz_solve.restype = i32
    lib.cans_helmholtz_solve.argtypes = [vp, vp, ctypes.c_double, vp]
    lib.cans_probe_fp64_fma.restype = i32
    lib.cans_probe_fp64_fma.argtypes = [ctypes.POINTER(ctypes.c_double), vp]
    lib.cans_probe_tile_copy.restype = i32
    lib.cans_probe_tile_copy.argtypes = [vp, vp, i32, ctypes.POINTER(ctypes.c_float), vp]
    lib.cans_projection_step.restype = i32
    lib.cans_projection_step.argtypes = [vp, vp, vp, vp, vp, vp, ctypes.c_double, vp, vp]
    lib.cans_projection_step_implicit.restype = i32
    lib.cans_projection_step_implicit.argtypes = [vp, vp, vp, vp, vp, vp, dbl, dbl, vp, vp]
    lib.cans_chkdt.restype = i32
    lib.cans_chkdt.argtypes = [vp, vp, vp, vp, vp, vp]
    lib.cans_chkdt_static.restype = i32
    lib.cans_chkdt_static.argtypes = [i32, i32, i32, dbl, dbl, dbl, ctypes.c_char_p] + [vp] * 10
    lib.cans_plan_set_profiling.restype = i32
    lib.cans_plan_set_profiling.argtypes = [vp, i32]
    lib.cans_plan_kernel_times.restype = i32
    lib.cans_plan_kernel_times.argtypes = [vp, ctypes.POINTER(ctypes.c_float), i32]
    lib.cans_plan_kernel_name.restype = ctypes.c_char_p
    lib.cans_plan_kernel_name.argtypes = [vp, i32]
    lib.cans_version.restype = ctypes.c_char_p
    lib.cans_version.argtypes = []
    return lib


_lib = _load()


def version() -> str:
    return _lib.cans_version().decode()


def last_error() -> str:
    return _lib.cans_last_error().decode()


def _check(rc: int):
    if rc != CANS_OK:
        raise CansError(rc, last_error())


def _bc_bytes(bc) -> bytes:
    flat = "".join(str(bc[d][s]) for d in range(3) for s in range(2))
    return flat.encode("ascii")


def _dev_ptr(t: torch.Tensor, shape) -> int:
    if not (t.is_cuda and t.dtype == torch.float64 and t.is_contiguous() and tuple(t.shape) == tuple(shape)):
        raise ValueError(f"expected a contiguous CUDA float64 tensor of shape {tuple(shape)}")
    return t.data_ptr()


def _host_ptr(t: torch.Tensor, shape) -> int:
    if t.is_cuda or t.dtype != torch.float64 or not t.is_contiguous() or tuple(t.shape) != tuple(shape):
        raise ValueError(f"expected a contiguous CPU float64 tensor of shape {tuple(shape)}")
    return t.data_ptr()


def _stream_ptr(stream) -> int:
    if stream is None:
        stream = torch.cuda.current_stream()
    return stream.cuda_stream


def probe_fp64_fma(stream=None) -> float:
    """cans_probe_fp64_fma: measured FP64 FMA instructions per second of the current device."""
    out = ctypes.c_double(0.0)
    _check(_lib.cans_probe_fp64_fma(ctypes.byref(out), _stream_ptr(stream)))
    return float(out.value)


STATIC_MAX_NZ = 1024         # CANS_STATIC_MAX_NZ
STATIC_MAX_CTAS = 65536      # CANS_STATIC_MAX_CTAS


def chkdt_static(u, v, w, dti, lx: float, ly: float, lz: float, bc, dzc=None, dzf=None, faces=None, stream=None):
    """cans_chkdt_static: the chkdt reduction without a plan and without any device allocation inside the library -- for
    a caller whose own pool already holds all of the GPU's memory, or whose other streams must not stall behind a
    cudaMalloc / cudaFree.  The scratch is a fixed 528 KB array in the library image, shared by all calls: calls that may
    overlap on the GPU race.  u, v, w: CUDA float64 tensors (nz, ny, nx); dzc / dzf: CUDA float64 tensors of nz+1 / nz
    entries or both None (uniform); faces: {direction: lower-face plane tensor} (required on lower 'D' sides);
    dti: one-element CUDA float64 tensor, overwritten.  Grids beyond the fixed array raise CansError (status 3)."""
    nz, ny, nx = u.shape
    shape = (nz, ny, nx)
    faces = faces or {}
    want = {0: (nz, ny, 1), 1: (nz, 1, nx), 2: (1, ny, nx)}
    fptr = [None if faces.get(d) is None else _dev_ptr(faces[d], want[d]) for d in range(3)]
    _check(_lib.cans_chkdt_static(nx, ny, nz, float(lx), float(ly), float(lz), _bc_bytes(bc),
                                  None if dzc is None else _dev_ptr(dzc, (nz + 1,)),
                                  None if dzf is None else _dev_ptr(dzf, (nz,)),
                                  _dev_ptr(u, shape), _dev_ptr(v, shape), _dev_ptr(w, shape),
                                  fptr[0], fptr[1], fptr[2], _dev_ptr(dti, (1,)), _stream_ptr(stream)))


class PoissonPlan:
    """cans_poisson_plan_create / _destroy.  Fields are torch CUDA float64 tensors of shape (nz, ny, nx)."""

    def __init__(self, nx: int, ny: int, nz: int, lx: float, ly: float, lz: float, bc,
                 dzc: Optional[Sequence[float]] = None, dzf: Optional[Sequence[float]] = None,
                 stagger: Optional[int] = None):
        self.shape = (nz, ny, nx)
        self._h = None
        dzc_t = dzf_t = None
        pc = pf = None
        if dzc is not None:
            dzc_t = torch.as_tensor(dzc, dtype=torch.float64, device="cpu").contiguous()
            if dzc_t.numel() != nz + 1:
                raise ValueError("dzc must have nz+1 entries")
            pc = dzc_t.data_ptr()
        if dzf is not None:
            dzf_t = torch.as_tensor(dzf, dtype=torch.float64, device="cpu").contiguous()
            if dzf_t.numel() != nz:
                raise ValueError("dzf must have nz entries")
            pf = dzf_t.data_ptr()
        if stagger is None:
            h = _lib.cans_poisson_plan_create(nx, ny, nz, float(lx), float(ly), float(lz), _bc_bytes(bc), pc, pf)
        else:       # cans_helmholtz_plan_create: the unknown lives on the faces of direction `stagger` (-1: centres)
            h = _lib.cans_helmholtz_plan_create(nx, ny, nz, float(lx), float(ly), float(lz), _bc_bytes(bc), pc, pf, int(stagger))
        if not h:
            raise CansError(_lib.cans_last_status(), last_error())
        self._h = h

    def close(self):
        if self._h:
            _lib.cans_poisson_plan_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # --- device entry points -------------------------------------------------------------------
    def poisson_solve(self, p: torch.Tensor, stream=None):
        """cans_poisson_solve: p (f on entry) is overwritten with Phi."""
        _check(_lib.cans_poisson_solve(self._h, _dev_ptr(p, self.shape), _stream_ptr(stream)))

    def helmholtz_solve(self, q: torch.Tensor, alpha: float, stream=None):
        """cans_helmholtz_solve: q (f on entry) is overwritten with Phi, (L + alpha I) Phi = f, alpha < 0 (eq. 3b)."""
        _check(_lib.cans_helmholtz_solve(self._h, _dev_ptr(q, self.shape), float(alpha), _stream_ptr(stream)))

    def projection(self, u, v, w, p, dt: float, stream=None):
        """cans_projection: u, v, w corrected in place, p overwritten with Phi."""
        _check(_lib.cans_projection(self._h, _dev_ptr(u, self.shape), _dev_ptr(v, self.shape),
                                    _dev_ptr(w, self.shape), _dev_ptr(p, self.shape), float(dt),
                                    _stream_ptr(stream)))

    def projection_step(self, u, v, w, p, dt: float, p_acc=None, dti=None, stream=None, nu_dt_half: float = 0.0):
        """cans_projection_step: the projection, plus p_acc += Phi (eq. 2d) in the correction kernel when p_acc is
        given, plus the chkdt reduction of the corrected velocities into the one-element CUDA tensor dti when given.
        nu_dt_half > 0: cans_projection_step_implicit, p_acc += Phi - nu_dt_half * L Phi (eq. 3e)."""
        pa = None if p_acc is None else _dev_ptr(p_acc, self.shape)
        dp = None if dti is None else _dev_ptr(dti, (1,))
        fields = (_dev_ptr(u, self.shape), _dev_ptr(v, self.shape), _dev_ptr(w, self.shape), _dev_ptr(p, self.shape))
        if nu_dt_half == 0.0:
            _check(_lib.cans_projection_step(self._h, *fields, pa, float(dt), dp, _stream_ptr(stream)))
        else:
            _check(_lib.cans_projection_step_implicit(self._h, *fields, pa, float(dt), float(nu_dt_half), dp, _stream_ptr(stream)))

    def chkdt(self, u, v, w, dti, stream=None):
        """cans_chkdt: dti[0] = max over cells of the per-face sums of Listing 1 (one-element CUDA float64 tensor)."""
        _check(_lib.cans_chkdt(self._h, _dev_ptr(u, self.shape), _dev_ptr(v, self.shape), _dev_ptr(w, self.shape),
                               _dev_ptr(dti, (1,)), _stream_ptr(stream)))

    def set_lower_face(self, direction: int, plane: Optional[torch.Tensor]):
        """cans_projection_set_lower_face: register (or, with None, unregister) the boundary-normal velocity on the
        lower face of `direction`: a contiguous float64 CUDA tensor with the field's shape and extent 1 along that
        direction.  The library keeps the pointer, not the tensor: keep it alive while it is registered."""
        ptr = None
        if plane is not None:
            nz, ny, nx = self.shape
            want = {0: (nz, ny, 1), 1: (nz, 1, nx), 2: (1, ny, nx)}.get(int(direction))
            if want is None:
                raise ValueError("direction must be 0, 1 or 2")
            if plane.dtype != torch.float64 or not plane.is_cuda or not plane.is_contiguous() or tuple(plane.shape) != want:
                raise ValueError(f"lower-face plane must be a contiguous float64 CUDA tensor of shape {want}")
            ptr = plane.data_ptr()
        _check(_lib.cans_projection_set_lower_face(self._h, int(direction), ptr))

    # --- host-buffer entry points (end-to-end timing) ---------------------------------------------
    def poisson_solve_host(self, p_host: torch.Tensor, stream=None):
        _check(_lib.cans_poisson_solve_host(self._h, _host_ptr(p_host, self.shape), _stream_ptr(stream)))

    def projection_host(self, u, v, w, p, dt: float, stream=None):
        _check(_lib.cans_projection_host(self._h, _host_ptr(u, self.shape), _host_ptr(v, self.shape),
                                         _host_ptr(w, self.shape), _host_ptr(p, self.shape), float(dt),
                                         _stream_ptr(stream)))

    def probe_tile_copy(self, p: torch.Tensor, which: int, stream=None) -> float:
        """cans_probe_tile_copy: ms of a bare TMA copy of p with the z-solve (0) or y-transform (1) tiles."""
        ms = ctypes.c_float(0.0)
        _check(_lib.cans_probe_tile_copy(self._h, _dev_ptr(p, self.shape), int(which), ctypes.byref(ms), _stream_ptr(stream)))
        return float(ms.value)

    def set_profiling(self, enable: bool):
        _check(_lib.cans_plan_set_profiling(self._h, 1 if enable else 0))

    def kernel_times(self):
        """[(kernel name, ms)] of the last call, in launch order (profiling must be enabled)."""
        buf = (ctypes.c_float * MAX_KERNEL_RECORDS)()
        n = _lib.cans_plan_kernel_times(self._h, buf, MAX_KERNEL_RECORDS)
        if n < 0:
            raise CansError(_lib.cans_last_status(), last_error())
        return [(_lib.cans_plan_kernel_name(self._h, i).decode(), float(buf[i])) for i in range(n)]

    @property
    def launches_per_solve(self) -> int:
        return _lib.cans_plan_launches_per_solve(self._h)

    @property
    def launches_per_projection(self) -> int:
        return _lib.cans_plan_launches_per_projection(self._h)


def plan_for(workload) -> PoissonPlan:
    """Plan for a workloads.Workload."""
    nx, ny, nz = workload.n
    lx, ly, lz = workload.lengths
    return PoissonPlan(nx, ny, nz, lx, ly, lz, workload.bc, workload.dzc, workload.dzf)
