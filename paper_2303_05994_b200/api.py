"""Thin ctypes binding of libbsl6d.so (include/bsl6d.h).  Argument marshalling only: every step of the path
runs in the CUDA kernels behind the C ABI.  torch is used for device memory and streams, nothing else.

There is no CPU fallback: if the shared library is missing or no CUDA device is present, calls raise.
"""
from __future__ import annotations

import ctypes as C
import os
from typing import Optional, Sequence

import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libbsl6d.so")

#: every symbol include/bsl6d.h declares (tests check that the library exports exactly these)
SYMBOLS = (
    "bsl6d_create", "bsl6d_destroy", "bsl6d_advect", "bsl6d_advect_generic", "bsl6d_rotate",
    "bsl6d_strang_step", "bsl6d_density", "bsl6d_run_host", "bsl6d_run_host_begin", "bsl6d_run_host_end", "bsl6d_advect_x1_peer", "bsl6d_strerror", "bsl6d_last_cuda_error",
    "bsl6d_launch_count", "bsl6d_kernel_name", "bsl6d_version", "bsl6d_advect_seq", "bsl6d_seq_passes",
    "bsl6d_set_fusion", "bsl6d_field_poisson", "bsl6d_field_adiabatic", "bsl6d_vp_step",
    "bsl6d_advect_pointwise", "bsl6d_set_boundary", "bsl6d_density_static", "bsl6d_density_scratch",
    "bsl6d_density_scratch_doubles",
)

OK, EINVAL, EALIAS, EUNSUPPORTED, ECUDA, ENOMEM, ESCRATCH = 0, -1, -2, -3, -4, -5, -6

#: doubles of scratch compiled into the library for density_static (BSL6D_STATIC_SCRATCH_DOUBLES, 2 MiB per GPU)
STATIC_SCRATCH_DOUBLES = 262144


class Grid(C.Structure):
    """bsl6d_grid: node i of dim d at lo[d] + i*dx[d]."""
    _fields_ = [("n", C.c_int32 * 6), ("lo", C.c_double * 6), ("dx", C.c_double * 6)]


class HostOp(C.Structure):
    """bsl6d_host_op."""
    _fields_ = [("kind", C.c_int32), ("dim", C.c_int32), ("shift_source", C.c_void_p), ("dt", C.c_double),
                ("B", C.c_double * 3), ("rho_host", C.c_void_p)]


class Sweep(C.Structure):
    """bsl6d_sweep."""
    _fields_ = [("dim", C.c_int32), ("src_dim_mask", C.c_uint32), ("src", C.c_void_p), ("scale", C.c_double)]


class Bsl6dError(RuntimeError):
    def __init__(self, code: int, what: str, detail: str = ""):
        self.code = code
        super().__init__(f"{what}: error {code} ({detail})")


_lib = None


def load_library() -> C.CDLL:
    """dlopen libbsl6d.so (built in-tree by paper_2303_05994_b200.build); raises if it is not there."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise FileNotFoundError(
            f"{LIB_PATH} is missing: run `python -m paper_2303_05994_b200.build` (there is no CPU fallback)")
    lib = C.CDLL(LIB_PATH)
    vp, dp = C.c_void_p, C.c_void_p
    lib.bsl6d_create.argtypes = [C.POINTER(Grid), C.c_int, C.POINTER(vp)]
    lib.bsl6d_destroy.argtypes = [vp]
    lib.bsl6d_destroy.restype = None
    lib.bsl6d_advect.argtypes = [vp, dp, dp, C.c_int, dp, C.c_double, vp]
    lib.bsl6d_advect_generic.argtypes = [vp, dp, dp, C.c_int, dp, C.c_uint, C.c_double, vp]
    lib.bsl6d_rotate.argtypes = [vp, dp, dp, C.POINTER(C.c_double), C.c_double, vp]
    lib.bsl6d_strang_step.argtypes = [vp, dp, dp, C.POINTER(C.c_void_p), C.POINTER(C.c_double), C.c_double, vp]
    lib.bsl6d_density.argtypes = [vp, dp, dp, vp]
    lib.bsl6d_density_scratch.argtypes = [vp, dp, dp, dp, vp]
    lib.bsl6d_density_scratch_doubles.argtypes = [vp]
    lib.bsl6d_density_scratch_doubles.restype = C.c_longlong
    lib.bsl6d_density_static.argtypes = [C.POINTER(C.c_int32), C.POINTER(C.c_double), dp, dp, vp, C.POINTER(C.c_int)]
    lib.bsl6d_run_host.argtypes = [vp, dp, dp, C.POINTER(HostOp), C.c_int]
    lib.bsl6d_run_host_begin.argtypes = [vp, dp, dp, C.POINTER(HostOp), C.c_int, C.c_int]
    lib.bsl6d_run_host_end.argtypes = [vp, C.c_int]
    lib.bsl6d_advect_x1_peer.argtypes = [vp, dp, dp, dp, dp, C.c_int, dp, C.c_double, vp]
    lib.bsl6d_strerror.argtypes = [C.c_int]
    lib.bsl6d_strerror.restype = C.c_char_p
    lib.bsl6d_last_cuda_error.argtypes = [vp]
    lib.bsl6d_launch_count.argtypes = [vp]
    lib.bsl6d_launch_count.restype = C.c_longlong
    lib.bsl6d_kernel_name.argtypes = [vp, C.c_int, C.c_char_p, C.c_int]
    lib.bsl6d_version.restype = C.c_int
    lib.bsl6d_advect_seq.argtypes = [vp, dp, dp, C.POINTER(Sweep), C.c_int, vp]
    lib.bsl6d_seq_passes.argtypes = [vp, C.POINTER(Sweep), C.c_int]
    lib.bsl6d_set_fusion.argtypes = [vp, C.c_int]
    lib.bsl6d_set_boundary.argtypes = [vp, C.c_int, C.c_int]
    lib.bsl6d_advect_pointwise.argtypes = [vp, dp, dp, C.c_int, dp, C.c_int, vp]
    lib.bsl6d_field_poisson.argtypes = [vp, dp, C.c_double, C.c_double, C.POINTER(C.c_void_p), vp]
    lib.bsl6d_field_adiabatic.argtypes = [vp, dp, C.c_double, C.c_double, C.POINTER(C.c_void_p), vp]
    lib.bsl6d_vp_step.argtypes = [vp, dp, dp, dp, C.POINTER(C.c_void_p), C.POINTER(C.c_double), C.c_double, C.c_int,
                                  C.c_double, C.c_double, vp]
    _lib = lib
    return lib


def _dev_ptr(t: Optional[torch.Tensor], what: str) -> Optional[int]:
    if t is None:
        return None
    if not (t.is_cuda and t.dtype == torch.float64 and t.is_contiguous()):
        raise TypeError(f"{what}: want a contiguous float64 CUDA tensor")
    return t.data_ptr()


def _host_ptr(t: Optional[torch.Tensor], what: str) -> Optional[int]:
    if t is None:
        return None
    if t.is_cuda or t.dtype != torch.float64 or not t.is_contiguous():
        raise TypeError(f"{what}: want a contiguous float64 CPU tensor")
    return t.data_ptr()


def _stream(stream) -> Optional[int]:
    if stream is None:
        stream = torch.cuda.current_stream()
    return stream.cuda_stream or None


class Context:
    """bsl6d_ctx*.  Methods carry the names of the C entry points."""

    def __init__(self, n: Sequence[int], lo: Sequence[float], dx: Sequence[float], degree: int):
        self._lib = load_library()
        self._h = C.c_void_p()
        g = Grid()
        for d in range(6):
            g.n[d], g.lo[d], g.dx[d] = int(n[d]), float(lo[d]), float(dx[d])
        self.n = tuple(int(v) for v in n)
        self.degree = int(degree)
        self.npts = 1
        for v in self.n:
            self.npts *= v
        self.nx = self.n[0] * self.n[1] * self.n[2]
        self.device = torch.cuda.current_device() if torch.cuda.is_available() else None
        rc = self._lib.bsl6d_create(C.byref(g), int(degree), C.byref(self._h))
        if rc != OK:
            self._h = C.c_void_p()
            raise Bsl6dError(rc, "bsl6d_create", self._lib.bsl6d_strerror(rc).decode())

    # -- plumbing ---------------------------------------------------------------------------------------
    def _check(self, rc: int, what: str):
        if rc != OK:
            detail = self._lib.bsl6d_strerror(rc).decode()
            if rc == ECUDA:
                detail += f"; cudaError {self._lib.bsl6d_last_cuda_error(self._h)}"
            raise Bsl6dError(rc, what, detail)

    def destroy(self):
        if getattr(self, "_h", None) and self._h.value:
            self._lib.bsl6d_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.destroy()

    def _shape_ok(self, t: torch.Tensor, what: str):
        self._count_ok(t, self.npts, what)

    def _count_ok(self, t: Optional[torch.Tensor], want: int, what: str):
        """Element count and device of a tensor argument (the C ABI takes bare pointers and cannot check either)."""
        if t is None:
            return
        if t.numel() != want:
            raise ValueError(f"{what}: {t.numel()} elements, want {want} for grid {self.n}")
        if t.is_cuda and self.device is not None and t.device.index != self.device:
            raise ValueError(f"{what}: lives on cuda:{t.device.index}, the context was created on cuda:{self.device}")

    def _mask_count(self, mask: int) -> int:
        want = 1
        for d in range(6):
            if mask >> d & 1:
                want *= self.n[d]
        return want

    # -- the C entry points -------------------------------------------------------------------------------
    def advect(self, f_in, f_out, dim: int, shift_source, dt: float, stream=None):
        self._shape_ok(f_in, "f_in"); self._shape_ok(f_out, "f_out")
        if 0 <= int(dim) <= 5:
            self._count_ok(shift_source, self.n[dim + 3] if dim < 3 else self.nx, "shift_source")
        self._check(self._lib.bsl6d_advect(self._h, _dev_ptr(f_in, "f_in"), _dev_ptr(f_out, "f_out"), int(dim),
                                           _dev_ptr(shift_source, "shift_source"), float(dt), _stream(stream)),
                    "bsl6d_advect")
        return f_out

    def advect_generic(self, f_in, f_out, dim: int, src, src_dim_mask: int, scale: float, stream=None):
        self._shape_ok(f_in, "f_in"); self._shape_ok(f_out, "f_out")
        self._count_ok(src, self._mask_count(int(src_dim_mask)), "src")
        self._check(self._lib.bsl6d_advect_generic(self._h, _dev_ptr(f_in, "f_in"), _dev_ptr(f_out, "f_out"),
                                                   int(dim), _dev_ptr(src, "src"), int(src_dim_mask), float(scale),
                                                   _stream(stream)), "bsl6d_advect_generic")
        return f_out

    def rotate(self, f_in, f_out, B: Sequence[float], dt: float, stream=None):
        self._shape_ok(f_in, "f_in"); self._shape_ok(f_out, "f_out")
        Bc = (C.c_double * 3)(*[float(b) for b in B])
        self._check(self._lib.bsl6d_rotate(self._h, _dev_ptr(f_in, "f_in"), _dev_ptr(f_out, "f_out"), Bc, float(dt),
                                           _stream(stream)), "bsl6d_rotate")
        return f_out

    def strang_step(self, f, f_tmp, E, B, dt: float, stream=None):
        self._shape_ok(f, "f"); self._count_ok(f_tmp, self.npts, "f_tmp")
        Ep = None
        if E is not None:
            for e in E:
                self._count_ok(e, self.nx, "E")
            Ep = (C.c_void_p * 3)(*[_dev_ptr(e, "E") for e in E])
        Bc = None if B is None else (C.c_double * 3)(*[float(b) for b in B])
        self._check(self._lib.bsl6d_strang_step(self._h, _dev_ptr(f, "f"), _dev_ptr(f_tmp, "f_tmp"), Ep, Bc, float(dt),
                                                _stream(stream)), "bsl6d_strang_step")
        return f

    def _sweeps(self, sweeps):
        """sweeps: (dim, src tensor or None, src_dim_mask, scale) tuples -> bsl6d_sweep array."""
        arr = (Sweep * max(1, len(sweeps)))()
        for i, (dim, src, mask, scale) in enumerate(sweeps):
            self._count_ok(src, self._mask_count(int(mask)), f"sweeps[{i}].src")
            arr[i].dim, arr[i].src_dim_mask, arr[i].scale = int(dim), int(mask), float(scale)
            arr[i].src = _dev_ptr(src, "src")
        return arr

    def advect_seq(self, f_in, f_out, sweeps, stream=None):
        self._shape_ok(f_in, "f_in"); self._shape_ok(f_out, "f_out")
        arr = self._sweeps(sweeps)
        self._check(self._lib.bsl6d_advect_seq(self._h, _dev_ptr(f_in, "f_in"), _dev_ptr(f_out, "f_out"), arr,
                                               len(sweeps), _stream(stream)), "bsl6d_advect_seq")
        return f_out

    def seq_passes(self, sweeps) -> int:
        rc = self._lib.bsl6d_seq_passes(self._h, self._sweeps(sweeps), len(sweeps))
        if rc < 0:
            self._check(rc, "bsl6d_seq_passes")
        return rc

    def set_fusion(self, mode) -> int:
        """0 / False: off; 1 / True: default policy; 2: fuse wherever a kernel exists.  Returns the old mode."""
        rc = self._lib.bsl6d_set_fusion(self._h, int(mode))
        if rc < 0:
            self._check(rc, "bsl6d_set_fusion")
        return rc

    def advect_x1_peer(self, f_in, f_left, f_right, f_out, halo_planes: int, shift_source, dt: float, stream=None):
        """x1 sweep of a slab reading its neighbours' planes in place (peer memory or same device); out of place."""
        self._shape_ok(f_in, "f_in"); self._shape_ok(f_out, "f_out")
        for t, nm in ((f_left, "f_left"), (f_right, "f_right")):      # may live on a peer GPU: element count only
            if t.numel() != self.npts:
                raise ValueError(f"{nm}: {t.numel()} elements, want {self.npts} for grid {self.n}")
        self._count_ok(shift_source, self.n[3], "shift_source")
        self._check(self._lib.bsl6d_advect_x1_peer(self._h, _dev_ptr(f_in, "f_in"), _dev_ptr(f_left, "f_left"),
                                                   _dev_ptr(f_right, "f_right"), _dev_ptr(f_out, "f_out"),
                                                   int(halo_planes), _dev_ptr(shift_source, "shift_source"), float(dt),
                                                   _stream(stream)), "bsl6d_advect_x1_peer")
        return f_out

    def set_boundary(self, dim: int, open_: bool) -> int:
        """Open (zero-extend) or close (periodic) x dim `dim`; returns the old setting (slab decomposition)."""
        rc = self._lib.bsl6d_set_boundary(self._h, int(dim), 1 if open_ else 0)
        if rc < 0:
            self._check(rc, "bsl6d_set_boundary")
        return rc

    def advect_pointwise(self, f_in, f_out, dim: int, alpha_cells, q: int, stream=None):
        self._shape_ok(f_in, "f_in"); self._shape_ok(f_out, "f_out"); self._shape_ok(alpha_cells, "alpha_cells")
        self._check(self._lib.bsl6d_advect_pointwise(self._h, _dev_ptr(f_in, "f_in"), _dev_ptr(f_out, "f_out"),
                                                     int(dim), _dev_ptr(alpha_cells, "alpha_cells"), int(q),
                                                     _stream(stream)), "bsl6d_advect_pointwise")
        return f_out

    def _E3(self, E):
        for e in E:
            self._count_ok(e, self.nx, "E")
        return (C.c_void_p * 3)(*[_dev_ptr(e, "E") for e in E])

    def field_poisson(self, rho, rho_fac: float, e_fac: float, E, stream=None):
        self._count_ok(rho, self.nx, "rho")
        self._check(self._lib.bsl6d_field_poisson(self._h, _dev_ptr(rho, "rho"), float(rho_fac), float(e_fac),
                                                  self._E3(E), _stream(stream)), "bsl6d_field_poisson")
        return E

    def field_adiabatic(self, rho, phi_fac: float, e_fac: float, E, stream=None):
        self._count_ok(rho, self.nx, "rho")
        self._check(self._lib.bsl6d_field_adiabatic(self._h, _dev_ptr(rho, "rho"), float(phi_fac), float(e_fac),
                                                    self._E3(E), _stream(stream)), "bsl6d_field_adiabatic")
        return E

    def vp_step(self, f, f_tmp, rho, E, B, dt: float, closure: int, c1: float, e_fac: float, stream=None):
        self._shape_ok(f, "f"); self._count_ok(f_tmp, self.npts, "f_tmp"); self._count_ok(rho, self.nx, "rho")
        Bc = None if B is None else (C.c_double * 3)(*[float(b) for b in B])
        self._check(self._lib.bsl6d_vp_step(self._h, _dev_ptr(f, "f"), _dev_ptr(f_tmp, "f_tmp"), _dev_ptr(rho, "rho"),
                                            self._E3(E), Bc, float(dt), int(closure), float(c1), float(e_fac),
                                            _stream(stream)), "bsl6d_vp_step")
        return f

    def density(self, f, rho, stream=None):
        self._shape_ok(f, "f"); self._count_ok(rho, self.nx, "rho")
        self._check(self._lib.bsl6d_density(self._h, _dev_ptr(f, "f"), _dev_ptr(rho, "rho"), _stream(stream)),
                    "bsl6d_density")
        return rho

    def density_scratch_doubles(self) -> int:
        return int(self._lib.bsl6d_density_scratch_doubles(self._h))

    def density_scratch(self, f, rho, scratch, stream=None):
        """bsl6d_density_scratch: the moment with a caller-owned work array (one per stream in flight)."""
        self._shape_ok(f, "f"); self._count_ok(rho, self.nx, "rho")
        need = self.density_scratch_doubles()
        if need and (scratch is None or scratch.numel() < need):
            raise ValueError(f"scratch: want {need} doubles")
        self._check(self._lib.bsl6d_density_scratch(self._h, _dev_ptr(f, "f"), _dev_ptr(rho, "rho"),
                                                    _dev_ptr(scratch, "scratch"), _stream(stream)), "bsl6d_density_scratch")
        return rho

    def _host_ops(self, ops: Sequence[dict]):
        arr = (HostOp * max(1, len(ops)))()
        for i, op in enumerate(ops):
            kind = {"advect": 0, "rotate": 1, "density": 2}[op["kind"]]
            arr[i].kind = kind
            arr[i].dim = int(op.get("dim", 0))
            arr[i].dt = float(op.get("dt", 0.0))
            arr[i].shift_source = _host_ptr(op.get("shift_source"), "shift_source")
            arr[i].rho_host = _host_ptr(op.get("rho_host"), "rho_host")
            for k, b in enumerate(op.get("B", (0.0, 0.0, 0.0))):
                arr[i].B[k] = float(b)
        return arr

    def run_host(self, f_in_host, f_out_host, ops: Sequence[dict]):
        """ops: dicts with kind in {'advect','rotate','density'} and dim / shift_source / dt / B / rho_host."""
        self._shape_ok(f_in_host, "f_in_host"); self._shape_ok(f_out_host, "f_out_host")
        arr = self._host_ops(ops)
        self._check(self._lib.bsl6d_run_host(self._h, _host_ptr(f_in_host, "f_in_host"),
                                             _host_ptr(f_out_host, "f_out_host"), arr, len(ops)), "bsl6d_run_host")
        return f_out_host

    def run_host_begin(self, f_in_host, f_out_host, ops: Sequence[dict], slot: int):
        """Enqueue upload, ops and download on `slot` (0 or 1) without waiting; the caller keeps every host tensor of
        the call alive and untouched until run_host_end(slot)."""
        self._shape_ok(f_in_host, "f_in_host"); self._shape_ok(f_out_host, "f_out_host")
        arr = self._host_ops(ops)
        self._check(self._lib.bsl6d_run_host_begin(self._h, _host_ptr(f_in_host, "f_in_host"),
                                                   _host_ptr(f_out_host, "f_out_host"), arr, len(ops), int(slot)),
                    "bsl6d_run_host_begin")

    def run_host_end(self, slot: int):
        self._check(self._lib.bsl6d_run_host_end(self._h, int(slot)), "bsl6d_run_host_end")

    # -- introspection --------------------------------------------------------------------------------------
    def launch_count(self) -> int:
        return int(self._lib.bsl6d_launch_count(self._h))

    def kernel_name(self, dim: int) -> str:
        buf = C.create_string_buffer(128)
        self._check(self._lib.bsl6d_kernel_name(self._h, int(dim), buf, 128), "bsl6d_kernel_name")
        return buf.value.decode()


def create(n, lo, dx, degree) -> Context:
    return Context(n, lo, dx, degree)


def density_static(n: Sequence[int], dv: Sequence[float], f, rho, stream=None):
    """bsl6d_density_static: rho[x] = dv1*dv2*dv3 * sum_v f[x, v] without a context and without any allocation.

    For users whose code may not allocate device memory while it runs -- a module inside an application that owns all
    GPU memory through an allocator of its own, or a diagnostic between time steps that must not trigger the
    synchronisation an allocation can bring.  The partial sums a long velocity block needs are kept in a 2 MiB array
    compiled into the library (STATIC_SCRATCH_DOUBLES doubles; each GPU that loads the library holds it until the
    process ends).  A grid that needs more raises Bsl6dError with code ESCRATCH.  The result has the same bits as
    Context.density.  All calls on a GPU share that array: keep them on one stream or order them with events.  The
    first call on a GPU looks the array's address up, so make it before you start capturing a stream.

    n: the six extents; dv: spacings of v1, v2, v3; f: float64 CUDA tensor of shape n on the current device;
    rho: float64 CUDA tensor with n[0]*n[1]*n[2] elements."""
    lib = load_library()
    n = [int(v) for v in n]
    if len(n) != 6 or len(dv) != 3:
        raise ValueError("n has six extents, dv three spacings")
    if tuple(f.shape) != tuple(n):
        raise ValueError(f"f: shape {tuple(f.shape)} != grid {tuple(n)}")
    if rho.numel() != n[0] * n[1] * n[2]:
        raise ValueError(f"rho: {rho.numel()} elements, want {n[0] * n[1] * n[2]}")
    cn = (C.c_int32 * 6)(*n)
    cdv = (C.c_double * 3)(*[float(v) for v in dv])
    cuda_err = C.c_int(0)
    rc = lib.bsl6d_density_static(cn, cdv, _dev_ptr(f, "f"), _dev_ptr(rho, "rho"), _stream(stream), C.byref(cuda_err))
    if rc != OK:
        detail = lib.bsl6d_strerror(rc).decode()
        if rc == ECUDA:
            detail += f"; cudaError {cuda_err.value}"
        if rc == ESCRATCH:
            detail += f" ({STATIC_SCRATCH_DOUBLES} doubles)"
        raise Bsl6dError(rc, "bsl6d_density_static", detail)
    return rho


def version() -> int:
    return int(load_library().bsl6d_version())
