"""Thin ctypes binding of libscatman (include/scatman.h): argument marshalling only.

Every step of the hot path runs inside the library's CUDA kernels.  PyTorch is used for device
memory and streams; tensors are passed as raw pointers.  There is NO fallback: if the shared
library is missing or the device is not a B200-class (cc 10.x) GPU, calls raise.
"""
from __future__ import annotations

import ctypes as C
import os
from typing import Optional, Sequence

HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(HERE, "libscatman.so")

OK, INVALID_ARGUMENT, UNSUPPORTED_DEVICE, WORKSPACE_TOO_SMALL, CUDA_ERROR, NOT_IMPLEMENTED = range(6)
RHO_LINEAR, RHO_N2M1 = 0, 1
METHOD_AUTO, METHOD_TENSOR, METHOD_SIMT_SINCOS, METHOD_SIMT_TABLE = 0, 1, 2, 3
LOSS_L2_NORMALISED, LOSS_POISSON_DEVIANCE = 0, 1
PRECISION_AUTO, PRECISION_FP16X3 = 0, 1
FLAG_SINGLE_CTA = 1
FLAG_COUNT_ISSUED = 2
FLAG_REUSE_TABLES = 4

EXPORTS = [
    "scatman_create", "scatman_destroy", "scatman_workspace_bytes", "scatman_qmap", "scatman_orient_workspace_bytes", "scatman_orient",
    "scatman_effective_strength", "scatman_simulate", "scatman_simulate_q", "scatman_simulate_host",
    "scatman_simulate_nufft_host", "scatman_simulate_qgrid_host",
    "scatman_qgrid_workspace_bytes", "scatman_simulate_qgrid", "scatman_shapes_workspace_bytes", "scatman_simulate_shapes",
    "scatman_shapes_qgrid_workspace_bytes", "scatman_simulate_shapes_qgrid",
    "scatman_nufft_workspace_bytes", "scatman_nufft_grid_dims", "scatman_simulate_nufft",
    "scatman_shapes_nufft_workspace_bytes", "scatman_simulate_shapes_nufft",
    "scatman_render", "scatman_fit_workspace_bytes", "scatman_discrepancy", "scatman_discrepancy_static", "scatman_ideal_detector", "scatman_last_launch_count", "scatman_last_contraction_ms", "scatman_last_issued_blocks", "scatman_status_string", "scatman_last_error",
    "scatman_version",
]


class Grid(C.Structure):
    _fields_ = [("nx", C.c_int32), ("ny", C.c_int32), ("nz", C.c_int32),
                ("dx", C.c_double), ("dy", C.c_double), ("dz", C.c_double)]


class Detector(C.Structure):
    _fields_ = [("npx", C.c_int32), ("npy", C.c_int32), ("theta_max_deg", C.c_double),
                ("cx", C.c_double), ("cy", C.c_double)]


class Options(C.Structure):
    _fields_ = [("rho_mode", C.c_int32), ("method", C.c_int32), ("precision", C.c_int32), ("flags", C.c_uint32)]


STATIC_SCRATCH_BYTES = 1 << 20     # SCATMAN_STATIC_SCRATCH_BYTES
SHAPE_ELLIPSOID, SHAPE_SPHERICAL_HARMONICS, SHAPE_RADIAL_MAP, SHAPE_VOLUME_MAP = range(4)


class Shape(C.Structure):
    _fields_ = [("kind", C.c_int32), ("delta", C.c_float), ("beta", C.c_float), ("quat", C.c_double * 4),
                ("a", C.c_double), ("b", C.c_double), ("c", C.c_double),
                ("ncoef", C.c_int32), ("h_coef", C.c_void_p),
                ("nlat", C.c_int32), ("nlon", C.c_int32), ("d_radii", C.c_void_p),
                ("nvx", C.c_int32), ("nvy", C.c_int32), ("nvz", C.c_int32), ("d_volume", C.c_void_p),
                ("vdx", C.c_double)]


class ScatmanError(RuntimeError):
    def __init__(self, status: int, msg: str):
        super().__init__(f"scatman status {status}: {msg}")
        self.status = status


_lib = None


def load_library() -> C.CDLL:
    """dlopen libscatman.so (built in-tree by paper_2202_03411_b200/build.py).  Fails loudly if absent."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise FileNotFoundError(f"{LIB_PATH} is missing: run `python -m paper_2202_03411_b200.build` "
                                "(or __graft_entry__.build()).  There is no CPU fallback.")
    L = C.CDLL(LIB_PATH)
    vp, i32, i64, dbl = C.c_void_p, C.c_int32, C.c_int64, C.c_double
    L.scatman_create.argtypes = [C.POINTER(vp), C.c_int]
    L.scatman_destroy.argtypes = [vp]
    L.scatman_workspace_bytes.argtypes = [vp, C.POINTER(Grid), i64, i32, C.POINTER(Options), C.POINTER(C.c_size_t)]
    L.scatman_qmap.argtypes = [vp, C.POINTER(Detector), dbl, vp, vp]
    L.scatman_orient_workspace_bytes.argtypes = [vp, i32, C.POINTER(C.c_size_t)]
    L.scatman_orient.argtypes = [vp, vp, C.POINTER(Grid), C.POINTER(dbl), i32, vp, C.c_size_t, vp, vp]
    L.scatman_effective_strength.argtypes = [vp, vp, C.POINTER(Grid), dbl, i32, i32, vp, vp]
    L.scatman_simulate.argtypes = [vp, vp, C.POINTER(Grid), dbl, C.POINTER(Detector), C.POINTER(dbl), i32,
                                   C.POINTER(Options), vp, C.c_size_t, vp, vp]
    L.scatman_simulate_q.argtypes = [vp, vp, C.POINTER(Grid), dbl, vp, i64, C.POINTER(dbl), i32,
                                     C.POINTER(Options), vp, C.c_size_t, vp, vp]
    L.scatman_simulate_host.argtypes = [vp, vp, C.POINTER(Grid), dbl, C.POINTER(Detector), C.POINTER(dbl), i32,
                                        C.POINTER(Options), vp]
    L.scatman_simulate_nufft_host.argtypes = L.scatman_simulate_host.argtypes
    L.scatman_simulate_qgrid_host.argtypes = [vp, vp, C.POINTER(Grid), dbl, C.POINTER(dbl), i32, C.POINTER(dbl), i32,
                                              C.POINTER(dbl), i32, C.POINTER(Options), vp]
    L.scatman_nufft_workspace_bytes.argtypes = [vp, C.POINTER(Grid), dbl, C.POINTER(Detector), i32, C.POINTER(C.c_size_t)]
    L.scatman_nufft_grid_dims.argtypes = [vp, C.POINTER(Grid), dbl, C.POINTER(Detector), C.POINTER(i32)]
    L.scatman_simulate_nufft.argtypes = [vp, vp, C.POINTER(Grid), dbl, C.POINTER(Detector), C.POINTER(dbl), i32,
                                         C.POINTER(Options), vp, C.c_size_t, vp, vp]
    L.scatman_shapes_nufft_workspace_bytes.argtypes = [vp, C.POINTER(Grid), dbl, C.POINTER(Detector), i32, C.POINTER(C.c_size_t)]
    L.scatman_simulate_shapes_nufft.argtypes = [vp, C.POINTER(Shape), i32, C.POINTER(Grid), dbl, C.POINTER(Detector),
                                                C.POINTER(Options), vp, C.c_size_t, vp, vp]
    L.scatman_qgrid_workspace_bytes.argtypes = [vp, C.POINTER(Grid), i32, i32, i32, C.POINTER(Options), C.POINTER(C.c_size_t)]
    L.scatman_simulate_qgrid.argtypes = [vp, vp, C.POINTER(Grid), dbl, vp, i32, vp, i32, C.POINTER(dbl), i32,
                                         C.POINTER(Options), vp, C.c_size_t, vp, vp]
    L.scatman_shapes_workspace_bytes.argtypes = [vp, C.POINTER(Grid), i64, i32, C.POINTER(Options), C.POINTER(C.c_size_t)]
    L.scatman_simulate_shapes.argtypes = [vp, C.POINTER(Shape), i32, C.POINTER(Grid), dbl, C.POINTER(Detector),
                                          C.POINTER(Options), vp, C.c_size_t, vp, vp]
    L.scatman_shapes_qgrid_workspace_bytes.argtypes = [vp, C.POINTER(Grid), i32, i32, i32, C.POINTER(Options), C.POINTER(C.c_size_t)]
    L.scatman_simulate_shapes_qgrid.argtypes = [vp, C.POINTER(Shape), i32, C.POINTER(Grid), dbl, vp, i32, vp, i32,
                                                C.POINTER(Options), vp, C.c_size_t, vp, vp]
    L.scatman_render.argtypes = [vp, C.POINTER(Shape), i32, C.POINTER(Grid), vp, vp]
    L.scatman_fit_workspace_bytes.argtypes = [vp, i64, i32, C.POINTER(C.c_size_t)]
    L.scatman_discrepancy.argtypes = [vp, vp, vp, i64, vp, i64, i32, i32, vp, C.c_size_t, vp, vp]
    L.scatman_discrepancy_static.argtypes = [vp, vp, vp, i64, vp, i64, i32, i32, vp, vp]
    L.scatman_ideal_detector.argtypes = [vp, vp, i64, i32, C.POINTER(dbl), C.c_uint64, vp, C.c_size_t, vp, vp]
    L.scatman_last_launch_count.argtypes = [vp, C.POINTER(i32)]
    L.scatman_last_contraction_ms.argtypes = [vp, C.POINTER(C.c_float)]
    L.scatman_last_issued_blocks.argtypes = [vp, C.POINTER(i64)]
    L.scatman_status_string.argtypes = [C.c_int]
    L.scatman_status_string.restype = C.c_char_p
    L.scatman_last_error.argtypes = [vp]
    L.scatman_last_error.restype = C.c_char_p
    L.scatman_version.restype = C.c_int
    for name in EXPORTS:
        getattr(L, name)
    _lib = L
    return L


def _quat_arg(quat, batch: int):
    if quat is None:
        return None, None
    flat = [float(v) for row in quat for v in row]
    if len(flat) != 4 * batch:
        raise ValueError("quat must be [batch][4]")
    arr = (C.c_double * len(flat))(*flat)
    return arr, C.cast(arr, C.POINTER(C.c_double))


class Scatman:
    """One context per device.  Methods mirror the C entry points one to one."""

    def __init__(self, device: int = 0):
        self.lib = load_library()
        self._ctx = C.c_void_p()
        rc = self.lib.scatman_create(C.byref(self._ctx), int(device))
        if rc != OK:
            raise ScatmanError(rc, self.lib.scatman_status_string(rc).decode())
        self.device = int(device)

    def close(self):
        if getattr(self, "_ctx", None) is not None and self._ctx.value:
            self.lib.scatman_destroy(self._ctx)
            self._ctx = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _check(self, rc: int):
        if rc != OK:
            msg = self.lib.scatman_last_error(self._ctx).decode() or self.lib.scatman_status_string(rc).decode()
            raise ScatmanError(rc, msg)

    # -- marshalling helpers -------------------------------------------------------------------
    @staticmethod
    def _stream(stream) -> C.c_void_p:
        if stream is None:
            import torch
            stream = torch.cuda.current_stream()
        return C.c_void_p(int(getattr(stream, "cuda_stream", stream)))

    @staticmethod
    def _empty(shape, dtype, device, stream):
        """torch.empty allocated in the ORDER OF `stream`: the caching allocator hands out blocks that are free in the order
        of the stream that is current at allocation time, so a buffer the library's kernels use on `stream` must be allocated
        (and is then freed) under that stream, not under whatever stream happens to be current."""
        import torch
        if stream is None:
            return torch.empty(shape, dtype=dtype, device=device)
        if not isinstance(stream, torch.cuda.Stream):
            stream = torch.cuda.ExternalStream(int(stream))
        with torch.cuda.stream(stream):
            return torch.empty(shape, dtype=dtype, device=device)

    @staticmethod
    def _grid_of(dn, voxel) -> Grid:
        if dn.dim() == 4:
            nz, ny, nx, two = dn.shape
        else:
            _, nz, ny, nx, two = dn.shape
        assert two == 2
        return Grid(nx, ny, nz, float(voxel[0]), float(voxel[1]), float(voxel[2]))

    @staticmethod
    def _batch_of(dn) -> int:
        return 1 if dn.dim() == 4 else int(dn.shape[0])

    @staticmethod
    def _check_dn(dn):
        import torch
        if not (dn.is_cuda and dn.dtype == torch.float32 and dn.is_contiguous()):
            raise ValueError("grid must be a contiguous CUDA float32 tensor [B][nz][ny][nx][2]")

    # -- entry points --------------------------------------------------------------------------
    def workspace_bytes(self, grid: Grid, npix: int, batch: int, opts: Optional[Options] = None) -> int:
        out = C.c_size_t(0)
        self._check(self.lib.scatman_workspace_bytes(self._ctx, C.byref(grid), int(npix), int(batch),
                                                     C.byref(opts) if opts else None, C.byref(out)))
        return int(out.value)

    def qmap(self, npx: int, npy: int, theta_max_deg: float, lam: float, cx: float = 0.0, cy: float = 0.0, stream=None):
        import torch
        q = self._empty((npx * npy, 3), torch.float64, f"cuda:{self.device}", stream)
        det = Detector(npx, npy, float(theta_max_deg), float(cx), float(cy))
        self._check(self.lib.scatman_qmap(self._ctx, C.byref(det), float(lam), C.c_void_p(q.data_ptr()), self._stream(stream)))
        return q

    def orient(self, dn, voxel, quat, stream=None):
        import torch
        self._check_dn(dn)
        grid, batch = self._grid_of(dn, voxel), self._batch_of(dn)
        out = self._empty(tuple(dn.shape), dn.dtype, dn.device, stream)
        need = C.c_size_t(0)
        self._check(self.lib.scatman_orient_workspace_bytes(self._ctx, batch, C.byref(need)))
        ws = self._empty(int(need.value), torch.uint8, dn.device, stream)
        keep, qp = _quat_arg(quat, batch)
        self._check(self.lib.scatman_orient(self._ctx, C.c_void_p(dn.data_ptr()), C.byref(grid), qp, batch,
                                            C.c_void_p(ws.data_ptr()), ws.numel(), C.c_void_p(out.data_ptr()), self._stream(stream)))
        return out

    def effective_strength(self, dn, voxel, lam: float, rho_mode: int = RHO_LINEAR, stream=None):
        import torch
        self._check_dn(dn)
        grid, batch = self._grid_of(dn, voxel), self._batch_of(dn)
        out = self._empty(tuple(dn.shape), dn.dtype, dn.device, stream)
        self._check(self.lib.scatman_effective_strength(self._ctx, C.c_void_p(dn.data_ptr()), C.byref(grid), float(lam),
                                                        int(rho_mode), batch, C.c_void_p(out.data_ptr()),
                                                        self._stream(stream)))
        return out

    @staticmethod
    def _shape_array(shapes: Sequence[dict]):
        """ctypes array of scatman_shape from descriptor dicts (+ the objects that must outlive the call)."""
        import numpy as np
        import torch
        batch = len(shapes)
        arr = (Shape * batch)()
        keep = []
        kinds = {"ellipsoid": SHAPE_ELLIPSOID, "spherical_harmonics": SHAPE_SPHERICAL_HARMONICS,
                 "radial_map": SHAPE_RADIAL_MAP, "volume_map": SHAPE_VOLUME_MAP}
        for i, sh in enumerate(shapes):
            s = arr[i]
            s.kind = kinds[sh["kind"]]
            s.delta, s.beta = float(sh["delta"]), float(sh["beta"])
            q = sh.get("quat")
            s.quat[:] = [1.0, 0.0, 0.0, 0.0] if q is None else [float(v) for v in q]
            if s.kind == SHAPE_ELLIPSOID:
                s.a, s.b, s.c = float(sh["a"]), float(sh["b"]), float(sh["c"])
            elif s.kind == SHAPE_SPHERICAL_HARMONICS:
                co = np.ascontiguousarray(np.asarray(sh["coeffs"], dtype=np.float64).reshape(-1, 3))
                keep.append(co)
                s.ncoef, s.h_coef = co.shape[0], co.ctypes.data
            elif s.kind == SHAPE_RADIAL_MAP:
                r = sh["radii"]
                if not (r.is_cuda and r.dtype == torch.float64 and r.is_contiguous() and r.dim() == 2):
                    raise ValueError("radii must be a contiguous CUDA float64 tensor [nlat][nlon]")
                keep.append(r)
                s.nlat, s.nlon, s.d_radii = int(r.shape[0]), int(r.shape[1]), r.data_ptr()
            else:
                v = sh["volume"]
                if not (v.is_cuda and v.dtype == torch.uint8 and v.is_contiguous() and v.dim() == 3):
                    raise ValueError("volume must be a contiguous CUDA uint8 tensor [nvz][nvy][nvx]")
                keep.append(v)
                s.nvz, s.nvy, s.nvx, s.d_volume, s.vdx = int(v.shape[0]), int(v.shape[1]), int(v.shape[2]), v.data_ptr(), float(sh["dx"])
        return arr, keep

    def render(self, shapes: Sequence[dict], dims, voxel, out=None, stream=None):
        """(delta, beta) grids float32 [B][nz][ny][nx][2] of shape descriptors (dicts with the keys of include/scatman.h's
        scatman_shape: kind, delta, beta, quat, and a/b/c | coeffs [(l, m, c)] | radii (CUDA float64 [nlat][nlon]) |
        volume (CUDA uint8 [nvz][nvy][nvx]) + dx).  Marshalling only: the shapes are evaluated by render_kernel."""
        import numpy as np
        import torch
        nx, ny, nz = (int(v) for v in dims)
        grid = Grid(nx, ny, nz, float(voxel[0]), float(voxel[1]), float(voxel[2]))
        batch = len(shapes)
        if out is None:
            out = self._empty((batch, nz, ny, nx, 2), torch.float32, f"cuda:{self.device}", stream)
        arr, keep = self._shape_array(shapes)
        self._check(self.lib.scatman_render(self._ctx, arr, batch, C.byref(grid), C.c_void_p(out.data_ptr()), self._stream(stream)))
        return out

    def simulate(self, dn, voxel, lam: float, npx: int, npy: int, theta_max_deg: float, quat=None,
                 rho_mode: int = RHO_LINEAR, method: int = METHOD_AUTO, cx: float = 0.0, cy: float = 0.0,
                 workspace=None, out=None, stream=None, flags: int = 0):
        """I float32 [B][npy][npx] on the device ([npy][npx] for a 4-D grid).  Asynchronous."""
        import torch
        self._check_dn(dn)
        grid, batch = self._grid_of(dn, voxel), self._batch_of(dn)
        det = Detector(int(npx), int(npy), float(theta_max_deg), float(cx), float(cy))
        opts = Options(int(rho_mode), int(method), 0, int(flags))
        need = self.workspace_bytes(grid, npx * npy, batch, opts)
        if workspace is None:
            workspace = self._empty(need, torch.uint8, dn.device, stream)
        if out is None:
            out = self._empty((batch, npy, npx), torch.float32, dn.device, stream)
        keep, qp = _quat_arg(quat, batch)
        self._check(self.lib.scatman_simulate(self._ctx, C.c_void_p(dn.data_ptr()), C.byref(grid), float(lam),
                                              C.byref(det), qp, batch, C.byref(opts), C.c_void_p(workspace.data_ptr()),
                                              workspace.numel(), C.c_void_p(out.data_ptr()), self._stream(stream)))
        return out if dn.dim() == 5 else out[0]

    def nufft_grid_dims(self, grid, lam: float, det):
        """(nqx, nqy, nqz): points per axis of the uniform grid scatman_simulate_nufft transforms onto."""
        nq = (C.c_int32 * 3)()
        self._check(self.lib.scatman_nufft_grid_dims(self._ctx, C.byref(grid), float(lam), C.byref(det), nq))
        return int(nq[0]), int(nq[1]), int(nq[2])

    def simulate_nufft(self, dn, voxel, lam: float, npx: int, npy: int, theta_max_deg: float, quat=None,
                       rho_mode: int = RHO_LINEAR, cx: float = 0.0, cy: float = 0.0, workspace=None, out=None, stream=None,
                       flags: int = 0, method: int = METHOD_AUTO):
        """Same result as simulate() by the 3-D type-2 NUFFT route (scatman_simulate_nufft).  Asynchronous.
        method: AUTO / TENSOR = GEMM stages on tcgen05 (FP16x3), SIMT_TABLE = FP64 CUDA-core stages."""
        import torch
        self._check_dn(dn)
        grid, batch = self._grid_of(dn, voxel), self._batch_of(dn)
        det = Detector(int(npx), int(npy), float(theta_max_deg), float(cx), float(cy))
        opts = Options(int(rho_mode), int(method), 0, int(flags))
        need = C.c_size_t(0)
        self._check(self.lib.scatman_nufft_workspace_bytes(self._ctx, C.byref(grid), float(lam), C.byref(det), batch,
                                                           C.byref(need)))
        if workspace is None:
            workspace = self._empty(int(need.value), torch.uint8, dn.device, stream)
        if out is None:
            out = self._empty((batch, npy, npx), torch.float32, dn.device, stream)
        keep, qp = _quat_arg(quat, batch)
        self._check(self.lib.scatman_simulate_nufft(self._ctx, C.c_void_p(dn.data_ptr()), C.byref(grid), float(lam),
                                                    C.byref(det), qp, batch, C.byref(opts), C.c_void_p(workspace.data_ptr()),
                                                    workspace.numel(), C.c_void_p(out.data_ptr()), self._stream(stream)))
        return out if dn.dim() == 5 else out[0]

    def simulate_q(self, dn, voxel, lam: float, q, quat=None, rho_mode: int = RHO_LINEAR, method: int = METHOD_AUTO,
                   workspace=None, out=None, stream=None, flags: int = 0):
        """I float32 [B][npix] at the explicit device q list [npix][3] (float64)."""
        import torch
        self._check_dn(dn)
        if not (q.is_cuda and q.dtype == torch.float64 and q.is_contiguous() and q.shape[-1] == 3):
            raise ValueError("q must be a contiguous CUDA float64 tensor [npix][3]")
        grid, batch = self._grid_of(dn, voxel), self._batch_of(dn)
        npix = int(q.shape[0])
        opts = Options(int(rho_mode), int(method), 0, int(flags))
        need = self.workspace_bytes(grid, npix, batch, opts)
        if workspace is None:
            workspace = self._empty(need, torch.uint8, dn.device, stream)
        if out is None:
            out = self._empty((batch, npix), torch.float32, dn.device, stream)
        keep, qp = _quat_arg(quat, batch)
        self._check(self.lib.scatman_simulate_q(self._ctx, C.c_void_p(dn.data_ptr()), C.byref(grid), float(lam),
                                                C.c_void_p(q.data_ptr()), npix, qp, batch, C.byref(opts),
                                                C.c_void_p(workspace.data_ptr()), workspace.numel(),
                                                C.c_void_p(out.data_ptr()), self._stream(stream)))
        return out if dn.dim() == 5 else out[0]

    def simulate_shapes(self, shapes: Sequence[dict], dims, voxel, lam: float, npx: int, npy: int, theta_max_deg: float,
                        rho_mode: int = RHO_LINEAR, method: int = METHOD_AUTO, workspace=None, out=None, stream=None,
                        flags: int = 0):
        """Shape descriptors (see render) -> I float32 [B][npy][npx]: rendered and simulated on the device."""
        import torch
        nx, ny, nz = (int(v) for v in dims)
        grid = Grid(nx, ny, nz, float(voxel[0]), float(voxel[1]), float(voxel[2]))
        batch = len(shapes)
        det = Detector(int(npx), int(npy), float(theta_max_deg), 0.0, 0.0)
        opts = Options(int(rho_mode), int(method), 0, int(flags))
        need = C.c_size_t(0)
        self._check(self.lib.scatman_shapes_workspace_bytes(self._ctx, C.byref(grid), npx * npy, batch, C.byref(opts), C.byref(need)))
        dev = f"cuda:{self.device}"
        if workspace is None:
            workspace = self._empty(int(need.value), torch.uint8, dev, stream)
        if out is None:
            out = self._empty((batch, npy, npx), torch.float32, dev, stream)
        arr, keep = self._shape_array(shapes)
        self._check(self.lib.scatman_simulate_shapes(self._ctx, arr, batch, C.byref(grid), float(lam), C.byref(det), C.byref(opts),
                                                     C.c_void_p(workspace.data_ptr()), workspace.numel(),
                                                     C.c_void_p(out.data_ptr()), self._stream(stream)))
        return out

    def simulate_shapes_qgrid(self, shapes: Sequence[dict], dims, voxel, lam: float, qx, qy, rho_mode: int = RHO_LINEAR,
                              method: int = METHOD_AUTO, workspace=None, out=None, stream=None):
        """Shape descriptors -> I float32 [B][npy][npx] on the tensor grid (qx[a], qy[b]): rendered on the device, then the
        separable route (scatman_simulate_shapes_qgrid)."""
        import torch
        for q in (qx, qy):
            if not (q.is_cuda and q.dtype == torch.float64 and q.is_contiguous() and q.dim() == 1):
                raise ValueError("qx, qy must be contiguous 1-D CUDA float64 tensors")
        nx, ny, nz = (int(v) for v in dims)
        grid = Grid(nx, ny, nz, float(voxel[0]), float(voxel[1]), float(voxel[2]))
        batch, npx, npy = len(shapes), int(qx.numel()), int(qy.numel())
        opts = Options(int(rho_mode), int(method), 0, 0)
        need = C.c_size_t(0)
        self._check(self.lib.scatman_shapes_qgrid_workspace_bytes(self._ctx, C.byref(grid), npx, npy, batch, C.byref(opts),
                                                                  C.byref(need)))
        if workspace is None:
            workspace = self._empty(int(need.value), torch.uint8, qx.device, stream)
        if out is None:
            out = self._empty((batch, npy, npx), torch.float32, qx.device, stream)
        arr, keep = self._shape_array(shapes)
        self._check(self.lib.scatman_simulate_shapes_qgrid(self._ctx, arr, batch, C.byref(grid), float(lam),
                                                           C.c_void_p(qx.data_ptr()), npx, C.c_void_p(qy.data_ptr()), npy,
                                                           C.byref(opts), C.c_void_p(workspace.data_ptr()), workspace.numel(),
                                                           C.c_void_p(out.data_ptr()), self._stream(stream)))
        return out

    def simulate_shapes_nufft(self, shapes: Sequence[dict], dims, voxel, lam: float, npx: int, npy: int, theta_max_deg: float,
                              rho_mode: int = RHO_LINEAR, cx: float = 0.0, cy: float = 0.0, workspace=None, out=None, stream=None):
        """Shape descriptors -> I float32 [B][npy][npx] on the flat detector: rendered on the device, then the NUFFT route
        (scatman_simulate_shapes_nufft)."""
        import torch
        nx, ny, nz = (int(v) for v in dims)
        grid = Grid(nx, ny, nz, float(voxel[0]), float(voxel[1]), float(voxel[2]))
        det = Detector(int(npx), int(npy), float(theta_max_deg), float(cx), float(cy))
        batch = len(shapes)
        opts = Options(int(rho_mode), 0, 0, 0)
        need = C.c_size_t(0)
        self._check(self.lib.scatman_shapes_nufft_workspace_bytes(self._ctx, C.byref(grid), float(lam), C.byref(det), batch,
                                                                  C.byref(need)))
        if workspace is None:
            workspace = self._empty(int(need.value), torch.uint8, "cuda", stream)
        if out is None:
            out = self._empty((batch, npy, npx), torch.float32, "cuda", stream)
        arr, keep = self._shape_array(shapes)
        self._check(self.lib.scatman_simulate_shapes_nufft(self._ctx, arr, batch, C.byref(grid), float(lam), C.byref(det),
                                                           C.byref(opts), C.c_void_p(workspace.data_ptr()), workspace.numel(),
                                                           C.c_void_p(out.data_ptr()), self._stream(stream)))
        return out

    def simulate_qgrid(self, dn, voxel, lam: float, qx, qy, quat=None, rho_mode: int = RHO_LINEAR, method: int = METHOD_AUTO,
                       workspace=None, out=None, stream=None, flags: int = 0):
        """I float32 [B][npy][npx] on the tensor grid (qx[a], qy[b]) of transverse momentum transfers (CUDA float64 1-D
        tensors): the separable route (scatman_simulate_qgrid).  method: AUTO / TENSOR = both GEMM stages on tcgen05,
        SIMT_TABLE = FP32 CUDA cores."""
        import torch
        self._check_dn(dn)
        for q in (qx, qy):
            if not (q.is_cuda and q.dtype == torch.float64 and q.is_contiguous() and q.dim() == 1):
                raise ValueError("qx, qy must be contiguous 1-D CUDA float64 tensors")
        grid, batch = self._grid_of(dn, voxel), self._batch_of(dn)
        npx, npy = int(qx.numel()), int(qy.numel())
        need = C.c_size_t(0)
        opts = Options(int(rho_mode), int(method), 0, int(flags))
        self._check(self.lib.scatman_qgrid_workspace_bytes(self._ctx, C.byref(grid), npx, npy, batch, C.byref(opts),
                                                           C.byref(need)))
        if workspace is None:
            workspace = self._empty(int(need.value), torch.uint8, dn.device, stream)
        if out is None:
            out = self._empty((batch, npy, npx), torch.float32, dn.device, stream)
        keep, qp = _quat_arg(quat, batch)
        self._check(self.lib.scatman_simulate_qgrid(self._ctx, C.c_void_p(dn.data_ptr()), C.byref(grid), float(lam),
                                                    C.c_void_p(qx.data_ptr()), npx, C.c_void_p(qy.data_ptr()), npy, qp, batch,
                                                    C.byref(opts), C.c_void_p(workspace.data_ptr()), workspace.numel(),
                                                    C.c_void_p(out.data_ptr()), self._stream(stream)))
        return out if dn.dim() == 5 else out[0]

    def _fit_ws(self, npix: int, batch: int, device, stream):
        """Workspace of the fit entry points, kept per (size, stream) so that a fitting loop allocates it once."""
        import torch
        need = C.c_size_t(0)
        self._check(self.lib.scatman_fit_workspace_bytes(self._ctx, npix, batch, C.byref(need)))
        key = (int(need.value), str(device), int(self._stream(stream).value or 0))
        cache = self.__dict__.setdefault("_fit_ws_cache", {})
        if key not in cache:
            cache.clear()
            cache[key] = self._empty(int(need.value), torch.uint8, device, stream)
        return cache[key]

    def discrepancy(self, I, M, mask=None, metric: int = LOSS_L2_NORMALISED, out=None, stream=None):
        """float64 [B]: discrepancy of each simulated pattern I[B][...] (CUDA float32) against the measured pattern M (same
        pixel shape, or [B][...] for one per item); mask: CUDA uint8 per pixel, 0 = ignored (scatman_discrepancy)."""
        import torch
        if not (I.is_cuda and I.dtype == torch.float32 and I.is_contiguous() and I.dim() >= 2):
            raise ValueError("I must be a contiguous CUDA float32 tensor [B][...pixels]")
        batch, npix = int(I.shape[0]), int(I[0].numel())
        if not (M.is_cuda and M.dtype == torch.float32 and M.is_contiguous() and M.numel() in (npix, batch * npix)):
            raise ValueError("M must be a contiguous CUDA float32 tensor with the pixels of one pattern or of every item")
        m_stride = 0 if M.numel() == npix else npix
        if mask is not None and not (mask.is_cuda and mask.dtype == torch.uint8 and mask.is_contiguous() and mask.numel() == npix):
            raise ValueError("mask must be a contiguous CUDA uint8 tensor with one byte per pixel")
        ws = self._fit_ws(npix, batch, I.device, stream)
        if out is None:
            out = self._empty(batch, torch.float64, I.device, stream)
        self._check(self.lib.scatman_discrepancy(self._ctx, C.c_void_p(I.data_ptr()), C.c_void_p(M.data_ptr()), m_stride,
                                                 C.c_void_p(mask.data_ptr()) if mask is not None else None, npix, batch,
                                                 int(metric), C.c_void_p(ws.data_ptr()), ws.numel(), C.c_void_p(out.data_ptr()),
                                                 self._stream(stream)))
        return out

    def discrepancy_static(self, I, M, out, mask=None, metric: int = LOSS_L2_NORMALISED, stream=None):
        """discrepancy() without any allocation: the scratch is the library's static device array of STATIC_SCRATCH_BYTES
        (scatman_discrepancy_static), `out` (CUDA float64 [B]) is the caller's.  Calls share that array: do not overlap them."""
        import torch
        if not (I.is_cuda and I.dtype == torch.float32 and I.is_contiguous() and I.dim() >= 2):
            raise ValueError("I must be a contiguous CUDA float32 tensor [B][...pixels]")
        batch, npix = int(I.shape[0]), int(I[0].numel())
        if not (M.is_cuda and M.dtype == torch.float32 and M.is_contiguous() and M.numel() in (npix, batch * npix)):
            raise ValueError("M must be a contiguous CUDA float32 tensor with the pixels of one pattern or of every item")
        if mask is not None and not (mask.is_cuda and mask.dtype == torch.uint8 and mask.is_contiguous() and mask.numel() == npix):
            raise ValueError("mask must be a contiguous CUDA uint8 tensor with one byte per pixel")
        if not (out.is_cuda and out.dtype == torch.float64 and out.is_contiguous() and out.numel() == batch):
            raise ValueError("out must be a contiguous CUDA float64 tensor [B]")
        self._check(self.lib.scatman_discrepancy_static(self._ctx, C.c_void_p(I.data_ptr()), C.c_void_p(M.data_ptr()),
                                                        0 if M.numel() == npix else npix,
                                                        C.c_void_p(mask.data_ptr()) if mask is not None else None, npix, batch,
                                                        int(metric), C.c_void_p(out.data_ptr()), self._stream(stream)))
        return out

    def ideal_detector(self, I, n_photons, seed: int, out=None, stream=None):
        """float32 counts of I's shape: Poisson(n_photons[b] I[b] / sum I[b]) from the (pixel, item, seed) Philox stream
        (scatman_ideal_detector).  n_photons: a number or one per item."""
        import numpy as np
        import torch
        if not (I.is_cuda and I.dtype == torch.float32 and I.is_contiguous() and I.dim() >= 2):
            raise ValueError("I must be a contiguous CUDA float32 tensor [B][...pixels]")
        batch, npix = int(I.shape[0]), int(I[0].numel())
        ph = np.ascontiguousarray(np.broadcast_to(np.asarray(n_photons, dtype=np.float64), (batch,)))
        ws = self._fit_ws(npix, batch, I.device, stream)
        if out is None:
            out = self._empty(tuple(I.shape), I.dtype, I.device, stream)
        self._check(self.lib.scatman_ideal_detector(self._ctx, C.c_void_p(I.data_ptr()), npix, batch,
                                                    ph.ctypes.data_as(C.POINTER(C.c_double)), C.c_uint64(int(seed) & (2 ** 64 - 1)),
                                                    C.c_void_p(ws.data_ptr()), ws.numel(), C.c_void_p(out.data_ptr()),
                                                    self._stream(stream)))
        return out

    def simulate_host(self, h_dn, voxel, lam: float, npx: int, npy: int, theta_max_deg: float, quat=None,
                      rho_mode: int = RHO_LINEAR, method: int = METHOD_AUTO, h_out=None, flags: int = 0, cx: float = 0.0, cy: float = 0.0):
        """Host-buffer end-to-end call: h_dn / h_out are CPU float32 tensors (pinned for speed). Synchronous."""
        import torch
        if h_dn.is_cuda or h_dn.dtype != torch.float32 or not h_dn.is_contiguous():
            raise ValueError("h_dn must be a contiguous CPU float32 tensor")
        grid, batch = self._grid_of(h_dn, voxel), self._batch_of(h_dn)
        det = Detector(int(npx), int(npy), float(theta_max_deg), float(cx), float(cy))
        opts = Options(int(rho_mode), int(method), 0, int(flags))
        if h_out is None:
            h_out = torch.empty((batch, npy, npx), dtype=torch.float32).pin_memory()
        keep, qp = _quat_arg(quat, batch)
        self._check(self.lib.scatman_simulate_host(self._ctx, C.c_void_p(h_dn.data_ptr()), C.byref(grid), float(lam),
                                                   C.byref(det), qp, batch, C.byref(opts), C.c_void_p(h_out.data_ptr())))
        return h_out

    def simulate_nufft_host(self, h_dn, voxel, lam: float, npx: int, npy: int, theta_max_deg: float, quat=None,
                            rho_mode: int = RHO_LINEAR, h_out=None, cx: float = 0.0, cy: float = 0.0, method: int = METHOD_AUTO):
        """scatman_simulate_nufft_host: host tensors in and out, upload / compute / download overlapped chunk by chunk."""
        import torch
        if h_dn.is_cuda or h_dn.dtype != torch.float32 or not h_dn.is_contiguous():
            raise ValueError("h_dn must be a contiguous CPU float32 tensor")
        grid, batch = self._grid_of(h_dn, voxel), self._batch_of(h_dn)
        det = Detector(int(npx), int(npy), float(theta_max_deg), float(cx), float(cy))
        opts = Options(int(rho_mode), int(method), 0, 0)
        if h_out is None:
            h_out = torch.empty((batch, npy, npx), dtype=torch.float32).pin_memory()
        keep, qp = _quat_arg(quat, batch)
        self._check(self.lib.scatman_simulate_nufft_host(self._ctx, C.c_void_p(h_dn.data_ptr()), C.byref(grid), float(lam),
                                                         C.byref(det), qp, batch, C.byref(opts), C.c_void_p(h_out.data_ptr())))
        return h_out

    def simulate_qgrid_host(self, h_dn, voxel, lam: float, qx, qy, quat=None, rho_mode: int = RHO_LINEAR,
                            method: int = METHOD_AUTO, h_out=None):
        """scatman_simulate_qgrid_host: host tensors in and out; qx, qy are host sequences / numpy arrays of float64."""
        import numpy as np
        import torch
        if h_dn.is_cuda or h_dn.dtype != torch.float32 or not h_dn.is_contiguous():
            raise ValueError("h_dn must be a contiguous CPU float32 tensor")
        grid, batch = self._grid_of(h_dn, voxel), self._batch_of(h_dn)
        qx = np.ascontiguousarray(np.asarray(qx, dtype=np.float64))
        qy = np.ascontiguousarray(np.asarray(qy, dtype=np.float64))
        npx, npy = int(qx.size), int(qy.size)
        opts = Options(int(rho_mode), int(method), 0, 0)
        if h_out is None:
            h_out = torch.empty((batch, npy, npx), dtype=torch.float32).pin_memory()
        keep, qp = _quat_arg(quat, batch)
        self._check(self.lib.scatman_simulate_qgrid_host(self._ctx, C.c_void_p(h_dn.data_ptr()), C.byref(grid), float(lam),
                                                         qx.ctypes.data_as(C.POINTER(C.c_double)), npx,
                                                         qy.ctypes.data_as(C.POINTER(C.c_double)), npy, qp, batch, C.byref(opts),
                                                         C.c_void_p(h_out.data_ptr())))
        return h_out

    def last_launch_count(self) -> int:
        n = C.c_int32(0)
        self._check(self.lib.scatman_last_launch_count(self._ctx, C.byref(n)))
        return int(n.value)

    def last_issued_blocks(self) -> int:
        n = C.c_int64(-1)
        self._check(self.lib.scatman_last_issued_blocks(self._ctx, C.byref(n)))
        return int(n.value)

    def last_contraction_ms(self) -> float:
        ms = C.c_float(0)
        self._check(self.lib.scatman_last_contraction_ms(self._ctx, C.byref(ms)))
        return float(ms.value)
