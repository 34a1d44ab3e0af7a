"""ctypes front-end of oracle/msft_oracle.c (FP64 CPU oracle; TEST INFRASTRUCTURE ONLY).

Every function cites the passage it follows in msft_oracle.c.  Arrays are numpy; the grid is
float32 [nz][ny][nx][2] = (delta, beta) in the paper's sense (Eq. 7).
"""
from __future__ import annotations

import ctypes as C
from typing import Optional

import numpy as np

from . import build as _build

RHO_LINEAR = 0
RHO_N2M1 = 1

_lib = None


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(_build.build())
        dp, fp = C.POINTER(C.c_double), C.POINTER(C.c_float)
        L.oracle_num_threads.restype = C.c_int
        L.oracle_qmap.argtypes = [C.c_int, C.c_int, C.c_double, C.c_double, C.c_double, C.c_double, dp]
        L.oracle_orient.argtypes = [fp, C.c_int, C.c_int, C.c_int, C.c_double, C.c_double, C.c_double, dp, fp]
        L.oracle_effective_strength.argtypes = [fp, C.c_int, C.c_int, C.c_int, C.c_double, C.c_double, C.c_double,
                                                C.c_double, C.c_int, dp]
        for f in (L.oracle_amplitude_direct, L.oracle_amplitude_tables):
            f.argtypes = [dp, C.c_int, C.c_int, C.c_int, C.c_double, C.c_double, C.c_double, dp, C.c_int64, dp]
        L.oracle_simulate_q.argtypes = [fp, C.c_int, C.c_int, C.c_int, C.c_double, C.c_double, C.c_double,
                                        C.c_double, dp, C.c_int, dp, C.c_int64, C.c_int, dp, dp]
        L.oracle_simulate_q.restype = C.c_int
        _lib = L
    return _lib


def _d(a):
    return a.ctypes.data_as(C.POINTER(C.c_double))


def _f(a):
    return a.ctypes.data_as(C.POINTER(C.c_float))


def num_threads() -> int:
    return int(lib().oracle_num_threads())


def qmap(npx: int, npy: int, theta_max_deg: float, lam: float, cx: float = 0.0, cy: float = 0.0) -> np.ndarray:
    """Ewald-sphere q of every pixel of the flat detector, float64 [npy*npx][3] (Eq. 3)."""
    q = np.empty((npx * npy, 3), dtype=np.float64)
    lib().oracle_qmap(npx, npy, float(theta_max_deg), float(cx), float(cy), float(lam), _d(q))
    return q


def _grid(dn: np.ndarray):
    dn = np.ascontiguousarray(dn, dtype=np.float32)
    assert dn.ndim == 4 and dn.shape[3] == 2, "grid must be [nz][ny][nx][2]"
    nz, ny, nx, _ = dn.shape
    return dn, nx, ny, nz


def orient(dn: np.ndarray, voxel, quat) -> np.ndarray:
    """Beam-frame grid = trilinear resample of the body-frame grid (Block 5; Fig. 6)."""
    dn, nx, ny, nz = _grid(dn)
    out = np.empty_like(dn)
    qa = np.ascontiguousarray(quat, dtype=np.float64)
    lib().oracle_orient(_f(dn), nx, ny, nz, *map(float, voxel), _d(qa), _f(out))
    return out


def effective_strength(dn: np.ndarray, voxel, lam: float, rho_mode: int = RHO_LINEAR) -> np.ndarray:
    """rho~_j(x,y) dV as complex128 [nz][ny][nx] (Eq. 6/8/9)."""
    dn, nx, ny, nz = _grid(dn)
    rho = np.empty((nz, ny, nx, 2), dtype=np.float64)
    lib().oracle_effective_strength(_f(dn), nx, ny, nz, *map(float, voxel), float(lam), int(rho_mode), _d(rho))
    return rho[..., 0] + 1j * rho[..., 1]


def amplitude(rho: np.ndarray, voxel, q: np.ndarray, method: str = "tables") -> np.ndarray:
    """A(p) = sum_j sum_y sum_x rho e^{i q.r} at the rows of q (Eq. 2)."""
    nz, ny, nx = rho.shape
    r2 = np.ascontiguousarray(np.stack([rho.real, rho.imag], axis=-1), dtype=np.float64)
    q = np.ascontiguousarray(q, dtype=np.float64).reshape(-1, 3)
    A = np.empty((q.shape[0], 2), dtype=np.float64)
    fn = lib().oracle_amplitude_direct if method == "direct" else lib().oracle_amplitude_tables
    fn(_d(r2), nx, ny, nz, *map(float, voxel), _d(q), q.shape[0], _d(A))
    return A[:, 0] + 1j * A[:, 1]


def simulate_q(dn: np.ndarray, voxel, lam: float, q: np.ndarray, quat=None, rho_mode: int = RHO_LINEAR,
               method: str = "tables", return_amplitude: bool = False):
    """Whole path for one grid at an explicit q list -> I float64 [npix] (and A complex128)."""
    dn, nx, ny, nz = _grid(dn)
    q = np.ascontiguousarray(q, dtype=np.float64).reshape(-1, 3)
    n = q.shape[0]
    I = np.empty(n, dtype=np.float64)
    A = np.empty((n, 2), dtype=np.float64)
    qa = None if quat is None else np.ascontiguousarray(quat, dtype=np.float64)
    rc = lib().oracle_simulate_q(_f(dn), nx, ny, nz, *map(float, voxel), float(lam),
                                 None if qa is None else _d(qa), int(rho_mode), _d(q), n,
                                 1 if method == "direct" else 0, _d(I), _d(A))
    if rc != 0:
        raise MemoryError("oracle_simulate_q failed")
    return (I, A[:, 0] + 1j * A[:, 1]) if return_amplitude else I


def simulate(dn: np.ndarray, voxel, lam: float, npx: int, npy: int, theta_max_deg: float, quat=None,
             rho_mode: int = RHO_LINEAR, pixels: Optional[np.ndarray] = None, method: str = "tables",
             cx: float = 0.0, cy: float = 0.0) -> np.ndarray:
    """I on the flat detector: float64 [npy][npx], or [len(pixels)] for a pixel subset."""
    q = qmap(npx, npy, theta_max_deg, lam, cx, cy)
    if pixels is not None:
        return simulate_q(dn, voxel, lam, q[np.asarray(pixels)], quat, rho_mode, method)
    return simulate_q(dn, voxel, lam, q, quat, rho_mode, method).reshape(npy, npx)


def qgrid_q(qx: np.ndarray, qy: np.ndarray, lam: float):
    """Momentum transfers of a tensor-grid detector: pixel (b, a) has transverse components (qx[a], qy[b]) and lies on the
    Ewald sphere, |q + k z^| = k (Eq. 3-4; the paper's q = k0 - k has qz = k0 (1 - cos theta) >= 0, north_star's
    q = k (s^ - z^) has the opposite sign): qz = -(k - sqrt(k^2 - qx^2 - qy^2)).  Returns (q float64 [npy*npx][3], propagating
    bool [npy*npx]); points with qx^2 + qy^2 > k^2 have no scattering direction (propagating False, qz set to 0)."""
    qx = np.asarray(qx, dtype=np.float64)
    qy = np.asarray(qy, dtype=np.float64)
    k = 2.0 * np.pi / float(lam)
    QX, QY = np.meshgrid(qx, qy, indexing="xy")          # [npy][npx]
    kz2 = k * k - QX * QX - QY * QY
    ok = kz2 >= 0.0
    qz = np.where(ok, -(k - np.sqrt(np.where(ok, kz2, 0.0))), 0.0)
    q = np.stack([QX.ravel(), QY.ravel(), qz.ravel()], axis=1)
    return q, ok.ravel()


def simulate_qgrid(dn: np.ndarray, voxel, lam: float, qx, qy, quat=None, rho_mode: int = RHO_LINEAR) -> np.ndarray:
    """Whole path on a tensor-grid detector: the same direct triple sum, at qgrid_q's points; I = 0 where nothing propagates.
    float64 [npy][npx]."""
    q, ok = qgrid_q(qx, qy, lam)
    I = simulate_q(dn, voxel, lam, q, quat, rho_mode)
    return np.where(ok, I, 0.0).reshape(len(np.atleast_1d(qy)), len(np.atleast_1d(qx)))
