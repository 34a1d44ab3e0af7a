"""FP64 CPU oracle of shape rendering (Block 5 of Fig. 4: "render the slice at the proper spatial
coordinates"; shape models of section 5).  TEST INFRASTRUCTURE ONLY: nothing in the
product path may import this module.

A shape is rendered directly in the beam frame: voxel centre r_beam (centred coordinates, R6) is taken to
the body frame, r_body = R^T r_beam (R = rotation of the unit quaternion body -> beam, R11), and the voxel
is (delta, beta) if r_body lies inside the shape, else vacuum (0, 0): binary voxelisation at voxel centres, like
PyScatman's boolean VolumeMap.  Everything is plain numpy in float64, no blocking, no shortcuts.

Readings (R18-R21):
  * Ellipsoid(a, b, c): (x/a)^2 + (y/b)^2 + (z/c)^2 <= 1, semi-axes along body x, y, z.
  * SphericalHarmonics([[l, m, c], ...]): R(theta, phi) = sum of c * Y_lm ("the final shape is the sum of
    all triplets"), theta = polar angle from body +z (the North-South axis), phi = atan2(y, x).
    Y_l^m of Eq. 10 is complex while a radius is real and the scaling parameter is a real number; the
    reading is the REAL orthonormal combinations: m = 0: Y_l^0 of Eq. 10; m > 0: sqrt(2) Re Y_l^m = sqrt(2) N_lm P_l^m(cos theta) cos(m phi);
    m < 0: sqrt(2) Im Y_l^|m| = sqrt(2) N_l|m| P_l^|m|(cos theta) sin(|m| phi), N_lm and P_l^m (Condon-Shortley phase)
    as in Eq. 10.  Inside: |r| <= R(theta, phi).
  * RadialMap(radii[nlat][nlon]): sample (i, j) holds the radius at latitude -pi/2 + i pi/nlat and longitude
    j 2pi/nlon (the paper's 4 x 4 example: theta = -pi/2, -pi/4, 0, pi/4 and phi = 0, pi/2, pi, 3pi/2);
    "linearly interpolated": bilinear, periodic in longitude, latitudes above the last sample hold the last row.
    latitude = asin(z/|r|), longitude = atan2(y, x) mod 2pi.  Inside: |r| <= R(lat, lon).
  * VolumeMap(vol[nvz][nvy][nvx] bool, dx): a block of cubic cells of side dx centred on the origin; inside if the
    cell containing r_body is True (a 10^3 all-True array with dx = 2 is a 20 x 20 x 20 cube).
"""
from __future__ import annotations

from math import factorial, pi, sqrt

import numpy as np


def rotation_matrix(quat) -> np.ndarray:
    """Row-major R (body -> beam) of a unit quaternion (w, x, y, z)."""
    w, a, b, c = (float(v) for v in quat)
    return np.array([[1 - 2 * (b * b + c * c), 2 * (a * b - w * c), 2 * (a * c + w * b)],
                     [2 * (a * b + w * c), 1 - 2 * (a * a + c * c), 2 * (b * c - w * a)],
                     [2 * (a * c - w * b), 2 * (b * c + w * a), 1 - 2 * (a * a + b * b)]], dtype=np.float64)


def body_coordinates(dims, voxel, quat=None):
    """r_body = R^T r_beam of every voxel centre; three float64 arrays [nz][ny][nx]."""
    nx, ny, nz = dims
    dx, dy, dz = voxel
    x = ((np.arange(nx, dtype=np.float64) - 0.5 * (nx - 1)) * dx)[None, None, :]
    y = ((np.arange(ny, dtype=np.float64) - 0.5 * (ny - 1)) * dy)[None, :, None]
    z = ((np.arange(nz, dtype=np.float64) - 0.5 * (nz - 1)) * dz)[:, None, None]
    if quat is None:
        shape = (nz, ny, nx)
        return np.broadcast_to(x, shape), np.broadcast_to(y, shape), np.broadcast_to(z, shape)
    R = rotation_matrix(quat)
    xb = R[0, 0] * x + R[1, 0] * y + R[2, 0] * z
    yb = R[0, 1] * x + R[1, 1] * y + R[2, 1] * z
    zb = R[0, 2] * x + R[1, 2] * y + R[2, 2] * z
    return xb, yb, zb


def legendre_p(l: int, m: int, x: np.ndarray) -> np.ndarray:
    """Associated Legendre function P_l^m(x), m >= 0, with the Condon-Shortley phase (Eq. 10's P_l^m), by the
    standard recurrences: P_m^m = (-1)^m (2m-1)!! (1-x^2)^(m/2), P_{m+1}^m = x (2m+1) P_m^m,
    (l-m) P_l^m = (2l-1) x P_{l-1}^m - (l+m-1) P_{l-2}^m."""
    x = np.asarray(x, dtype=np.float64)
    s = np.sqrt(np.maximum(0.0, 1.0 - x * x))
    pmm = np.ones_like(x)
    for k in range(1, m + 1):
        pmm = -pmm * (2 * k - 1) * s
    if l == m:
        return pmm
    pm1 = x * (2 * m + 1) * pmm
    if l == m + 1:
        return pm1
    for ll in range(m + 2, l + 1):
        pmm, pm1 = pm1, ((2 * ll - 1) * x * pm1 - (ll + m - 1) * pmm) / (ll - m)
    return pm1


def real_sph_harm(l: int, m: int, cos_theta: np.ndarray, phi: np.ndarray) -> np.ndarray:
    """Real orthonormal Y_lm (module docstring): Eq. 10's normalisation N_lm = sqrt((2l+1)/(4pi) (l-|m|)!/(l+|m|)!)."""
    am = abs(m)
    n = sqrt((2 * l + 1) / (4 * pi) * factorial(l - am) / factorial(l + am))
    p = legendre_p(l, am, cos_theta)
    if m == 0:
        return n * p
    if m > 0:
        return sqrt(2.0) * n * p * np.cos(am * phi)
    return sqrt(2.0) * n * p * np.sin(am * phi)


def sh_radius(coeffs, cos_theta, phi) -> np.ndarray:
    """R(theta, phi) = sum over triplets (l, m, c) of c * Y_lm."""
    out = np.zeros(np.broadcast(cos_theta, phi).shape, dtype=np.float64)
    for (l, m, c) in coeffs:
        out = out + float(c) * real_sph_harm(int(l), int(m), cos_theta, phi)
    return out


def radial_map_radius(radii: np.ndarray, lat: np.ndarray, lon: np.ndarray) -> np.ndarray:
    """Bilinear lookup of radii[nlat][nlon] at latitude lat in [-pi/2, pi/2] and longitude lon in [0, 2pi)."""
    radii = np.asarray(radii, dtype=np.float64)
    nlat, nlon = radii.shape
    fi = np.clip((np.asarray(lat, dtype=np.float64) + 0.5 * pi) / (pi / nlat), 0.0, float(nlat - 1))
    fj = np.asarray(lon, dtype=np.float64) / (2.0 * pi / nlon)
    i0 = np.minimum(np.floor(fi).astype(np.int64), nlat - 1)
    i1 = np.minimum(i0 + 1, nlat - 1)
    ti = fi - i0
    j0f = np.floor(fj)
    tj = fj - j0f
    j0 = np.mod(j0f.astype(np.int64), nlon)
    j1 = np.mod(j0 + 1, nlon)
    lo = radii[i0, j0] * (1.0 - tj) + radii[i0, j1] * tj
    hi = radii[i1, j0] * (1.0 - tj) + radii[i1, j1] * tj
    return lo * (1.0 - ti) + hi * ti


# ------------------------------------------------------------------------------------------------ inside tests
# Each returns (inside, margin): margin = signed distance-like quantity whose sign decides (inside = margin <= 0 or
# >= 0 as stated), so that a test can tell a genuine mismatch from a rounding tie at the surface.
def inside_ellipsoid(xb, yb, zb, a, b, c):
    v = (xb / a) ** 2 + (yb / b) ** 2 + (zb / c) ** 2
    return v <= 1.0, v - 1.0


def inside_spherical_harmonics(xb, yb, zb, coeffs):
    r = np.sqrt(xb * xb + yb * yb + zb * zb)
    ct = np.where(r > 0.0, zb / np.where(r > 0.0, r, 1.0), 1.0)
    ph = np.arctan2(yb, xb)
    R = sh_radius(coeffs, ct, ph)
    return r <= R, r - R


def inside_radial_map(xb, yb, zb, radii):
    r = np.sqrt(xb * xb + yb * yb + zb * zb)
    lat = np.arcsin(np.clip(np.where(r > 0.0, zb / np.where(r > 0.0, r, 1.0), 0.0), -1.0, 1.0))
    lon = np.arctan2(yb, xb)
    lon = np.where(lon < 0.0, lon + 2.0 * pi, lon)
    R = radial_map_radius(radii, lat, lon)
    return r <= R, r - R


def inside_volume_map(xb, yb, zb, vol, dx):
    vol = np.asarray(vol).astype(bool)
    nvz, nvy, nvx = vol.shape
    fx = xb / dx + 0.5 * nvx
    fy = yb / dx + 0.5 * nvy
    fz = zb / dx + 0.5 * nvz
    ix, iy, iz = np.floor(fx).astype(np.int64), np.floor(fy).astype(np.int64), np.floor(fz).astype(np.int64)
    ok = (ix >= 0) & (ix < nvx) & (iy >= 0) & (iy < nvy) & (iz >= 0) & (iz < nvz)
    inside = np.zeros(ok.shape, dtype=bool)
    inside[ok] = vol[iz[ok], iy[ok], ix[ok]]
    # margin: distance (in cells) of the nearest coordinate to a cell face
    edge = np.minimum(np.minimum(np.abs(fx - np.round(fx)), np.abs(fy - np.round(fy))), np.abs(fz - np.round(fz)))
    return inside, edge


def render(shape: dict, dims, voxel, return_margin: bool = False):
    """(delta, beta) grid float32 [nz][ny][nx][2] of one shape.  shape = {"kind": "ellipsoid" | "spherical_harmonics" |
    "radial_map" | "volume_map", "delta", "beta", "quat" (optional), and the kind's own parameters}."""
    xb, yb, zb = body_coordinates(dims, voxel, shape.get("quat"))
    kind = shape["kind"]
    if kind == "ellipsoid":
        inside, margin = inside_ellipsoid(xb, yb, zb, shape["a"], shape["b"], shape["c"])
    elif kind == "spherical_harmonics":
        inside, margin = inside_spherical_harmonics(xb, yb, zb, shape["coeffs"])
    elif kind == "radial_map":
        inside, margin = inside_radial_map(xb, yb, zb, shape["radii"])
    elif kind == "volume_map":
        inside, margin = inside_volume_map(xb, yb, zb, shape["volume"], shape["dx"])
    else:
        raise ValueError(kind)
    nx, ny, nz = dims
    out = np.zeros((nz, ny, nx, 2), dtype=np.float32)
    out[..., 0] = np.where(inside, np.float32(shape["delta"]), np.float32(0.0))
    out[..., 1] = np.where(inside, np.float32(shape["beta"]), np.float32(0.0))
    return (out, np.broadcast_to(margin, (nz, ny, nx))) if return_margin else out
