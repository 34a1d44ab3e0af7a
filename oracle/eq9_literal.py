"""The paper's Eq. 9 / Fig. 4 main loop, followed LITERALLY in the paper's order, notation and
sign convention (numpy, FP64; TEST INFRASTRUCTURE ONLY).

PAPER.md:127-131 (Eq. 9), Blocks 4-11:

    out = 0 ; E = E_0 = 1                                   Block 4
    for s in 0..S-1:
        slice_n  = 1 - delta_s + i beta_s                   Block 5 (Eq. 7)
        F        = DFT[(slice_n^2 - 1) * E](q_x, q_y)       Block 6 (direct sum at the given q)
        F       *= exp(-i sqrt(k0^2 - q_x^2 - q_y^2) s dz)  Block 7 (R5 for the garbled exponent)
        out     += F                                        Block 8
        E        = E * exp(i k0 dz slice_n)                 Block 9 (Eq. 8; keeps the vacuum phase)
    I = |out|^2                                             Block 11

The paper's momentum transfer is q = k_0 - k (Fig. 3 caption), the opposite sign of
north_star's q = k(s - z^); pass q_paper = -q_northstar.  `strength="n-1"` replaces n^2-1 by
n-1 (the north_star's linear contrast).  Positions are the oracle's centred x, y and z_s = s dz
for the slices (the paper's slice origin): origin shifts are unit phase factors (R6).
"""
from __future__ import annotations

import numpy as np


def eq9_field(dn: np.ndarray, voxel, lam: float, q_paper: np.ndarray, strength: str = "n2-1") -> np.ndarray:
    dn = np.asarray(dn, dtype=np.float64)
    nz, ny, nx, _ = dn.shape
    dx, dy, dz = voxel
    k0 = 2.0 * np.pi / lam
    x = (np.arange(nx) - (nx - 1) / 2.0) * dx
    y = (np.arange(ny) - (ny - 1) / 2.0) * dy
    qx, qy = q_paper[:, 0], q_paper[:, 1]
    kz = np.sqrt(k0 ** 2 - qx ** 2 - qy ** 2)
    out = np.zeros(q_paper.shape[0], dtype=np.complex128)          # Block 4
    E = np.ones((ny, nx), dtype=np.complex128)
    ex = np.exp(1j * np.outer(qx, x))                               # e^{i q_x x}
    ey = np.exp(1j * np.outer(qy, y))
    for s in range(nz):
        n_s = 1.0 - dn[s, :, :, 0] + 1j * dn[s, :, :, 1]            # Block 5, Eq. 7
        src = (n_s ** 2 - 1.0 if strength == "n2-1" else n_s - 1.0) * E
        F = np.einsum("py,yx,px->p", ey, src, ex)                   # Block 6
        F = F * np.exp(-1j * kz * s * dz)                           # Block 7
        out += F                                                    # Block 8
        E = E * np.exp(1j * k0 * dz * n_s)                          # Block 9, Eq. 8
    return out * (dx * dy * dz)
