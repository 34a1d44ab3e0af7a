"""The error bound DESIGN.md (R25, section 5) states for the NUFFT route's window, checked with numpy / scipy alone (no CUDA, no oracle):
e^{i u t} = (1 / Phi(t)) sum_m phi(u - m) e^{i m t} up to the aliases, for the Kaiser-Bessel window of 8 cells at oversampling 2
(|t| <= pi / 2), and the degree-11 per-cell polynomials reproduce the window to 1e-12."""
import numpy as np
from scipy.special import i0

W = 8
HALF = W / 2.0
BETA = np.pi * np.sqrt(HALF * HALF * 2.25 - 0.8)


def phi(s):
    a = 1.0 - (s / HALF) ** 2
    return np.where(a >= 0, i0(BETA * np.sqrt(np.maximum(a, 0.0))) / i0(BETA), 0.0)


def Phi(t):
    r = np.sqrt(BETA ** 2 - (HALF * t) ** 2)
    return 2.0 * HALF * np.sinh(r) / (i0(BETA) * r)


def test_window_identity_error_is_below_the_stated_bound():
    rng = np.random.default_rng(220203411)
    worst = 0.0
    for _ in range(4000):
        u = rng.uniform(-200.0, 200.0)
        t = rng.uniform(-np.pi / 2, np.pi / 2)
        if rng.random() < 0.3:                       # the edge voxels of the box are the worst case
            t = np.sign(t) * np.pi / 2 * (1.0 - 1e-3 * rng.random())
        m0 = int(np.ceil(u - HALF))
        m = np.arange(m0, m0 + W)
        approx = np.sum(phi(u - m) * np.exp(1j * m * t)) / Phi(t)
        worst = max(worst, abs(approx - np.exp(1j * u * t)))
    assert worst <= 4e-7, worst   # 2.4e-7 measured; three factors per voxel -> 7e-7 of sum |rho~|, below the 1e-3 per-pixel tolerance at 1e-6 of the peak


def test_Phi_is_the_windows_fourier_transform():
    s = np.linspace(-HALF, HALF, 200001)
    for t in (0.0, 0.7, -1.3, np.pi / 2):
        f = phi(s) * np.cos(s * t)
        num = float(np.sum(0.5 * (f[1:] + f[:-1]) * np.diff(s)))
        assert abs(num - Phi(t)) <= 1e-8 * Phi(0.0)


def test_per_cell_polynomials_of_degree_11_reproduce_the_window():
    n = 12
    xk = np.cos(np.pi * (np.arange(n) + 0.5) / n)
    t = np.linspace(0.0, 1.0, 1001)[:-1]
    for c in range(W):
        f = phi(HALF - c - 0.5 * (xk + 1.0))
        cheb = np.array([(2.0 / n) * np.sum(f * np.cos(j * np.pi * (np.arange(n) + 0.5) / n)) for j in range(n)])
        cheb[0] *= 0.5
        y = np.polynomial.chebyshev.chebval(2.0 * t - 1.0, cheb)
        assert np.max(np.abs(y - phi(HALF - c - t))) <= 1e-12
