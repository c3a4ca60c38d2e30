"""Pins for the oracle's scatter denoiser (paper Eq. (5)) against things other than itself:
one sweep written out independently in numpy slicing, the fixed point of a constant image, the closed-form
amplification factor of the cosine eigenmodes of the replicate-boundary Laplacian (first order), and the
optimality condition Eq. (4) plus its summed form at convergence."""
import math

import numpy as np
import pytest

import oracle

OMEGA = 0.8


def numpy_sweep(s, s_hat, beta, omega=OMEGA):
    p = np.pad(s, 1, mode="edge")                              # replicate boundary [Q28]
    total = p[1:-1, 2:] + p[2:, 1:-1] + p[1:-1, :-2] + p[:-2, 1:-1]
    return (1 - omega) * s + omega / 4 * (total - (1 - s_hat / s) / beta)


def test_d1_one_and_three_sweeps_against_numpy_slicing():
    rng = np.random.default_rng(1)
    s_hat = rng.poisson(40.0, size=(7, 9)).astype(float) + 1.0
    ref = s_hat.copy()
    for k in range(1, 4):
        ref = numpy_sweep(ref, s_hat, beta=0.3)
        np.testing.assert_allclose(oracle.denoise(s_hat, beta=0.3, n_iter=k), ref, rtol=1e-13)
    assert np.array_equal(oracle.denoise(s_hat, beta=0.3, n_iter=0), s_hat)     # S(0) = S_hat


def test_d2_constant_image_is_a_fixed_point():
    s_hat = np.full((6, 5), 17.25)
    assert np.array_equal(oracle.denoise(s_hat, beta=0.7, n_iter=11), s_hat)


@pytest.mark.parametrize("p,q", [(0, 1), (2, 0), (3, 2), (5, 4)])
def test_d3_eigenmode_amplification_factor(p, q):
    """S_hat = c, S(0) = c + eps cos(pi p (i + 1/2) / nu) cos(pi q (j + 1/2) / nv): these modes are eigenvectors
    of the 5-point sum with replicated edges (eigenvalue 2 cos(pi p / nu) + 2 cos(pi q / nv)), and to first order
    1 - c / (c + e) = e / c, so one sweep multiplies the mode by g = 1 - w + w/4 (lambda - 1 / (beta c))."""
    nu, nv, c, beta, eps = 12, 10, 30.0, 0.05, 1e-6
    i, j = np.arange(nu)[None, :], np.arange(nv)[:, None]
    mode = np.cos(math.pi * p * (i + 0.5) / nu) * np.cos(math.pi * q * (j + 0.5) / nv)
    out = oracle.denoise(np.full((nv, nu), c), beta=beta, n_iter=1, s0=c + eps * mode)
    lam = 2 * math.cos(math.pi * p / nu) + 2 * math.cos(math.pi * q / nv)
    g = 1 - OMEGA + OMEGA / 4 * (lam - 1 / (beta * c))
    np.testing.assert_allclose((out - c) / eps, g * mode, atol=5e-6)


def test_d4_converged_image_satisfies_eq4_and_its_sum():
    rng = np.random.default_rng(4)
    i, j = np.arange(40)[None, :], np.arange(32)[:, None]
    truth = 50 + 30 * np.exp(-((i - 18) ** 2 + (j - 12) ** 2) / 150.0)
    s_hat = rng.poisson(truth).astype(float)
    beta = 0.2
    s = oracle.denoise(s_hat, beta=beta, n_iter=4000)
    p = np.pad(s, 1, mode="edge")
    lap = p[1:-1, 2:] + p[2:, 1:-1] + p[1:-1, :-2] + p[:-2, 1:-1] - 4 * s
    residual = (1 - s_hat / s) - beta * lap                     # Eq. (4)
    assert np.abs(residual).max() < 1e-9
    assert abs((s_hat / s).sum() - s.size) < 1e-6               # Eq. (4) summed: the Laplacian sums to 0
    assert np.abs(np.diff(s, axis=1)).sum() < 0.3 * np.abs(np.diff(s_hat, axis=1)).sum()     # smoother
    assert np.abs(s - truth).mean() < 0.6 * np.abs(s_hat - truth).mean()                     # and closer to the mean


def test_d5_floor_keeps_empty_pixels_defined():
    s_hat = np.zeros((5, 5)); s_hat[2, 2] = 9.0
    out = oracle.denoise(s_hat, beta=1.0, n_iter=50, floor=1e-3)
    assert np.all(np.isfinite(out)) and out.min() >= 1e-3
    with pytest.raises(ValueError):
        oracle.denoise(s_hat, beta=0.0, n_iter=1)


def test_denoise_golden_regression():
    """tests/golden/oracle_denoise_regression.txt (written by tests/golden/make_golden.py from oracle/ only)."""
    import os
    path = os.path.join(os.path.dirname(__file__), "golden", "oracle_denoise_regression.txt")
    want = np.array([[float(x) for x in l.split()] for l in open(path) if not l.startswith("#")])
    rng = np.random.default_rng(12046367)
    img = rng.poisson(30.0, size=(6, 8)).astype(np.float64) + 1.0
    np.testing.assert_allclose(oracle.denoise(img, beta=0.25, n_iter=7), want, rtol=1e-13)
