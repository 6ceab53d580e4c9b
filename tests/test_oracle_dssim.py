"""Pins of the oracle's D-SSIM term (Eq. 8; reading S25): identity, the closed form on constant
images, bounds and symmetry, central finite differences of the gradient, and a cross-check of the window sums against
scipy's correlation with the same Gaussian window (a library routine, not the oracle's loops)."""
import numpy as np
import pytest

C1, C2 = 0.01 ** 2, 0.03 ** 2


def test_identical_images_have_zero_loss_and_zero_gradient(oracle_mod):
    rng = np.random.default_rng(0)
    x = rng.uniform(0, 1, (3, 20, 23))
    L, g = oracle_mod.dssim(x, x)
    assert abs(L) < 1e-12 and np.abs(g).max() < 1e-12


def test_constant_images_closed_form(oracle_mod):
    # constant a against constant b: variances vanish; with zero padding the window mass m(p) < 1 near the border
    # scales both means, so ssim(p) = (2 m^2 a b + C1) / (m^2 (a^2 + b^2) + C1) everywhere
    a, b, H, W = 0.7, 0.4, 17, 19
    g1 = np.exp(-((np.arange(11) - 5.0) ** 2) / (2 * 1.5 ** 2))
    g1 /= g1.sum()
    my = np.array([g1[max(0, 5 - y):min(11, 5 + H - y)].sum() for y in range(H)])
    mx = np.array([g1[max(0, 5 - x):min(11, 5 + W - x)].sum() for x in range(W)])
    m = np.outer(my, mx)
    # E[x^2] = m a^2 but mu^2 = m^2 a^2: the "variance" of a constant under an un-normalised window is m(1-m)a^2
    s11, s22, s12 = m * (1 - m) * a * a, m * (1 - m) * b * b, m * (1 - m) * a * b
    ssim = ((2 * m * m * a * b + C1) * (2 * s12 + C2)) / ((m * m * (a * a + b * b) + C1) * (s11 + s22 + C2))
    L, _ = oracle_mod.dssim(np.full((3, H, W), a), np.full((3, H, W), b), grad=False)
    assert abs(L - (1 - ssim.mean())) < 1e-12
    assert abs(ssim[8, 9] - (2 * a * b + C1) / (a * a + b * b + C1)) < 1e-6     # interior: the textbook value


def test_bounds_and_symmetry(oracle_mod):
    rng = np.random.default_rng(1)
    x, y = rng.uniform(0, 1, (3, 16, 18)), rng.uniform(0, 1, (3, 16, 18))
    Lxy, _ = oracle_mod.dssim(x, y, grad=False)
    Lyx, _ = oracle_mod.dssim(y, x, grad=False)
    assert abs(Lxy - Lyx) < 1e-13 and 0 < Lxy < 2
    L32, _ = oracle_mod.dssim(x, y, "f32", grad=False)
    assert abs(L32 - Lxy) < 1e-5


def test_gradient_matches_central_differences(oracle_mod):
    rng = np.random.default_rng(2)
    x, y = rng.uniform(0.1, 0.9, (3, 14, 15)), rng.uniform(0.1, 0.9, (3, 14, 15))
    L, g = oracle_mod.dssim(x, y)
    h = 1e-6
    for _ in range(40):
        c, i, j = rng.integers(3), rng.integers(14), rng.integers(15)
        xp, xm = x.copy(), x.copy()
        xp[c, i, j] += h
        xm[c, i, j] -= h
        fd = (oracle_mod.dssim(xp, y, grad=False)[0] - oracle_mod.dssim(xm, y, grad=False)[0]) / (2 * h)
        assert abs(fd - g[c, i, j]) <= 1e-7 + 1e-5 * abs(fd)
    # a random direction in the whole image
    d = rng.normal(size=x.shape)
    fd = (oracle_mod.dssim(x + h * d, y, grad=False)[0] - oracle_mod.dssim(x - h * d, y, grad=False)[0]) / (2 * h)
    assert abs(fd - (g * d).sum()) <= 1e-7 + 1e-5 * abs(fd)


def test_window_sums_against_scipy(oracle_mod):
    # mean SSIM rebuilt from scipy.ndimage.correlate with the separable 11-tap Gaussian, zero padding
    from scipy.ndimage import correlate1d
    rng = np.random.default_rng(3)
    x, y = rng.uniform(0, 1, (3, 21, 20)), rng.uniform(0, 1, (3, 21, 20))
    g1 = np.exp(-((np.arange(11) - 5.0) ** 2) / (2 * 1.5 ** 2))
    g1 /= g1.sum()
    blur = lambda a: correlate1d(correlate1d(a, g1, axis=1, mode="constant"), g1, axis=2, mode="constant")
    mu1, mu2 = blur(x), blur(y)
    s11, s22, s12 = blur(x * x) - mu1 ** 2, blur(y * y) - mu2 ** 2, blur(x * y) - mu1 * mu2
    ssim = ((2 * mu1 * mu2 + C1) * (2 * s12 + C2)) / ((mu1 ** 2 + mu2 ** 2 + C1) * (s11 + s22 + C2))
    L, _ = oracle_mod.dssim(x, y, grad=False)
    assert abs(L - (1 - ssim.mean())) < 1e-12
