"""Pin P23: the `min` face-opacity variant ("routes gradients solely to the vertex with
the lowest opacity"; "+ min opacity" row of Table S3) of the oracle."""
import numpy as np

from conftest import IDENT, SimpleCam, SimpleParams, unproject
from test_oracle_gradients import small_scene


def test_p23_closed_form_and_gradient_routing(oracle_mod):
    """The 30-40-50 screen triangle with vertex opacities (0.9, 0.6, 0.3): alpha at the incentre is 0.6 (mean) or 0.3
    (min); with a single face dL/dalpha does not depend on the mode when only A carries a cotangent, so the whole
    min-mode gradient on the third vertex is three times one of the equal mean-mode thirds."""
    cam = SimpleCam(64, 48, 60.0, 60.0, 0.0, 0.0)
    pos = unproject([(6.0, 6.0, 2.0), (46.0, 6.0, 2.0), (6.0, 36.0, 2.0)], cam)     # incentre (16,16), r = 10
    col, opa = np.ones((3, 3)), np.array([0.9, 0.6, 0.3])
    a = {}
    for mode in (False, True):
        prm = SimpleParams(sigma=1.0, min_opacity=mode)
        o = oracle_mod.Oracle(pos, col, opa, None, IDENT, cam, prm, "f64")
        f = o.forward()
        a[mode] = f.alpha
        assert abs(f.alpha[16, 16] - (0.3 if mode else 0.6)) < 1e-12
    assert np.allclose(a[True] * 2.0, a[False], atol=1e-12)                          # one layer: alpha = obar I
    gA = np.random.default_rng(0).normal(size=a[True].shape)
    g_mean = oracle_mod.Oracle(pos, col, opa, None, IDENT, cam, SimpleParams(sigma=1.0), "f64").backward(None, None, gA)
    g_min = oracle_mod.Oracle(pos, col, opa, None, IDENT, cam, SimpleParams(sigma=1.0, min_opacity=True), "f64").backward(None, None, gA)
    assert np.allclose(g_mean.grad_opacity, g_mean.grad_opacity[0])                  # equal thirds
    assert g_min.grad_opacity[0] == 0 and g_min.grad_opacity[1] == 0
    assert abs(g_min.grad_opacity[2] - 3.0 * g_mean.grad_opacity[0]) < 1e-12 * abs(g_min.grad_opacity[2]) + 1e-15
    # ties: the lowest index takes the gradient
    g_tie = oracle_mod.Oracle(pos, col, np.array([0.5, 0.3, 0.3]), None, IDENT, cam,
                              SimpleParams(sigma=1.0, min_opacity=True), "f64").backward(None, None, gA)
    assert g_tie.grad_opacity[1] != 0 and g_tie.grad_opacity[2] == 0 and g_tie.grad_opacity[0] == 0


def test_p23_finite_differences(oracle_mod):
    """Central differences of <gC,C> + <gD,D> + <gA,A> in min mode, for opacities (away from ties) and positions."""
    cam, prm, pos, col, opa, T = small_scene(13, n=70)
    prm.min_opacity = True
    rng = np.random.default_rng(5)
    gC, gD, gA = rng.normal(size=(3, cam.height, cam.width)), rng.normal(size=(cam.height, cam.width)), rng.normal(size=(cam.height, cam.width))

    def value(p, a):
        f = oracle_mod.Oracle(p, col, a, None, T, cam, prm, "f64").forward()
        return float((gC * f.color).sum() + (gD * f.depth).sum() + (gA * f.alpha).sum()), f.sig

    L0, sig0 = value(pos, opa)
    g = oracle_mod.Oracle(pos, col, opa, None, T, cam, prm, "f64").backward(gC, gD, gA)
    tri = opa.reshape(-1, 3)
    is_min = (tri == tri.min(axis=1, keepdims=True)).reshape(-1)
    assert np.all(g.grad_opacity[~is_min] == 0) and np.abs(g.grad_opacity[is_min]).max() > 0
    h, checked = 1e-6, 0
    for kind, arr, grad in (("opa", opa, g.grad_opacity), ("pos", pos, g.grad_pos)):
        scale = np.abs(grad).max()
        for fi in rng.choice(arr.size, 90, replace=False):
            ap, am = arr.copy(), arr.copy()
            ap.flat[fi] += h
            am.flat[fi] -= h
            (lp, sp), (lm, sm) = (value(pos, ap), value(pos, am)) if kind == "opa" else (value(ap, opa), value(am, opa))
            if not (np.array_equal(sp, sig0) and np.array_equal(sm, sig0)):
                continue
            checked += 1
            d = (lp - lm) / (2 * h)
            assert abs(d - grad.flat[fi]) <= 1e-5 * scale + 1e-4 * abs(d), (kind, fi, d, grad.flat[fi])
    assert checked > 120
