"""Pin P24: the screen-space gradient statistic (reading S28) against a finite difference through
the CAMERA INTRINSICS: moving the principal point by (dx, dy) translates every projected vertex by (dx, dy) in the
image plane, so for a scene with one face dL/d(cx, cy) is that face's statistic vector, and for several faces the sum
of theirs."""
import numpy as np

from conftest import IDENT, SimpleCam, SimpleParams
from test_oracle_gradients import small_scene


def _value(oracle_mod, cam, prm, pos, col, opa, T, gC, gD, gA, dcx=0.0, dcy=0.0):
    c = SimpleCam(cam.width, cam.height, cam.fx, cam.fy, cam.cx + dcx, cam.cy + dcy, cam.znear)
    f = oracle_mod.Oracle(pos, col, opa, None, T, c, prm, "f64").forward()
    return float((gC * f.color).sum() + (gD * f.depth).sum() + (gA * f.alpha).sum()), f.sig


def test_p24_principal_point_finite_difference(oracle_mod):
    cam, prm, pos, col, opa, T = small_scene(21, n=60)
    rng = np.random.default_rng(2)
    gC = rng.normal(size=(3, cam.height, cam.width))
    gD, gA = rng.normal(size=(cam.height, cam.width)), rng.normal(size=(cam.height, cam.width))
    # one face at a time (the statistic is per face), then all together (the sum of the vectors)
    h = 1e-6
    for sel in ([7], [23], list(range(60))):
        idx = np.concatenate([[3 * m, 3 * m + 1, 3 * m + 2] for m in sel])
        p, c, a = pos[idx], col[idx], opa[idx]
        o = oracle_mod.Oracle(p, c, a, None, T, cam, prm, "f64")
        if o.project().n_visible == 0:
            continue
        g = o.backward(gC, gD, gA, want=("pos", "stat"))
        vec = np.stack([g.g_scr[:, 0] + g.g_scr[:, 3] + g.g_scr[:, 6], g.g_scr[:, 1] + g.g_scr[:, 4] + g.g_scr[:, 7]], axis=1)
        assert np.allclose(g.face_grad2d, np.linalg.norm(vec, axis=1), rtol=1e-13, atol=0)
        assert np.array_equal(g.face_views, (np.abs(g.g_scr).sum(1) > 0).astype(np.uint32))
        L0, sig0 = _value(oracle_mod, cam, prm, p, c, a, T, gC, gD, gA)
        d = []
        for dcx, dcy in ((h, 0.0), (0.0, h)):
            (lp, sp), (lm, sm) = (_value(oracle_mod, cam, prm, p, c, a, T, gC, gD, gA, dcx, dcy),
                                  _value(oracle_mod, cam, prm, p, c, a, T, gC, gD, gA, -dcx, -dcy))
            assert np.array_equal(sp, sig0) and np.array_equal(sm, sig0)
            d.append((lp - lm) / (2 * h))
        tot = vec.sum(0)
        assert np.allclose(d, tot, rtol=2e-5, atol=2e-6 * np.abs(vec).max()), (sel, d, tot)
        if len(sel) == 1:
            assert abs(np.hypot(*d) - g.face_grad2d[0]) <= 2e-5 * g.face_grad2d[0]


def test_p24_accumulates_over_views(oracle_mod):
    cam, prm, pos, col, opa, T = small_scene(22, n=40)
    rng = np.random.default_rng(3)
    gC = rng.normal(size=(3, cam.height, cam.width))
    o = oracle_mod.Oracle(pos, col, opa, None, T, cam, prm, "f64")
    g = o.backward(gC, None, None, want=("stat",))
    pr = o.project()
    acc, views = np.zeros(o.M), np.zeros(o.M, np.uint32)
    for _ in range(3):
        oracle_mod.lib().tso_screen_grad_stat_f64(o.M, oracle_mod._p(pr.visible), oracle_mod._p(g.g_scr),
                                                  oracle_mod._p(acc), oracle_mod._p(views))
    assert np.allclose(acc, 3 * g.face_grad2d) and np.array_equal(views, 3 * g.face_views)
    assert np.all(acc[pr.visible == 0] == 0)
