"""Pins P18-P21 of the oracle's rendered normal map (Eq. 12; reading S26):
closed forms that do not go through a cross product of the vertices (plane coefficients, Eq. 11 applied to the
rendered depth), winding / rigid-motion invariants, two-layer compositing and central finite differences of the
float64 forward pass for every gradient, incl. SE(3) perturbations."""
import numpy as np
import pytest

from conftest import IDENT, SimpleCam, SimpleParams, unproject
from paper_2605_31419_b200 import scenes
from test_oracle_gradients import small_scene


def plane_triangle(cam, a, b, c, uv):
    """Three world points (identity pose) on the plane Z = a X + b Y + c whose projections are the pixels uv."""
    uv = np.asarray(uv, np.float64)
    xn, yn = (uv[:, 0] - cam.cx) / cam.fx, (uv[:, 1] - cam.cy) / cam.fy
    Z = c / (1.0 - a * xn - b * yn)
    return np.stack([xn * Z, yn * Z, Z], axis=1)


def test_p18_plane_coefficients_and_winding(oracle_mod):
    """One opaque face on Z = aX + bY + c: N(p)/A(p) is the plane normal (a, b, -1)/|.| (pointing at the camera,
    which looks along +Z), whatever the vertex order; fronto-parallel gives (0, 0, -1)."""
    cam = SimpleCam(48, 40, 50.0, 47.0, 23.5, 19.5)
    prm = SimpleParams(sigma=1.0)
    uv = [(4.3, 5.1), (43.2, 8.7), (20.9, 36.4)]
    for a, b, c in [(0.0, 0.0, 2.0), (0.3, -0.2, 2.5), (-0.6, 0.45, 3.0)]:
        expect = np.array([a, b, -1.0]) / np.sqrt(a * a + b * b + 1.0)
        for order in ([0, 1, 2], [0, 2, 1]):
            pos = plane_triangle(cam, a, b, c, uv)[order]
            o = oracle_mod.Oracle(pos, np.ones((3, 3)), np.ones(3), None, IDENT, cam, prm, "f64")
            n = o.face_normals()
            assert np.allclose(n[0], expect, atol=1e-12)
            N, A = o.normal_forward(), o.forward().alpha
            cov = A > 1e-3
            assert cov.sum() > 300
            assert np.allclose(N[:, cov] / A[cov], expect[:, None], atol=1e-10)
            assert np.all(N[:, ~(A > 0)] == 0)


def test_p19_sensor_normal_of_the_rendered_depth(oracle_mod):
    """Eq. 11 applied to the oracle's own rendered depth D/A of a planar face -- back-projection and
    finite differences of neighbouring pixels, no vertex involved -- reproduces the rendered normal N/A."""
    cam = SimpleCam(64, 48, 60.0, 58.0, 31.5, 23.5)
    prm = SimpleParams(sigma=1.0)
    pos = plane_triangle(cam, 0.25, -0.4, 2.2, [(3.2, 2.6), (60.1, 9.4), (25.5, 45.2)])
    o = oracle_mod.Oracle(pos, np.ones((3, 3)), np.ones(3), None, IDENT, cam, prm, "f64")
    f, N = o.forward(), o.normal_forward()
    cov = f.alpha > 1e-3
    z = np.where(cov, f.depth / np.where(cov, f.alpha, 1.0), np.nan)
    ys, xs = np.mgrid[0:cam.height, 0:cam.width]
    P = np.stack([(xs - cam.cx) / cam.fx * z, (ys - cam.cy) / cam.fy * z, z])
    dx, dy = P[:, :, 1:] - P[:, :, :-1], P[:, 1:, :] - P[:, :-1, :]
    nb = np.cross(dx[:, :-1, :], dy[:, :, :-1], axis=0)
    nb /= np.linalg.norm(nb, axis=0)
    nb *= -np.sign((nb * P[:, :-1, :-1]).sum(0))                      # towards the camera
    ok = np.isfinite(nb).all(0)
    assert ok.sum() > 300
    Nn = (N / np.where(cov, f.alpha, 1.0))[:, :-1, :-1]
    assert np.allclose(Nn[:, ok], nb[:, ok], atol=1e-9)


def test_p20_two_layers_and_flat_colour_equivalence(oracle_mod):
    """Eq. 4 with two faces: N = n1 a1 + n2 a2 (1 - a1); and on a random scene the normal map equals the COLOUR image of
    the same scene whose three vertex colours of face m are all n_m (a flat attribute interpolates to itself)."""
    cam = SimpleCam(32, 32, 40.0, 40.0, 15.5, 15.5)
    prm = SimpleParams(sigma=1.0)
    uv = [(2.2, 3.1), (29.3, 4.4), (15.8, 29.6)]
    near, far = plane_triangle(cam, 0.2, 0.1, 2.0, uv), plane_triangle(cam, -0.3, 0.25, 3.0, uv)
    pos = np.concatenate([far, near])
    opa = np.array([0.9, 0.9, 0.9, 0.6, 0.6, 0.6])
    o = oracle_mod.Oracle(pos, np.ones((6, 3)), opa, None, IDENT, cam, prm, "f64")
    n = o.face_normals()
    o1 = oracle_mod.Oracle(near, np.ones((3, 3)), opa[3:], None, IDENT, cam, prm, "f64")
    o2 = oracle_mod.Oracle(far, np.ones((3, 3)), opa[:3], None, IDENT, cam, prm, "f64")
    a1, a2 = o1.forward().alpha, o2.forward().alpha
    expect = n[1][:, None, None] * a1 + n[0][:, None, None] * a2 * (1 - a1)
    assert np.allclose(o.normal_forward(), expect, atol=1e-12)

    cam2, prm2, pos2, col2, opa2, T2 = small_scene(11, n=120)
    oo = oracle_mod.Oracle(pos2, col2, opa2, None, T2, cam2, prm2, "f64")
    nn = oo.face_normals()
    flat = np.repeat(nn, 3, axis=0)
    as_colour = oracle_mod.Oracle(pos2, flat, opa2, None, T2, cam2, prm2, "f64").forward().color
    assert np.abs(as_colour).max() > 0.3
    assert np.allclose(oo.normal_forward(), as_colour, atol=1e-12)
    # unit length, towards the camera, zero for culled faces
    pr = oo.project()
    vis = pr.visible.astype(bool)
    assert np.allclose(np.linalg.norm(nn[vis], axis=1), 1.0, atol=1e-12)
    assert np.all((nn[vis] * pr.Q[vis, :3]).sum(1) < 0) and np.all(nn[~vis] == 0)
    # brute == tiled
    assert np.allclose(oo.normal_forward("brute"), oo.normal_forward("tiled"), atol=1e-13)


def test_p20_rigid_motion(oracle_mod):
    """Moving the world by G and the camera by G^-1 leaves the camera-space normal map unchanged."""
    cam, prm, pos, col, opa, T = small_scene(5, n=100)
    G = scenes.left_perturb(IDENT, np.array([0.3, -0.2, 0.5, 0.4, -0.3, 0.2]))
    R, t = G[:, :3], G[:, 3]
    pos2 = pos @ R.T + t
    T4 = np.vstack([T, [0, 0, 0, 1]])
    Ginv = np.linalg.inv(np.vstack([G, [0, 0, 0, 1]]))
    T2 = (T4 @ Ginv)[:3]
    a = oracle_mod.Oracle(pos, col, opa, None, T, cam, prm, "f64").normal_forward()
    b = oracle_mod.Oracle(pos2, col, opa, None, T2, cam, prm, "f64").normal_forward()
    assert np.abs(a).max() > 0.3 and np.allclose(a, b, atol=1e-9)


@pytest.mark.parametrize("sigma", [1.0, 2.0])
def test_p21_finite_differences(oracle_mod, sigma):
    """d<gN, N>/d(pos, opacity, pose): analytic (B2-B9 with the flat attribute + the normal's own dependence on the
    vertices) against Richardson central differences of the float64 forward pass."""
    cam, prm, pos, col, opa, T = small_scene(7, n=90, sigma=sigma)
    rng = np.random.default_rng(17)
    gN = rng.normal(size=(3, cam.height, cam.width))

    def value(p, a, Tm):
        o = oracle_mod.Oracle(p, col, a, None, Tm, cam, prm, "f64")
        return float((gN * o.normal_forward()).sum()), o.forward().sig

    L0, sig0 = value(pos, opa, T)
    g = oracle_mod.Oracle(pos, col, opa, None, T, cam, prm, "f64").normal_backward(gN)

    def fd(plus, minus, h):
        (lp, sp), (lm, sm) = value(*plus), value(*minus)
        return None if not (np.array_equal(sp, sig0) and np.array_equal(sm, sig0)) else (lp - lm) / (2 * h)

    def rich(make, h):
        d1, d2 = fd(make(h), make(-h), h), fd(make(h / 2), make(-h / 2), h / 2)
        return None if d1 is None or d2 is None else (4 * d2 - d1) / 3

    h = 1e-6
    checked = 0
    sp, so = np.abs(g.grad_pos).max(), np.abs(g.grad_opacity).max()
    for fi in rng.choice(pos.size, 150, replace=False):
        def make(s, fi=fi):
            p = pos.copy()
            p.flat[fi] += s
            return p, opa, T
        d = rich(make, h)
        if d is None:
            continue
        checked += 1
        assert abs(d - g.grad_pos.flat[fi]) <= 2e-5 * sp + 1e-4 * abs(d), (fi, d, g.grad_pos.flat[fi])
    assert checked > 100
    checked = 0
    for fi in rng.choice(opa.size, 80, replace=False):
        def make(s, fi=fi):
            a = opa.copy()
            a[fi] += s
            return pos, a, T
        d = rich(make, h)
        if d is None:
            continue
        checked += 1
        assert abs(d - g.grad_opacity[fi]) <= 2e-6 * so + 1e-5 * abs(d), (fi, d, g.grad_opacity[fi])
    assert checked > 60
    # pose: Exp(+-h e_k) o T
    st = np.abs(g.dL_dtau).max()
    for k in range(6):
        def make(s, k=k):
            tau = np.zeros(6)
            tau[k] = s
            return pos, opa, oracle_mod.left_perturb(T, tau)
        d = rich(make, h)
        assert d is not None
        assert abs(d - g.dL_dtau[k]) <= 2e-5 * st, (k, d, g.dL_dtau[k])
    # a translation of the camera does not turn the normals: the rho part comes from the window path only
    only_n = np.zeros(6)
    o = oracle_mod.Oracle(pos, col, opa, None, T, cam, prm, "f64")
    pr = o.project()
    oracle_mod.lib().tso_face_normal_bwd_f64(
        oracle_mod._p(o.pos), None, o.M, oracle_mod._p(o.T_cw), oracle_mod._p(pr.visible), oracle_mod._p(pr.Q),
        oracle_mod._p(g.g_nrm), None, oracle_mod._p(only_n))
    assert np.all(only_n[:3] == 0) and np.abs(only_n[3:]).max() > 0


def test_p22_normal_loss_closed_forms(oracle_mod):
    """E_norm (Eq. 12): 0 when the maps agree on unit normals, 2 when they are opposite, 1 when orthogonal or when
    nothing was rendered; pixels without a sensor normal do not count; the gradient is -w Nbar / (H W) on valid pixels
    (the loss is linear in N, so a finite difference is exact)."""
    rng = np.random.default_rng(3)
    H, W = 7, 9
    nb = rng.normal(size=(3, H, W))
    nb /= np.linalg.norm(nb, axis=0)
    for prec in ("f64", "f32"):
        tol = 1e-12 if prec == "f64" else 1e-6
        assert abs(oracle_mod.normal_loss(nb, nb, 1.0, prec)[0]) < tol
        assert abs(oracle_mod.normal_loss(-nb, nb, 1.0, prec)[0] - 2.0) < tol
        assert abs(oracle_mod.normal_loss(np.zeros_like(nb), nb, 0.05, prec)[0] - 0.05) < tol
        t = np.cross(nb, np.array([0.3, -0.5, 0.8])[:, None, None], axis=0)
        assert abs(oracle_mod.normal_loss(t, nb, 1.0, prec)[0] - 1.0) < tol
    holes = nb.copy()
    holes[:, 2:4, 3:6] = 0.0                      # 6 pixels without a sensor normal
    L, g = oracle_mod.normal_loss(-nb, holes, 3.0)
    assert abs(L - 3.0 * 2.0 * (H * W - 6) / (H * W)) < 1e-12
    assert np.all(g[:, 2:4, 3:6] == 0) and np.allclose(g, -3.0 * holes / (H * W), atol=1e-15)
    N = rng.normal(size=(3, H, W))
    dN = rng.normal(size=(3, H, W))
    L0, g0 = oracle_mod.normal_loss(N, holes, 0.7)
    L1, _ = oracle_mod.normal_loss(N + dN, holes, 0.7)
    assert abs((L1 - L0) - (g0 * dN).sum()) < 1e-12
