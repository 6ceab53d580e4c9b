"""Pins P26-P27: the normalised depth D / A with its backward pass, and the normal of the highest-opacity hit (Fig. 3,
PAPER.md:145).  Expectations are closed forms (worked example of tests/golden, ray-plane geometry, single-face alphas)
and central finite differences through the float64 oracle; none re-types the oracle's formulas."""
import os

import numpy as np
import pytest

from conftest import IDENT, SimpleCam, SimpleParams, unproject
from test_oracle_closed_form import CAM, RGB, load_gold


def test_p26_normalised_depth_is_the_ray_plane_depth(oracle_mod):
    g = load_gold()
    uvz = np.stack([g["tri_u"], g["tri_v"], g["Z"]], axis=1)            # worked example: depths (2, 4, 4)
    pos = unproject(uvz, CAM)
    px, py = g["pixel"].astype(int)
    for opa in ((0.9, 0.6, 0.3), (0.3, 0.2, 0.1), (1.0, 1.0, 1.0)):
        o = oracle_mod.Oracle(pos, RGB, np.array(opa), None, IDENT, CAM, SimpleParams(sigma=1.0), "f64")
        f = o.forward("brute")
        Dn = oracle_mod.depth_normalise(f.depth, f.alpha, 1e-9, "f64")
        # D = alpha z and A = alpha for a single face, so D / A = z = 3.2 at the worked pixel whatever the opacity
        assert abs(Dn[py, px] - g["z"][0]) < 1e-12
        # ... and everywhere on the face it is the depth of the ray-plane intersection (independent geometry)
        n = np.cross(pos[1] - pos[0], pos[2] - pos[0])
        ys, xs = np.nonzero(f.alpha > 1e-6)
        d = np.stack([(xs - CAM.cx) / CAM.fx, (ys - CAM.cy) / CAM.fy, np.ones(len(xs))], axis=1)
        z_plane = (n @ pos[0]) / (d @ n)
        assert np.allclose(Dn[ys, xs], z_plane, rtol=1e-10)
        assert np.all(Dn[f.alpha <= 1e-9] == 0.0)
    # float32 agrees
    f32 = oracle_mod.Oracle(pos, RGB, np.array((0.9, 0.6, 0.3)), None, IDENT, CAM, SimpleParams(sigma=1.0), "f32").forward("brute")
    assert abs(oracle_mod.depth_normalise(f32.depth, f32.alpha, 1e-6, "f32")[py, px] - 3.2) < 1e-5


def test_p26_normalised_depth_backward_finite_differences(oracle_mod):
    """L = sum w * (D / A): analytic gradient = depth_normalise_bwd -> oracle backward (gD, gA), against central
    differences of L on vertex coordinates and opacities (float64, alpha_min = t_min = 0)."""
    rng = np.random.default_rng(26)
    cam = SimpleCam(32, 24, 30.0, 30.0, 15.5, 11.5)
    prm = SimpleParams(sigma=1.0)
    M = 12
    cen = np.stack([rng.uniform(-0.8, 0.8, M), rng.uniform(-0.6, 0.6, M), rng.uniform(2.0, 3.0, M)], axis=1)
    pos = (cen[:, None, :] + rng.normal(0, 0.25, (M, 3, 3))).reshape(-1, 3)
    pos[:, 2] = np.maximum(pos[:, 2], 1.0)
    col, opa = rng.uniform(0, 1, (3 * M, 3)), rng.uniform(0.3, 0.9, 3 * M)
    w = rng.normal(size=(cam.height, cam.width))

    def loss(p, op):
        f = oracle_mod.Oracle(p, col, op, None, IDENT, cam, prm, "f64").forward("brute")
        return float((w * oracle_mod.depth_normalise(f.depth, f.alpha, 1e-4, "f64")).sum()), f

    L0, f0 = loss(pos, opa)
    gD, gA = oracle_mod.depth_normalise_bwd(f0.depth, f0.alpha, w, 1e-4, "f64")
    g = oracle_mod.Oracle(pos, col, opa, None, IDENT, cam, prm, "f64").backward(None, gD, gA)
    h, checked = 1e-6, 0
    for idx in rng.choice(pos.size, 40, replace=False):
        v, k = divmod(int(idx), 3)
        pp, pm = pos.copy(), pos.copy()
        pp[v, k] += h
        pm[v, k] -= h
        Lp, fp = loss(pp, opa)
        Lm, fm = loss(pm, opa)
        if not (np.array_equal(fp.n_contrib, f0.n_contrib) and np.array_equal(fm.n_contrib, f0.n_contrib)):
            continue                                            # the step crossed a kink (hit set changed)
        if ((fp.alpha > 1e-4) != (f0.alpha > 1e-4)).any() or ((fm.alpha > 1e-4) != (f0.alpha > 1e-4)).any():
            continue                                            # ... or the A > eps mask
        fd = (Lp - Lm) / (2 * h)
        assert abs(fd - g.grad_pos[v, k]) <= 1e-5 * max(1.0, abs(fd)), (v, k, fd, g.grad_pos[v, k])
        checked += 1
    for v in rng.choice(3 * M, 10, replace=False):
        op_p, op_m = opa.copy(), opa.copy()
        op_p[v] += h
        op_m[v] -= h
        fd = (loss(pos, op_p)[0] - loss(pos, op_m)[0]) / (2 * h)
        assert abs(fd - g.grad_opacity[v]) <= 1e-5 * max(1.0, abs(fd))
        checked += 1
    assert checked >= 30
    # a single face: D / A does not depend on its opacity at all, so that gradient is exactly zero
    o1 = oracle_mod.Oracle(pos[:3], col[:3], opa[:3], None, IDENT, cam, prm, "f64")
    f1 = o1.forward("brute")
    gD1, gA1 = oracle_mod.depth_normalise_bwd(f1.depth, f1.alpha, w, 1e-4, "f64")
    assert np.abs(o1.backward(None, gD1, gA1).grad_opacity).max() < 1e-12


def test_p27_normal_of_the_highest_opacity_hit(oracle_mod):
    """Two overlapping faces on different planes: the top normal at a pixel is the normal of whichever face has the
    larger alpha THERE (alphas taken from single-face renders, normals from the plane equations)."""
    cam = SimpleCam(48, 48, 60.0, 60.0, 23.5, 23.5)
    prm = SimpleParams(sigma=1.0)

    def plane_face(a, b, c, shift=(0.0, 0.0)):            # Z = a X + b Y + c over a big screen triangle
        uv = np.array([[4.0, 4.0], [44.0, 6.0], [20.0, 44.0]]) + np.asarray(shift)
        P = []
        for u, v in uv:
            dx, dy = (u - cam.cx) / cam.fx, (v - cam.cy) / cam.fy
            Z = c / (1.0 - a * dx - b * dy)
            P.append([dx * Z, dy * Z, Z])
        return np.array(P)

    A_, B_ = plane_face(0.3, 0.1, 2.0), plane_face(-0.2, 0.4, 3.0, (-3.0, 2.5))   # A in front of B; windows differ
    nA = np.array([0.3, 0.1, -1.0]) / np.linalg.norm([0.3, 0.1, -1.0])
    nB = np.array([-0.2, 0.4, -1.0]) / np.linalg.norm([-0.2, 0.4, -1.0])
    col = np.ones((6, 3))
    for oa, ob in ((0.6, 0.5), (0.5, 0.6), (0.2, 0.9)):
        opa = np.array([oa] * 3 + [ob] * 3)
        o = oracle_mod.Oracle(np.vstack([A_, B_]), col, opa, None, IDENT, cam, prm, "f64")
        top = o.normal_top("brute")
        aA = oracle_mod.Oracle(A_, col[:3], opa[:3], None, IDENT, cam, prm, "f64").forward("brute").alpha
        aB = oracle_mod.Oracle(B_, col[3:], opa[3:], None, IDENT, cam, prm, "f64").forward("brute").alpha
        both = (aA > 1e-3) & (aB > 1e-3) & (np.abs(aA - aB) > 1e-6)
        assert both.sum() > 200
        want = np.where((aA > aB)[None], nA[:, None, None], nB[:, None, None])
        assert np.allclose(top[:, both], want[:, both], atol=1e-12)
        if abs(oa - ob) < 0.2:
            assert (aA > aB)[both].any() and (aB > aA)[both].any()           # both cases occur inside one image
        only_a = (aA > 1e-3) & (aB == 0)
        assert np.allclose(top[:, only_a], nA[:, None], atol=1e-12)
        none = o.forward("brute").n_contrib == 0            # (alpha = 1 - T reads 0 for a hit with alpha below 1e-16)
        assert none.sum() > 500 and not top[:, none].any()
        # single layer: the top normal is the direction of the composited normal map
        N = o.normal_forward("brute")
        assert np.allclose(N[:, only_a] / aA[only_a], top[:, only_a], atol=1e-10)
        # tiled mode agrees
        assert np.array_equal(o.normal_top("tiled"), top)
