"""Pins P1-P6: the oracle against closed forms fixed by the paper's definitions.

Eq. 2-3: window = (distance to nearest edge / inradius)^sigma inside, 0 on/outside the boundary,
exactly 1 at the incentre.  PAPER.md:82: barycentric colour, mean opacity.  Eq. 4: compositing.
None of these tests re-types the oracle's formulas: expectations are hand-computed numbers (tests/golden) or
independent geometry (ray-plane intersection, point-to-segment distance).
"""
import os

import numpy as np
import pytest

from conftest import IDENT, SimpleCam, SimpleParams, unproject

GOLD = os.path.join(os.path.dirname(__file__), "golden", "worked_example.txt")


def load_gold():
    g = {}
    for line in open(GOLD):
        if line.startswith("#") or not line.strip():
            continue
        k, *v = line.split()
        g[k] = np.array([float(x) for x in v])
    return g


def render(tso, cam, prm, uvz, col, opa, prec="f64", mode="brute", T=IDENT):
    pos = unproject(np.asarray(uvz, dtype=np.float64).reshape(-1, 3), cam)
    o = tso.Oracle(pos, col, opa, None, T, cam, prm, prec)
    return o, o.forward(mode)


CAM = SimpleCam(64, 64, 100.0, 100.0, 0.0, 0.0)
RGB = np.eye(3)


@pytest.mark.parametrize("prec,tol", [("f64", 1e-12), ("f32", 2e-6)])
@pytest.mark.parametrize("sigma,key", [(1.0, "I_sigma1"), (0.5, "I_sigma05"), (2.0, "I_sigma2")])
def test_p1_window_values(oracle_mod, prec, tol, sigma, key):
    g = load_gold()
    uvz = np.stack([g["tri_u"], g["tri_v"], np.full(3, 2.0)], axis=1)
    o, f = render(oracle_mod, CAM, SimpleParams(sigma=sigma), uvz, RGB, np.ones(3), prec)
    # fronto-parallel, opacity 1: alpha(p) = I(p)
    sx, sy = g["incentre"].astype(int)
    assert abs(f.alpha[sy, sx] - 1.0) < tol                       # exactly 1 at the incentre
    px, py = g["pixel"].astype(int)
    assert abs(f.alpha[py, px] - g[key][0]) < tol
    # P3 fronto-parallel: lambda = screen barycentrics, D = Z * A
    assert np.allclose(f.color[:, py, px] / f.alpha[py, px], g["bary"], atol=10 * tol)
    assert np.allclose(f.depth, 2.0 * f.alpha, atol=10 * tol)
    # zero on every boundary pixel, at the vertices and outside
    # (boundary pixels sit on the edge only up to the rounding of the unprojection: x ~ 1 ulp, I ~ ulp^sigma)
    btol = (1e-14 if prec == "f64" else 1e-6) ** min(sigma, 1.0)
    for (x, y) in [(8, 8), (38, 8), (8, 48), (8, 20), (20, 8), (23, 28)]:
        assert f.alpha[y, x] < btol
    for (x, y) in [(7, 20), (20, 7), (40, 40), (0, 0), (24, 28), (39, 8)]:
        assert f.alpha[y, x] == 0.0


@pytest.mark.parametrize("sigma", [0.5, 1.0, 2.0])
def test_p1_window_is_edge_distance_over_inradius(oracle_mod, sigma):
    """Everywhere: I(p) = (min point-to-segment-line distance / r)^sigma for inside pixels; independent geometry."""
    g = load_gold()
    q = np.stack([g["tri_u"], g["tri_v"]], axis=1)
    uvz = np.concatenate([q, np.full((3, 1), 3.0)], axis=1)
    o, f = render(oracle_mod, CAM, SimpleParams(sigma=sigma), uvz, RGB, np.ones(3), "f64")
    ys, xs = np.mgrid[0:64, 0:64]
    P = np.stack([xs, ys], axis=-1).astype(np.float64)
    dist = np.full((64, 64), np.inf)
    inside = np.ones((64, 64), bool)
    for a, b, c in [(0, 1, 2), (1, 2, 0), (2, 0, 1)]:
        e = q[b] - q[a]
        cr = e[0] * (P[..., 1] - q[a][1]) - e[1] * (P[..., 0] - q[a][0])
        cr_c = e[0] * (q[c][1] - q[a][1]) - e[1] * (q[c][0] - q[a][0])
        inside &= (cr * np.sign(cr_c) > 0)
        dist = np.minimum(dist, np.abs(cr) / np.linalg.norm(e))
    expect = np.where(inside, (dist / g["inradius"][0]) ** sigma, 0.0)
    off_edge = dist > 1e-9      # pixels exactly on an edge are decided by the unprojection's last bit
    assert off_edge.sum() > 3900 and inside.sum() > 500
    assert np.allclose(f.alpha[off_edge], expect[off_edge], atol=1e-12)
    assert f.alpha[~off_edge].max() < 1e-6


@pytest.mark.parametrize("prec,tol", [("f64", 1e-12), ("f32", 3e-6)])
def test_p2_worked_example(oracle_mod, prec, tol):
    g = load_gold()
    uvz = np.stack([g["tri_u"], g["tri_v"], g["Z"]], axis=1)
    o, f = render(oracle_mod, CAM, SimpleParams(sigma=1.0), uvz, RGB, g["opacity"], prec)
    px, py = g["pixel"].astype(int)
    assert np.allclose(f.color[:, py, px], g["C_sigma1"], atol=tol)
    assert abs(f.depth[py, px] - g["D_sigma1"][0]) < 10 * tol
    assert abs(f.alpha[py, px] - g["A_sigma1"][0]) < tol
    pr = o.project()
    assert abs(float(pr.zbar[0]) - g["mean_depth"][0]) < 10 * tol
    assert pr.depth_key[0] == np.float32(pr.zbar[0]).view(np.uint32)
    assert tuple(pr.rect[0]) == (8, 8, 38, 48) and pr.tiles_touched[0] == 3 * 4


def test_p4_perspective_correct_is_ray_plane(oracle_mod):
    """Tilted face: D/A is the ray-plane intersection depth and C/A the 3-D barycentrics of that point."""
    cam = SimpleCam(96, 80, 90.0, 85.0, 47.3, 39.6)
    rng = np.random.default_rng(5)
    uvz = np.array([[10.2, 12.7, 1.5], [80.4, 20.1, 4.0], [35.5, 70.3, 2.5]])
    pos = unproject(uvz, cam)
    o = oracle_mod.Oracle(pos, RGB, np.ones(3), None, IDENT, cam, SimpleParams(sigma=0.5), "f64")
    f = o.forward("brute")
    n = np.cross(pos[1] - pos[0], pos[2] - pos[0])
    ys, xs = np.nonzero(f.alpha > 0)
    assert len(ys) > 500
    for y, x in zip(ys[::7], xs[::7]):
        d = np.array([(x - cam.cx) / cam.fx, (y - cam.cy) / cam.fy, 1.0])
        tz = n.dot(pos[0]) / n.dot(d)
        X = tz * d
        lam = np.linalg.solve(np.stack([pos[0], pos[1], pos[2]], axis=1), X)
        assert abs(f.depth[y, x] / f.alpha[y, x] - tz) < 1e-10
        assert np.allclose(f.color[:, y, x] / f.alpha[y, x], lam, atol=1e-10)


def test_p5_opaque_face_gives_interpolated_colour(oracle_mod):
    g = load_gold()
    uvz = np.stack([g["tri_u"], g["tri_v"], g["Z"]], axis=1)
    col = np.array([[0.9, 0.1, 0.3], [0.2, 0.8, 0.5], [0.4, 0.6, 0.7]])
    for prec, tol in [("f64", 1e-13), ("f32", 1e-6)]:
        o, f = render(oracle_mod, CAM, SimpleParams(sigma=0.5), uvz, col, np.ones(3), prec)
        # at the incentre s=(18,18): b = r/h_k = (10/24, 10/30, 10/40); alpha = 1 exactly (no clamp, S8)
        b = np.array([10 / 24, 10 / 30, 10 / 40])
        om = b / g["Z"]
        lam = om / om.sum()
        assert abs(f.alpha[18, 18] - 1.0) < tol
        assert np.allclose(f.color[:, 18, 18], lam @ col, atol=tol)
        assert abs(f.depth[18, 18] - 1.0 / om.sum()) < 10 * tol


def test_p6_two_layers_and_tie_break(oracle_mod):
    """C = a1 c1 + (1-a1) a2 c2 (Eq. 4); swapping depths swaps roles; equal depth keys -> lower index in front."""
    g = load_gold()
    tri = np.stack([g["tri_u"], g["tri_v"]], axis=1)

    def scene(z_a, z_b):
        uvz = np.concatenate([np.c_[tri, np.full(3, z_a)], np.c_[tri, np.full(3, z_b)]])
        col = np.concatenate([np.tile([1.0, 0.0, 0.0], (3, 1)), np.tile([0.0, 0.0, 1.0], (3, 1))])
        opa = np.concatenate([np.full(3, 0.5), np.full(3, 0.8)])
        return render(oracle_mod, CAM, SimpleParams(sigma=1.0), uvz, col, opa, "f64", mode="tiled")[1]

    a1, a2 = 0.5 * 0.6, 0.8 * 0.6   # window 0.6 at pixel (23,18)
    f = scene(2.0, 3.0)
    assert np.allclose(f.color[:, 18, 23], [a1, 0, (1 - a1) * a2], atol=1e-12)
    assert abs(f.alpha[18, 23] - (1 - (1 - a1) * (1 - a2))) < 1e-12
    assert abs(f.depth[18, 23] - (a1 * 2.0 + (1 - a1) * a2 * 3.0)) < 1e-12
    f = scene(3.0, 2.0)
    assert np.allclose(f.color[:, 18, 23], [(1 - a2) * a1, 0, a2], atol=1e-12)
    f = scene(2.5, 2.5)             # tie: face 0 in front
    assert np.allclose(f.color[:, 18, 23], [a1, 0, (1 - a1) * a2], atol=1e-12)
