"""Pins P11-P13: every analytic gradient of the oracle against central finite differences
of its own float64 FORWARD pass (the backward shares only eval() with it), incl. SE(3) perturbations
Exp(+-h e_k) o T (Eq. 5-7), plus exact identities."""
import numpy as np
import pytest

from paper_2605_31419_b200 import scenes


def small_scene(seed, n=80, sigma=1.0):
    """Overlapping triangles a few pixels to tens of pixels wide, several layers deep, varying depth."""
    rng = np.random.default_rng(seed)
    cam = scenes.Camera(40, 32, 45.0, 42.0, 19.3, 15.6)
    cen = np.stack([rng.uniform(-0.9, 0.9, n), rng.uniform(-0.7, 0.7, n), rng.uniform(2.0, 4.0, n)], axis=1)
    verts = cen[:, None, :] + rng.normal(0, 0.35, size=(n, 3, 3)) * np.array([1.0, 1.0, 0.6])
    pos = verts.reshape(-1, 3)
    col = rng.uniform(0, 1, size=(3 * n, 3))
    opa = rng.uniform(0.2, 1.0, size=3 * n)
    th = rng.normal(0, 0.05, 3)
    T = scenes.left_perturb(np.concatenate([np.eye(3), [[0.02], [-0.03], [0.1]]], axis=1), np.concatenate([[0, 0, 0], th]))
    prm = scenes.Params(sigma=sigma, alpha_min=0.0, t_min=0.0)
    return cam, prm, pos, col, opa, T


class Functional:
    """L = <gC,C> + <gD,D> + <gA,A> with fixed random cotangents (exercises gA != 0)."""

    def __init__(self, tso, cam, prm, seed):
        rng = np.random.default_rng(seed + 100)
        self.tso, self.cam, self.prm = tso, cam, prm
        self.gC = rng.normal(size=(3, cam.height, cam.width))
        self.gD = rng.normal(size=(cam.height, cam.width))
        self.gA = rng.normal(size=(cam.height, cam.width))

    def oracle(self, pos, col, opa, T):
        return self.tso.Oracle(pos, col, opa, None, T, self.cam, self.prm, "f64")

    def value(self, pos, col, opa, T):
        f = self.oracle(pos, col, opa, T).forward("tiled")
        return float((self.gC * f.color).sum() + (self.gD * f.depth).sum() + (self.gA * f.alpha).sum()), f.sig

    def grad(self, pos, col, opa, T):
        return self.oracle(pos, col, opa, T).backward(self.gC, self.gD, self.gA)


def fd(fun, base_sig, plus, minus, h):
    """Central difference; returns None when the step crossed a kink (hit sequence changed)."""
    (lp, sp), (lm, sm) = fun(*plus), fun(*minus)
    if not (np.array_equal(sp, base_sig) and np.array_equal(sm, base_sig)):
        return None
    return (lp - lm) / (2 * h)


def fd_dir(fun, base_sig, x0, dx, h):
    """Richardson-extrapolated central difference along dx (tuples of arrays): (4 D(h/2) - D(h)) / 3."""
    step = lambda s: tuple(a + s * d for a, d in zip(x0, dx))
    d1 = fd(fun, base_sig, step(h), step(-h), h)
    d2 = fd(fun, base_sig, step(h / 2), step(-h / 2), h / 2)
    return None if d1 is None or d2 is None else (4 * d2 - d1) / 3


@pytest.mark.parametrize("sigma", [0.5, 1.0, 2.0])
def test_p11_finite_differences_all_parameters(oracle_mod, sigma):
    cam, prm, pos, col, opa, T = small_scene(3, sigma=sigma)
    F = Functional(oracle_mod, cam, prm, 3)
    L0, sig0 = F.value(pos, col, opa, T)
    g = F.grad(pos, col, opa, T)
    assert (sig0 != sig0.flat[0]).mean() > 0.5          # most pixels are covered
    rng = np.random.default_rng(99)
    h = 1e-7   # sigma = 0.5 makes d3I/dx3 large next to an edge; the FD error falls as h^2 (checked down to 1e-8)
    scale = {"pos": np.abs(g.grad_pos).max(), "col": np.abs(g.grad_color).max(), "opa": np.abs(g.grad_opacity).max()}
    checked = {"pos": 0, "col": 0, "opa": 0}
    for kind, arr, grad in (("pos", pos, g.grad_pos), ("col", col, g.grad_color), ("opa", opa, g.grad_opacity)):
        flat_idx = rng.choice(arr.size, size=min(arr.size, 260), replace=False)
        for fi in flat_idx:
            ap, am = arr.copy(), arr.copy()
            ap.flat[fi] += h
            am.flat[fi] -= h
            args = {"pos": (pos, col, opa), "col": (pos, col, opa), "opa": (pos, col, opa)}[kind]
            sub = lambda a: tuple(a if k == kind else x for k, x in zip(("pos", "col", "opa"), args)) + (T,)
            d = fd(F.value, sig0, sub(ap), sub(am), h)
            if d is None:
                continue
            checked[kind] += 1
            assert abs(d - grad.flat[fi]) <= 2e-5 * scale[kind] + 1e-5 * abs(d), (kind, fi, d, grad.flat[fi])
    assert min(checked.values()) >= 200
    # 32 random directions in the full parameter space
    n_ok = 0
    for _ in range(32):
        dp, dc, do = rng.normal(size=pos.shape), rng.normal(size=col.shape), rng.normal(size=opa.shape)
        d = fd_dir(F.value, sig0, (pos, col, opa, T), (dp, dc, do, np.zeros_like(T)), h)
        if d is None:
            continue
        n_ok += 1
        ana = (g.grad_pos * dp).sum() + (g.grad_color * dc).sum() + (g.grad_opacity * do).sum()
        assert abs(d - ana) <= 1e-5 * (abs(ana) + np.sqrt((g.grad_pos**2).sum()))
    assert n_ok >= 16


@pytest.mark.parametrize("sigma", [0.5, 1.0, 2.0])
def test_p11_pose_jacobian_se3(oracle_mod, sigma):
    cam, prm, pos, col, opa, T = small_scene(7, sigma=sigma)
    F = Functional(oracle_mod, cam, prm, 7)
    L0, sig0 = F.value(pos, col, opa, T)
    g = F.grad(pos, col, opa, T)
    h = 1e-7   # sigma = 0.5 makes d3I/dx3 large next to an edge; the FD error falls as h^2 (checked down to 1e-8)
    n_ok = 0
    for k in range(6):
        e = np.zeros(6)
        e[k] = h
        P = lambda s: (pos, col, opa, oracle_mod.left_perturb(T, s * e))
        d1 = fd(F.value, sig0, P(1.0), P(-1.0), h)
        d2 = fd(F.value, sig0, P(0.5), P(-0.5), h / 2)
        if d1 is None or d2 is None:
            continue
        d = (4 * d2 - d1) / 3          # Richardson: every vertex moves, so the h^2 terms of all edges add up
        n_ok += 1
        assert abs(d - g.dL_dtau[k]) <= 1e-5 * np.abs(g.dL_dtau).max(), (k, d, g.dL_dtau)
    assert n_ok >= 5
    # the numpy Exp used by the input generators and the oracle's Exp agree
    tau = np.array([0.01, -0.02, 0.03, 0.02, -0.01, 0.015])
    assert np.allclose(scenes.left_perturb(T, tau), oracle_mod.left_perturb(T, tau), atol=1e-14)


def test_p11_l1_loss_gradient(oracle_mod):
    cam, prm, pos, col, opa, T = small_scene(5, sigma=0.5)
    o = oracle_mod.Oracle(pos, col, opa, None, T, cam, prm, "f64")
    f = o.forward("tiled")
    tgt = oracle_mod.Oracle(pos + np.random.default_rng(1).normal(0, 0.01, pos.shape), col, opa, None, T, cam, prm, "f64").forward("tiled")
    Dhat = np.where(tgt.alpha > 0.3, tgt.depth, 0.0)            # invalid (0) target depth where coverage is thin
    L, gC, gD = o.l1_loss(f.color, f.depth, tgt.color, Dhat, 0.05)
    n = cam.width * cam.height
    # independent numpy statement of Eq. 8-10 with the S19 normalisation
    Lnp = np.abs(f.color - tgt.color).sum() / (3 * n) + 0.05 * np.abs(f.depth - Dhat)[Dhat > 0].sum() / n
    assert abs(L - Lnp) < 1e-14
    assert np.allclose(gC, np.sign(f.color - tgt.color) / (3 * n)) and np.allclose(gD, np.where(Dhat > 0, np.sign(f.depth - Dhat), 0) * 0.05 / n)
    # and the chain through the renderer: d L1 / d tau by finite differences
    g = o.backward(gC, gD, None)
    h = 1e-7   # sigma = 0.5 makes d3I/dx3 large next to an edge; the FD error falls as h^2 (checked down to 1e-8)
    for k in (0, 2, 4):
        e = np.zeros(6)
        e[k] = h
        vals = []
        for s in (+1, -1):
            oo = oracle_mod.Oracle(pos, col, opa, None, oracle_mod.left_perturb(T, s * e), cam, prm, "f64")
            ff = oo.forward("tiled")
            vals.append(oo.l1_loss(ff.color, ff.depth, tgt.color, Dhat, 0.05)[0])
        assert abs((vals[0] - vals[1]) / (2 * h) - g.dL_dtau[k]) <= 2e-4 * np.abs(g.dL_dtau).max()


def test_p12_pose_gradient_identity_from_grad_pos(oracle_mod):
    """dL/dtau == sum_v [R g_W,v ; Q_v x (R g_W,v)] recomputed in numpy from grad_pos (soup: one entry per vertex)."""
    cam, prm, pos, col, opa, T = small_scene(11, sigma=0.5)
    F = Functional(oracle_mod, cam, prm, 11)
    g = F.grad(pos, col, opa, T)
    R, t = T[:, :3], T[:, 3]
    gc = g.grad_pos @ R.T
    Q = pos @ R.T + t
    tau = np.concatenate([gc.sum(0), np.cross(Q, gc).sum(0)])
    assert np.allclose(tau, g.dL_dtau, rtol=1e-10, atol=1e-10 * np.abs(tau).max())


def test_p13_identities(oracle_mod):
    cam, prm, pos, col, opa, T = small_scene(13, sigma=0.5)
    F = Functional(oracle_mod, cam, prm, 13)
    g = F.grad(pos, col, opa, T)
    # the three vertex-opacity gradients of a face are equal (mean opacity)
    go = g.grad_opacity.reshape(-1, 3)
    assert np.allclose(go[:, 0], go[:, 1]) and np.allclose(go[:, 1], go[:, 2]) and np.abs(go).max() > 0
    # sum_k dL/dc_k over a face == sum_p T alpha gC (since sum lambda = 1): compare against colour-shift FD
    h = 1e-7   # sigma = 0.5 makes d3I/dx3 large next to an edge; the FD error falls as h^2 (checked down to 1e-8)
    for m in (0, 5, 17, 33):
        for ch in range(3):
            cp, cm = col.copy(), col.copy()
            cp[3 * m:3 * m + 3, ch] += h
            cm[3 * m:3 * m + 3, ch] -= h
            d = (F.value(pos, cp, opa, T)[0] - F.value(pos, cm, opa, T)[0]) / (2 * h)
            assert abs(d - g.grad_color[3 * m:3 * m + 3, ch].sum()) < 1e-7 * max(1.0, abs(d))
    # rigid-motion identity: moving every vertex by a small rigid transform == left-multiplying the pose by it,
    # hence  sum_v [g_W ; P_v x g_W]  (world frame)  ==  Ad^T-transported dL/dtau.  Checked by direct FD instead:
    e = np.array([2e-7, -1e-7, 3e-7, 1e-7, 2e-7, -2e-7])
    G = scenes.se3_exp(e)
    pos_moved = pos @ G[:3, :3].T + G[:3, 3]
    Tm = np.eye(4)
    Tm[:3] = T
    T_right = (Tm @ G)[:3]                                 # T o G acts on the world points first
    assert abs(F.value(pos_moved, col, opa, T)[0] - F.value(pos, col, opa, T_right)[0]) < 1e-9
