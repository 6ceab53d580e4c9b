"""Pin P29: per-face window smoothness (reading S32; Triangle Splatting's learnable sigma): closed form on
the worked triangle, equivalence with the global constant, and central finite differences of dL/dsigma_m."""
import numpy as np

from conftest import IDENT, SimpleCam, SimpleParams, unproject
from test_oracle_closed_form import CAM, RGB, load_gold


def test_p29_window_value_per_face(oracle_mod):
    g = load_gold()
    uvz = np.stack([g["tri_u"], g["tri_v"], np.full(3, 2.0)], axis=1)
    # the same screen triangle twice, far apart in depth order does not matter: two faces side by side instead
    shift = np.array([0.0, 0.0, 0.0])
    pos_a = unproject(uvz, CAM)
    uvz_b = uvz.copy()
    uvz_b[:, 0] += 0.0
    uvz_b[:, 1] += 0.0
    px, py = g["pixel"].astype(int)
    for sa, want in ((0.5, g["I_sigma05"][0]), (1.0, g["I_sigma1"][0]), (2.0, g["I_sigma2"][0]), (1.7, 0.6 ** 1.7)):
        # global sigma is a decoy: the per-face value must win
        o = oracle_mod.Oracle(pos_a, RGB, np.ones(3), None, IDENT, CAM, SimpleParams(sigma=3.3), "f64", face_sigma=np.array([sa]))
        f = o.forward("brute")
        assert abs(f.alpha[py, px] - want) < 1e-12
    # a constant per-face array equals the global constant, bit for bit, forward and backward
    rng = np.random.default_rng(29)
    M = 40
    cen = np.stack([rng.uniform(-0.2, 0.4, M), rng.uniform(-0.2, 0.4, M), rng.uniform(2, 3, M)], 1)
    pos = (cen[:, None] + rng.normal(0, 0.08, (M, 3, 3))).reshape(-1, 3)
    col, opa = rng.uniform(0, 1, (3 * M, 3)), rng.uniform(0.3, 0.9, 3 * M)
    a = oracle_mod.Oracle(pos, col, opa, None, IDENT, CAM, SimpleParams(sigma=0.7), "f32")
    b = oracle_mod.Oracle(pos, col, opa, None, IDENT, CAM, SimpleParams(sigma=9.9), "f32", face_sigma=np.full(M, 0.7))
    fa, fb = a.forward("tiled"), b.forward("tiled")
    assert np.array_equal(fa.color, fb.color) and np.array_equal(fa.alpha, fb.alpha)
    gC = rng.normal(size=fa.color.shape)
    ga, gb = a.backward(gC, None, None), b.backward(gC, None, None)
    assert np.array_equal(ga.grad_pos, gb.grad_pos) and ga.grad_sigma is None and gb.grad_sigma is not None


def test_p29_sigma_gradient_finite_differences(oracle_mod):
    rng = np.random.default_rng(290)
    cam = SimpleCam(40, 30, 40.0, 40.0, 19.5, 14.5)
    prm = SimpleParams(sigma=1.0)
    M = 25
    cen = np.stack([rng.uniform(-0.7, 0.7, M), rng.uniform(-0.5, 0.5, M), rng.uniform(2, 3, M)], 1)
    pos = (cen[:, None] + rng.normal(0, 0.2, (M, 3, 3))).reshape(-1, 3)
    pos[:, 2] = np.maximum(pos[:, 2], 1.0)
    col, opa = rng.uniform(0, 1, (3 * M, 3)), rng.uniform(0.3, 0.9, 3 * M)
    sig = rng.uniform(0.4, 2.0, M)
    wC, wD, wA = rng.normal(size=(3, 30, 40)), rng.normal(size=(30, 40)), rng.normal(size=(30, 40))

    def loss(s):
        f = oracle_mod.Oracle(pos, col, opa, None, IDENT, cam, prm, "f64", face_sigma=s).forward("brute")
        return float((wC * f.color).sum() + (wD * f.depth).sum() + (wA * f.alpha).sum())

    o = oracle_mod.Oracle(pos, col, opa, None, IDENT, cam, prm, "f64", face_sigma=sig)
    g = o.backward(wC, wD, wA, mode="brute")
    assert np.abs(g.grad_sigma).max() > 0
    h = 1e-6
    for m in range(M):
        sp, sm = sig.copy(), sig.copy()
        sp[m] += h
        sm[m] -= h
        fd = (loss(sp) - loss(sm)) / (2 * h)
        assert abs(fd - g.grad_sigma[m]) <= 1e-6 * max(1.0, abs(fd)), (m, fd, g.grad_sigma[m])
    # positions still differentiate correctly with per-face sigma (the dI/dx factor uses the face's own sigma)
    for idx in rng.choice(pos.size, 15, replace=False):
        v, k = divmod(int(idx), 3)
        pp, pm = pos.copy(), pos.copy()
        pp[v, k] += h
        pm[v, k] -= h
        lp = oracle_mod.Oracle(pp, col, opa, None, IDENT, cam, prm, "f64", face_sigma=sig).forward("brute")
        lm = oracle_mod.Oracle(pm, col, opa, None, IDENT, cam, prm, "f64", face_sigma=sig).forward("brute")
        f0 = o.forward("brute")
        if not (np.array_equal(lp.n_contrib, f0.n_contrib) and np.array_equal(lm.n_contrib, f0.n_contrib)):
            continue
        fd = (float((wC * lp.color).sum() + (wD * lp.depth).sum() + (wA * lp.alpha).sum())
              - float((wC * lm.color).sum() + (wD * lm.depth).sum() + (wA * lm.alpha).sum())) / (2 * h)
        assert abs(fd - g.grad_pos[v, k]) <= 2e-5 * max(1.0, abs(fd)), (v, k, fd, g.grad_pos[v, k])
