"""Pin P28: tight binning (reading S31: a face is binned only into the tiles its triangle meets).  The rule may only
drop (tile, face) pairs that cannot contribute, so what it must leave unchanged is fixed by the definition of the
image itself: the tiled render with tight lists equals the BRUTE-FORCE render (no tiles at all) bit for bit, and the
gradients do too; what it must change is counted by independent geometry (exact rational triangle-box overlap)."""
from fractions import Fraction

import numpy as np
import pytest

from paper_2605_31419_b200 import scenes


def _params(sc, tight):
    p = scenes.Params(**{**sc.params.__dict__, "tight_binning": tight})
    return p


@pytest.mark.parametrize("maker", [lambda: scenes.config0(n_faces=1500), lambda: scenes.config2(n_faces=6000)])
@pytest.mark.parametrize("prec", ["f32", "f64"])
def test_p28_tight_lists_render_the_brute_force_image(oracle_mod, maker, prec):
    sc = maker()
    if sc.cam.width > 400:                                   # keep the brute-force pass affordable
        sc.cam = scenes.Camera(240, 136, 120.0, 120.0, 119.5, 67.5)
    loose = oracle_mod.Oracle(sc.pos, sc.color, sc.opacity, None, sc.T_start[0], sc.cam, _params(sc, False), prec)
    tight = oracle_mod.Oracle(sc.pos, sc.color, sc.opacity, None, sc.T_start[0], sc.cam, _params(sc, True), prec)
    bl, bt = loose.bin_sort(), tight.bin_sort()
    assert bt.P < bl.P and bt.P > 0.5 * bl.P                # pairs are dropped, not many
    # the tight list is a sub-list of the loose one, in the same order
    kl = {(int(k), int(v)) for k, v in zip(bl.keys, bl.vals)}
    assert all((int(k), int(v)) in kl for k, v in zip(bt.keys, bt.vals))
    assert np.all(np.diff(bt.keys.astype(np.uint64)) >= 0) if prec == "f32" else True
    assert np.array_equal(tight.project().tiles_touched.sum(dtype=np.int64), bt.P)
    fb, ft, fl = tight.forward("brute"), tight.forward("tiled"), loose.forward("tiled")
    for a, b in ((ft.color, fb.color), (ft.depth, fb.depth), (ft.alpha, fb.alpha), (ft.color, fl.color), (ft.alpha, fl.alpha)):
        assert np.array_equal(a, b)
    rng = np.random.default_rng(28)
    gC, gD = rng.normal(size=ft.color.shape), rng.normal(size=ft.depth.shape)
    gt, gl = tight.backward(gC, gD, None), loose.backward(gC, gD, None)
    assert np.array_equal(gt.grad_pos, gl.grad_pos) and np.array_equal(gt.dL_dtau, gl.dL_dtau)


def _tri_box_overlap_exact(tri, x0, y0, x1, y1):
    """Exact (rational) test: does the closed triangle meet the closed box?  Separating axes: box axes + edge normals."""
    P = [(Fraction(float(a)), Fraction(float(b))) for a, b in tri]
    xs, ys = [p[0] for p in P], [p[1] for p in P]
    if max(xs) < x0 or min(xs) > x1 or max(ys) < y0 or min(ys) > y1:
        return False
    corners = [(Fraction(x0), Fraction(y0)), (Fraction(x1), Fraction(y0)), (Fraction(x0), Fraction(y1)), (Fraction(x1), Fraction(y1))]
    for k in range(3):
        a, b, c = P[k], P[(k + 1) % 3], P[(k + 2) % 3]
        nx, ny = b[1] - a[1], -(b[0] - a[0])
        side_c = nx * (c[0] - a[0]) + ny * (c[1] - a[1])
        vals = [nx * (q[0] - a[0]) + ny * (q[1] - a[1]) for q in corners]
        if side_c > 0 and max(vals) < 0:
            return False
        if side_c < 0 and min(vals) > 0:
            return False
    return True


def test_p28_rule_against_exact_overlap(oracle_mod):
    """Every pair the rule keeps-or-drops is checked against exact rational geometry: a dropped pair's triangle misses
    the tile's pixel box (n rect) altogether, and a pair whose triangle reaches more than 2e-3 px into the box is kept."""
    sc = scenes.config2(n_faces=4000)
    sc.cam = scenes.Camera(240, 136, 120.0, 120.0, 119.5, 67.5)
    loose = oracle_mod.Oracle(sc.pos, sc.color, sc.opacity, None, sc.T_start[0], sc.cam, _params(sc, False), "f32")
    tight = oracle_mod.Oracle(sc.pos, sc.color, sc.opacity, None, sc.T_start[0], sc.cam, _params(sc, True), "f32")
    pr = loose.project()
    kept = {(int(k) >> 32, int(v)) for k, v in zip(tight.bin_sort().keys, tight.bin_sort().vals)}
    tiles_x = (sc.cam.width + 15) // 16
    dropped = 0
    for k, m in zip(loose.bin_sort().keys, loose.bin_sort().vals):
        t, m = int(k) >> 32, int(m)
        tx, ty = t % tiles_x, t // tiles_x
        x0, y0, x1, y1 = (int(v) for v in pr.rect[m])
        bx0, bx1, by0, by1 = max(x0, 16 * tx), min(x1, 16 * tx + 15), max(y0, 16 * ty), min(y1, 16 * ty + 15)
        tri = pr.scr[m].reshape(3, 3)[:, :2]
        if (t, m) in kept:
            continue
        dropped += 1
        assert not _tri_box_overlap_exact(tri, bx0, by0, bx1, by1), (t, m)
    assert dropped > 20
