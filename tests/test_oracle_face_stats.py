"""Pins of the oracle's per-face statistics (map-management inputs): pixel counts against
Pick's theorem on the 30-40-50 triangle of the worked example, the projected area against the triangle's area,
occlusion by a fully opaque pixel, consistency with the forward render's hit counter, brute == tiled."""
import numpy as np
import pytest

from conftest import IDENT, SimpleCam, SimpleParams, unproject
from paper_2605_31419_b200 import scenes

CAM = SimpleCam(64, 64, 100.0, 100.0, 0.0, 0.0)
TRI = np.array([[8.0, 8.0], [38.0, 8.0], [8.0, 48.0]])      # legs 30 and 40: area 600, 80 boundary lattice points


def oracle_for(tso, uvz, opa, prm, prec="f64"):
    pos = unproject(np.asarray(uvz, dtype=np.float64).reshape(-1, 3), CAM)
    n = pos.shape[0]
    return tso.Oracle(pos, np.tile(np.eye(3), (n // 3, 1)), opa, None, IDENT, CAM, prm, prec)


@pytest.mark.parametrize("prec", ["f64", "f32"])
def test_pixel_count_is_picks_theorem_and_area(oracle_mod, prec):
    # interior lattice points I = A - B/2 + 1 = 600 - 40 + 1 = 561; boundary pixels have I(p) = 0 up to rounding of the
    # unprojection, alpha_min = 1e-6 removes them (the nearest interior pixel has x >= 0.02)
    uvz = np.concatenate([TRI, np.full((3, 1), 2.0)], axis=1)
    o = oracle_for(oracle_mod, uvz, np.ones(3), SimpleParams(sigma=1.0, alpha_min=1e-6), prec)
    for mode in ("brute", "tiled"):
        st = o.face_stats(mode)
        assert st.face_pixels.tolist() == [561]
        assert abs(st.proj_area[0] - 600.0) < (1e-9 if prec == "f64" else 1e-3)


def test_opaque_pixel_hides_the_face_behind(oracle_mod):
    # two copies of the triangle, opacity 1: only at the incentre (18,18) is alpha exactly 1, the walk of that pixel
    # stops there (T = 0 <= t_min), so the face behind is counted on one pixel fewer
    uvz = np.concatenate([np.concatenate([TRI, np.full((3, 1), 2.0)], axis=1),
                          np.concatenate([TRI, np.full((3, 1), 3.0)], axis=1)])
    o = oracle_for(oracle_mod, uvz, np.ones(6), SimpleParams(sigma=1.0, alpha_min=1e-6, t_min=1e-4))
    st = o.face_stats("tiled")
    assert st.face_pixels.tolist() == [561, 560]
    # a culled face (behind the camera) has neither pixels nor area
    uvz[3:, 2] = -1.0
    o = oracle_for(oracle_mod, uvz, np.ones(6), SimpleParams(sigma=1.0, alpha_min=1e-6, t_min=1e-4))
    st = o.face_stats("tiled")
    assert st.face_pixels.tolist() == [561, 0] and st.proj_area[1] == 0.0


@pytest.mark.parametrize("prec", ["f64", "f32"])
def test_counts_sum_to_the_hit_counter_and_brute_equals_tiled(oracle_mod, prec):
    sc = scenes.config0(n_faces=400)
    o = oracle_mod.Oracle(sc.pos, sc.color, sc.opacity, None, sc.T_gt[0], sc.cam, sc.params, prec)
    f = o.forward("tiled")
    st, sb = o.face_stats("tiled"), o.face_stats("brute")
    assert int(st.face_pixels.sum()) == int(f.counters[2]) > 0
    assert np.array_equal(st.face_pixels, sb.face_pixels)
    pr = o.project()
    assert np.all(st.face_pixels[pr.visible == 0] == 0) and np.all(st.proj_area[pr.visible == 0] == 0)
    assert np.all(st.proj_area[pr.visible == 1] > 0)
    # every pixel of a face lies in its rect: count <= rect area
    rect_area = (pr.rect[:, 2] - pr.rect[:, 0] + 1).astype(np.int64) * (pr.rect[:, 3] - pr.rect[:, 1] + 1)
    assert np.all(st.face_pixels[pr.visible == 1] <= rect_area[pr.visible == 1])
