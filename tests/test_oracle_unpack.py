"""P30: the sensor-frame unpacking of reading S33 (oracle.unpack_rgbd) against what the definition fixes: closed-form
values, a hand-typed layout example, exact invertibility over all 8-bit / 16-bit codes."""
import numpy as np
import pytest


def test_p30_closed_forms(oracle_mod):
    rgb = np.zeros((1, 4, 3), np.uint8)
    rgb[0, :, 0] = [0, 255, 51, 128]
    dep = np.array([[0, 5000, 2500, 65535]], np.uint16)
    for prec, dt in (("f64", np.float64), ("f32", np.float32)):
        C, D = oracle_mod.unpack_rgbd(rgb, dep, 5000.0, prec)
        assert C.dtype == dt and D.dtype == dt and C.shape == (3, 1, 4) and D.shape == (1, 4)
        assert C[0, 0, 0] == 0.0 and C[0, 0, 1] == 1.0                         # exact end points
        assert C[0, 0, 2] == dt(51) / dt(255) and abs(C[0, 0, 2] - 0.2) < 1e-7
        assert abs(C[0, 0, 3] - 0.50196078431372548) < 1e-7
        assert D[0, 0] == 0.0 and D[0, 1] == 1.0 and D[0, 2] == 0.5             # 0 = no measurement; 5000 units = 1 m
        assert abs(D[0, 3] - 13.107) < 1e-6
        assert np.all(C[1:] == 0.0)


def test_p30_layout_hand_typed(oracle_mod):
    """A 2 x 3 frame with eighteen distinct colour codes: interleaved [y][x][c] in, planar [c][y][x] out."""
    rgb = np.array([[[10, 20, 30], [11, 21, 31], [12, 22, 32]],
                    [[13, 23, 33], [14, 24, 34], [15, 25, 35]]], np.uint8)
    dep = np.array([[100, 200, 300], [400, 500, 600]], np.uint16)
    C, D = oracle_mod.unpack_rgbd(rgb, dep, 1000.0)
    want = np.array([[[10, 11, 12], [13, 14, 15]],
                     [[20, 21, 22], [23, 24, 25]],
                     [[30, 31, 32], [33, 34, 35]]], np.float64) / 255.0
    assert np.array_equal(C, want)
    assert np.array_equal(D, np.array([[0.1, 0.2, 0.3], [0.4, 0.5, 0.6]]))


@pytest.mark.parametrize("prec", ["f32", "f64"])
def test_p30_every_code_survives_the_round_trip(oracle_mod, prec):
    """Quantising the unpacked values again gives back every 8-bit and every 16-bit code (both precisions)."""
    rgb = np.arange(256, dtype=np.uint8).reshape(1, 256, 1).repeat(3, axis=2)
    dep = np.zeros((1, 256), np.uint16)
    C, _ = oracle_mod.unpack_rgbd(rgb, dep, 5000.0, prec)
    assert np.array_equal(np.rint(C[1, 0].astype(np.float64) * 255.0).astype(np.int64), np.arange(256))
    assert np.all(np.diff(C[2, 0]) > 0)
    d = np.arange(65536, dtype=np.uint16).reshape(256, 256)
    for scale in (5000.0, 6553.5, 1000.0):
        _, D = oracle_mod.unpack_rgbd(np.zeros((256, 256, 3), np.uint8), d, scale, prec)
        assert np.array_equal(np.rint(D.astype(np.float64) * scale).astype(np.int64), d.astype(np.int64))
