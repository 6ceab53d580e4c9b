"""Pins of the oracle's equilateral regulariser E_equi (Eq. 14): zero on an equilateral face,
the hand value of a right isosceles face, invariance under rigid motion and scale, finite differences."""
import numpy as np


def test_equilateral_is_zero_and_right_isosceles_closed_form(oracle_mod):
    eq = np.array([[0, 0, 0], [1, 0, 0], [0.5, np.sqrt(3) / 2, 0]], float)
    E, g = oracle_mod.equi(eq)
    assert abs(E) < 1e-30 and np.abs(g).max() < 1e-15
    # angles 90, 45, 45 degrees: cosines 0, 1/sqrt2, 1/sqrt2
    ri = np.array([[0, 0, 0], [2, 0, 0], [0, 2, 0]], float)
    E, _ = oracle_mod.equi(ri, grad=False)
    assert abs(E - (0.25 + 2 * (np.sqrt(0.5) - 0.5) ** 2) / 3) < 1e-15
    # mean over faces
    E2, _ = oracle_mod.equi(np.concatenate([eq, ri]), grad=False)
    assert abs(E2 - E / 2) < 1e-15


def test_invariances_and_indexed_faces(oracle_mod):
    rng = np.random.default_rng(0)
    pos = rng.normal(size=(30, 3))
    E, _ = oracle_mod.equi(pos, grad=False)
    Q, _ = np.linalg.qr(rng.normal(size=(3, 3)))
    E2, _ = oracle_mod.equi(3.7 * pos @ Q.T + np.array([1.0, -2.0, 0.5]), grad=False)
    assert abs(E - E2) < 1e-13                       # angles do not change under similarity transforms
    faces = np.arange(30, dtype=np.int32).reshape(-1, 3)
    E3, g3 = oracle_mod.equi(pos, faces)
    _, g = oracle_mod.equi(pos)
    assert abs(E - E3) < 1e-15 and np.allclose(g, g3)
    assert np.abs(g.reshape(-1, 3, 3).sum(axis=1)).max() < 1e-12    # translation invariance: face gradients sum to 0


def test_gradient_matches_central_differences(oracle_mod):
    rng = np.random.default_rng(1)
    pos = rng.normal(size=(24, 3))
    faces = rng.integers(0, 24, size=(20, 3)).astype(np.int32)
    faces = faces[(faces[:, 0] != faces[:, 1]) & (faces[:, 1] != faces[:, 2]) & (faces[:, 0] != faces[:, 2])]
    E, g = oracle_mod.equi(pos, faces, weight=2.5)
    h = 1e-6
    for _ in range(30):
        i, a = rng.integers(24), rng.integers(3)
        pp, pm = pos.copy(), pos.copy()
        pp[i, a] += h
        pm[i, a] -= h
        fd = 2.5 * (oracle_mod.equi(pp, faces, grad=False)[0] - oracle_mod.equi(pm, faces, grad=False)[0]) / (2 * h)
        assert abs(fd - g[i, a]) <= 1e-8 + 1e-6 * abs(fd)
    E32, g32 = oracle_mod.equi(pos, faces, weight=2.5, prec="f32")
    assert abs(E32 - E) < 1e-6 and np.abs(g32 - g).max() < 1e-5
