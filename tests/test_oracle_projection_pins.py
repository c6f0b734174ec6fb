"""Pins of the oracle's tomographic projection matrix (sec. 2.5) against things other than itself."""
import numpy as np

from oracle import oracle as O

IDENT = [1.0, 0.0, 0.0, 0.0, 1.0, 0.0]


def _modes(n, ny, nx, seed):
    rng = np.random.default_rng(seed)
    yy, xx = np.mgrid[0:ny, 0:nx].astype(np.float64)
    out = []
    for _ in range(n):
        fx, fy = rng.uniform(-2, 2, 2) * 2 * np.pi / nx
        out.append(rng.normal() * np.cos(fx * xx + fy * yy + rng.uniform(0, 6)) + 0.2 * rng.normal(size=(ny, nx)))
    return np.array(out, dtype=np.float32)


def test_operand_is_the_modes_themselves_under_the_identity_and_a_shifted_copy_under_an_integer_shift():
    """One direction, identity map, grid = pupil grid: P is the cube, pixel-major, times the pupil; a direction whose
    map is an integer shift shows the shifted modes (zero fill), scaled by the square root of its weight."""
    cube = _modes(3, 12, 12, 1)
    pupil = (np.hypot(*np.mgrid[-5.5:6, -5.5:6]) <= 5.6).astype(np.float32)
    p = O.projection_operand(cube, [IDENT, [1, 0, 2.0, 0, 1, -1.0]], pupil, weights=[1.0, 4.0])
    assert p.shape == (2 * 144, 3)
    assert np.array_equal(p[:144], (cube.astype(np.float64) * pupil).reshape(3, 144).T)
    sh = np.zeros((3, 12, 12))
    sh[:, 1:, :10] = cube[:, :11, 2:]
    assert np.array_equal(p[144:], 2.0 * (sh * pupil).reshape(3, 144).T)


def test_exact_recovery_when_the_layer_lies_in_the_span_of_the_mirrors():
    """P_Layer = P_DM X and lambda = 0: the least-squares projection is X itself."""
    rng = np.random.default_rng(2)
    p_dm = rng.normal(size=(300, 12))
    x = rng.normal(size=(12, 5))
    assert np.allclose(O.projection_matrix(p_dm, p_dm @ x, 0.0), x, rtol=0, atol=1e-10)


def test_equals_ridge_regression_solved_without_normal_equations():
    """(A^T A + lambda I)^-1 A^T B is the minimiser of |A X - B|^2 + lambda |X|^2, i.e. the least-squares solution
    of the stacked system [A; sqrt(lambda) I] X = [B; 0] -- solved here by numpy's SVD-based lstsq."""
    rng = np.random.default_rng(3)
    a, b, lam = rng.normal(size=(200, 15)), rng.normal(size=(200, 7)), 0.37
    ref = np.linalg.lstsq(np.vstack([a, np.sqrt(lam) * np.eye(15)]), np.vstack([b, np.zeros((15, 7))]), rcond=None)[0]
    assert np.allclose(O.projection_matrix(a, b, lam), ref, rtol=0, atol=1e-11)


def test_strong_regularisation_limit_and_a_hand_computed_two_by_two():
    rng = np.random.default_rng(4)
    a, b = rng.normal(size=(50, 4)), rng.normal(size=(50, 3))
    lam = 1.0e9
    assert np.allclose(O.projection_matrix(a, b, lam) * lam, a.T @ b, rtol=1e-6)
    # A = [[1,0],[0,2],[0,0]], B = [[1],[1],[5]], lambda = 1: (A^T A + I) = diag(2, 5), A^T B = (1, 2) -> (1/2, 2/5)
    x = O.projection_matrix(np.array([[1.0, 0], [0, 2.0], [0, 0]]), np.array([[1.0], [1.0], [5.0]]), 1.0)
    assert np.allclose(x.ravel(), [0.5, 0.4], rtol=0, atol=1e-15)


def test_end_to_end_a_layer_that_is_a_mirror_seen_in_every_direction():
    """Two directions with different integer footprints, a 'layer' whose modes are mixtures of the mirror's own
    influence functions at the same altitude (same maps): P_opt is the mixing matrix."""
    cube = _modes(6, 20, 20, 5)
    pupil = np.ones((12, 12), np.float32)
    maps = [[1, 0, 3.0, 0, 1, -2.0], [1, 0, -1.0, 0, 1, 2.0]]
    mix = np.random.default_rng(6).normal(size=(6, 4))
    layer = np.tensordot(mix.T, cube.astype(np.float64), axes=1).astype(np.float32)
    p_dm = O.projection_operand(cube, maps, pupil)
    p_l = O.projection_operand(layer, maps, pupil)
    assert np.allclose(O.projection_matrix(p_dm, p_l, 0.0), mix, rtol=0, atol=1e-5)   # (float32 rounding of the mixtures)
