"""Pins of the float64 oracle against things other than itself (CPU only).

The paper prints no worked numerical example, so the oracle is pinned by what the
mathematics fixes: closed forms, invariants, library special cases and brute force; each test
names the step of oracle/synim_oracle.c it would catch a mistake in.
"""
import math

import numpy as np
import pytest

from oracle import oracle as O
from paper_2606_07759_b200 import workloads as W

IDENT = [1.0, 0.0, 0.0, 0.0, 1.0, 0.0]


def rot_affine(deg, mag=1.0, sx=0.0, sy=0.0):
    t = math.radians(deg)
    return [math.cos(t) / mag, math.sin(t) / mag, sx, -math.sin(t) / mag, math.cos(t) / mag, sy]


def centred(ny, nx):
    yy, xx = np.mgrid[0:ny, 0:nx].astype(np.float64)
    return xx - (nx - 1) / 2.0, yy - (ny - 1) / 2.0


def full_wfs(n_subap, n_pix, rng=None):
    m = n_subap * n_pix
    pupil = np.ones((m, m), np.float32) if rng is None else rng.uniform(0.1, 1.0, (m, m)).astype(np.float32)
    return pupil, np.ones((n_subap, n_subap), np.uint8)


# ---------------------------------------------------------------- steps 1-2: resampling
def test_identity_leaves_input_unchanged_bitwise():
    rng = np.random.default_rng(1)
    g = rng.normal(size=(24, 24)).astype(np.float32)
    assert np.array_equal(O.resample(g, 24, IDENT), g.astype(np.float64))


def test_integer_shift_is_shifted_array_with_zero_fill():
    rng = np.random.default_rng(2)
    g = rng.normal(size=(20, 20)).astype(np.float32)
    phi = O.resample(g, 20, [1, 0, 3.0, 0, 1, -2.0])          # col = j+3, row = i-2
    ref = np.zeros((20, 20))
    ref[2:, :17] = g[:18, 3:]
    assert np.array_equal(phi, ref)


@pytest.mark.parametrize("k", [0, 1, 2, 3])
def test_quarter_turns_equal_rot90_bitwise(k):
    """Exactly integer rotation matrices reproduce np.rot90(g, -k): fixes the pixel-centre
    convention (R2) and the sense of rotation (+theta turns +x toward +y)."""
    rng = np.random.default_rng(3)
    g = rng.normal(size=(16, 16)).astype(np.float32)
    c, s = [(1, 0), (0, 1), (-1, 0), (0, -1)][k]
    phi = O.resample(g, 16, [c, s, 0, -s, c, 0])
    assert np.array_equal(phi, np.rot90(g, -k).astype(np.float64))
    # and the composed matrix for rot_deg = 90k agrees to rounding
    a = O.compose_affine(W.physical(rot_deg=90.0 * k))
    assert np.allclose(O.resample(g, 16, a), np.rot90(g, -k), atol=1e-12)


def test_bilinear_equals_scipy_affine_transform_and_torch_grid_sample():
    """Step 2 against two library routines (R3/R4): order-1 spline with zero 'grid-constant'
    boundary, and grid_sample(bilinear, zeros, align_corners=True)."""
    import scipy.ndimage as ndi
    import torch
    rng = np.random.default_rng(4)
    ny, nx, m = 30, 34, 36                       # WFS grid overruns the source grid
    g = rng.normal(size=(ny, nx)).astype(np.float32)
    a = rot_affine(33.0, mag=0.9, sx=1.7, sy=-2.3)
    a[1] *= 1.1                                  # not a pure similarity
    phi = O.resample(g, m, a)
    cw, cx, cy = (m - 1) / 2.0, (nx - 1) / 2.0, (ny - 1) / 2.0
    mat = np.array([[a[4], a[3]], [a[1], a[0]]])
    off = np.array([a[5] + cy - cw * (a[3] + a[4]), a[2] + cx - cw * (a[0] + a[1])])
    ref = ndi.affine_transform(g.astype(np.float64), mat, offset=off, output_shape=(m, m), order=1,
                               mode="grid-constant", cval=0.0)
    assert np.allclose(phi, ref, atol=1e-12)
    ii, jj = np.mgrid[0:m, 0:m].astype(np.float64)
    col = a[0] * (jj - cw) + a[1] * (ii - cw) + a[2] + cx
    row = a[3] * (jj - cw) + a[4] * (ii - cw) + a[5] + cy
    grid = torch.from_numpy(np.stack([2 * col / (nx - 1) - 1, 2 * row / (ny - 1) - 1], axis=-1))[None]
    t = torch.nn.functional.grid_sample(torch.from_numpy(g.astype(np.float64))[None, None], grid,
                                        mode="bilinear", padding_mode="zeros", align_corners=True)
    assert np.allclose(phi, t[0, 0].numpy(), atol=1e-12)


def test_halo_grid_is_the_same_map_evaluated_one_pixel_further():
    rng = np.random.default_rng(5)
    g = rng.normal(size=(20, 20)).astype(np.float32)
    a = rot_affine(10.0, 1.05, 0.3, 0.4)
    h = O.resample(g, 12, a, halo=True)
    assert np.array_equal(h[1:-1, 1:-1], O.resample(g, 12, a))
    # halo pixel (-1,-1) of a 12-grid == pixel (0,0) of a 14-grid with the same matrix
    assert np.array_equal(h, O.resample(g, 14, a))


# ---------------------------------------------------------------- steps 3-4: slopes
@pytest.mark.parametrize("mode", [O.ND, O.GTILT])
def test_pure_tilt_gives_constant_slopes_equal_to_AT_tilt(mode):
    """phi = a x_s + b y_s  ->  every slope = (a a0 + b a3, a a1 + b a4): catches a transposed
    matrix, a wrong stencil width, a missing /2, differentiation in the wrong frame (R5, R6)."""
    xs, ys = centred(96, 96)
    ta, tb = 0.37, -0.52
    g = (ta * xs + tb * ys).astype(np.float32)[None]
    ta, tb = float(np.float32(ta)), float(np.float32(tb))
    rng = np.random.default_rng(6)
    pupil, valid = full_wfs(6, 5, rng)
    a = rot_affine(27.0, mag=1.07, sx=0.31, sy=-0.44)
    s = O.slopes_wfs(g, pupil, 6, 5, valid, a, scale=1.5, mode=mode)[0]
    assert np.allclose(s[:36], 1.5 * (ta * a[0] + tb * a[3]), atol=1e-6)
    assert np.allclose(s[36:], 1.5 * (ta * a[1] + tb * a[4]), atol=1e-6)


def test_quadratic_gives_linear_slopes_under_fractional_shift():
    """g = x^2 with a pure shift d: linear interpolation of a parabola adds the constant
    f(1-f), so the central difference is exactly 2(x_w+d); the weighted subaperture mean is
    2(sum P x / sum P + d).  Same for y.  Catches weighting / normalisation mistakes (R7)."""
    xs, ys = centred(64, 64)
    rng = np.random.default_rng(7)
    n_subap, n_pix = 5, 8
    pupil, valid = full_wfs(n_subap, n_pix, rng)
    xw, yw = centred(40, 40)
    p = pupil.astype(np.float64).reshape(n_subap, n_pix, n_subap, n_pix)
    w = p.sum(axis=(1, 3))
    xbar = (p * xw.reshape(n_subap, n_pix, n_subap, n_pix)).sum(axis=(1, 3)) / w
    ybar = (p * yw.reshape(n_subap, n_pix, n_subap, n_pix)).sum(axis=(1, 3)) / w
    dx, dy = 0.3, -1.6
    a = [1, 0, dx, 0, 1, dy]
    sx = O.slopes_wfs((xs ** 2).astype(np.float32)[None], pupil, n_subap, n_pix, valid, a)[0]
    sy = O.slopes_wfs((ys ** 2).astype(np.float32)[None], pupil, n_subap, n_pix, valid, a)[0]
    assert np.allclose(sx[:25], 2 * (xbar.ravel() + dx), atol=1e-10)
    assert np.allclose(sx[25:], 0, atol=1e-10)
    assert np.allclose(sy[25:], 2 * (ybar.ravel() + dy), atol=1e-10)
    assert np.allclose(sy[:25], 0, atol=1e-10)


def test_row_order_valid_subaps_row_major_x_then_y():
    """With g = x^2 + 10 y^2... each subaperture has its own (sx, sy); a mask with holes must
    drop exactly those entries and keep row-major order (R9, R10)."""
    xs, ys = centred(48, 48)
    g = (xs ** 2 + 3.0 * ys ** 2).astype(np.float32)[None]
    n_subap, n_pix = 6, 6
    pupil = np.ones((36, 36), np.float32)
    rng = np.random.default_rng(8)
    valid = (rng.uniform(size=(6, 6)) > 0.4).astype(np.uint8)
    s = O.slopes_wfs(g, pupil, n_subap, n_pix, valid, IDENT)[0]
    centre = (np.arange(6) * 6 + 2.5) - 17.5
    exp_x = np.array([2 * centre[b] for a in range(6) for b in range(6) if valid[a, b]])
    exp_y = np.array([6 * centre[a] for a in range(6) for b in range(6) if valid[a, b]])
    nv = int(valid.sum())
    assert s.shape == (2 * nv,)
    assert np.allclose(s[:nv], exp_x, atol=1e-10) and np.allclose(s[nv:], exp_y, atol=1e-10)


def test_columns_are_linear_under_sums_of_influence_functions():
    rng = np.random.default_rng(9)
    g1 = (rng.integers(-64, 64, size=(40, 40)) / 16.0).astype(np.float32)
    g2 = (rng.integers(-64, 64, size=(40, 40)) / 8.0).astype(np.float32)
    cube = np.stack([g1, g2, 2.0 * g1 - 0.5 * g2]).astype(np.float32)   # exact in float32
    pupil, valid = full_wfs(4, 8, rng)
    for mode in (O.ND, O.GTILT):
        s = O.slopes_wfs(cube, pupil, 4, 8, valid, rot_affine(12.0, 0.97, 0.2, 0.1), mode=mode)
        assert np.allclose(s[2], 2.0 * s[0] - 0.5 * s[1], atol=1e-12)


def test_telescoping_identity_on_full_subapertures():
    """P = 1 on a full subaperture: sum_S Dx = 1/2 sum_rows (phi[.,j0+n]+phi[.,j0+n-1]-phi[.,j0]-phi[.,j0-1])."""
    rng = np.random.default_rng(10)
    g = rng.normal(size=(40, 40)).astype(np.float32)
    n_subap, n_pix = 4, 7
    m = n_subap * n_pix
    a = rot_affine(-21.0, 1.1, 0.6, -0.2)
    pupil, valid = full_wfs(n_subap, n_pix)
    s = O.slopes_wfs(g[None], pupil, n_subap, n_pix, valid, a)[0]
    h = O.resample(g, m, a, halo=True)           # h[i+1][j+1] = phi[i][j]
    k = 0
    for sa in range(n_subap):
        for sb in range(n_subap):
            i0, j0 = sa * n_pix, sb * n_pix
            rows = slice(i0 + 1, i0 + n_pix + 1)
            cols = slice(j0 + 1, j0 + n_pix + 1)
            ex = 0.5 * (h[rows, j0 + n_pix + 1] + h[rows, j0 + n_pix] - h[rows, j0 + 1] - h[rows, j0]).sum()
            ey = 0.5 * (h[i0 + n_pix + 1, cols] + h[i0 + n_pix, cols] - h[i0 + 1, cols] - h[i0, cols]).sum()
            assert abs(s[k] - ex / n_pix ** 2) < 1e-12
            assert abs(s[n_subap ** 2 + k] - ey / n_pix ** 2) < 1e-12
            k += 1


def _brute_force(g, ny, nx, pupil, n_subap, n_pix, valid, a, scale):
    """Scalar pure-Python evaluation straight from the definitions (independent code)."""
    m = n_subap * n_pix

    def sample(i, j):
        xw, yw = j - (m - 1) / 2.0, i - (m - 1) / 2.0
        col = a[0] * xw + a[1] * yw + a[2] + (nx - 1) / 2.0
        row = a[3] * xw + a[4] * yw + a[5] + (ny - 1) / 2.0
        c0, r0 = math.floor(col), math.floor(row)
        tot = 0.0
        for dr in (0, 1):
            for dc in (0, 1):
                r, c = r0 + dr, c0 + dc
                if 0 <= r < ny and 0 <= c < nx:
                    wgt = (1 - abs(col - c)) * (1 - abs(row - r))      # tent weights
                    tot += wgt * float(g[r][c])
        return tot

    sx, sy = [], []
    for sa in range(n_subap):
        for sb in range(n_subap):
            if not valid[sa][sb]:
                continue
            wsum = ax = ay = 0.0
            for i in range(sa * n_pix, (sa + 1) * n_pix):
                for j in range(sb * n_pix, (sb + 1) * n_pix):
                    p = float(pupil[i][j])
                    wsum += p
                    ax += p * (sample(i, j + 1) - sample(i, j - 1)) / 2
                    ay += p * (sample(i + 1, j) - sample(i - 1, j)) / 2
            sx.append(scale * ax / wsum)
            sy.append(scale * ay / wsum)
    return np.array(sx + sy)


@pytest.mark.parametrize("seed", [11, 12, 13])
def test_brute_force_per_pixel_evaluation_on_tiny_grids(seed):
    rng = np.random.default_rng(seed)
    ny, nx, n_subap, n_pix = 14, 16, 3, 4
    g = rng.normal(size=(ny, nx)).astype(np.float32)
    pupil = rng.uniform(0, 1, (12, 12)).astype(np.float32)
    valid = np.ones((3, 3), np.uint8)
    valid[rng.integers(0, 3), rng.integers(0, 3)] = 0
    a = rot_affine(rng.uniform(-180, 180), rng.uniform(0.8, 1.3), rng.uniform(-2, 2), rng.uniform(-2, 2))
    a[0] *= 1.07                                 # anamorphic
    s = O.slopes_wfs(g[None], pupil, n_subap, n_pix, valid, a, scale=0.7)[0]
    assert np.allclose(s, _brute_force(g, ny, nx, pupil, n_subap, n_pix, valid, a, 0.7), atol=1e-12)


def test_impulse_responses_assemble_the_linear_operator():
    rng = np.random.default_rng(14)
    n = 10
    imp = np.eye(n * n, dtype=np.float32).reshape(n * n, n, n)
    pupil, valid = full_wfs(2, 4, rng)
    a = rot_affine(40.0, 0.9, 0.4, -0.3)
    S = O.slopes_wfs(imp, pupil, 2, 4, valid, a).T                 # [rows][n*n]
    g = rng.normal(size=(n, n)).astype(np.float32)
    direct = O.slopes_wfs(g[None], pupil, 2, 4, valid, a)[0]
    assert np.allclose(S @ g.astype(np.float64).ravel(), direct, atol=1e-12)


def test_integer_subaperture_shift_moves_the_response_by_whole_subapertures():
    """Translation equivariance (used for R12: a footprint shift of k*n_pix pixels moves the
    response by k subapertures)."""
    wl = W.make_config(1)
    g = wl.cube[48:49]
    pupil, valid = full_wfs(10, 8)
    s0 = O.slopes_wfs(g, pupil, 10, 8, valid, IDENT)[0].reshape(2, 10, 10)
    s1 = O.slopes_wfs(g, pupil, 10, 8, valid, [1, 0, 8.0, 0, 1, -16.0])[0].reshape(2, 10, 10)
    assert np.abs(s0).max() > 1e-3
    assert np.allclose(s1[:, 2:, :9], s0[:, :8, 1:], atol=1e-14)


# ---------------------------------------------------------------- G-tilt comparison mode
def test_gtilt_is_exact_on_parabola_and_differs_from_nd_on_a_gaussian():
    xs, _ = centred(64, 64)
    pupil, valid = full_wfs(5, 8)
    s = O.slopes_wfs((xs ** 2).astype(np.float32)[None], pupil, 5, 8, valid, IDENT, mode=O.GTILT)[0]
    xw, _ = centred(40, 40)
    mid = np.array([0.5 * (xw[0, b * 8] + xw[0, b * 8 + 7]) for b in range(5)])
    assert np.allclose(s[:25].reshape(5, 5), 2 * mid[None, :], atol=1e-10)
    wl = W.make_config(1)
    w = wl.wfs[0]
    nd = O.slopes_wfs(wl.cube[40:41], w.pupil, 10, 8, w.valid, IDENT, mode=O.ND)[0]
    gt = O.slopes_wfs(wl.cube[40:41], w.pupil, 10, 8, w.valid, IDENT, mode=O.GTILT)[0]
    rel = np.linalg.norm(nd - gt) / np.linalg.norm(nd)
    assert 1e-3 < rel < 0.2                      # the two estimators are distinguishable


def test_gtilt_partial_subaperture_uses_first_and_last_valid_pixel():
    xs, ys = centred(32, 32)
    g = (0.25 * xs).astype(np.float32)[None]
    pupil = np.zeros((16, 16), np.float32)
    pupil[:, 3:14] = 1.0                        # columns 0-2 and 14-15 dark
    valid = np.ones((2, 2), np.uint8)
    s = O.slopes_wfs(g, pupil, 2, 8, valid, IDENT, mode=O.GTILT)[0]
    assert np.allclose(s[:4], 0.25, atol=1e-12) and np.allclose(s[4:], 0.0, atol=1e-12)


def test_gtilt_threshold_and_aggregation_on_a_ragged_fractional_pupil():
    """Pins the two decisions of reading R13 that a tilt or a full pupil cannot see (PAPER.md:61
    "evaluates the phase difference strictly at the subaperture edges"):
      * a pixel is valid iff P >= 0.5 (a pixel with 0 < P < 0.5 is NOT an edge; P == 0.5 is),
      * the estimator is sum(num) / sum(den) over the pixel rows, not the mean of per-row ratios.
    phi = x^2 (y^2) under the identity map is exact on integer pixels, so the closed form is
    sum_rows(x_l^2 - x_f^2) / sum_rows(x_l - x_f) with (f, l) the first / last pixel of each row
    with P >= 0.5.  Rows have different spans and the span ends are flanked by pixels of weight
    0.3 / 0.49 (invalid) or exactly 0.5 (valid), so either mistake changes the value."""
    n = 12
    m = 2 * n
    xs, ys = centred(m, m)
    spans = [(2, 9), (1, 10), (3, 9), (0, 11), (4, 10), (2, 9), (4, 11), (1, 9), (3, 11), (0, 9), (1, 10), (2, 11)]
    for axis in (0, 1):
        pupil = np.zeros((m, m), np.float32)
        expect = np.zeros((2, 2))
        for a in range(2):
            for b in range(2):
                num = den = 0.0
                ratios = []
                for q, (f, l) in enumerate(spans):
                    f, l = (f + a + b) % 5, l - ((a + 2 * b) % 3)           # a different ragged shape per subaperture
                    line = np.zeros(n, np.float32)
                    line[f:l + 1] = 1.0
                    line[f] = 0.5                                           # exactly 0.5 counts as valid
                    if f > 0:
                        line[f - 1] = 0.3 if q % 2 else 0.49                # fractional, below the threshold
                    if l + 1 < n:
                        line[l + 1] = 0.3
                    if axis == 0:
                        pupil[a * n + q, b * n:(b + 1) * n] = line
                        c = xs[0, b * n:(b + 1) * n]
                    else:
                        pupil[a * n:(a + 1) * n, b * n + q] = line
                        c = ys[a * n:(a + 1) * n, 0]
                    num += c[l] ** 2 - c[f] ** 2
                    den += c[l] - c[f]
                    ratios.append((c[l] ** 2 - c[f] ** 2) / (c[l] - c[f]))
                expect[a, b] = num / den
                assert abs(np.mean(ratios) - expect[a, b]) > 1e-2           # the aggregation is visible here
        g = ((xs if axis == 0 else ys) ** 2).astype(np.float32)[None]
        s = O.slopes_wfs(g, pupil, 2, n, np.ones((2, 2), np.uint8), IDENT, scale=1.0, mode=O.GTILT)[0]
        got = s[:4] if axis == 0 else s[4:]
        assert np.allclose(got.reshape(2, 2), expect, rtol=0, atol=1e-12), (axis, got, expect)
        # the value with every lit pixel (P > 0) taken as valid is different: the threshold is visible too
        lit = pupil > 0
        alt = np.zeros((2, 2))
        for a in range(2):
            for b in range(2):
                num = den = 0.0
                for q in range(n):
                    row = lit[a * n + q, b * n:(b + 1) * n] if axis == 0 else lit[a * n:(a + 1) * n, b * n + q]
                    c = xs[0, b * n:(b + 1) * n] if axis == 0 else ys[a * n:(a + 1) * n, 0]
                    k = np.flatnonzero(row)
                    num += c[k[-1]] ** 2 - c[k[0]] ** 2
                    den += c[k[-1]] - c[k[0]]
                alt[a, b] = num / den
        assert np.abs(alt - expect).min() > 1e-2


# ---------------------------------------------------------------- composition helper
def _sequential(phys, pt):
    """Apply the individual maps to a point one after another (independent restatement)."""
    x = np.array(pt, dtype=np.float64) * phys["wfs_pitch_src_px"]
    x = x - np.array([phys["shift_x"], phys["shift_y"]])
    t = math.radians(phys["rot_deg"])
    x = np.array([math.cos(t) * x[0] + math.sin(t) * x[1], -math.sin(t) * x[0] + math.cos(t) * x[1]])
    x = x / np.array([phys["mag_x"], phys["mag_y"]])
    h, H = phys["dm_height_m"], phys["gs_range_m"]
    kappa = 1.0 if math.isinf(H) else 1.0 - h / H
    th = phys["gs_theta_arcsec"] * W.ARCSEC
    az = math.radians(phys["gs_azimuth_deg"])
    x = kappa * x + h * th * np.array([math.cos(az), math.sin(az)]) / phys["src_pixel_pitch_m"]
    x = x - np.array([phys["dm_shift_x"], phys["dm_shift_y"]])
    t = math.radians(phys["dm_rot_deg"])
    x = np.array([math.cos(t) * x[0] + math.sin(t) * x[1], -math.sin(t) * x[0] + math.cos(t) * x[1]])
    return x / phys["dm_mag"]


def test_composite_matrix_equals_sequential_point_mapping():
    rng = np.random.default_rng(15)
    phys = W.physical(shift_x=0.4, shift_y=-0.7, rot_deg=31.0, mag_x=1.03, mag_y=0.98,
                      dm_shift_x=-1.2, dm_shift_y=0.5, dm_rot_deg=-4.0, dm_mag=1.01,
                      dm_height_m=12000.0, gs_range_m=90000.0, gs_theta_arcsec=50.0,
                      gs_azimuth_deg=77.0, src_pixel_pitch_m=0.08, wfs_pitch_src_px=1.004)
    a = O.compose_affine(phys)
    for _ in range(10):
        pt = rng.uniform(-200, 200, size=2)
        got = np.array([a[0] * pt[0] + a[1] * pt[1] + a[2], a[3] * pt[0] + a[4] * pt[1] + a[5]])
        assert np.allclose(got, _sequential(phys, pt), atol=1e-10)
    assert np.allclose(O.compose_affine(W.physical()), IDENT, atol=0)


def test_cone_factor_and_footprint_shift_of_config_4():
    """BASELINE.json config 4 prints 1-h/H = 0.81 and a footprint shift h*theta (R12)."""
    wl = W.make_config(4, max_modes=4)
    a = O.compose_affine(wl.wfs[1].phys)                     # LGS at azimuth 60 deg
    kappa = 1 - 17.0 / 90.0
    assert abs(kappa - 0.81) < 0.005
    shift = 17000.0 * 45.0 * W.ARCSEC / (38.5 / 476.0)
    assert np.allclose(a, [kappa, 0, shift * math.cos(math.radians(60)), 0, kappa,
                           shift * math.sin(math.radians(60))], atol=1e-9)
    n = O.compose_affine(wl.wfs[6].phys)                     # NGS at azimuth 90 deg, infinite range
    assert np.allclose(n, [1, 0, 0, 0, 1, 17000.0 * 80.0 * W.ARCSEC / (38.5 / 476.0)], atol=1e-9)


# ---------------------------------------------------------------- inputs
def test_workload_shapes_match_baseline_configs():
    c1 = W.make_config(1)
    assert c1.n_modes == 97 and c1.wfs[0].n_valid == 80 and c1.n_rows == 160
    c2 = W.make_config(2, max_modes=8)
    assert c2.wfs[0].n_valid == 1240 and c2.cube.shape == (8, 400, 400)
    assert len(W.actuator_grid(41, 10.0, 205.0)) == 1313
    assert len(W.actuator_grid(81, 6.0, 241.0)) == 5065
    assert len(W.actuator_grid(60, 10.0, 305.0)) == 2912
    c4 = W.make_config(4, max_modes=4)
    assert [w.n_valid for w in c4.wfs] == [3356] * 6 + [4] * 3 and c4.n_rows == 40296
    assert np.array_equal(W.tight_bboxes(c1.cube), c1.bbox)


def test_zernike_modes_are_orthonormal_low_order_and_bounded_high_order():
    n = 128
    pup = W.make_pupil(n, 128.0, 0.0)
    cube = W.zernike_cube(n, n, 64.0, pup, 2, 29).astype(np.float64)
    m = pup > 0
    gram = np.einsum("kp,lp->kl", cube[:, m], cube[:, m]) / m.sum()
    assert np.allclose(np.diag(gram), 1.0, atol=1e-6)
    assert np.abs(gram - np.diag(np.diag(gram))).max() < 0.05   # pixelated disc: nearly orthogonal
    # high radial order stays finite and O(sqrt(n+1)): the recurrence does not blow up
    hi = W.zernike_cube(n, n, 64.0, pup, 1954, 1954)[0]
    assert W.noll_to_nm(1954) == (62, 0) and np.isfinite(hi).all() and np.abs(hi).max() < 40
    # R_62^0(1) = 1: centre-to-edge ratio is fixed by the radial polynomial
    x, _ = centred(n, n)
    # (inside the disc only: rho is clamped to 1 outside it)
    assert W.noll_to_nm(2) == (1, 1)
    assert np.allclose((cube[0] / cube[0, 64, 100] * x[64, 100])[m], x[m], rtol=1e-5, atol=1e-4)


def test_oracle_runs_clean_under_address_and_undefined_behaviour_sanitizers(tmp_path):
    """the oracle's C source built with -fsanitize=address,undefined runs every entry point
    (numerical derivative, G-tilt, edge repair, halo resampling, composition) on odd-sized inputs whose samples leave
    the source grid, in a subprocess; any out-of-bounds access or undefined operation aborts it."""
    import os
    import subprocess
    import sys
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    lib = str(tmp_path / "liboracle_san.so")
    subprocess.check_call(["gcc", "-O1", "-g", "-std=c11", "-fPIC", "-shared", "-fopenmp", "-fsanitize=address,undefined",
                           "-fno-sanitize-recover=undefined", "-o", lib, os.path.join(root, "oracle", "synim_oracle.c"), "-lm"])
    asan = subprocess.check_output(["gcc", "-print-file-name=libasan.so"], text=True).strip()
    code = (
        "import numpy as np\n"
        "from oracle import oracle as O\n"
        "from paper_2606_07759_b200 import workloads as W\n"
        "rng = np.random.default_rng(0)\n"
        "cube = rng.normal(size=(3, 20, 28)).astype(np.float32)\n"
        "pup = W.make_pupil(21, 21.0, 0.2)\n"
        "val = W.valid_subaps(pup, 3, 7)\n"
        "a = [0.7, 0.9, 6.0, -0.9, 0.7, -5.0]\n"
        "for mode in (O.ND, O.GTILT):\n"
        "    assert np.isfinite(O.slopes_wfs(cube, pup, 3, 7, val, a, 1.5, mode, modes=[2, 0], n_threads=2)).all()\n"
        "mask = (rng.uniform(size=(20, 28)) > 0.2).astype(np.float32)\n"
        "assert np.isfinite(O.slopes_wfs_repair(cube, mask, pup, 3, 7, val, a)).all()\n"
        "O.repair_screen(cube[0], mask, 21, a); O.resample(cube[1], 21, a, halo=True)\n"
        "O.compose_affine(W.physical(rot_deg=33.0, dm_height_m=17000.0, gs_range_m=90000.0, gs_theta_arcsec=45.0, src_pixel_pitch_m=0.08))\n"
        "print('clean')\n")
    env = dict(os.environ, SYNIM_ORACLE_LIB=lib, LD_PRELOAD=asan, ASAN_OPTIONS="detect_leaks=0", PYTHONPATH=root)
    out = subprocess.run([sys.executable, "-c", code], env=env, capture_output=True, text=True, cwd=root, timeout=300)
    assert out.returncode == 0 and "clean" in out.stdout, out.stderr[-2000:]
