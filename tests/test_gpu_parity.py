"""Parity of the CUDA path (through the C ABI) against the float64 oracle, on a B200.

Tolerance (BASELINE.json north_star): per (mode, WFS) column relative L2 error <= 1e-5 and
elementwise |err| <= 1e-5 * max|column| in float32.  A (mode, WFS) column the oracle gives as exactly 0
is exactly 0; single entries the oracle gives as exactly 0 are exactly 0 too, except the few on the
one-pixel rim of a support described in DESIGN.md reading R15 (counted and bounded in _check_block).
Every input is seeded and synthetic (paper_2606_07759_b200/workloads.py).
"""
import math

import numpy as np
import pytest

from oracle import oracle as O
from paper_2606_07759_b200 import workloads as W

pytestmark = pytest.mark.gpu

TOL = 1e-5


@pytest.fixture(scope="module")
def S():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("the -m gpu tests need a CUDA device")
    from paper_2606_07759_b200 import build, synim
    build.build_library()
    synim.lib()
    return synim


def gpu_im(S, wl, affines=None, scales=None, use_bbox=True, ld_pad=0, hint=True, octagon=True, mode=0, mask=None,
           threshold=O.REPAIR_THRESHOLD):
    """IM of a workload through the C ABI -> numpy float32 [rows][n_modes].  ``mask`` (source frame) switches the
    edge repair on (synim_interaction_matrix_repaired)."""
    import torch
    geom = S.create_geometry(wl.ny, wl.nx, wl.wfs)
    cube = torch.from_numpy(wl.cube).cuda()
    bbox, diag, bmax = None, None, (0, 0)
    if use_bbox and wl.bbox is not None:
        bbox = torch.from_numpy(wl.bbox).cuda()
        if octagon:
            diag = S.compute_supports(cube)[1]
        if hint:
            bmax = S.bbox_extent(bbox)
    rows = geom.num_rows
    assert rows == wl.n_rows
    out = torch.full((wl.n_modes, rows + ld_pad), float("nan"), dtype=torch.float32, device="cuda")
    if affines is None:
        affines = S.affines_of(wl)
    if scales is None:
        scales = [w.slope_scale for w in wl.wfs]
    if mask is not None:
        S.interaction_matrix(geom, cube, bbox, affines, scales, out=out, bbox_max=bmax, diag=diag, mode=mode,
                             repair_mask=torch.from_numpy(np.ascontiguousarray(mask, dtype=np.float32)).cuda(),
                             threshold=threshold)
    else:
        S.interaction_matrix(geom, cube, bbox, affines, scales, out=out, bbox_max=bmax, diag=diag, mode=mode)
    torch.cuda.synchronize()
    res = out.cpu().numpy()
    if ld_pad:
        assert np.isnan(res[:, rows:]).all()      # padding rows are left untouched
    geom.destroy()
    return res[:, :rows].T.copy()


EPS32 = 2.0 ** -24


def _check_block(g, r, tol, floor, stats):
    """One sensor's block: g, r float64 [2*n_valid][n]; floor [n].  north_star's bar per (mode, WFS) column
    -- rel-L2 <= tol and |err| <= tol * max|column| -- with the absolute floor of DESIGN.md reading R17 added
    ONLY to columns that are (nearly) pure cancellation, max|column| < 100 * floor."""
    err = np.abs(g - r)
    cmax = np.abs(r).max(axis=0)
    nrm = np.linalg.norm(r, axis=0)
    dead = (cmax < 100.0 * floor) | (cmax == 0.0)      # (an all-zero column, e.g. of an empty mode, has no relative error)
    fl = np.where(dead, floor, 0.0)
    assert (err <= tol * cmax[None, :] + fl[None, :]).all(), float((err.max(axis=0) / (cmax + 1e-300))[~dead].max(initial=0.0))
    assert (np.linalg.norm(g - r, axis=0) <= tol * nrm + fl * math.sqrt(r.shape[0])).all()
    live = ~dead
    if live.any():
        stats["l2"] = max(stats["l2"], float((np.linalg.norm(g - r, axis=0)[live] / nrm[live]).max()))
        stats["el"] = max(stats["el"], float((err.max(axis=0)[live] / cmax[live]).max()))
    stats["floored"] += int((dead & (cmax > 0.0)).sum())
    stats["columns"] += int(dead.size)
    assert (g[:, cmax == 0] == 0).all(), "a (mode, WFS) column the oracle gives as exactly 0 is not 0"
    # Skipping is exact (R15): wherever the oracle is exactly 0 the GPU is exactly 0, except on the
    # one-pixel rim of the support where a float32 coordinate can land on the other side of an
    # integer and pick up a weight of a few ulp; those entries are few and far below tolerance.
    stray = (r == 0) & (g != 0)
    assert stray.sum() <= 0.05 * max(1, (r != 0).sum()), (int(stray.sum()), int((r != 0).sum()))
    assert (err[stray] <= (1e-6 * cmax[None, :] + fl[None, :]).repeat(r.shape[0], 0)[stray]).all()
    stats["stray"] += int(stray.sum())


def assert_parity(got, ref, wl, tol=TOL):
    """got float32 [rows][n], ref float64 [rows][n]; checked per (mode, WFS) column.

    north_star's bar (rel-L2 <= 1e-5, |err| <= 1e-5 max|column|).  Columns that are pure cancellation (an
    actuator strictly inside one fully lit giant subaperture has an exactly zero net slope; the oracle
    returns ~1e-17 of float64 noise there) get the absolute floor of DESIGN.md reading R17, one float32
    rounding of the mode's amplitude eps32*|scale|*max|IF_m|; the number of such columns is printed.
    Entries the oracle gives as exactly 0 are exactly 0 on the GPU except for the few rim entries of
    reading R15 (counted, bounded by 1e-6 max|column|)."""
    assert got.shape == ref.shape
    assert np.isfinite(got).all()
    amp = np.abs(wl.cube).reshape(wl.n_modes, -1).max(axis=1).astype(np.float64)
    r0 = 0
    stats = {"l2": 0.0, "el": 0.0, "floored": 0, "columns": 0, "stray": 0}
    for w in wl.wfs:
        r1 = r0 + 2 * w.n_valid
        if r1 > r0:      # (a sensor without a valid subaperture has no rows)
            _check_block(got[r0:r1].astype(np.float64), ref[r0:r1], tol, EPS32 * abs(w.slope_scale) * amp, stats)
        r0 = r1
    print(f"parity {wl.name}: worst rel-L2 {stats['l2']:.2e}, worst elementwise {stats['el']:.2e}, "
          f"{stats['floored']} of {stats['columns']} columns on the R17 floor, {stats['stray']} rim entries")
    return stats["l2"], stats["el"]


def assert_parity_whole(S, wl, out, modes=None, omode=0, tol=TOL):
    """The WHOLE matrix (or the given modes of it) against the oracle, one sensor at a time so that the
    float64 reference never exceeds a few hundred MB.  out: CUDA float32 [n_modes][ld]."""
    import torch
    sel = np.arange(wl.n_modes) if modes is None else np.asarray(modes)
    amp = np.abs(wl.cube[sel]).reshape(len(sel), -1).max(axis=1).astype(np.float64)
    idx = torch.from_numpy(sel).cuda()
    stats = {"l2": 0.0, "el": 0.0, "floored": 0, "columns": 0, "stray": 0}
    r0 = 0
    for w in wl.wfs:
        r1 = r0 + 2 * w.n_valid
        ref = O.slopes_wfs(wl.cube, w.pupil, w.n_subap, w.n_pix, w.valid, O.compose_affine(w.phys),
                           w.slope_scale, omode, None if modes is None else sel).T
        got = out[idx, r0:r1].cpu().numpy().T.astype(np.float64)
        _check_block(got, ref, tol, EPS32 * abs(w.slope_scale) * amp, stats)
        r0 = r1
    print(f"parity {wl.name}: {len(sel)} of {wl.n_modes} modes x {len(wl.wfs)} sensors, worst rel-L2 {stats['l2']:.2e}, "
          f"worst elementwise {stats['el']:.2e}, {stats['floored']} of {stats['columns']} columns on the R17 floor, "
          f"{stats['stray']} rim entries")
    return stats


def test_config1_scao_tiny_full(S):
    wl = W.make_config(1)
    assert_parity(gpu_im(S, wl), O.interaction_matrix(wl), wl)


def test_config1_with_padding_rows_scale_and_no_hint(S):
    wl = W.make_config(1)
    wl.wfs[0].slope_scale = 2.5
    ref = O.interaction_matrix(wl)
    assert_parity(gpu_im(S, wl, ld_pad=24), ref, wl)
    assert_parity(gpu_im(S, wl, ld_pad=3), ref, wl)          # columns no longer 16-byte aligned
    assert_parity(gpu_im(S, wl, hint=False), ref, wl)


def test_config2_vlt_subset(S):
    wl = W.make_config(2, max_modes=96)
    assert_parity(gpu_im(S, wl), O.interaction_matrix(wl), wl)


def test_config3_elt_ground_six_rotated_lgs(S):
    wl = W.make_config(3, max_modes=64)
    assert_parity(gpu_im(S, wl), O.interaction_matrix(wl), wl)


def test_config4_altitude_dm_cone_footprint_and_giant_ngs_subaps(S):
    wl = W.make_config(4, max_modes=48)
    assert [w.n_pix for w in wl.wfs] == [7] * 6 + [238] * 3
    assert_parity(gpu_im(S, wl), O.interaction_matrix(wl), wl)


def test_config5_dense_zernike_modes(S):
    wl = W.make_config(5, max_modes=10)
    assert wl.bbox is None
    assert_parity(gpu_im(S, wl), O.interaction_matrix(wl), wl)


def _full_size(S, cfg, n_sample=None, seed=0):
    """The whole config in bench.py's launch configuration (device-computed supports, size hint), and the
    WHOLE matrix against the oracle (n_sample: a seeded draw of that many modes instead, for the dense
    config whose oracle pass is the slowest)."""
    import torch
    wl = W.make_config(cfg)
    geom = S.create_geometry(wl.ny, wl.nx, wl.wfs)
    cube = torch.from_numpy(wl.cube).cuda()
    bbox = diag = None
    bmax = (0, 0)
    if wl.bbox is not None:
        bbox, diag = S.compute_supports(cube)
        assert np.array_equal(bbox.cpu().numpy(), wl.bbox)
        bmax = S.bbox_extent(bbox)
    out = torch.full((wl.n_modes, geom.num_rows), float("nan"), dtype=torch.float32, device="cuda")
    S.interaction_matrix(geom, cube, bbox, S.affines_of(wl), [w.slope_scale for w in wl.wfs], out=out, bbox_max=bmax,
                         diag=diag)
    torch.cuda.synchronize()
    assert bool(torch.isfinite(out).all())          # every element of every column was written
    sel = None
    if n_sample is not None and n_sample < wl.n_modes:
        sel = np.sort(np.random.default_rng(seed).choice(wl.n_modes, size=n_sample, replace=False))
    assert_parity_whole(S, wl, out, sel)
    if wl.bbox is not None:
        # compact support: a column has at most (footprint / subaperture + 2)^2 non-zero slopes per sensor
        nnz = (out != 0).sum(dim=1).cpu().numpy()
        bound = 0
        for w in wl.wfs:
            aff = np.asarray(S.compose_affine(w.phys))[:6].reshape(2, 3)[:, :2]
            ext = (max(bmax) + 2) * np.abs(np.linalg.inv(aff)).sum(axis=1).max() + 2
            bound += 2 * (int(ext // w.n_pix) + 2) ** 2
        assert nnz.max() <= bound, (int(nnz.max()), bound)
        assert nnz.min() >= 0 and (nnz > 0).mean() > 0.9     # nearly every actuator is seen by some sensor
    geom.destroy()


def test_config3_full_size_whole_matrix_in_the_bench_configuration(S):
    _full_size(S, 3)


def test_config2_and_config4_full_size_whole_matrices(S):
    _full_size(S, 2)
    _full_size(S, 4)


def test_config5_full_size_dense(S):
    _full_size(S, 5, n_sample=256, seed=15)


def test_more_than_sixteen_sensors_take_a_second_launch(S):
    """17 sensors (MORFEO has 12; a launch batches 16): the second launch has its own row range
    and its own zeros.  Compact and dense modes, both estimators."""
    rng = np.random.default_rng(41)
    wl = W.make_config(1, max_modes=40)
    base = wl.wfs[0]
    sensors = []
    for k in range(17):
        phys = W.physical(shift_x=rng.uniform(-1, 1), shift_y=rng.uniform(-1, 1), rot_deg=rng.uniform(-180, 180),
                          mag_x=rng.uniform(0.95, 1.05), mag_y=rng.uniform(0.95, 1.05))
        sensors.append(W.WfsInput(base.n_subap, base.n_pix, base.pupil, base.valid, phys, slope_scale=1.0 + 0.1 * k))
    wl.wfs = sensors
    ref = O.interaction_matrix(wl)
    assert_parity(gpu_im(S, wl), ref, wl)
    assert_parity(gpu_im(S, wl, use_bbox=False), ref, wl)
    assert_parity(gpu_im(S, wl, mode=S.SLOPES_GTILT, ld_pad=5), O.interaction_matrix(wl, mode=O.GTILT), wl)


def test_more_than_65535_dense_modes_take_a_second_batch(S):
    """The tile kernel keeps the modes in grid.y (<= 65535): a larger cube goes in batches, each with descriptors
    re-encoded on its part of the cube and its own part of the matrix (synim_api.cu, run_interaction_matrix)."""
    n = 65700
    cube = np.random.default_rng(5).normal(size=(n, 8, 8)).astype(np.float32)
    s = [W.WfsInput(2, 4, np.ones((8, 8), np.float32), np.ones((2, 2), np.uint8), W.physical(rot_deg=7.0, shift_x=0.3))]
    wl = W.Workload(f"{n} small dense modes", 0, 8, 8, cube, None, s)
    assert_parity(gpu_im(S, wl), O.interaction_matrix(wl), wl)


def test_dense_modes_with_padding_rows(S):
    """Dense modes into a matrix with ld > rows (padding rows must stay untouched), aligned and not."""
    wl = W.make_config(5, max_modes=4)
    ref = O.interaction_matrix(wl)
    assert_parity(gpu_im(S, wl, ld_pad=8), ref, wl)
    assert_parity(gpu_im(S, wl, ld_pad=3), ref, wl)
    wl = W.make_config(1, max_modes=12)
    assert_parity(gpu_im(S, wl, use_bbox=False, ld_pad=7), O.interaction_matrix(wl), wl)


def test_gtilt_estimator_on_the_gpu(S):
    """SYNIM_SLOPES_GTILT (reading R13) against the oracle's G-tilt mode: small subapertures under
    rotation, partially lit ones, the 238-pixel NGS subapertures, the split-support and dense paths; and it
    is a different estimator from the numerical derivative (they differ by a few per cent on a Gaussian)."""
    wl = W.make_config(1)
    ref = O.interaction_matrix(wl, mode=O.GTILT)
    got = gpu_im(S, wl, mode=S.SLOPES_GTILT)
    assert_parity(got, ref, wl)
    nd = O.interaction_matrix(wl, mode=O.ND)
    assert np.abs(ref - nd).max() > 1e-3 * np.abs(nd).max()
    assert_parity(gpu_im(S, wl, mode=S.SLOPES_GTILT, hint=False, use_bbox=False), ref, wl)     # dense path
    wl = W.make_config(3, max_modes=48)
    assert_parity(gpu_im(S, wl, mode=S.SLOPES_GTILT), O.interaction_matrix(wl, mode=O.GTILT), wl)
    wl = W.make_config(4, max_modes=32)
    assert_parity(gpu_im(S, wl, mode=S.SLOPES_GTILT, hint=False), O.interaction_matrix(wl, mode=O.GTILT), wl)


def test_dense_path_on_zonal_cube_equals_bbox_path(S):
    """bbox = NULL must give the same matrix as the tile-skipping path (skipping is exact, R15)."""
    wl = W.make_config(1, max_modes=24)
    ref = O.interaction_matrix(wl)
    assert_parity(gpu_im(S, wl, use_bbox=False), ref, wl)


def test_identity_transform_is_exact_on_integer_data(S):
    """Identity map: phi == input bit for bit, so slopes of an integer-valued screen with P = 1
    are exactly representable sums: the GPU must match the oracle to the last bit."""
    rng = np.random.default_rng(31)
    n_subap, n_pix = 6, 8
    m = n_subap * n_pix
    cube = rng.integers(-8, 9, size=(5, m, m)).astype(np.float32)
    w = W.WfsInput(n_subap, n_pix, np.ones((m, m), np.float32), np.ones((n_subap, n_subap), np.uint8), W.physical())
    wl = W.Workload("identity", 0, m, m, cube, None, [w])
    got = gpu_im(S, wl)
    ref = O.interaction_matrix(wl)
    assert np.array_equal(got.astype(np.float64), ref)


def test_tilt_and_quadratic_closed_forms_on_the_gpu(S):
    """The oracle's closed-form pins, applied directly to the CUDA path."""
    n = 96
    yy, xx = np.mgrid[0:n, 0:n].astype(np.float64)
    xs, ys = xx - (n - 1) / 2.0, yy - (n - 1) / 2.0
    ta, tb = 0.375, -0.5
    cube = np.stack([ta * xs + tb * ys, xs ** 2 / 64.0]).astype(np.float32)
    rng = np.random.default_rng(32)
    n_subap, n_pix = 6, 5
    pupil = rng.uniform(0.1, 1.0, (30, 30)).astype(np.float32)
    w = W.WfsInput(n_subap, n_pix, pupil, np.ones((6, 6), np.uint8), W.physical(), slope_scale=1.5)
    wl = W.Workload("closed forms", 0, n, n, cube, None, [w])
    t = math.radians(27.0)
    a = [math.cos(t) / 1.07, math.sin(t) / 1.07, 0.31, -math.sin(t) / 1.07, math.cos(t) / 1.07, -0.44]
    got = gpu_im(S, wl, affines=[a])
    assert np.allclose(got[:36, 0], 1.5 * (ta * a[0] + tb * a[3]), rtol=0, atol=1e-5)
    assert np.allclose(got[36:, 0], 1.5 * (ta * a[1] + tb * a[4]), rtol=0, atol=1e-5)
    got = gpu_im(S, wl, affines=[[1, 0, 0.25, 0, 1, -1.5]])
    p = pupil.astype(np.float64).reshape(6, 5, 6, 5)
    xw = (np.arange(30) - 14.5).reshape(1, 1, 6, 5)
    xbar = (p * xw).sum(axis=(1, 3)) / p.sum(axis=(1, 3))
    assert np.allclose(got[:36, 1], 1.5 * 2 * (xbar.ravel() + 0.25) / 64.0, rtol=0, atol=1e-5)
    assert np.allclose(got[36:, 1], 0.0, atol=1e-5)


def test_empty_and_degenerate_inputs(S):
    import torch
    wl = W.make_config(1, max_modes=6)
    wl.cube[2] = 0.0                               # an identically-zero mode
    wl.bbox[2] = (0, 0, -1, -1)
    wl.bbox[4] = (0, 0, wl.nx - 1, wl.ny - 1)      # a loose, full-grid bbox is still correct
    ref = O.interaction_matrix(wl)
    got = gpu_im(S, wl, hint=False)
    assert (got[:, 2] == 0).all()
    assert_parity(got, ref, wl)
    # n_modes = 0 is a no-op
    geom = S.create_geometry(wl.ny, wl.nx, wl.wfs)
    empty = torch.empty((0, wl.ny, wl.nx), dtype=torch.float32, device="cuda")
    out = S.interaction_matrix(geom, empty, None, S.affines_of(wl))
    assert out.shape == (0, geom.num_rows)
    # singular affine and a too-small ld are argument errors
    cube = torch.from_numpy(wl.cube).cuda()
    with pytest.raises(S.SynimError) as e:
        S.interaction_matrix(geom, cube, None, [[1, 2, 0, 2, 4, 0]])
    assert e.value.status == S.ERR_INVALID_ARG
    with pytest.raises(S.SynimError) as e:
        S.interaction_matrix(geom, cube, None, S.affines_of(wl), mode=7)
    assert e.value.status == S.ERR_INVALID_ARG
    small = torch.empty((wl.n_modes, geom.num_rows - 1), dtype=torch.float32, device="cuda")
    assert S.lib().synim_interaction_matrix(geom._h, cube.data_ptr(), wl.n_modes, None, None, 0, 0,
                                            S._affine_array(S.affines_of(wl), None), 0, small.data_ptr(),
                                            geom.num_rows - 1, None) == S.ERR_INVALID_ARG
    geom.destroy()
    # sensors without any valid subaperture: a matrix without rows, a no-op whatever the output pointer is
    blind = W.WfsInput(2, 4, np.ones((8, 8), np.float32), np.zeros((2, 2), np.uint8), W.physical())
    geom = S.create_geometry(wl.ny, wl.nx, [blind])
    assert geom.num_rows == 0
    out = S.interaction_matrix(geom, cube, None, [S.compose_affine(blind.phys)])
    assert out.shape == (wl.n_modes, 0)
    geom.destroy()
    # a valid subaperture without light is refused at geometry creation
    dark = W.WfsInput(2, 4, np.zeros((8, 8), np.float32), np.ones((2, 2), np.uint8), W.physical())
    with pytest.raises(S.SynimError) as e:
        S.create_geometry(8, 8, [dark])
    assert e.value.status == S.ERR_EMPTY_SUBAP


def test_wfs_looking_past_the_source_grid_and_strong_magnification(S):
    """Footprints that overrun the grid (R4), a demagnified and an anamorphic sensor, partial pupil."""
    rng = np.random.default_rng(33)
    ny, nx = 72, 88
    cube = W.random_smooth_cube(6, ny, nx, 34)
    pup = W.make_pupil(60, 60.0, 0.2)
    sensors = []
    for phys in (W.physical(shift_x=20.0, shift_y=-17.5, rot_deg=33.0),
                 W.physical(mag_x=0.55, mag_y=0.6, rot_deg=-75.0),
                 W.physical(mag_x=1.7, mag_y=1.5, shift_x=3.3, rot_deg=140.0)):
        sensors.append(W.WfsInput(10, 6, pup, W.valid_subaps(pup, 10, 6), phys))
    wl = W.Workload("overrun", 0, ny, nx, cube, None, sensors)
    ref = O.interaction_matrix(wl)
    assert_parity(gpu_im(S, wl), ref, wl)
    wl.bbox = W.tight_bboxes(cube)
    assert_parity(gpu_im(S, wl), ref, wl)
    assert_parity(gpu_im(S, wl, hint=False), ref, wl)


def test_full_physical_chain_and_degenerate_sensor_grids(S):
    """Every parameter of the composite matrix at once (DM shift / rotation / magnification, cone effect,
    off-axis footprint, sub-pixel alignment scale s != 1), sensors with one pixel per subaperture and with
    a single subaperture, both estimators, zonal and dense."""
    ny, nx = 64, 64
    cube = W.random_smooth_cube(5, ny, nx, 77)
    sensors = []
    for n_subap, n_pix, phys in (
            (8, 6, W.physical(shift_x=0.4, shift_y=-0.7, rot_deg=12.0, mag_x=1.03, mag_y=0.98, dm_shift_x=-1.3,
                              dm_shift_y=0.6, dm_rot_deg=-4.0, dm_mag=1.05, dm_height_m=9000.0, gs_range_m=90000.0,
                              gs_theta_arcsec=20.0, gs_azimuth_deg=40.0, src_pixel_pitch_m=0.35, wfs_pitch_src_px=1.1)),
            (40, 1, W.physical(rot_deg=-20.0, shift_x=1.5)),          # one pixel per subaperture
            (1, 44, W.physical(rot_deg=5.0, mag_x=1.1, mag_y=1.1))):  # a single subaperture
        m = n_subap * n_pix
        pup = W.make_pupil(m, float(m), 0.0) if n_subap > 1 else np.ones((m, m), np.float32)
        sensors.append(W.WfsInput(n_subap, n_pix, pup, W.valid_subaps(pup, n_subap, n_pix), phys))
    wl = W.Workload("chain", 0, ny, nx, cube, None, sensors)
    for mode, omode in ((S.SLOPES_ND, O.ND), (S.SLOPES_GTILT, O.GTILT)):
        ref = O.interaction_matrix(wl, mode=omode)
        wl.bbox = None
        assert_parity(gpu_im(S, wl, mode=mode), ref, wl)
        wl.bbox = W.tight_bboxes(cube)
        assert_parity(gpu_im(S, wl, mode=mode), ref, wl)


def test_debug_build_traps_on_nothing(S, tmp_path):
    """The -DSYNIM_CHECKS build traps on any shared-memory, weight-map or slope-table access outside its
    bounds; every launch configuration runs through it cleanly (compute-sanitizer is closed on this pool)."""
    from paper_2606_07759_b200 import build
    lib = build.build_library(extra=("-DSYNIM_CHECKS",), out=str(tmp_path / "libsynim_checks.so"))
    saved = (S.LIB_PATH, S._lib)
    S.LIB_PATH, S._lib = lib, None
    try:
        for cfg, n, kw in ((1, None, {}), (1, None, dict(hint=False)), (1, None, dict(use_bbox=False)),
                           (1, None, dict(mode=S.SLOPES_GTILT)), (3, 24, {}), (4, 16, {}), (4, 8, dict(hint=False)),
                           (5, 1, {})):
            wl = W.make_config(cfg, max_modes=n)
            got = gpu_im(S, wl, **kw)
            assert np.isfinite(got).all()
        wl = W.masked(W.make_config(1), W.make_pupil(80, 80.0, 0.14))          # edge repair, strips and tiles
        for kw in ({}, dict(use_bbox=False)):
            assert np.isfinite(gpu_im(S, wl, mask=wl.mask, **kw)).all()
    finally:
        S.LIB_PATH, S._lib = saved


def test_compute_bboxes_matches_the_generator(S):
    import torch
    wl = W.make_config(2, max_modes=40)
    wl.cube[7] = 0
    got = S.compute_bboxes(torch.from_numpy(wl.cube).cuda())
    exp = W.tight_bboxes(wl.cube)
    assert np.array_equal(got.cpu().numpy(), exp)
    assert S.bbox_extent(got) == (int((exp[:, 2] - exp[:, 0] + 1).max()), int((exp[:, 3] - exp[:, 1] + 1).max()))
    # diagonal extents: min/max of x+y and x-y over the non-zero pixels, written out with numpy
    bb, dg = S.compute_supports(torch.from_numpy(wl.cube).cuda())
    assert np.array_equal(bb.cpu().numpy(), exp)
    dg = dg.cpu().numpy()
    for m in range(wl.n_modes):
        yy, xx = np.nonzero(wl.cube[m])
        want = (0, -1, 0, -1) if len(xx) == 0 else ((xx + yy).min(), (xx + yy).max(), (xx - yy).min(), (xx - yy).max())
        assert tuple(int(v) for v in dg[m]) == tuple(int(v) for v in want), m


def test_octagon_footprints_change_nothing_but_the_work(S):
    """The diagonal extents only narrow what is sampled: same IM with and without them, on rotated
    sensors (config 3) and on the split-support path (no size hint, config 4's 60-pixel supports)."""
    wl = W.make_config(3, max_modes=96)
    a = gpu_im(S, wl, octagon=True)
    b = gpu_im(S, wl, octagon=False)
    ref = O.interaction_matrix(wl)
    assert_parity(a, ref, wl)
    assert_parity(b, ref, wl)
    scale = np.abs(ref).max()
    assert np.abs(a.astype(np.float64) - b.astype(np.float64)).max() <= 1e-6 * scale
    wl = W.make_config(4, max_modes=24)
    assert_parity(gpu_im(S, wl, octagon=True, hint=False), O.interaction_matrix(wl), wl)


def test_host_buffer_entry_point(S):
    import torch
    wl = W.make_config(1)
    geom = S.create_geometry(wl.ny, wl.nx, wl.wfs)
    out = S.interaction_matrix_host(geom, torch.from_numpy(wl.cube).pin_memory(), wl.bbox, S.affines_of(wl))
    assert_parity(out.numpy().T.copy(), O.interaction_matrix(wl), wl)
    geom.destroy()


def test_host_entry_point_packs_supports_edges_empty_modes_and_dense(S):
    """With bboxes only the supports cross the bus (packed, per-mode origins): supports touching the grid
    edge (origin -4), an all-zero mode, pageable memory, a repeated call on the same geometry; without
    bboxes the whole cube goes (dense path)."""
    import torch
    wl = W.make_config(4, max_modes=40)           # 600-px grid, 60-px supports, some cut by the grid edge
    rng = np.random.default_rng(5)
    wl.cube[5] = 0
    wl.bbox[5] = (0, 0, -1, -1)
    wl.cube[6] = 0                                  # a support in the upper-left corner: packed origin (-4, -1)
    wl.cube[6, 0:20, 0:17] = rng.uniform(0.1, 1.0, (20, 17)).astype(np.float32)
    wl.bbox[6] = (0, 0, 16, 19)
    wl.cube[7] = 0                                  # ... and one against the far edges
    wl.cube[7, wl.ny - 31:, wl.nx - 25:] = rng.uniform(0.1, 1.0, (31, 25)).astype(np.float32)
    wl.bbox[7] = (wl.nx - 25, wl.ny - 31, wl.nx - 1, wl.ny - 1)
    ref = O.interaction_matrix(wl)
    geom = S.create_geometry(wl.ny, wl.nx, wl.wfs)
    for _ in range(2):
        out = S.interaction_matrix_host(geom, wl.cube, wl.bbox, S.affines_of(wl))      # numpy, pageable
        assert_parity(out.numpy().T.copy(), ref, wl)
    bad = wl.bbox.copy()
    bad[0, 2] = wl.nx
    with pytest.raises(S.SynimError) as e:
        S.interaction_matrix_host(geom, wl.cube, bad, S.affines_of(wl))
    assert e.value.status == S.ERR_INVALID_ARG
    geom.destroy()
    wl = W.make_config(5, max_modes=3)
    geom = S.create_geometry(wl.ny, wl.nx, wl.wfs)
    out = S.interaction_matrix_host(geom, torch.from_numpy(wl.cube).pin_memory(), None, S.affines_of(wl))
    assert_parity(out.numpy().T.copy(), O.interaction_matrix(wl), wl)
    geom.destroy()


def test_host_entry_point_in_chunks(S, monkeypatch):
    """The host entry point's pipeline with chunks of a few modes (SYNIM_HOST_CHUNK_BYTES): buffers alternate, the
    copies of one chunk overlap the kernel of the next, and the matrix is the same as in one piece."""
    import torch
    wl = W.make_config(1)
    ref = O.interaction_matrix(wl)
    geom = S.create_geometry(wl.ny, wl.nx, wl.wfs)
    for chunk in ("8000", "100000", None):
        if chunk is None:
            monkeypatch.delenv("SYNIM_HOST_CHUNK_BYTES", raising=False)
        else:
            monkeypatch.setenv("SYNIM_HOST_CHUNK_BYTES", chunk)
        out = S.interaction_matrix_host(geom, torch.from_numpy(wl.cube).pin_memory(), wl.bbox, S.affines_of(wl))
        assert_parity(out.numpy().T.copy(), ref, wl)
        out = S.interaction_matrix_host(geom, wl.cube, None, S.affines_of(wl), mode=S.SLOPES_GTILT)     # dense, pageable
        assert_parity(out.numpy().T.copy(), O.interaction_matrix(wl, mode=O.GTILT), wl)
    geom.destroy()


def test_dictionary_host_streams_layers_with_their_own_grids(S, monkeypatch):
    """synim_dictionary_host: components at different altitudes, each with its own meta-pupil
    grid, cone factor and footprints, through one set of sensors; a dense and an empty layer among them; every
    layer's matrix against the oracle."""
    layers = W.make_dictionary(n_layers=4, acts_across=40, max_modes=20)
    dense = W.make_config(5, max_modes=2)
    dense.wfs = layers[0].wfs                      # same sensors, the ground layer's transforms
    layers.insert(2, dense)
    geom = S.create_geometry(layers[0].ny, layers[0].nx, layers[0].wfs)
    spec = [dict(cube=l.cube, bbox=l.bbox, affines=S.affines_of(l), scales=[1.0 + 0.1 * k] * len(l.wfs)) for k, l in enumerate(layers)]
    spec.insert(1, dict(cube=np.zeros((0, 480, 480), np.float32), bbox=np.zeros((0, 4), np.int32), affines=S.affines_of(layers[0])))
    monkeypatch.setenv("SYNIM_HOST_CHUNK_BYTES", str(6 * 40272 * 4))       # six modes per chunk
    outs = S.dictionary_host(geom, spec)
    outs.pop(1)
    for k, (l, o) in enumerate(zip(layers, outs)):
        for w in l.wfs:
            w.slope_scale = 1.0 + 0.1 * k
        assert_parity(o.numpy().T.copy(), O.interaction_matrix(l), l)
    assert len({l.ny for l in layers}) >= 3 and layers[-1].wfs[0].phys["dm_height_m"] == 22000.0
    geom.destroy()


def test_one_geometry_many_transforms(S):
    """The on-line regime (what bench.py times): the geometry is built once and the transforms change from
    call to call -- compact and dense modes, both estimators, a map that comes back (the tile plans are memoised per
    sensor and map).  Every call against the oracle."""
    import dataclasses
    import torch
    base = W.make_config(1, max_modes=10)
    geom = S.create_geometry(base.ny, base.nx, base.wfs)
    cube = torch.from_numpy(base.cube).cuda()
    bbox, diag = S.compute_supports(cube)
    bmax = S.bbox_extent(bbox)
    out = torch.empty((base.n_modes, geom.num_rows), dtype=torch.float32, device="cuda")
    maps = [dict(), dict(rot_deg=31.0, mag_x=0.9, mag_y=1.1), dict(shift_x=2.5, shift_y=-1.25), dict(rot_deg=31.0, mag_x=0.9, mag_y=1.1),
            dict(rot_deg=-120.0, mag_x=1.2, mag_y=1.2, shift_x=-0.4)]
    for dense in (False, True):
        for k, phys in enumerate(maps):
            mode = k % 2 if k else 0
            wfs = [dataclasses.replace(w, phys=W.physical(**phys), slope_scale=1.0 + 0.5 * k) for w in base.wfs]
            wl = W.Workload(f"call {k}", 0, base.ny, base.nx, base.cube, None if dense else base.bbox, wfs)
            out.fill_(float("nan"))
            S.interaction_matrix(geom, cube, None if dense else bbox, S.affines_of(wl), [w.slope_scale for w in wfs], out=out,
                                 bbox_max=(0, 0) if dense else bmax, diag=None if dense else diag, mode=mode)
            torch.cuda.synchronize()
            assert_parity(out.cpu().numpy().T, O.interaction_matrix(wl, mode=O.GTILT if mode else O.ND), wl)
    geom.destroy()


def test_flat_one_shot_entry_point(S):
    """synim_interaction_matrix_flat (north_star's argument list: create -> supports -> matrix -> destroy in one call)
    gives the matrix of the piecewise calls bit for bit, and meets the bar on its own."""
    import torch
    for cfg, n in ((1, None), (4, 12)):
        wl = W.make_config(cfg, max_modes=n)
        cube = torch.from_numpy(wl.cube).cuda()
        aff, sc = S.affines_of(wl), [w.slope_scale for w in wl.wfs]
        flat = S.interaction_matrix_flat(cube, wl.wfs, aff, sc).cpu().numpy().T
        assert np.array_equal(flat, gpu_im(S, wl))
        assert_parity(flat, O.interaction_matrix(wl), wl)
        dense = S.interaction_matrix_flat(cube, wl.wfs, aff, sc, compact=False).cpu().numpy().T
        assert np.array_equal(dense, gpu_im(S, wl, use_bbox=False))


def test_mode_ranges_through_the_library_concatenate_to_the_unsharded_matrix(S):
    """the mode axis shards with no exchange.  The ranges of sharding.partition_modes go through
    synim_interaction_matrix one by one (as the ranks of a job would, each on its slice of the cube and its block of
    the column-major matrix); the concatenation equals the unsharded matrix bit for bit, zonal and dense."""
    import torch
    from paper_2606_07759_b200 import sharding
    for cfg, n, dense in ((3, 61, False), (1, 23, True)):
        wl = W.make_config(cfg, max_modes=n)
        geom = S.create_geometry(wl.ny, wl.nx, wl.wfs)
        cube = torch.from_numpy(wl.cube).cuda()
        bbox = diag = None
        bmax = (0, 0)
        if not dense:
            bbox, diag = S.compute_supports(cube)
            bmax = S.bbox_extent(bbox)
        aff = S.affines_of(wl)
        whole = S.interaction_matrix(geom, cube, bbox, aff, bbox_max=bmax, diag=diag).clone()
        for world in (2, 3, 5):
            out = torch.full_like(whole, float("nan"))
            for b, e in sharding.partition_modes(wl.n_modes, world):
                if e > b:
                    S.interaction_matrix(geom, cube[b:e], None if bbox is None else bbox[b:e], aff, out=out[b:e],
                                         bbox_max=bmax, diag=None if diag is None else diag[b:e])
            torch.cuda.synchronize()
            assert torch.equal(out, whole)
        geom.destroy()
    assert_parity(whole.cpu().numpy().T.copy(), O.interaction_matrix(wl), wl)


def test_edge_repair_on_masked_modes(S):
    """synim_interaction_matrix_repaired against the oracle's edge repair, on modes cut by a
    source-frame mask: every BASELINE geometry (small subapertures under rotation, the cone effect with giant NGS
    subapertures, dense Zernikes through the tile kernel), zonal and dense, with and without size hint / octagon."""
    def check(wl, **kw):
        ref = O.interaction_matrix(wl, repair_mask=wl.mask, threshold=kw.get("threshold", O.REPAIR_THRESHOLD))
        raw = O.interaction_matrix(wl)
        assert np.abs(ref - raw).max() > 1e-3 * np.abs(ref).max()      # the repair changes the matrix
        assert_parity(gpu_im(S, wl, mask=wl.mask, **kw), ref, wl)
    wl = W.masked(W.make_config(1), W.make_pupil(80, 80.0, 0.14))
    check(wl)
    check(wl, hint=False, octagon=False, ld_pad=3)
    check(wl, use_bbox=False)                                          # dense: tiles of the WFS grid
    check(W.masked(W.make_config(3, max_modes=48), W.make_pupil(480, 476.0, 0.28)))
    check(W.masked(W.make_config(4, max_modes=24), W.make_pupil(600, 560.0, 0.1)))
    check(W.masked(W.make_config(5, max_modes=2), W.make_pupil(480, 476.0, 0.28)))


def test_edge_repair_soft_mask_thresholds_and_odd_sensors(S):
    """A mask with soft (fractional) edges, holes and thin parts, sensors that look past the grid, strongly
    (de)magnified ones, a single giant subaperture, one pixel per subaperture; the paper's threshold and 0.5."""
    import scipy.ndimage as ndi
    rng = np.random.default_rng(5)
    ny, nx = 72, 88
    cube = W.random_smooth_cube(4, ny, nx, 34)
    blob = ndi.gaussian_filter(rng.normal(size=(ny, nx)), 4.0)
    mask = np.clip(ndi.gaussian_filter((blob > np.quantile(blob, 0.3)).astype(float), 0.8) * 1.3, 0, 1).astype(np.float32)
    pup = W.make_pupil(60, 60.0, 0.2)
    sensors = []
    for phys in (W.physical(shift_x=20.0, shift_y=-17.5, rot_deg=33.0), W.physical(mag_x=0.55, mag_y=0.6, rot_deg=-75.0),
                 W.physical(mag_x=1.7, mag_y=1.5, shift_x=3.3, rot_deg=140.0)):
        sensors.append(W.WfsInput(10, 6, pup, W.valid_subaps(pup, 10, 6), phys, slope_scale=1.7))
    sensors.append(W.WfsInput(1, 44, np.ones((44, 44), np.float32), np.ones((1, 1), np.uint8),
                              W.physical(rot_deg=5.0, mag_x=1.1, mag_y=1.1)))
    p1 = W.make_pupil(40, 40.0, 0.0)
    sensors.append(W.WfsInput(40, 1, p1, W.valid_subaps(p1, 40, 1), W.physical(rot_deg=-20.0, shift_x=1.5)))
    wl = W.masked(W.Workload("soft mask", 0, ny, nx, cube, None, sensors), mask)
    for thr in (O.REPAIR_THRESHOLD, 0.5):
        ref = O.interaction_matrix(wl, repair_mask=mask, threshold=thr)
        wl.bbox = None
        assert_parity(gpu_im(S, wl, mask=mask, threshold=thr), ref, wl)
        wl.bbox = W.tight_bboxes(wl.cube)
        assert_parity(gpu_im(S, wl, mask=mask, threshold=thr), ref, wl)


def test_edge_repair_argument_errors(S):
    import torch
    wl = W.masked(W.make_config(1, max_modes=4), W.make_pupil(80, 80.0, 0.14))
    geom = S.create_geometry(wl.ny, wl.nx, wl.wfs)
    cube = torch.from_numpy(wl.cube).cuda()
    mask = torch.from_numpy(wl.mask).cuda()
    for thr in (0.0, 1.5, float("nan")):
        with pytest.raises(S.SynimError) as e:
            S.interaction_matrix(geom, cube, None, S.affines_of(wl), repair_mask=mask, threshold=thr)
        assert e.value.status == S.ERR_INVALID_ARG
    with pytest.raises(ValueError):
        S.interaction_matrix(geom, cube, None, S.affines_of(wl), repair_mask=mask, mode=S.SLOPES_GTILT)
    geom.destroy()


def test_seeded_random_cases_on_the_gpu(S):
    """The committed fuzz campaign (workloads.random_case, the seeds tests/test_kernel_logic_emulated.py runs through the
    host emulation) through the real library: random grids, sensors, pupils, maps, compact and dense modes, every call
    option, both estimators, edge repair -- each case against the oracle at the north_star bar."""
    worst = 0.0
    for seed in range(64):
        wl, o = W.random_case(seed)
        rep = o.pop("repair")
        mask = wl.mask if rep else None
        ref = O.interaction_matrix(wl, mode=O.GTILT if o["mode"] else O.ND, repair_mask=mask)
        try:
            worst = max(worst, assert_parity(gpu_im(S, wl, mask=mask, **o), ref, wl)[1])
        except AssertionError as exc:
            raise AssertionError(f"random case {seed} ({o}, repair={rep})") from exc
    print(f"64 random cases: worst elementwise error {worst:.2e} of the column maximum")


def test_packed_zonal_walk_is_opt_in_and_agrees_with_the_oracle(S, monkeypatch):
    """SYNIM_ZONAL_PACKED=1 (not the default until it has been timed): zonal footprints rounded out to whole units, their
    edge-sum units sampled on the boundary rows and columns only.  Same matrix within the bar."""
    monkeypatch.setenv("SYNIM_ZONAL_PACKED", "1")
    for cfg, n in ((1, None), (3, 48), (2, 60), (4, 24)):
        wl = W.make_config(cfg, max_modes=n)
        assert_parity(gpu_im(S, wl), O.interaction_matrix(wl), wl)
    wl = W.make_config(1)
    assert_parity(gpu_im(S, wl, hint=False, octagon=False, ld_pad=5), O.interaction_matrix(wl), wl)
