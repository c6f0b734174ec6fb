"""The CUDA kernels' LOGIC, checked on a CPU: the library's own sources (paper_2606_07759_b200/csrc/*.cu) are compiled
for the host against tests/emu -- an emulation of the CUDA execution model (fibers for threads, rendezvous for warp
collectives and barriers, a bounds-checked shared-memory arena, TMA box loads with the hardware's zero fill, checked
global accesses) -- and driven through the C ABI against the float64 oracle, at the north_star tolerance.

What this does and does not show is spelt out in tests/emu/README.md: indexing, masks, segment logic, memory safety and
float32 numerics yes (where both exist the figures agree with the GPU's to the digit); timing, bank conflicts, races
between warps and real descriptor encodings no.  It is test infrastructure: no product path is built this way, and the
parity claims proper are the `-m gpu` tests.
"""
import os
import subprocess
import sys

import numpy as np
import pytest

from oracle import oracle as O
from paper_2606_07759_b200 import workloads as W

HERE = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, os.path.join(HERE, "emu"))

TOL = 1e-5
EPS32 = 2.0 ** -24


@pytest.fixture(scope="module")
def emu(tmp_path_factory):
    import harness
    out = str(tmp_path_factory.mktemp("emu"))
    lib = harness.build(out)
    e = harness.Emu(lib)
    e.dir = out
    return e


def check(got, ref, wl, tol=TOL):
    """north_star's bar per (mode, sensor) column, with the absolute floor of DESIGN.md reading R17 on columns that are
    (nearly) pure cancellation -- the rule of tests/test_gpu_parity._check_block, restated."""
    amp = np.abs(wl.cube).reshape(wl.n_modes, -1).max(axis=1).astype(np.float64)
    r0, worst = 0, 0.0
    for w in wl.wfs:
        r1 = r0 + 2 * w.n_valid
        if r1 > r0:
            g, r = got[r0:r1], ref[r0:r1]
            cmax = np.abs(r).max(axis=0)
            floor = EPS32 * abs(w.slope_scale) * amp
            fl = np.where(cmax < 100.0 * floor, floor, 0.0)
            err = np.abs(g - r)
            assert (err <= tol * cmax[None, :] + fl[None, :]).all()
            assert (np.linalg.norm(g - r, axis=0) <= tol * np.linalg.norm(r, axis=0) + fl * np.sqrt(r.shape[0])).all()
            live = (cmax >= 100.0 * floor) & (cmax > 0.0)
            if live.any():
                worst = max(worst, float((err.max(axis=0)[live] / cmax[live]).max()))
        r0 = r1
    return worst


def emu_last_nonzero(emu, wl):
    """Where the strip kernel's slope table held a non-zero value (it stores only those on top of the zeros): the
    non-zero entries of the matrix itself."""
    return emu.interaction_matrix(wl).T != 0


def test_strip_kernel_zonal_modes(emu):
    wl = W.make_config(1, max_modes=30)
    ref = O.interaction_matrix(wl)
    check(emu.interaction_matrix(wl, count_stores=True), ref, wl)
    cnt = emu.store_counts                             # the column's zeros once, the non-zero slopes once more on top
    assert cnt.min() == 1 and cnt.max() == 2 and ((cnt == 2) == (emu_last_nonzero(emu, wl))).all()
    check(emu.interaction_matrix(wl, hint=False, octagon=False, ld_pad=3), ref, wl)
    check(emu.interaction_matrix(wl, mode=1), O.interaction_matrix(wl, mode=O.GTILT), wl)
    for cfg, n in ((3, 6), (4, 4)):                    # six rotated LGS sensors; the cone effect and giant NGS subapertures
        wl = W.make_config(cfg, max_modes=n)
        check(emu.interaction_matrix(wl), O.interaction_matrix(wl), wl)
    # supports larger than the staged box and no size hint: one CTA walks nine pieces, re-arming its mbarrier for each
    # (the emulated barrier checks the transaction bytes and the phase parity of every wait)
    cube = W.random_smooth_cube(2, 160, 160, 3)
    pup = W.make_pupil(60, 60.0, 0.0)
    s = [W.WfsInput(10, 6, pup, W.valid_subaps(pup, 10, 6), W.physical(rot_deg=10.0, mag_x=0.4, mag_y=0.4))]
    wl = W.Workload("split supports", 0, 160, 160, cube, W.tight_bboxes(cube), s)
    check(emu.interaction_matrix(wl, hint=False), O.interaction_matrix(wl), wl)
    # a geometry without any valid subaperture: a matrix without rows, a no-op whatever the output pointer is
    import ctypes
    import harness
    blind = W.WfsInput(10, 6, pup, np.zeros((10, 10), np.uint8), W.physical())
    h, keep = emu.geometry([blind], 160, 160)
    assert emu.L.synim_num_rows(h) == 0
    arr = harness.S._affine_array(emu.affines([blind]), [1.0])
    assert emu.L.synim_interaction_matrix(h, emu.reg(cube).ctypes.data, 2, None, None, 0, 0, arr, 0, None, 0, None) == 0
    emu.L.synim_destroy(h)


def test_flat_one_shot_entry_point(emu):
    """synim_interaction_matrix_flat (north_star's argument list: create -> supports -> matrix -> destroy) gives the
    matrix of the piecewise calls bit for bit, compact and dense, both estimators."""
    wl = W.make_config(1, max_modes=5)
    assert np.array_equal(emu.interaction_matrix_flat(wl), emu.interaction_matrix(wl))
    assert np.array_equal(emu.interaction_matrix_flat(wl, compact=False), emu.interaction_matrix(wl, use_bbox=False))
    check(emu.interaction_matrix_flat(wl, mode=1), O.interaction_matrix(wl, mode=O.GTILT), wl)
    wl = W.make_config(4, max_modes=2)        # sensors of two classes: two launches inside the one call
    check(emu.interaction_matrix_flat(wl), O.interaction_matrix(wl), wl)


def test_tile_kernel_dense_modes(emu):
    """Tiles of the WFS grid: narrow last strips (the lanes beyond a strip's halo column once read outside the staged box
    -- the emulator aborts on such an access), partially lit units, skipped units, both estimators, padding rows."""
    wl = W.make_config(1, max_modes=12)
    check(emu.interaction_matrix(wl, use_bbox=False, ld_pad=5), O.interaction_matrix(wl), wl)
    check(emu.interaction_matrix(wl, use_bbox=False, mode=1), O.interaction_matrix(wl, mode=O.GTILT), wl)
    wl = W.make_config(5, max_modes=1)
    assert check(emu.interaction_matrix(wl, count_stores=True), O.interaction_matrix(wl), wl) < 3e-6
    assert (emu.store_counts == 1).all()               # output-stationary: every slope is stored exactly once
    # a sensor demagnified until no tile fits a TMA box (falls back to source-space pieces), and a strongly magnified one
    cube = W.random_smooth_cube(2, 64, 64, 3)
    pup = W.make_pupil(42, 42.0, 0.0)
    for mag in (0.05, 3.0):
        s = [W.WfsInput(6, 7, pup, W.valid_subaps(pup, 6, 7), W.physical(mag_x=mag, mag_y=mag, rot_deg=20.0))]
        wl = W.Workload(f"mag {mag}", 0, 64, 64, cube, None, s)
        check(emu.interaction_matrix(wl), O.interaction_matrix(wl), wl)


def test_tile_kernel_batches_of_modes(emu, monkeypatch):
    """grid.y holds the modes of the tile kernel, at most 65535 of them: larger cubes are cut into batches, each with
    descriptors re-encoded on its part of the cube and its own part of the matrix.  The emulation of a CTA costs
    milliseconds, so the batch size comes down through the library's test knob (tests/test_gpu_parity.py runs the real
    65,700 modes)."""
    monkeypatch.setenv("SYNIM_TILE_BATCH_MODES", "300")
    cube = np.random.default_rng(5).normal(size=(700, 8, 8)).astype(np.float32)
    s = [W.WfsInput(2, 4, np.ones((8, 8), np.float32), np.ones((2, 2), np.uint8), W.physical(rot_deg=7.0, shift_x=0.3))]
    wl = W.Workload("700 small dense modes", 0, 8, 8, cube, None, s)
    check(emu.interaction_matrix(wl, count_stores=True), O.interaction_matrix(wl), wl)
    assert (emu.store_counts == 1).all()


def test_edge_repair_in_both_kernels(emu):
    wl = W.masked(W.make_config(1, max_modes=20), W.make_pupil(80, 80.0, 0.14))
    ref = O.interaction_matrix(wl, repair_mask=wl.mask)
    assert np.abs(ref - O.interaction_matrix(wl)).max() > 1e-3 * np.abs(ref).max()
    check(emu.interaction_matrix(wl, mask=wl.mask), ref, wl)
    check(emu.interaction_matrix(wl, mask=wl.mask, use_bbox=False), ref, wl)
    # rotated, (de)magnified sensors and a soft mask with holes, dense and zonal
    import scipy.ndimage as ndi
    rng = np.random.default_rng(5)
    ny, nx = 72, 88
    cube = W.random_smooth_cube(3, ny, nx, 34)
    blob = ndi.gaussian_filter(rng.normal(size=(ny, nx)), 4.0)
    mask = np.clip(ndi.gaussian_filter((blob > np.quantile(blob, 0.3)).astype(float), 0.8) * 1.3, 0, 1).astype(np.float32)
    pup = W.make_pupil(60, 60.0, 0.2)
    sensors = [W.WfsInput(10, 6, pup, W.valid_subaps(pup, 10, 6), phys, slope_scale=1.7)
               for phys in (W.physical(shift_x=20.0, shift_y=-17.5, rot_deg=33.0), W.physical(mag_x=0.55, mag_y=0.6, rot_deg=-75.0))]
    sensors.append(W.WfsInput(1, 44, np.ones((44, 44), np.float32), np.ones((1, 1), np.uint8), W.physical(rot_deg=5.0, mag_x=1.1, mag_y=1.1)))
    wl = W.masked(W.Workload("soft mask", 0, ny, nx, cube, None, sensors), mask)
    ref = O.interaction_matrix(wl, repair_mask=mask)
    check(emu.interaction_matrix(wl, mask=mask), ref, wl)
    wl.bbox = W.tight_bboxes(wl.cube)
    check(emu.interaction_matrix(wl, mask=mask), ref, wl)


def test_packed_zonal_walk_opt_in(emu, monkeypatch):
    monkeypatch.setenv("SYNIM_ZONAL_PACKED", "1")
    for cfg, n in ((1, 30), (3, 6), (4, 6)):       # (config 4: the LGS launch packed, the giant NGS subapertures as ever)
        wl = W.make_config(cfg, max_modes=n)
        check(emu.interaction_matrix(wl), O.interaction_matrix(wl), wl)


def test_host_pipeline_and_dictionary_in_chunks(emu, monkeypatch):
    """Chunking, buffer alternation, packed supports and per-layer grids of the host entry points (their streams and
    events are synchronous in the emulation: ordering on real hardware is the GPU tests' business)."""
    import ctypes
    from paper_2606_07759_b200 import synim as S
    monkeypatch.setenv("SYNIM_HOST_CHUNK_BYTES", "9000")
    L = emu.L
    wl = W.make_config(1, max_modes=23)
    h, keep = emu.geometry(wl.wfs, wl.ny, wl.nx)
    rows = int(L.synim_num_rows(h))
    arr = S._affine_array(emu.affines(wl.wfs), None)
    ref = O.interaction_matrix(wl)
    for bbox in (wl.bbox, None):
        out = np.full((wl.n_modes, rows), np.nan, np.float32)
        emu.chk(L.synim_interaction_matrix_host(h, wl.cube.ctypes.data, wl.n_modes, None if bbox is None else bbox.ctypes.data,
                                                arr, 0, out.ctypes.data, None))
        check(out.T.astype(np.float64), ref, wl)
    # two layers with their own grids and cone factors, one of them dense
    specs = []
    for li, (n, alt, zonal) in enumerate(((88, 6000.0, True), (96, 12000.0, False))):
        cube, bbox = W.gaussian_cube(n, n, W.actuator_grid(7, 9.0, n / 2.0)[: 11 + li], 9.0)
        ws = [W.WfsInput(s.n_subap, s.n_pix, s.pupil, s.valid, W.physical(rot_deg=3.0, dm_height_m=alt, gs_range_m=90000.0,
                         gs_theta_arcsec=40.0, gs_azimuth_deg=70.0, src_pixel_pitch_m=0.5), slope_scale=1.0 + li) for s in wl.wfs]
        specs.append(W.Workload(f"layer {li}", 0, n, n, cube, bbox if zonal else None, ws))
    lay = (S.Layer * len(specs))()
    outs, arrs = [], []
    for li, w_ in enumerate(specs):
        a = S._affine_array(emu.affines(w_.wfs), [x.slope_scale for x in w_.wfs])
        o = np.full((w_.n_modes, rows), np.nan, np.float32)
        arrs.append(a)
        outs.append(o)
        lay[li].h_influence, lay[li].n_modes, lay[li].ny, lay[li].nx = w_.cube.ctypes.data, w_.n_modes, w_.ny, w_.nx
        lay[li].h_bbox = None if w_.bbox is None else w_.bbox.ctypes.data
        lay[li].affine = ctypes.cast(a, ctypes.POINTER(S.WfsAffine))
        lay[li].h_out = o.ctypes.data
    emu.chk(L.synim_dictionary_host(h, lay, len(specs), 0, None))
    for w_, o in zip(specs, outs):
        check(o.T.astype(np.float64), O.interaction_matrix(w_), w_)
    L.synim_destroy(h)


def test_projection_matrix_call_sequence(emu):
    """synim_projection_matrix with CPU stand-ins for cuBLAS / cuSOLVER (so: the operand kernel, the argument plumbing
    and the call sequence), in a process of its own so that dlopen finds the stand-ins and nothing else."""
    code = r'''
import sys, ctypes, math
sys.path.insert(0, sys.argv[1]); sys.path.insert(0, sys.argv[2])
import numpy as np
import harness
from oracle import oracle as O
from paper_2606_07759_b200 import workloads as W, synim as S
e = harness.Emu(sys.argv[3])
def rot(deg, mag, sx, sy):
    t = math.radians(deg); return [math.cos(t)/mag, math.sin(t)/mag, sx, -math.sin(t)/mag, math.cos(t)/mag, sy]
mp = 20
pupil = e.reg(W.make_pupil(mp, 20.0, 0.2))
c0, _ = W.gaussian_cube(36, 36, W.actuator_grid(5, 5.0, 16.0), 5.0)
c1, _ = W.gaussian_cube(44, 44, W.actuator_grid(4, 8.0, 20.0), 8.0)
cl = W.random_smooth_cube(4, 52, 52, 9)
dirs = [(0.0, 0.0), (3.3, -1.2), (-2.1, 2.7)]
maps = ([rot(1.0, 1.0, 0.0, 0.0) for _ in dirs], [rot(-2.0, 1.02, dx, dy) for dx, dy in dirs])
mapsl = [rot(0.0, 1.0, 2.0 * dx, 2.0 * dy) for dx, dy in dirs]
wts = [1.0, 0.5, 2.0]
p_dm = np.hstack([O.projection_operand(c, m, pupil, wts) for c, m in zip((c0, c1), maps)])
p_l = O.projection_operand(cl, mapsl, pupil, wts)
lam = 0.05 * np.trace(p_dm.T @ p_dm) / p_dm.shape[1]
ref = O.projection_matrix(p_dm, p_l, lam)
comps = (S.Component * 2)(); keep = []
for k, (c, m) in enumerate(zip((c0, c1), maps)):
    c = e.reg(np.ascontiguousarray(c)); a = S._affine_array(m, None); keep.append((c, a))
    comps[k].d_cube = c.ctypes.data; comps[k].n_modes, comps[k].ny, comps[k].nx = c.shape
    comps[k].maps = ctypes.cast(a, ctypes.POINTER(S.WfsAffine))
lay = S.Component(); clr = e.reg(np.ascontiguousarray(cl)); al = S._affine_array(mapsl, None)
lay.d_cube = clr.ctypes.data; lay.n_modes, lay.ny, lay.nx = clr.shape; lay.maps = ctypes.cast(al, ctypes.POINTER(S.WfsAffine))
n_a = ref.shape[0]
out = e.reg(np.full((cl.shape[0], n_a + 3), np.nan, np.float32))
w = (ctypes.c_double * 3)(*wts)
e.chk(e.L.synim_projection_matrix(comps, 2, ctypes.byref(lay), 3, w, pupil.ctypes.data, mp, lam, out.ctypes.data, n_a + 3, None))
assert np.isnan(out[:, n_a:]).all()
err = np.abs(out[:, :n_a].T - ref).max() / np.abs(ref).max()
assert err < 1e-4, err
assert e.L.synim_projection_matrix(comps, 2, ctypes.byref(lay), 3, w, pupil.ctypes.data, mp, -1.0, out.ctypes.data, n_a + 3, None) == -1
print("ok %.2e" % err)
'''
    root = os.path.dirname(HERE)
    env = dict(os.environ, LD_LIBRARY_PATH=emu.dir + os.pathsep + os.environ.get("LD_LIBRARY_PATH", ""))
    res = subprocess.run([sys.executable, "-c", code, root, os.path.join(HERE, "emu"), os.path.join(emu.dir, "libsynim_emu.so")],
                         capture_output=True, text=True, env=env, timeout=600, cwd=root)
    assert res.returncode == 0 and res.stdout.startswith("ok"), res.stderr[-2000:]


def _shard_worker(rank, world, port, lib_path, q):
    """One rank of a two-process gloo job: its sharding.partition_modes range of config 1 through the EMULATED library,
    then sharding.sharded_columns' all_gather of the column blocks."""
    import torch
    import torch.distributed as dist
    sys.path.insert(0, os.path.join(HERE, "emu"))
    import harness
    from paper_2606_07759_b200 import sharding
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        e = harness.Emu(lib_path)
        wl = W.make_config(1, max_modes=21)

        def compute(b, e_):
            import copy
            part = copy.copy(wl)
            part.cube = np.ascontiguousarray(wl.cube[b:e_])
            part.bbox = np.ascontiguousarray(wl.bbox[b:e_])
            if e_ == b:
                return torch.zeros((0, wl.n_rows), dtype=torch.float32)
            return torch.from_numpy(e.interaction_matrix(part).T.astype(np.float32).copy())
        full, (b, e_) = sharding.sharded_columns(wl.n_modes, compute, gather=True)
        q.put((rank, b, e_, full.numpy()))
    finally:
        dist.destroy_process_group()


@pytest.mark.timeout(300)
def test_two_gloo_ranks_shard_the_modes_through_the_kernels(emu):
    """SURVEY sec. 8(e) on CPU with the kernels in the loop (the stand-in `compute` of tests/test_sharding_gloo.py replaced
    by the emulated library): two ranks, contiguous mode ranges, no exchange but the final all_gather; the gathered matrix
    is bit for bit the unsharded one."""
    import socket
    import torch.multiprocessing as mp
    from paper_2606_07759_b200 import sharding
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    world = 2
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    lib = os.path.join(emu.dir, "libsynim_emu.so")
    procs = [ctx.Process(target=_shard_worker, args=(r, world, port, lib, q)) for r in range(world)]
    for p in procs:
        p.start()
    got = [q.get(timeout=240) for _ in range(world)]
    for p in procs:
        p.join(60)
        assert p.exitcode == 0
    wl = W.make_config(1, max_modes=21)
    whole = emu.interaction_matrix(wl).T.astype(np.float32)
    ranges = sharding.partition_modes(wl.n_modes, world)
    for rank, b, e_, full in got:
        assert (b, e_) == ranges[rank]
        assert np.array_equal(full, whole)
    check(whole.T.astype(np.float64), O.interaction_matrix(wl), wl)


def test_seeded_random_cases_against_the_oracle(emu):
    """Fuzzing, committed: the first cases of workloads.random_case (random grids, 1-3 sensors of 1..14 subapertures of
    1..40 pixels with binary or fractional pupils, rotations over +-180 degrees, anamorphic magnifications, compact or
    dense modes, every call option, both estimators, edge repair with binary and soft masks, sensors without a valid
    subaperture, empty modes) through the emulated library, each against the oracle at the north_star bar.
    SYNIM_FUZZ_CASES widens the campaign (default 64; the same seeds run on the GPU in tests/test_gpu_parity.py)."""
    n = int(os.environ.get("SYNIM_FUZZ_CASES", "64"))
    worst, kinds = 0.0, set()
    for seed in range(n):
        wl, o = W.random_case(seed)
        rep = o.pop("repair")
        mask = wl.mask if rep else None
        ref = O.interaction_matrix(wl, mode=O.GTILT if o["mode"] else O.ND, repair_mask=mask)
        try:
            worst = max(worst, check(emu.interaction_matrix(wl, mask=mask, **o), ref, wl))
        except AssertionError as exc:
            raise AssertionError(f"random case {seed} ({o}, repair={rep})") from exc
        kinds.add((wl.bbox is None or not o["use_bbox"], o["mode"], rep))
    print(f"{n} random cases, worst elementwise error {worst:.2e} of the column maximum")
    assert worst <= TOL
    if n >= 64:      # the campaign reaches every path: compact / dense x estimator x repair
        assert {(False, 0, None), (True, 0, None), (False, 1, None), (True, 1, None)} <= kinds
        assert any(k[2] == "binary" for k in kinds) and any(k[2] == "soft" for k in kinds)


@pytest.mark.skipif(not os.environ.get("SYNIM_EMU_FULL"), reason="opt-in (about 25 minutes): SYNIM_EMU_FULL=1")
@pytest.mark.timeout(7200)
def test_full_size_configurations_whole_matrices(emu):
    """The bodies of the full-size GPU tests (tests/test_gpu_parity.py::_full_size) through the emulated library: the WHOLE
    matrices of configs 2, 3 and 4 and the 256 seeded modes of config 5 the GPU test draws, by the GPU tests' own rule
    (assert_parity).  Round 2, last commit: 6.0e-7, 4.9e-6, 6.9e-6 and 1.05e-6 of the column maximum."""
    import test_gpu_parity as T
    for cfg, n_sample, chunk in ((2, None, 256), (3, None, 256), (4, None, 256), (5, 256, 16)):
        wl = W.make_config(cfg)
        sel = np.arange(wl.n_modes)
        if n_sample is not None:
            sel = np.sort(np.random.default_rng(15).choice(wl.n_modes, size=n_sample, replace=False))
        worst = 0.0
        for c0 in range(0, len(sel), chunk):
            idx = sel[c0:c0 + chunk]
            sub = W.Workload(wl.name, wl.cfg, wl.ny, wl.nx, np.ascontiguousarray(wl.cube[idx]),
                             None if wl.bbox is None else np.ascontiguousarray(wl.bbox[idx]), wl.wfs)
            worst = max(worst, T.assert_parity(emu.interaction_matrix(sub).astype(np.float32), O.interaction_matrix(sub), sub)[1])
        print(f"config {cfg}: {len(sel)} modes x {len(wl.wfs)} sensors, worst elementwise error {worst:.2e}")


def test_one_geometry_many_transforms(emu):
    """The on-line regime (what bench.py times): the geometry is built once and the transforms change from
    call to call -- compact and dense modes, both estimators, a map that comes back (the tile plans are memoised per
    sensor and map).  Every call against the oracle."""
    import ctypes
    import dataclasses
    import harness
    L = emu.L
    base = W.make_config(1, max_modes=10)
    h, keep = emu.geometry(base.wfs, base.ny, base.nx)
    rows = int(L.synim_num_rows(h))
    cube = emu.reg(np.ascontiguousarray(base.cube))
    bbox = emu.reg(np.zeros((base.n_modes, 4), np.int32))
    diag = emu.reg(np.zeros((base.n_modes, 4), np.int32))
    emu.chk(L.synim_compute_bboxes(cube.ctypes.data, base.n_modes, base.ny, base.nx, bbox.ctypes.data, diag.ctypes.data, None))
    bw, bh = ctypes.c_int32(), ctypes.c_int32()
    emu.chk(L.synim_bbox_extent(bbox.ctypes.data, base.n_modes, ctypes.byref(bw), ctypes.byref(bh), None))
    out = emu.reg(np.empty((base.n_modes, rows), np.float32))
    maps = [dict(), dict(rot_deg=31.0, mag_x=0.9, mag_y=1.1), dict(shift_x=2.5, shift_y=-1.25), dict(rot_deg=31.0, mag_x=0.9, mag_y=1.1),
            dict(rot_deg=-120.0, mag_x=1.2, mag_y=1.2, shift_x=-0.4)]
    for dense in (False, True):
        for k, phys in enumerate(maps):
            mode = k % 2 if k else 0                       # both estimators along the way
            wfs = [dataclasses.replace(w, phys=W.physical(**phys), slope_scale=1.0 + 0.5 * k) for w in base.wfs]
            wl = W.Workload(f"call {k}", 0, base.ny, base.nx, base.cube, None if dense else base.bbox, wfs)
            arr = harness.S._affine_array(emu.affines(wfs), [w.slope_scale for w in wfs])
            out[:] = np.nan
            emu.chk(L.synim_interaction_matrix(h, cube.ctypes.data, base.n_modes, None if dense else bbox.ctypes.data,
                                               None if dense else diag.ctypes.data, 0 if dense else bw.value, 0 if dense else bh.value,
                                               arr, mode, out.ctypes.data, rows, None))
            assert np.isfinite(out).all()
            check(out.T.astype(np.float64), O.interaction_matrix(wl, mode=O.GTILT if mode else O.ND), wl)
    L.synim_destroy(h)
