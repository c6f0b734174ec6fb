"""Seeded synthetic inputs for the five BASELINE.json configurations.

This module is the ONLY code shared by the CUDA path and the oracle.  It holds
none of the method's arithmetic: no affine composition, no interpolation, no
slopes.  It only manufactures the *inputs* of the synthetic interaction-matrix
computation (section 2.1-2.2):

  * the influence-function cube ``[n_modes][ny][nx]`` float32 (zonal Gaussian
    actuators or Zernike modes) and, for zonal cubes, the tight non-zero
    bounding box of every influence function,
  * per wavefront sensor: the Shack-Hartmann subaperture grid, the pupil
    weights in the WFS frame, the valid-subaperture mask, and the *physical*
    misregistration / guide-star parameters.  Turning those parameters into a
    composite affine matrix is method arithmetic and is done
    separately by each side (``synim_compose_affine`` in the library,
    ``oracle_compose_affine`` in the oracle).

The real MORFEO influence functions, modal bases and YAML files the paper
measures on are not available; these inputs stand in
for them with the same shapes, sizes and structure ("Input
recipe").  Everything is generated in float64 and cast to float32 once.
Seeds are ``7759 + cfg``.
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field
from typing import List, Optional, Sequence

import numpy as np

ARCSEC = math.pi / (180.0 * 3600.0)

#: keys of the physical parameter record of one WFS (all float64); the same
#: field list as ``synim_wfs_physical`` in include/synim.h.
PHYSICAL_FIELDS = (
    "shift_x", "shift_y", "rot_deg", "mag_x", "mag_y",
    "dm_shift_x", "dm_shift_y", "dm_rot_deg", "dm_mag",
    "dm_height_m", "gs_range_m", "gs_theta_arcsec", "gs_azimuth_deg",
    "src_pixel_pitch_m", "wfs_pitch_src_px",
)


def physical(**kw) -> dict:
    """A physical-parameter record with neutral defaults."""
    p = dict(shift_x=0.0, shift_y=0.0, rot_deg=0.0, mag_x=1.0, mag_y=1.0,
             dm_shift_x=0.0, dm_shift_y=0.0, dm_rot_deg=0.0, dm_mag=1.0,
             dm_height_m=0.0, gs_range_m=math.inf, gs_theta_arcsec=0.0,
             gs_azimuth_deg=0.0, src_pixel_pitch_m=1.0, wfs_pitch_src_px=1.0)
    for k, v in kw.items():
        if k not in p:
            raise KeyError(k)
        p[k] = float(v)
    return p


@dataclass
class WfsInput:
    n_subap: int
    n_pix: int
    pupil: np.ndarray        # float32 [M][M], M = n_subap*n_pix, weights in the WFS frame
    valid: np.ndarray        # uint8 [n_subap][n_subap], 1 = valid
    phys: dict               # PHYSICAL_FIELDS -> float
    slope_scale: float = 1.0

    @property
    def m(self) -> int:
        return self.n_subap * self.n_pix

    @property
    def n_valid(self) -> int:
        return int(self.valid.sum())


@dataclass
class Workload:
    name: str
    cfg: int
    ny: int
    nx: int
    cube: np.ndarray                 # float32 [n_modes][ny][nx]
    bbox: Optional[np.ndarray]       # int32 [n_modes][4] (x0,y0,x1,y1 inclusive) or None (dense)
    wfs: List[WfsInput] = field(default_factory=list)
    mode_ids: Optional[np.ndarray] = None   # index of each kept mode in the full config
    mask: Optional[np.ndarray] = None       # float32 [ny][nx]: the modes exist only inside this SOURCE-frame mask
                                            # (the edge-repair case); None: defined everywhere

    @property
    def n_modes(self) -> int:
        return int(self.cube.shape[0])

    @property
    def n_rows(self) -> int:
        return 2 * sum(w.n_valid for w in self.wfs)

    @property
    def n_columns(self) -> int:
        """IM columns in the metric's sense: one per (mode, WFS) pair."""
        return self.n_modes * len(self.wfs)


# --------------------------------------------------------------------------
# pupil, subapertures
# --------------------------------------------------------------------------
def make_pupil(m: int, diameter: float, obstruction: float) -> np.ndarray:
    """Binary annular pupil on an m x m grid, pixel k at k-(m-1)/2."""
    c = (m - 1) / 2.0
    y, x = np.mgrid[0:m, 0:m].astype(np.float64)
    r = np.hypot(x - c, y - c)
    p = (r <= diameter / 2.0) & (r >= obstruction * diameter / 2.0)
    return p.astype(np.float32)


def valid_subaps(pupil: np.ndarray, n_subap: int, n_pix: int, min_frac: float = 0.5) -> np.ndarray:
    """Subaperture (a,b) is valid iff its summed weight >= min_frac*n_pix^2 (ties valid)."""
    s = pupil.astype(np.float64).reshape(n_subap, n_pix, n_subap, n_pix).sum(axis=(1, 3))
    return (s >= min_frac * n_pix * n_pix).astype(np.uint8)


# --------------------------------------------------------------------------
# zonal Gaussian influence functions
# --------------------------------------------------------------------------
def actuator_grid(n_act: int, pitch: float, r_keep: float) -> np.ndarray:
    """Centred positions (x,y) of the n_act x n_act actuators kept (r <= r_keep), row-major."""
    u = (np.arange(n_act) - (n_act - 1) / 2.0) * pitch
    yy, xx = np.meshgrid(u, u, indexing="ij")
    keep = np.hypot(xx, yy) <= r_keep
    return np.stack([xx[keep], yy[keep]], axis=1)


def gaussian_cube(ny: int, nx: int, act_xy: np.ndarray, pitch: float,
                  coupling: float = 0.3, support_pitches: float = 3.0):
    """Gaussian influence functions exp(ln(coupling) r^2/pitch^2), zero for r > support*pitch.

    Returns (cube float32 [n][ny][nx], bbox int32 [n][4] tight non-zero extent)."""
    n = act_xy.shape[0]
    cube = np.zeros((n, ny, nx), dtype=np.float32)
    bbox = np.zeros((n, 4), dtype=np.int32)
    cx, cy = (nx - 1) / 2.0, (ny - 1) / 2.0
    rad = support_pitches * pitch
    lnc = math.log(coupling)
    for k in range(n):
        ax, ay = act_xy[k, 0] + cx, act_xy[k, 1] + cy     # actuator centre in pixel indices
        x0 = max(0, int(math.floor(ax - rad)))
        x1 = min(nx - 1, int(math.ceil(ax + rad)))
        y0 = max(0, int(math.floor(ay - rad)))
        y1 = min(ny - 1, int(math.ceil(ay + rad)))
        if x1 < x0 or y1 < y0:
            bbox[k] = (0, 0, -1, -1)
            continue
        ys, xs = np.mgrid[y0:y1 + 1, x0:x1 + 1].astype(np.float64)
        r2 = (xs - ax) ** 2 + (ys - ay) ** 2
        patch = np.where(r2 <= rad * rad, np.exp(lnc * r2 / (pitch * pitch)), 0.0).astype(np.float32)
        cube[k, y0:y1 + 1, x0:x1 + 1] = patch
        nz_r = np.flatnonzero(patch.any(axis=1))
        nz_c = np.flatnonzero(patch.any(axis=0))
        if nz_r.size == 0:
            bbox[k] = (0, 0, -1, -1)
        else:
            bbox[k] = (x0 + nz_c[0], y0 + nz_r[0], x0 + nz_c[-1], y0 + nz_r[-1])
    return cube, bbox


def tight_bboxes(cube: np.ndarray) -> np.ndarray:
    """Tight non-zero extent of every mode: (x0,y0,x1,y1) inclusive; (0,0,-1,-1) if all zero."""
    n = cube.shape[0]
    out = np.zeros((n, 4), dtype=np.int32)
    for k in range(n):
        nz = cube[k] != 0
        r = np.flatnonzero(nz.any(axis=1))
        c = np.flatnonzero(nz.any(axis=0))
        out[k] = (c[0], r[0], c[-1], r[-1]) if r.size else (0, 0, -1, -1)
    return out


# --------------------------------------------------------------------------
# Zernike modes (Noll ordering), stable to high radial order
# --------------------------------------------------------------------------
def noll_to_nm(j: int):
    """Noll index j>=1 -> (n, m) with m>0 for the cosine and m<0 for the sine term."""
    n = 0
    while (n + 1) * (n + 2) // 2 < j:
        n += 1
    p = j - n * (n + 1) // 2 - 1                 # 0..n inside radial order n
    am = 2 * ((p + 1) // 2) if n % 2 == 0 else 2 * (p // 2) + 1
    if am == 0:
        return n, 0
    return (n, am) if j % 2 == 0 else (n, -am)


def _radial_family(rho: np.ndarray, m: int, n_max: int):
    """Yield (n, R_n^m(rho)) for n = m, m+2, ... <= n_max.

    R_n^m(rho) = rho^m P_k^{(0,m)}(2 rho^2 - 1), k = (n-m)/2, with the Jacobi
    three-term recurrence (the factorial sum loses all digits beyond n ~ 40)."""
    x = 2.0 * rho * rho - 1.0
    rm = rho ** m
    a, b = 0.0, float(m)
    p_prev = np.ones_like(x)
    yield m, rm * p_prev
    if m + 2 > n_max:
        return
    p_cur = 0.5 * ((a - b) + (a + b + 2.0) * x)
    yield m + 2, rm * p_cur
    k = 2
    while m + 2 * k <= n_max:
        c = 2.0 * k + a + b
        a1 = 2.0 * k * (k + a + b) * (c - 2.0)
        a2 = (c - 1.0) * (a * a - b * b)
        a3 = (c - 2.0) * (c - 1.0) * c
        a4 = 2.0 * (k + a - 1.0) * (k + b - 1.0) * c
        p_next = ((a2 + a3 * x) * p_cur - a4 * p_prev) / a1
        p_prev, p_cur = p_cur, p_next
        yield m + 2 * k, rm * p_cur
        k += 1


def zernike_cube(ny: int, nx: int, radius: float, pupil_src: np.ndarray,
                 j_first: int, j_last: int, j_keep: Optional[Sequence[int]] = None) -> np.ndarray:
    """Zernike modes Noll j_first..j_last on the source grid, unit RMS over ``pupil_src`` pixels.

    rho is clamped to 1 outside the unit disc (the polynomials explode beyond it)."""
    js = list(range(j_first, j_last + 1)) if j_keep is None else list(j_keep)
    slot = {j: i for i, j in enumerate(js)}
    cube = np.zeros((len(js), ny, nx), dtype=np.float32)
    cx, cy = (nx - 1) / 2.0, (ny - 1) / 2.0
    yy, xx = np.mgrid[0:ny, 0:nx].astype(np.float64)
    rho = np.minimum(np.hypot(xx - cx, yy - cy) / radius, 1.0)
    theta = np.arctan2(yy - cy, xx - cx)
    pmask = pupil_src > 0
    want = {}
    for j in js:
        n, m = noll_to_nm(j)
        want.setdefault(abs(m), {}).setdefault(n, []).append((j, m))
    n_max = max(noll_to_nm(j)[0] for j in js)
    for am, by_n in sorted(want.items()):
        cosm = np.cos(am * theta) if am else None
        sinm = np.sin(am * theta) if am else None
        for n, rad in _radial_family(rho, am, n_max):
            for (j, m) in by_n.get(n, ()):
                z = rad if m == 0 else (rad * cosm if m > 0 else rad * sinm)
                rms = math.sqrt(float(np.mean(z[pmask] ** 2)))
                cube[slot[j]] = (z / rms).astype(np.float32)
    return cube


# --------------------------------------------------------------------------
# the five configurations (BASELINE.json "configs")
# --------------------------------------------------------------------------
def _subset(n_total: int, max_modes: Optional[int], seed: int) -> np.ndarray:
    if max_modes is None or max_modes >= n_total:
        return np.arange(n_total)
    rng = np.random.default_rng(seed + 1000)
    return np.sort(rng.choice(n_total, size=max_modes, replace=False))


def _cfg3_physical(seed: int):
    """Per-WFS parameters of config 3 (also used by config 5): rot k*60+U(+-0.5) deg,
    shift U(+-0.5) px, magnification 1+U(+-0.01); draw order rot, shift_x, shift_y, mag."""
    rng = np.random.default_rng(seed)
    out = []
    for k in range(6):
        rot = 60.0 * k + rng.uniform(-0.5, 0.5)
        sx = rng.uniform(-0.5, 0.5)
        sy = rng.uniform(-0.5, 0.5)
        mag = 1.0 + rng.uniform(-0.01, 0.01)
        out.append(physical(shift_x=sx, shift_y=sy, rot_deg=rot, mag_x=mag, mag_y=mag))
    return out


def make_config(cfg: int, max_modes: Optional[int] = None) -> Workload:
    """Build configuration ``cfg`` (1..5).  ``max_modes`` keeps a seeded, sorted subset of
    the modes (same WFS set) so that tests can run a structurally identical smaller case."""
    seed = 7759 + cfg
    if cfg == 1:
        n, npix, nsub = 80, 8, 10
        pup = make_pupil(n, 80.0, 0.14)
        acts = actuator_grid(11, 8.0, 40.0 + 4.0)
        keep = _subset(len(acts), max_modes, seed)
        cube, bbox = gaussian_cube(n, n, acts[keep], 8.0)
        w = WfsInput(nsub, npix, pup, valid_subaps(pup, nsub, npix),
                     physical(shift_x=0.3, shift_y=-0.2, rot_deg=1.5, mag_x=1.02, mag_y=1.02))
        return Workload("SCAO tiny", 1, n, n, cube, bbox, [w], keep)
    if cfg == 2:
        n, npix, nsub = 400, 10, 40
        pup = make_pupil(n, 400.0, 0.14)
        acts = actuator_grid(41, 10.0, 200.0 + 5.0)
        keep = _subset(len(acts), max_modes, seed)
        cube, bbox = gaussian_cube(n, n, acts[keep], 10.0)
        rng = np.random.default_rng(seed)
        sx, sy = rng.uniform(-0.5, 0.5), rng.uniform(-0.5, 0.5)
        rot = rng.uniform(-2.0, 2.0)
        mag = 1.0 + rng.uniform(-0.02, 0.02)
        w = WfsInput(nsub, npix, pup, valid_subaps(pup, nsub, npix),
                     physical(shift_x=sx, shift_y=sy, rot_deg=rot, mag_x=mag, mag_y=mag))
        return Workload("VLT-class SCAO", 2, n, n, cube, bbox, [w], keep)
    if cfg in (3, 5):
        n, npix, nsub = 480, 7, 68
        m = nsub * npix                                  # 476
        pup = make_pupil(m, 476.0, 0.28)
        val = valid_subaps(pup, nsub, npix)
        wfs = [WfsInput(nsub, npix, pup, val, p) for p in _cfg3_physical(7759 + 3)]
        if cfg == 3:
            acts = actuator_grid(81, 6.0, 238.0 + 3.0)
            keep = _subset(len(acts), max_modes, seed)
            cube, bbox = gaussian_cube(n, n, acts[keep], 6.0)
            return Workload("ELT MCAO ground DM, 6 LGS", 3, n, n, cube, bbox, wfs, keep)
        keep = _subset(2000, max_modes, seed)
        cube = zernike_cube(n, n, 238.0, make_pupil(n, 476.0, 0.28), 2, 2001,
                            j_keep=[2 + int(k) for k in keep])
        return Workload("Modal ELT IM, 2000 Zernikes, 6 LGS", 5, n, n, cube, None, wfs, keep)
    if cfg == 4:
        n = 600
        pitch_m = 38.5 / 476.0
        pup = make_pupil(476, 476.0, 0.28)
        acts = actuator_grid(60, 10.0, 300.0 + 5.0)
        keep = _subset(len(acts), max_modes, seed)
        cube, bbox = gaussian_cube(n, n, acts[keep], 10.0)
        wfs = []
        val_l = valid_subaps(pup, 68, 7)
        for k in range(6):
            wfs.append(WfsInput(68, 7, pup, val_l, physical(
                dm_height_m=17000.0, gs_range_m=90000.0, gs_theta_arcsec=45.0,
                gs_azimuth_deg=60.0 * k, src_pixel_pitch_m=pitch_m)))
        val_n = valid_subaps(pup, 2, 238)
        for az in (90.0, 210.0, 330.0):
            wfs.append(WfsInput(2, 238, pup, val_n, physical(
                dm_height_m=17000.0, gs_range_m=math.inf, gs_theta_arcsec=80.0,
                gs_azimuth_deg=az, src_pixel_pitch_m=pitch_m)))
        return Workload("ELT MCAO altitude DM, 6 LGS + 3 NGS", 4, n, n, cube, bbox, wfs, keep)
    raise ValueError(f"unknown config {cfg}")


def random_smooth_cube(n_modes: int, ny: int, nx: int, seed: int) -> np.ndarray:
    """Dense test modes: a few random low-order 2-D cosines per mode (no compact support)."""
    rng = np.random.default_rng(seed)
    yy, xx = np.mgrid[0:ny, 0:nx].astype(np.float64)
    cube = np.empty((n_modes, ny, nx), dtype=np.float32)
    for k in range(n_modes):
        z = np.zeros((ny, nx))
        for _ in range(4):
            fx, fy = rng.uniform(-3, 3, size=2) * 2 * math.pi / max(nx, ny)
            z += rng.normal() * np.cos(fx * xx + fy * yy + rng.uniform(0, 2 * math.pi))
        cube[k] = z.astype(np.float32)
    return cube


def masked(wl: Workload, mask: np.ndarray) -> Workload:
    """The edge-repair variant of a workload: the same modes cut by a mask given in the source
    frame (a DM or pupil mask; values in [0, 1]), as a real M4 influence-function file or modal basis would be.
    Supports are recomputed (a masked influence function can only shrink)."""
    mask = np.ascontiguousarray(mask, dtype=np.float32)
    assert mask.shape == (wl.ny, wl.nx)
    cube = np.ascontiguousarray(wl.cube * mask[None], dtype=np.float32)
    bbox = None if wl.bbox is None else tight_bboxes(cube)
    return Workload(wl.name + ", masked", wl.cfg, wl.ny, wl.nx, cube, bbox, wl.wfs, wl.mode_ids, mask)


def make_dictionary(n_layers: int = 12, acts_across: int = 66, max_modes: Optional[int] = None,
                    top_km: float = 22.0, grid_lo: int = 480, grid_hi: int = 692) -> List[Workload]:
    """A multi-layer dictionary of the shape of PAPER.md:132 (MORFEO: 3 DMs + 9 layers = 12 altitude components
    between 0 and 22 km, six LGS WFS of 68x68 subapertures, meta-pupil grids of 480^2 ... 690^2 pixels): one
    Workload per component, all looking through the SAME six sensors (the config-3 sensors, 45 arcsec off axis on a
    hexagonal ring, 90 km range), each with its own grid, cone factor and footprints (the physical records carry
    dm_height_m); every third layer is seen anamorphically and every fourth with a sub-pixel alignment scale s != 1.  Zonal Gaussian influence functions on a centred grid of ``acts_across`` actuators across the
    meta-pupil; ``max_modes`` keeps a seeded subset per layer.  Stand-in for the MORFEO modal bases, which are not
    available here."""
    npix, nsub = 7, 68
    m = nsub * npix
    pup = make_pupil(m, 476.0, 0.28)
    val = valid_subaps(pup, nsub, npix)
    base = _cfg3_physical(7759 + 3)
    pitch_m = 38.5 / 476.0
    out = []
    for li in range(n_layers):
        h_km = top_km * li / max(1, n_layers - 1)
        n = (int(round(grid_lo + (grid_hi - grid_lo) * h_km / top_km)) + 3) & ~3
        d_meta = 476.0 + (n - 480.0)
        pitch = d_meta / acts_across
        acts = actuator_grid(acts_across + 1, pitch, d_meta / 2.0 + pitch / 2.0)
        keep = _subset(len(acts), max_modes, 7759 + 100 + li)
        cube, bbox = gaussian_cube(n, n, acts[keep], pitch)
        wfs = []
        for k, p in enumerate(base):
            q = dict(p)
            q.update(dm_height_m=1000.0 * h_km, gs_range_m=90000.0, gs_theta_arcsec=45.0, gs_azimuth_deg=60.0 * k,
                     src_pixel_pitch_m=pitch_m)
            if li % 3 == 1:          # an anamorphic sensor-to-layer registration ("anamorphic distortions")
                q.update(mag_x=q["mag_x"] * 1.012, mag_y=q["mag_y"] * 0.991)
            if li % 4 == 2:          # a sub-pixel alignment scale s != 1 (reading R11)
                q.update(wfs_pitch_src_px=1.003)
            wfs.append(WfsInput(nsub, npix, pup, val, q))
        out.append(Workload(f"dictionary layer {li} ({h_km:.1f} km, {n}x{n})", 0, n, n, cube, bbox, wfs, keep))
    return out


# --------------------------------------------------------------------------
# seeded random small problems (fuzzing the kernels against the oracle)
# --------------------------------------------------------------------------
def random_case(seed: int):
    """A seeded random SMALL problem and the call options to run it with -> (Workload, options).

    Inputs only, like everything here.  Grids of 32..116 pixels (widths in multiples of 4: the TMA rule of
    include/synim.h), 1-3 sensors of 1..14 subapertures of 1..40 pixels (at most 120 pixels across) with an annular
    binary pupil or random fractional weights, rotations over +-180 degrees, anamorphic magnifications 0.6..1.7,
    shifts of a few pixels, 2-5 modes that are either compact (cut Gaussians of random width and place: the bbox
    path) or smooth and dense.  ``options``: use_bbox / hint / octagon / ld_pad as in tests/test_gpu_parity.gpu_im,
    ``mode`` (0 = numerical derivative, 1 = G-tilt) and ``repair`` (None, "binary" or "soft": the modes are then cut by
    a source-frame mask, Workload.mask, and the repaired entry point applies)."""
    rng = np.random.default_rng([7759, 2, int(seed)])
    ny, nx = 4 * int(rng.integers(8, 30)), 4 * int(rng.integers(8, 30))
    sensors = []
    for _ in range(int(rng.integers(1, 4))):
        n_pix = int(rng.choice([1, 2, 3, 4, 5, 6, 7, 8, 10, 12, 16, 23, 31, 40]))
        n_subap = int(rng.integers(1, max(2, min(14, 120 // n_pix) + 1)))
        m = n_subap * n_pix
        pupil = make_pupil(m, rng.uniform(0.8, 1.1) * m, rng.uniform(0.0, 0.3)) if m > 2 else np.ones((m, m), np.float32)
        if rng.random() < 0.35:      # fractional weights (a soft, unevenly lit pupil)
            pupil = (pupil * rng.uniform(0.05, 1.0, size=pupil.shape)).astype(np.float32)
        valid = valid_subaps(pupil, n_subap, n_pix, min_frac=float(rng.uniform(0.15, 0.6)))
        lit = pupil.astype(np.float64).reshape(n_subap, n_pix, n_subap, n_pix).sum(axis=(1, 3)) > 0
        valid = (valid.astype(bool) & lit).astype(np.uint8)      # (a valid subaperture with no light is an input error)
        s = min(ny, nx) / m * rng.uniform(0.6, 1.25)             # source pixels per sensor pixel
        phys = physical(shift_x=rng.uniform(-3, 3), shift_y=rng.uniform(-3, 3), rot_deg=rng.uniform(-180, 180),
                        mag_x=rng.uniform(0.6, 1.7), mag_y=rng.uniform(0.6, 1.7), wfs_pitch_src_px=s)
        if rng.random() < 0.3:
            phys["mag_y"] = phys["mag_x"]
        sensors.append(WfsInput(n_subap, n_pix, pupil, valid, phys, slope_scale=float(rng.choice([1.0, 1.0, -0.37, 2.5]))))
    n_modes = int(rng.integers(2, 6))
    compact = rng.random() < 0.6
    if compact:
        yy, xx = np.mgrid[0:ny, 0:nx].astype(np.float64)
        cube = np.zeros((n_modes, ny, nx), np.float32)
        for k in range(n_modes):
            cx, cy = rng.uniform(-4, nx + 3), rng.uniform(-4, ny + 3)
            sig, cut = rng.uniform(1.5, 12.0), rng.uniform(1.5, 3.0)
            r2 = (xx - cx) ** 2 + (yy - cy) ** 2
            z = rng.normal() * np.exp(-0.5 * r2 / sig ** 2)
            z[r2 > (cut * sig) ** 2] = 0.0
            if k == n_modes - 1 and rng.random() < 0.25:
                z[:] = 0.0                                           # an empty mode
            cube[k] = z.astype(np.float32)
        bbox = tight_bboxes(cube)
    else:
        cube, bbox = random_smooth_cube(n_modes, ny, nx, 1000 + int(seed)), None
    wl = Workload(f"random case {seed}", 0, ny, nx, cube, bbox, sensors)
    opts = dict(use_bbox=bool(rng.random() < 0.8), hint=bool(rng.random() < 0.7), octagon=bool(rng.random() < 0.7),
                ld_pad=int(rng.choice([0, 0, 3])), mode=int(rng.random() < 0.25), repair=None)
    if opts["mode"] == 0 and rng.random() < 0.35:
        import scipy.ndimage as ndi
        opts["repair"] = "soft" if rng.random() < 0.5 else "binary"
        blob = ndi.gaussian_filter(rng.normal(size=(ny, nx)), 5.0)
        mask = (blob > np.quantile(blob, rng.uniform(0.1, 0.4))).astype(np.float64)
        if opts["repair"] == "soft":
            mask = np.clip(ndi.gaussian_filter(mask, 0.8) * 1.3, 0.0, 1.0)
        wl = masked(wl, mask.astype(np.float32))
    return wl, opts
