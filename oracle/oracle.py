"""ctypes front end of the float64 CPU oracle (oracle/synim_oracle.c).

TEST INFRASTRUCTURE, NOT PRODUCT CODE: only tests/, __graft_entry__.smoke() and
bench.py's cpu_baseline / --impl reference legs may import this module.  It shares
nothing with the CUDA path (paper_2606_07759_b200/csrc) and never imports it.
See the header of synim_oracle.c for the passages of PAPER.md each step follows.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from typing import Optional, Sequence

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "synim_oracle.c")
#: SYNIM_ORACLE_LIB points the front end at another build of the same source (the sanitizer run of the tests)
_LIB = os.environ.get("SYNIM_ORACLE_LIB") or os.path.join(_HERE, "liboracle.so")

ND, GTILT = 0, 1

#: order of the physical parameters in the double[15] record synim_oracle_compose reads
_FIELDS = ("shift_x", "shift_y", "rot_deg", "mag_x", "mag_y",
           "dm_shift_x", "dm_shift_y", "dm_rot_deg", "dm_mag",
           "dm_height_m", "gs_range_m", "gs_theta_arcsec", "gs_azimuth_deg",
           "src_pixel_pitch_m", "wfs_pitch_src_px")


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (plain C, OpenMP over modes)."""
    if os.environ.get("SYNIM_ORACLE_LIB"):
        return _LIB
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        subprocess.check_call(["gcc", "-O2", "-std=c11", "-fPIC", "-shared", "-fopenmp",
                               "-o", _LIB, _SRC, "-lm"])
    return _LIB


_lib = None


def _load():
    global _lib
    if _lib is None:
        lib = ctypes.CDLL(build())
        f64p = ctypes.POINTER(ctypes.c_double)
        lib.synim_oracle_wfs.restype = ctypes.c_int
        lib.synim_oracle_wfs.argtypes = [
            ctypes.c_void_p, ctypes.c_int64, ctypes.c_void_p, ctypes.c_int32, ctypes.c_int32, ctypes.c_int32,
            ctypes.c_void_p, ctypes.c_int32, ctypes.c_int32, ctypes.c_void_p, f64p, ctypes.c_double,
            ctypes.c_int32, ctypes.c_int32, ctypes.c_void_p]
        lib.synim_oracle_wfs_repair.restype = ctypes.c_int
        lib.synim_oracle_wfs_repair.argtypes = [
            ctypes.c_void_p, ctypes.c_int64, ctypes.c_void_p, ctypes.c_int32, ctypes.c_int32, ctypes.c_int32,
            ctypes.c_void_p, ctypes.c_double, ctypes.c_void_p, ctypes.c_int32, ctypes.c_int32, ctypes.c_void_p, f64p,
            ctypes.c_double, ctypes.c_int32, ctypes.c_void_p]
        lib.synim_oracle_repair_screen.restype = ctypes.c_int
        lib.synim_oracle_repair_screen.argtypes = [ctypes.c_void_p, ctypes.c_void_p, ctypes.c_int32, ctypes.c_int32,
                                                   ctypes.c_int32, f64p, ctypes.c_double, ctypes.c_void_p,
                                                   ctypes.c_void_p, ctypes.c_void_p]
        lib.synim_oracle_resample.restype = ctypes.c_int
        lib.synim_oracle_resample.argtypes = [ctypes.c_void_p, ctypes.c_int32, ctypes.c_int32, ctypes.c_int32,
                                              f64p, ctypes.c_int32, ctypes.c_void_p]
        lib.synim_oracle_compose.restype = ctypes.c_int
        lib.synim_oracle_compose.argtypes = [f64p, f64p]
        lib.synim_oracle_num_threads.restype = ctypes.c_int
        _lib = lib
    return _lib


def num_threads() -> int:
    return int(_load().synim_oracle_num_threads())


def compose_affine(phys: dict) -> np.ndarray:
    """Physical parameters -> composite 2x3 matrix a[6] (output -> input, centred pixels)."""
    p = (ctypes.c_double * 15)(*[float(phys[k]) for k in _FIELDS])
    a = (ctypes.c_double * 6)()
    if _load().synim_oracle_compose(p, a) != 0:
        raise ValueError("oracle: bad physical parameters")
    return np.array(list(a), dtype=np.float64)


def resample(g: np.ndarray, m: int, a: Sequence[float], halo: bool = False) -> np.ndarray:
    """The resampled screen of one mode (steps 1-2), float64: [M][M], or with ``halo`` the
    [M+2][M+2] grid of pixels -1..M."""
    g = np.ascontiguousarray(g, dtype=np.float32)
    out = np.empty((m + 2, m + 2) if halo else (m, m), dtype=np.float64)
    aa = (ctypes.c_double * 6)(*[float(v) for v in a])
    rc = _load().synim_oracle_resample(g.ctypes.data, g.shape[0], g.shape[1], m, aa, int(halo),
                                       out.ctypes.data)
    if rc != 0:
        raise RuntimeError(f"oracle resample failed ({rc})")
    return out


REPAIR_THRESHOLD = 0.999999   #: the paper's example value


def repair_screen(g: np.ndarray, mask: np.ndarray, m: int, a: Sequence[float],
                  threshold: float = REPAIR_THRESHOLD):
    """Edge repair of one mode: (phi_repaired float64, core uint8, ring uint8), each on the
    [M+2][M+2] halo grid of pixels -1..M."""
    g = np.ascontiguousarray(g, dtype=np.float32)
    mask = np.ascontiguousarray(mask, dtype=np.float32)
    assert g.shape == mask.shape
    phi = np.empty((m + 2, m + 2), dtype=np.float64)
    core = np.empty((m + 2, m + 2), dtype=np.uint8)
    ring = np.empty((m + 2, m + 2), dtype=np.uint8)
    aa = (ctypes.c_double * 6)(*[float(v) for v in a])
    rc = _load().synim_oracle_repair_screen(g.ctypes.data, mask.ctypes.data, g.shape[0], g.shape[1], m, aa,
                                            float(threshold), phi.ctypes.data, core.ctypes.data, ring.ctypes.data)
    if rc != 0:
        raise RuntimeError(f"oracle repair failed ({rc})")
    return phi, core, ring


def slopes_wfs_repair(cube: np.ndarray, mask: np.ndarray, pupil: np.ndarray, n_subap: int, n_pix: int,
                      valid: np.ndarray, a: Sequence[float], scale: float = 1.0,
                      threshold: float = REPAIR_THRESHOLD, modes: Optional[Sequence[int]] = None,
                      n_threads: int = 0) -> np.ndarray:
    """Edge-repaired numerical-derivative slopes of the selected modes for one WFS:
    float64 [n_sel][2*n_valid] (x then y)."""
    cube = np.ascontiguousarray(cube, dtype=np.float32)
    mask = np.ascontiguousarray(mask, dtype=np.float32)
    pupil = np.ascontiguousarray(pupil, dtype=np.float32)
    valid = np.ascontiguousarray(valid, dtype=np.uint8)
    n_tot, ny, nx = cube.shape
    assert mask.shape == (ny, nx)
    assert pupil.shape == (n_subap * n_pix, n_subap * n_pix) and valid.shape == (n_subap, n_subap)
    if modes is None:
        idx_p, n_sel = None, n_tot
    else:
        idx = np.ascontiguousarray(modes, dtype=np.int32)
        idx_p, n_sel = idx.ctypes.data, idx.size
    nv = int(valid.sum())
    out = np.zeros((n_sel, 2 * nv), dtype=np.float64)
    aa = (ctypes.c_double * 6)(*[float(v) for v in a])
    rc = _load().synim_oracle_wfs_repair(cube.ctypes.data, n_tot, idx_p, n_sel, ny, nx, mask.ctypes.data,
                                         float(threshold), pupil.ctypes.data, n_subap, n_pix, valid.ctypes.data, aa,
                                         float(scale), int(n_threads), out.ctypes.data)
    if rc != 0:
        raise RuntimeError(f"oracle failed ({rc})")
    return out


def slopes_wfs(cube: np.ndarray, pupil: np.ndarray, n_subap: int, n_pix: int, valid: np.ndarray,
               a: Sequence[float], scale: float = 1.0, mode: int = ND,
               modes: Optional[Sequence[int]] = None, n_threads: int = 0) -> np.ndarray:
    """Slopes of the selected modes for one WFS: float64 [n_sel][2*n_valid] (x then y)."""
    cube = np.ascontiguousarray(cube, dtype=np.float32)
    pupil = np.ascontiguousarray(pupil, dtype=np.float32)
    valid = np.ascontiguousarray(valid, dtype=np.uint8)
    n_tot, ny, nx = cube.shape
    assert pupil.shape == (n_subap * n_pix, n_subap * n_pix) and valid.shape == (n_subap, n_subap)
    if modes is None:
        idx_p, n_sel = None, n_tot
    else:
        idx = np.ascontiguousarray(modes, dtype=np.int32)
        idx_p, n_sel = idx.ctypes.data, idx.size
    nv = int(valid.sum())
    out = np.zeros((n_sel, 2 * nv), dtype=np.float64)
    aa = (ctypes.c_double * 6)(*[float(v) for v in a])
    rc = _load().synim_oracle_wfs(cube.ctypes.data, n_tot, idx_p, n_sel, ny, nx, pupil.ctypes.data,
                                  n_subap, n_pix, valid.ctypes.data, aa, float(scale), int(mode),
                                  int(n_threads), out.ctypes.data)
    if rc != 0:
        raise RuntimeError(f"oracle failed ({rc})")
    return out


def interaction_matrix(wl, mode: int = ND, modes: Optional[Sequence[int]] = None,
                       wfs: Optional[Sequence[int]] = None, n_threads: int = 0,
                       affines: Optional[Sequence[Sequence[float]]] = None,
                       repair_mask: Optional[np.ndarray] = None,
                       threshold: float = REPAIR_THRESHOLD) -> np.ndarray:
    """IM of a workload: float64 [rows][n_sel], rows = WFS 0..n-1, each x slopes then y slopes.

    ``wfs`` restricts to some sensors (rows of the others are left out);
    ``affines`` overrides the composite matrices (else composed from ``phys``);
    ``repair_mask`` (float32 [ny][nx], source frame) switches the edge repair of PAPER.md:69-76 on
    (numerical-derivative mode only)."""
    sel = list(range(len(wl.wfs))) if wfs is None else list(wfs)
    blocks = []
    for k in sel:
        w = wl.wfs[k]
        a = compose_affine(w.phys) if affines is None else affines[k]
        if repair_mask is not None:
            assert mode == ND, "edge repair belongs to the numerical-derivative engine"
            blocks.append(slopes_wfs_repair(wl.cube, repair_mask, w.pupil, w.n_subap, w.n_pix, w.valid, a,
                                            w.slope_scale, threshold, modes, n_threads).T)
        else:
            blocks.append(slopes_wfs(wl.cube, w.pupil, w.n_subap, w.n_pix, w.valid, a, w.slope_scale,
                                     mode, modes, n_threads).T)
    return np.concatenate(blocks, axis=0)


# ------------------------------------------------------------------------------------------------------------------
# Tomographic projection matrix (sec. 2.5; readings R24-R26 of DESIGN.md)
# ------------------------------------------------------------------------------------------------------------------
def projection_operand(cube: np.ndarray, maps: Sequence[Sequence[float]], pupil: np.ndarray,
                       weights: Optional[Sequence[float]] = None) -> np.ndarray:
    """P of PAPER.md:90: the influence functions of one component "mapped over the optimized directions".
    Row (d, p) = direction d, pixel p of the mp x mp pupil grid (row-major); column m = mode m; entry
    sqrt(w_d) * pupil[p] * phi_m(A_d x_p), phi_m resampled through the direction's composite map with the same single
    bilinear interpolation as everywhere else (steps 1-2 of the interaction matrix, without the halo).
    float64 [n_dir * mp * mp][n_modes]."""
    cube = np.ascontiguousarray(cube, dtype=np.float32)
    pupil = np.ascontiguousarray(pupil, dtype=np.float64)
    mp = pupil.shape[0]
    assert pupil.shape == (mp, mp)
    n_dir = len(maps)
    w = np.ones(n_dir) if weights is None else np.asarray(weights, dtype=np.float64)
    out = np.empty((n_dir, mp * mp, cube.shape[0]), dtype=np.float64)
    for d in range(n_dir):
        for m in range(cube.shape[0]):
            out[d, :, m] = float(np.sqrt(w[d])) * (pupil * resample(cube[m], mp, maps[d])).ravel()
    return out.reshape(n_dir * mp * mp, cube.shape[0])


def projection_matrix(p_dm: np.ndarray, p_layer: np.ndarray, lam: float) -> np.ndarray:
    """P_opt = (P_DM^T P_DM + lambda I)^-1 P_DM^T P_Layer, written out as the paper gives it:
    float64 [n_dm_modes][n_layer_modes].  P_DM holds the columns of ALL deformable mirrors side by side."""
    g = p_dm.T @ p_dm + float(lam) * np.eye(p_dm.shape[1])
    return np.linalg.solve(g, p_dm.T @ p_layer)
