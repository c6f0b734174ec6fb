"""Thin ctypes binding of the C-ABI library (include/synim.h), same names without the prefix.

Argument marshalling only: every step of the path runs in the CUDA kernels of ``libsynim.so``.
PyTorch supplies device memory and streams.  There is no CPU fallback: if the library has not been
built (``python -m paper_2606_07759_b200.build``) importing this module's functions raises.
"""
from __future__ import annotations

import ctypes
import os
from typing import Optional, Sequence

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libsynim.so")

OK, ERR_INVALID_ARG, ERR_ALIGNMENT, ERR_EMPTY_SUBAP = 0, -1, -2, -3
ERR_UNSUPPORTED_DEVICE, ERR_OUT_OF_MEMORY, ERR_CUDA, ERR_UNSUPPORTED = -4, -5, -6, -7
SLOPES_ND, SLOPES_GTILT = 0, 1

#: every symbol include/synim.h declares
EXPORTS = ("synim_compose_affine", "synim_create_geometry", "synim_num_rows", "synim_num_valid",
           "synim_row_offset", "synim_interaction_matrix", "synim_interaction_matrix_repaired",
           "synim_interaction_matrix_flat", "synim_compute_bboxes",
           "synim_bbox_extent",
           "synim_interaction_matrix_host", "synim_dictionary_host", "synim_projection_matrix", "synim_destroy", "synim_last_error", "synim_version",
           "synim_launch_count")

PHYSICAL_FIELDS = ("shift_x", "shift_y", "rot_deg", "mag_x", "mag_y",
                   "dm_shift_x", "dm_shift_y", "dm_rot_deg", "dm_mag",
                   "dm_height_m", "gs_range_m", "gs_theta_arcsec", "gs_azimuth_deg",
                   "src_pixel_pitch_m", "wfs_pitch_src_px")


class WfsGrid(ctypes.Structure):
    _fields_ = [("n_subap", ctypes.c_int32), ("n_pix", ctypes.c_int32),
                ("valid_mask", ctypes.c_void_p), ("d_pupil", ctypes.c_void_p)]


class WfsAffine(ctypes.Structure):
    _fields_ = [("a", ctypes.c_double * 6), ("slope_scale", ctypes.c_double)]


class WfsPhysical(ctypes.Structure):
    _fields_ = [(k, ctypes.c_double) for k in PHYSICAL_FIELDS]


class Layer(ctypes.Structure):
    _fields_ = [("h_influence", ctypes.c_void_p), ("n_modes", ctypes.c_int32), ("ny", ctypes.c_int32),
                ("nx", ctypes.c_int32), ("h_bbox", ctypes.c_void_p), ("affine", ctypes.POINTER(WfsAffine)),
                ("h_out", ctypes.c_void_p)]


class Component(ctypes.Structure):
    _fields_ = [("d_cube", ctypes.c_void_p), ("n_modes", ctypes.c_int32), ("ny", ctypes.c_int32),
                ("nx", ctypes.c_int32), ("maps", ctypes.POINTER(WfsAffine))]


class SynimError(RuntimeError):
    def __init__(self, status: int, text: str):
        super().__init__(f"synim status {status}: {text}")
        self.status = status


_lib = None


def lib() -> ctypes.CDLL:
    """The loaded library; raises if it was never built (no fallback of any kind)."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise RuntimeError(f"{LIB_PATH} is missing: build it with `python -m paper_2606_07759_b200.build`; "
                               "there is no CPU fallback")
        L = ctypes.CDLL(LIB_PATH)
        vp, i32, i64 = ctypes.c_void_p, ctypes.c_int32, ctypes.c_int64
        L.synim_compose_affine.restype = ctypes.c_int
        L.synim_compose_affine.argtypes = [ctypes.POINTER(WfsPhysical), ctypes.POINTER(WfsAffine)]
        L.synim_create_geometry.restype = ctypes.c_int
        L.synim_create_geometry.argtypes = [i32, i32, i32, ctypes.POINTER(WfsGrid), vp, ctypes.POINTER(vp)]
        for name in ("synim_num_rows",):
            getattr(L, name).restype = i64
            getattr(L, name).argtypes = [vp]
        for name in ("synim_num_valid", "synim_row_offset"):
            getattr(L, name).restype = i64
            getattr(L, name).argtypes = [vp, i32]
        L.synim_interaction_matrix.restype = ctypes.c_int
        L.synim_interaction_matrix.argtypes = [vp, vp, i32, vp, vp, i32, i32, ctypes.POINTER(WfsAffine), ctypes.c_int,
                                               vp, i64, vp]
        L.synim_interaction_matrix_repaired.restype = ctypes.c_int
        L.synim_interaction_matrix_repaired.argtypes = [vp, vp, i32, vp, vp, i32, i32, ctypes.POINTER(WfsAffine), vp,
                                                        ctypes.c_double, vp, i64, vp]
        L.synim_interaction_matrix_flat.restype = ctypes.c_int
        L.synim_interaction_matrix_flat.argtypes = [vp, i32, i32, i32, i32, ctypes.POINTER(WfsGrid), ctypes.POINTER(WfsAffine),
                                                    i32, ctypes.c_int, vp, i64, ctypes.POINTER(i64), vp]
        L.synim_compute_bboxes.restype = ctypes.c_int
        L.synim_compute_bboxes.argtypes = [vp, i32, i32, i32, vp, vp, vp]
        L.synim_bbox_extent.restype = ctypes.c_int
        L.synim_bbox_extent.argtypes = [vp, i32, ctypes.POINTER(i32), ctypes.POINTER(i32), vp]
        L.synim_interaction_matrix_host.restype = ctypes.c_int
        L.synim_interaction_matrix_host.argtypes = [vp, vp, i32, vp, ctypes.POINTER(WfsAffine), ctypes.c_int, vp, vp]
        L.synim_dictionary_host.restype = ctypes.c_int
        L.synim_dictionary_host.argtypes = [vp, ctypes.POINTER(Layer), i32, ctypes.c_int, vp]
        L.synim_projection_matrix.restype = ctypes.c_int
        L.synim_projection_matrix.argtypes = [ctypes.POINTER(Component), i32, ctypes.POINTER(Component), i32,
                                              ctypes.POINTER(ctypes.c_double), vp, i32, ctypes.c_double, vp, i64, vp]
        L.synim_destroy.restype = None
        L.synim_destroy.argtypes = [vp]
        L.synim_last_error.restype = ctypes.c_char_p
        L.synim_last_error.argtypes = []
        L.synim_version.restype = i32
        L.synim_version.argtypes = []
        L.synim_launch_count.restype = i64
        L.synim_launch_count.argtypes = []
        _lib = L
    return _lib


def _check(status: int) -> None:
    if status != OK:
        raise SynimError(status, lib().synim_last_error().decode("utf-8", "replace"))


def version() -> int:
    return int(lib().synim_version())


def launch_count() -> int:
    """Kernels launched by the library in this process so far (synim_launch_count)."""
    return int(lib().synim_launch_count())


def hot_kernel_name(dense: bool, gtilt: bool = False, repair: bool = False) -> str:
    """Name of the kernel that dominates a step (for reports; the launch lists under profiles/ show it)."""
    g, r = ("true" if gtilt else "false"), ("true" if repair else "false")
    if dense:
        return f"synim_tile_kernel<{g}, {r}> (dense modes: tiles of the WFS grid)"
    return f"synim_strip_kernel<{g}, true, {r}>"


def last_error() -> str:
    return lib().synim_last_error().decode("utf-8", "replace")


def compose_affine(phys: dict) -> np.ndarray:
    """Physical parameters (PHYSICAL_FIELDS) -> composite matrix a[6] (pure host call)."""
    p = WfsPhysical(*[float(phys[k]) for k in PHYSICAL_FIELDS])
    out = WfsAffine()
    _check(lib().synim_compose_affine(ctypes.byref(p), ctypes.byref(out)))
    return np.array(list(out.a), dtype=np.float64)


def _affine_array(affines: Sequence[Sequence[float]], scales: Optional[Sequence[float]]):
    n = len(affines)
    arr = (WfsAffine * n)()
    for k in range(n):
        for q in range(6):
            arr[k].a[q] = float(affines[k][q])
        arr[k].slope_scale = 1.0 if scales is None else float(scales[k])
    return arr


def _stream_ptr(stream) -> int:
    import torch
    if stream is None:
        stream = torch.cuda.current_stream()
    return int(stream.cuda_stream)


class Geometry:
    """Owner of a ``synim_geometry*`` (synim_create_geometry / synim_destroy)."""

    def __init__(self, ny: int, nx: int, wfs: Sequence, stream=None):
        """``wfs``: objects with n_subap, n_pix, valid (uint8 [n_subap][n_subap], host) and pupil
        (float32 [M][M]; a CUDA tensor, or a numpy array that is copied to the device here)."""
        import torch
        n = len(wfs)
        grids = (WfsGrid * n)()
        keep = []
        on_device = {}   # sensors that pass the SAME pupil object get the same device buffer (the library then shares their maps)
        for k, w in enumerate(wfs):
            valid = np.ascontiguousarray(w.valid, dtype=np.uint8)
            pupil = on_device.get(id(w.pupil))
            if pupil is None:
                pupil = w.pupil
                if not isinstance(pupil, torch.Tensor):
                    pupil = torch.from_numpy(np.ascontiguousarray(pupil, dtype=np.float32))
                pupil = pupil.to(device="cuda", dtype=torch.float32).contiguous()
                on_device[id(w.pupil)] = pupil
            m = int(w.n_subap) * int(w.n_pix)
            if tuple(pupil.shape) != (m, m) or valid.shape != (w.n_subap, w.n_subap):
                raise ValueError(f"sensor {k}: pupil must be [{m}][{m}] and valid [{w.n_subap}][{w.n_subap}]")
            keep.append((valid, pupil))
            grids[k].n_subap, grids[k].n_pix = int(w.n_subap), int(w.n_pix)
            grids[k].valid_mask = valid.ctypes.data
            grids[k].d_pupil = pupil.data_ptr()
        handle = ctypes.c_void_p()
        _check(lib().synim_create_geometry(int(ny), int(nx), n, grids, _stream_ptr(stream), ctypes.byref(handle)))
        self._h = handle
        self.ny, self.nx, self.n_wfs = int(ny), int(nx), n
        del keep   # synim_create_geometry synchronised the stream; the inputs are no longer read

    @property
    def num_rows(self) -> int:
        return int(lib().synim_num_rows(self._h))

    def num_valid(self, w: int) -> int:
        return int(lib().synim_num_valid(self._h, int(w)))

    def row_offset(self, w: int) -> int:
        return int(lib().synim_row_offset(self._h, int(w)))

    def destroy(self) -> None:
        if getattr(self, "_h", None):
            lib().synim_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass


def create_geometry(ny: int, nx: int, wfs: Sequence, stream=None) -> Geometry:
    return Geometry(ny, nx, wfs, stream)


def destroy(geom: Geometry) -> None:
    geom.destroy()


def num_rows(geom: Geometry) -> int:
    return geom.num_rows


def compute_bboxes(cube, stream=None):
    """Tight non-zero extents of a CUDA float32 cube [n][ny][nx] -> CUDA int32 [n][4]."""
    return compute_supports(cube, stream, diagonals=False)[0]


def compute_supports(cube, stream=None, diagonals=True):
    """(bbox, diag): tight non-zero extents [n][4] and, if asked for, the diagonal extents
    (min x+y, max x+y, min x-y, max x-y) [n][4] of every mode of a CUDA float32 cube [n][ny][nx]."""
    import torch
    assert cube.is_cuda and cube.dtype == torch.float32 and cube.is_contiguous() and cube.dim() == 3
    n, ny, nx = cube.shape
    out = torch.empty((n, 4), dtype=torch.int32, device=cube.device)
    diag = torch.empty((n, 4), dtype=torch.int32, device=cube.device) if diagonals else None
    _check(lib().synim_compute_bboxes(cube.data_ptr(), n, ny, nx, out.data_ptr(),
                                      None if diag is None else diag.data_ptr(), _stream_ptr(stream)))
    return out, diag


def bbox_extent(bbox, stream=None):
    """(max width, max height) of CUDA int32 bboxes [n][4]; synchronises the stream."""
    w, h = ctypes.c_int32(), ctypes.c_int32()
    _check(lib().synim_bbox_extent(bbox.data_ptr(), int(bbox.shape[0]), ctypes.byref(w), ctypes.byref(h),
                                   _stream_ptr(stream)))
    return int(w.value), int(h.value)


REPAIR_THRESHOLD = 0.999999   #: the paper's example value for the strict binarisation


def interaction_matrix(geom: Geometry, cube, bbox, affines: Sequence[Sequence[float]],
                       scales: Optional[Sequence[float]] = None, out=None, bbox_max=(0, 0),
                       mode: int = SLOPES_ND, stream=None, diag=None, repair_mask=None,
                       threshold: float = REPAIR_THRESHOLD):
    """synim_interaction_matrix on CUDA tensors.  Returns ``out`` viewed as [n_modes][ld] (row k of the
    view is IM column k: the buffer is the column-major IM).  With ``repair_mask`` (CUDA float32 [ny][nx], the
    modes' mask in the source frame) the call is synim_interaction_matrix_repaired (edge repair)."""
    import torch
    assert cube.is_cuda and cube.dtype == torch.float32 and cube.is_contiguous() and cube.dim() == 3
    n = int(cube.shape[0])
    if tuple(cube.shape[1:]) != (geom.ny, geom.nx):
        raise ValueError("cube shape does not match the geometry's source grid")
    if len(affines) != geom.n_wfs:
        raise ValueError("one affine per sensor")
    rows = geom.num_rows
    if out is None:
        out = torch.empty((n, rows), dtype=torch.float32, device=cube.device)
    assert out.is_cuda and out.dtype == torch.float32 and out.dim() == 2 and out.stride(1) == 1
    assert out.shape[0] >= n
    ld = int(out.stride(0)) if out.shape[0] > 1 else int(out.shape[1])
    bptr = None
    if bbox is not None:
        assert bbox.is_cuda and bbox.dtype == torch.int32 and bbox.is_contiguous() and tuple(bbox.shape) == (n, 4)
        bptr = bbox.data_ptr()
    dptr = None
    if diag is not None:
        assert diag.is_cuda and diag.dtype == torch.int32 and diag.is_contiguous() and tuple(diag.shape) == (n, 4)
        dptr = diag.data_ptr()
    arr = _affine_array(affines, scales)
    if repair_mask is not None:
        assert repair_mask.is_cuda and repair_mask.dtype == torch.float32 and repair_mask.is_contiguous()
        assert tuple(repair_mask.shape) == (geom.ny, geom.nx)
        if mode != SLOPES_ND:
            raise ValueError("edge repair belongs to the numerical-derivative engine")
        _check(lib().synim_interaction_matrix_repaired(geom._h, cube.data_ptr(), n, bptr, dptr, int(bbox_max[0]),
                                                       int(bbox_max[1]), arr, repair_mask.data_ptr(), float(threshold),
                                                       out.data_ptr(), ld, _stream_ptr(stream)))
        return out
    _check(lib().synim_interaction_matrix(geom._h, cube.data_ptr(), n, bptr, dptr, int(bbox_max[0]), int(bbox_max[1]),
                                          arr, int(mode), out.data_ptr(), ld, _stream_ptr(stream)))
    return out


def interaction_matrix_flat(cube, wfs: Sequence, affines: Sequence[Sequence[float]], scales: Optional[Sequence[float]] = None,
                            compact: bool = True, mode: int = SLOPES_ND, stream=None):
    """synim_interaction_matrix_flat: the one-shot call with north_star's argument list (cube, per-sensor pupil mask,
    subaperture grid and valid mask, per-sensor composite matrices) -> CUDA float32 [n_modes][rows].  ``wfs`` as for
    ``Geometry``; the library builds and frees its own geometry and synchronises the device."""
    import torch
    assert cube.is_cuda and cube.dtype == torch.float32 and cube.is_contiguous() and cube.dim() == 3
    n, ny, nx = (int(v) for v in cube.shape)
    grids = (WfsGrid * len(wfs))()
    keep, rows, on_device = [], 0, {}
    for k, w in enumerate(wfs):
        valid = np.ascontiguousarray(w.valid, dtype=np.uint8)
        pupil = on_device.get(id(w.pupil))     # the SAME pupil object -> the same device buffer -> shared maps (as in Geometry)
        if pupil is None:
            pupil = w.pupil if isinstance(w.pupil, torch.Tensor) else torch.from_numpy(np.ascontiguousarray(w.pupil, dtype=np.float32))
            pupil = pupil.to(device="cuda", dtype=torch.float32).contiguous()
            on_device[id(w.pupil)] = pupil
        keep.append((valid, pupil))
        grids[k].n_subap, grids[k].n_pix = int(w.n_subap), int(w.n_pix)
        grids[k].valid_mask = valid.ctypes.data
        grids[k].d_pupil = pupil.data_ptr()
        rows += 2 * int(np.count_nonzero(valid))
    out = torch.empty((n, max(rows, 1)), dtype=torch.float32, device=cube.device)[:, :rows]
    got = ctypes.c_int64(-1)
    _check(lib().synim_interaction_matrix_flat(cube.data_ptr(), n, ny, nx, len(wfs), grids, _affine_array(affines, scales),
                                               1 if compact else 0, int(mode), out.data_ptr(), int(out.stride(0)),
                                               ctypes.byref(got), _stream_ptr(stream)))
    assert got.value == rows
    del keep
    return out


def interaction_matrix_host(geom: Geometry, cube_host, bbox_host, affines: Sequence[Sequence[float]],
                            scales: Optional[Sequence[float]] = None, out_host=None, mode: int = SLOPES_ND,
                            stream=None):
    """synim_interaction_matrix_host: HOST buffers in and out (torch CPU tensors, pinned or not, or
    numpy arrays); copies and the final synchronisation happen inside the C call."""
    import torch

    def ptr(x):
        return x.data_ptr() if isinstance(x, torch.Tensor) else x.ctypes.data

    def check(x, name, dtype_t, dtype_n, shape):
        if isinstance(x, torch.Tensor):
            ok = (not x.is_cuda) and x.dtype == dtype_t and x.is_contiguous()
        else:
            ok = isinstance(x, np.ndarray) and x.dtype == dtype_n and x.flags["C_CONTIGUOUS"]
        if not ok or tuple(x.shape) != tuple(shape):
            raise ValueError(f"{name} must be a C-contiguous host array of {dtype_n.__name__} with shape {tuple(shape)}")

    n = int(cube_host.shape[0])
    rows = geom.num_rows
    check(cube_host, "cube_host", torch.float32, np.float32, (n, geom.ny, geom.nx))
    if bbox_host is not None:
        check(bbox_host, "bbox_host", torch.int32, np.int32, (n, 4))
    if len(affines) != geom.n_wfs:
        raise ValueError("one affine per sensor")
    if out_host is None:
        out_host = torch.empty((n, rows), dtype=torch.float32).pin_memory()
    check(out_host, "out_host", torch.float32, np.float32, (n, rows))
    arr = _affine_array(affines, scales)
    _check(lib().synim_interaction_matrix_host(geom._h, ptr(cube_host), n,
                                               None if bbox_host is None else ptr(bbox_host),
                                               arr, int(mode), ptr(out_host), _stream_ptr(stream)))
    return out_host


def dictionary_host(geom: Geometry, layers: Sequence[dict], mode: int = SLOPES_ND, stream=None):
    """synim_dictionary_host: ``layers`` is a list of dicts with ``cube`` (host float32 [n][ny][nx], torch CPU tensor or
    numpy), ``bbox`` (host int32 [n][4] or None), ``affines`` ([n_wfs][6]), optional ``scales`` and ``out`` (host float32
    [n][rows]; allocated pinned if missing).  Returns the list of output buffers."""
    import torch

    def ptr(x):
        return x.data_ptr() if isinstance(x, torch.Tensor) else x.ctypes.data

    def ok(x, dt_t, dt_n):
        if isinstance(x, torch.Tensor):
            return (not x.is_cuda) and x.dtype == dt_t and x.is_contiguous()
        return isinstance(x, np.ndarray) and x.dtype == dt_n and x.flags["C_CONTIGUOUS"]

    rows = geom.num_rows
    arr = (Layer * len(layers))()
    keep, outs = [], []
    for k, lay in enumerate(layers):
        cube, bbox = lay["cube"], lay.get("bbox")
        if not ok(cube, torch.float32, np.float32) or len(cube.shape) != 3:
            raise ValueError(f"layer {k}: cube must be a C-contiguous host float32 array [n][ny][nx]")
        n, ny, nx = (int(v) for v in cube.shape)
        if bbox is not None and (not ok(bbox, torch.int32, np.int32) or tuple(bbox.shape) != (n, 4)):
            raise ValueError(f"layer {k}: bbox must be a C-contiguous host int32 array [n][4]")
        if len(lay["affines"]) != geom.n_wfs:
            raise ValueError(f"layer {k}: one affine per sensor")
        out = lay.get("out")
        if out is None:
            out = torch.empty((n, rows), dtype=torch.float32).pin_memory()
        if not ok(out, torch.float32, np.float32) or tuple(out.shape) != (n, rows):
            raise ValueError(f"layer {k}: out must be a C-contiguous host float32 array [{n}][{rows}]")
        aff = _affine_array(lay["affines"], lay.get("scales"))
        keep.append((cube, bbox, out, aff))
        arr[k].h_influence, arr[k].n_modes, arr[k].ny, arr[k].nx = ptr(cube), n, ny, nx
        arr[k].h_bbox = None if bbox is None else ptr(bbox)
        arr[k].affine = ctypes.cast(aff, ctypes.POINTER(WfsAffine))
        arr[k].h_out = ptr(out)
        outs.append(out)
    _check(lib().synim_dictionary_host(geom._h, arr, len(layers), int(mode), _stream_ptr(stream)))
    del keep
    return outs


def projection_matrix(dm_cubes: Sequence, dm_maps: Sequence[Sequence[Sequence[float]]], layer_cube,
                      layer_maps: Sequence[Sequence[float]], pupil, lam: float, weights: Optional[Sequence[float]] = None,
                      out=None, stream=None):
    """synim_projection_matrix: ``dm_cubes`` CUDA float32 cubes [n][ny][nx] of the mirrors with their
    per-direction maps ``dm_maps[k][d]`` (a[6]); ``layer_cube`` / ``layer_maps`` likewise; ``pupil`` CUDA float32
    [mp][mp].  Returns P_opt as a CUDA tensor viewed [n_layer_modes][ld] (row l = column l of the column-major
    matrix: the projection of layer mode l onto all mirrors' modes)."""
    import torch
    n_dir = len(layer_maps)
    comps = (Component * len(dm_cubes))()
    keep = []
    n_a = 0
    for k, (cube, maps) in enumerate(zip(dm_cubes, dm_maps)):
        assert cube.is_cuda and cube.dtype == torch.float32 and cube.is_contiguous() and cube.dim() == 3
        assert len(maps) == n_dir
        arr = _affine_array(maps, None)
        keep.append(arr)
        comps[k].d_cube, comps[k].n_modes, comps[k].ny, comps[k].nx = cube.data_ptr(), int(cube.shape[0]), int(cube.shape[1]), int(cube.shape[2])
        comps[k].maps = ctypes.cast(arr, ctypes.POINTER(WfsAffine))
        n_a += int(cube.shape[0])
    assert layer_cube.is_cuda and layer_cube.dtype == torch.float32 and layer_cube.is_contiguous() and layer_cube.dim() == 3
    lay = Component()
    larr = _affine_array(layer_maps, None)
    lay.d_cube, lay.n_modes, lay.ny, lay.nx = layer_cube.data_ptr(), int(layer_cube.shape[0]), int(layer_cube.shape[1]), int(layer_cube.shape[2])
    lay.maps = ctypes.cast(larr, ctypes.POINTER(WfsAffine))
    assert pupil.is_cuda and pupil.dtype == torch.float32 and pupil.is_contiguous() and pupil.dim() == 2 and pupil.shape[0] == pupil.shape[1]
    n_l = int(layer_cube.shape[0])
    if out is None:
        out = torch.empty((n_l, n_a), dtype=torch.float32, device=layer_cube.device)
    assert out.is_cuda and out.dtype == torch.float32 and out.dim() == 2 and out.stride(1) == 1 and out.shape[0] >= n_l
    ld = int(out.stride(0)) if out.shape[0] > 1 else int(out.shape[1])
    w = None
    if weights is not None:
        assert len(weights) == n_dir
        w = (ctypes.c_double * n_dir)(*[float(v) for v in weights])
    _check(lib().synim_projection_matrix(comps, len(dm_cubes), ctypes.byref(lay), n_dir, w, pupil.data_ptr(), int(pupil.shape[0]),
                                         float(lam), out.data_ptr(), ld, _stream_ptr(stream)))
    del keep, larr
    return out


def affines_of(workload) -> list:
    """Composite matrices of a ``workloads.Workload`` through the library's own helper."""
    return [compose_affine(w.phys) for w in workload.wfs]
