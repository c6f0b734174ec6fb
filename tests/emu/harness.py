"""TEST INFRASTRUCTURE (tests/emu/README.md): build the library's own sources for the host against the emulation of
the CUDA execution model and drive its C ABI with numpy buffers.  Not a product path: nothing under
paper_2606_07759_b200/ knows about it, and the library proper is never built this way."""
from __future__ import annotations

import ctypes
import os
import subprocess
import sys

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.abspath(os.path.join(HERE, "..", ".."))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)
if HERE not in sys.path:
    sys.path.insert(0, HERE)

import convert  # noqa: E402
from paper_2606_07759_b200 import synim as S  # noqa: E402  (ctypes structure definitions only; its lib() is not used)

CXX = ["g++", "-O1", "-g", "-std=c++17", "-fPIC", "-shared", "-mfma", "-ffp-contract=fast", "-Wno-psabi"]


def build(out_dir: str, defines=()) -> str:
    """Convert csrc/*.cu, compile them with emu.cpp into libsynim_emu.so, and build the CPU stand-ins of cuBLAS /
    cuSOLVER under the sonames synim_popt.cu asks dlopen for.  Returns the path of the emulated library."""
    gen = os.path.join(out_dir, "gen")
    srcs = convert.convert_all(gen)
    lib = os.path.join(out_dir, "libsynim_emu.so")
    # SYNIM_EMU_CXXFLAGS: extra compiler flags, e.g. "-fsanitize=address,undefined" for a run with libasan preloaded
    extra = os.environ.get("SYNIM_EMU_CXXFLAGS", "").split()
    subprocess.check_call(CXX + extra + [f"-D{d}" for d in defines] +
                          ["-I" + HERE, "-I" + gen, "-I" + os.path.join(ROOT, "include"), "-o", lib] + srcs +
                          [os.path.join(HERE, "emu.cpp"), "-ldl"])
    fake = os.path.join(out_dir, "libcublas.so.12")
    subprocess.check_call(["g++", "-O2", "-fPIC", "-shared", "-o", fake, os.path.join(HERE, "fake_blas.cpp")])
    subprocess.check_call(["cp", fake, os.path.join(out_dir, "libcusolver.so.11")])
    return lib


class Emu:
    """The emulated library behind its C ABI.  "Device" buffers are numpy arrays registered with the emulator, so
    that every global access of a kernel is checked against them."""

    def __init__(self, lib_path: str):
        # (synim_projection_matrix dlopens "libcublas.so.12" / "libcusolver.so.11": run it in a process whose
        # LD_LIBRARY_PATH starts with the directory of the stand-ins that build() put beside the library)
        L = ctypes.CDLL(lib_path)
        vp, i32, i64 = ctypes.c_void_p, ctypes.c_int32, ctypes.c_int64
        L.synim_compose_affine.argtypes = [ctypes.POINTER(S.WfsPhysical), ctypes.POINTER(S.WfsAffine)]
        L.synim_create_geometry.argtypes = [i32, i32, i32, ctypes.POINTER(S.WfsGrid), vp, ctypes.POINTER(vp)]
        L.synim_num_rows.restype = i64
        L.synim_num_rows.argtypes = [vp]
        L.synim_interaction_matrix.argtypes = [vp, vp, i32, vp, vp, i32, i32, ctypes.POINTER(S.WfsAffine), ctypes.c_int, vp, i64, vp]
        L.synim_interaction_matrix_repaired.argtypes = [vp, vp, i32, vp, vp, i32, i32, ctypes.POINTER(S.WfsAffine), vp,
                                                        ctypes.c_double, vp, i64, vp]
        L.synim_interaction_matrix_flat.argtypes = [vp, i32, i32, i32, i32, ctypes.POINTER(S.WfsGrid), ctypes.POINTER(S.WfsAffine),
                                                    i32, ctypes.c_int, vp, i64, ctypes.POINTER(i64), vp]
        L.synim_compute_bboxes.argtypes = [vp, i32, i32, i32, vp, vp, vp]
        L.synim_bbox_extent.argtypes = [vp, i32, ctypes.POINTER(i32), ctypes.POINTER(i32), vp]
        L.synim_interaction_matrix_host.argtypes = [vp, vp, i32, vp, ctypes.POINTER(S.WfsAffine), ctypes.c_int, vp, vp]
        L.synim_dictionary_host.argtypes = [vp, ctypes.POINTER(S.Layer), i32, ctypes.c_int, vp]
        L.synim_projection_matrix.argtypes = [ctypes.POINTER(S.Component), i32, ctypes.POINTER(S.Component), i32,
                                              ctypes.POINTER(ctypes.c_double), vp, i32, ctypes.c_double, vp, i64, vp]
        L.synim_destroy.argtypes = [vp]
        L.synim_destroy.restype = None
        L.synim_last_error.restype = ctypes.c_char_p
        L.emu_register.argtypes = [vp, ctypes.c_size_t]
        L.emu_track_stores.argtypes = [vp, ctypes.c_size_t]
        L.emu_store_counts.argtypes = [vp]
        self.L = L
        self.store_counts = None     # after interaction_matrix(count_stores=True): uint8 [n_modes][rows + ld_pad]
        self.pre_launch = None       # optional callable run right before the interaction-matrix call (op_counts.py)

    def reg(self, a: np.ndarray) -> np.ndarray:
        self.L.emu_register(a.ctypes.data, a.nbytes)
        return a

    def chk(self, rc: int) -> None:
        if rc != 0:
            raise RuntimeError(f"status {rc}: {self.L.synim_last_error().decode()}")

    def affines(self, wfs_list):
        out = []
        for w in wfs_list:
            p = S.WfsPhysical(*[float(w.phys[k]) for k in S.PHYSICAL_FIELDS])
            o = S.WfsAffine()
            self.chk(self.L.synim_compose_affine(ctypes.byref(p), ctypes.byref(o)))
            out.append(list(o.a))
        return out

    def geometry(self, wfs_list, ny, nx):
        n = len(wfs_list)
        grids = (S.WfsGrid * n)()
        keep, shared = [], {}
        for k, w in enumerate(wfs_list):
            valid = np.ascontiguousarray(w.valid, dtype=np.uint8)
            pupil = shared.get(id(w.pupil))
            if pupil is None:
                pupil = self.reg(np.ascontiguousarray(w.pupil, dtype=np.float32).copy())
                shared[id(w.pupil)] = pupil
            keep.append((valid, pupil))
            grids[k].n_subap, grids[k].n_pix = int(w.n_subap), int(w.n_pix)
            grids[k].valid_mask = valid.ctypes.data
            grids[k].d_pupil = pupil.ctypes.data
        h = ctypes.c_void_p()
        self.chk(self.L.synim_create_geometry(ny, nx, n, grids, None, ctypes.byref(h)))
        return h, keep

    def interaction_matrix_flat(self, wl, compact=True, mode=0):
        """synim_interaction_matrix_flat (create -> supports -> matrix -> destroy in one call) -> float64 [rows][n_modes]."""
        L = self.L
        n = len(wl.wfs)
        grids = (S.WfsGrid * n)()
        keep, shared = [], {}
        for k, w in enumerate(wl.wfs):
            valid = np.ascontiguousarray(w.valid, dtype=np.uint8)
            pupil = shared.get(id(w.pupil))      # (sensors that pass the same buffer share their maps, as in geometry())
            if pupil is None:
                pupil = self.reg(np.ascontiguousarray(w.pupil, dtype=np.float32).copy())
                shared[id(w.pupil)] = pupil
            keep.append((valid, pupil))
            grids[k].n_subap, grids[k].n_pix = int(w.n_subap), int(w.n_pix)
            grids[k].valid_mask = valid.ctypes.data
            grids[k].d_pupil = pupil.ctypes.data
        cube = self.reg(np.ascontiguousarray(wl.cube, dtype=np.float32))
        out = self.reg(np.full((wl.n_modes, wl.n_rows), np.nan, np.float32))
        arr = S._affine_array(self.affines(wl.wfs), [w.slope_scale for w in wl.wfs])
        rows = ctypes.c_int64(-1)
        self.chk(L.synim_interaction_matrix_flat(cube.ctypes.data, wl.n_modes, wl.ny, wl.nx, n, grids, arr, 1 if compact else 0, mode,
                                                 out.ctypes.data, wl.n_rows, ctypes.byref(rows), None))
        assert rows.value == wl.n_rows
        res = out.T.astype(np.float64)
        assert np.isfinite(res).all(), "unwritten IM elements"
        return res

    def interaction_matrix(self, wl, use_bbox=True, ld_pad=0, hint=True, octagon=True, mode=0, affines=None, scales=None,
                           mask=None, threshold=0.999999, count_stores=False):
        """The IM of a workload through the emulated C ABI -> float64 [rows][n_modes] (as tests/test_gpu_parity.gpu_im)."""
        L = self.L
        h, keep = self.geometry(wl.wfs, wl.ny, wl.nx)
        rows = int(L.synim_num_rows(h))
        assert rows == wl.n_rows
        cube = self.reg(np.ascontiguousarray(wl.cube, dtype=np.float32))
        assert cube.ctypes.data % 16 == 0
        bptr = dptr = None
        bw = bh = 0
        if use_bbox and wl.bbox is not None:
            bbox = self.reg(np.zeros((wl.n_modes, 4), np.int32))
            diag = self.reg(np.zeros((wl.n_modes, 4), np.int32))
            self.chk(L.synim_compute_bboxes(cube.ctypes.data, wl.n_modes, wl.ny, wl.nx, bbox.ctypes.data, diag.ctypes.data, None))
            assert np.array_equal(bbox, wl.bbox)
            bptr = bbox.ctypes.data
            if octagon:
                dptr = diag.ctypes.data
            if hint:
                a, b = ctypes.c_int32(), ctypes.c_int32()
                self.chk(L.synim_bbox_extent(bptr, wl.n_modes, ctypes.byref(a), ctypes.byref(b), None))
                bw, bh = a.value, b.value
        out = self.reg(np.full((wl.n_modes, rows + ld_pad), np.nan, np.float32))
        if affines is None:
            affines = self.affines(wl.wfs)
        if scales is None:
            scales = [w.slope_scale for w in wl.wfs]
        arr = S._affine_array(affines, scales)
        if self.pre_launch:
            self.pre_launch()
        if count_stores:
            L.emu_track_stores(out.ctypes.data, out.nbytes)
        if mask is not None:
            mk = self.reg(np.ascontiguousarray(mask, dtype=np.float32).copy())
            self.chk(L.synim_interaction_matrix_repaired(h, cube.ctypes.data, wl.n_modes, bptr, dptr, bw, bh, arr, mk.ctypes.data,
                                                         threshold, out.ctypes.data, rows + ld_pad, None))
        else:
            self.chk(L.synim_interaction_matrix(h, cube.ctypes.data, wl.n_modes, bptr, dptr, bw, bh, arr, mode, out.ctypes.data,
                                                rows + ld_pad, None))
        if count_stores:
            cnt = np.zeros(out.shape, np.uint8)
            L.emu_store_counts(cnt.ctypes.data)
            self.store_counts = cnt
        L.synim_destroy(h)
        if ld_pad:
            assert np.isnan(out[:, rows:]).all()          # padding rows are left untouched
        res = out[:, :rows].T.astype(np.float64)
        assert np.isfinite(res).all(), "unwritten IM elements"
        return res
