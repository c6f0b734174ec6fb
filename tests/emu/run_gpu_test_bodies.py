"""TEST INFRASTRUCTURE (tests/emu/README.md): the BODIES of the `-m gpu` tests that reach the library through
tests/test_gpu_parity.gpu_im only, run against the emulated library with the GPU tests' own strict rule (assert_parity:
north_star's bar, exact zeros, rim entries counted and bounded).  What a hardware run of those tests will compute, bar the
things only hardware has (tests/emu/README.md).  Tests that also drive torch / the real binding directly (argument errors,
host buffers, the one-shot call, compute_bboxes) have their own emulated counterparts in tests/test_kernel_logic_emulated.py.

    python tests/emu/run_gpu_test_bodies.py [test names]        # about 5 minutes for the default list
"""
import inspect
import os
import sys
import tempfile
import time
import traceback

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, HERE)
sys.path.insert(0, os.path.join(HERE, ".."))
import harness  # noqa: E402
import test_gpu_parity as T  # noqa: E402
from paper_2606_07759_b200 import synim as S  # noqa: E402  (constants only)

DEFAULT = ("test_config1_scao_tiny_full", "test_config1_with_padding_rows_scale_and_no_hint", "test_config2_vlt_subset",
           "test_config3_elt_ground_six_rotated_lgs", "test_config4_altitude_dm_cone_footprint_and_giant_ngs_subaps",
           "test_config5_dense_zernike_modes", "test_more_than_sixteen_sensors_take_a_second_launch",
           "test_dense_modes_with_padding_rows", "test_gtilt_estimator_on_the_gpu", "test_dense_path_on_zonal_cube_equals_bbox_path",
           "test_identity_transform_is_exact_on_integer_data", "test_tilt_and_quadratic_closed_forms_on_the_gpu",
           "test_wfs_looking_past_the_source_grid_and_strong_magnification", "test_full_physical_chain_and_degenerate_sensor_grids",
           "test_octagon_footprints_change_nothing_but_the_work", "test_packed_zonal_walk_is_opt_in_and_agrees_with_the_oracle",
           "test_edge_repair_on_masked_modes", "test_edge_repair_soft_mask_thresholds_and_odd_sensors",
           "test_seeded_random_cases_on_the_gpu")


class _Env:      # stands in for pytest's monkeypatch fixture
    def setenv(self, k, v):
        os.environ[k] = v

    def delenv(self, k, raising=True):
        os.environ.pop(k, None)


def main(names):
    emu = harness.Emu(harness.build(tempfile.mkdtemp(prefix="emu_bodies_")))

    def gpu_im(S_, wl, affines=None, scales=None, use_bbox=True, ld_pad=0, hint=True, octagon=True, mode=0, mask=None,
               threshold=0.999999):
        return emu.interaction_matrix(wl, use_bbox=use_bbox, ld_pad=ld_pad, hint=hint, octagon=octagon, mode=mode,
                                      affines=affines, scales=scales, mask=mask, threshold=threshold).astype(np.float32)
    T.gpu_im = gpu_im
    failed = 0
    for n in names:
        f = getattr(T, n)
        args = [S if p == "S" else _Env() if p == "monkeypatch" else None for p in inspect.signature(f).parameters]
        t = time.time()
        try:
            f(*args)
            print(f"PASS {n} ({time.time() - t:.0f} s)", flush=True)
        except Exception:
            failed += 1
            print(f"FAIL {n}: {traceback.format_exc()[-800:]}", flush=True)
        os.environ.pop("SYNIM_ZONAL_PACKED", None)
    return failed


if __name__ == "__main__":
    sys.exit(1 if main(sys.argv[1:] or DEFAULT) else 0)
