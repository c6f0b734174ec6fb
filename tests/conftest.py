import os
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box with -m gpu)")


# The GPU run is `pytest -x`: one failure hides every test after it.  So the GPU tests run in the order of how
# much hardware time the path under test has already seen: first the strip kernel on zonal modes
# (measured on a B200 in rounds 1 and 2), then everything that (also) goes through the tile kernel, then the host pipeline
# and the dictionary, then the paths written after GPU access closed (edge repair, the packed zonal walk, P_opt), and last
# the -DSYNIM_CHECKS trap build, which drives every one of those paths again (a trap is a device fault: nothing after it
# in the process can run).
# The order inside a class is the files' own; tests that need no GPU are not touched.
_GPU_FIRST = ("test_config1_", "test_config2_", "test_config3_", "test_config4_", "test_compute_bboxes", "test_octagon_")
_GPU_LATER = (
    ("test_host_", "test_dictionary_host", "test_mode_ranges_through", "test_flat_one_shot", "test_one_geometry_many"),
    ("test_edge_repair", "test_packed_zonal", "test_projection_matrix"),
    ("test_seeded_random_cases",),
    ("test_debug_build",),
)


def _gpu_rank(item):
    if item.get_closest_marker("gpu") is None or item.name.startswith(_GPU_FIRST):
        return 0
    for rank, names in enumerate(_GPU_LATER, start=2):
        if item.name.startswith(names):
            return rank
    return 1


def pytest_collection_modifyitems(config, items):
    items.sort(key=_gpu_rank)          # (stable: ties keep the collection order)
