"""TEST INFRASTRUCTURE (tests/emu/README.md): dynamic operation counts of the hot kernels from the emulated library --
shared-memory loads and stores, warp collectives and global accesses per (mode, sensor) column, in warp-instruction
equivalents (lane operations / 32; a predicated-off lane does not count, so these are lower bounds of the issued
instructions).  Not a timing: a way to compare variants of a kernel without hardware.

    python tests/emu/op_counts.py            # prints a markdown table (profiles/r02_emulated_op_counts.md)
"""
import ctypes
import os
import sys
import tempfile

HERE = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, HERE)
import harness  # noqa: E402
from paper_2606_07759_b200 import workloads as W  # noqa: E402


def main():
    out = tempfile.mkdtemp(prefix="emu_counts_")
    e = harness.Emu(harness.build(out))
    e.L.emu_counters.argtypes = [ctypes.POINTER(ctypes.c_ulonglong)]

    def counts():
        a = (ctypes.c_ulonglong * 4)()
        e.L.emu_counters(a)
        return [int(v) for v in a]

    rows = []
    for cfg, n, variants in ((2, 60, ("default", "packed")), (3, 60, ("default", "packed")), (4, 40, ("default", "packed")),
                             (5, 2, ("tiles",))):
        wl = W.make_config(cfg, max_modes=n)
        for v in variants:
            os.environ["SYNIM_ZONAL_PACKED"] = "1" if v == "packed" else "0"
            e.pre_launch = counts          # reset right before the interaction-matrix call (set-up kernels excluded)
            e.interaction_matrix(wl)
            c = counts()
            k = 32.0 * wl.n_columns
            rows.append((cfg, v, wl.n_modes, c[0] / k, c[1] / k, c[2] / k, c[3] / k))
    print("| config | kernel variant | modes run | LDS | shared stores | shuffles / votes / syncwarps | global loads + stores |")
    print("|---|---|---|---|---|---|---|")
    for r in rows:
        print("| %d | %s | %d | %.0f | %.0f | %.0f | %.0f |" % r)


if __name__ == "__main__":
    main()
