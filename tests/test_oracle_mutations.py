"""Every pin must earn its keep: plausible mistakes are planted in a copy of the oracle's source, one at a time, and each
must make at least one of the oracle's pins (tests/test_oracle_pins.py, test_oracle_repair_pins.py) fail.  This is the
check a reviewer would otherwise do by hand; it shows that the pins, not the oracle's own formula, decide what is right
(a dropped term, a wrong sign or index, a transposed operand, a threshold, an aggregation).  The mutated library is built
in a scratch directory and reaches the pins through SYNIM_ORACLE_LIB; nothing under oracle/ is touched."""
import os
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
SRC = os.path.join(ROOT, "oracle", "synim_oracle.c")

# (name, text in synim_oracle.c, replacement, occurrences to replace: 0 = all)
MUTATIONS = [
    # numerical-derivative engine
    ("nd: /2 of D_x dropped", "const double dx = (PHI(i, j + 1) - PHI(i, j - 1)) / 2.0;", "const double dx = (PHI(i, j + 1) - PHI(i, j - 1));", 1),
    ("nd: forward difference", "const double dy = (PHI(i + 1, j) - PHI(i - 1, j)) / 2.0;", "const double dy = (PHI(i + 1, j) - PHI(i, j));", 1),
    ("nd: D_x along rows", "const double dx = (PHI(i, j + 1) - PHI(i, j - 1)) / 2.0;", "const double dx = (PHI(i + 1, j) - PHI(i - 1, j)) / 2.0;", 1),
    ("nd: weights squared", "ax += p * dx;", "ax += p * p * dx;", 1),
    ("nd: plain mean instead of the P-weighted one", "w += p;\n                    ax += p * dx;", "w += 1.0;\n                    ax += p * dx;", 1),
    ("nd: slope scale ignored", "sx[k] = scale * ax / w;", "sx[k] = ax / w;", 1),
    # single bilinear resampling
    ("resample: fx and fy swapped", "(1.0 - fy) * ((1.0 - fx) * v00 + fx * v01) + fy * ((1.0 - fx) * v10 + fx * v11)",
     "(1.0 - fx) * ((1.0 - fy) * v00 + fy * v01) + fx * ((1.0 - fy) * v10 + fy * v11)", 1),
    ("resample: WFS centre at M/2", "const double cw = (M - 1) / 2.0, cx = (nx - 1) / 2.0, cy = (ny - 1) / 2.0;",
     "const double cw = M / 2.0, cx = (nx - 1) / 2.0, cy = (ny - 1) / 2.0;", 1),
    ("resample: source centre at nx/2", "const double cw = (M - 1) / 2.0, cx = (nx - 1) / 2.0, cy = (ny - 1) / 2.0;",
     "const double cw = (M - 1) / 2.0, cx = nx / 2.0, cy = (ny - 1) / 2.0;", 1),
    ("resample: transposed matrix", "const double xs = a[0] * xw + a[1] * yw + a[2];", "const double xs = a[0] * xw + a[3] * yw + a[2];", 1),
    ("resample: first column dropped", "if (c0 >= 0 && c0 < nx) v00 = g[r0 * (long)nx + c0];", "if (c0 > 0 && c0 < nx) v00 = g[r0 * (long)nx + c0];", 1),
    ("resample: nearest neighbour in x", "const double fx = col - fc, fy = row - fr;", "const double fx = 0.0, fy = row - fr;", 1),
    # G-tilt telescoping sum (reading R13)
    ("gtilt: validity threshold P > 0", ">= 0.5f", "> 0.0f", 0),
    ("gtilt: mean of the per-row ratios", "{ num += PHI(i, jl) - PHI(i, jf); den += jl - jf; }",
     "{ num += (PHI(i, jl) - PHI(i, jf)) / (jl - jf); den += 1.0; }", 1),
    ("gtilt: denominator counts pixels, not steps", "den += l - f;", "den += l - f + 1;", 1),
    ("gtilt: one pixel inside the edge", "{ num += PHI(l, j) - PHI(f, j); den += l - f; }", "{ num += PHI(l - 1, j) - PHI(f, j); den += l - f; }", 1),
    # composite matrix
    ("compose: footprint shift with the wrong sign", "+ fx - ddx;", "- fx - ddx;", 1),
    ("compose: cone factor 1 + h/H", "1.0 - h / H", "1.0 + h / H", 1),
    ("compose: WFS rotation the other way", "B01 = sw / mx, B10 = -sw / my", "B01 = -sw / mx, B10 = sw / my", 1),
    ("compose: WFS shift not scaled by the cone factor", "const double c0 = -kappa * (B00 * dwx + B01 * dwy)", "const double c0 = -(B00 * dwx + B01 * dwy)", 1),
    ("compose: DM rotation dropped", "a[3] = -sd * C00 + cd * C10;", "a[3] = cd * C10;", 1),
    # edge repair
    ("repair: 2*P2 - P1", "sum += 2.0 * p1 - phi[(long)i2 * P + j2];", "sum += 2.0 * phi[(long)i2 * P + j2] - p1;", 1),
    ("repair: sum not normalised", "phi[q] = sum / n_dir;", "phi[q] = sum;", 1),
    ("repair: loose threshold", "core[q] = mu[q] >= threshold ? 1 : 0;", "core[q] = mu[q] >= 0.5 ? 1 : 0;", 1),
    ("repair: diagonal neighbours", "di[4] = {0, 0, 1, -1}, dj[4] = {1, -1, 0, 0}", "di[4] = {1, 1, -1, -1}, dj[4] = {1, -1, 1, -1}", 1),
    ("repair: screen not cleared outside the core", "if (!core[q]) phi[q] = 0.0;", ";", 1),
    ("repair: slopes averaged over ring pixels too", "if (!core[(long)(i + 1) * P + (j + 1)]) continue;", ";", 1),
    ("repair: linear extrapolation never used", "if (i2 >= 0 && i2 < P && j2 >= 0 && j2 < P && core[(long)i2 * P + j2]) sum +=", "if (0) sum +=", 1),
]

PINS = ["tests/test_oracle_pins.py", "tests/test_oracle_repair_pins.py"]


def _survives(args):
    """Build the mutant and run the pins against it; True if every pin still passes (the mutant survives)."""
    idx, (name, old, new, count), out_dir = args
    src = open(SRC).read()
    assert old in src, f"mutation '{name}' no longer applies to oracle/synim_oracle.c"
    mutated = src.replace(old, new) if count == 0 else src.replace(old, new, count)
    c = os.path.join(out_dir, f"m{idx}.c")
    lib = os.path.join(out_dir, f"libmutant{idx}.so")
    with open(c, "w") as f:
        f.write(mutated)
    subprocess.check_call(["gcc", "-O1", "-std=c11", "-fPIC", "-shared", "-fopenmp", "-o", lib, c, "-lm"])
    env = dict(os.environ, SYNIM_ORACLE_LIB=lib, OMP_NUM_THREADS="1", PYTHONPATH=ROOT)
    # (the sanitizer and mutation tests themselves are left out: they build their own libraries)
    res = subprocess.run([sys.executable, "-m", "pytest", *PINS, "-x", "-q", "-p", "no:cacheprovider",
                          "-k", "not sanitiz and not mutation"], cwd=ROOT, env=env, capture_output=True, text=True, timeout=600)
    return res.returncode == 0


@pytest.mark.timeout(900)
def test_every_planted_mistake_fails_a_pin(tmp_path):
    # control: the same pipeline on the unmutated source passes every pin (so a "failure" below is a pin's, not the harness's)
    control = ("control: a comment", "/* Steps 3-4, numerical derivative. */", "/* Steps 3-4, numerical derivative */", 1)
    assert _survives((len(MUTATIONS), control, str(tmp_path)))
    jobs = [(i, m, str(tmp_path)) for i, m in enumerate(MUTATIONS)]
    with ThreadPoolExecutor(max_workers=min(8, os.cpu_count() or 1)) as pool:
        survived = list(pool.map(_survives, jobs))
    alive = [MUTATIONS[i][0] for i, s in enumerate(survived) if s]
    assert not alive, f"mutants no pin catches: {alive}"


# The projection-matrix oracle is numpy code in oracle/oracle.py: the same game, with the mutated module
# installed as oracle.oracle in a child interpreter before the pins (tests/test_oracle_projection_pins.py) are collected.
PY_MUTATIONS = [
    ("popt: regulariser subtracted", "+ float(lam) * np.eye(p_dm.shape[1])", "- float(lam) * np.eye(p_dm.shape[1])"),
    ("popt: regulariser ignored", "+ float(lam) * np.eye(p_dm.shape[1])", "+ 0.0 * np.eye(p_dm.shape[1])"),
    ("popt: no inverse", "return np.linalg.solve(g, p_dm.T @ p_layer)", "return g @ (p_dm.T @ p_layer)"),
    ("popt: direction weights not square-rooted", "float(np.sqrt(w[d])) *", "float(w[d]) *"),
    ("popt: pupil weighting dropped", "(pupil * resample(cube[m], mp, maps[d])).ravel()", "(resample(cube[m], mp, maps[d])).ravel()"),
    ("popt: every direction seen through the first map", "resample(cube[m], mp, maps[d])", "resample(cube[m], mp, maps[0])"),
]

_CHILD = r"""
import sys, types
root, old, new = sys.argv[1], sys.argv[2], sys.argv[3]
sys.path.insert(0, root)
import oracle as pkg
path = root + "/oracle/oracle.py"
src = open(path).read()
assert old in src, "mutation no longer applies to oracle/oracle.py"
mod = types.ModuleType("oracle.oracle")
mod.__file__ = path
mod.__package__ = "oracle"
sys.modules["oracle.oracle"] = mod
exec(compile(src.replace(old, new, 1), path, "exec"), mod.__dict__)
pkg.oracle = mod
import pytest
sys.exit(pytest.main([root + "/tests/test_oracle_projection_pins.py", "-x", "-q", "-p", "no:cacheprovider"]))
"""


def _py_survives(m):
    name, old, new = m
    res = subprocess.run([sys.executable, "-c", _CHILD, ROOT, old, new], cwd=ROOT, capture_output=True, text=True, timeout=600)
    assert "no longer applies" not in res.stderr, name
    return res.returncode == 0


@pytest.mark.timeout(600)
def test_every_planted_mistake_in_the_projection_oracle_fails_a_pin():
    assert _py_survives(("control", "written out as the paper gives it", "written out as the paper gives it "))
    with ThreadPoolExecutor(max_workers=min(6, os.cpu_count() or 1)) as pool:
        survived = list(pool.map(_py_survives, PY_MUTATIONS))
    alive = [PY_MUTATIONS[i][0] for i, s in enumerate(survived) if s]
    assert not alive, f"mutants no pin catches: {alive}"
