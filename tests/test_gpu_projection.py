"""The tomographic projection matrix (synim_projection_matrix) against the oracle, on a B200.

Tolerance (R26): the operands are float32 samples (relative error ~1e-7), the contractions accumulate
K = n_dir * mp^2 products in float32 (relative error of an entry of P_DM^T P_DM <~ sqrt(K) * 2^-24) and the solve
amplifies that by the condition number of P_DM^T P_DM + lambda I; the bound used is 4 * cond * sqrt(K) * 2^-24 of
max|P_opt|, with lambda chosen so that cond is a few hundred.
"""
import math

import numpy as np
import pytest

from oracle import oracle as O
from paper_2606_07759_b200 import workloads as W

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def S():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("the -m gpu tests need a CUDA device")
    from paper_2606_07759_b200 import build, synim
    build.build_library()
    synim.lib()
    return synim


def rot(deg, mag, sx, sy):
    t = math.radians(deg)
    return [math.cos(t) / mag, math.sin(t) / mag, sx, -math.sin(t) / mag, math.cos(t) / mag, sy]


def _case(mp, lam_frac):
    pupil = W.make_pupil(mp, float(mp), 0.2)
    c0, _ = W.gaussian_cube(mp + 16, mp + 16, W.actuator_grid(7, mp / 6.0, mp / 2.0 + 2.0), mp / 6.0)
    c1, _ = W.gaussian_cube(mp + 24, mp + 24, W.actuator_grid(5, mp / 4.0, mp / 2.0 + 6.0), mp / 4.0)
    cl = W.random_smooth_cube(9, mp + 32, mp + 32, 9)
    dirs = [(0.0, 0.0), (3.3, -1.2), (-2.1, 2.7), (0.4, 3.9)]
    maps0 = [rot(1.0, 1.0, 0.0, 0.0) for _ in dirs]                       # ground mirror: no footprint
    maps1 = [rot(-2.0, 1.02, 1.0 * dx, 1.0 * dy) for dx, dy in dirs]      # altitude mirror
    mapsl = [rot(0.0, 1.0, 2.0 * dx, 2.0 * dy) for dx, dy in dirs]        # a higher layer
    wts = [1.0, 0.5, 2.0, 1.5]
    p_dm = np.hstack([O.projection_operand(c0, maps0, pupil, wts), O.projection_operand(c1, maps1, pupil, wts)])
    p_l = O.projection_operand(cl, mapsl, pupil, wts)
    lam = lam_frac * np.trace(p_dm.T @ p_dm) / p_dm.shape[1]
    cond = np.linalg.cond(p_dm.T @ p_dm + lam * np.eye(p_dm.shape[1]))
    return pupil, (c0, c1), (maps0, maps1), cl, mapsl, wts, lam, O.projection_matrix(p_dm, p_l, lam), cond, p_dm.shape[0]


def test_projection_matrix_against_the_oracle(S):
    import torch
    for mp, lam_frac in ((24, 0.05), (40, 0.08)):
        pupil, cubes, maps, cl, mapsl, wts, lam, ref, cond, k = _case(mp, lam_frac)
        n_a = ref.shape[0]
        out = torch.full((cl.shape[0], n_a + 5), float("nan"), dtype=torch.float32, device="cuda")
        S.projection_matrix([torch.from_numpy(c).cuda() for c in cubes], maps, torch.from_numpy(cl).cuda(), mapsl,
                            torch.from_numpy(pupil).cuda(), lam, weights=wts, out=out)
        res = out.cpu().numpy()
        assert np.isnan(res[:, n_a:]).all()                                   # padding rows untouched
        got = res[:, :n_a].T.astype(np.float64)
        tol = 4.0 * cond * math.sqrt(k) * 2.0 ** -24
        err = np.abs(got - ref).max() / np.abs(ref).max()
        print(f"P_opt {ref.shape}: cond {cond:.0f}, K {k}, max err {err:.2e} (bound {tol:.2e})")
        assert tol < 1e-2 and err <= tol


def test_projection_matrix_argument_errors(S):
    import torch
    pupil, cubes, maps, cl, mapsl, wts, lam, ref, cond, k = _case(16, 0.05)
    dev = [torch.from_numpy(c).cuda() for c in cubes]
    with pytest.raises(S.SynimError) as e:
        S.projection_matrix(dev, maps, torch.from_numpy(cl).cuda(), mapsl, torch.from_numpy(pupil).cuda(), -1.0)
    assert e.value.status == S.ERR_INVALID_ARG
    # lambda = 0 with more mirror modes than the operand has rows that see them: not positive definite -> reported
    dark = torch.zeros((16, 16), dtype=torch.float32, device="cuda")
    with pytest.raises(S.SynimError) as e:
        S.projection_matrix(dev, maps, torch.from_numpy(cl).cuda(), mapsl, dark, 0.0)
    assert e.value.status == S.ERR_INVALID_ARG
