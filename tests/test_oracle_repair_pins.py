"""Pins of the oracle's edge repair (sec. 2.3; readings R18-R22 of DESIGN.md) against things
other than itself (CPU only): a hand-computed example, exactness on constant and linear phases, the no-op
case, the threshold, and an independent restatement built on scipy.ndimage.binary_dilation.

Set-up used throughout: with the identity transform and a source grid of (M+2) x (M+2) pixels, WFS pixel
(i, j), i, j in -1..M, samples source pixel (i+1, j+1) exactly, so the halo-grid screens ARE the source arrays.
"""
import math

import numpy as np
import pytest
import scipy.ndimage as ndi

from oracle import oracle as O

IDENT = [1.0, 0.0, 0.0, 0.0, 1.0, 0.0]
TAU = O.REPAIR_THRESHOLD


def rot_affine(deg, mag=1.0, sx=0.0, sy=0.0):
    t = math.radians(deg)
    return [math.cos(t) / mag, math.sin(t) / mag, sx, -math.sin(t) / mag, math.cos(t) / mag, sy]


def test_threshold_constant_is_the_papers_example():
    assert TAU == 0.999999          # PAPER.md:71 "(e.g., 0.999999)"


# ------------------------------------------------------------------------------- the worked example
def _hand_example():
    core = [(3, 1), (3, 2), (3, 3), (2, 3), (1, 3), (2, 4)]
    val = {(3, 1): 2.0, (3, 2): 3.0, (3, 3): 5.0, (2, 3): 7.0, (1, 3): 11.0, (2, 4): 13.0}
    mask = np.zeros((7, 7), np.float32)
    g = np.full((7, 7), 100.0, np.float32)       # whatever lies outside the core must not matter
    for q in core:
        mask[q] = 1.0
        g[q] = val[q]
    return core, val, mask, g


def test_hand_computed_example_every_kind_of_ring_pixel():
    """Worked by hand from PAPER.md:71-74.  Core: a run (3,1)-(3,3), a run (1,3)-(3,3) and (2,4).
    (3,0): one direction, two reference pixels  -> 2*2-3 = 1          (linear extrapolation)
    (2,1): one direction, one reference pixel   -> 2                  (constant extrapolation)
    (2,2): east linear 2*7-13 = 1, south constant 3 -> (1+3)/2 = 2    (normalised average of mixed kinds)
    (3,4): west linear 2*5-3 = 7, north constant 13 -> 10
    (4,4): touches the core only diagonally     -> not a ring pixel, stays 0 (4-neighbour dilation)."""
    core, val, mask, g = _hand_example()
    phi, c, r = O.repair_screen(g, mask, 5, IDENT)
    exp = np.zeros((7, 7))
    for q in core:
        exp[q] = val[q]
    ring = {(3, 0): 1.0, (2, 1): 2.0, (2, 2): 2.0, (3, 4): 10.0, (1, 4): 12.0, (2, 5): 19.0, (0, 3): 15.0,
            (1, 2): 11.0, (4, 1): 2.0, (4, 2): 3.0, (4, 3): 3.0}
    for q, v in ring.items():
        exp[q] = v
    assert np.array_equal(phi, exp)
    assert {tuple(q) for q in np.argwhere(c)} == set(core)
    assert {tuple(q) for q in np.argwhere(r)} == set(ring)
    # slopes of the one 5x5 subaperture: mean over the six core pixels of the central differences of the
    # repaired screen (worked by hand: sum D_x = 1+1.5+3.5+5.5+0.5+6 = 18, sum D_y = 0+0.5-2-3-4-1 = -9.5)
    s = O.slopes_wfs_repair(g[None], mask, np.ones((5, 5), np.float32), 1, 5, np.ones((1, 1), np.uint8), IDENT)
    assert np.allclose(s[0], [3.0, -9.5 / 6.0], rtol=0, atol=1e-14)
    # the pupil weights enter as P*core: doubling P on pixel (2,4) [WFS pixel (1,3)] changes the weighted mean
    p = np.ones((5, 5), np.float32)
    p[1, 3] = 2.0
    s = O.slopes_wfs_repair(g[None], mask, p, 1, 5, np.ones((1, 1), np.uint8), IDENT, scale=2.0)
    assert np.allclose(s[0], [2.0 * (18.0 + 6.0) / 7.0, 2.0 * (-9.5 - 1.0) / 7.0], rtol=0, atol=1e-14)


# ------------------------------------------------------------------------------- no-op and exactness
def test_all_ones_mask_changes_nothing():
    """Every pixel core, no ring: the repaired engine IS the numerical-derivative engine, bit for bit."""
    rng = np.random.default_rng(5)
    n, m = 40, 24                                        # the halo of the 24-px sensor stays inside the grid
    cube = rng.normal(size=(3, n, n)).astype(np.float32)
    pupil = rng.uniform(0.1, 1.0, (m, m)).astype(np.float32)
    valid = np.ones((4, 4), np.uint8)
    a = rot_affine(17.0, 1.05, 0.3, -0.6)
    ref = O.slopes_wfs(cube, pupil, 4, 6, valid, a, 1.3)
    got = O.slopes_wfs_repair(cube, np.ones((n, n), np.float32), pupil, 4, 6, valid, a, 1.3)
    assert np.array_equal(got, ref)
    _, c, r = O.repair_screen(cube[0], np.ones((n, n), np.float32), m, a)
    assert c.all() and not r.any()


@pytest.mark.parametrize("shift", [(0.0, 0.0), (2.0, -1.0), (0.37, -0.81)])
def test_constant_and_linear_phase_are_restored_exactly_up_to_the_mask_edge(shift):
    """A rectangular mask at least two pixels thick: every valid direction has both reference pixels, and
    2*P1 - P2 continues a linear phase exactly.  So the slopes of a MASKED tilt are the tilt in every subaperture
    that holds a core pixel -- while the unrepaired engine is wrong by tens of per cent along the edge
    ('phase values artificially collapse towards zero')."""
    n, nsub, npix = 48, 6, 6
    m = nsub * npix
    yy, xx = np.mgrid[0:n, 0:n].astype(np.float64)
    xs, ys = xx - (n - 1) / 2.0, yy - (n - 1) / 2.0
    mask = np.zeros((n, n), np.float32)
    mask[15:37, 19:41] = 1.0
    ta, tb = 0.25, -0.375
    cube = np.stack([np.full((n, n), 3.5), ta * xs + tb * ys]).astype(np.float32) * mask
    a = [1.0, 0.0, shift[0], 0.0, 1.0, shift[1]]
    pupil = np.ones((m, m), np.float32)
    valid = np.ones((nsub, nsub), np.uint8)
    phi_c, core, ring = O.repair_screen(cube[0], mask, m, a)
    assert ring.any() and np.allclose(phi_c[(core | ring) == 1], 3.5, rtol=0, atol=1e-12)
    assert (phi_c[(core | ring) == 0] == 0).all()
    phi_l, _, _ = O.repair_screen(cube[1], mask, m, a)
    ii, jj = np.mgrid[-1:m + 1, -1:m + 1].astype(np.float64)
    lin = ta * (jj - (m - 1) / 2.0 + shift[0]) + tb * (ii - (m - 1) / 2.0 + shift[1])
    sel = (core | ring) == 1
    assert np.allclose(phi_l[sel], lin[sel], rtol=0, atol=1e-12)
    s = O.slopes_wfs_repair(cube, mask, pupil, nsub, npix, valid, a)
    has_core = core[1:-1, 1:-1].reshape(nsub, npix, nsub, npix).sum(axis=(1, 3)).ravel() > 0
    assert has_core.sum() >= 16 and (~has_core).sum() >= 8
    nv = nsub * nsub
    assert np.allclose(s[0], 0.0, atol=1e-13)                                   # constant: no slope anywhere
    assert np.allclose(s[1, :nv][has_core], ta, rtol=0, atol=1e-12)
    assert np.allclose(s[1, nv:][has_core], tb, rtol=0, atol=1e-12)
    assert (s[1, :nv][~has_core] == 0).all() and (s[1, nv:][~has_core] == 0).all()   # no core pixel: slope 0 (R22)
    raw = O.slopes_wfs(cube, pupil, nsub, npix, valid, a)                       # the unrepaired engine
    assert np.abs(raw[1, :nv][has_core] - ta).max() > 0.1 * abs(ta)


def test_threshold_is_inclusive_and_is_the_value_given():
    """mu >= threshold (R19).  Under the identity map mu is the mask itself: float32 values just below and just
    above 0.999999, and a pixel exactly on a custom threshold of 0.5."""
    mask = np.zeros((7, 7), np.float32)
    mask[2:5, 2:5] = 1.0
    mask[3, 2] = np.float32(0.9999985)       # < 0.999999: not core
    mask[3, 4] = np.float32(0.9999995)       # >= 0.999999: core
    mask[2, 3] = 0.5
    g = np.arange(49, dtype=np.float32).reshape(7, 7)
    _, c, _ = O.repair_screen(g, mask, 5, IDENT)
    assert not c[3, 2] and c[3, 4] and not c[2, 3] and c.sum() == 7
    _, c, _ = O.repair_screen(g, mask, 5, IDENT, threshold=0.5)
    assert c[3, 2] and c[3, 4] and c[2, 3] and c.sum() == 9
    _, c, _ = O.repair_screen(g, mask, 5, IDENT, threshold=np.nextafter(0.5, 1.0))
    assert not c[2, 3]


def test_directions_that_leave_the_halo_grid_are_invalid():
    """A core that touches the border of the halo grid: pixels beyond it do not exist (R20), so a ring pixel
    in the corner region only uses the directions that stay inside."""
    mask = np.ones((7, 7), np.float32)
    mask[0, :] = 0.0                              # top halo row is not core; everything else is
    g = (np.arange(49, dtype=np.float32).reshape(7, 7)) ** 2
    phi, c, r = O.repair_screen(g, mask, 5, IDENT)
    assert r[0].all() and r.sum() == 7 and c[1:].all()
    # every ring pixel of row 0 has the single valid direction 'down': 2*g[1] - g[2]
    assert np.array_equal(phi[0], 2.0 * g[1].astype(np.float64) - g[2])


# ------------------------------------------------------------------------------- independent restatement
def _restated(phi, mu, thr):
    """The same three steps written with whole-array operations and scipy's dilation (default structuring
    element: the 4-neighbour cross)."""
    core = mu >= thr
    ring = ndi.binary_dilation(core) & ~core
    pc = np.where(core, phi, 0.0)
    pad = np.pad(pc, 2)
    cpad = np.pad(core, 2)
    n0, n1 = phi.shape
    num = np.zeros_like(phi)
    cnt = np.zeros_like(phi)
    for dy, dx in ((0, 1), (0, -1), (1, 0), (-1, 0)):
        p1 = pad[2 + dy:2 + dy + n0, 2 + dx:2 + dx + n1]
        p2 = pad[2 + 2 * dy:2 + 2 * dy + n0, 2 + 2 * dx:2 + 2 * dx + n1]
        c1 = cpad[2 + dy:2 + dy + n0, 2 + dx:2 + dx + n1]
        c2 = cpad[2 + 2 * dy:2 + 2 * dy + n0, 2 + 2 * dx:2 + 2 * dx + n1]
        num += np.where(c1, np.where(c2, 2.0 * p1 - p2, p1), 0.0)
        cnt += c1
    out = pc.copy()
    out[ring] = num[ring] / cnt[ring]
    return out, core, ring


@pytest.mark.parametrize("seed", [0, 1, 2, 3])
def test_independent_restatement_on_random_masks_under_rotation(seed):
    rng = np.random.default_rng(100 + seed)
    n, nsub, npix = 56, 5, 8
    m = nsub * npix
    # a blobby binary mask with holes and thin parts, and one with soft (fractional) edges
    blob = ndi.gaussian_filter(rng.normal(size=(n, n)), 3.0)
    mask = (blob > np.quantile(blob, 0.35)).astype(np.float32)
    if seed % 2:
        mask = np.clip(ndi.gaussian_filter(mask, 0.7) * 1.2, 0.0, 1.0).astype(np.float32)
    g = (rng.normal(size=(n, n)) * 2.0 + 1.0).astype(np.float32)
    a = rot_affine(rng.uniform(-180, 180), rng.uniform(0.9, 1.15), rng.uniform(-3, 3), rng.uniform(-3, 3))
    phi, core, ring = O.repair_screen(g, mask, m, a)
    exp, ecore, ering = _restated(O.resample(g, m, a, halo=True), O.resample(mask, m, a, halo=True), TAU)
    assert np.array_equal(core.astype(bool), ecore) and np.array_equal(ring.astype(bool), ering)
    assert ering.sum() > 50 and (~ecore & ~ering).sum() > 50
    assert np.allclose(phi, exp, rtol=0, atol=1e-12)
    # slopes: weights P*core, central differences of the repaired screen, zero where no core pixel
    pupil = rng.uniform(0.2, 1.0, (m, m)).astype(np.float32)
    valid = (rng.uniform(size=(nsub, nsub)) > 0.2).astype(np.uint8)
    s = O.slopes_wfs_repair(g[None], mask, pupil, nsub, npix, valid, a, scale=0.7)[0]
    dx = (exp[1:-1, 2:] - exp[1:-1, :-2]) / 2.0
    dy = (exp[2:, 1:-1] - exp[:-2, 1:-1]) / 2.0
    wgt = pupil.astype(np.float64) * ecore[1:-1, 1:-1]
    blk = lambda z: z.reshape(nsub, npix, nsub, npix).sum(axis=(1, 3))
    den = blk(wgt)
    with np.errstate(invalid="ignore", divide="ignore"):
        ex = np.where(den > 0, 0.7 * blk(wgt * dx) / den, 0.0)[valid == 1]
        ey = np.where(den > 0, 0.7 * blk(wgt * dy) / den, 0.0)[valid == 1]
    assert np.allclose(s, np.concatenate([ex, ey]), rtol=0, atol=1e-12)


def test_repair_recovers_the_slopes_of_a_smooth_mode_cut_by_a_round_pupil():
    """The purpose of the algorithm: a smooth mode that exists only inside a round pupil mask.
    Its repaired slopes agree with those of the uncut mode on every subaperture of the core to the accuracy of a
    linear extrapolation, where the unrepaired ones are off by a large factor at the edge."""
    n, nsub, npix = 96, 10, 8
    m = nsub * npix
    yy, xx = np.mgrid[0:n, 0:n].astype(np.float64)
    xs, ys = xx - (n - 1) / 2.0, yy - (n - 1) / 2.0
    mask = (np.hypot(xs, ys) <= 36.0).astype(np.float32)
    full = (np.sin(xs / 17.0) * np.cos(ys / 23.0) + 0.01 * xs).astype(np.float32)
    a = rot_affine(11.0, 1.02, 0.4, -0.3)
    pupil = np.ones((m, m), np.float32)
    valid = np.ones((nsub, nsub), np.uint8)
    _, core, _ = O.repair_screen(full, mask, m, a)
    w = core[1:-1, 1:-1].astype(np.float32)
    inside = w.reshape(nsub, npix, nsub, npix).sum(axis=(1, 3)).ravel() >= 8
    truth = O.slopes_wfs(full[None], w, nsub, npix, inside.reshape(nsub, nsub).astype(np.uint8), a)[0]
    rep = O.slopes_wfs_repair((full * mask)[None], mask, pupil, nsub, npix, valid, a)[0]
    raw = O.slopes_wfs((full * mask)[None], w, nsub, npix, inside.reshape(nsub, nsub).astype(np.uint8), a)[0]
    nv, ni = nsub * nsub, int(inside.sum())
    rep_in = np.concatenate([rep[:nv][inside], rep[nv:][inside]])
    scale = np.abs(truth).max()
    assert np.abs(rep_in - truth).max() < 0.02 * scale         # second-order error of the extrapolation only
    assert np.abs(raw - truth).max() > 0.5 * scale             # the collapse the paper describes
    assert ni >= 50
