/*
 * synim_oracle.c -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.
 *
 * A plain, slow, float64 CPU restatement of the synthetic Shack-Hartmann
 * interaction-matrix computation of SynIM (arxiv/paper_2606_07759), written from
 * the paper's prose (/root/reference/PAPER.md; the paper has no numbered
 * equations) under the readings R1..R13 listed in DESIGN.md.  Only tests/,
 * __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
 * call it.  It shares no code, header, table or helper with the CUDA path.
 *
 * What it computes, per (mode m, WFS w)  [one IM column in the metric's sense]:
 *
 *   1. composite affine, ONE matrix per WFS (sec. 2.1 "multiplied into a
 *      single composite matrix"): for every WFS pixel (i,j), i,j in {-1..M} (a one
 *      pixel halo so that central differences exist at the border, reading R5),
 *        x_w = j-(M-1)/2, y_w = i-(M-1)/2           (pixel centres, reading R2)
 *        x_s = a0 x_w + a1 y_w + a2,  y_s = a3 x_w + a4 y_w + a5     (reading R1)
 *        col = x_s+(Nx-1)/2, row = y_s+(Ny-1)/2
 *   2. single bilinear interpolation ("interpolating the high-resolution
 *      grid exactly once", :63/:67 "bilinear"), zero outside the grid (reading R4):
 *        phi[i][j] = (1-fy)((1-fx) g(r0,c0) + fx g(r0,c0+1)) + fy((1-fx) g(r0+1,c0) + fx g(r0+1,c0+1))
 *   3. finite central differences at every pixel (sec. 2.2):
 *        Dx = (phi[i][j+1]-phi[i][j-1])/2,  Dy = (phi[i+1][j]-phi[i-1][j])/2
 *   4. spatial average over the subaperture, weighted by the pupil
 *      weights P given in the WFS frame (reading R7):
 *        s_x = scale * sum_S P Dx / sum_S P          (same for y)
 *   5. row order inside a column: all x slopes of the valid subapertures in row-major
 *      (a,b) order, then all y slopes (reading R9).
 *
 * SYNIM_ORACLE_GTILT replaces 3-4 by the boundary-driven telescoping sum (PAPER.md:61
 * "evaluates the phase difference strictly at the subaperture edges", reading R13):
 * pixel valid iff P >= 0.5; for each pixel row of S with first/last valid columns
 * jf < jl: num += phi[row][jl]-phi[row][jf], den += jl-jf; s_x = scale*num/den.
 *
 * EDGE REPAIR (sec. 2.3 "_repair_interpolated_phase"; readings R18-R22 of DESIGN.md), for modes
 * that exist only inside a mask given in the SOURCE frame (a DM or pupil mask): see repair_interpolated_phase()
 * and slopes_nd_core() below.  Pins (tests/test_oracle_repair_pins.py): an all-ones mask changes nothing; a constant
 * and a linear phase are restored exactly on the ring, so the slopes of a masked tilt are the tilt right up to the
 * edge; a hand-computed 7x7 example (one valid direction with one reference pixel, two directions of different
 * kinds); the threshold; an independent restatement with scipy.ndimage.binary_dilation on random masks.
 *
 * Pins (tests/test_oracle_pins.py): pure tilt -> constant slopes A^T(a,b); quadratic ->
 * linear slopes; identity / integer shift / 90-degree rotations reproduce the input
 * bit for bit; linearity; telescoping identity on full subapertures; equality with
 * scipy.ndimage.affine_transform(order=1, mode='grid-constant') and
 * torch.grid_sample(bilinear, zeros, align_corners=True); a scalar pure-Python brute
 * force on tiny grids; the explicit sparse operator assembled from impulse responses.
 * The composition helper is pinned by applying the individual maps to points one
 * after another; its sign / order conventions (R1) and the row order (R9) are
 * conventions and therefore "parity unpinned".
 *
 * No blocking, fusion, bbox skipping, tiling or telescoping: full (M+2)^2 grid per
 * (mode, WFS).  OpenMP only distributes whole modes over host cores.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define SYNIM_ORACLE_ND 0
#define SYNIM_ORACLE_GTILT 1

/* Step 1+2 for one mode: phi on the halo grid, (M+2) x (M+2), phi[(i+1)*(M+2)+(j+1)]. */
static void resample_once(const float *g, int ny, int nx, int M, const double a[6], double *phi)
{
    const double cw = (M - 1) / 2.0, cx = (nx - 1) / 2.0, cy = (ny - 1) / 2.0;
    const int P = M + 2;
    for (int i = -1; i <= M; ++i) {
        for (int j = -1; j <= M; ++j) {
            const double xw = j - cw, yw = i - cw;
            const double xs = a[0] * xw + a[1] * yw + a[2];
            const double ys = a[3] * xw + a[4] * yw + a[5];
            const double col = xs + cx, row = ys + cy;
            const double fc = floor(col), fr = floor(row);
            const double fx = col - fc, fy = row - fr;
            double v00 = 0.0, v01 = 0.0, v10 = 0.0, v11 = 0.0;
            /* far outside: every neighbour is out of range */
            if (fc >= -1.0 && fc <= (double)nx && fr >= -1.0 && fr <= (double)ny) {
                const long c0 = (long)fc, r0 = (long)fr;
                if (r0 >= 0 && r0 < ny) {
                    if (c0 >= 0 && c0 < nx) v00 = g[r0 * (long)nx + c0];
                    if (c0 + 1 >= 0 && c0 + 1 < nx) v01 = g[r0 * (long)nx + c0 + 1];
                }
                if (r0 + 1 >= 0 && r0 + 1 < ny) {
                    if (c0 >= 0 && c0 < nx) v10 = g[(r0 + 1) * (long)nx + c0];
                    if (c0 + 1 >= 0 && c0 + 1 < nx) v11 = g[(r0 + 1) * (long)nx + c0 + 1];
                }
            }
            phi[(long)(i + 1) * P + (j + 1)] =
                (1.0 - fy) * ((1.0 - fx) * v00 + fx * v01) + fy * ((1.0 - fx) * v10 + fx * v11);
        }
    }
}

#define PHI(i, j) phi[(long)((i) + 1) * P + ((j) + 1)]

/* Steps 3-4, numerical derivative. */
static void slopes_nd(const double *phi, int M, int n_subap, int n_pix, const float *pupil,
                      const uint8_t *valid, double scale, double *sx, double *sy)
{
    const int P = M + 2;
    int k = 0;
    for (int a = 0; a < n_subap; ++a) {
        for (int b = 0; b < n_subap; ++b) {
            if (!valid[a * n_subap + b]) continue;
            double w = 0.0, ax = 0.0, ay = 0.0;
            for (int i = a * n_pix; i < (a + 1) * n_pix; ++i) {
                for (int j = b * n_pix; j < (b + 1) * n_pix; ++j) {
                    const double p = pupil[(long)i * M + j];
                    const double dx = (PHI(i, j + 1) - PHI(i, j - 1)) / 2.0;
                    const double dy = (PHI(i + 1, j) - PHI(i - 1, j)) / 2.0;
                    w += p;
                    ax += p * dx;
                    ay += p * dy;
                }
            }
            sx[k] = scale * ax / w;
            sy[k] = scale * ay / w;
            ++k;
        }
    }
}

/* Steps 3-4 replaced by the G-tilt telescoping sum. */
static void slopes_gtilt(const double *phi, int M, int n_subap, int n_pix, const float *pupil,
                         const uint8_t *valid, double scale, double *sx, double *sy)
{
    const int P = M + 2;
    int k = 0;
    for (int a = 0; a < n_subap; ++a) {
        for (int b = 0; b < n_subap; ++b) {
            if (!valid[a * n_subap + b]) continue;
            const int i0 = a * n_pix, j0 = b * n_pix;
            double num = 0.0, den = 0.0;
            for (int i = i0; i < i0 + n_pix; ++i) {
                int jf = -1, jl = -1;
                for (int j = j0; j < j0 + n_pix; ++j)
                    if (pupil[(long)i * M + j] >= 0.5f) { if (jf < 0) jf = j; jl = j; }
                if (jf >= 0 && jl > jf) { num += PHI(i, jl) - PHI(i, jf); den += jl - jf; }
            }
            sx[k] = den > 0.0 ? scale * num / den : 0.0;
            num = 0.0; den = 0.0;
            for (int j = j0; j < j0 + n_pix; ++j) {
                int f = -1, l = -1;
                for (int i = i0; i < i0 + n_pix; ++i)
                    if (pupil[(long)i * M + j] >= 0.5f) { if (f < 0) f = i; l = i; }
                if (f >= 0 && l > f) { num += PHI(l, j) - PHI(f, j); den += l - f; }
            }
            sy[k] = den > 0.0 ? scale * num / den : 0.0;
            ++k;
        }
    }
}

/*
 * Edge repair.  In: phi = the interpolated mode, mu = the mask interpolated through the SAME
 * composite transform with the same bilinear rule (R18), both on the halo grid (M+2)^2.  Steps, in the paper's order:
 *   1. strict binarisation and clearing: core = (mu >= threshold), "e.g. 0.999999", compared in
 *      float64 (R19); phi is set to 0 outside the core;
 *   2. edge identification: ring = (binary dilation of core) and not core, with the 4-neighbour cross as
 *      structuring element, one iteration (R20); pixels beyond the halo grid are not core;
 *   3. omnidirectional extrapolation: for every ring pixel q and each of the four cardinal directions
 *      d: P1 = q+d, P2 = q+2d ("consecutive reference pixels"); the direction is valid iff P1 is core; its estimate is
 *      2*phi[P1] - phi[P2] if P2 is core too, else phi[P1]; phi[q] = sum of the estimates / number of valid
 *      directions (R21).
 * Out: phi repaired in place (core: unchanged; ring: restored; elsewhere 0), core[] (1/0), ring[] (1/0; may be NULL).
 */
static void repair_interpolated_phase(double *phi, const double *mu, int M, double threshold, uint8_t *core, uint8_t *ring)
{
    const int P = M + 2;
    const long n = (long)P * P;
    for (long q = 0; q < n; ++q) {
        core[q] = mu[q] >= threshold ? 1 : 0;
        if (!core[q]) phi[q] = 0.0;
    }
    static const int di[4] = {0, 0, 1, -1}, dj[4] = {1, -1, 0, 0};
    for (int i = 0; i < P; ++i) {
        for (int j = 0; j < P; ++j) {
            const long q = (long)i * P + j;
            if (ring) ring[q] = 0;
            if (core[q]) continue;
            double sum = 0.0;
            int n_dir = 0;
            for (int d = 0; d < 4; ++d) {
                const int i1 = i + di[d], j1 = j + dj[d], i2 = i + 2 * di[d], j2 = j + 2 * dj[d];
                if (i1 < 0 || i1 >= P || j1 < 0 || j1 >= P || !core[(long)i1 * P + j1]) continue;
                const double p1 = phi[(long)i1 * P + j1];
                if (i2 >= 0 && i2 < P && j2 >= 0 && j2 < P && core[(long)i2 * P + j2]) sum += 2.0 * p1 - phi[(long)i2 * P + j2];
                else sum += p1;
                ++n_dir;
            }
            if (n_dir > 0) {          /* q is a 4-neighbour of the core: a ring pixel */
                if (ring) ring[q] = 1;
                phi[q] = sum / n_dir;  /* (reads core pixels only, which this loop never writes) */
            }
        }
    }
}

/* Steps 3-4 after edge repair (R22): central differences of the repaired screen, averaged over the CORE pixels of
 * the subaperture with the weights P (a pixel outside the core has a stencil that reaches past the ring: no valid
 * derivative).  A valid subaperture without any weighted core pixel gets slope 0. */
static void slopes_nd_core(const double *phi, const uint8_t *core, int M, int n_subap, int n_pix, const float *pupil,
                           const uint8_t *valid, double scale, double *sx, double *sy)
{
    const int P = M + 2;
    int k = 0;
    for (int a = 0; a < n_subap; ++a) {
        for (int b = 0; b < n_subap; ++b) {
            if (!valid[a * n_subap + b]) continue;
            double w = 0.0, ax = 0.0, ay = 0.0;
            for (int i = a * n_pix; i < (a + 1) * n_pix; ++i) {
                for (int j = b * n_pix; j < (b + 1) * n_pix; ++j) {
                    if (!core[(long)(i + 1) * P + (j + 1)]) continue;
                    const double p = pupil[(long)i * M + j];
                    const double dx = (PHI(i, j + 1) - PHI(i, j - 1)) / 2.0;
                    const double dy = (PHI(i + 1, j) - PHI(i - 1, j)) / 2.0;
                    w += p;
                    ax += p * dx;
                    ay += p * dy;
                }
            }
            sx[k] = w > 0.0 ? scale * ax / w : 0.0;
            sy[k] = w > 0.0 ? scale * ay / w : 0.0;
            ++k;
        }
    }
}

/*
 * Slopes of the selected modes for ONE wavefront sensor.
 *   cube      float32 [n_modes_total][ny][nx]
 *   mode_idx  n_sel indices into the cube, or NULL for 0..n_sel-1
 *   pupil     float32 [M][M], M = n_subap*n_pix, weights in the WFS frame
 *   valid     uint8 [n_subap][n_subap]
 *   a         composite 2x3 matrix (output -> input, centred pixel coordinates)
 *   out       float64 [n_sel][2*n_valid]: per mode, x slopes then y slopes
 *   n_threads <=0: all host cores (OpenMP over modes)
 * Returns 0, or -1 on bad arguments / a valid subaperture of zero weight, -2 on OOM.
 */
int synim_oracle_wfs(const float *cube, int64_t n_modes_total, const int32_t *mode_idx, int32_t n_sel,
                     int32_t ny, int32_t nx, const float *pupil, int32_t n_subap, int32_t n_pix,
                     const uint8_t *valid, const double *a, double scale, int32_t mode, int32_t n_threads,
                     double *out)
{
    if (!cube || !pupil || !valid || !a || !out || ny <= 0 || nx <= 0 || n_subap <= 0 || n_pix <= 0) return -1;
    if (mode != SYNIM_ORACLE_ND && mode != SYNIM_ORACLE_GTILT) return -1;
    const int M = n_subap * n_pix;
    int n_valid = 0;
    for (int s = 0; s < n_subap * n_subap; ++s) n_valid += valid[s] ? 1 : 0;
    if (mode == SYNIM_ORACLE_ND) {
        for (int sa = 0; sa < n_subap; ++sa)
            for (int sb = 0; sb < n_subap; ++sb) {
                if (!valid[sa * n_subap + sb]) continue;
                double w = 0.0;
                for (int i = sa * n_pix; i < (sa + 1) * n_pix; ++i)
                    for (int j = sb * n_pix; j < (sb + 1) * n_pix; ++j) w += pupil[(long)i * M + j];
                if (!(w > 0.0)) return -1;
            }
    }
    int err = 0;
#ifdef _OPENMP
    if (n_threads > 0) omp_set_num_threads(n_threads);
    else omp_set_num_threads(omp_get_num_procs());
#endif
#pragma omp parallel
    {
        double *phi = (double *)malloc(sizeof(double) * (size_t)(M + 2) * (size_t)(M + 2));
        if (!phi) {
#pragma omp atomic write
            err = -2;
        }
#pragma omp for schedule(dynamic, 1)
        for (int s = 0; s < n_sel; ++s) {
            if (!phi) continue;
            const int64_t m = mode_idx ? mode_idx[s] : s;
            if (m < 0 || m >= n_modes_total) {
#pragma omp atomic write
                err = -1;
                continue;
            }
            const float *g = cube + (size_t)m * (size_t)ny * (size_t)nx;
            double *sx = out + (size_t)s * 2 * (size_t)n_valid;
            double *sy = sx + n_valid;
            resample_once(g, ny, nx, M, a, phi);
            if (mode == SYNIM_ORACLE_ND) slopes_nd(phi, M, n_subap, n_pix, pupil, valid, scale, sx, sy);
            else slopes_gtilt(phi, M, n_subap, n_pix, pupil, valid, scale, sx, sy);
        }
        free(phi);
    }
    return err;
}

/*
 * Edge-repaired slopes of the selected modes for ONE wavefront sensor: as synim_oracle_wfs in
 * numerical-derivative mode, with the mode's screen repaired before it is differentiated.
 *   mask       float32 [ny][nx], the mask of the modes in the SOURCE frame (values in [0, 1])
 *   threshold  the strict-binarisation threshold (the paper's example: 0.999999)
 * Returns 0, -1 on bad arguments, -2 on OOM.
 */
int synim_oracle_wfs_repair(const float *cube, int64_t n_modes_total, const int32_t *mode_idx, int32_t n_sel,
                            int32_t ny, int32_t nx, const float *mask, double threshold, const float *pupil,
                            int32_t n_subap, int32_t n_pix, const uint8_t *valid, const double *a, double scale,
                            int32_t n_threads, double *out)
{
    if (!cube || !mask || !pupil || !valid || !a || !out || ny <= 0 || nx <= 0 || n_subap <= 0 || n_pix <= 0) return -1;
    const int M = n_subap * n_pix;
    const size_t np = (size_t)(M + 2) * (size_t)(M + 2);
    int n_valid = 0;
    for (int s = 0; s < n_subap * n_subap; ++s) n_valid += valid[s] ? 1 : 0;
    double *mu = (double *)malloc(sizeof(double) * np);
    if (!mu) return -2;
    resample_once(mask, ny, nx, M, a, mu);   /* the mask goes through the same transform, once (R18) */
    int err = 0;
#ifdef _OPENMP
    if (n_threads > 0) omp_set_num_threads(n_threads);
    else omp_set_num_threads(omp_get_num_procs());
#endif
#pragma omp parallel
    {
        double *phi = (double *)malloc(sizeof(double) * np);
        uint8_t *core = (uint8_t *)malloc(np);
        if (!phi || !core) {
#pragma omp atomic write
            err = -2;
        }
#pragma omp for schedule(dynamic, 1)
        for (int s = 0; s < n_sel; ++s) {
            if (!phi || !core) continue;
            const int64_t m = mode_idx ? mode_idx[s] : s;
            if (m < 0 || m >= n_modes_total) {
#pragma omp atomic write
                err = -1;
                continue;
            }
            double *sx = out + (size_t)s * 2 * (size_t)n_valid;
            resample_once(cube + (size_t)m * (size_t)ny * (size_t)nx, ny, nx, M, a, phi);
            repair_interpolated_phase(phi, mu, M, threshold, core, NULL);
            slopes_nd_core(phi, core, M, n_subap, n_pix, pupil, valid, scale, sx, sx + n_valid);
        }
        free(phi);
        free(core);
    }
    free(mu);
    return err;
}

/* For the pins: the repaired screen of one mode on the halo grid, with its core and ring maps
 * (all [(M+2)][(M+2)], pixel (i, j) at [(i+1)][(j+1)]). */
int synim_oracle_repair_screen(const float *g, const float *mask, int32_t ny, int32_t nx, int32_t M, const double *a,
                               double threshold, double *phi_out, uint8_t *core_out, uint8_t *ring_out)
{
    if (!g || !mask || !a || !phi_out || !core_out || !ring_out || M <= 0) return -1;
    const size_t np = (size_t)(M + 2) * (size_t)(M + 2);
    double *mu = (double *)malloc(sizeof(double) * np);
    if (!mu) return -2;
    resample_once(mask, ny, nx, M, a, mu);
    resample_once(g, ny, nx, M, a, phi_out);
    repair_interpolated_phase(phi_out, mu, M, threshold, core_out, ring_out);
    free(mu);
    return 0;
}

/* Steps 1-2 only, for the pins: the resampled screen of one mode, either on the M x M grid
 * (halo = 0) or on the (M+2) x (M+2) halo grid i,j in {-1..M} (halo = 1). */
int synim_oracle_resample(const float *g, int32_t ny, int32_t nx, int32_t M, const double *a, int32_t halo,
                          double *out)
{
    if (!g || !a || !out || M <= 0) return -1;
    const int P = M + 2;
    double *phi = (double *)malloc(sizeof(double) * (size_t)P * (size_t)P);
    if (!phi) return -2;
    resample_once(g, ny, nx, M, a, phi);
    if (halo) memcpy(out, phi, sizeof(double) * (size_t)P * (size_t)P);
    else
        for (int i = 0; i < M; ++i)
            for (int j = 0; j < M; ++j) out[(long)i * M + j] = PHI(i, j);
    free(phi);
    return 0;
}

/*
 * Composite matrix from physical parameters ("altitude-dependent perspective
 * scalings", :49 DM (shift, rotation, magnification) and WFS (incl. anamorphosis) matrices
 * "mathematically multiplied into a single composite matrix"; readings R1, R11, R12).
 * p[15] in the field order of workloads.PHYSICAL_FIELDS.  Output -> input chain:
 *   u1 = s*x_w - d_w                         WFS pixel -> pupil plane, remove WFS shift
 *   u2 = diag(1/m_x,1/m_y) R(-th_w) u1       undo WFS rotation / (anamorphic) magnification
 *   u3 = kappa*u2 + f                        propagate to the DM's conjugate altitude:
 *                                            kappa = 1-h/H (1 for H=inf), f = h*theta*(cos az, sin az)/pitch
 *   x_s = (1/m_d) R(-th_d) (u3 - d_d)        into the DM's own (misregistered) frame
 * R(-t) = [[cos t, sin t], [-sin t, cos t]].
 */
int synim_oracle_compose(const double *p, double *a)
{
    const double PI = 3.14159265358979323846;
    const double dwx = p[0], dwy = p[1], thw = p[2] * PI / 180.0, mx = p[3], my = p[4];
    const double ddx = p[5], ddy = p[6], thd = p[7] * PI / 180.0, md = p[8];
    const double h = p[9], H = p[10], theta = p[11] * PI / (180.0 * 3600.0), az = p[12] * PI / 180.0;
    const double pitch = p[13], s = p[14];
    if (!(mx != 0.0) || !(my != 0.0) || !(md != 0.0) || !(pitch > 0.0)) return -1;
    const double kappa = isinf(H) ? 1.0 : 1.0 - h / H;
    const double fx = h * theta * cos(az) / pitch, fy = h * theta * sin(az) / pitch;
    /* B = diag(1/m) R(-th_w) */
    const double cw = cos(thw), sw = sin(thw);
    const double B00 = cw / mx, B01 = sw / mx, B10 = -sw / my, B11 = cw / my;
    /* u3 = kappa*B*(s*x - d_w) + f */
    const double C00 = kappa * B00 * s, C01 = kappa * B01 * s, C10 = kappa * B10 * s, C11 = kappa * B11 * s;
    const double c0 = -kappa * (B00 * dwx + B01 * dwy) + fx - ddx;
    const double c1 = -kappa * (B10 * dwx + B11 * dwy) + fy - ddy;
    /* x_s = (1/m_d) R(-th_d) (C x + c) */
    const double cd = cos(thd) / md, sd = sin(thd) / md;
    a[0] = cd * C00 + sd * C10;  a[1] = cd * C01 + sd * C11;  a[2] = cd * c0 + sd * c1;
    a[3] = -sd * C00 + cd * C10; a[4] = -sd * C01 + cd * C11; a[5] = -sd * c0 + cd * c1;
    return 0;
}

int synim_oracle_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_num_procs();
#else
    return 1;
#endif
}
