/*
 * synim.h -- C ABI of the B200-native synthetic Shack-Hartmann interaction-matrix engine.
 *
 * What the library computes (SynIM, arxiv/paper_2606_07759; citations are lines of
 * /root/reference/PAPER.md, "R<n>" are the readings listed in DESIGN.md):
 *
 *   for every (mode m, wavefront sensor w)            -- one IM column in the metric's sense
 *     1. ONE composite affine transform per WFS maps every WFS pixel to the DM / meta-pupil grid
 *        (sec. 2.1: DM and WFS matrices "multiplied into a single composite matrix";
 *        :47 altitude-dependent perspective scaling),
 *     2. the influence function is bilinearly interpolated exactly once,
 *        zero outside the grid (R4),
 *     3. finite central differences at every WFS pixel (sec. 2.2),
 *     4. spatial average over each valid subaperture, weighted by the pupil weights (PAPER.md:61,
 *        :116), times the caller's slope scale,
 *   assembled into IM[rows][n_modes], rows = 2 * sum_w n_valid_w.
 *
 * Conventions
 *   - Pixel k of an N-pixel axis sits at k-(N-1)/2 (R2).  x = column direction, y = row direction.
 *   - The composite matrix maps WFS pixel coordinates (x_w, y_w) to source-grid coordinates:
 *       x_s = a[0]*x_w + a[1]*y_w + a[2],   y_s = a[3]*x_w + a[4]*y_w + a[5]        (R1)
 *   - Row order inside a column: WFS 0..n_wfs-1; inside a WFS all x slopes of the valid
 *     subapertures in row-major (a,b) order, then all y slopes (R9).
 *   - The IM is column-major: element (r, m) is d_out[m*ld + r]  (float32).
 *   - "HOST" / "DEVICE" say where a pointer lives.  The caller owns every buffer it passes in;
 *     HOST arrays are consumed during the call and may be freed on return.  DEVICE buffers must
 *     stay valid until the work enqueued on `stream` has finished.  The library owns only the
 *     geometry object and its small internal device buffers.
 *   - `stream` is a cudaStream_t passed as void* (NULL = the legacy default stream).  Calls
 *     enqueue work and return without synchronising unless stated otherwise.
 *   - Every entry point returns a synim_status; nothing throws or aborts across the ABI.  There is
 *     NO CPU fallback: without a CUDA device of compute capability 10.x the compute entry points
 *     return SYNIM_ERR_UNSUPPORTED_DEVICE / SYNIM_ERR_CUDA.  synim_last_error() gives the text
 *     of the calling thread's last failure.
 */
#ifndef SYNIM_H_
#define SYNIM_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define SYNIM_VERSION_MAJOR 0
#define SYNIM_VERSION_MINOR 3

typedef struct synim_geometry synim_geometry; /* opaque, library-owned */

typedef enum {
    SYNIM_OK = 0,
    SYNIM_ERR_INVALID_ARG = -1,        /* NULL pointer, non-positive size, ld < rows, singular matrix ... */
    SYNIM_ERR_ALIGNMENT = -2,          /* cube pointer not 16-byte aligned or nx % 4 != 0 (TMA) */
    SYNIM_ERR_EMPTY_SUBAP = -3,        /* a subaperture flagged valid has zero summed pupil weight */
    SYNIM_ERR_UNSUPPORTED_DEVICE = -4, /* current device is not compute capability 10.x */
    SYNIM_ERR_OUT_OF_MEMORY = -5,
    SYNIM_ERR_CUDA = -6,               /* any other CUDA runtime / driver failure */
    SYNIM_ERR_UNSUPPORTED = -7         /* edge repair with the G-tilt estimator; cuBLAS / cuSOLVER not loadable */
} synim_status;

/* Slope estimator.  ND = finite central differences averaged over the subaperture
 * (the paper's engine).  GTILT = boundary-driven telescoping sum: the first/last valid pixel
 * (P >= 0.5) of every pixel row / column of the subaperture (R13). */
typedef enum { SYNIM_SLOPES_ND = 0, SYNIM_SLOPES_GTILT = 1 } synim_slope_mode;

/* One Shack-Hartmann sensor's static description.  M = n_subap*n_pix WFS pixels per side;
 * subaperture (a,b) owns pixels i in [a*n_pix,(a+1)*n_pix), j in [b*n_pix,(b+1)*n_pix). */
typedef struct {
    int32_t n_subap;
    int32_t n_pix;
    const uint8_t *valid_mask;   /* HOST  [n_subap][n_subap] row-major, non-zero = valid (R10) */
    const float *d_pupil;        /* DEVICE [M][M] row-major non-negative weights P in the WFS frame (R7) */
} synim_wfs_grid;

/* Per-call geometry of one sensor: the composite output->input matrix in centred pixel
 * coordinates (see Conventions) and the factor every slope of this sensor is multiplied by (R8). */
typedef struct {
    double a[6];
    double slope_scale;
} synim_wfs_affine;

/* Physical parameters the composite matrix is built from (R1, R11, R12).
 * Lengths in source-grid pixels unless stated; angles as named.  Chain, WFS pixel -> source grid:
 *   u1 = wfs_pitch_src_px * x_w - (shift_x, shift_y)
 *   u2 = diag(1/mag_x, 1/mag_y) * R(-rot_deg) * u1
 *   u3 = kappa * u2 + f,   kappa = 1 - dm_height_m/gs_range_m (1 if gs_range_m is +inf),
 *                          f = dm_height_m * theta * (cos az, sin az) / src_pixel_pitch_m
 *   x_s = (1/dm_mag) * R(-dm_rot_deg) * (u3 - (dm_shift_x, dm_shift_y))
 * with R(-t) = [[cos t, sin t], [-sin t, cos t]]. */
typedef struct {
    double shift_x, shift_y, rot_deg, mag_x, mag_y;
    double dm_shift_x, dm_shift_y, dm_rot_deg, dm_mag;
    double dm_height_m, gs_range_m, gs_theta_arcsec, gs_azimuth_deg, src_pixel_pitch_m;
    double wfs_pitch_src_px;
} synim_wfs_physical;

/* Pure host helper (no CUDA): compose the single matrix of PAPER.md:49 from physical parameters.
 * out->slope_scale is set to 1.  SYNIM_ERR_INVALID_ARG on NULL, zero magnification or pitch <= 0. */
synim_status synim_compose_affine(const synim_wfs_physical *phys, synim_wfs_affine *out);

/* Build the static geometry for n_wfs sensors looking at an ny x nx source grid (S0 of SURVEY.md
 * sec. 8(a)): per sensor the valid-subaperture row map, the per-pixel reduction weights
 * 0.5*P/W_S (W_S = summed weight of the pixel's subaperture, 0 for invalid ones) and the row offsets
 * of the sensor inside a column.  Runs small kernels on `stream` and SYNCHRONISES it once to
 * report SYNIM_ERR_EMPTY_SUBAP.  grids[w].d_pupil is only read during this call.
 * Requirements: 1 <= n_wfs <= 64, n_subap >= 1, n_pix >= 1, nx % 4 == 0. */
synim_status synim_create_geometry(int32_t ny, int32_t nx, int32_t n_wfs, const synim_wfs_grid *grids,
                                   void *stream, synim_geometry **out);

/* rows of the IM = 2 * sum_w n_valid_w; -1 on NULL. */
int64_t synim_num_rows(const synim_geometry *geom);
/* number of valid subapertures of sensor w, and the row where its x slopes start; -1 on error. */
int64_t synim_num_valid(const synim_geometry *geom, int32_t wfs);
int64_t synim_row_offset(const synim_geometry *geom, int32_t wfs);

/* The hot path (S1-S4): all (mode, WFS) pairs, fused coordinate generation, shared-memory gather of
 * TMA-staged influence-function tiles, central differences, subaperture reduction and the
 * column-major store including the zeros.
 *   d_influence  DEVICE float32 [n_modes][ny][nx], 16-byte aligned
 *   d_bbox       DEVICE int32 [n_modes][4] = (x0,y0,x1,y1) inclusive extent outside which the mode is
 *                exactly zero (x1 < x0: the mode is identically zero), or NULL = dense modes.
 *                A bbox that leaves out non-zero samples gives wrong results (not checked).
 *   d_diag       DEVICE int32 [n_modes][4] = (min x+y, max x+y, min x-y, max x-y) over the mode's non-zero
 *                pixels, or NULL.  With the bbox this is the support's bounding octagon: under a rotated
 *                sensor the footprint of a round influence function is then its own size, not that of
 *                its rotated bounding box.  Only ever narrows what is sampled (same "not checked" rule);
 *                requires d_bbox.  16-byte aligned.
 *   bbox_max_w/h HOST upper bounds of x1-x0+1 / y1-y0+1 over all modes, used only to size the
 *                shared-memory tiles (<= 0: unknown).  Wrong bounds cost speed, never correctness.
 *   affine       HOST [n_wfs]
 *   mode         SYNIM_SLOPES_ND (the paper's engine) or SYNIM_SLOPES_GTILT (comparison estimator: same
 *                kernel, the slopes are sums of phi weighted by the G-tilt coefficient maps built at
 *                synim_create_geometry); anything else is INVALID_ARG
 *   d_out        DEVICE float32, column-major, ld >= synim_num_rows(); every element of rows
 *                [0, num_rows) of columns [0, n_modes) is written (padding rows are left untouched)
 *                n_modes == 0, or a geometry without any valid subaperture (num_rows == 0), is a no-op that
 *                returns SYNIM_OK whatever the buffers are
 * Errors: INVALID_ARG (NULL, n_modes < 0, ld < rows, singular affine), ALIGNMENT, CUDA. */
synim_status synim_interaction_matrix(const synim_geometry *geom, const float *d_influence, int32_t n_modes,
                                      const int32_t *d_bbox, const int32_t *d_diag, int32_t bbox_max_w,
                                      int32_t bbox_max_h,
                                      const synim_wfs_affine *affine, synim_slope_mode mode, float *d_out,
                                      int64_t ld, void *stream);

/* The same hot path with the paper's EDGE REPAIR (sec. 2.3, "_repair_interpolated_phase"), for modes
 * that exist only inside a mask given in the SOURCE frame (a DM or pupil mask): their interpolated screen collapses
 * towards zero along the mask's edge and would corrupt the derivative there.  Per call and sensor (DESIGN.md readings
 * R18-R22):
 *   1. d_mask goes through the same composite transform and bilinear rule as the modes (in float64); the strict core
 *      is mu >= threshold (the paper's example: 0.999999), and the screen is cleared outside it;
 *   2. the ring is the 4-neighbour dilation of the core minus the core;
 *   3. a ring pixel becomes the normalised average, over the cardinal directions whose neighbour P1 is core, of
 *      2*P1 - P2 (P2, the next pixel, core too) or P1;
 *   then central differences of the repaired screen, averaged over the CORE pixels of each valid subaperture with the
 *   weights P (a valid subaperture without a weighted core pixel gets slope 0).
 * Numerical-derivative engine only.  Everything runs on `stream`: three small set-up kernels per sensor, then the fused
 * kernel (the ring is restored inside it, from extra samples of the staged tile -- the repaired screen is never stored).
 *   d_mask     DEVICE float32 [ny][nx], values in [0, 1]
 *   threshold  in (0, 1]
 * All other arguments, the output layout and the errors as for synim_interaction_matrix. */
synim_status synim_interaction_matrix_repaired(const synim_geometry *geom, const float *d_influence, int32_t n_modes,
                                               const int32_t *d_bbox, const int32_t *d_diag, int32_t bbox_max_w,
                                               int32_t bbox_max_h, const synim_wfs_affine *affine, const float *d_mask,
                                               double threshold, float *d_out, int64_t ld, void *stream);

/* Tight non-zero extent of every mode of a cube (DEVICE in, DEVICE out int32 [n_modes][4]);
 * an all-zero mode gets (0,0,-1,-1).  d_diag (DEVICE int32 [n_modes][4], or NULL) receives the
 * diagonal extents described above; an all-zero mode gets (0,-1,0,-1).  Asynchronous. */
synim_status synim_compute_bboxes(const float *d_influence, int32_t n_modes, int32_t ny, int32_t nx,
                                  int32_t *d_bbox, int32_t *d_diag, void *stream);
/* Largest bbox width / height (HOST out); synchronises `stream`. */
synim_status synim_bbox_extent(const int32_t *d_bbox, int32_t n_modes, int32_t *max_w, int32_t *max_h,
                               void *stream);

/* One-shot form with north_star's argument list (BASELINE.json; "a flat convenience wrapper ... may
 * wrap create -> compute -> destroy"): influence cube, per-sensor pupil mask + subaperture grid + valid mask (grids),
 * per-sensor composite matrices (affine), out IM [2 * sum_w n_valid_w][n_modes] column-major.  All buffers DEVICE except
 * grids[w].valid_mask and affine (HOST), exactly as in the calls it wraps:
 *   synim_create_geometry -> (compact != 0: synim_compute_bboxes + synim_bbox_extent, so that empty tiles are skipped;
 *   compact == 0: dense modes) -> synim_interaction_matrix -> synim_destroy.
 * ld >= 2 * sum_w n_valid_w, which the caller derives from its own valid masks; rows_out (may be NULL) receives it.
 * The supports live in a stream-ordered allocation of 32 * n_modes bytes for the duration of the call.  SYNCHRONISES the
 * device before returning (the geometry it built is freed).  For repeated use keep a geometry and call the pieces. */
synim_status synim_interaction_matrix_flat(const float *d_influence, int32_t n_modes, int32_t ny, int32_t nx, int32_t n_wfs,
                                           const synim_wfs_grid *grids, const synim_wfs_affine *affine, int32_t compact,
                                           synim_slope_mode mode, float *d_out, int64_t ld, int64_t *rows_out, void *stream);

/* Convenience wrapper with HOST buffers, for one-shot use and end-to-end timing: brings the cube to
 * the device, runs synim_interaction_matrix, copies the IM back and synchronises.  h_out is column-major
 * with ld = synim_num_rows().  With h_bbox (HOST int32 [n_modes][4], every bbox inside the grid, else
 * INVALID_ARG) only the supports cross the bus: each mode's bbox plus the ring of zeros the kernel stages
 * with it is packed into a pinned buffer of [n_modes][max_h + 2][roundup4(max_w + 5)] floats (host
 * threads), copied, and the kernel reads the packed cube through per-mode origins.  With h_bbox == NULL
 * (dense modes) the whole cube is copied.  The modes are processed in chunks whose packing, copies and kernels
 * overlap (see synim_dictionary_host).  Pinned h_influence / h_out make the copies asynchronous but are not required. */
synim_status synim_interaction_matrix_host(const synim_geometry *geom, const float *h_influence, int32_t n_modes,
                                           const int32_t *h_bbox, const synim_wfs_affine *affine,
                                           synim_slope_mode mode, float *h_out, void *stream);

/* One component of a multi-layer dictionary (sec. 4.2: DMs and atmospheric layers at different
 * conjugation altitudes, each with its own meta-pupil grid, modes and per-sensor composite transforms). */
typedef struct {
    const float *h_influence;         /* HOST float32 [n_modes][ny][nx] */
    int32_t n_modes, ny, nx;          /* nx % 4 == 0; the layer's own source grid (the geometry's is not used) */
    const int32_t *h_bbox;            /* HOST int32 [n_modes][4] inside the grid, or NULL = dense modes */
    const synim_wfs_affine *affine;   /* HOST [n_wfs]: this layer's composite transforms (cone factor, footprints ...) */
    float *h_out;                     /* HOST float32, column-major, ld = synim_num_rows(): the layer's own matrix */
} synim_layer;

/* The whole dictionary in one call, HOST buffers in and out: every layer's cube is fetched exactly once for all
 * sensors and streamed -- the modes of all layers are cut into chunks of about 64 MB of matrix, and
 * while chunk k is packed on the host (compact supports only) and copied in, chunk k-1 is computed and chunk k-2's
 * columns travel back, on two internal streams with two buffers of everything.  The sensors (geometry) are shared by
 * all layers; only the per-layer transforms differ.  Work queued on `stream` before the call is waited for; the call
 * returns when every matrix is in host memory.  synim_interaction_matrix_host is this call with one layer on the
 * geometry's own grid.  Pinned host buffers make the copies asynchronous but are not required.
 * Errors: INVALID_ARG (NULL, sizes, a bbox that leaves its grid, singular affine), ALIGNMENT, OUT_OF_MEMORY, CUDA. */
synim_status synim_dictionary_host(const synim_geometry *geom, const synim_layer *layers, int32_t n_layers,
                                   synim_slope_mode mode, void *stream);

/* ---- Tomographic projection matrix (sec. 2.5) ------------------------------------------------------
 * P_opt = (P_DM^T P_DM + lambda I)^-1 P_DM^T P_Layer, "where P_DM and P_Layer map the influence functions over the
 * optimized directions".  Readings (R24-R26): row (d, p) of an operand = optimisation direction d, pixel p of
 * an mp x mp pupil grid; column m = mode m of the component; entry = sqrt(weight_d) * pupil[p] * phi_m(A_d x_p), phi_m
 * resampled through the direction's composite map with the library's single bilinear interpolation (zero outside the
 * grid).  P_DM holds the columns of ALL mirrors side by side (component 0 first).
 * One component = one deformable mirror or one reconstructed layer: */
typedef struct {
    const float *d_cube;            /* DEVICE float32 [n_modes][ny][nx] */
    int32_t n_modes, ny, nx;        /* n_modes <= 65535 */
    const synim_wfs_affine *maps;   /* HOST [n_dir]: pupil pixel -> this component's grid, centred pixel coordinates as
                                       for a sensor (footprint h*theta of the direction, misregistration ...); slope_scale
                                       is ignored */
} synim_component;

/* The operands are built by a kernel of this library (HBM-bound by their store); the two contractions and the Cholesky
 * solve are cuBLAS (SYRK, GEMM, float32) and cuSOLVER (POTRF, POTRS) calls, loaded with dlopen at the first call
 * (SYNIM_ERR_UNSUPPORTED if they cannot be found).  Temporaries (the operands: 4*n_dir*mp*mp bytes per mode) come from
 * the stream-ordered allocator.  SYNCHRONISES `stream` once, to report a matrix that is not positive definite.
 *   dir_weight  HOST [n_dir] non-negative weights of the directions, or NULL = all 1
 *   d_pupil     DEVICE float32 [mp][mp] pupil weights (0 = outside)
 *   d_popt      DEVICE float32, column-major: element (a, l) = actuator / DM mode a (all mirrors, in order), layer mode
 *               l, at d_popt[l*ld + a]; ld >= sum of the mirrors' modes
 * Errors: INVALID_ARG (NULL, sizes, lambda < 0, not positive definite), UNSUPPORTED, OUT_OF_MEMORY, CUDA. */
synim_status synim_projection_matrix(const synim_component *dms, int32_t n_dms, const synim_component *layer,
                                     int32_t n_dir, const double *dir_weight, const float *d_pupil, int32_t mp,
                                     double lambda, float *d_popt, int64_t ld, void *stream);

void synim_destroy(synim_geometry *geom); /* NULL-safe; frees the internal device buffers */
const char *synim_last_error(void);       /* thread-local, never NULL */
int32_t synim_version(void);              /* major*1000 + minor */
/* Number of CUDA kernels this library has launched in this process so far (all entry points, all threads);
 * bench.py reports the difference around its timed steps as gpu_launches. */
int64_t synim_launch_count(void);

#ifdef __cplusplus
}
#endif
#endif /* SYNIM_H_ */
