// synim_api.cu -- host side of the C ABI declared in include/synim.h: argument checks, the static
// geometry object (S0 of SURVEY.md sec. 8(a)), float64 composition / inversion of the per-sensor
// affine maps, tile sizing, and the launches.  No compute happens here and there is no CPU path.
#include "../../include/synim.h"
#include "synim_device.h"

#include <cuda.h>   // CUtensorMap and its enums; cuTensorMapEncodeTiled is fetched through the runtime

#include <algorithm>
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstring>
#include <cstdlib>
#include <mutex>
#include <new>
#include <thread>
#include <vector>

namespace {

thread_local char g_err[512] = "";

synim_status fail(synim_status s, const char *fmt, ...)
{
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_err, sizeof(g_err), fmt, ap);
    va_end(ap);
    return s;
}

synim_status cuda_fail(cudaError_t e, const char *what)
{
    if (e == cudaErrorMemoryAllocation) return fail(SYNIM_ERR_OUT_OF_MEMORY, "%s: %s", what, cudaGetErrorString(e));
    return fail(SYNIM_ERR_CUDA, "%s: %s", what, cudaGetErrorString(e));
}

}  // namespace

namespace synim {
// the other translation units' way to set the calling thread's error text (synim_last_error)
synim_status report(synim_status s, const char *fmt, ...)
{
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_err, sizeof(g_err), fmt, ap);
    va_end(ap);
    return s;
}
}  // namespace synim

namespace {

#define SYNIM_CUDA(call)                                       \
    do {                                                       \
        cudaError_t e_ = (call);                               \
        if (e_ != cudaSuccess) return cuda_fail(e_, #call);    \
    } while (0)

struct WfsHost {
    int n_subap = 0, n_pix = 0, M = 0, n_valid = 0;
    int row_x = 0, row_y = 0;
    float *d_wmap = nullptr;
    float *d_gx = nullptr, *d_gy = nullptr;   // G-tilt coefficient maps
    int *d_subap_row = nullptr;
    int owner = -1;   // sensor that owns the four device maps (sensors with the same pupil, grid and valid mask
                      // share one set: their lines then hit in L1 / L2 whichever sensor a warp works on)
};

}  // namespace

struct synim_geometry {
    int ny = 0, nx = 0, device = 0;
    long long rows = 0;
    std::vector<WfsHost> wfs;
    mutable std::mutex lock;   // one host-buffer call at a time per geometry (they share the pipeline's buffers)
    // the host entry points' pipeline (synim_interaction_matrix_host / synim_dictionary_host): two chunks in flight
    struct Pipe {
        bool ready = false;
        cudaStream_t s_compute = nullptr, s_copy = nullptr;
        cudaEvent_t start = nullptr, h2d_done[2] = {nullptr, nullptr}, kern_done[2] = {nullptr, nullptr}, d2h_done[2] = {nullptr, nullptr};
        float *d_cube[2] = {nullptr, nullptr}; size_t d_cube_bytes[2] = {0, 0};
        float *d_out[2] = {nullptr, nullptr};  size_t d_out_bytes[2] = {0, 0};
        int *d_meta[2] = {nullptr, nullptr};   size_t d_meta_bytes[2] = {0, 0};
        char *h_stage[2] = {nullptr, nullptr}; size_t h_stage_bytes[2] = {0, 0};
    };
    mutable Pipe pipe;
    // the last tile plan of every sensor (dense modes): planning simulates bank conflicts (about a millisecond of host
    // time per sensor), and an on-line loop calls with the same transforms again and again
    struct PlanMemo { bool set = false; double key[7] = {0, 0, 0, 0, 0, 0, 0}; int ns = 0, nr = 0, pitch = 0, h = 0; bool fits = false; };
    mutable std::mutex plan_lock;
    mutable std::vector<PlanMemo> plans;
};

namespace {

synim_status check_device()
{
    int dev = 0, major = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return cuda_fail(e, "cudaGetDevice");
    SYNIM_CUDA(cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev));
    if (major != 10)
        return fail(SYNIM_ERR_UNSUPPORTED_DEVICE, "device %d has compute capability %d.x; this library is sm_100a only",
                    dev, major);
    return SYNIM_OK;
}

template <typename T>
synim_status grow(T *&ptr, size_t &have, size_t want)
{
    if (want <= have) return SYNIM_OK;
    if (ptr) cudaFree(ptr);
    ptr = nullptr;
    have = 0;
    cudaError_t e = cudaMalloc(reinterpret_cast<void **>(&ptr), want);
    if (e != cudaSuccess) return cuda_fail(e, "cudaMalloc(workspace)");
    have = want;
    return SYNIM_OK;
}

// The absolute-index forward map and its inverse, in float64 (R1, R2).
bool build_maps(const synim_wfs_affine &af, int M, int ny, int nx, double fwd[6], double inv[6])
{
    const double cw = (M - 1) / 2.0, cx = (nx - 1) / 2.0, cy = (ny - 1) / 2.0;
    const double *a = af.a;
    fwd[0] = a[0]; fwd[1] = a[1]; fwd[2] = a[2] + cx - cw * (a[0] + a[1]);
    fwd[3] = a[3]; fwd[4] = a[4]; fwd[5] = a[5] + cy - cw * (a[3] + a[4]);
    const double det = a[0] * a[4] - a[1] * a[3];
    for (int k = 0; k < 6; ++k)
        if (!std::isfinite(a[k])) return false;
    if (!std::isfinite(af.slope_scale) || !(std::fabs(det) > 1e-300)) return false;
    inv[0] = a[4] / det; inv[1] = -a[1] / det;
    inv[3] = -a[3] / det; inv[4] = a[0] / det;
    inv[2] = -(inv[0] * fwd[2] + inv[1] * fwd[5]);
    inv[5] = -(inv[3] * fwd[2] + inv[4] * fwd[5]);
    return true;
}

// TMA descriptor over the cube [n_modes][ny][nx] with box {box_w, box_h, 1}; out-of-range elements read
// as zero.  The driver entry point comes from the runtime, so libcuda is never linked.
synim_status encode_cube_map(const float *d_cube, int n_modes, int ny, int nx, int box_w, int box_h, CUtensorMap *out)
{
    typedef CUresult (*encode_fn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *,
                                  const cuuint64_t *, const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
    static encode_fn fn = nullptr;
    if (!fn) {
        void *sym = nullptr;
        cudaDriverEntryPointQueryResult q = cudaDriverEntryPointSymbolNotFound;
        cudaError_t e = cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &sym, cudaEnableDefault, &q);
        if (e != cudaSuccess || q != cudaDriverEntryPointSuccess || !sym)
            return fail(SYNIM_ERR_CUDA, "cuTensorMapEncodeTiled is not available from this driver");
        fn = reinterpret_cast<encode_fn>(sym);
    }
    if (box_w < 4 || box_w > 256 || box_h < 1 || box_h > 256 || box_w % 4 != 0)
        return fail(SYNIM_ERR_INVALID_ARG, "internal: TMA box %d x %d out of range", box_w, box_h);
    const cuuint64_t dims[3] = {(cuuint64_t)nx, (cuuint64_t)ny, (cuuint64_t)n_modes};
    const cuuint64_t strides[2] = {(cuuint64_t)nx * 4, (cuuint64_t)nx * (cuuint64_t)ny * 4};
    const cuuint32_t box[3] = {(cuuint32_t)box_w, (cuuint32_t)box_h, 1};
    const cuuint32_t estr[3] = {1, 1, 1};
    CUresult r = fn(out, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 3, const_cast<float *>(d_cube), dims, strides, box, estr,
                    CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_NONE,
                    CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) return fail(SYNIM_ERR_CUDA, "cuTensorMapEncodeTiled failed (CUresult %d)", (int)r);
    return SYNIM_OK;
}

}  // namespace

extern "C" {

const char *synim_last_error(void) { return g_err; }

int32_t synim_version(void) { return SYNIM_VERSION_MAJOR * 1000 + SYNIM_VERSION_MINOR; }

int64_t synim_launch_count(void) { return (int64_t)synim::launches_so_far(); }

synim_status synim_compose_affine(const synim_wfs_physical *p, synim_wfs_affine *out)
{
    if (!p || !out) return fail(SYNIM_ERR_INVALID_ARG, "synim_compose_affine: NULL argument");
    if (p->mag_x == 0.0 || p->mag_y == 0.0 || p->dm_mag == 0.0 || !(p->src_pixel_pitch_m > 0.0))
        return fail(SYNIM_ERR_INVALID_ARG, "synim_compose_affine: zero magnification or non-positive pixel pitch");
    const double deg = 3.14159265358979323846 / 180.0;
    // 3x3 homogeneous matrices, multiplied right to left in the order of synim.h
    struct H { double m[3][3]; };
    auto mul = [](const H &A, const H &B) {
        H C;
        for (int i = 0; i < 3; ++i)
            for (int j = 0; j < 3; ++j) C.m[i][j] = A.m[i][0] * B.m[0][j] + A.m[i][1] * B.m[1][j] + A.m[i][2] * B.m[2][j];
        return C;
    };
    auto rotm = [](double t) { return H{{{std::cos(t), std::sin(t), 0}, {-std::sin(t), std::cos(t), 0}, {0, 0, 1}}}; };
    auto scal = [](double sx, double sy) { return H{{{sx, 0, 0}, {0, sy, 0}, {0, 0, 1}}}; };
    auto tran = [](double tx, double ty) { return H{{{1, 0, tx}, {0, 1, ty}, {0, 0, 1}}}; };
    const double kappa = std::isinf(p->gs_range_m) ? 1.0 : 1.0 - p->dm_height_m / p->gs_range_m;
    const double theta = p->gs_theta_arcsec * deg / 3600.0, az = p->gs_azimuth_deg * deg;
    const double fx = p->dm_height_m * theta * std::cos(az) / p->src_pixel_pitch_m;
    const double fy = p->dm_height_m * theta * std::sin(az) / p->src_pixel_pitch_m;
    H T = scal(p->wfs_pitch_src_px, p->wfs_pitch_src_px);          // WFS pixel -> pupil-plane source pixels
    T = mul(tran(-p->shift_x, -p->shift_y), T);                    // remove the WFS shift
    T = mul(rotm(p->rot_deg * deg), T);                            // R(-rot)
    T = mul(scal(1.0 / p->mag_x, 1.0 / p->mag_y), T);              // undo (anamorphic) magnification
    T = mul(scal(kappa, kappa), T);                                // cone effect at the DM's altitude
    T = mul(tran(fx - p->dm_shift_x, fy - p->dm_shift_y), T);      // footprint shift, DM shift
    T = mul(rotm(p->dm_rot_deg * deg), T);                         // R(-dm_rot)
    T = mul(scal(1.0 / p->dm_mag, 1.0 / p->dm_mag), T);
    out->a[0] = T.m[0][0]; out->a[1] = T.m[0][1]; out->a[2] = T.m[0][2];
    out->a[3] = T.m[1][0]; out->a[4] = T.m[1][1]; out->a[5] = T.m[1][2];
    out->slope_scale = 1.0;
    return SYNIM_OK;
}

void synim_destroy(synim_geometry *g)
{
    if (!g) return;
    for (size_t k = 0; k < g->wfs.size(); ++k) {
        auto &w = g->wfs[k];
        if (w.owner != (int)k) continue;   // shared maps are freed by their owner
        if (w.d_wmap) cudaFree(w.d_wmap);
        if (w.d_gx) cudaFree(w.d_gx);
        if (w.d_gy) cudaFree(w.d_gy);
        if (w.d_subap_row) cudaFree(w.d_subap_row);
    }
    synim_geometry::Pipe &pp = g->pipe;
    for (int b = 0; b < 2; ++b) {
        if (pp.d_cube[b]) cudaFree(pp.d_cube[b]);
        if (pp.d_out[b]) cudaFree(pp.d_out[b]);
        if (pp.d_meta[b]) cudaFree(pp.d_meta[b]);
        if (pp.h_stage[b]) cudaFreeHost(pp.h_stage[b]);
        if (pp.h2d_done[b]) cudaEventDestroy(pp.h2d_done[b]);
        if (pp.kern_done[b]) cudaEventDestroy(pp.kern_done[b]);
        if (pp.d2h_done[b]) cudaEventDestroy(pp.d2h_done[b]);
    }
    if (pp.start) cudaEventDestroy(pp.start);
    if (pp.s_compute) cudaStreamDestroy(pp.s_compute);
    if (pp.s_copy) cudaStreamDestroy(pp.s_copy);
    delete g;
}

synim_status synim_create_geometry(int32_t ny, int32_t nx, int32_t n_wfs, const synim_wfs_grid *grids, void *stream,
                                   synim_geometry **out)
{
    if (!out) return fail(SYNIM_ERR_INVALID_ARG, "synim_create_geometry: out is NULL");
    *out = nullptr;
    if (!grids || ny <= 0 || nx <= 0 || n_wfs < 1 || n_wfs > 64)
        return fail(SYNIM_ERR_INVALID_ARG, "synim_create_geometry: need grids, ny,nx > 0 and 1 <= n_wfs <= 64");
    if (nx % 4 != 0) return fail(SYNIM_ERR_ALIGNMENT, "synim_create_geometry: nx = %d is not a multiple of 4", nx);
    for (int w = 0; w < n_wfs; ++w) {
        if (grids[w].n_subap < 1 || grids[w].n_pix < 1 || !grids[w].valid_mask || !grids[w].d_pupil)
            return fail(SYNIM_ERR_INVALID_ARG, "synim_create_geometry: sensor %d: bad n_subap / n_pix / NULL mask", w);
        if ((long long)grids[w].n_subap * grids[w].n_pix > 32768)
            return fail(SYNIM_ERR_INVALID_ARG, "synim_create_geometry: sensor %d: more than 32768 pixels per side", w);
    }
    synim_status st = check_device();
    if (st != SYNIM_OK) return st;
    cudaStream_t s = static_cast<cudaStream_t>(stream);

    synim_geometry *g = new (std::nothrow) synim_geometry;
    if (!g) return fail(SYNIM_ERR_OUT_OF_MEMORY, "synim_create_geometry: host allocation failed");
    g->ny = ny; g->nx = nx;
    cudaGetDevice(&g->device);
    g->wfs.resize(n_wfs);

    int *d_err = nullptr;
    uint8_t *d_valid = nullptr;
    size_t max_sub = 0;
    for (int w = 0; w < n_wfs; ++w) max_sub = std::max(max_sub, (size_t)grids[w].n_subap * grids[w].n_subap);
    auto cleanup = [&](synim_status r) {
        if (d_err) cudaFree(d_err);
        if (d_valid) cudaFree(d_valid);
        if (r != SYNIM_OK) synim_destroy(g);
        return r;
    };
    cudaError_t e;
    if ((e = cudaMalloc(reinterpret_cast<void **>(&d_err), sizeof(int))) != cudaSuccess) return cleanup(cuda_fail(e, "cudaMalloc"));
    if ((e = cudaMalloc(reinterpret_cast<void **>(&d_valid), max_sub)) != cudaSuccess) return cleanup(cuda_fail(e, "cudaMalloc"));
    if ((e = cudaMemsetAsync(d_err, 0, sizeof(int), s)) != cudaSuccess) return cleanup(cuda_fail(e, "cudaMemsetAsync"));

    long long row = 0;
    std::vector<int> rowmap;
    std::vector<uint8_t> valid01;
    for (int w = 0; w < n_wfs; ++w) {
        WfsHost &h = g->wfs[w];
        h.n_subap = grids[w].n_subap; h.n_pix = grids[w].n_pix; h.M = h.n_subap * h.n_pix;
        h.owner = w;
        const size_t ns = (size_t)h.n_subap * h.n_subap;
        rowmap.assign(ns, -1);
        valid01.assign(ns, 0);
        int k = 0;
        for (size_t q = 0; q < ns; ++q)
            if (grids[w].valid_mask[q]) { rowmap[q] = k++; valid01[q] = 1; }
        h.n_valid = k;
        if (row + 2LL * k > 0x3fffffffLL) return cleanup(fail(SYNIM_ERR_INVALID_ARG, "synim_create_geometry: more than 2^30 rows"));
        h.row_x = (int)row; h.row_y = (int)row + k;
        row += 2LL * k;
        // the same pupil buffer, grid and valid mask as an earlier sensor: share its maps
        for (int v = 0; v < w; ++v) {
            if (g->wfs[v].owner != v || grids[v].d_pupil != grids[w].d_pupil || grids[v].n_subap != h.n_subap ||
                grids[v].n_pix != h.n_pix)
                continue;
            bool same = true;
            for (size_t q = 0; q < ns && same; ++q) same = (grids[v].valid_mask[q] != 0) == (valid01[q] != 0);
            if (!same) continue;
            h.owner = v;
            h.d_wmap = g->wfs[v].d_wmap; h.d_gx = g->wfs[v].d_gx; h.d_gy = g->wfs[v].d_gy; h.d_subap_row = g->wfs[v].d_subap_row;
            break;
        }
        if (h.owner != w) continue;
        // rows of zeros below the map: the strip kernel's halo lanes and row look-ahead read them
        const size_t wmap_bytes = sizeof(float) * (size_t)(h.M + synim::kWmapPadRows) * h.M;
        if ((e = cudaMalloc(reinterpret_cast<void **>(&h.d_wmap), wmap_bytes)) != cudaSuccess)
            return cleanup(cuda_fail(e, "cudaMalloc(wmap)"));
        if ((e = cudaMemsetAsync(h.d_wmap, 0, wmap_bytes, s)) != cudaSuccess) return cleanup(cuda_fail(e, "cudaMemsetAsync(wmap)"));
        if ((e = cudaMalloc(reinterpret_cast<void **>(&h.d_subap_row), sizeof(int) * ns)) != cudaSuccess)
            return cleanup(cuda_fail(e, "cudaMalloc(subap_row)"));
        // pageable sources: these copies are staged by the runtime before the call returns
        if ((e = cudaMemcpyAsync(h.d_subap_row, rowmap.data(), sizeof(int) * ns, cudaMemcpyHostToDevice, s)) != cudaSuccess)
            return cleanup(cuda_fail(e, "cudaMemcpyAsync(subap_row)"));
        if ((e = cudaMemcpyAsync(d_valid, valid01.data(), ns, cudaMemcpyHostToDevice, s)) != cudaSuccess)
            return cleanup(cuda_fail(e, "cudaMemcpyAsync(valid)"));
        if ((e = synim::launch_subap_weights(grids[w].d_pupil, d_valid, h.n_subap, h.n_pix, h.d_wmap, h.d_subap_row, d_err, s)) != cudaSuccess)
            return cleanup(cuda_fail(e, "subap_weights_kernel"));
        // the G-tilt estimator's coefficient maps, same layout
        if ((e = cudaMalloc(reinterpret_cast<void **>(&h.d_gx), wmap_bytes)) != cudaSuccess) return cleanup(cuda_fail(e, "cudaMalloc(gx)"));
        if ((e = cudaMalloc(reinterpret_cast<void **>(&h.d_gy), wmap_bytes)) != cudaSuccess) return cleanup(cuda_fail(e, "cudaMalloc(gy)"));
        if ((e = cudaMemsetAsync(h.d_gx, 0, wmap_bytes, s)) != cudaSuccess) return cleanup(cuda_fail(e, "cudaMemsetAsync(gx)"));
        if ((e = cudaMemsetAsync(h.d_gy, 0, wmap_bytes, s)) != cudaSuccess) return cleanup(cuda_fail(e, "cudaMemsetAsync(gy)"));
        if ((e = synim::launch_gtilt_maps(grids[w].d_pupil, d_valid, h.n_subap, h.n_pix, h.d_gx, h.d_gy, s)) != cudaSuccess)
            return cleanup(cuda_fail(e, "gtilt_maps_kernel"));
        // d_valid is reused by the next sensor: stream order keeps this safe
    }
    g->rows = row;
    int herr = 0;
    if ((e = cudaMemcpyAsync(&herr, d_err, sizeof(int), cudaMemcpyDeviceToHost, s)) != cudaSuccess)
        return cleanup(cuda_fail(e, "cudaMemcpyAsync(err)"));
    if ((e = cudaStreamSynchronize(s)) != cudaSuccess) return cleanup(cuda_fail(e, "cudaStreamSynchronize"));
    if (herr) return cleanup(fail(SYNIM_ERR_EMPTY_SUBAP, "synim_create_geometry: a valid subaperture has zero summed pupil weight"));
    *out = g;
    return cleanup(SYNIM_OK);
}

int64_t synim_num_rows(const synim_geometry *g) { return g ? g->rows : -1; }

int64_t synim_num_valid(const synim_geometry *g, int32_t w)
{
    return (g && w >= 0 && w < (int)g->wfs.size()) ? g->wfs[w].n_valid : -1;
}

int64_t synim_row_offset(const synim_geometry *g, int32_t w)
{
    return (g && w >= 0 && w < (int)g->wfs.size()) ? g->wfs[w].row_x : -1;
}

// Dense modes, sensors whose subapertures fit a strip: tiles of the WFS grid (synim_tile_kernel).  A tile is
// tile_ns strips x tile_nr subaperture rows, about 119 pixels square, shrunk until the bounding box of its
// pre-image (+ halo, bilinear reach, one pixel of margin, alignment slack) fits a TMA box (<= 256 per side) and the
// shared-memory budget of two CTAs per SM; then the tile counts are evened out (68 rows -> 4 x 17, not 16+...+4).
// Returns false if not even a 1 x 1 tile fits (extreme magnification): the caller falls back to source-space pieces.
struct TilePlan { int ns, nr, pitch, h; };
static bool plan_tiles(const synim::WfsDev &d, size_t budget_floats, int reach, TilePlan *out)
{
    const int strip_px = d.spb * d.n_pix, n_strips = (d.n_subap + d.spb - 1) / d.spb;
    auto box = [&](int ns, int nr, int *pitch, int *h) {
        // phi pixels - 1 (one more row: look-ahead; reach: what a restored pixel reads beside itself, edge repair)
        const double wt = (double)std::min(ns * strip_px, d.M) + 1.0 + 2.0 * reach, ht = (double)std::min(nr * d.n_pix, d.M) + 2.0 + 2.0 * reach;
        const double ex = std::fabs(d.fwd[0]) * wt + std::fabs(d.fwd[1]) * ht, ey = std::fabs(d.fwd[3]) * wt + std::fabs(d.fwd[4]) * ht;
        if (!(ex < 1.0e6) || !(ey < 1.0e6)) { *pitch = *h = 1 << 20; return; }
        *pitch = ((int)std::ceil(ex) + 8 + 3) & ~3;   // floor(cmin)-1-slack(<=3) .. floor(cmax)+2
        *h = (int)std::ceil(ey) + 5;
    };
    int ns = std::max(1, std::min(n_strips, (119 + strip_px / 2) / strip_px));
    int nr = std::max(1, std::min(d.n_subap, (119 + d.n_pix / 2) / d.n_pix));
    int pitch = 0, h = 0;
    while (true) {
        box(ns, nr, &pitch, &h);
        if (pitch <= 256 && h <= 256 && (size_t)pitch * h + 3 * (size_t)ns * d.spb * nr <= budget_floats) break;
        if (ns == 1 && nr == 1) return false;
        // shrink the height first while the tile is not much flatter than wide: a CTA has one warp per strip, so a tile
        // of fewer strips than warps leaves warps idle, whereas fewer rows only shorten the strips
        const bool keep_width = ns <= synim::kTileWarpsPerCta && 10 * nr * d.n_pix >= 6 * ns * strip_px;
        if (nr > 1 && (keep_width || nr * d.n_pix >= ns * strip_px || ns == 1)) --nr; else --ns;
    }
    auto even_out = [&](int *pns, int *pnr) {
        const int ty = (d.n_subap + *pnr - 1) / *pnr, tx = (n_strips + *pns - 1) / *pns;
        *pnr = (d.n_subap + ty - 1) / ty;
        *pns = (n_strips + tx - 1) / tx;
    };
    // Shared-memory bank conflicts of the gather.  The 32 lanes of a warp sample 32 neighbouring WFS pixels of one row;
    // under a rotated sensor their four taps land on ~28 different box rows, and how those fall onto the 32 banks
    // depends on the box pitch modulo 32 alone: simulated for config 5, 1.1 to 4.0 wavefronts per LDS request on the
    // 60-degree sensors (ncu on the first version, fixed pitches: 1.9 on average).  So the pitch is padded by the
    // multiple of 4 floats (TMA rows are 16-byte multiples) with the fewest wavefronts; if even the best one that fits
    // stays above 1.6, a shorter tile (more room for padding) is tried.
    auto wavefronts = [&](int pit) {
        double tot = 0.0;
        int cnt = 0;
        for (int s = 0; s < 24; ++s) {
            const double j0 = (double)((s * 37) % std::max(1, d.M - 31)), i = (double)((s * 53 + 11) % d.M);
            long long c0[32], r0[32];
            for (int l = 0; l < 32; ++l) {
                const double j = j0 + l;
                c0[l] = (long long)std::floor(d.fwd[0] * j + d.fwd[1] * i + d.fwd[2]);
                r0[l] = (long long)std::floor(d.fwd[3] * j + d.fwd[4] * i + d.fwd[5]);
            }
            for (int tap = 0; tap < 4; ++tap) {
                long long word[32];
                int per_bank[32] = {0}, worst = 0;
                for (int l = 0; l < 32; ++l) {
                    word[l] = (r0[l] + (tap >> 1)) * pit + c0[l] + (tap & 1);
                    bool seen = false;
                    for (int q = 0; q < l && !seen; ++q) seen = word[q] == word[l];
                    if (!seen) worst = std::max(worst, ++per_bank[(int)(((word[l] % 32) + 32) % 32)]);
                }
                tot += worst; ++cnt;
            }
        }
        return tot / cnt;
    };
    auto best_pad = [&](int ns_, int nr_, int *ppitch, int *ph) {   // -> wavefronts per request; 1e9 if nothing fits
        int p0 = 0, h0 = 0;
        box(ns_, nr_, &p0, &h0);
        double best = 1.0e9;
        for (int pad = 0; pad < 32; pad += 4) {
            const int pit = p0 + pad;
            if (pit > 256 || h0 > 256 || (size_t)pit * h0 + 3 * (size_t)ns_ * d.spb * nr_ > budget_floats) break;
            const double w = wavefronts(pit);
            if (w < best - 1.0e-9) { best = w; *ppitch = pit; *ph = h0; }
        }
        return best;
    };
    even_out(&ns, &nr);
    double got = best_pad(ns, nr, &pitch, &h);
    for (int shorter = nr - 1; got > 1.6 && shorter >= std::max(4, nr - 3); --shorter) {
        int ns2 = ns, nr2 = shorter, p2 = 0, h2 = 0;
        even_out(&ns2, &nr2);
        const double w2 = best_pad(ns2, nr2, &p2, &h2);
        if (w2 < got - 0.2) { got = w2; ns = ns2; nr = nr2; pitch = p2; h = h2; }
    }
    if (got > 1.0e8) box(ns, nr, &pitch, &h);   // (cannot happen: the unpadded box of this tile fitted above)
    if (std::getenv("SYNIM_DEBUG_TILES"))
        std::fprintf(stderr, "synim: tile %d strips x %d rows, box %d x %d floats, %.2f shared-memory wavefronts per request\n", ns, nr,
                     pitch, h, got);
    out->ns = ns; out->nr = nr; out->pitch = pitch; out->h = h;
    return true;
}

// The launch behind both entry points.  The cube may be PACKED (synim_interaction_matrix_host): mode m
// then holds only the neighbourhood of its support, cube_ny x cube_nx pixels whose pixel (0, 0) is source
// pixel d_origin[m] = (ox, oy); bboxes and affine maps stay in source-grid coordinates.
static synim_status run_interaction_matrix(const synim_geometry *g, const float *d_influence, int cube_ny, int cube_nx,
                                           const int32_t *d_origin, int32_t n_modes, const int32_t *d_bbox,
                                           const int32_t *d_diag, int32_t bbox_max_w, int32_t bbox_max_h,
                                           const synim_wfs_affine *affine, synim_slope_mode mode, float *d_out, int64_t ld,
                                           void *stream, const float *d_mask = nullptr, double threshold = 0.0,
                                           int src_ny = 0, int src_nx = 0)
{
    if (!g || !affine || n_modes < 0) return fail(SYNIM_ERR_INVALID_ARG, "synim_interaction_matrix: NULL geometry/affine or n_modes < 0");
    const bool repair = d_mask != nullptr;
    if (repair && mode != SYNIM_SLOPES_ND)
        return fail(SYNIM_ERR_UNSUPPORTED, "edge repair belongs to the numerical-derivative engine (SYNIM_SLOPES_ND)");
    if (repair && !(threshold > 0.0 && threshold <= 1.0))
        return fail(SYNIM_ERR_INVALID_ARG, "synim_interaction_matrix_repaired: threshold %g is not in (0, 1]", threshold);
    if (mode != SYNIM_SLOPES_ND && mode != SYNIM_SLOPES_GTILT) return fail(SYNIM_ERR_INVALID_ARG, "synim_interaction_matrix: unknown slope mode %d", (int)mode);
    if (n_modes == 0) return SYNIM_OK;
    {   // the geometry's buffers live on the device it was created on (an sm_100 one: checked there)
        int cur = -1;
        SYNIM_CUDA(cudaGetDevice(&cur));
        if (cur != g->device)
            return fail(SYNIM_ERR_INVALID_ARG, "synim_interaction_matrix: current device %d is not the geometry's device %d", cur, g->device);
    }
    if (g->rows == 0) return SYNIM_OK;   // no sensor has a valid subaperture: the matrix has no rows, nothing is read or written
    if (!d_influence || !d_out) return fail(SYNIM_ERR_INVALID_ARG, "synim_interaction_matrix: NULL device buffer");
    if (ld < g->rows) return fail(SYNIM_ERR_INVALID_ARG, "synim_interaction_matrix: ld = %lld < rows = %lld", (long long)ld, g->rows);
    if (reinterpret_cast<uintptr_t>(d_influence) % 16 != 0)
        return fail(SYNIM_ERR_ALIGNMENT, "synim_interaction_matrix: influence cube is not 16-byte aligned");
    if (d_diag && !d_bbox) return fail(SYNIM_ERR_INVALID_ARG, "synim_interaction_matrix: d_diag without d_bbox");
    if (reinterpret_cast<uintptr_t>(d_out) % 4 != 0 || (d_bbox && reinterpret_cast<uintptr_t>(d_bbox) % 16 != 0) ||
        (d_diag && reinterpret_cast<uintptr_t>(d_diag) % 16 != 0))
        return fail(SYNIM_ERR_ALIGNMENT, "synim_interaction_matrix: output / bbox pointer misaligned");
    cudaStream_t s = static_cast<cudaStream_t>(stream);
    const int n_wfs = (int)g->wfs.size();
    const bool dense = (d_bbox == nullptr);
    // (a dictionary layer brings its own source grid; everything the geometry holds belongs to the sensors)
    const int ny = src_ny > 0 ? src_ny : g->ny, nx = src_nx > 0 ? src_nx : g->nx;

    // ---- shared-memory sizing ------------------------------------------------------------------
    // The staged box: <= 3 columns of TMA alignment slack, ring, support (or a piece of it), ring.  With a
    // size hint the whole support is one piece; without one, and for dense modes (the support is the
    // whole grid), 63 x 62 pieces -- by linearity a piece is its own mode and the pieces' slopes add up.
    const int kPatchMax = 128;
    int bw = bbox_max_w, bh = bbox_max_h;
    const bool hinted = !dense && bw > 0 && bh > 0 && bw + 5 <= kPatchMax && bh + 2 <= kPatchMax;
    int patch_pitch = 68, patch_h = 64;
    if (hinted) {
        patch_pitch = (std::min(bw, nx) + 5 + 3) & ~3;
        patch_h = std::min(bh, ny) + 2;
    }
    const int cap_w = patch_pitch - 5, cap_h = patch_h - 2;

    std::vector<synim::WfsDev> dev;
    try {
        dev.resize(n_wfs);
    } catch (...) {
        return fail(SYNIM_ERR_OUT_OF_MEMORY, "synim_interaction_matrix: host allocation failed");
    }
    for (int w = 0; w < n_wfs; ++w) {
        const WfsHost &h = g->wfs[w];
        synim::WfsDev &d = dev[w];
        if (!build_maps(affine[w], h.M, ny, nx, d.fwd, d.inv))
            return fail(SYNIM_ERR_INVALID_ARG, "synim_interaction_matrix: sensor %d: singular or non-finite affine", w);
        d.wmap = h.d_wmap; d.gx = h.d_gx; d.gy = h.d_gy; d.subap_row = h.d_subap_row;
        d.scale = (float)affine[w].slope_scale;
        d.M = h.M; d.n_subap = h.n_subap; d.n_pix = h.n_pix; d.row_x = h.row_x; d.row_y = h.row_y;
        d.tab_off = 0; d.tab_cap = 0;
        d.w_uniform = (float)(0.5 / ((double)h.n_pix * (double)h.n_pix));
        d.spb = h.n_pix <= synim::kStripMaxCols ? synim::kStripMaxCols / h.n_pix : 0;
        d.red_steps = 0;
        while (d.red_steps < 5 && (1 << d.red_steps) < h.n_pix) ++d.red_steps;
        d.npx_magic = (unsigned)((0x100000000ULL + (unsigned long long)h.n_pix - 1) / (unsigned long long)h.n_pix);   // (unused for 1)
    }
    // Edge repair: per call and sensor, the mask goes through the sensor's map and becomes pixel
    // classes, core-restricted weights and a row map that keeps the edge-sum path off anything not core.  The maps
    // live in ONE stream-ordered allocation, freed (on the stream) after the launches below.
    struct AsyncBlock {
        void *p = nullptr; cudaStream_t s = nullptr;
        ~AsyncBlock() { if (p) cudaFreeAsync(p, s); }
    } block;
    const int reach = repair ? synim::kRepairReach : 0;
    if (repair) {
        size_t total = 0;
        std::vector<size_t> off(n_wfs);
        auto up = [](size_t v) { return (v + 255) & ~(size_t)255; };
        for (int w = 0; w < n_wfs; ++w) {
            const WfsHost &h = g->wfs[w];
            const size_t np = (size_t)(h.M + 2) * (h.M + 2);
            off[w] = total;
            total += up(np) + up(np * sizeof(unsigned short)) + up(sizeof(float) * (size_t)(h.M + synim::kWmapPadRows) * h.M) +
                     up(sizeof(int) * (size_t)h.n_subap * h.n_subap);
        }
        block.s = s;
        SYNIM_CUDA(cudaMallocAsync(&block.p, total, s));
        for (int w = 0; w < n_wfs; ++w) {
            const WfsHost &h = g->wfs[w];
            const size_t np = (size_t)(h.M + 2) * (h.M + 2);
            const size_t wbytes = sizeof(float) * (size_t)(h.M + synim::kWmapPadRows) * h.M;
            char *base = static_cast<char *>(block.p) + off[w];
            unsigned char *core = reinterpret_cast<unsigned char *>(base);
            unsigned short *rcode = reinterpret_cast<unsigned short *>(base + up(np));
            float *wm = reinterpret_cast<float *>(base + up(np) + up(np * sizeof(unsigned short)));
            int *rows = reinterpret_cast<int *>(base + up(np) + up(np * sizeof(unsigned short)) + up(wbytes));
            SYNIM_CUDA(cudaMemsetAsync(wm, 0, wbytes, s));   // (the rows of zeros below the map)
            SYNIM_CUDA(synim::launch_repair_maps(d_mask, ny, nx, dev[w].fwd, threshold, h.n_subap, h.n_pix, h.d_wmap, h.d_subap_row,
                                                 core, rcode, wm, rows, s));
            dev[w].wmap = wm; dev[w].subap_row = rows; dev[w].rcode = rcode;
        }
    }
    // launch groups: consecutive sensors of one class (subapertures that fit a strip / giant ones), at most
    // kMaxWfsPerLaunch each; a group's rows are contiguous in the column
    std::vector<std::pair<int, int>> groups;   // [first, last) sensor
    for (int w = 0; w < n_wfs;) {
        int e = w + 1;
        while (e < n_wfs && e - w < synim::kMaxWfsPerLaunch && (dev[e].spb > 0) == (dev[w].spb > 0)) ++e;
        groups.emplace_back(w, e);
        w = e;
    }
    // per sensor a table of (x, y) partial slopes over the window of subapertures one piece's footprint
    // can span (the kernel derives the window from the same bounds and traps if it ever needed more)
    int tab_floats_max = 0;
    for (const auto &gr : groups) {
        int off = 0;
        for (int w = gr.first; w < gr.second; ++w) {
            synim::WfsDev &d = dev[w];
            const double ej = (cap_w + 2) * std::fabs(d.inv[0]) + (cap_h + 2) * std::fabs(d.inv[1]) + 2.0 * reach;
            const double ei = (cap_w + 2) * std::fabs(d.inv[3]) + (cap_h + 2) * std::fabs(d.inv[4]) + 2.0 * reach;
            auto span = [&](double e) {   // subapertures that floor(x) .. ceil(x + e) can touch
                const double s_ = std::floor((std::min(e, 1.0e8) + 2.0) / d.n_pix) + 2.0;
                return (int)std::min<double>(s_, d.n_subap);
            };
            d.tab_off = off;
            d.tab_cap = 2 * span(ej) * span(ei);
            off += d.tab_cap;
        }
        tab_floats_max = std::max(tab_floats_max, (off + 3) & ~3);
    }
    const size_t smem = sizeof(float) * ((size_t)patch_pitch * patch_h + (size_t)tab_floats_max) +
                        sizeof(int) * (size_t)(tab_floats_max / 2);
    CUtensorMap tmap;
    synim_status st = encode_cube_map(d_influence, n_modes, cube_ny, cube_nx, patch_pitch, patch_h, &tmap);
    if (st != SYNIM_OK) return st;
    if (smem > synim::max_dynamic_smem())
        return fail(SYNIM_ERR_CUDA, "synim_interaction_matrix: %zu bytes of shared memory exceed the device limit", smem);

    // ---- launches ------------------------------------------------------------------------------
    // Compact modes: the CTA that owns a column writes its zeros itself.  Dense modes: sensors whose subapertures
    // fit a strip go through the tile kernel (output-stationary: every slope stored once); the others (giant
    // subapertures, or a map so magnified that no tile fits) through source-space pieces spread over `chunks` CTAs
    // that add into the column, whose rows are cleared first (one strided memset per group).
    int chunks = 1;
    if (dense) {
        const int npieces = ((nx - 1 + cap_w) / cap_w) * ((ny - 1 + cap_h) / cap_h);
        chunks = std::max(1, std::min(npieces, 32));   // (2 .. 64 measured at config 5: 12.3 .. 9.6 ms, flat from 16 on)
    }
    for (const auto &gr : groups) {
        const int w0 = gr.first, nw = gr.second - gr.first;
        synim::ImParams p;
        std::memset(&p, 0, sizeof(p));
        p.cube = d_influence; p.bbox = d_bbox; p.diag = d_diag; p.origin = d_origin; p.out = d_out; p.ld = ld;
        p.n_modes = n_modes; p.ny = ny; p.nx = nx; p.n_wfs = nw;
        p.addr_bias = 0x4B400000u << 2;
        p.reach = reach;
        for (int w = 0; w < nw; ++w) p.wfs[w] = dev[w0 + w];
        if (dense && dev[w0].spb > 0) {
            // two CTAs per SM: half the SM's shared memory less the per-CTA reserve and the static part
            const size_t budget = (synim::max_dynamic_smem() + 1024) / 2 - 2048 - (size_t)synim::kTileScratchBytesPerCta;   // (less the warps' scratch)
            bool fits = true;
            int tiles = 0, box_floats = 0, tab = 0;
            for (int w = 0; w < nw && fits; ++w) {
                TilePlan tp = {0, 0, 0, 0};
                {
                    std::lock_guard<std::mutex> memo_guard(g->plan_lock);
                    if (g->plans.size() != g->wfs.size()) g->plans.assign(g->wfs.size(), synim_geometry::PlanMemo());
                    synim_geometry::PlanMemo &pm = g->plans[w0 + w];
                    const synim::WfsDev &dd = p.wfs[w];
                    const double key[7] = {dd.fwd[0], dd.fwd[1], dd.fwd[2], dd.fwd[3], dd.fwd[4], dd.fwd[5], (double)reach};
                    if (!pm.set || std::memcmp(pm.key, key, sizeof(key)) != 0) {
                        pm.fits = plan_tiles(dd, budget / sizeof(float), reach, &tp);
                        pm.ns = tp.ns; pm.nr = tp.nr; pm.pitch = tp.pitch; pm.h = tp.h;
                        std::memcpy(pm.key, key, sizeof(key));
                        pm.set = true;
                    }
                    fits = pm.fits;
                    tp.ns = pm.ns; tp.nr = pm.nr; tp.pitch = pm.pitch; tp.h = pm.h;
                }
                if (!fits) break;
                synim::WfsDev &d = p.wfs[w];
                d.tile_ns = tp.ns; d.tile_nr = tp.nr; d.box_pitch = tp.pitch; d.box_h = tp.h;
                d.tiles_x = ((d.n_subap + d.spb - 1) / d.spb + tp.ns - 1) / tp.ns;
                d.tiles_y = (d.n_subap + tp.nr - 1) / tp.nr;
                d.tile_first = tiles;
                tiles += d.tiles_x * d.tiles_y;
                d.tab_off = 0; d.tab_cap = 2 * tp.ns * d.spb * tp.nr;
                box_floats = std::max(box_floats, tp.pitch * tp.h);
                tab = std::max(tab, d.tab_cap);
            }
            if (fits) {
                synim::TileMaps maps;
                std::memset(&maps, 0, sizeof(maps));
                static_assert(sizeof(CUtensorMap) == 128, "TileMaps holds 128-byte descriptors");
                for (int w = 0; w < nw; ++w) {
                    CUtensorMap tm;
                    st = encode_cube_map(d_influence, n_modes, cube_ny, cube_nx, p.wfs[w].box_pitch, p.wfs[w].box_h, &tm);
                    if (st != SYNIM_OK) return st;
                    std::memcpy(maps.m[w], &tm, sizeof(tm));
                }
                // the kernel's layout: [ box | table | rows ], the box region sized for the largest sensor
                p.patch_pitch = box_floats; p.patch_h = 1; p.patch_pitchf = (float)box_floats;
                p.tab_floats = (tab + 3) & ~3;
                p.tiles_total = tiles;
                const size_t tsmem = sizeof(float) * ((size_t)box_floats + (size_t)p.tab_floats) + sizeof(int) * (size_t)(p.tab_floats / 2);
                int batch = 65535;   // grid.y holds the modes
                if (const char *env = std::getenv("SYNIM_TILE_BATCH_MODES")) {   // test knob: smaller batches
                    const int v = std::atoi(env);
                    if (v >= 1 && v < batch) batch = v;
                }
                for (int m0 = 0; m0 < n_modes; m0 += batch) {
                    synim::ImParams q = p;
                    q.n_modes = std::min(batch, n_modes - m0);
                    q.out = d_out + (size_t)m0 * (size_t)ld;
                    if (m0 > 0) {   // the descriptors address modes from the cube's start: re-encode on the batch
                        const float *sub = d_influence + (size_t)m0 * (size_t)cube_ny * (size_t)cube_nx;
                        for (int w = 0; w < nw; ++w) {
                            CUtensorMap tm;
                            st = encode_cube_map(sub, q.n_modes, cube_ny, cube_nx, p.wfs[w].box_pitch, p.wfs[w].box_h, &tm);
                            if (st != SYNIM_OK) return st;
                            std::memcpy(maps.m[w], &tm, sizeof(tm));
                        }
                    }
                    SYNIM_CUDA(synim::launch_tiles(q, maps, tsmem, mode == SYNIM_SLOPES_GTILT, repair, s));
                }
                continue;
            }
            for (int w = 0; w < nw; ++w) p.wfs[w] = dev[w0 + w];   // no tile fits: source-space pieces
        }
        p.patch_pitchf = (float)patch_pitch;
        p.patch_pitch = patch_pitch; p.patch_h = patch_h;
        // opt-in until measured on hardware: the packed boundary-only walk for zonal modes
        p.unit_rows = (!dense && !repair && mode == SYNIM_SLOPES_ND && dev[w0].spb > 0 && std::getenv("SYNIM_ZONAL_PACKED") &&
                       std::atoi(std::getenv("SYNIM_ZONAL_PACKED")) != 0) ? 1 : 0;
        p.tab_floats = nw > 0 ? (dev[w0 + nw - 1].tab_off + dev[w0 + nw - 1].tab_cap + 3) & ~3 : 0;
        p.chunks = chunks;
        if (dense) {
            p.zero_begin = 0; p.zero_count = 0;
            const int r_begin = g->wfs[w0].row_x;
            const WfsHost &last = g->wfs[w0 + nw - 1];
            const size_t r_count = (size_t)(last.row_x + 2 * last.n_valid - r_begin);
            if (r_count > 0)
                SYNIM_CUDA(cudaMemset2DAsync(d_out + r_begin, sizeof(float) * (size_t)ld, 0, sizeof(float) * r_count, n_modes, s));
        } else {
            p.zero_begin = g->wfs[w0].row_x;
            const WfsHost &last = g->wfs[w0 + nw - 1];
            p.zero_count = last.row_x + 2 * last.n_valid - p.zero_begin;
        }
        SYNIM_CUDA(synim::launch_strip(p, &tmap, smem, mode == SYNIM_SLOPES_GTILT, repair, s));
    }
    return SYNIM_OK;
}

synim_status synim_interaction_matrix(const synim_geometry *g, const float *d_influence, int32_t n_modes,
                                      const int32_t *d_bbox, const int32_t *d_diag, int32_t bbox_max_w, int32_t bbox_max_h,
                                      const synim_wfs_affine *affine, synim_slope_mode mode, float *d_out, int64_t ld,
                                      void *stream)
{
    if (!g) return fail(SYNIM_ERR_INVALID_ARG, "synim_interaction_matrix: NULL geometry/affine or n_modes < 0");
    return run_interaction_matrix(g, d_influence, g->ny, g->nx, nullptr, n_modes, d_bbox, d_diag, bbox_max_w, bbox_max_h, affine,
                                  mode, d_out, ld, stream);
}

synim_status synim_interaction_matrix_repaired(const synim_geometry *g, const float *d_influence, int32_t n_modes,
                                               const int32_t *d_bbox, const int32_t *d_diag, int32_t bbox_max_w, int32_t bbox_max_h,
                                               const synim_wfs_affine *affine, const float *d_mask, double threshold, float *d_out,
                                               int64_t ld, void *stream)
{
    if (!g) return fail(SYNIM_ERR_INVALID_ARG, "synim_interaction_matrix_repaired: NULL geometry");
    if (!d_mask) return fail(SYNIM_ERR_INVALID_ARG, "synim_interaction_matrix_repaired: NULL mask");
    return run_interaction_matrix(g, d_influence, g->ny, g->nx, nullptr, n_modes, d_bbox, d_diag, bbox_max_w, bbox_max_h, affine,
                                  SYNIM_SLOPES_ND, d_out, ld, stream, d_mask, threshold);
}

synim_status synim_compute_bboxes(const float *d_influence, int32_t n_modes, int32_t ny, int32_t nx, int32_t *d_bbox,
                                  int32_t *d_diag, void *stream)
{
    if (n_modes < 0 || ny <= 0 || nx <= 0) return fail(SYNIM_ERR_INVALID_ARG, "synim_compute_bboxes: bad sizes");
    if (n_modes == 0) return SYNIM_OK;
    if (!d_influence || !d_bbox) return fail(SYNIM_ERR_INVALID_ARG, "synim_compute_bboxes: NULL device buffer");
    if (nx % 4 != 0 || reinterpret_cast<uintptr_t>(d_influence) % 16 != 0 || reinterpret_cast<uintptr_t>(d_bbox) % 16 != 0 ||
        reinterpret_cast<uintptr_t>(d_diag) % 16 != 0)
        return fail(SYNIM_ERR_ALIGNMENT, "synim_compute_bboxes: need nx %% 4 == 0 and 16-byte aligned buffers");
    SYNIM_CUDA(synim::launch_compute_bboxes(d_influence, n_modes, ny, nx, d_bbox, d_diag, static_cast<cudaStream_t>(stream)));
    return SYNIM_OK;
}

synim_status synim_bbox_extent(const int32_t *d_bbox, int32_t n_modes, int32_t *max_w, int32_t *max_h, void *stream)
{
    if (!max_w || !max_h || n_modes < 0) return fail(SYNIM_ERR_INVALID_ARG, "synim_bbox_extent: bad arguments");
    *max_w = 0; *max_h = 0;
    if (n_modes == 0) return SYNIM_OK;
    if (!d_bbox) return fail(SYNIM_ERR_INVALID_ARG, "synim_bbox_extent: NULL device buffer");
    cudaStream_t s = static_cast<cudaStream_t>(stream);
    // two ints of device scratch per device, allocated once per process (the call synchronises anyway, so
    // concurrent callers are serialised by the lock)
    static std::mutex lock;
    static int *scratch[64] = {};
    int dev = 0;
    SYNIM_CUDA(cudaGetDevice(&dev));
    if (dev < 0 || dev >= 64) return fail(SYNIM_ERR_INVALID_ARG, "synim_bbox_extent: device index %d out of range", dev);
    std::lock_guard<std::mutex> guard(lock);
    if (!scratch[dev]) SYNIM_CUDA(cudaMalloc(reinterpret_cast<void **>(&scratch[dev]), 2 * sizeof(int)));
    int *d_wh = scratch[dev];
    int wh[2] = {0, 0};
    cudaError_t e = synim::launch_bbox_extent(d_bbox, n_modes, d_wh, s);
    if (e == cudaSuccess) e = cudaMemcpyAsync(wh, d_wh, sizeof(wh), cudaMemcpyDeviceToHost, s);
    if (e == cudaSuccess) e = cudaStreamSynchronize(s);
    if (e != cudaSuccess) return cuda_fail(e, "synim_bbox_extent");
    *max_w = wh[0]; *max_h = wh[1];
    return SYNIM_OK;
}

synim_status synim_interaction_matrix_flat(const float *d_influence, int32_t n_modes, int32_t ny, int32_t nx, int32_t n_wfs,
                                           const synim_wfs_grid *grids, const synim_wfs_affine *affine, int32_t compact,
                                           synim_slope_mode mode, float *d_out, int64_t ld, int64_t *rows_out, void *stream)
{
    if (rows_out) *rows_out = -1;
    if (!affine || n_modes < 0) return fail(SYNIM_ERR_INVALID_ARG, "synim_interaction_matrix_flat: NULL affine or n_modes < 0");
    synim_geometry *g = nullptr;
    synim_status st = synim_create_geometry(ny, nx, n_wfs, grids, stream, &g);
    if (st != SYNIM_OK) return st;
    if (rows_out) *rows_out = g->rows;
    cudaStream_t s = static_cast<cudaStream_t>(stream);
    int32_t *d_sup = nullptr;   // [n_modes][4] bboxes, then [n_modes][4] diagonal extents
    int32_t bw = 0, bh = 0;
    if (compact && n_modes > 0) {
        cudaError_t e = cudaMallocAsync(reinterpret_cast<void **>(&d_sup), sizeof(int32_t) * 8 * (size_t)n_modes, s);
        if (e != cudaSuccess) st = cuda_fail(e, "cudaMallocAsync(supports)");
        if (st == SYNIM_OK) st = synim_compute_bboxes(d_influence, n_modes, ny, nx, d_sup, d_sup + 4 * (size_t)n_modes, stream);
        if (st == SYNIM_OK) st = synim_bbox_extent(d_sup, n_modes, &bw, &bh, stream);
    }
    if (st == SYNIM_OK)
        st = run_interaction_matrix(g, d_influence, ny, nx, nullptr, n_modes, d_sup, d_sup ? d_sup + 4 * (size_t)n_modes : nullptr, bw, bh,
                                    affine, mode, d_out, ld, stream);
    if (d_sup) cudaFreeAsync(d_sup, s);
    const cudaError_t e = cudaDeviceSynchronize();   // the geometry's maps are in use until the launches have drained
    synim_destroy(g);
    if (st == SYNIM_OK && e != cudaSuccess) st = cuda_fail(e, "synim_interaction_matrix_flat");
    return st;
}

// The pipeline behind both host entry points.  The modes of every layer are cut into chunks; chunk k is packed on the
// host (compact supports only) while chunk k-1 runs and chunk k-2 goes home:
//     host: pack k | s_compute: H2D k, kernel k | s_copy: D2H k        (two buffers of everything, events between)
// so the bus carries the matrix back (the bulk of the bytes) while the next supports are packed, copied and computed.
#define SYNIM_PIPE(call)                                              \
    do {                                                              \
        cudaError_t e_ = (call);                                      \
        if (e_ != cudaSuccess) return drain(cuda_fail(e_, #call));    \
    } while (0)
static synim_status host_pipeline(const synim_geometry *g, const synim_layer *layers, int32_t n_layers, synim_slope_mode mode,
                                  void *stream)
{
    std::lock_guard<std::mutex> guard(g->lock);
    synim_geometry::Pipe &pp = g->pipe;
    if (!pp.ready) {
        SYNIM_CUDA(cudaStreamCreateWithFlags(&pp.s_compute, cudaStreamNonBlocking));
        SYNIM_CUDA(cudaStreamCreateWithFlags(&pp.s_copy, cudaStreamNonBlocking));
        SYNIM_CUDA(cudaEventCreateWithFlags(&pp.start, cudaEventDisableTiming));
        for (int b = 0; b < 2; ++b) {
            SYNIM_CUDA(cudaEventCreateWithFlags(&pp.h2d_done[b], cudaEventDisableTiming));
            SYNIM_CUDA(cudaEventCreateWithFlags(&pp.kern_done[b], cudaEventDisableTiming));
            SYNIM_CUDA(cudaEventCreateWithFlags(&pp.d2h_done[b], cudaEventDisableTiming));
        }
        pp.ready = true;
    }
    // whatever the caller queued on `stream` comes first
    SYNIM_CUDA(cudaEventRecord(pp.start, static_cast<cudaStream_t>(stream)));
    SYNIM_CUDA(cudaStreamWaitEvent(pp.s_compute, pp.start, 0));

    auto grow_pinned = [&](int b, size_t want) -> synim_status {
        if (want <= pp.h_stage_bytes[b]) return SYNIM_OK;
        if (pp.h_stage[b]) cudaFreeHost(pp.h_stage[b]);
        pp.h_stage[b] = nullptr; pp.h_stage_bytes[b] = 0;
        cudaError_t e = cudaMallocHost(reinterpret_cast<void **>(&pp.h_stage[b]), want);
        if (e != cudaSuccess) return cuda_fail(e, "cudaMallocHost(staging)");
        pp.h_stage_bytes[b] = want;
        return SYNIM_OK;
    };
    auto drain = [&](synim_status st) {   // buffers are reused by the next call: nothing may still be in flight
        cudaStreamSynchronize(pp.s_compute);
        cudaStreamSynchronize(pp.s_copy);
        return st;
    };

    size_t kChunkBytes = (size_t)64 << 20;   // of matrix (and of dense cube) per chunk
    if (const char *env = std::getenv("SYNIM_HOST_CHUNK_BYTES")) {   // tuning / test knob
        const long long v = std::atoll(env);
        if (v >= 4096) kChunkBytes = (size_t)v;
    }
    const int nthreads = (int)std::max(1u, std::min(8u, std::thread::hardware_concurrency()));
    long long k = 0;                                // chunks issued so far (buffer = k & 1)
    bool used[2] = {false, false};
    for (int32_t li = 0; li < n_layers; ++li) {
        const synim_layer &L = layers[li];
        if (L.n_modes == 0) continue;
        const int ny = L.ny, nx = L.nx;
        const size_t col_bytes = sizeof(float) * (size_t)g->rows;
        const bool dense = L.h_bbox == nullptr;
        // compact supports: every mode of the layer is packed into one pny x pnx image (see the header)
        int bw = 0, bh = 0, pnx = 0, pny = 0;
        if (!dense) {
            for (int m = 0; m < L.n_modes; ++m) {
                const int32_t *b = L.h_bbox + 4 * (size_t)m;
                if (b[2] < b[0] || b[3] < b[1]) continue;
                if (b[0] < 0 || b[1] < 0 || b[2] >= nx || b[3] >= ny)
                    return drain(fail(SYNIM_ERR_INVALID_ARG, "host entry point: layer %d: bbox of mode %d leaves the grid", (int)li, m));
                bw = std::max(bw, b[2] - b[0] + 1);
                bh = std::max(bh, b[3] - b[1] + 1);
            }
            pnx = std::max(8, (bw + 5 + 3) & ~3); pny = std::max(4, bh + 2);
        }
        const size_t img = dense ? (size_t)ny * nx : (size_t)pnx * pny;
        size_t per_mode = std::max(col_bytes, dense ? sizeof(float) * img : (size_t)1);
        const int chunk_modes = (int)std::max<size_t>(1, std::min<size_t>((size_t)L.n_modes, kChunkBytes / std::max<size_t>(per_mode, 1)));
        for (int m0 = 0; m0 < L.n_modes; m0 += chunk_modes, ++k) {
            const int b = (int)(k & 1), nm = std::min(chunk_modes, L.n_modes - m0);
            const size_t cube_bytes = sizeof(float) * img * nm, meta_bytes = dense ? 0 : sizeof(int) * 6 * (size_t)nm;
            const size_t out_bytes = col_bytes * nm;
            synim_status st;
            if ((st = grow(pp.d_out[b], pp.d_out_bytes[b], std::max<size_t>(out_bytes, 16))) != SYNIM_OK) return drain(st);
            if ((st = grow(pp.d_cube[b], pp.d_cube_bytes[b], cube_bytes)) != SYNIM_OK) return drain(st);
            const float *src_chunk = L.h_influence + (size_t)m0 * ny * nx;
            if (dense) {
                // the staging buffer of two chunks ago is free once its copy has left the host
                if (used[b]) SYNIM_PIPE(cudaEventSynchronize(pp.h2d_done[b]));
                SYNIM_PIPE(cudaMemcpyAsync(pp.d_cube[b], src_chunk, cube_bytes, cudaMemcpyHostToDevice, pp.s_compute));
                SYNIM_PIPE(cudaEventRecord(pp.h2d_done[b], pp.s_compute));
            } else {
                if ((st = grow(pp.d_meta[b], pp.d_meta_bytes[b], meta_bytes)) != SYNIM_OK) return drain(st);
                if (used[b]) SYNIM_PIPE(cudaEventSynchronize(pp.h2d_done[b]));
                if ((st = grow_pinned(b, cube_bytes + meta_bytes)) != SYNIM_OK) return drain(st);
                float *stage = reinterpret_cast<float *>(pp.h_stage[b]);
                int *meta = reinterpret_cast<int *>(pp.h_stage[b] + cube_bytes);
                std::memcpy(meta, L.h_bbox + 4 * (size_t)m0, sizeof(int) * 4 * (size_t)nm);
                int *origin = meta + 4 * (size_t)nm;
                auto pack = [&](int q0, int q1) {
                    for (int q = q0; q < q1; ++q) {
                        const int32_t *bb = L.h_bbox + 4 * (size_t)(m0 + q);
                        float *dst = stage + img * q;
                        std::memset(dst, 0, sizeof(float) * img);
                        origin[2 * q] = 0; origin[2 * q + 1] = 0;
                        if (bb[2] < bb[0] || bb[3] < bb[1]) continue;
                        const int ox = (bb[0] - 1) & ~3, oy = bb[1] - 1;
                        origin[2 * q] = ox; origin[2 * q + 1] = oy;
                        const float *src = src_chunk + (size_t)q * ny * nx;
                        const size_t row_bytes = sizeof(float) * (size_t)(bb[2] - bb[0] + 1);
                        for (int y = bb[1]; y <= bb[3]; ++y)
                            std::memcpy(dst + (size_t)(y - oy) * pnx + (bb[0] - ox), src + (size_t)y * nx + bb[0], row_bytes);
                    }
                };
                int done = 0;   // modes [0, done) of the chunk are packed (or handed to a thread)
                if (nthreads > 1 && nm >= 64) {
                    std::vector<std::thread> pool;
                    try {   // no exception crosses the C ABI: what the threads could not be started for is packed here
                        pool.reserve(nthreads);
                        for (int t = 0; t < nthreads; ++t) {
                            const int q1 = (int)((long long)nm * (t + 1) / nthreads);
                            pool.emplace_back(pack, done, q1);
                            done = q1;
                        }
                    } catch (...) {
                    }
                    for (auto &th : pool) th.join();
                }
                pack(done, nm);
                SYNIM_PIPE(cudaMemcpyAsync(pp.d_cube[b], stage, cube_bytes, cudaMemcpyHostToDevice, pp.s_compute));
                SYNIM_PIPE(cudaMemcpyAsync(pp.d_meta[b], meta, meta_bytes, cudaMemcpyHostToDevice, pp.s_compute));
                SYNIM_PIPE(cudaEventRecord(pp.h2d_done[b], pp.s_compute));
            }
            // the output buffer of two chunks ago must have gone home before the kernel overwrites it
            if (used[b]) SYNIM_PIPE(cudaStreamWaitEvent(pp.s_compute, pp.d2h_done[b], 0));
            if (dense)
                st = run_interaction_matrix(g, pp.d_cube[b], ny, nx, nullptr, nm, nullptr, nullptr, 0, 0, L.affine, mode, pp.d_out[b],
                                            g->rows, pp.s_compute, nullptr, 0.0, ny, nx);
            else
                st = run_interaction_matrix(g, pp.d_cube[b], pny, pnx, pp.d_meta[b] + 4 * (size_t)nm, nm, pp.d_meta[b], nullptr, bw, bh,
                                            L.affine, mode, pp.d_out[b], g->rows, pp.s_compute, nullptr, 0.0, ny, nx);
            if (st != SYNIM_OK) return drain(st);
            SYNIM_PIPE(cudaEventRecord(pp.kern_done[b], pp.s_compute));
            SYNIM_PIPE(cudaStreamWaitEvent(pp.s_copy, pp.kern_done[b], 0));
            SYNIM_PIPE(cudaMemcpyAsync(L.h_out + (size_t)m0 * (size_t)g->rows, pp.d_out[b], out_bytes, cudaMemcpyDeviceToHost, pp.s_copy));
            SYNIM_PIPE(cudaEventRecord(pp.d2h_done[b], pp.s_copy));
            used[b] = true;
        }
    }
    cudaError_t e1 = cudaStreamSynchronize(pp.s_compute), e2 = cudaStreamSynchronize(pp.s_copy);
    if (e1 != cudaSuccess) return cuda_fail(e1, "cudaStreamSynchronize(compute)");
    if (e2 != cudaSuccess) return cuda_fail(e2, "cudaStreamSynchronize(copy)");
    return SYNIM_OK;
}

static synim_status check_layers(const synim_geometry *g, const synim_layer *layers, int32_t n_layers, const char *who)
{
    for (int32_t li = 0; li < n_layers; ++li) {
        const synim_layer &L = layers[li];
        if (L.n_modes < 0 || L.ny <= 0 || L.nx <= 0) return fail(SYNIM_ERR_INVALID_ARG, "%s: layer %d: bad sizes", who, (int)li);
        if (L.nx % 4 != 0) return fail(SYNIM_ERR_ALIGNMENT, "%s: layer %d: nx = %d is not a multiple of 4", who, (int)li, L.nx);
        if (L.n_modes > 0 && (!L.h_influence || !L.h_out || !L.affine))
            return fail(SYNIM_ERR_INVALID_ARG, "%s: layer %d: NULL host buffer or affine", who, (int)li);
    }
    (void)g;
    return SYNIM_OK;
}

synim_status synim_interaction_matrix_host(const synim_geometry *g, const float *h_influence, int32_t n_modes,
                                           const int32_t *h_bbox, const synim_wfs_affine *affine, synim_slope_mode mode,
                                           float *h_out, void *stream)
{
    if (!g || !affine || n_modes < 0) return fail(SYNIM_ERR_INVALID_ARG, "synim_interaction_matrix_host: bad arguments");
    if (n_modes == 0) return SYNIM_OK;
    if (!h_influence || !h_out) return fail(SYNIM_ERR_INVALID_ARG, "synim_interaction_matrix_host: NULL host buffer");
    synim_layer L;
    L.h_influence = h_influence; L.n_modes = n_modes; L.ny = g->ny; L.nx = g->nx; L.h_bbox = h_bbox; L.affine = affine; L.h_out = h_out;
    return host_pipeline(g, &L, 1, mode, stream);
}

synim_status synim_dictionary_host(const synim_geometry *g, const synim_layer *layers, int32_t n_layers, synim_slope_mode mode,
                                   void *stream)
{
    if (!g || n_layers < 0 || (n_layers > 0 && !layers)) return fail(SYNIM_ERR_INVALID_ARG, "synim_dictionary_host: bad arguments");
    if (mode != SYNIM_SLOPES_ND && mode != SYNIM_SLOPES_GTILT) return fail(SYNIM_ERR_INVALID_ARG, "synim_dictionary_host: unknown slope mode %d", (int)mode);
    synim_status st = check_layers(g, layers, n_layers, "synim_dictionary_host");
    if (st != SYNIM_OK) return st;
    if (n_layers == 0) return SYNIM_OK;
    return host_pipeline(g, layers, n_layers, mode, stream);
}

}  // extern "C"
