// synim_kernels.cu -- set-up kernels of the synthetic Shack-Hartmann interaction matrix for sm_100a:
// the per-pixel reduction weights of a sensor (S0 of SURVEY.md sec. 8(a)) and the supports of a cube
// (bounding boxes and diagonal extents).  The hot path (S1-S4) is synim_strip.cu.
#include "synim_device.h"

#include <atomic>

namespace synim {

namespace {

// ---- geometry-time kernels ----------------------------------------------------------------------
// one CTA per subaperture: W_S = sum of P, then wmap = 0.5*P/W_S (0 if invalid).  A valid subaperture whose
// n_pix^2 weights are not all equal gets kSubapGeneral set in its row-map entry: the others ("uniform":
// fully and evenly lit, the common case under a binary pupil) have the constant weight 0.5/n_pix^2, which the
// strip kernel applies once per subaperture to edge sums instead of once per pixel (synim_strip.cu).
__global__ void __launch_bounds__(128) subap_weights_kernel(const float *__restrict__ pupil,
                                                            const uint8_t *__restrict__ valid, int n_subap,
                                                            int n_pix, float *__restrict__ wmap, int *__restrict__ subap_row,
                                                            int *err)
{
    __shared__ double part[4];
    __shared__ float pmin[4], pmax[4];
    __shared__ double total;
    const int s = blockIdx.x, a = s / n_subap, b = s - a * n_subap;
    const int M = n_subap * n_pix, n = n_pix * n_pix;
    double acc = 0.0;
    float lo = 3.0e38f, hi = -3.0e38f;
    for (int e = threadIdx.x; e < n; e += 128) {
        const int r = e / n_pix, c = e - r * n_pix;
        const float pv = pupil[(size_t)(a * n_pix + r) * M + b * n_pix + c];
        acc += (double)pv;
        lo = fminf(lo, pv); hi = fmaxf(hi, pv);
    }
    for (int o = 16; o > 0; o >>= 1) {
        acc += __shfl_xor_sync(0xffffffffu, acc, o);
        lo = fminf(lo, __shfl_xor_sync(0xffffffffu, lo, o));
        hi = fmaxf(hi, __shfl_xor_sync(0xffffffffu, hi, o));
    }
    if ((threadIdx.x & 31) == 0) { part[threadIdx.x >> 5] = acc; pmin[threadIdx.x >> 5] = lo; pmax[threadIdx.x >> 5] = hi; }
    __syncthreads();
    if (threadIdx.x == 0) {
        total = part[0] + part[1] + part[2] + part[3];
        if (valid[s] && !(total > 0.0)) atomicExch(err, 1);
        const float l = fminf(fminf(pmin[0], pmin[1]), fminf(pmin[2], pmin[3]));
        const float h = fmaxf(fmaxf(pmax[0], pmax[1]), fmaxf(pmax[2], pmax[3]));
        if (valid[s] && !(l == h)) subap_row[s] |= kSubapGeneral;   // (the host wrote the row index, >= 0, before this launch)
    }
    __syncthreads();
    const bool ok = valid[s] && total > 0.0;
    for (int e = threadIdx.x; e < n; e += 128) {
        const int r = e / n_pix, c = e - r * n_pix;
        const size_t at = (size_t)(a * n_pix + r) * M + b * n_pix + c;
        wmap[at] = ok ? (float)(0.5 * (double)pupil[at] / total) : 0.0f;
    }
}

// G-tilt (reading R13) as two coefficient maps.  A pixel is valid iff
// P >= 0.5.  For every pixel row of a subaperture with first / last valid columns jf < jl the estimator
// adds phi[row][jl] - phi[row][jf] to a numerator and jl - jf to a denominator; s_x = num / den (0 if
// den = 0), and the same over pixel columns for s_y.  That is s_x = sum gx*phi, s_y = sum gy*phi with
// gx = +-1/den_x on those end pixels and 0 elsewhere.  One CTA per subaperture; gx, gy arrive zeroed.
__global__ void __launch_bounds__(128) gtilt_maps_kernel(const float *__restrict__ pupil, const uint8_t *__restrict__ valid,
                                                         int n_subap, int n_pix, float *__restrict__ gx,
                                                         float *__restrict__ gy)
{
    __shared__ int den[2];
    const int s = blockIdx.x, a = s / n_subap, b = s - a * n_subap;
    if (!valid[s]) return;   // CTA-uniform
    const int M = n_subap * n_pix, i0 = a * n_pix, j0 = b * n_pix;
    if (threadIdx.x < 2) den[threadIdx.x] = 0;
    __syncthreads();
    // pass 1: the two denominators
    for (int r = threadIdx.x; r < 2 * n_pix; r += 128) {
        const int axis = r >= n_pix, q = axis ? r - n_pix : r;   // axis 0: pixel row i0+q; axis 1: pixel column j0+q
        int f = -1, l = -1;
        for (int t = 0; t < n_pix; ++t) {
            const float pv = axis ? pupil[(size_t)(i0 + t) * M + j0 + q] : pupil[(size_t)(i0 + q) * M + j0 + t];
            if (pv >= 0.5f) { if (f < 0) f = t; l = t; }
        }
        if (f >= 0 && l > f) atomicAdd(&den[axis], l - f);
    }
    __syncthreads();
    // pass 2: +-1/den on the end pixels
    for (int r = threadIdx.x; r < 2 * n_pix; r += 128) {
        const int axis = r >= n_pix, q = axis ? r - n_pix : r;
        if (den[axis] <= 0) continue;
        int f = -1, l = -1;
        for (int t = 0; t < n_pix; ++t) {
            const float pv = axis ? pupil[(size_t)(i0 + t) * M + j0 + q] : pupil[(size_t)(i0 + q) * M + j0 + t];
            if (pv >= 0.5f) { if (f < 0) f = t; l = t; }
        }
        if (f >= 0 && l > f) {
            const float c = (float)(1.0 / (double)den[axis]);
            if (axis) {
                gy[(size_t)(i0 + l) * M + j0 + q] = c;
                gy[(size_t)(i0 + f) * M + j0 + q] = -c;
            } else {
                gx[(size_t)(i0 + q) * M + j0 + l] = c;
                gx[(size_t)(i0 + q) * M + j0 + f] = -c;
            }
        }
    }
}

// ---- edge repair, per call (readings R18-R22) -----------------------------------------
// Step 1, the strict core: the mask goes through the SAME map and the same bilinear rule as the modes (zero outside
// the grid), in float64 -- float32 coordinates could not tell a weight of 1e-6 from 0 -- and core = (mu >= threshold).
struct Fwd6 { double a[6]; };
__global__ void __launch_bounds__(256) repair_core_kernel(const float *__restrict__ mask, int ny, int nx, Fwd6 f, double threshold,
                                                          int M, unsigned char *__restrict__ core)
{
    const int P = M + 2;
    const int q = blockIdx.x * 256 + threadIdx.x;
    if (q >= P * P) return;
    const int i = q / P - 1, j = q - (i + 1) * P - 1;
    const double col = f.a[0] * (double)j + f.a[1] * (double)i + f.a[2];
    const double row = f.a[3] * (double)j + f.a[4] * (double)i + f.a[5];
    const double fc = floor(col), fr = floor(row);
    double v00 = 0.0, v01 = 0.0, v10 = 0.0, v11 = 0.0;
    if (fc >= -1.0 && fc <= (double)nx && fr >= -1.0 && fr <= (double)ny) {
        const int c0 = (int)fc, r0 = (int)fr;
        const bool cl = c0 >= 0 && c0 < nx, ch = c0 + 1 >= 0 && c0 + 1 < nx;
        if (r0 >= 0 && r0 < ny) {
            if (cl) v00 = (double)__ldg(mask + (size_t)r0 * nx + c0);
            if (ch) v01 = (double)__ldg(mask + (size_t)r0 * nx + c0 + 1);
        }
        if (r0 + 1 >= 0 && r0 + 1 < ny) {
            if (cl) v10 = (double)__ldg(mask + (size_t)(r0 + 1) * nx + c0);
            if (ch) v11 = (double)__ldg(mask + (size_t)(r0 + 1) * nx + c0 + 1);
        }
    }
    const double fx = col - fc, fy = row - fr;
    const double mu = (1.0 - fy) * ((1.0 - fx) * v00 + fx * v01) + fy * ((1.0 - fx) * v10 + fx * v11);
    core[q] = mu >= threshold ? 1 : 0;
}

// Steps 2-3 as pixel classes: the ring is the 4-neighbour dilation of the core minus the core, and a ring pixel's
// restored value averages, over the directions whose P1 is core, 2*phi[P1] - phi[P2] (P2 core) or phi[P1].  Pixels
// beyond the halo grid are not core.
__global__ void __launch_bounds__(256) repair_code_kernel(const unsigned char *__restrict__ core, int M, unsigned short *__restrict__ code)
{
    const int P = M + 2;
    const int q = blockIdx.x * 256 + threadIdx.x;
    if (q >= P * P) return;
    const int i = q / P, j = q - i * P;
    if (core[q]) { code[q] = (unsigned short)kRepairCore; return; }
    const int di[4] = {0, 0, 1, -1}, dj[4] = {1, -1, 0, 0};
    int c = 0;
#pragma unroll
    for (int d = 0; d < 4; ++d) {
        const int i1 = i + di[d], j1 = j + dj[d], i2 = i + 2 * di[d], j2 = j + 2 * dj[d];
        if (i1 < 0 || i1 >= P || j1 < 0 || j1 >= P || !core[i1 * P + j1]) continue;
        c |= 1 << (kRepairP1Shift + d);
        if (i2 >= 0 && i2 < P && j2 >= 0 && j2 < P && core[i2 * P + j2]) c |= 1 << (kRepairP2Shift + d);
    }
    code[q] = (unsigned short)c;
}

// The reduction weights over the core (R22) and the subapertures that may keep the edge-sum path: one CTA per
// subaperture.  wmap_in = 0.5*P/W_S, so 0.5*P*core / sum_S(P*core) = 0.5 * wmap_in*core / sum_S(wmap_in*core).
__global__ void __launch_bounds__(128) repair_weights_kernel(const unsigned char *__restrict__ core, int n_subap, int n_pix,
                                                             const float *__restrict__ wmap_in, const int *__restrict__ rows_in,
                                                             float *__restrict__ wmap_out, int *__restrict__ rows_out)
{
    __shared__ double part[4];
    __shared__ int bad[4];
    const int s = blockIdx.x, a = s / n_subap, b = s - a * n_subap;
    const int M = n_subap * n_pix, P = M + 2, n = n_pix * n_pix;
    const int row_in = rows_in[s];
    double acc = 0.0;
    int notcore = 0;
    for (int e = threadIdx.x; e < n; e += 128) {
        const int r = e / n_pix, c = e - r * n_pix;
        const int i = a * n_pix + r, j = b * n_pix + c;
        const bool co = core[(i + 1) * P + (j + 1)] != 0;
        if (co) acc += (double)wmap_in[(size_t)i * M + j];
        notcore |= !co;
    }
    // the pixels the edge sums read beside the subaperture: one row above and below, one column left and right
    for (int e = threadIdx.x; e < 4 * n_pix; e += 128) {
        const int side = e / n_pix, t = e - side * n_pix;
        const int i = side == 0 ? a * n_pix - 1 : (side == 1 ? (a + 1) * n_pix : a * n_pix + t);
        const int j = side == 2 ? b * n_pix - 1 : (side == 3 ? (b + 1) * n_pix : b * n_pix + t);
        notcore |= core[(i + 1) * P + (j + 1)] == 0;
    }
    for (int o = 16; o > 0; o >>= 1) {
        acc += __shfl_xor_sync(0xffffffffu, acc, o);
        notcore |= __shfl_xor_sync(0xffffffffu, notcore, o);
    }
    if ((threadIdx.x & 31) == 0) { part[threadIdx.x >> 5] = acc; bad[threadIdx.x >> 5] = notcore; }
    __syncthreads();
    const double total = part[0] + part[1] + part[2] + part[3];
    if (threadIdx.x == 0) {
        int r = row_in;
        if (r >= 0 && (bad[0] | bad[1] | bad[2] | bad[3])) r |= kSubapGeneral;
        rows_out[s] = r;
    }
    const bool ok = row_in >= 0 && total > 0.0;
    for (int e = threadIdx.x; e < n; e += 128) {
        const int r = e / n_pix, c = e - r * n_pix;
        const int i = a * n_pix + r, j = b * n_pix + c;
        const size_t at = (size_t)i * M + j;
        const bool co = core[(i + 1) * P + (j + 1)] != 0;
        wmap_out[at] = (ok && co) ? (float)(0.5 * (double)wmap_in[at] / total) : 0.0f;
    }
}

// one CTA per mode: tight non-zero extent (x0,y0,x1,y1) and, if asked for, the diagonal extents
// (min x+y, max x+y, min x-y, max x-y) of the non-zero pixels: together the support's bounding octagon
__global__ void __launch_bounds__(256) bbox_kernel(const float *__restrict__ cube, int ny, int nx,
                                                   int *__restrict__ bbox, int *__restrict__ diag)
{
    const float4 *img = reinterpret_cast<const float4 *>(cube + (size_t)blockIdx.x * ny * nx);
    const int nx4 = nx >> 2, n4 = ny * nx4;
    const int big = 0x3fffffff;
    int lo[4] = {big, big, big, big};      // x0, y0, min x+y, min x-y
    int hi[4] = {-big, -big, -big, -big};  // x1, y1, max x+y, max x-y
    for (int e = threadIdx.x; e < n4; e += 256) {
        const float4 v = __ldg(img + e);
        if (v.x != 0.f || v.y != 0.f || v.z != 0.f || v.w != 0.f) {
            const int r = e / nx4, c = (e - r * nx4) << 2;
            const int l = v.x != 0.f ? 0 : (v.y != 0.f ? 1 : (v.z != 0.f ? 2 : 3));
            const int h = v.w != 0.f ? 3 : (v.z != 0.f ? 2 : (v.y != 0.f ? 1 : 0));
            // within one row x+y and x-y are both extreme at the first / last non-zero pixel
            lo[0] = min(lo[0], c + l); hi[0] = max(hi[0], c + h); lo[1] = min(lo[1], r); hi[1] = max(hi[1], r);
            lo[2] = min(lo[2], c + l + r); hi[2] = max(hi[2], c + h + r);
            lo[3] = min(lo[3], c + l - r); hi[3] = max(hi[3], c + h - r);
        }
    }
    __shared__ int sh[8][8];
#pragma unroll
    for (int q = 0; q < 4; ++q) {
        for (int o = 16; o > 0; o >>= 1) {
            lo[q] = min(lo[q], __shfl_xor_sync(0xffffffffu, lo[q], o));
            hi[q] = max(hi[q], __shfl_xor_sync(0xffffffffu, hi[q], o));
        }
        if ((threadIdx.x & 31) == 0) { sh[threadIdx.x >> 5][q] = lo[q]; sh[threadIdx.x >> 5][4 + q] = hi[q]; }
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        for (int k = 1; k < 8; ++k)
            for (int q = 0; q < 4; ++q) { lo[q] = min(lo[q], sh[k][q]); hi[q] = max(hi[q], sh[k][4 + q]); }
        const bool none = hi[0] < 0;
        reinterpret_cast<int4 *>(bbox)[blockIdx.x] = none ? make_int4(0, 0, -1, -1) : make_int4(lo[0], lo[1], hi[0], hi[1]);
        if (diag) reinterpret_cast<int4 *>(diag)[blockIdx.x] = none ? make_int4(0, -1, 0, -1) : make_int4(lo[2], hi[2], lo[3], hi[3]);
    }
}

__global__ void __launch_bounds__(256) bbox_extent_kernel(const int *__restrict__ bbox, int n_modes, int *wh)
{
    int w = 0, h = 0;
    for (int m = threadIdx.x; m < n_modes; m += 256) {
        const int4 b = __ldg(reinterpret_cast<const int4 *>(bbox) + m);
        w = max(w, b.z - b.x + 1); h = max(h, b.w - b.y + 1);
    }
    for (int o = 16; o > 0; o >>= 1) {
        w = max(w, __shfl_xor_sync(0xffffffffu, w, o)); h = max(h, __shfl_xor_sync(0xffffffffu, h, o));
    }
    __shared__ int sh[8][2];
    if ((threadIdx.x & 31) == 0) { sh[threadIdx.x >> 5][0] = w; sh[threadIdx.x >> 5][1] = h; }
    __syncthreads();
    if (threadIdx.x == 0) {
        for (int k = 1; k < 8; ++k) { w = max(w, sh[k][0]); h = max(h, sh[k][1]); }
        wh[0] = w; wh[1] = h;
    }
}

}  // namespace

static std::atomic<long long> g_launches{0};
void note_launch() { g_launches.fetch_add(1, std::memory_order_relaxed); }
long long launches_so_far() { return g_launches.load(std::memory_order_relaxed); }

size_t max_dynamic_smem()
{
    int dev = 0, v = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return 0;
    if (cudaDeviceGetAttribute(&v, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev) != cudaSuccess) return 0;
    return (size_t)v;
}

cudaError_t launch_subap_weights(const float *d_pupil, const uint8_t *d_valid, int n_subap, int n_pix,
                                 float *d_wmap, int *d_subap_row, int *d_error_flag, cudaStream_t stream)
{
    note_launch();
    subap_weights_kernel<<<n_subap * n_subap, 128, 0, stream>>>(d_pupil, d_valid, n_subap, n_pix, d_wmap, d_subap_row,
                                                                d_error_flag);
    return cudaGetLastError();
}

cudaError_t launch_gtilt_maps(const float *d_pupil, const uint8_t *d_valid, int n_subap, int n_pix, float *d_gx, float *d_gy,
                              cudaStream_t stream)
{
    note_launch();
    gtilt_maps_kernel<<<n_subap * n_subap, 128, 0, stream>>>(d_pupil, d_valid, n_subap, n_pix, d_gx, d_gy);
    return cudaGetLastError();
}

cudaError_t launch_compute_bboxes(const float *d_cube, int n_modes, int ny, int nx, int *d_bbox, int *d_diag,
                                  cudaStream_t stream)
{
    if (n_modes <= 0) return cudaSuccess;
    note_launch();
    bbox_kernel<<<n_modes, 256, 0, stream>>>(d_cube, ny, nx, d_bbox, d_diag);
    return cudaGetLastError();
}

cudaError_t launch_repair_maps(const float *d_mask, int ny, int nx, const double *fwd, double threshold, int n_subap, int n_pix,
                               const float *wmap_in, const int *rows_in, unsigned char *core, unsigned short *rcode,
                               float *wmap_out, int *rows_out, cudaStream_t stream)
{
    const int M = n_subap * n_pix, np = (M + 2) * (M + 2);
    Fwd6 f;
    for (int k = 0; k < 6; ++k) f.a[k] = fwd[k];
    note_launch();
    repair_core_kernel<<<(np + 255) / 256, 256, 0, stream>>>(d_mask, ny, nx, f, threshold, M, core);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return e;
    note_launch();
    repair_code_kernel<<<(np + 255) / 256, 256, 0, stream>>>(core, M, rcode);
    e = cudaGetLastError();
    if (e != cudaSuccess) return e;
    note_launch();
    repair_weights_kernel<<<n_subap * n_subap, 128, 0, stream>>>(core, n_subap, n_pix, wmap_in, rows_in, wmap_out, rows_out);
    return cudaGetLastError();
}

cudaError_t launch_bbox_extent(const int *d_bbox, int n_modes, int *d_wh, cudaStream_t stream)
{
    note_launch();
    bbox_extent_kernel<<<1, 256, 0, stream>>>(d_bbox, n_modes, d_wh);
    return cudaGetLastError();
}

}  // namespace synim
