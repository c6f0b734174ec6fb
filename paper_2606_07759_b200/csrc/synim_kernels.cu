// synim_kernels.cu -- sm_100a kernels of the synthetic Shack-Hartmann interaction matrix.
//
// One fused launch per call:
//   S1 composite-affine coordinates generated on the fly per WFS pixel,
//   S2 bilinear gather from an influence-function patch staged in shared memory,
//   S3 central differences + weighted subaperture sums with warp shuffles,
//   S4 all (mode, WFS) pairs in the launch, column-major store including the zeros.
// The resampled screen phi lives only in shared memory.
#include "synim_device.h"

namespace synim {

namespace {

constexpr float kMagicFloor = 12582912.0f;   // 1.5 * 2^23: fadd.rm(x, magic) = magic + floor(x), |x| < 2^22
constexpr int kMagicFloorBits = 0x4B400000;
constexpr float kMagicInt = 8388608.0f;      // 2^23: int_as_float(n | bits) - 2^23 = (float)n, 0 <= n < 2^23
constexpr int kMagicIntBits = 0x4B000000;

__device__ __forceinline__ float small_int_to_float(int n)
{
    return __int_as_float(n | kMagicIntBits) - kMagicInt;
}

// floor and fractional part of a tile-local coordinate with full-rate FP32 adds only
__device__ __forceinline__ void floor_frac(float x, int &i, float &f)
{
    const float t = __fadd_rd(x, kMagicFloor);
    i = __float_as_int(t) - kMagicFloorBits;
    f = x - (t - kMagicFloor);
}

// ---- zero fill of one column segment (S4: the zeros are part of the column-major write) --------
template <int NT>
__device__ __forceinline__ void zero_fill(float *dst, int n)
{
    const int tid = threadIdx.x;
    const int mis = (int)((reinterpret_cast<uintptr_t>(dst) >> 2) & 3);
    int head = (4 - mis) & 3;
    if (head > n) head = n;
    if (tid < head) dst[tid] = 0.0f;
    float4 *v = reinterpret_cast<float4 *>(dst + head);
    const int nv = (n - head) >> 2;
    const float4 z = make_float4(0.f, 0.f, 0.f, 0.f);
    for (int t = tid; t < nv; t += NT) v[t] = z;
    const int done = head + (nv << 2);
    if (tid < n - done) dst[done + tid] = 0.0f;
}

// ---- patch staging: rows [py0, py0+ph) x cols [px0, px0+pw) of one mode, zero outside the grid ---
template <int NT>
__device__ __forceinline__ void load_patch(float *patch, int pitch, const float *__restrict__ img, int ny, int nx,
                                           int px0, int py0, int pw, int ph)
{
    const int n = pw * ph;
    const unsigned magic = 0xFFFFFFFFu / (unsigned)pw + 1u;
    for (int e = threadIdx.x; e < n; e += NT) {
        const int r = (int)__umulhi((unsigned)e, magic);
        const int c = e - r * pw;
        const int gx = px0 + c, gy = py0 + r;
        float v = 0.0f;
        if ((unsigned)gx < (unsigned)nx && (unsigned)gy < (unsigned)ny) v = __ldg(img + (size_t)gy * nx + gx);
        patch[r * pitch + c] = v;
    }
}

struct Tile {
    int ti0, ti1, tj0, tj1;   // D pixels, absolute WFS indices, inclusive
};
struct Patch {
    int x0, y0, w, h;         // absolute source origin and extent currently staged
};

// S1 + S2: phi on the tile plus its 1-pixel halo -> shared memory
template <int NT>
__device__ __forceinline__ void resample_tile(const WfsDev &W, const Tile &t, const Patch &pa,
                                              const float *patch, int patch_pitch, float *phi, int phi_pitch)
{
    const int tw2 = t.tj1 - t.tj0 + 3, th2 = t.ti1 - t.ti0 + 3;
    const int n = tw2 * th2;
    // tile base in float64 (absolute coordinates), then tile-local float32 offsets
    const double jb = (double)(t.tj0 - 1), ib = (double)(t.ti0 - 1);
    const float bc = (float)(W.fwd[0] * jb + W.fwd[1] * ib + W.fwd[2] - (double)pa.x0);
    const float br = (float)(W.fwd[3] * jb + W.fwd[4] * ib + W.fwd[5] - (double)pa.y0);
    const float a0 = (float)W.fwd[0], a1 = (float)W.fwd[1], a3 = (float)W.fwd[3], a4 = (float)W.fwd[4];
    const unsigned magic = 0xFFFFFFFFu / (unsigned)tw2 + 1u;
    const unsigned cmax = (unsigned)(pa.w - 1), rmax = (unsigned)(pa.h - 1);
    for (int idx = threadIdx.x; idx < n; idx += NT) {
        const int ii = (int)__umulhi((unsigned)idx, magic);
        const int jj = idx - ii * tw2;
        const float jf = small_int_to_float(jj), yf = small_int_to_float(ii);
        const float col = fmaf(a0, jf, fmaf(a1, yf, bc));
        const float row = fmaf(a3, jf, fmaf(a4, yf, br));
        int c0, r0;
        float fx, fy;
        floor_frac(col, c0, fx);
        floor_frac(row, r0, fy);
        float v = 0.0f;
        if ((unsigned)c0 < cmax && (unsigned)r0 < rmax) {
            const float *q = patch + r0 * patch_pitch + c0;
            const float v00 = q[0], v01 = q[1], v10 = q[patch_pitch], v11 = q[patch_pitch + 1];
            const float top = fmaf(fx, v01 - v00, v00);
            const float bot = fmaf(fx, v11 - v10, v10);
            v = fmaf(fy, bot - top, top);
        }
        phi[ii * phi_pitch + jj] = v;
    }
}

// S3: central differences, weighted sums over the pixels of each subaperture that fall in the tile,
// warp-shuffle reduction over the G lanes that share a subaperture, then accumulate into the column.
template <int NT>
__device__ __forceinline__ void reduce_tile(const WfsDev &W, const Tile &t, const float *phi, int phi_pitch,
                                            float *__restrict__ colp)
{
    const int npx = W.n_pix, G = W.group;
    const int sa0 = t.ti0 / npx, sa1 = t.ti1 / npx, sb0 = t.tj0 / npx, sb1 = t.tj1 / npx;
    const int nsb = sb1 - sb0 + 1, ngroups = (sa1 - sa0 + 1) * nsb;
    const int gl = threadIdx.x & (G - 1);
    const int gshift = 31 - __clz(G);
    const int gpc = NT >> gshift;
    for (int g0 = 0; g0 < ngroups; g0 += gpc) {
        const int gi = g0 + (threadIdx.x >> gshift);
        float sx = 0.0f, sy = 0.0f;
        int k = -1;
        if (gi < ngroups) {
            const int ga = gi / nsb, gb = gi - ga * nsb;
            const int a = sa0 + ga, b = sb0 + gb;
            k = __ldg(W.subap_row + a * W.n_subap + b);
            if (k >= 0) {
                const int jb = max(b * npx, t.tj0), je = min(b * npx + npx - 1, t.tj1);
                const int nq = je - jb + 1;
                for (int r = gl; r < npx; r += G) {
                    const int i = a * npx + r;
                    if (i < t.ti0 || i > t.ti1) continue;
                    const float *prow = phi + (i - t.ti0 + 1) * phi_pitch + (jb - t.tj0 + 1);
                    const float *wrow = W.wmap + (size_t)i * W.M + jb;
                    for (int q = 0; q < nq; ++q) {
                        const float wgt = __ldg(wrow + q);
                        sx = fmaf(wgt, prow[q + 1] - prow[q - 1], sx);
                        sy = fmaf(wgt, prow[q + phi_pitch] - prow[q - phi_pitch], sy);
                    }
                }
            }
        }
        for (int o = G >> 1; o > 0; o >>= 1) {
            sx += __shfl_xor_sync(0xffffffffu, sx, o);
            sy += __shfl_xor_sync(0xffffffffu, sy, o);
        }
        if (gl == 0 && k >= 0) {
            atomicAdd(colp + W.row_x + k, sx * W.scale);
            atomicAdd(colp + W.row_y + k, sy * W.scale);
        }
    }
}

template <int NT>
__global__ void __launch_bounds__(NT) synim_im_kernel(const __grid_constant__ ImParams p)
{
    extern __shared__ __align__(128) float smem[];
    float *patch = smem;
    float *phi = smem + p.patch_pitch * p.patch_h;

    const int mode = blockIdx.x / p.jobs_per_mode;
    const int job = blockIdx.x - mode * p.jobs_per_mode;
    int w_begin = 0, w_end = p.n_wfs, chunk = 0, nchunk = 1;
    if (p.jobs_per_mode > 1) {
        w_begin = job / p.chunks;
        w_end = w_begin + 1;
        chunk = job - w_begin * p.chunks;
        nchunk = p.chunks;
    }
    float *colp = p.out + (long long)mode * p.ld;

    int bx0 = 0, by0 = 0, bx1 = p.nx - 1, by1 = p.ny - 1;
    if (p.bbox != nullptr) {
        const int4 b = __ldg(reinterpret_cast<const int4 *>(p.bbox) + mode);
        bx0 = max(b.x, 0); by0 = max(b.y, 0); bx1 = min(b.z, p.nx - 1); by1 = min(b.w, p.ny - 1);
    }
    if (p.zero_count > 0) zero_fill<NT>(colp + p.zero_begin, p.zero_count);
    if (bx1 < bx0 || by1 < by0) return;

    const float *img = p.cube + (size_t)mode * p.ny * p.nx;
    // the support plus the one-pixel ring of zeros a bilinear sample can still touch
    Patch pa;
    const bool fixed = (bx1 - bx0 + 3 <= p.patch_pitch) && (by1 - by0 + 3 <= p.patch_h);
    if (fixed) {
        pa.x0 = bx0 - 1; pa.y0 = by0 - 1; pa.w = bx1 - bx0 + 3; pa.h = by1 - by0 + 3;
        load_patch<NT>(patch, p.patch_pitch, img, p.ny, p.nx, pa.x0, pa.y0, pa.w, pa.h);
    }
    __syncthreads();   // patch visible; zero fill ordered before this CTA's accumulations

    for (int w = w_begin; w < w_end; ++w) {
        const WfsDev &W = p.wfs[w];
        // WFS pixels whose bilinear footprint can touch the support: image of the open source box
        // (bx0-1, bx1+1) x (by0-1, by1+1) under the inverse map, then +-1 pixel for the stencil
        double jmin = 1e300, jmax = -1e300, imin = 1e300, imax = -1e300;
#pragma unroll
        for (int cr = 0; cr < 4; ++cr) {
            const double c = (cr & 1) ? (double)(bx1 + 1) : (double)(bx0 - 1);
            const double r = (cr & 2) ? (double)(by1 + 1) : (double)(by0 - 1);
            const double j = W.inv[0] * c + W.inv[1] * r + W.inv[2];
            const double i = W.inv[3] * c + W.inv[4] * r + W.inv[5];
            jmin = fmin(jmin, j); jmax = fmax(jmax, j); imin = fmin(imin, i); imax = fmax(imax, i);
        }
        const double lim = 1.0e9;
        const int j_lo = max(0, (int)floor(fmax(jmin, -lim)) - 1), j_hi = min(W.M - 1, (int)ceil(fmin(jmax, lim)) + 1);
        const int i_lo = max(0, (int)floor(fmax(imin, -lim)) - 1), i_hi = min(W.M - 1, (int)ceil(fmin(imax, lim)) + 1);
        if (j_hi < j_lo || i_hi < i_lo) continue;
        const int T = fixed ? W.tile_fixed : W.tile_dense;
        const int ntx = (j_hi - j_lo + T) / T, nty = (i_hi - i_lo + T) / T;
        for (int tt = chunk; tt < ntx * nty; tt += nchunk) {
            const int ty = tt / ntx, tx = tt - ty * ntx;
            Tile t;
            t.tj0 = j_lo + tx * T; t.tj1 = min(t.tj0 + T - 1, j_hi);
            t.ti0 = i_lo + ty * T; t.ti1 = min(t.ti0 + T - 1, i_hi);
            if (!fixed) {
                // source box of this tile's phi rectangle (+1 pixel of slack), clipped to the support
                double cmin = 1e300, cmax = -1e300, rmin = 1e300, rmax = -1e300;
#pragma unroll
                for (int cr = 0; cr < 4; ++cr) {
                    const double j = (cr & 1) ? (double)(t.tj1 + 1) : (double)(t.tj0 - 1);
                    const double i = (cr & 2) ? (double)(t.ti1 + 1) : (double)(t.ti0 - 1);
                    const double c = W.fwd[0] * j + W.fwd[1] * i + W.fwd[2];
                    const double r = W.fwd[3] * j + W.fwd[4] * i + W.fwd[5];
                    cmin = fmin(cmin, c); cmax = fmax(cmax, c); rmin = fmin(rmin, r); rmax = fmax(rmax, r);
                }
                const int x_lo = max((int)floor(fmax(cmin, -lim)) - 1, bx0 - 1);
                const int x_hi = min((int)floor(fmin(cmax, lim)) + 2, bx1 + 1);
                const int y_lo = max((int)floor(fmax(rmin, -lim)) - 1, by0 - 1);
                const int y_hi = min((int)floor(fmin(rmax, lim)) + 2, by1 + 1);
                pa.x0 = x_lo; pa.y0 = y_lo;
                pa.w = min(x_hi - x_lo + 1, p.patch_pitch);
                pa.h = min(y_hi - y_lo + 1, p.patch_h);
                if (pa.w < 2 || pa.h < 2) continue;   // the tile sees nothing of the support (CTA-uniform)
                load_patch<NT>(patch, p.patch_pitch, img, p.ny, p.nx, pa.x0, pa.y0, pa.w, pa.h);
                __syncthreads();
            }
            resample_tile<NT>(W, t, pa, patch, p.patch_pitch, phi, p.phi_pitch);
            __syncthreads();
            reduce_tile<NT>(W, t, phi, p.phi_pitch, colp);
            __syncthreads();
        }
    }
}

// ---- geometry-time kernels ----------------------------------------------------------------------
// one CTA per subaperture: W_S = sum of P, then wmap = 0.5*P/W_S (0 if invalid)
__global__ void __launch_bounds__(128) subap_weights_kernel(const float *__restrict__ pupil,
                                                            const uint8_t *__restrict__ valid, int n_subap,
                                                            int n_pix, float *__restrict__ wmap, int *err)
{
    __shared__ double part[4];
    __shared__ double total;
    const int s = blockIdx.x, a = s / n_subap, b = s - a * n_subap;
    const int M = n_subap * n_pix, n = n_pix * n_pix;
    double acc = 0.0;
    for (int e = threadIdx.x; e < n; e += 128) {
        const int r = e / n_pix, c = e - r * n_pix;
        acc += (double)pupil[(size_t)(a * n_pix + r) * M + b * n_pix + c];
    }
    for (int o = 16; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
    if ((threadIdx.x & 31) == 0) part[threadIdx.x >> 5] = acc;
    __syncthreads();
    if (threadIdx.x == 0) {
        total = part[0] + part[1] + part[2] + part[3];
        if (valid[s] && !(total > 0.0)) atomicExch(err, 1);
    }
    __syncthreads();
    const bool ok = valid[s] && total > 0.0;
    for (int e = threadIdx.x; e < n; e += 128) {
        const int r = e / n_pix, c = e - r * n_pix;
        const size_t at = (size_t)(a * n_pix + r) * M + b * n_pix + c;
        wmap[at] = ok ? (float)(0.5 * (double)pupil[at] / total) : 0.0f;
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

size_t max_dynamic_smem()
{
    int dev = 0, v = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return 0;
    if (cudaDeviceGetAttribute(&v, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev) != cudaSuccess) return 0;
    return (size_t)v;
}

cudaError_t launch_interaction_matrix(const ImParams &p, size_t smem_bytes, cudaStream_t stream)
{
    if (p.n_modes <= 0) return cudaSuccess;
    cudaError_t e = cudaFuncSetAttribute(synim_im_kernel<kThreads>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                         (int)smem_bytes);
    if (e != cudaSuccess) return e;
    const long long grid = (long long)p.n_modes * p.jobs_per_mode;
    if (grid > 0x7fffffffLL) return cudaErrorInvalidConfiguration;
    synim_im_kernel<kThreads><<<(unsigned)grid, kThreads, smem_bytes, stream>>>(p);
    return cudaGetLastError();
}

cudaError_t launch_subap_weights(const float *d_pupil, const uint8_t *d_valid, int n_subap, int n_pix,
                                 float *d_wmap, int *d_error_flag, cudaStream_t stream)
{
    subap_weights_kernel<<<n_subap * n_subap, 128, 0, stream>>>(d_pupil, d_valid, n_subap, n_pix, d_wmap,
                                                                d_error_flag);
    return cudaGetLastError();
}

cudaError_t launch_compute_bboxes(const float *d_cube, int n_modes, int ny, int nx, int *d_bbox, int *d_diag,
                                  cudaStream_t stream)
{
    if (n_modes <= 0) return cudaSuccess;
    bbox_kernel<<<n_modes, 256, 0, stream>>>(d_cube, ny, nx, d_bbox, d_diag);
    return cudaGetLastError();
}

cudaError_t launch_bbox_extent(const int *d_bbox, int n_modes, int *d_wh, cudaStream_t stream)
{
    bbox_extent_kernel<<<1, 256, 0, stream>>>(d_bbox, n_modes, d_wh);
    return cudaGetLastError();
}

}  // namespace synim
