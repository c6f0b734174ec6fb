// synim_strip.cu -- the compact-support ("zonal") interaction-matrix kernel for sm_100a.
//
// One CTA per mode.  The mode's support (its bbox plus the one-pixel ring a bilinear sample can still
// touch) is staged ONCE in shared memory by a TMA 3-D box load (cp.async.bulk.tensor, out-of-range
// elements zero-filled by the hardware = reading R4) and reused by every sensor of the batch
// (the cube is fetched once for all WFS).  While the load is in flight the CTA streams
// the zeros of its whole IM column (S4).  Then each warp takes "strips": 30 WFS pixel columns (one
// per lane, plus one halo column on either side) of one sensor's footprint, and walks down the pixel
// rows keeping phi of the previous two rows in registers:
//   S1  col/row = tile-local float32 offsets from a float64 per-lane base,
//   S2  4 LDS + 3 lerps from the staged patch,
//   S3  D_y from registers, D_x from the two neighbouring lanes (shuffles), weighted by the
//       precomputed 0.5*P/W_S map, summed down the rows of a subaperture in registers and across
//       its columns with a segmented warp-shuffle reduction,
//   S4  one float add into the (already zeroed) column per (subaperture, axis).
// Rows of a strip that cannot touch the support are never sampled (exact: phi is 0 there, R15).
// phi is never written anywhere.
#include "synim_device.h"

#include <cstring>
#include <cuda.h>   // CUtensorMap (type only; the encoder is fetched at run time, no libcuda link)

namespace synim {

namespace {

constexpr int kStripThreads = 128;
constexpr int kStripCols = 30;               // D columns per strip: lanes 1..30, halo on lanes 0 and 31
constexpr float kMagicFloor = 12582912.0f;   // 1.5 * 2^23
constexpr int kMagicFloorBits = 0x4B400000;
constexpr unsigned kFull = 0xffffffffu;

__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint64_t *bar, int count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void fence_barrier_init() { asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory"); }
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }
__device__ __forceinline__ void mbar_expect_tx(uint64_t *bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ bool mbar_try_wait(uint64_t *bar, uint32_t parity)
{
    uint32_t ok;
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
        "selp.u32 %0, 1, 0, p;\n\t}"
        : "=r"(ok)
        : "r"(smem_u32(bar)), "r"(parity)
        : "memory");
    return ok != 0;
}
// Bounded wait: a lost transaction becomes a trap (launch error), never a hung GPU.
__device__ __forceinline__ void mbar_wait(uint64_t *bar, uint32_t parity)
{
#pragma unroll 1
    for (int spin = 0; spin < (1 << 24); ++spin)
        if (mbar_try_wait(bar, parity)) return;
    __trap();
}
__device__ __forceinline__ void tma_load_box(void *dst, const CUtensorMap *map, uint64_t *bar, int x, int y, int z)
{
    asm volatile(
        "cp.async.bulk.tensor.3d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5}], [%2];"
        ::"r"(smem_u32(dst)), "l"(map), "r"(smem_u32(bar)), "r"(x), "r"(y), "r"(z)
        : "memory");
}

__device__ __forceinline__ float lds_f32(uint32_t addr)
{
    float v;
    asm volatile("ld.shared.f32 %0, [%1];" : "=f"(v) : "r"(addr));
    return v;
}

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
#pragma unroll 4
    for (int t = tid; t < nv; t += NT) v[t] = z;
    const int done = head + (nv << 2);
    if (tid < n - done) dst[done + tid] = 0.0f;
}

struct PatchBox {
    int x0, y0, w, h;   // absolute source origin of the staged box; extent that may be sampled
};

// One strip: D columns jA .. jA+nC-1 (lanes 1..nC), D rows i0 .. i1 of sensor W.
__device__ __forceinline__ void process_strip(const WfsDev &W, int i0, int i1, int jA, int nC, const PatchBox &pa,
                                              const float *__restrict__ patch, int pitch, float *__restrict__ colp)
{
    const int lane = threadIdx.x & 31;
    const int nR = i1 - i0 + 1;   // D rows; phi row rr (0 .. nR+1) is absolute row i0-1+rr
    const int jcol = jA - 1 + lane;

    // S1: float64 per-lane base, then float32 tile-local offsets
    const double jl = (double)jcol, ib = (double)(i0 - 1);
    const float bc = (float)(W.fwd[0] * jl + W.fwd[1] * ib + W.fwd[2] - (double)pa.x0);
    const float br = (float)(W.fwd[3] * jl + W.fwd[4] * ib + W.fwd[5] - (double)pa.y0);
    const float a1 = (float)W.fwd[1], a4 = (float)W.fwd[4];

    // phi rows whose pixel segment [lane 0 .. lane nC+1] can reach the box (a sample is non-zero only
    // if 0 <= col < w-1 and 0 <= row < h-1); every sample of a row lies between its two end points
    const float bcL = __shfl_sync(kFull, bc, 0), brL = __shfl_sync(kFull, br, 0);
    const float bcR = __shfl_sync(kFull, bc, nC + 1), brR = __shfl_sync(kFull, br, nC + 1);
    const float cw1 = (float)(pa.w - 1) + 0.01f, ch1 = (float)(pa.h - 1) + 0.01f;
    int first = 0x7fffffff, last = -1;
    for (int g = 0; g < nR + 2; g += 32) {
        const int rr = g + lane;
        const float rf = (float)rr;
        const float cl = fmaf(a1, rf, bcL), cr = fmaf(a1, rf, bcR);
        const float rl = fmaf(a4, rf, brL), rq = fmaf(a4, rf, brR);
        const bool act = rr < nR + 2 && fmaxf(cl, cr) > -0.01f && fminf(cl, cr) < cw1 && fmaxf(rl, rq) > -0.01f &&
                         fminf(rl, rq) < ch1;
        const unsigned m = __ballot_sync(kFull, act);
        if (m) {
            first = min(first, g + __ffs(m) - 1);
            last = g + 31 - __clz(m);
        }
    }
    if (last < 0) return;
    const int d_lo = max(first - 1, 1), d_hi = min(last + 1, nR);   // D rows that can be non-zero
    if (d_hi < d_lo) return;

    // segments of lanes that belong to one subaperture column
    const int npx = W.n_pix;
    const bool isD = lane >= 1 && lane <= nC;
    const int seg = isD ? jcol / npx : -1;
    const int segL = __shfl_up_sync(kFull, seg, 1);
    const bool head = isD && (lane == 1 || segL != seg);
    unsigned okm = 0;
    int nsteps = 0;
    while ((1 << nsteps) < min(npx, kStripCols)) ++nsteps;
    for (int s = 0; s < 5; ++s) {
        const int sd = __shfl_down_sync(kFull, seg, 1 << s);
        if (isD && lane + (1 << s) < 32 && sd == seg) okm |= 1u << s;
    }

    const unsigned cmax = (unsigned)(pa.w - 1), rmax = (unsigned)(pa.h - 1);
    const int i_first = i0 - 1 + d_lo;           // absolute row of D row d_lo
    int a_cur = i_first / npx;
    int rem = i_first - a_cur * npx;
    const int M = W.M;
    const float *wp = W.wmap + ((size_t)i_first * M + (isD ? jcol : 0));
    uint32_t pbase;   // volatile: keeps the shared-window address in a register instead of re-deriving it per row
    asm volatile("{\n\t.reg .u64 t;\n\tcvta.to.shared.u64 t, %1;\n\tcvt.u32.u64 %0, t;\n\t}" : "=r"(pbase) : "l"(patch));
    const uint32_t pitch4 = (uint32_t)pitch * 4u;

    // S2: bilinear gather of phi row rr from the staged patch (0 outside it)
    auto sample = [&](int rr) -> float {
        const float rf = (float)rr;
        const float col = fmaf(a1, rf, bc), row = fmaf(a4, rf, br);
        const float tc = __fadd_rd(col, kMagicFloor), tr = __fadd_rd(row, kMagicFloor);
        const int c0 = __float_as_int(tc) - kMagicFloorBits, r0 = __float_as_int(tr) - kMagicFloorBits;
        const float fx = col - (tc - kMagicFloor), fy = row - (tr - kMagicFloor);
        const bool inb = (unsigned)c0 < cmax && (unsigned)r0 < rmax;
        const uint32_t at = inb ? pbase + (uint32_t)(r0 * pitch + c0) * 4u : pbase;
        const float v00 = lds_f32(at), v01 = lds_f32(at + 4u), v10 = lds_f32(at + pitch4), v11 = lds_f32(at + pitch4 + 4u);
        const float top = fmaf(fx, v01 - v00, v00);
        const float bot = fmaf(fx, v11 - v10, v10);
        return inb ? fmaf(fy, bot - top, top) : 0.0f;
    };

    float pm2 = sample(d_lo - 1), pm1 = sample(d_lo), sx = 0.0f, sy = 0.0f;
#pragma unroll 1
    for (int rr = d_lo + 1; rr <= d_hi + 1; ++rr) {
        const float cur = sample(rr);
        // S3: D row d = rr-1: D_y = phi[d+1]-phi[d-1] from registers, D_x from the neighbouring lanes
        const float wgt = isD ? __ldg(wp) : 0.0f;
        wp += M;
        const float dy = cur - pm2;
        const float dx = __shfl_down_sync(kFull, pm1, 1) - __shfl_up_sync(kFull, pm1, 1);
        sx = fmaf(wgt, dx, sx);
        sy = fmaf(wgt, dy, sy);
        pm2 = pm1;
        pm1 = cur;
        ++rem;
        if (rem == npx || rr == d_hi + 1) {
            for (int s = 0; s < nsteps; ++s) {
                const float tx = __shfl_down_sync(kFull, sx, 1 << s), ty = __shfl_down_sync(kFull, sy, 1 << s);
                if ((okm >> s) & 1u) { sx += tx; sy += ty; }
            }
            if (head && (sx != 0.0f || sy != 0.0f)) {
                const int k = __ldg(W.subap_row + a_cur * W.n_subap + seg);
                if (k >= 0) {
                    atomicAdd(colp + W.row_x + k, sx * W.scale);   // S4 (result unused: RED)
                    atomicAdd(colp + W.row_y + k, sy * W.scale);
                }
            }
            sx = 0.0f; sy = 0.0f; rem = 0; ++a_cur;
        }
    }
}

__global__ void __launch_bounds__(kStripThreads) synim_strip_kernel(const __grid_constant__ ImParams p,
                                                                    const __grid_constant__ CUtensorMap tmap)
{
    extern __shared__ __align__(128) float patch[];
    __shared__ __align__(8) uint64_t bar;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    constexpr int nwarps = kStripThreads / 32;
    const int mode = blockIdx.x;
    float *colp = p.out + (long long)mode * p.ld;

    const int4 b = __ldg(reinterpret_cast<const int4 *>(p.bbox) + mode);
    const int bx0 = max(b.x, 0), by0 = max(b.y, 0), bx1 = min(b.z, p.nx - 1), by1 = min(b.w, p.ny - 1);
    const bool empty = bx1 < bx0 || by1 < by0;

    // pieces of the support that fit the staged box (one piece unless the bbox hint was too small)
    // (the box must start on a 16-byte boundary of the source row: up to 3 columns of slack on the left)
    const int cap_w = p.patch_pitch - 5, cap_h = p.patch_h - 2;
    const int npcx = empty ? 0 : (bx1 - bx0 + cap_w) / cap_w, npcy = empty ? 0 : (by1 - by0 + cap_h) / cap_h;
    const int npieces = npcx * npcy;
    const uint32_t box_bytes = (uint32_t)(p.patch_pitch * p.patch_h) * 4u;

    if (tid == 0 && npieces > 0) {
        mbar_init(&bar, 1);
        fence_barrier_init();
        fence_proxy_async();
        mbar_expect_tx(&bar, box_bytes);
        tma_load_box(patch, &tmap, &bar, (bx0 - 1) & ~3, by0 - 1, mode);
    }
    if (p.zero_count > 0) zero_fill<kStripThreads>(colp + p.zero_begin, p.zero_count);
    __syncthreads();   // barrier initialised; this CTA's zeros are ordered before its accumulations
    uint32_t parity = 0;

    for (int pc = 0; pc < npieces; ++pc) {
        const int pcy = pc / npcx, pcx = pc - pcy * npcx;
        const int qx0 = bx0 + pcx * cap_w, qx1 = min(qx0 + cap_w - 1, bx1);
        const int qy0 = by0 + pcy * cap_h, qy1 = min(qy0 + cap_h - 1, by1);
        PatchBox pa;
        pa.x0 = (qx0 - 1) & ~3; pa.y0 = qy0 - 1; pa.w = qx1 + 2 - pa.x0; pa.h = qy1 - qy0 + 3;
        const int slack = qx0 - 1 - pa.x0;   // columns 0..slack are left of the piece
        mbar_wait(&bar, parity);
        parity ^= 1u;
        if (npieces > 1) {
            // by linearity a piece is its own mode: zero outside its box, so clear the ring just staged
            for (int e = tid; e < pa.w; e += kStripThreads) { patch[e] = 0.0f; patch[(pa.h - 1) * p.patch_pitch + e] = 0.0f; }
            for (int e = tid; e < pa.h; e += kStripThreads) {
                for (int c = 0; c <= slack; ++c) patch[e * p.patch_pitch + c] = 0.0f;
                patch[e * p.patch_pitch + pa.w - 1] = 0.0f;
            }
            __syncthreads();
        }

        // lane w: footprint of this piece on sensor w = image of the open box (qx0-1,qx1+1)x(qy0-1,qy1+1)
        // under the inverse map, +-1 pixel for the stencil, clipped to the sensor
        int r_i0 = 0, r_i1 = -1, r_j0 = 0, r_j1 = -1, r_n = 0;
        if (lane < p.n_wfs) {
            const WfsDev &W = p.wfs[lane];
            double jmin = 1e300, jmax = -1e300, imin = 1e300, imax = -1e300;
#pragma unroll
            for (int cr = 0; cr < 4; ++cr) {
                const double c = (cr & 1) ? (double)(qx1 + 1) : (double)(qx0 - 1);
                const double r = (cr & 2) ? (double)(qy1 + 1) : (double)(qy0 - 1);
                const double j = W.inv[0] * c + W.inv[1] * r + W.inv[2];
                const double i = W.inv[3] * c + W.inv[4] * r + W.inv[5];
                jmin = fmin(jmin, j); jmax = fmax(jmax, j); imin = fmin(imin, i); imax = fmax(imax, i);
            }
            const double lim = 1.0e9;
            r_j0 = max(0, (int)floor(fmax(jmin, -lim)) - 1); r_j1 = min(W.M - 1, (int)ceil(fmin(jmax, lim)) + 1);
            r_i0 = max(0, (int)floor(fmax(imin, -lim)) - 1); r_i1 = min(W.M - 1, (int)ceil(fmin(imax, lim)) + 1);
            if (r_j1 >= r_j0 && r_i1 >= r_i0) r_n = (r_j1 - r_j0 + kStripCols) / kStripCols;
        }
        int incl = r_n;
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) {
            const int t = __shfl_up_sync(kFull, incl, d);
            if (lane >= d) incl += t;
        }
        const int total = __shfl_sync(kFull, incl, 31);
        for (int t = warp; t < total; t += nwarps) {
            const int w = __popc(__ballot_sync(kFull, incl <= t));
            const int base = __shfl_sync(kFull, incl - r_n, w);
            const int i0 = __shfl_sync(kFull, r_i0, w), i1 = __shfl_sync(kFull, r_i1, w);
            const int j0 = __shfl_sync(kFull, r_j0, w), j1 = __shfl_sync(kFull, r_j1, w);
            const int jA = j0 + (t - base) * kStripCols;
            const int nC = min(kStripCols, j1 - jA + 1);
            process_strip(p.wfs[w], i0, i1, jA, nC, pa, patch, p.patch_pitch, colp);
        }

        if (pc + 1 < npieces) {
            __syncthreads();   // every warp is done with this piece
            if (tid == 0) {
                const int ny_ = (pc + 1) / npcx, nx_ = (pc + 1) - ny_ * npcx;
                fence_proxy_async();
                mbar_expect_tx(&bar, box_bytes);
                tma_load_box(patch, &tmap, &bar, (bx0 + nx_ * cap_w - 1) & ~3, by0 + ny_ * cap_h - 1, mode);
            }
        }
    }
}

}  // namespace

cudaError_t launch_strip(const ImParams &p, const void *tensor_map, size_t smem_bytes, cudaStream_t stream)
{
    if (p.n_modes <= 0) return cudaSuccess;
    cudaError_t e = cudaFuncSetAttribute(synim_strip_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_bytes);
    if (e != cudaSuccess) return e;
    CUtensorMap tm;
    memcpy(&tm, tensor_map, sizeof(tm));
    synim_strip_kernel<<<(unsigned)p.n_modes, kStripThreads, smem_bytes, stream>>>(p, tm);
    return cudaGetLastError();
}

}  // namespace synim
