// synim_strip.cu -- the interaction-matrix kernels for sm_100a (S1-S4 of SURVEY.md sec. 8(a)).
//
// Two kernels around one strip walker (process_strip):
//   synim_strip_kernel  compact-support ("zonal") modes: one CTA per mode, all sensors -- described below;
//   synim_tile_kernel   dense (modal) cubes: one CTA per (mode, sensor, tile of the WFS grid), output-stationary --
//                       described above its definition.
// Template flags: kGtilt (the G-tilt estimator instead of the numerical derivative), kAligned (strips hold whole
// subaperture columns; edge-sum path on uniformly lit subapertures), kTile (the strip is a piece of a staged tile),
// kRepair (edge repair) -- see process_strip.
//
// Zonal modes: the mode's support (its bbox plus the one-pixel ring a bilinear sample can still
// touch) is staged ONCE in shared memory by a TMA 3-D box load (cp.async.bulk.tensor, out-of-range
// elements zero-filled by the hardware = reading R4) and reused by every sensor of the batch
// (the cube is fetched once for all WFS).  Each warp then takes "strips": 30 WFS pixel
// columns (one per lane, plus one halo column on either side) of one sensor's footprint -- the image of
// the support's bounding OCTAGON under the inverse map -- and walks down the pixel rows, keeping phi
// of the previous two rows in registers:
//   S1  col/row = tile-local float32 offsets from a float64 per-lane base,
//   S2  floor/fraction with the 1.5*2^23 trick, the shared-memory address straight from the float
//       mantissa, 4 predicated LDS + 3 lerps per sample, branch-free; a sample outside the staged box
//       is 0 (R4, R15),
//   S3  D_y from registers, D_x from the two neighbouring lanes (shuffles), weighted by the
//       precomputed 0.5*P/W_S map, summed down the rows of a subaperture in registers, across its
//       columns with a segmented warp-shuffle reduction, and into a per-CTA shared table of
//       (sensor, subaperture, axis) slopes; on uniformly lit subapertures the sums telescope to the
//       boundary rows and columns (edge-sum path: no stencil, no weights),
//   S4  the column is written once: its zeros by plain 16-byte stores PACED through the sampling loop
//       (one per thread per iteration), then the table's non-zero entries on top.
// Rows of a strip that cannot touch the support are never sampled (exact: phi is 0 there, R15).
// phi is never written anywhere.  A support larger than the staged box (no size hint, > 128 px, or dense
// modes seen by subapertures wider than a strip) is split into pieces whose slopes add up (global RED).
//
// Measured on B200, round 1 (profiles/README.md): FFMA2/FADD2 occupy the issue port for two cycles, so
// packing pixel pairs into f32x2 saves nothing; LDS and SHFL each run at about one warp instruction
// per clock per SM; and dumping a CTA's 161 KB of zeros in one go (plain stores, TMA bulk copies, or
// a warp of its own) delays every load of the SM behind the store data -- hence the pacing.
#include "synim_device.h"

#include <cstring>
#include <cuda.h>   // CUtensorMap (type only; the encoder is fetched at run time, no libcuda link)

namespace synim {

namespace {

// Build parameters (measured on B200: these values are the fastest at config 3)
#ifndef SYNIM_STRIP_WARPS
#define SYNIM_STRIP_WARPS 4    // warps per CTA
#endif
#ifndef SYNIM_STRIP_MINB
#define SYNIM_STRIP_MINB 7     // CTAs per SM the register allocation aims at (72 registers)
#endif
#ifndef SYNIM_STRIP_ROWS
#define SYNIM_STRIP_ROWS 2     // pixel rows per loop iteration (independent samples in flight per lane)
#endif
#ifndef SYNIM_STRIP_UNROLL
#define SYNIM_STRIP_UNROLL 1   // unrolling of the row loop
#endif
#ifndef SYNIM_TILE_PACKED_EDGES
#define SYNIM_TILE_PACKED_EDGES 1    // 0: the tile kernel samples every pixel of an edge-sum unit (comparisons)
#endif
#ifndef SYNIM_TILE_BATCHED_EDGES
#define SYNIM_TILE_BATCHED_EDGES 1   // 0: the tile kernel combines the lanes of every edge-sum unit with shuffles (comparisons)
#endif
#ifndef SYNIM_EDGE_SUM
#define SYNIM_EDGE_SUM 1       // 0: uniformly lit subapertures take the general path too (for comparisons)
#endif
constexpr int kComputeWarps = SYNIM_STRIP_WARPS, kComputeThreads = 32 * kComputeWarps;
constexpr int kStripThreads = kComputeThreads;
constexpr int kStripUnroll = SYNIM_STRIP_UNROLL;
constexpr int kStripRows = SYNIM_STRIP_ROWS;
static_assert(2 * kStripRows <= kWmapPadRows, "weight look-ahead runs past the rows of zeros");
constexpr int kStripCols = kStripMaxCols;     // D columns per strip: lanes 1..30, halo on lanes 0 and 31
constexpr float kMagicFloor = 12582912.0f;   // 1.5 * 2^23: fadd.rm(x, magic) = magic + floor(x), |x| < 2^22
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
    // L2 evict-first: a box is read once.  (Measured, config 3: this hint together with the streaming stores of
    // the column is worth 7 % -- 0.231 -> 0.216 ms; either alone about 1-2 %.)
    asm volatile(
        "{\n\t.reg .b64 pol;\n\tcreatepolicy.fractional.L2::evict_first.b64 pol, 1.0;\n\t"
        "cp.async.bulk.tensor.3d.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1, {%3, %4, %5}], [%2], pol;\n\t}"
        ::"r"(smem_u32(dst)), "l"(map), "r"(smem_u32(bar)), "r"(x), "r"(y), "r"(z)
        : "memory");
}

__device__ __forceinline__ float lds_f32(uint32_t addr)
{
    float v;
    asm volatile("ld.shared.f32 %0, [%1];" : "=f"(v) : "r"(addr));
    return v;
}
__device__ __forceinline__ void cp_async_4(uint32_t dst, const void *src)
{
    asm volatile("cp.async.ca.shared.global [%0], [%1], 4;" ::"r"(dst), "l"(src) : "memory");
}
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_all;" ::: "memory"); }
__device__ __forceinline__ int lds_s32(uint32_t addr)
{
    int v;
    asm volatile("ld.shared.s32 %0, [%1];" : "=r"(v) : "r"(addr));
    return v;
}
__device__ __forceinline__ void red_shared_f32(uint32_t addr, float v)
{
    asm volatile("red.shared.add.f32 [%0], %1;" ::"r"(addr), "f"(v) : "memory");
}
__device__ __forceinline__ void sts_f32(uint32_t addr, float v) { asm volatile("st.shared.f32 [%0], %1;" ::"r"(addr), "f"(v) : "memory"); }
__device__ __forceinline__ void sts_s32(uint32_t addr, int v) { asm volatile("st.shared.s32 [%0], %1;" ::"r"(addr), "r"(v) : "memory"); }
__device__ __forceinline__ void bar_sync(int id, int nthreads) { asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(nthreads) : "memory"); }
template <int NT>
__device__ __forceinline__ void zero_fill(float *dst, int n, int tid)
{
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

// One staged piece.  Cell (r, c) covers source pixels x0+c .. x0+c+1, y0+r .. y0+r+1, where (x0, y0) is
// the upper-left pixel of the piece's ring of zeros; a sample at (col, row) relative to (x0, y0) can be
// non-zero only for 0 <= col < cw, 0 <= row < ch.
struct CellBox {
    int x0, y0;      // absolute source pixel of cell (0, 0)
    int cw, ch;      // cells per row / rows of cells: piece width + 1, piece height + 1
    uint32_t base;   // shared-window byte address of pixel (x0, y0) in the staged box
    int pitch;       // floats per row of the staged box
    float pitchf;    // the same, as float
    uint32_t limit;  // end of the staged box (debug checks only)
    // a sample can be non-zero only for s_lo < col+row < s_hi and d_lo < col-row < d_hi as well (the
    // support's bounding octagon, grown by the reach of a bilinear sample)
    float s_lo, s_hi, d_lo, d_hi;
};

// Everything a strip needs from its sensor, read once from the kernel parameters.
struct StripSensor {
    const float *wmap;    // weights of the x sums: 0.5*P/W_S, or gx
    const float *wmap2;   // weights of the y sums: the same map, or gy
    int M, n_subap, n_pix;
};

// S4, the zeros of the column, paced: every thread owns the 16-byte pieces tid, tid+NT, ... of its CTA's
// column and stores ONE of them per iteration of the sampling loop, so that the column is written at
// the rate the CTA computes.  (Dumping the whole column at the start of the CTA -- plain stores, bulk
// copies, or a warp of its own: all measured -- fills the SM's path to L2, and every load of the other
// warps then waits behind 161 KB of store data.)
struct ZeroPacer {
    float4 *base;    // first 16-byte piece of the column (CTA-uniform)
    uint32_t next;   // the thread's next piece
    uint32_t end;    // number of pieces
    __device__ __forceinline__ void step()
    {
        if (next < end) {
            __stcs(base + next, make_float4(0.0f, 0.0f, 0.0f, 0.0f));   // streaming: the column is not read again
            next += kStripThreads;
        }
    }
    __device__ __forceinline__ bool pending() const { return next < end; }
};

// A weight (or G-tilt coefficient): read-only path, kept in L1 as long as possible.  The maps are the only
// global data the sampling loop reads, and their L1 hits matter; measured at config 3: L1::evict_last and
// plain ld.global.nc 0.215-0.217 ms, bypassing L1 (ld.global.cg) 0.242 ms, L1::no_allocate 0.251 ms.
__device__ __forceinline__ float wld(const float *p)
{
    float v;
    asm volatile("ld.global.nc.L1::evict_last.f32 %0, [%1];" : "=f"(v) : "l"(p));
    return v;
}

// x / n_pix for 0 <= x < 2^15 without the integer-division sequence: magic = ceil(2^32 / n_pix) (exact while
// x * n_pix < 2^32; n_pix = 1 would need 2^32 itself)
__device__ __forceinline__ int div_npx(int x, int npx, unsigned magic) { return npx == 1 ? x : (int)__umulhi((unsigned)x, magic); }

// One strip: D columns jA .. jA+nC-1 (lanes 1..nC), D rows i0 .. i1 of sensor W.
// Its partial slopes go to the CTA's shared table: entry (a, b, axis) of the sensor's window of
// subapertures (first row a0, first column b0, nb columns) sits at tab + ((a-a0)*nb + (b-b0))*8 + axis*4.
//
// kAligned (the sensor's subapertures are at most a strip wide): the strip starts on a subaperture boundary
// and holds whole subaperture columns only, so (a) each table entry is written by exactly one warp, with a
// plain store, and (b) the rows of the strip are cut into SEGMENTS of consecutive "units" (the strip's
// subapertures of one subaperture row) of one kind.  A unit none of whose valid subapertures has unequal
// pixel weights (the row map flags those with kSubapGeneral at geometry time) is an EDGE-SUM unit: with a
// constant weight w = 0.5/n^2 the weighted sum of central differences telescopes,
//     sum_S w*D_x = w * sum_rows (phi[.,j0+n] + phi[.,j0+n-1] - phi[.,j0] - phi[.,j0-1]),
//     sum_S w*D_y = w * sum_cols (phi[i0+n,.] + phi[i0+n-1,.] - phi[i0,.] - phi[i0-1,.]),
// (the identity behind tests/test_oracle_pins.py::test_telescoping_identity_on_full_subapertures), so a pixel
// row costs its sample and ONE add: no stencil shuffles, no weight loads, no multiply; the lanes are combined
// once per subaperture.  The other units (a partially lit subaperture among them) take the general path:
// D_y from registers, D_x from the neighbouring lanes, one weight per pixel.  Each segment primes its own
// two rows of phi, so the two loops share no state but the table.
// kGtilt: the G-tilt estimator (reading R13) instead of the numerical derivative: the slopes are then two
// weighted sums of phi itself (coefficient maps gx, gy: +-1/den on the first / last valid pixel of every
// pixel row / column of a subaperture), so the stencil and its shuffles drop out (general path only).
//
// kTile (dense modes, synim_tile_kernel): the strip is a piece of a tile of the WFS grid whose whole pre-image
// (halo and bilinear reach included) is staged, so (a) no sample can leave the staged box: no range test, no row
// pruning; (b) coordinates are taken relative to the pre-image of the strip's own centre (an integer source pixel
// folded into the address base), which keeps |col|, |row| below ~64 and their float32 spacing below 4e-6 pixels
// however large the box is; (c) a unit none of whose subapertures is valid is SKIPPED (nothing is sampled for it).
// kRepair (edge repair; numerical derivative only): the stencil reads the REPAIRED screen -- phi on
// the strict core, the normalised average of 2*P1-P2 / P1 over the valid cardinal directions on the ring (each P a
// bilinear sample of its own, taken by the lane that needs it), 0 elsewhere -- per the pixel classes W.rcode that
// repair_maps built for this call; W.wmap then holds 0.5*P*core/sum(P*core) and W.subap_row flags as general every
// subaperture that is not core throughout, so the edge-sum path only ever sees unrepaired pixels.
// kWalk: 0 = the classic walk of a footprint (rows pruned to the support, partial units at either end); 1 = kTile;
// 2 = a zonal footprint whose rows were rounded out to whole units (ImParams::unit_rows), so that its edge-sum units can
// take the packed boundary-only path of the tile kernel (opt-in, SYNIM_ZONAL_PACKED=1: not the default until measured).
template <bool kGtilt, bool kAligned, int kWalk, bool kRepair>
__device__ __forceinline__ void process_strip(const WfsDev &W, int i0, int i1, int jA, int nC, const CellBox &cb,
                                              uint32_t addr_bias, uint32_t tab, int a0, int b0, int nb, ZeroPacer &zp,
                                              uint32_t scr = 0u)
{
    constexpr bool kTile = kWalk == 1, kWhole = kWalk != 0;   // kWhole: the walk consists of whole units
    static_assert(!kWhole || kAligned, "whole-unit walks are made of aligned strips");
    static_assert(!kRepair || !kGtilt, "edge repair belongs to the numerical-derivative engine");
    constexpr bool kEdge = kAligned && !kGtilt && SYNIM_EDGE_SUM != 0;   // the edge-sum path exists
    constexpr int kRows = kStripRows;
    static_assert(kRows == 2, "the segment loops are written for two rows per iteration");
    const int lane = threadIdx.x & 31;
    const int nR = i1 - i0 + 1;   // D rows; phi row rr (0 .. nR+1) is absolute row i0-1+rr
    const int jcol = jA - 1 + lane;

    // S1: float64 per-lane base, then float32 tile-local offsets.  (kTile samples without a range test: the lanes
    // beyond the strip's right halo column stay on it, inside the staged pre-image.)
    const double jl = (double)(kTile ? min(jcol, jA + nC) : jcol);
    float bc = (float)(W.fwd[0] * jl + W.fwd[1] * (double)(i0 - 1) + W.fwd[2] - (double)cb.x0);
    float br = (float)(W.fwd[3] * jl + W.fwd[4] * (double)(i0 - 1) + W.fwd[5] - (double)cb.y0);
    // byte address of element 0 minus (bits of the magic number << 2) mod 2^32.  The bias is a kernel
    // parameter, not a literal, so that ptxas keeps the difference in one register and an address is one LEA
    uint32_t cbase = cb.base - addr_bias;
    int roff = 0;   // phi row rr (counted from absolute row i0-1) is sampled at rf = rr - roff
    // kTile: coordinates are re-based every few units on the pre-image of the centre of the rows ahead (an integer
    // source pixel, folded into the address base) and counted from their first row: |col|, |row| and rf stay below
    // ~40, so the float32 roundings of the base, of the product a1*rf and of the sum stay near 2e-6 pixels however
    // tall the strip is.  rr0 .. rr1: the phi rows (counted from i0-1) sampled until the next call.
    // Packed interior samples of edge-sum units (kTile): the telescoped sums need phi on the first and last row of a
    // unit in every column, but on its n-2 interior rows only in the boundary columns of the subapertures (their first
    // and last column, and the strip's two halo columns): ncol = 2*nsb + 2 columns.  Those (n-2)*ncol samples are
    // packed over the lanes, at most two per lane: lane l takes samples q = l and q = 32 + l, sample q being interior
    // row 1 + q / ncol of boundary column q % ncol.  pj / pk: that sample's pixel column and row inside the unit.
    constexpr bool kPacked = kWhole && kEdge && SYNIM_TILE_PACKED_EDGES != 0;
    const int p_nsb = kPacked ? div_npx(nC, W.n_pix, W.npx_magic) : 0, p_ncol = 2 * p_nsb + 2;
    const int p_total = (W.n_pix - 2) * p_ncol;
    const bool packed_ok = kPacked && W.n_pix >= 3 && p_total <= 64;
    int pj[2] = {0, 0}, pk[2] = {0, 0};
    bool pv[2] = {false, false};
    float bcP[2] = {0.f, 0.f}, brP[2] = {0.f, 0.f};
    if (packed_ok) {
#pragma unroll
        for (int s2 = 0; s2 < 2; ++s2) {
            const int q = s2 * 32 + lane;
            pv[s2] = q < p_total;
            const int kr = q / p_ncol, kc = q - kr * p_ncol;
            const int b = (kc - 1) >> 1, side = (kc - 1) & 1;
            const int ln = kc == 0 ? 0 : (kc == p_ncol - 1 ? nC + 1 : 1 + b * W.n_pix + side * (W.n_pix - 1));
            pj[s2] = jA - 1 + ln; pk[s2] = kr + 1;
            if (kWalk == 2) {   // (no re-basing in a zonal walk: relative to the staged box, once per strip)
                const double pjd = (double)pj[s2], pid = (double)(i0 - 1 + pk[s2]);
                bcP[s2] = (float)(W.fwd[0] * pjd + W.fwd[1] * pid + W.fwd[2] - (double)cb.x0);
                brP[s2] = (float)(W.fwd[3] * pjd + W.fwd[4] * pid + W.fwd[5] - (double)cb.y0);
            }
        }
    }
    auto rebase = [&](int rr0, int rr1) {
        const double jm = (double)jA + 0.5 * (double)nC, im = (double)(i0 - 1) + 0.5 * (double)(rr0 + rr1);
        const int xc = __double2int_rn(W.fwd[0] * jm + W.fwd[1] * im + W.fwd[2] - (double)cb.x0);
        const int yc = __double2int_rn(W.fwd[3] * jm + W.fwd[4] * im + W.fwd[5] - (double)cb.y0);
        const double ib = (double)(i0 - 1 + rr0);
        bc = (float)(W.fwd[0] * jl + W.fwd[1] * ib + W.fwd[2] - (double)(cb.x0 + xc));
        br = (float)(W.fwd[3] * jl + W.fwd[4] * ib + W.fwd[5] - (double)(cb.y0 + yc));
        cbase = cb.base + (uint32_t)(yc * cb.pitch + xc) * 4u - addr_bias;
        roff = rr0;
        if (packed_ok) {   // the packed samples' bases: pk rows below the unit's first row (whose rf is passed), column pj
#pragma unroll
            for (int s2 = 0; s2 < 2; ++s2) {
                const double pjd = (double)pj[s2], pid = ib + (double)pk[s2];
                bcP[s2] = (float)(W.fwd[0] * pjd + W.fwd[1] * pid + W.fwd[2] - (double)(cb.x0 + xc));
                brP[s2] = (float)(W.fwd[3] * pjd + W.fwd[4] * pid + W.fwd[5] - (double)(cb.y0 + yc));
            }
        }
    };
    const float a1 = (float)W.fwd[1], a4 = (float)W.fwd[4];
    const float cwf = (float)cb.cw, chf = (float)cb.ch;

    // phi rows whose pixel segment [lane 0 .. lane nC+1] can reach the support's octagon (a sample is
    // non-zero only if 0 <= col < cw, 0 <= row < ch and inside the diagonal limits); every sample of a
    // row lies between its two end points, and each limit is a half-plane
    // (kRepair: a restored pixel reads up to kRepairReach pixels away, along its row or its column)
    const float a0f = (float)W.fwd[0], a3f = (float)W.fwd[3];
    float bcL = __shfl_sync(kFull, bc, 0), brL = __shfl_sync(kFull, br, 0);
    float bcR = __shfl_sync(kFull, bc, nC + 1), brR = __shfl_sync(kFull, br, nC + 1);
    if (kRepair) {
        bcL -= (float)kRepairReach * a0f; brL -= (float)kRepairReach * a3f;
        bcR += (float)kRepairReach * a0f; brR += (float)kRepairReach * a3f;
    }
    int first = 0x7fffffff, last = -1;
    if (kTile) { first = 0; last = nR + 1; }
    for (int g = 0; !kTile && g < nR + 2; g += 32) {
        const int rr = g + lane;
        const float rf = (float)rr;
        const float cl = fmaf(a1, rf, bcL), cr = fmaf(a1, rf, bcR);
        const float rl = fmaf(a4, rf, brL), rq = fmaf(a4, rf, brR);
        const float sl = cl + rl, sr = cr + rq, dl = cl - rl, dr = cr - rq;
        const bool act = rr < nR + 2 && fmaxf(cl, cr) > -0.01f && fminf(cl, cr) < cwf + 0.01f && fmaxf(rl, rq) > -0.01f &&
                         fminf(rl, rq) < chf + 0.01f && fmaxf(sl, sr) > cb.s_lo && fminf(sl, sr) < cb.s_hi &&
                         fmaxf(dl, dr) > cb.d_lo && fminf(dl, dr) < cb.d_hi;
        const unsigned m = __ballot_sync(kFull, act);
        if (m) {
            first = min(first, g + __ffs(m) - 1);
            last = g + 31 - __clz(m);
        }
    }
    if (last < 0) return;
    const int row_reach = kRepair ? 1 + kRepairReach : 1;
    int d_lo = max(first - row_reach, 1), d_hi = min(last + row_reach, nR);   // D rows that can be non-zero
    if (d_hi < d_lo) return;
    if (kWalk == 2) {   // whole units (the footprint starts and ends on unit boundaries; the rows added hold phi = 0)
        d_lo = ((d_lo - 1) / W.n_pix) * W.n_pix + 1;
        d_hi = min(((d_hi + W.n_pix - 1) / W.n_pix) * W.n_pix, nR);
    }

    // segments of lanes that belong to one subaperture column
    const int npx = W.n_pix, n_subap = W.n_subap;
    const bool isD = lane >= 1 && lane <= nC;
    const int seg = isD ? div_npx(jcol, npx, W.npx_magic) : -1;
    const int seg_first = div_npx(jA, npx, W.npx_magic);   // (aligned strips start on a subaperture boundary)
    const int segL = __shfl_up_sync(kFull, seg, 1);
    const bool head = isD && (lane == 1 || segL != seg);
    unsigned okm = 0;
#pragma unroll
    for (int s = 0; s < 5; ++s) {
        const int sd = __shfl_down_sync(kFull, seg, 1 << s);
        if (isD && lane + (1 << s) < 32 && sd == seg) okm |= 1u << s;
    }
    const int nsteps = kAligned ? W.red_steps : 5;   // (warp-uniform) a lane segment is at most n_pix lanes long

    const int i_first = i0 - 1 + d_lo;           // absolute row of D row d_lo
    const int a_first = div_npx(i_first, npx, W.npx_magic);
    int a_cur = a_first;
    int rem = i_first - a_cur * npx;             // rows of subaperture row a_cur already behind us
    const int M = W.M;
    uint32_t tent = tab + (uint32_t)((a_cur - a0) * nb + (isD ? seg - b0 : 0)) * 8u;   // this lane's table entry
    const uint32_t tstep = (uint32_t)nb * 8u;

    // bit u of genmask: unit a_first+u needs the general path (lane u looks at the strip's subapertures of
    // its unit; units beyond 32 are simply taken as general)
    // bit u of skipmask (kTile): none of the strip's subapertures of unit a_first+u is valid
    unsigned genmask = 0xffffffffu, skipmask = 0u;
    if (kEdge || kWhole) {
        const int bA = div_npx(jA, npx, W.npx_magic), nsb = div_npx(nC, npx, W.npx_magic);
        const int a_mine = a_first + lane;
        bool gflag = false, vflag = false;
        if (a_mine < n_subap) {
            const int *rp = W.subap_row + a_mine * n_subap + bA;
            for (int q = 0; q < nsb; ++q)
                if (bA + q < n_subap) {
                    const int c = __ldg(rp + q);
                    gflag = gflag || (c >= 0 && (c & kSubapGeneral) != 0);
                    vflag = vflag || c >= 0;
                }
        }
        if (kEdge) genmask = __ballot_sync(kFull, gflag);
        if (kWhole) skipmask = __ballot_sync(kFull, a_mine < n_subap && !vflag);
        genmask &= ~skipmask;
    }

    // S3 (columns), general path: segmented sum over the lanes of a subaperture, then one shared-memory
    // store (this warp owns the entry) or add (another warp may hold the other columns of this subaperture)
    auto flush_general = [&](float sx, float sy) {
        unsigned m = okm;
        asm volatile("" : "+r"(m));   // keeps the five lane masks out of predicate registers between flushes
#pragma unroll
        for (int s = 0; s < 5; ++s) {   // (a step beyond the segment length has no lane mask set: cheaper than a branch)
            if (kAligned && s >= nsteps) break;
            const float tx = __shfl_down_sync(kFull, sx, 1 << s), ty = __shfl_down_sync(kFull, sy, 1 << s);
            if ((m >> s) & 1u) { sx += tx; sy += ty; }
        }
        if (head && (kAligned || sx != 0.0f || sy != 0.0f) && a_cur < n_subap) {
#ifdef SYNIM_CHECKS
            if (tent < tab || tent + 8u > tab + (uint32_t)W.tab_cap * 4u) __trap();
#endif
            if (kAligned) {
                sts_f32(tent, sx);
                sts_f32(tent + 4u, sy);
            } else {
                red_shared_f32(tent, sx);
                red_shared_f32(tent + 4u, sy);
            }
        }
    };
    // edge-sum path: cs = this lane's column sum of phi over the unit's rows, v = (phi[i0+n] + phi[i0+n-1]) -
    // (phi[i0] + phi[i0-1]) of this lane's column
    const float wu = W.w_uniform;
    auto flush_edges = [&](float cs, float v) {
        const float pr = cs + __shfl_up_sync(kFull, cs, 1);                  // columns j-1 and j
        const float sx = (__shfl_down_sync(kFull, pr, npx) - pr) * wu;       // at the head lane: the two edge pairs
        unsigned m = okm;
        asm volatile("" : "+r"(m));
#pragma unroll
        for (int s = 0; s < 5; ++s) {
            if (s >= nsteps) break;
            const float t = __shfl_down_sync(kFull, v, 1 << s);
            if ((m >> s) & 1u) v += t;
        }
        if (head && a_cur < n_subap) {
#ifdef SYNIM_CHECKS
            if (tent < tab || tent + 8u > tab + (uint32_t)W.tab_cap * 4u) __trap();
#endif
            sts_f32(tent, sx);
            sts_f32(tent + 4u, v * wu);
        }
    };

    // S2: one bilinear sample of phi row rf from the staged pixels; 0 outside them.  Non-negative floats order like
    // their bit patterns and negative ones have the sign bit set, so one unsigned compare per axis
    // tests 0 <= x < limit.  Branch-free (predicated LDS), so that the kRows samples of an iteration
    // overlap: the kernel is latency-bound otherwise (ncu, round 1).
    const uint32_t cw_bits = __float_as_uint(cwf), ch_bits = __float_as_uint(chf);
    const float pitchf = cb.pitchf;
    const uint32_t rpitch4 = (uint32_t)cb.pitch * 4u;
    auto sample_xy = [&](float col, float row) -> float {
        const float tc = __fadd_rd(col, kMagicFloor), tr = __fadd_rd(row, kMagicFloor);   // magic + floor
        const float fx = col - (tc - kMagicFloor), fy = row - (tr - kMagicFloor);
        // magic + c0 + r0*pitch is exact: its mantissa is the element index (a negative index borrows from
        // the mantissa's leading bit: still exact, and the address arithmetic is modulo 2^32)
        const uint32_t idx = __float_as_uint(fmaf(tr - kMagicFloor, pitchf, tc));
        const uint32_t at = idx * 4u + cbase;
        if (kTile) {   // the whole pre-image of the tile is staged: nothing to test
#ifdef SYNIM_CHECKS
            if (at < cb.base || at + rpitch4 + 8u > cb.limit) __trap();
#endif
            const float v00 = lds_f32(at), v01 = lds_f32(at + 4u), v10 = lds_f32(at + rpitch4), v11 = lds_f32(at + rpitch4 + 4u);
            const float t = fmaf(fx, v01 - v00, v00), u = fmaf(fx, v11 - v10, v10);
            return fmaf(fy, u - t, t);
        }
#ifdef SYNIM_CHECKS   // debug build: a sample that passes the range test must lie inside the staged box
        if (__float_as_uint(col) < cw_bits && __float_as_uint(row) < ch_bits &&
            (at < cb.base || at + rpitch4 + 8u > cb.limit)) __trap();
#endif
        float phi;
        asm volatile(
            "{\n\t.reg .pred p;\n\t.reg .f32 v00, v01, v10, v11, t, u;\n\t.reg .b32 at1;\n\t"
            "setp.lt.u32 p, %1, %2;\n\t"
            "setp.lt.and.u32 p, %3, %4, p;\n\t"
            "add.u32 at1, %5, %8;\n\t"
            "@p ld.shared.f32 v00, [%5];\n\t"
            "@p ld.shared.f32 v01, [%5+4];\n\t"
            "@p ld.shared.f32 v10, [at1];\n\t"
            "@p ld.shared.f32 v11, [at1+4];\n\t"
            "sub.rn.f32 t, v01, v00;\n\t"
            "fma.rn.f32 t, %6, t, v00;\n\t"
            "sub.rn.f32 u, v11, v10;\n\t"
            "fma.rn.f32 u, %6, u, v10;\n\t"
            "sub.rn.f32 u, u, t;\n\t"
            "fma.rn.f32 t, %7, u, t;\n\t"
            "selp.f32 %0, t, 0f00000000, p;\n\t}"
            : "=f"(phi)
            : "r"(__float_as_uint(col)), "r"(cw_bits), "r"(__float_as_uint(row)), "r"(ch_bits), "r"(at), "f"(fx), "f"(fy),
              "r"(rpitch4));
        return phi;
    };
    auto sample = [&](float rf) -> float { return sample_xy(fmaf(a1, rf, bc), fmaf(a4, rf, br)); };
    // the repaired screen (kRepair) at phi row rr (counted from i0-1; rf is its float, re-based) of this lane's column
    const int jhalo = (kTile ? min(jcol, jA + nC) : jcol) + 1;   // column on the halo grid, >= 0
    auto sample_r = [&](float rf, int rr) -> float {
        float v = sample(rf);
        if (kRepair) {
            const int irow = i0 + rr;   // row on the halo grid (absolute row i0-1+rr, plus one)
            int code = 0;
            if (irow <= W.M + 1 && jhalo <= W.M + 1) code = (int)__ldg(W.rcode + (size_t)irow * (size_t)(W.M + 2) + jhalo);
            if (!(code & kRepairCore)) {
                v = 0.0f;                              // cleared outside the strict core
                if (code & kRepairRingMask) {          // ring: restored from the core
                    float acc = 0.0f, cnt = 0.0f;
#pragma unroll 1
                    for (int dir = 0; dir < 4; ++dir) {   // +x, -x, +y, -y (rare: one copy of the code is enough)
                        if (!((code >> (kRepairP1Shift + dir)) & 1)) continue;
                        const float sgn = (dir & 1) ? -1.0f : 1.0f;
                        const float dj = dir < 2 ? sgn : 0.0f, di = dir < 2 ? 0.0f : sgn;
                        const float p1 = sample_xy(fmaf(a1, rf + di, fmaf(a0f, dj, bc)), fmaf(a4, rf + di, fmaf(a3f, dj, br)));
                        float est = p1;
                        if ((code >> (kRepairP2Shift + dir)) & 1)
                            est = 2.0f * p1 - sample_xy(fmaf(a1, rf + 2.0f * di, fmaf(a0f, 2.0f * dj, bc)),
                                                        fmaf(a4, rf + 2.0f * di, fmaf(a3f, 2.0f * dj, br)));
                        acc += est; cnt += 1.0f;
                    }
                    v = acc / cnt;
                }
            }
        }
        return v;
    };
#ifdef SYNIM_CHECKS
    const uint32_t wlimit = (uint32_t)(M + kWmapPadRows) * (uint32_t)M;
#define SYNIM_WCHECK(o) do { if ((o) >= wlimit) __trap(); } while (0)
#else
#define SYNIM_WCHECK(o) do { } while (0)
#endif

    int d = d_lo;
    while (d <= d_hi) {
        // the segment: units of one kind from the current one on; D rows d .. d_end
        const int u = a_cur - a_first;
        const bool skip = kWhole && u < 32 && ((skipmask >> u) & 1u);
        const bool gen = !skip && (!kEdge || u >= 32 || ((genmask >> u) & 1u));
        int d_end = d_hi;
        if ((kEdge || kWhole) && u < 32) {
            const unsigned mine = skip ? skipmask : (gen ? genmask : ~(genmask | skipmask));
            const unsigned other = ~mine >> u;   // bit k: unit u+k is of another kind
            if (other) d_end = min(d_hi, (a_cur + __ffs(other) - 1) * npx - i0);   // last D row before that unit
        }
        if (skip) {   // whole units (a tile's strips start and end on unit boundaries): nothing to sample
            const int nu = (d_end - d + 1) / npx;
            a_cur += nu; tent += tstep * (uint32_t)nu;
            d = d_end + 1;
            continue;
        }
        constexpr int kRebaseUnits = 4;   // kTile: units between two re-basings of the coordinates
        const int rebase_rows = kRebaseUnits * npx;
        if (kTile) rebase(d - 1, min(d_end, d - 1 + rebase_rows) + 1);
        float rf = (float)(d + 1 - roff);
        float pmA, pmB;   // phi[d-1], phi[d]
        if (kRepair && gen) { pmA = sample_r((float)(d - 1 - roff), d - 1); pmB = sample_r((float)(d - roff), d); }
        else { pmA = sample((float)(d - 1 - roff)); pmB = sample((float)(d - roff)); }
        if (gen) {
            const float *wm = kGtilt ? W.gx : W.wmap, *wm2 = kGtilt ? W.gy : W.wmap;
            // weight map offsets (elements).  The map has kWmapPadRows rows of zeros below row M-1: halo lanes
            // stay on the first of them (stride 0), and the look-ahead of the last rows may run onto them.
            uint32_t woff = isD ? (uint32_t)(i0 - 1 + d) * (uint32_t)M + (uint32_t)jcol : (uint32_t)M * (uint32_t)M;
            const uint32_t wrow = isD ? (uint32_t)M : 0u, wstride = isD ? (uint32_t)kRows * (uint32_t)M : 0u;
            float wgt[kRows], wg2[kRows];
#pragma unroll
            for (int k = 0; k < kRows; ++k) {
                SYNIM_WCHECK(woff + (uint32_t)k * wrow);
                wgt[k] = wld(wm + (woff + (uint32_t)k * wrow));
                wg2[k] = kGtilt ? wld(wm2 + (woff + (uint32_t)k * wrow)) : wgt[k];
            }
            float sx = 0.0f, sy = 0.0f;
#pragma unroll(kStripUnroll)
            for (; d <= d_end; d += kRows) {
#pragma unroll
                for (int q = 0; q < (kComputeWarps >= 4 ? 1 : 4 / kComputeWarps); ++q) zp.step();
                if (kTile && d + 1 - roff > rebase_rows) {   // (phi[d-1], phi[d] are in registers already)
                    rebase(d + 1, min(d_end, d + rebase_rows) + 2);
                    rf = 0.0f;
                }
                float cur[kRows];   // phi[d+1 .. d+kRows]
#pragma unroll
                for (int k = 0; k < kRows; ++k) cur[k] = kRepair ? sample_r(rf + (float)k, d + 1 + k) : sample(rf + (float)k);
                rf += (float)kRows;
                // D rows d, d+1: D_y from registers, D_x from the neighbouring lanes.  A row past d_hi has D = 0
                // exactly (or a weight from the rows of zeros); a row past d_end is the next segment's.
                const bool two = !(kEdge || kWhole) || d + 1 <= d_end;
#pragma unroll
                for (int k = 0; k < kRows; ++k) {
                    const float mid = k == 0 ? pmB : cur[k - 1];                         // phi[d+k]
                    const float above = k == 0 ? pmA : (k == 1 ? pmB : cur[k - 2]);     // phi[d+k-1]
                    float dx, dy;
                    if (kGtilt) {
                        dx = mid; dy = mid;   // the sums run over phi itself
                    } else {
                        dy = cur[k] - above;
                        dx = __shfl_down_sync(kFull, mid, 1) - __shfl_up_sync(kFull, mid, 1);
                    }
                    if (k == 0 || two) {
                        sx = fmaf(wgt[k], dx, sx); sy = fmaf(wg2[k], dy, sy);
                        if (++rem == npx) { flush_general(sx, sy); sx = 0.0f; sy = 0.0f; rem = 0; ++a_cur; tent += tstep; }
                    }
                }
                pmA = cur[kRows - 2]; pmB = cur[kRows - 1];
                // the weights of the next kRows rows, loaded into the registers just consumed: nothing touches
                // them until the end of the next iteration (a register-to-register copy would wait for the load)
                woff += wstride;
#pragma unroll
                for (int k = 0; k < kRows; ++k) {
                    SYNIM_WCHECK(woff + (uint32_t)k * wrow);
                    wgt[k] = wld(wm + (woff + (uint32_t)k * wrow));
                    wg2[k] = kGtilt ? wld(wm2 + (woff + (uint32_t)k * wrow)) : wgt[k];
                }
            }
            if (rem > 0 && d_end == d_hi) { flush_general(sx, sy); rem = 0; }   // the walk ended inside a unit
        } else if (packed_ok) {
            // Edge-sum units of a tile, boundary samples only (see kPacked above): per unit two full rows (its last row
            // and the next unit's first) and at most two packed samples per lane instead of n full rows.  Parked per
            // unit in the warp's scratch: csp = phi[first row] + phi[last row] of the lane's column, v = the difference
            // of the two row pairs, pk = the packed samples; combined kEdgeBatch units at a time.
            const int nu = (d_end - d + 1) / npx;
            const int nsb = max(p_nsb, 1), ncol = p_ncol;   // (p_nsb >= 1 here; the max keeps dead instantiations quiet)
            constexpr uint32_t kSlot4 = (uint32_t)kEdgeSlotFloats * 4u;
            auto packed_phase2 = [&](int a_start, int cnt) {
                __syncwarp();
                for (int t = lane; t < cnt * nsb; t += 32) {
                    const int uu = t / nsb, sb = t - uu * nsb;
                    const uint32_t base = scr + (uint32_t)uu * kSlot4;
                    const uint32_t c0 = base + (uint32_t)(sb * npx) * 4u, c2 = base + (uint32_t)((sb + 1) * npx) * 4u;
                    float s_lo = lds_f32(c0) + lds_f32(c0 + 4u), s_hi = lds_f32(c2) + lds_f32(c2 + 4u);
                    uint32_t pr = base + (uint32_t)(66 + 2 * sb) * 4u;   // interior row 1, boundary column 2*sb
                    for (int k = 0; k < npx - 2; ++k, pr += (uint32_t)ncol * 4u) {
                        s_lo += lds_f32(pr) + lds_f32(pr + 4u);
                        s_hi += lds_f32(pr + 8u) + lds_f32(pr + 12u);
                    }
                    const uint32_t rv = base + (uint32_t)(33 + 1 + sb * npx) * 4u;
                    float sy = lds_f32(rv);
                    for (int k = 1; k < npx; ++k) sy += lds_f32(rv + (uint32_t)k * 4u);
                    const uint32_t te = tab + (uint32_t)((a_start + uu - a0) * nb + (seg_first - b0) + sb) * 8u;
#ifdef SYNIM_CHECKS
                    if (te < tab || te + 8u > tab + (uint32_t)W.tab_cap * 4u) __trap();
#endif
                    sts_f32(te, (s_hi - s_lo) * wu);
                    sts_f32(te + 4u, sy * wu);
                }
                __syncwarp();
            };
            float pairt = pmA + pmB, carry = pmB;   // phi[i0-1] + phi[i0] and phi[i0] of the current unit
            int slot = 0, a_batch = a_cur;
            int rr = d + 1;   // phi row after the unit's first (counted from i0-1): rf is its re-based float
            for (int uu = 0; uu < nu; ++uu, rr += npx) {
                if (kTile && uu != 0 && (uu & (kRebaseUnits - 1)) == 0) {
                    rebase(rr, min(d_end + 1, rr + rebase_rows));
                    rf = 0.0f;
                }
                if (!kTile) {   // (a zonal CTA paces its column's zeros through this loop: about n/2 iterations' worth)
#pragma unroll
                    for (int q = 0; q < 4; ++q) zp.step();
                }
                const float rfu = rf - 1.0f;   // the unit's first row
                const float fl = sample(rfu + (float)(npx - 1)), fn = sample(rfu + (float)npx);
                float k0 = 0.0f, k1 = 0.0f;
                if (pv[0]) k0 = sample_xy(fmaf(a1, rfu, bcP[0]), fmaf(a4, rfu, brP[0]));
                if (pv[1]) k1 = sample_xy(fmaf(a1, rfu, bcP[1]), fmaf(a4, rfu, brP[1]));
                rf += (float)npx;
                const float pairb = fl + fn;
                const uint32_t sl = scr + (uint32_t)slot * kSlot4 + (uint32_t)lane * 4u;
                sts_f32(sl, carry + fl);
                sts_f32(sl + 33u * 4u, pairb - pairt);
                sts_f32(sl + 66u * 4u, k0);
                sts_f32(sl + 98u * 4u, k1);
                pairt = pairb; carry = fn;
                if (++slot == kEdgeBatch) { packed_phase2(a_batch, slot); a_batch += slot; slot = 0; }
            }
            if (slot) packed_phase2(a_batch, slot);
            a_cur += nu; tent += tstep * (uint32_t)nu;
        } else if (kTile && SYNIM_TILE_BATCHED_EDGES != 0) {
            // Edge-sum units of a tile: whole units, four rows in flight.  Per unit and lane only the column sum cs
            // and the difference v of the two row pairs are formed; they are parked in the warp's scratch
            // ([kEdgeBatch units][33] floats each) and the lanes are combined kEdgeBatch units at a time
            // (edge_phase2): a handful of instructions per unit instead of five shuffle steps.
            const int nu = (d_end - d + 1) / npx;
            const int nsb = div_npx(nC, npx, W.npx_magic);
            auto edge_phase2 = [&](int a_start, int cnt) {
                __syncwarp();
                for (int t = lane; t < cnt * nsb; t += 32) {
                    const int uu = t / nsb, sb = t - uu * nsb;
                    const uint32_t rc = scr + (uint32_t)(uu * 33 + 1 + sb * npx) * 4u;       // cs of the subaperture's first column
                    const uint32_t rv = rc + (uint32_t)(kEdgeBatch * 33) * 4u;               // v of it
                    const uint32_t n4 = (uint32_t)npx * 4u;
                    const float sx = (lds_f32(rc + n4) + lds_f32(rc + n4 - 4u)) - (lds_f32(rc) + lds_f32(rc - 4u));
                    float sy = lds_f32(rv);
                    for (int k = 1; k < npx; ++k) sy += lds_f32(rv + (uint32_t)k * 4u);
                    const uint32_t te = tab + (uint32_t)((a_start + uu - a0) * nb + (seg_first - b0) + sb) * 8u;
#ifdef SYNIM_CHECKS
                    if (te < tab || te + 8u > tab + (uint32_t)W.tab_cap * 4u) __trap();
#endif
                    sts_f32(te, sx * wu);
                    sts_f32(te + 4u, sy * wu);
                }
                __syncwarp();
            };
            float pairt = pmA + pmB, carry = pmB;   // phi[i0-1] + phi[i0] and phi[i0] of the current unit
            int slot = 0, a_batch = a_cur;
            int rr = d + 1;   // next phi row to sample (counted from i0-1)
            for (int uu = 0; uu < nu; ++uu, rr += npx) {
                if (kTile && uu != 0 && (uu & (kRebaseUnits - 1)) == 0) {
                    rebase(rr, min(d_end + 1, rr + rebase_rows));
                    rf = 0.0f;
                }
                // rows i0+1 .. i0+n of the unit (the last one is the next unit's first row)
                float tot = 0.0f, prev = carry, last = carry;
                int k = 0;
                for (; k + 4 <= npx; k += 4) {
                    const float c0 = sample(rf), c1 = sample(rf + 1.0f), c2 = sample(rf + 2.0f), c3 = sample(rf + 3.0f);
                    rf += 4.0f;
                    tot += (c0 + c1) + (c2 + c3);
                    prev = c2; last = c3;
                }
                const int r = npx - k;
                if (r == 3) {
                    const float c0 = sample(rf), c1 = sample(rf + 1.0f), c2 = sample(rf + 2.0f);
                    tot += (c0 + c1) + c2; prev = c1; last = c2;
                } else if (r == 2) {
                    const float c0 = sample(rf), c1 = sample(rf + 1.0f);
                    tot += c0 + c1; prev = c0; last = c1;
                } else if (r == 1) {
                    const float c0 = sample(rf);
                    tot += c0; prev = last; last = c0;
                }
                rf += (float)r;
                const float pairb = prev + last;                      // phi[i0+n-1] + phi[i0+n]
                sts_f32(scr + (uint32_t)(slot * 33 + lane) * 4u, carry + (tot - last));                     // cs
                sts_f32(scr + (uint32_t)((kEdgeBatch + slot) * 33 + lane) * 4u, pairb - pairt);            // v
                pairt = pairb; carry = last;
                if (++slot == kEdgeBatch) { edge_phase2(a_batch, slot); a_batch += slot; slot = 0; }
            }
            if (slot) edge_phase2(a_batch, slot);
            a_cur += nu; tent += tstep * (uint32_t)nu;
        } else {
            float cs = 0.0f;   // sum of phi over the rows of the unit so far
            // phi[i0-1] + phi[i0] of the current unit: both rows lie above the walk (where phi is 0) unless the
            // segment starts on the unit's first row
            float utop = rem == 0 ? pmA + pmB : 0.0f;
            for (; d <= d_end; d += kRows) {
                zp.step();
                const float c0 = sample(rf), c1 = sample(rf + 1.0f);   // phi[d+1], phi[d+2]
                rf += 2.0f;
                cs += pmB;                                            // D row d: phi[d]
                if (++rem == npx) {   // the unit's last row: phi[i0+n-1] = phi[d], phi[i0+n] = phi[d+1]
                    const float ubot = pmB + c0;
                    flush_edges(cs, ubot - utop);
                    utop = ubot; cs = 0.0f; rem = 0; ++a_cur; tent += tstep;
                }
                if (d + 1 <= d_end) {                                 // D row d+1 (else it is the next segment's)
                    cs += c0;
                    if (++rem == npx) {
                        const float ubot = c0 + c1;
                        flush_edges(cs, ubot - utop);
                        utop = ubot; cs = 0.0f; rem = 0; ++a_cur; tent += tstep;
                    }
                }
                pmA = c0; pmB = c1;
            }
            if (rem > 0 && d_end == d_hi) { flush_edges(cs, 0.0f - utop); rem = 0; }   // rows below the walk hold phi = 0
        }
        d = d_end + 1;
    }
}


// Lane w of one warp: footprint of a piece (source pixels qx0..qx1 x qy0..qy1 of a support with diagonal
// extents sg0..sg1, dg0..dg1) on sensor w.  phi(i,j) can be non-zero only strictly inside the image, under
// the inverse map, of the piece's open octagon: the box (qx0-1,qx1+1)x(qy0-1,qy1+1) cut by
// sg0-2 < x+y < sg1+2 and dg0-2 < x-y < dg1+2.  So D(i,j) only for floor(jmin) <= j <= ceil(jmax) (one pixel
// of stencil either side), clipped to the sensor.  Results go to shared memory for the other warps.
template <bool kZPack>
__device__ __forceinline__ void footprint_of_piece(const ImParams &p, int lane, int qx0, int qx1, int qy0, int qy1, int sg0,
                                                   int sg1, int dg0, int dg1, int4 *s_box, int4 *s_win)
{
        int r_i0 = 0, r_i1 = -1, r_j0 = 0, r_j1 = -1, r_a0 = 0, r_b0 = 0, r_na = 0, r_nb = 0;
        const WfsDev &W = p.wfs[lane];
        const double X0 = qx0 - 1, X1 = qx1 + 1, Y0 = qy0 - 1, Y1 = qy1 + 1;
        const double S0 = sg0 - 2, S1 = sg1 + 2, D0 = dg0 - 2, D1 = dg1 + 2;
        double jmin = 1e300, jmax = -1e300, imin = 1e300, imax = -1e300;
        auto vertex = [&](double c, double r) {
            const double j = W.inv[0] * c + W.inv[1] * r + W.inv[2];
            const double i = W.inv[3] * c + W.inv[4] * r + W.inv[5];
            jmin = fmin(jmin, j); jmax = fmax(jmax, j); imin = fmin(imin, i); imax = fmax(imax, i);
        };
        // two vertices on each edge of the box; an edge the diagonals cut away altogether yields two
        // points outside the octagon but inside the box (a superset: still exact)
#pragma unroll
        for (int e = 0; e < 2; ++e) {
            const double X = e ? X1 : X0, Y = e ? Y1 : Y0;
            const double ya = fmax(fmax(Y0, S0 - X), X - D1), yb = fmin(fmin(Y1, S1 - X), X - D0);
            vertex(X, ya); vertex(X, yb);
            const double xa = fmax(fmax(X0, S0 - Y), D0 + Y), xb = fmin(fmin(X1, S1 - Y), D1 + Y);
            vertex(xa, Y); vertex(xb, Y);
        }
        const double lim = 1.0e9;
        // (p.reach: with edge repair a restored pixel carries phi up to kRepairReach pixels further)
        r_j0 = max(0, (int)floor(fmax(jmin, -lim)) - p.reach); r_j1 = min(W.M - 1, (int)ceil(fmin(jmax, lim)) + p.reach);
        r_i0 = max(0, (int)floor(fmax(imin, -lim)) - p.reach); r_i1 = min(W.M - 1, (int)ceil(fmin(imax, lim)) + p.reach);
        int4 win = make_int4(0, 0, 0, 0);
        // A footprint that lies inside ONE subaperture (giant subapertures: config 4's 238-pixel NGS ones) whose pixel
        // weights are all equal, or which is invalid, yields exactly nothing: the weighted sum of central differences
        // telescopes to phi on the subaperture's two boundary column / row pairs (process_strip), where phi is 0 -- the
        // D pixels that can be non-zero are uj0..uj1 x ui0..ui1, so phi vanishes outside uj0+1..uj1-1.  (The G-tilt sums
        // read phi on the first / last valid pixels only: 0 as well.)  The column's zeros are already on their way.
        {
            const double uj0 = floor(fmax(jmin, -lim)) - p.reach, uj1 = ceil(fmin(jmax, lim)) + p.reach;
            const double ui0 = floor(fmax(imin, -lim)) - p.reach, ui1 = ceil(fmin(imax, lim)) + p.reach;
            if (uj0 >= 0.0 && ui0 >= 0.0 && uj1 <= (double)(W.M - 1) && ui1 <= (double)(W.M - 1)) {
                const int sb = (int)uj0 / W.n_pix, sa = (int)ui0 / W.n_pix;
                if ((int)uj1 / W.n_pix == sb && (int)ui1 / W.n_pix == sa) {
                    const int c = __ldg(W.subap_row + sa * W.n_subap + sb);
                    if (c < 0 || (c & kSubapGeneral) == 0) { r_j1 = r_j0 - 1; r_i1 = r_i0 - 1; }
                }
            }
        }
        if (kZPack && W.spb > 0 && r_i1 >= r_i0) {   // whole subaperture rows (the rows added hold phi = 0)
            r_i0 = (r_i0 / W.n_pix) * W.n_pix;
            r_i1 = min(W.M - 1, (r_i1 / W.n_pix + 1) * W.n_pix - 1);
        }
        if (r_j1 >= r_j0 && r_i1 >= r_i0) {
            r_a0 = r_i0 / W.n_pix; r_b0 = r_j0 / W.n_pix;
            r_nb = r_j1 / W.n_pix - r_b0 + 1;
            r_na = r_i1 / W.n_pix - r_a0 + 1;
            win = make_int4(r_a0, r_b0, r_na, r_nb);
            if (win.z * win.w * 2 > W.tab_cap) __trap();   // the host sized the table from the same bounds
        }
        s_box[lane] = make_int4(r_i0, r_i1, r_j0, r_j1);
        s_win[lane] = win;   // also read by scatter_table
}

// All warps, after a barrier: fetch the IM rows of the windows' subapertures (needed only when the table
// is stored: asynchronously, so that the store at the end waits for nothing), then sample the strips of
// every sensor's footprint.
template <bool kGtilt, bool kAligned, bool kRepair, bool kZPack>
__device__ __forceinline__ void sample_footprints(const ImParams &p, int warp, int lane, const int4 *s_box, const int4 *s_win,
                                                  int *s_next_ptr, const CellBox &cb, uint32_t tab_base, uint32_t krow_base,
                                                  ZeroPacer &zp, uint32_t scr)
{
    // kAligned (every sensor of the launch has subapertures that fit a strip, spb > 0): strip t holds the spb
    // subaperture columns b0 + t*spb ... of the footprint's window; otherwise (giant subapertures) strips are
    // kStripCols columns of the footprint, wherever they fall.  (The host never mixes the two in one launch.)
    int r_i0 = 0, r_i1 = -1, r_j0 = 0, r_j1 = -1, r_n = 0, r_a0 = 0, r_b0 = 0, r_nb = 0, r_spb = 0;
    if (lane < p.n_wfs) {
        const int4 fb = s_box[lane], fw = s_win[lane];
        r_i0 = fb.x; r_i1 = fb.y; r_j0 = fb.z; r_j1 = fb.w;
        r_a0 = fw.x; r_b0 = fw.y; r_nb = fw.w;
        r_spb = p.wfs[lane].spb;
        if (r_j1 >= r_j0 && r_i1 >= r_i0) r_n = kAligned ? (r_nb + r_spb - 1) / r_spb : (r_j1 - r_j0 + kStripCols) / kStripCols;
    }
    // the IM rows of the windows' subapertures, needed only when the table is stored: fetched now,
    // asynchronously, so that the store at the end waits for nothing (sensor w by warp w mod 4)
    for (int w = warp; w < p.n_wfs; w += kComputeWarps) {
        const int4 fw = s_win[w];   // a0, b0, na, nb
        const WfsDev &W = p.wfs[w];
        const int n = fw.z * fw.w;
        const unsigned magic = 0xFFFFFFFFu / (unsigned)max(fw.w, 1) + 1u;   // (wraps to 0 for 1)
        for (int e = lane; e < n; e += 32) {
            const int ra = fw.w == 1 ? e : (int)__umulhi((unsigned)e, magic), rb = e - ra * fw.w;
            cp_async_4(krow_base + (uint32_t)((W.tab_off >> 1) + e) * 4u, W.subap_row + (fw.x + ra) * W.n_subap + (fw.y + rb));
        }
    }
    int incl = r_n;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
        const int t = __shfl_up_sync(kFull, incl, d);
        if (lane >= d) incl += t;
    }
    const int total = __shfl_sync(kFull, incl, 31);
    // strips are handed out first come, first served: their costs differ (a strip over the rim of a
    // round support has fewer live rows), and the CTA ends with its slowest warp
    while (true) {
        int t = 0;
        if (lane == 0) t = atomicAdd(s_next_ptr, 1);
        t = __shfl_sync(kFull, t, 0);
        if (t >= total) break;
        const int w = __popc(__ballot_sync(kFull, incl <= t));
        const int base = __shfl_sync(kFull, incl - r_n, w);
        const int i0 = __shfl_sync(kFull, r_i0, w), i1 = __shfl_sync(kFull, r_i1, w);
        const int j0 = __shfl_sync(kFull, r_j0, w), j1 = __shfl_sync(kFull, r_j1, w);
        const int a0 = __shfl_sync(kFull, r_a0, w), b0 = __shfl_sync(kFull, r_b0, w), nb = __shfl_sync(kFull, r_nb, w);
        const int spb = __shfl_sync(kFull, r_spb, w);
        const WfsDev &W = p.wfs[w];
        const uint32_t tab = tab_base + (uint32_t)W.tab_off * 4u;
        if (kAligned) {
            const int bA = b0 + (t - base) * spb;
            process_strip<kGtilt, true, kZPack ? 2 : 0, kRepair>(W, i0, i1, bA * W.n_pix, min(spb, b0 + nb - bA) * W.n_pix, cb, p.addr_bias, tab, a0, b0, nb, zp, scr);
        } else {
            const int jA = j0 + (t - base) * kStripCols;
            process_strip<kGtilt, false, 0, kRepair>(W, i0, i1, jA, min(kStripCols, j1 - jA + 1), cb, p.addr_bias, tab, a0, b0, nb, zp);
        }
    }
}

// The table's non-zero entries -> the IM column (S4).  kAtomic: the support was split into pieces, whose
// contributions add up (linearity); the entries are cleared for the next piece.
template <bool kAtomic, int NT>
__device__ __forceinline__ void scatter_table(const ImParams &p, const int4 *s_win, uint32_t tab_base, uint32_t krow_base,
                                              float *__restrict__ colp, int t0)
{
    for (int w = 0; w < p.n_wfs; ++w) {
        const int4 win = s_win[w];   // a0, b0, na, nb
        const int n = win.z * win.w * 2;
        if (n <= 0) continue;
        const WfsDev &W = p.wfs[w];
        const uint32_t tb = tab_base + (uint32_t)W.tab_off * 4u;
        for (int e = t0; e < n; e += NT) {
            const float v = lds_f32(tb + (uint32_t)e * 4u);
            if (v == 0.0f) continue;
            const int k = lds_s32(krow_base + (uint32_t)((W.tab_off >> 1) + (e >> 1)) * 4u);   // fetched while the strips ran
            if (kAtomic) sts_f32(tb + (uint32_t)e * 4u, 0.0f);
            if (k < 0) continue;
            float *dst = colp + ((e & 1) ? W.row_y : W.row_x) + (k & kSubapRowMask);
            if (kAtomic) {
                atomicAdd(dst, v * W.scale);
            } else {
                __stcs(dst, v * W.scale);
            }
        }
    }
}

template <bool kGtilt, bool kAligned, bool kRepair, bool kZPack>
__global__ void __launch_bounds__(kStripThreads, kRepair ? 4 : (kZPack ? 4 : SYNIM_STRIP_MINB)) synim_strip_kernel(const __grid_constant__ ImParams p,
                                                                                     const __grid_constant__ CUtensorMap tmap)
{
    // [ TMA box: patch_pitch x patch_h floats | table: tab_floats | rows: tab_floats / 2 ints ]
    extern __shared__ __align__(128) float patch[];
    __shared__ __align__(8) uint64_t bar;
    __shared__ int4 s_win[kMaxWfsPerLaunch];   // window of subapertures of each sensor: a0, b0, na, nb
    __shared__ int4 s_box[kMaxWfsPerLaunch];   // footprint of each sensor: i0, i1, j0, j1
    __shared__ int s_next;   // next strip of the current piece
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int mode = blockIdx.x;
    float *colp = p.out + (long long)mode * p.ld;
    const uint32_t raw_base = smem_u32(patch);
    const uint32_t tab_base = raw_base + (uint32_t)(p.patch_pitch * p.patch_h) * 4u;
    const uint32_t krow_base = tab_base + (uint32_t)p.tab_floats * 4u;   // IM row of each (a, b) of the windows
    // (kZPack) per-warp scratch of the packed edge-sum units, behind the rows
    const uint32_t scr = kZPack ? krow_base + (uint32_t)(p.tab_floats >> 1) * 4u + (uint32_t)(warp * (kEdgeBatch * kEdgeSlotFloats)) * 4u : 0u;

    // dense modes (no bboxes): the support is the whole grid, split into pieces; blockIdx.y takes every
    // gridDim.y-th piece, and the pieces' slopes add up in the column, which the host has cleared
    const int chunk = blockIdx.y, nchunk = gridDim.y;
    const int4 b = p.bbox != nullptr ? __ldg(reinterpret_cast<const int4 *>(p.bbox) + mode) : make_int4(0, 0, p.nx - 1, p.ny - 1);
    const int bx0 = max(b.x, 0), by0 = max(b.y, 0), bx1 = min(b.z, p.nx - 1), by1 = min(b.w, p.ny - 1);
    const bool empty = bx1 < bx0 || by1 < by0;
    // a packed cube holds mode m from source pixel org on (org.x is a multiple of 4: the alignment carries over)
    const int2 org = p.origin != nullptr ? __ldg(reinterpret_cast<const int2 *>(p.origin) + mode) : make_int2(0, 0);
    // diagonal extents of the support: min/max of x+y and of x-y over its non-zero pixels (the bbox's own
    // when the caller has none)
    int sg0 = b.x + b.y, sg1 = b.z + b.w, dg0 = b.x - b.w, dg1 = b.z - b.y;
    if (p.diag != nullptr) {
        const int4 dg = __ldg(reinterpret_cast<const int4 *>(p.diag) + mode);
        sg0 = max(sg0, dg.x); sg1 = min(sg1, dg.y); dg0 = max(dg0, dg.z); dg1 = min(dg1, dg.w);
    }

    // pieces of the support that fit the staged box (one piece unless the bbox hint was too small).
    // Box layout: up to 3 columns of slack (the box must start on a 16-byte boundary of the source row),
    // the ring, the piece, the ring.
    const int cap_w = p.patch_pitch - 5, cap_h = p.patch_h - 2;
    const int npcx = empty ? 0 : (bx1 - bx0 + cap_w) / cap_w, npcy = empty ? 0 : (by1 - by0 + cap_h) / cap_h;
    const int npieces = npcx * npcy;
    const bool multi = npieces > 1 || nchunk > 1;
    const uint32_t box_bytes = (uint32_t)(p.patch_pitch * p.patch_h) * 4u;

    if (tid == 0 && chunk < npieces) {
        mbar_init(&bar, 1);
        fence_barrier_init();
        fence_proxy_async();
        mbar_expect_tx(&bar, box_bytes);
        const int fy = chunk / npcx, fx = chunk - fy * npcx;
        tma_load_box(patch, &tmap, &bar, ((bx0 + fx * cap_w - 1) & ~3) - org.x, by0 + fy * cap_h - 1 - org.y, mode);
    }
    for (int e = tid; e < p.tab_floats; e += kStripThreads) sts_f32(tab_base + (uint32_t)e * 4u, 0.0f);
    if (tid < kMaxWfsPerLaunch) s_win[tid] = make_int4(0, 0, 0, 0);
    if (tid == 0) s_next = 0;
    // a split support adds into the column piece by piece: the zeros must be there first
    if (multi && p.zero_count > 0) zero_fill<kStripThreads>(colp + p.zero_begin, p.zero_count, tid);
    __syncthreads();   // mbarrier initialised, table cleared

    ZeroPacer zp;
    zp.base = nullptr; zp.next = 0; zp.end = 0;
    if (!multi && p.zero_count > 0) {
        float *z = colp + p.zero_begin;
        const int mis = (int)((reinterpret_cast<uintptr_t>(z) >> 2) & 3);
        const int headn = min((4 - mis) & 3, p.zero_count);
        const int body = (p.zero_count - headn) >> 2, tailn = p.zero_count - headn - (body << 2);
        if (tid < headn) z[tid] = 0.0f;
        if (tid < tailn) z[headn + (body << 2) + tid] = 0.0f;
        zp.base = reinterpret_cast<float4 *>(z + headn);
        zp.next = (uint32_t)tid; zp.end = (uint32_t)body;
    }
    {
        uint32_t parity = 0;
        for (int pc = chunk; pc < npieces; pc += nchunk) {
            const int pcy = pc / npcx, pcx = pc - pcy * npcx;
            const int qx0 = bx0 + pcx * cap_w, qx1 = min(qx0 + cap_w - 1, bx1);
            const int qy0 = by0 + pcy * cap_h, qy1 = min(qy0 + cap_h - 1, by1);
            const int raw_x0 = (qx0 - 1) & ~3;
            const int slack = qx0 - 1 - raw_x0;   // raw column `slack` is the left ring
            CellBox cb;
            cb.x0 = qx0 - 1; cb.y0 = qy0 - 1; cb.cw = qx1 - qx0 + 2; cb.ch = qy1 - qy0 + 2;
            cb.base = raw_base + (uint32_t)slack * 4u;
            cb.pitch = p.patch_pitch;
            cb.pitchf = p.patch_pitchf;
            cb.limit = raw_base + (uint32_t)(p.patch_pitch * p.patch_h) * 4u;
            cb.s_lo = (float)(sg0 - 2 - (cb.x0 + cb.y0)) - 0.01f; cb.s_hi = (float)(sg1 + 2 - (cb.x0 + cb.y0)) + 0.01f;
            cb.d_lo = (float)(dg0 - 2 - (cb.x0 - cb.y0)) - 0.01f; cb.d_hi = (float)(dg1 + 2 - (cb.x0 - cb.y0)) + 0.01f;
            if (warp == 0 && lane < p.n_wfs)   // once per CTA, while the box is still in flight
                footprint_of_piece<kZPack>(p, lane, qx0, qx1, qy0, qy1, sg0, sg1, dg0, dg1, s_box, s_win);
            mbar_wait(&bar, parity);
            parity ^= 1u;

            // By linearity a piece is its own mode, zero outside its box: when the support was split, whatever
            // the box holds on the piece's ring is read as 0.
            if (multi) {   // clear the ring just staged (pixels cw and ch are the far ring)
                const uint32_t org = raw_base + (uint32_t)slack * 4u, rp4 = (uint32_t)p.patch_pitch * 4u;
                for (int e = tid; e <= cb.cw; e += kComputeThreads) { sts_f32(org + (uint32_t)e * 4u, 0.0f); sts_f32(org + (uint32_t)cb.ch * rp4 + (uint32_t)e * 4u, 0.0f); }
                for (int e = tid + 1; e < cb.ch; e += kComputeThreads) { sts_f32(org + (uint32_t)e * rp4, 0.0f); sts_f32(org + (uint32_t)e * rp4 + (uint32_t)cb.cw * 4u, 0.0f); }   // (the corners belong to the rows above)
            }
            bar_sync(1, kComputeThreads);   // footprints (and a cleared ring) visible

            sample_footprints<kGtilt, kAligned, kRepair, kZPack>(p, warp, lane, s_box, s_win, &s_next, cb, tab_base, krow_base, zp, scr);
            if (multi) {
                cp_async_wait_all();
                bar_sync(1, kComputeThreads);   // every warp is done with this box and this piece's table
                if (pc + nchunk < npieces && tid == 0) {   // the box was being sampled until now
                    const int ny_ = (pc + nchunk) / npcx, nx_ = (pc + nchunk) - ny_ * npcx;
                    fence_proxy_async();
                    mbar_expect_tx(&bar, box_bytes);
                    tma_load_box(patch, &tmap, &bar, ((bx0 + nx_ * cap_w - 1) & ~3) - org.x, by0 + ny_ * cap_h - 1 - org.y, mode);
                }
                scatter_table<true, kComputeThreads>(p, s_win, tab_base, krow_base, colp, tid);
                if (tid == 0) s_next = 0;
                bar_sync(1, kComputeThreads);   // table clear again, windows free
            }
        }
    }
    while (zp.pending()) zp.step();   // what the sampling loop did not get to
    cp_async_wait_all();
    __syncthreads();                  // all zeros stored before anyone stores a value; table complete
    if (!multi && npieces > 0) scatter_table<false, kStripThreads>(p, s_win, tab_base, krow_base, colp, tid);
}


// ---- dense modes: tiles of the WFS grid -------------------------------------------------------------------------
// A dense mode has no support to skip, so the work is cut in WFS space, output-stationary: one CTA per (mode, sensor,
// tile of tile_ns strips x tile_nr subaperture rows).  The tile's pre-image under the sensor's map -- the bounding
// box of its four corners, plus the halo, the reach of a bilinear sample and the alignment slack -- is staged by ONE
// TMA box load (the sensor's own descriptor: the box of a sensor rotated by 60 degrees is twice that of an unrotated
// one), the warps take (strip, rows) pieces of the tile, and every slope of the tile is stored exactly once, by this
// CTA, with plain streaming stores: no memset, no atomics.  CTAs are ordered mode-major, so a mode's image is read
// from HBM once and served from L2 to the other tiles and sensors (the cube is fetched once for all
// WFS).  Units of invalid subapertures (outside the pupil) are skipped.
constexpr int kTileWarps = kTileWarpsPerCta, kTileThreads = 32 * kTileWarps;
constexpr int kTileScratchFloats = kEdgeBatch * kEdgeSlotFloats;   // per warp

__device__ __forceinline__ void tma_load_box_plain(void *dst, const void *map, uint64_t *bar, int x, int y, int z)
{
    asm volatile(
        "cp.async.bulk.tensor.3d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5}], [%2];"
        ::"r"(smem_u32(dst)), "l"(map), "r"(smem_u32(bar)), "r"(x), "r"(y), "r"(z)
        : "memory");
}

// grid: x = tile of the mode (all sensors of the launch), y = mode -- the tiles of a mode are neighbours in launch order
template <bool kGtilt, bool kRepair>
__global__ void __launch_bounds__(kTileThreads, 2) synim_tile_kernel(const __grid_constant__ ImParams p,
                                                                     const __grid_constant__ TileMaps maps)
{
    // [ TMA box: box_pitch x box_h floats of this sensor (<= patch_pitch floats) | table | rows | scratch ]
    extern __shared__ __align__(128) float patch[];
    __shared__ __align__(8) uint64_t bar;
    __shared__ int s_next;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int mode = blockIdx.y;
    int t = blockIdx.x;
    int w = 0;
    while (w + 1 < p.n_wfs && t >= p.wfs[w + 1].tile_first) ++w;
    const WfsDev &W = p.wfs[w];
    t -= W.tile_first;
    const int ty = t / W.tiles_x, tx = t - ty * W.tiles_x;
    const int spb = W.spb, npx = W.n_pix, n_subap = W.n_subap;
    const int b0 = tx * W.tile_ns * spb, nb = min(W.tile_ns * spb, n_subap - b0);
    const int a0 = ty * W.tile_nr, na = min(W.tile_nr, n_subap - a0);
    const uint32_t raw_base = smem_u32(patch);
    const uint32_t tab_base = raw_base + (uint32_t)p.patch_pitch * 4u;
    const uint32_t krow_base = tab_base + (uint32_t)p.tab_floats * 4u;
    const uint32_t scr = krow_base + (uint32_t)(p.tab_floats >> 1) * 4u + (uint32_t)(warp * kTileScratchFloats) * 4u;

    // the IM rows of the tile's subapertures; a tile without a valid one has nothing to compute or to store
    int any = 0;
    for (int ra = warp; ra < na; ra += kTileWarps)
        for (int rb = lane; rb < nb; rb += 32) {
            const int k = __ldg(W.subap_row + (a0 + ra) * n_subap + b0 + rb);
            sts_s32(krow_base + (uint32_t)(ra * nb + rb) * 4u, k);
            any |= (k >= 0);
        }
    if (!__syncthreads_or(any)) return;

    // pre-image of the tile's phi pixels (halo included): bounding box of the four corners, float64
    // (+1 below: the general path's row look-ahead; p.reach: what a restored pixel reads beside itself)
    const double jl = (double)(b0 * npx - 1 - p.reach), jh = (double)((b0 + nb) * npx + p.reach);
    const double il = (double)(a0 * npx - 1 - p.reach), ih = (double)((a0 + na) * npx + 1 + p.reach);
    const double cmin = W.fwd[2] + fmin(W.fwd[0] * jl, W.fwd[0] * jh) + fmin(W.fwd[1] * il, W.fwd[1] * ih);
    const double rmin = W.fwd[5] + fmin(W.fwd[3] * jl, W.fwd[3] * jh) + fmin(W.fwd[4] * il, W.fwd[4] * ih);
    const double lim = 1.0e9;
    const int x0 = ((int)floor(fmax(fmin(cmin, lim), -lim)) - 1) & ~3;   // one pixel of margin, 16-byte aligned
    const int y0 = (int)floor(fmax(fmin(rmin, lim), -lim)) - 1;
    if (tid == 0) {
        mbar_init(&bar, 1);
        fence_barrier_init();
        fence_proxy_async();
        mbar_expect_tx(&bar, (uint32_t)(W.box_pitch * W.box_h) * 4u);
        tma_load_box_plain(patch, &maps.m[w][0], &bar, x0, y0, mode);
        s_next = 0;
    }
    for (int e = tid; e < na * nb * 2; e += kTileThreads) sts_f32(tab_base + (uint32_t)e * 4u, 0.0f);
    __syncthreads();   // mbarrier initialised, table cleared

    CellBox cb;
    cb.x0 = x0; cb.y0 = y0; cb.cw = W.box_pitch; cb.ch = W.box_h;
    cb.base = raw_base; cb.pitch = W.box_pitch; cb.pitchf = (float)W.box_pitch;
    cb.limit = raw_base + (uint32_t)(W.box_pitch * W.box_h) * 4u;
    cb.s_lo = cb.d_lo = -3.0e38f; cb.s_hi = cb.d_hi = 3.0e38f;
    ZeroPacer zp;
    zp.base = nullptr; zp.next = 0; zp.end = 0;

    // pieces: strip s of the tile x chunk c of its subaperture rows (one chunk unless the tile has fewer strips than
    // the CTA has warps), first come, first served
    const int ns = (nb + spb - 1) / spb;
    int nch = max(1, min(na, kTileWarps / ns));
    const int cr = (na + nch - 1) / nch;
    nch = (na + cr - 1) / cr;
    const int total = ns * nch;
    mbar_wait(&bar, 0);
    while (true) {
        int it = 0;
        if (lane == 0) it = atomicAdd(&s_next, 1);
        it = __shfl_sync(kFull, it, 0);
        if (it >= total) break;
        const int c = it / ns, sidx = it - c * ns;
        const int bA = b0 + sidx * spb, aA = a0 + c * cr, aE = min(aA + cr, a0 + na);
        process_strip<kGtilt, true, 1, kRepair>(W, aA * npx, aE * npx - 1, bA * npx, min(spb, b0 + nb - bA) * npx, cb, p.addr_bias,
                                          tab_base, a0, b0, nb, zp, scr);
    }
    __syncthreads();   // table complete

    // S4: every slope of the tile, once (zeros included); consecutive valid subapertures of a subaperture row are
    // consecutive IM rows
    float *colp = p.out + (long long)mode * p.ld;
    const int n_sub = na * nb;
    for (int e = tid; e < 2 * n_sub; e += kTileThreads) {
        const int axis = e >= n_sub, q = axis ? e - n_sub : e;
        const int k = lds_s32(krow_base + (uint32_t)q * 4u);
        if (k < 0) continue;
        const float v = lds_f32(tab_base + (uint32_t)(2 * q + axis) * 4u);
        __stcs(colp + (axis ? W.row_y : W.row_x) + (k & kSubapRowMask), v * W.scale);
    }
}

}  // namespace

cudaError_t launch_strip(const ImParams &p, const void *tensor_map, size_t smem_bytes, bool gtilt, bool repair, cudaStream_t stream)
{
    if (p.n_modes <= 0) return cudaSuccess;
    if (gtilt && repair) return cudaErrorInvalidValue;
    bool aligned = true;   // one class of sensors per launch (the host groups them)
    for (int w = 0; w < p.n_wfs; ++w) aligned = aligned && p.wfs[w].spb > 0;
    for (int w = 0; w < p.n_wfs; ++w)
        if (!aligned && p.wfs[w].spb > 0) return cudaErrorInvalidValue;
    const bool zpack = p.unit_rows != 0 && aligned && !gtilt && !repair;
    if (p.unit_rows != 0 && !zpack) return cudaErrorInvalidValue;   // (the host sets unit_rows only where it applies)
    auto kernel = zpack ? synim_strip_kernel<false, true, false, true>
                  : repair ? (aligned ? synim_strip_kernel<false, true, true, false> : synim_strip_kernel<false, false, true, false>)
                  : gtilt ? (aligned ? synim_strip_kernel<true, true, false, false> : synim_strip_kernel<true, false, false, false>)
                          : (aligned ? synim_strip_kernel<false, true, false, false> : synim_strip_kernel<false, false, false, false>);
    if (zpack) smem_bytes += sizeof(float) * (size_t)(kComputeWarps * kEdgeBatch * kEdgeSlotFloats);
    // the opt-in shared-memory limit only ever has to grow (per device; a race sets it twice, harmlessly)
    static size_t granted[7][64] = {};
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    size_t &have = granted[zpack ? 6 : (repair ? 4 : (gtilt ? 2 : 0)) + (aligned ? 1 : 0)][dev & 63];
    if (smem_bytes > have) {
        e = cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_bytes);
        if (e != cudaSuccess) return e;
        have = smem_bytes;
    }
    CUtensorMap tm;
    memcpy(&tm, tensor_map, sizeof(tm));
    note_launch();
    kernel<<<dim3((unsigned)p.n_modes, (unsigned)(p.chunks > 0 ? p.chunks : 1)), kStripThreads, smem_bytes, stream>>>(p, tm);
    return cudaGetLastError();
}

cudaError_t launch_tiles(const ImParams &p, const TileMaps &maps, size_t smem_bytes, bool gtilt, bool repair, cudaStream_t stream)
{
    if (gtilt && repair) return cudaErrorInvalidValue;
    if (p.n_modes <= 0 || p.tiles_total <= 0) return cudaSuccess;
    for (int w = 0; w < p.n_wfs; ++w)
        if (p.wfs[w].spb <= 0) return cudaErrorInvalidValue;
    if (p.n_modes > 65535) return cudaErrorInvalidValue;   // (the host splits larger batches)
    auto kernel = repair ? synim_tile_kernel<false, true> : (gtilt ? synim_tile_kernel<true, false> : synim_tile_kernel<false, false>);
    static size_t granted[3][64] = {};
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    smem_bytes += sizeof(float) * (size_t)(kTileWarps * kTileScratchFloats);
    size_t &have = granted[repair ? 2 : (gtilt ? 1 : 0)][dev & 63];
    if (smem_bytes > have) {
        e = cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_bytes);
        if (e != cudaSuccess) return e;
        have = smem_bytes;
    }
    note_launch();
    kernel<<<dim3((unsigned)p.tiles_total, (unsigned)p.n_modes), kTileThreads, smem_bytes, stream>>>(p, maps);
    return cudaGetLastError();
}

}  // namespace synim
