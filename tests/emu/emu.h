// emu.h -- TEST INFRASTRUCTURE, NOT PRODUCT CODE (see tests/emu/README.md).
// Host emulation of the CUDA execution model, for checking kernel LOGIC and memory safety without a GPU.
// One OS thread; every CUDA thread of the running CTA is a ucontext fiber; warp / CTA synchronisation points yield.
#pragma once
#include <cstdint>
#include <cstddef>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <cmath>
#include <algorithm>
#include <functional>

struct dim3 { unsigned x, y, z; dim3(unsigned a = 1, unsigned b = 1, unsigned c = 1) : x(a), y(b), z(c) {} };
struct uint3 { unsigned x, y, z; };
struct alignas(16) float4 { float x, y, z, w; };
struct alignas(16) int4 { int x, y, z, w; };
struct alignas(8) int2 { int x, y; };
static inline float4 make_float4(float a, float b, float c, float d) { return float4{a, b, c, d}; }
static inline int4 make_int4(int a, int b, int c, int d) { return int4{a, b, c, d}; }
static inline int2 make_int2(int a, int b) { return int2{a, b}; }

namespace emu {
struct State {
    uint3 tid, bid; dim3 bdim, gdim;
};
extern State *cur;           // the running fiber's identity
extern char *smem;           // dynamic shared memory arena of the running CTA
extern size_t smem_bytes;
constexpr uint32_t kSmemBase = 4096;   // shared-window address of arena byte 0 (small negative offsets stay detectable)
void yield();
void fail(const char *fmt, ...);
void launch(const void *fn, dim3 grid, dim3 block, size_t smem, const std::function<void()> &body);
int set_max_dynamic_smem(const void *fn, int bytes);   // cudaFuncSetAttribute(MaxDynamicSharedMemorySize)
// mbarrier model (one CTA runs at a time; TMA is synchronous): arrival count, transaction bytes, phase parity
void mbar_init(const void *bar, int count);
void mbar_arrive_expect_tx(const void *bar, uint32_t bytes);
void mbar_complete_tx(const void *bar, uint32_t bytes);
bool mbar_try_wait(const void *bar, uint32_t parity);
void cta_barrier();
int cta_barrier_or(int pred);
// warp collective: every live lane contributes 8 bytes; afterwards all 32 slots are readable until the next collective
const uint64_t *warp_gather(uint64_t mine);
int lane_id();
void note_syncwarp();   // (race tracking: a __syncwarp orders the warp's shared-memory accesses)
void register_range(const void *p, size_t bytes);
void unregister_range(const void *p);
void check_global(const void *p, size_t bytes, const char *what);   // one access: in range and naturally aligned
void check_range(const void *p, size_t bytes, const char *what);    // a byte range (memset, memcpy)
char *shared_ptr(uint32_t addr, size_t bytes, const char *what);
uint32_t shared_addr(const void *p);
}

#define __global__
#define __device__
#define __host__
#define __forceinline__ inline
#define __launch_bounds__(...)
#define __grid_constant__
#define __align__(n) __attribute__((aligned(n)))
#define threadIdx (emu::cur->tid)
#define blockIdx (emu::cur->bid)
#define blockDim (emu::cur->bdim)
#define gridDim (emu::cur->gdim)

template <typename T> static inline T emu_shfl_from(T v, int src_lane)
{
    static_assert(sizeof(T) <= 8, "");
    uint64_t raw = 0; memcpy(&raw, &v, sizeof(T));
    const uint64_t *all = emu::warp_gather(raw);
    T out; memcpy(&out, &all[src_lane & 31], sizeof(T));
    return out;
}
template <typename T> static inline T __shfl_sync(unsigned, T v, int src) { return emu_shfl_from(v, src); }
template <typename T> static inline T __shfl_up_sync(unsigned, T v, unsigned d)
{
    const int l = emu::lane_id(); const int s = l - (int)d;
    T o = emu_shfl_from(v, s < 0 ? l : s); return o;
}
template <typename T> static inline T __shfl_down_sync(unsigned, T v, unsigned d)
{
    const int l = emu::lane_id(); const int s = l + (int)d;
    return emu_shfl_from(v, s > 31 ? l : s);
}
template <typename T> static inline T __shfl_xor_sync(unsigned, T v, int m) { return emu_shfl_from(v, emu::lane_id() ^ m); }
static inline unsigned __ballot_sync(unsigned, int pred)
{
    const uint64_t *all = emu::warp_gather(pred ? 1u : 0u);
    unsigned m = 0; for (int l = 0; l < 32; ++l) if (all[l] & 1u) m |= 1u << l;
    return m;
}
static inline void __syncwarp(unsigned = 0xffffffffu) { emu::warp_gather(0); emu::note_syncwarp(); emu::warp_gather(0); }
static inline void __syncthreads() { emu::cta_barrier(); }
static inline int __syncthreads_or(int p) { return emu::cta_barrier_or(p); }
template <typename T> static inline T __ldg(const T *p) { emu::check_global(p, sizeof(T), "__ldg"); return *p; }
template <typename T> static inline void __stcs(T *p, T v) { emu::check_global(p, sizeof(T), "__stcs"); *p = v; }
static inline float __fadd_rd(float a, float b)
{
    const double e = (double)a + (double)b;   // (exact unless the exponents are > 29 apart: then e is within 1 ulp_double)
    float s = (float)e;
    if ((double)s > e) s = nextafterf(s, -INFINITY);
    return s;
}
static inline unsigned __float_as_uint(float f) { unsigned u; memcpy(&u, &f, 4); return u; }
static inline float __uint_as_float(unsigned u) { float f; memcpy(&f, &u, 4); return f; }
static inline unsigned __umulhi(unsigned a, unsigned b) { return (unsigned)(((uint64_t)a * b) >> 32); }
static inline int __double2int_rn(double x) { return (int)nearbyint(x); }
static inline int __ffs(unsigned x) { return x ? __builtin_ctz(x) + 1 : 0; }
static inline int __clz(unsigned x) { return x ? __builtin_clz(x) : 32; }
static inline int __popc(unsigned x) { return __builtin_popcount(x); }
static inline size_t __cvta_generic_to_shared(const void *p) { return emu::shared_addr(p); }
static inline int atomicAdd(int *p, int v) { int o = *p; *p = o + v; return o; }
static inline float atomicAdd(float *p, float v) { emu::check_global(p, 4, "atomicAdd"); float o = *p; *p = o + v; return o; }
static inline int atomicExch(int *p, int v) { int o = *p; *p = v; return o; }
static inline void __trap() { emu::fail("__trap()"); }
using std::min; using std::max;
static inline int min(int a, unsigned b) { return std::min(a, (int)b); }

#define EMU_LAUNCH(kernel, grid, block, smemb, ...) emu::launch((const void *)(kernel), dim3(grid), dim3(block), (size_t)(smemb), [&]() { kernel(__VA_ARGS__); })

// ---- runtime API shim -------------------------------------------------------------------------------------------
typedef int cudaError_t;
typedef void *cudaStream_t;
enum { cudaSuccess = 0, cudaErrorInvalidValue = 1, cudaErrorMemoryAllocation = 2 };
enum cudaMemcpyKind { cudaMemcpyHostToDevice = 1, cudaMemcpyDeviceToHost = 2, cudaMemcpyDeviceToDevice = 3 };
enum { cudaDevAttrComputeCapabilityMajor = 75, cudaDevAttrMaxSharedMemoryPerBlockOptin = 97 };
enum { cudaFuncAttributeMaxDynamicSharedMemorySize = 8 };
enum cudaDriverEntryPointQueryResult { cudaDriverEntryPointSuccess = 0, cudaDriverEntryPointSymbolNotFound = 1 };
enum { cudaEnableDefault = 0 };
static inline const char *cudaGetErrorString(cudaError_t e) { return e == 0 ? "no error" : "emulated error"; }
static inline cudaError_t cudaGetLastError() { return cudaSuccess; }
static inline cudaError_t cudaGetDevice(int *d) { *d = 0; return cudaSuccess; }
static inline cudaError_t cudaDeviceGetAttribute(int *v, int attr, int) { *v = attr == cudaDevAttrComputeCapabilityMajor ? 10 : 232448; return cudaSuccess; }
template <typename F> static inline cudaError_t cudaFuncSetAttribute(F f, int attr, int v)
{
    return attr == cudaFuncAttributeMaxDynamicSharedMemorySize ? emu::set_max_dynamic_smem((const void *)f, v) : cudaSuccess;
}
cudaError_t cudaMalloc(void **p, size_t n);
cudaError_t cudaFree(void *p);
static inline cudaError_t cudaMallocAsync(void **p, size_t n, cudaStream_t) { return cudaMalloc(p, n); }
static inline cudaError_t cudaFreeAsync(void *p, cudaStream_t) { return cudaFree(p); }
static inline cudaError_t cudaMallocHost(void **p, size_t n) { *p = malloc(n); return *p ? cudaSuccess : cudaErrorMemoryAllocation; }
static inline cudaError_t cudaFreeHost(void *p) { free(p); return cudaSuccess; }
static inline cudaError_t cudaMemcpyAsync(void *d, const void *s, size_t n, cudaMemcpyKind, cudaStream_t) { memcpy(d, s, n); return cudaSuccess; }
static inline cudaError_t cudaMemsetAsync(void *d, int v, size_t n, cudaStream_t) { emu::check_range(d, n, "cudaMemsetAsync"); memset(d, v, n); return cudaSuccess; }
static inline cudaError_t cudaMemset2DAsync(void *d, size_t pitch, int v, size_t w, size_t h, cudaStream_t)
{
    for (size_t r = 0; r < h; ++r) { emu::check_range((char *)d + r * pitch, w, "cudaMemset2DAsync"); memset((char *)d + r * pitch, v, w); }
    return cudaSuccess;
}
static inline cudaError_t cudaStreamSynchronize(cudaStream_t) { return cudaSuccess; }
static inline cudaError_t cudaDeviceSynchronize() { return cudaSuccess; }
typedef void *cudaEvent_t;
enum { cudaStreamNonBlocking = 1, cudaEventDisableTiming = 2 };
static inline cudaError_t cudaStreamCreateWithFlags(cudaStream_t *s, int) { *s = (cudaStream_t)malloc(8); return cudaSuccess; }
static inline cudaError_t cudaStreamDestroy(cudaStream_t s) { free(s); return cudaSuccess; }
static inline cudaError_t cudaEventCreateWithFlags(cudaEvent_t *e, int) { *e = (cudaEvent_t)malloc(8); return cudaSuccess; }
static inline cudaError_t cudaEventDestroy(cudaEvent_t e) { free(e); return cudaSuccess; }
static inline cudaError_t cudaEventRecord(cudaEvent_t, cudaStream_t) { return cudaSuccess; }
static inline cudaError_t cudaEventSynchronize(cudaEvent_t) { return cudaSuccess; }
static inline cudaError_t cudaStreamWaitEvent(cudaStream_t, cudaEvent_t, int) { return cudaSuccess; }
cudaError_t cudaGetDriverEntryPoint(const char *name, void **fn, int, cudaDriverEntryPointQueryResult *q);
