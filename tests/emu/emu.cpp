// emu.cpp -- TEST INFRASTRUCTURE, NOT PRODUCT CODE (see tests/emu/README.md).
// The run-time half of the host emulation of the CUDA execution model: fibers, rendezvous points, the bounds-checked
// shared-memory arena, the registry of "device" buffers, and stand-ins for the few runtime / driver calls the library makes.
#include "emu.h"
#include "cuda.h"
#include <ucontext.h>
#include <cstdarg>
#include <map>
#include <vector>

namespace emu {
extern unsigned long long g_count_shared_ld, g_count_shared_st, g_count_gather, g_count_global;
State *cur = nullptr;
char *smem = nullptr;
size_t smem_bytes = 0;

namespace {
struct Fiber { ucontext_t ctx; State st; bool done = false; char *stack = nullptr; };
std::vector<Fiber> fibers;
ucontext_t sched_ctx;
int cur_fiber = -1;
const std::function<void()> *cur_body = nullptr;
constexpr size_t kStack = 512 << 10;
std::vector<char *> stack_pool;
long progress = 0;   // bumped whenever a sync point releases or a fiber finishes

// per-warp collective state
struct WarpSync { uint64_t slot[2][32]; int arrived = 0; unsigned gen = 0; };
std::vector<WarpSync> warps;
struct CtaSync { int arrived = 0; unsigned gen = 0; int acc = 0; int result[2] = {0, 0}; } cta;
std::map<const char *, size_t> ranges;

// Race tracking on the dynamic shared memory (a small racecheck): per 4-byte word the last writer and the last reader,
// each with the CTA-barrier generation and the issuing warp's __syncwarp generation at the time.  Two accesses to a word,
// at least one a plain write, conflict when they come from different warps with no CTA barrier in between, or from
// different lanes of one warp with no __syncwarp in between (shuffles and votes converge the lanes but order no memory, so
// they do not count).  Atomic adds conflict only with plain accesses.
struct Access { int warp = -1, lane = 0; unsigned cta_gen = 0, warp_gen = 0; char kind = 0; };   // kind: 'w' plain, 'a' atomic, 'r' read
std::vector<Access> last_write, last_read;
std::vector<unsigned> syncwarp_gen;   // per warp
unsigned long long races_found = 0;

void trampoline() { (*cur_body)(); fibers[cur_fiber].done = true; ++progress; swapcontext(&fibers[cur_fiber].ctx, &sched_ctx); }
int live_in_warp(int w)
{
    int n = 0;
    for (int l = 0; l < 32; ++l) { const size_t f = (size_t)w * 32 + l; if (f < fibers.size() && !fibers[f].done) ++n; }
    return n;
}
int live_in_cta() { int n = 0; for (auto &f : fibers) if (!f.done) ++n; return n; }
}  // namespace

void fail(const char *fmt, ...)
{
    va_list ap; va_start(ap, fmt);
    fprintf(stderr, "EMU FAILURE: ");
    vfprintf(stderr, fmt, ap);
    if (cur) fprintf(stderr, "  [block (%u,%u,%u) thread %u]", cur->bid.x, cur->bid.y, cur->bid.z, cur->tid.x);
    fprintf(stderr, "\n");
    va_end(ap);
    fflush(stderr);
    abort();
}
void yield() { swapcontext(&fibers[cur_fiber].ctx, &sched_ctx); }
int lane_id() { return (int)(cur->tid.x & 31); }

extern unsigned long long g_count_gather;
const uint64_t *warp_gather(uint64_t mine)
{
    ++g_count_gather;
    const int w = cur_fiber >> 5, l = cur_fiber & 31;
    WarpSync &ws = warps[w];
    const unsigned g = ws.gen;
    ws.slot[g & 1][l] = mine;
    if (++ws.arrived >= live_in_warp(w)) { ws.arrived = 0; ++ws.gen; ++progress; }
    else while (ws.gen == g) { yield(); if (ws.gen == g && ws.arrived >= live_in_warp(w)) { ws.arrived = 0; ++ws.gen; ++progress; } }
    return ws.slot[g & 1];
}
static int cta_sync(int pred)
{
    const unsigned g = cta.gen;
    cta.acc |= pred;
    if (++cta.arrived >= live_in_cta()) { cta.result[g & 1] = cta.acc; cta.acc = 0; cta.arrived = 0; ++cta.gen; ++progress; }
    else while (cta.gen == g) { yield(); if (cta.gen == g && cta.arrived >= live_in_cta()) { cta.result[g & 1] = cta.acc; cta.acc = 0; cta.arrived = 0; ++cta.gen; ++progress; } }
    return cta.result[g & 1];
}
void cta_barrier() { cta_sync(0); }
int cta_barrier_or(int pred) { return cta_sync(pred != 0); }

// ---- launch rules the hardware enforces: opt-in dynamic shared memory, grid limits ----------------------------------
static std::map<const void *, int> max_dyn_smem;
constexpr int kOptInSmem = 232448, kDefaultSmem = 48 << 10;
int set_max_dynamic_smem(const void *fn, int bytes)
{
    if (bytes < 0 || bytes > kOptInSmem) return 1;   // cudaErrorInvalidValue
    max_dyn_smem[fn] = bytes;
    return 0;
}

// ---- mbarrier: the current phase completes when its pending arrivals and its transaction bytes are both zero --------
namespace {
struct MBar { bool init = false; int count = 0, pending = 0; long long tx = 0; unsigned phase = 0; };
std::map<const void *, MBar> mbars;
MBar &mbar_of(const void *bar, const char *what)
{
    auto it = mbars.find(bar);
    if (it == mbars.end() || !it->second.init) fail("%s on an mbarrier this CTA has not initialised", what);
    return it->second;
}
void mbar_settle(MBar &b) { if (b.pending == 0 && b.tx == 0) { ++b.phase; b.pending = b.count; ++progress; } }
}  // namespace
void mbar_init(const void *bar, int count)
{
    if (count < 1) fail("mbarrier.init with count %d", count);
    MBar &b = mbars[bar];
    b = MBar(); b.init = true; b.count = b.pending = count;
}
void mbar_arrive_expect_tx(const void *bar, uint32_t bytes)
{
    MBar &b = mbar_of(bar, "mbarrier.arrive.expect_tx");
    if (b.pending <= 0) fail("mbarrier.arrive beyond the barrier's arrival count");
    if (bytes >= (1u << 20)) fail("mbarrier.expect_tx of %u bytes: the transaction count holds less than 2^20", bytes);
    b.tx += bytes; --b.pending;
    mbar_settle(b);
}
void mbar_complete_tx(const void *bar, uint32_t bytes)
{
    MBar &b = mbar_of(bar, "TMA complete_tx");
    b.tx -= bytes;
    mbar_settle(b);
}
bool mbar_try_wait(const void *bar, uint32_t parity)
{
    MBar &b = mbar_of(bar, "mbarrier.try_wait");
    if (parity > 1) fail("mbarrier.try_wait.parity with parity %u", parity);
    if ((b.phase & 1u) != parity) {
        if (b.phase == 0) fail("mbarrier.try_wait on the parity of a phase that never ran (returns at once on hardware: a race)");
        return true;
    }
    yield();   // the phase with this parity is still open: somebody else has to complete it
    return false;
}

void launch(const void *fn, dim3 grid, dim3 block, size_t smemb, const std::function<void()> &body)
{
    const size_t nt = (size_t)block.x * block.y * block.z;
    if (nt == 0 || nt > 1024) fail("bad block size");
    if (grid.x == 0 || grid.y == 0 || grid.z == 0 || grid.x > 2147483647u || grid.y > 65535u || grid.z > 65535u)
        fail("bad grid (%u, %u, %u): the launch fails on hardware", grid.x, grid.y, grid.z);
    {
        auto it = max_dyn_smem.find(fn);
        const size_t granted = it == max_dyn_smem.end() ? (size_t)kDefaultSmem : std::max<size_t>((size_t)it->second, (size_t)kDefaultSmem);
        if (smemb > granted)
            fail("launch with %zu bytes of dynamic shared memory, but this kernel was granted %zu (cudaFuncSetAttribute on THIS instantiation)", smemb, granted);
    }
    while (stack_pool.size() < nt) stack_pool.push_back((char *)malloc(kStack));
    std::vector<char> arena(smemb + 64, 0);
    for (unsigned bz = 0; bz < grid.z; ++bz) for (unsigned by = 0; by < grid.y; ++by) for (unsigned bx = 0; bx < grid.x; ++bx) {
        memset(arena.data(), 0xCD, arena.size());   // shared memory starts as garbage
        smem = arena.data(); smem_bytes = smemb;
        fibers.assign(nt, Fiber());
        warps.assign((nt + 31) / 32, WarpSync());
        last_write.assign(smemb / 4 + 1, Access());
        last_read.assign(smemb / 4 + 1, Access());
        syncwarp_gen.assign((nt + 31) / 32, 0u);
        cta = CtaSync();
        mbars.clear();   // static __shared__ barriers are garbage until this CTA initialises them
        cur_body = &body;
        for (size_t t = 0; t < nt; ++t) {
            Fiber &f = fibers[t];
            f.st.tid = uint3{(unsigned)(t % block.x), (unsigned)((t / block.x) % block.y), (unsigned)(t / ((size_t)block.x * block.y))};
            f.st.bid = uint3{bx, by, bz}; f.st.bdim = block; f.st.gdim = grid;
            getcontext(&f.ctx);
            f.ctx.uc_stack.ss_sp = stack_pool[t]; f.ctx.uc_stack.ss_size = kStack; f.ctx.uc_link = &sched_ctx;
            makecontext(&f.ctx, trampoline, 0);
        }
        size_t remaining = nt;
        long last_progress = -1; int idle_rounds = 0;
        while (remaining) {
            remaining = 0;
            for (size_t t = 0; t < nt; ++t) {
                if (fibers[t].done) continue;
                cur_fiber = (int)t; cur = &fibers[t].st;
                swapcontext(&sched_ctx, &fibers[t].ctx);
                if (!fibers[t].done) ++remaining;
            }
            if (progress == last_progress) { if (++idle_rounds > 4) { cur = nullptr; fail("deadlock: %zu threads wait at a synchronisation point nobody else reaches (block %u,%u)", remaining, bx, by); } }
            else { idle_rounds = 0; last_progress = progress; }
        }
        cur = nullptr; cur_fiber = -1;
    }
    smem = nullptr; smem_bytes = 0;
}

void register_range(const void *p, size_t bytes)
{
    const char *c = (const char *)p;
    // drop stale entries the new buffer overlaps (buffers the caller freed without telling us)
    auto it = ranges.lower_bound(c);
    if (it != ranges.begin()) { auto pr = std::prev(it); if (pr->first + pr->second > c) ranges.erase(pr); }
    it = ranges.lower_bound(c);
    while (it != ranges.end() && it->first < c + bytes) it = ranges.erase(it);
    ranges[c] = bytes;
}
void unregister_range(const void *p) { ranges.erase((const char *)p); }
extern unsigned long long g_count_global;
// (optional) one tracked buffer: how often each of its 4-byte words is stored with __stcs -- the tile kernel's claim that
// every slope is stored exactly once is checked with this
static const char *track_base = nullptr;
static std::vector<unsigned char> track_count;
void check_global(const void *p, size_t bytes, const char *what)
{
    if (track_base && what[0] == '_' && what[2] == 's') {   // "__stcs"
        const char *c = (const char *)p;
        if (c >= track_base && c + bytes <= track_base + track_count.size() * 4)
            for (size_t k = 0; k < bytes / 4; ++k) { unsigned char &n = track_count[(c - track_base) / 4 + k]; if (n < 255) ++n; }
    }
    ++g_count_global;
    if (bytes <= 16 && ((uintptr_t)p % bytes) != 0) fail("%s: misaligned global access of %zu bytes at %p", what, bytes, p);
    check_range(p, bytes, what);
}
void check_range(const void *p, size_t bytes, const char *what)
{
    const char *c = (const char *)p;
    auto it = ranges.upper_bound(c);
    if (it != ranges.begin()) { --it; if (c >= it->first && c + bytes <= it->first + it->second) return; }
    fail("%s: global access of %zu bytes at %p is outside every registered buffer", what, bytes, p);
}
unsigned long long g_count_shared_ld = 0, g_count_shared_st = 0, g_count_gather = 0, g_count_global = 0;
void note_syncwarp() { if (cur_fiber >= 0 && (cur_fiber & 31) == 0) ++syncwarp_gen[cur_fiber >> 5]; }
static void conflict(const char *what, const char *how, uint32_t addr, const Access &o)
{
    ++races_found;
    fail("%s: shared-memory race (%s) on window offset %u: the other access came from warp %d lane %d with no %s in between", what, how,
         addr - kSmemBase, o.warp, o.lane, o.warp == (cur_fiber >> 5) ? "__syncwarp" : "CTA barrier");
}
char *shared_ptr(uint32_t addr, size_t bytes, const char *what)
{
    if (what[0] == 'l') ++g_count_shared_ld; else ++g_count_shared_st;
    if (addr < kSmemBase || (size_t)(addr - kSmemBase) + bytes > smem_bytes)
        fail("%s: shared access of %zu bytes at window offset %lld is outside the CTA's %zu bytes of dynamic shared memory", what, bytes,
             (long long)addr - (long long)kSmemBase, smem_bytes);
    if (addr % bytes) fail("%s: misaligned shared access", what);
    if (cur_fiber >= 0 && what[0] != 't') {   // (TMA writes are ordered by their mbarrier; its waits are not modelled)
        const int w = cur_fiber >> 5, l = cur_fiber & 31;
        const char kind = what[0] == 'l' ? 'r' : (what[0] == 'r' ? 'a' : 'w');
        const size_t word = (addr - kSmemBase) / 4;
        const unsigned wg = syncwarp_gen[w];
        auto clashes = [&](const Access &o) {
            if (o.warp < 0) return false;
            if (o.warp != w) return o.cta_gen == cta.gen;
            return o.lane != l && o.warp_gen == wg && o.cta_gen == cta.gen;
        };
        Access &lw = last_write[word], &lr = last_read[word];
        if (kind == 'r') {
            if (clashes(lw)) conflict(what, "read after write", addr, lw);
            lr.warp = w; lr.lane = l; lr.cta_gen = cta.gen; lr.warp_gen = wg; lr.kind = 'r';
        } else {
            if (clashes(lw) && !(kind == 'a' && lw.kind == 'a')) conflict(what, "write after write", addr, lw);
            if (clashes(lr)) conflict(what, "write after read", addr, lr);
            lw.warp = w; lw.lane = l; lw.cta_gen = cta.gen; lw.warp_gen = wg; lw.kind = kind;
        }
    }
    return smem + (addr - kSmemBase);
}
uint32_t shared_addr(const void *p)
{
    const char *c = (const char *)p;
    if (smem && c >= smem && c < smem + smem_bytes + 64) return kSmemBase + (uint32_t)(c - smem);
    return 0x7f000000u;   // a static __shared__ variable: only ever handed to mbarrier operations, which are no-ops here
}
}  // namespace emu

cudaError_t cudaMalloc(void **p, size_t n)
{
    if (posix_memalign(p, 256, n ? n : 1) != 0) { *p = nullptr; return cudaErrorMemoryAllocation; }   // (exactly n bytes: a sanitizer sees the end)
    memset(*p, 0xA5, n);   // device memory starts as garbage
    emu::register_range(*p, n);
    return cudaSuccess;
}
cudaError_t cudaFree(void *p) { if (p) { emu::unregister_range(p); free(p); } return cudaSuccess; }

static CUresult emu_encode(CUtensorMap *out, CUtensorMapDataType, cuuint32_t rank, void *base, const cuuint64_t *dims, const cuuint64_t *strides,
                           const cuuint32_t *box, const cuuint32_t *, CUtensorMapInterleave, CUtensorMapSwizzle, CUtensorMapL2promotion,
                           CUtensorMapFloatOOBfill)
{
    if (rank != 3) return 1;
    if (((uintptr_t)base & 15) || (strides[0] & 15) || (strides[1] & 15) || ((box[0] * 4) & 15) || box[0] > 256 || box[1] > 256) return 1;
    EmuTensorMap m; m.base = (const float *)base;
    for (int k = 0; k < 3; ++k) { m.dims[k] = dims[k]; m.box[k] = box[k]; }
    m.strides[0] = strides[0]; m.strides[1] = strides[1];
    memset(out, 0, sizeof(*out)); memcpy(out, &m, sizeof(m));
    return CUDA_SUCCESS;
}
cudaError_t cudaGetDriverEntryPoint(const char *, void **fn, int, cudaDriverEntryPointQueryResult *q)
{
    *fn = (void *)&emu_encode; *q = cudaDriverEntryPointSuccess; return cudaSuccess;
}

extern "C" void emu_counters(unsigned long long *out) { out[0] = emu::g_count_shared_ld; out[1] = emu::g_count_shared_st; out[2] = emu::g_count_gather; out[3] = emu::g_count_global; emu::g_count_shared_ld = emu::g_count_shared_st = emu::g_count_gather = emu::g_count_global = 0; }
extern "C" void emu_track_stores(const void *p, size_t bytes) { emu::track_base = (const char *)p; emu::track_count.assign(bytes / 4, 0); }
extern "C" void emu_store_counts(unsigned char *out) { memcpy(out, emu::track_count.data(), emu::track_count.size()); emu::track_base = nullptr; }
extern "C" void emu_register(const void *p, size_t n) { emu::register_range(p, n); }
extern "C" void emu_unregister(const void *p) { emu::unregister_range(p); }
