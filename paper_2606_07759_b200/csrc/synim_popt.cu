// synim_popt.cu -- the tomographic projection matrix of PAPER.md:90 (sec. 2.5):
//     P_opt = (P_DM^T P_DM + lambda I)^-1 P_DM^T P_Layer,
// "where P_DM and P_Layer map the influence functions over the optimized directions" (readings R24-R26 of DESIGN.md).
//
// Two halves.  (1) The operands are this library's own steps S1-S2 without the derivative: every mode of a component,
// resampled ONCE through the direction's composite map onto the pupil grid (bilinear, zero outside the grid), times
// the pupil weight and the square root of the direction's weight -- popt_operand_kernel below, HBM-bound by the store
// of the operand.  (2) The contraction is a plain dense GEMM (the paper: "heavily dominated by large, dense
// matrix-matrix multiplications") followed by a Cholesky solve: both are library calls, cuBLAS (SYRK + GEMM) and
// cuSOLVER (POTRF + POTRS), loaded at the first call with dlopen so that libsynim.so itself links neither (the
// interaction-matrix path never needs them).  This is the one tensor-core candidate of the paper; cuBLAS chooses the
// kernels.
#include "../../include/synim.h"
#include "synim_device.h"

#include <dlfcn.h>

#include <cmath>
#include <cstdio>
#include <cstring>
#include <mutex>
#include <vector>

namespace synim {

// (synim_api.cu) thread-local error text behind synim_last_error()
synim_status report(synim_status s, const char *fmt, ...);

namespace {

// ---- (1) the operand ---------------------------------------------------------------------------------------------
// a[(d * mp*mp + p) + K * m] = sqrt(w_d) * pupil[p] * phi_m(A_d x_p); K = n_dir * mp * mp.  One thread per pupil pixel,
// grid (pixel blocks, directions, modes).  The map is the absolute-index one (centring folded in on the host, float64),
// evaluated in float64 per pixel; the four taps come through the read-only path (neighbouring threads share sectors).
struct DirMap { double f[6]; float sw; };

__global__ void __launch_bounds__(256) popt_operand_kernel(const float *__restrict__ cube, int ny, int nx, const DirMap *__restrict__ maps,
                                                           const float *__restrict__ pupil, int mp, long long K, float *__restrict__ out)
{
    const int p = blockIdx.x * 256 + threadIdx.x;
    if (p >= mp * mp) return;
    const int d = blockIdx.y, m = blockIdx.z;
    const DirMap M = maps[d];
    const float pw = __ldg(pupil + p);
    float v = 0.0f;
    if (pw != 0.0f) {
        const int i = p / mp, j = p - i * mp;
        const double col = M.f[0] * (double)j + M.f[1] * (double)i + M.f[2];
        const double row = M.f[3] * (double)j + M.f[4] * (double)i + M.f[5];
        const double fc = floor(col), fr = floor(row);
        if (fc >= -1.0 && fc <= (double)nx && fr >= -1.0 && fr <= (double)ny) {
            const int c0 = (int)fc, r0 = (int)fr;
            const float fx = (float)(col - fc), fy = (float)(row - fr);
            const float *img = cube + (size_t)m * (size_t)ny * (size_t)nx;
            const bool cl = c0 >= 0 && c0 < nx, ch = c0 + 1 >= 0 && c0 + 1 < nx;
            float v00 = 0.f, v01 = 0.f, v10 = 0.f, v11 = 0.f;
            if (r0 >= 0 && r0 < ny) {
                if (cl) v00 = __ldg(img + (size_t)r0 * nx + c0);
                if (ch) v01 = __ldg(img + (size_t)r0 * nx + c0 + 1);
            }
            if (r0 + 1 >= 0 && r0 + 1 < ny) {
                if (cl) v10 = __ldg(img + (size_t)(r0 + 1) * nx + c0);
                if (ch) v11 = __ldg(img + (size_t)(r0 + 1) * nx + c0 + 1);
            }
            const float t = fmaf(fx, v01 - v00, v00), u = fmaf(fx, v11 - v10, v10);
            v = fmaf(fy, u - t, t) * (pw * M.sw);
        }
    }
    __stcs(out + (size_t)K * (size_t)m + (size_t)d * (size_t)(mp * mp) + p, v);
}

__global__ void __launch_bounds__(256) popt_add_diagonal_kernel(float *g, int n, float lam)
{
    const int k = blockIdx.x * 256 + threadIdx.x;
    if (k < n) g[(size_t)k * n + k] += lam;
}

// ---- (2) cuBLAS / cuSOLVER, loaded on first use ----------------------------------------------------------------------
typedef void *Handle;
struct Libs {
    bool tried = false, ok = false;
    char why[256] = "";
    int (*blasCreate)(Handle *) = nullptr;
    int (*blasSetStream)(Handle, cudaStream_t) = nullptr;
    int (*ssyrk)(Handle, int, int, int, int, const float *, const float *, int, const float *, float *, int) = nullptr;
    int (*sgemm)(Handle, int, int, int, int, int, const float *, const float *, int, const float *, int, const float *, float *, int) = nullptr;
    int (*solCreate)(Handle *) = nullptr;
    int (*solSetStream)(Handle, cudaStream_t) = nullptr;
    int (*potrfSize)(Handle, int, int, float *, int, int *) = nullptr;
    int (*potrf)(Handle, int, int, float *, int, float *, int, int *) = nullptr;
    int (*potrs)(Handle, int, int, int, const float *, int, float *, int, int *) = nullptr;
    Handle blas[64] = {}, sol[64] = {};
};
Libs g_libs;
std::mutex g_libs_lock;

void *open_any(const char *const *names)
{
    for (; *names; ++names)
        if (void *h = dlopen(*names, RTLD_NOW | RTLD_GLOBAL)) return h;
    return nullptr;
}

bool load_libs()
{
    Libs &L = g_libs;
    if (L.tried) return L.ok;
    L.tried = true;
    static const char *const blas_names[] = {"libcublas.so.12", "libcublas.so", "/usr/local/cuda/lib64/libcublas.so.12", nullptr};
    static const char *const sol_names[] = {"libcusolver.so.11", "libcusolver.so", "/usr/local/cuda/lib64/libcusolver.so.11", nullptr};
    void *hb = open_any(blas_names), *hs = open_any(sol_names);
    if (!hb || !hs) {
        snprintf(L.why, sizeof(L.why), "%s could not be loaded: %s", hb ? "libcusolver" : "libcublas", dlerror() ? dlerror() : "not found");
        return false;
    }
#define SYNIM_SYM(field, handle, name)                                                         \
    do {                                                                                       \
        *reinterpret_cast<void **>(&L.field) = dlsym(handle, name);                            \
        if (!L.field) { snprintf(L.why, sizeof(L.why), "symbol %s not found", name); return false; } \
    } while (0)
    SYNIM_SYM(blasCreate, hb, "cublasCreate_v2");
    SYNIM_SYM(blasSetStream, hb, "cublasSetStream_v2");
    SYNIM_SYM(ssyrk, hb, "cublasSsyrk_v2");
    SYNIM_SYM(sgemm, hb, "cublasSgemm_v2");
    SYNIM_SYM(solCreate, hs, "cusolverDnCreate");
    SYNIM_SYM(solSetStream, hs, "cusolverDnSetStream");
    SYNIM_SYM(potrfSize, hs, "cusolverDnSpotrf_bufferSize");
    SYNIM_SYM(potrf, hs, "cusolverDnSpotrf");
    SYNIM_SYM(potrs, hs, "cusolverDnSpotrs");
#undef SYNIM_SYM
    L.ok = true;
    return true;
}

// absolute-index map of a direction: pupil pixel (i, j) of an mp x mp grid -> pixel (row, col) of an ny x nx grid
void absolute_map(const synim_wfs_affine &af, int mp, int ny, int nx, double f[6])
{
    const double cw = (mp - 1) / 2.0, cx = (nx - 1) / 2.0, cy = (ny - 1) / 2.0;
    const double *a = af.a;
    f[0] = a[0]; f[1] = a[1]; f[2] = a[2] + cx - cw * (a[0] + a[1]);
    f[3] = a[3]; f[4] = a[4]; f[5] = a[5] + cy - cw * (a[3] + a[4]);
}

struct AsyncMem {
    std::vector<void *> p;
    cudaStream_t s = nullptr;
    ~AsyncMem() { for (void *q : p) if (q) cudaFreeAsync(q, s); }
    cudaError_t get(void **out, size_t bytes)
    {
        cudaError_t e = cudaMallocAsync(out, bytes ? bytes : 16, s);
        if (e == cudaSuccess) p.push_back(*out);
        return e;
    }
};

}  // namespace

}  // namespace synim

using synim::report;

#define POPT_CUDA(call)                                                                                             \
    do {                                                                                                            \
        cudaError_t e_ = (call);                                                                                    \
        if (e_ != cudaSuccess)                                                                                      \
            return report(e_ == cudaErrorMemoryAllocation ? SYNIM_ERR_OUT_OF_MEMORY : SYNIM_ERR_CUDA, "%s: %s", #call, \
                          cudaGetErrorString(e_));                                                                  \
    } while (0)
#define POPT_LIB(call)                                                                                  \
    do {                                                                                                \
        int s_ = (call);                                                                                \
        if (s_ != 0) return report(SYNIM_ERR_CUDA, "synim_projection_matrix: %s returned status %d", #call, s_); \
    } while (0)

extern "C" synim_status synim_projection_matrix(const synim_component *dms, int32_t n_dms, const synim_component *layer, int32_t n_dir,
                                                const double *dir_weight, const float *d_pupil, int32_t mp, double lambda,
                                                float *d_popt, int64_t ld, void *stream)
{
    using namespace synim;
    if (!dms || n_dms < 1 || !layer || n_dir < 1 || !d_pupil || mp < 1 || !d_popt)
        return report(SYNIM_ERR_INVALID_ARG, "synim_projection_matrix: NULL argument or non-positive count");
    if (!(lambda >= 0.0) || !std::isfinite(lambda)) return report(SYNIM_ERR_INVALID_ARG, "synim_projection_matrix: lambda must be >= 0");
    long long n_a = 0;
    std::vector<const synim_component *> comps;
    for (int c = 0; c <= n_dms; ++c) {
        const synim_component *q = c < n_dms ? &dms[c] : layer;
        if (q->n_modes < 0 || q->ny <= 0 || q->nx <= 0 || !q->maps || (q->n_modes > 0 && !q->d_cube))
            return report(SYNIM_ERR_INVALID_ARG, "synim_projection_matrix: component %d: bad sizes or NULL pointer", c);
        if (q->n_modes > 65535) return report(SYNIM_ERR_INVALID_ARG, "synim_projection_matrix: component %d: more than 65535 modes", c);
        for (int d = 0; d < n_dir; ++d)
            for (int k = 0; k < 6; ++k)
                if (!std::isfinite(q->maps[d].a[k])) return report(SYNIM_ERR_INVALID_ARG, "synim_projection_matrix: non-finite map");
        if (c < n_dms) n_a += q->n_modes;
        comps.push_back(q);
    }
    const long long n_l = layer->n_modes;
    const long long K = (long long)n_dir * mp * mp;
    if (ld < n_a) return report(SYNIM_ERR_INVALID_ARG, "synim_projection_matrix: ld = %lld < rows = %lld", (long long)ld, n_a);
    if (n_a == 0 || n_l == 0) return SYNIM_OK;
    if (K > 0x7fffffffLL || n_a > 0x7fffffffLL / 2 || ld > 0x7fffffffLL || n_dir > 65535)
        return report(SYNIM_ERR_INVALID_ARG, "synim_projection_matrix: sizes beyond the 32-bit interface of the BLAS");
    for (int d = 0; dir_weight && d < n_dir; ++d)
        if (!(dir_weight[d] >= 0.0) || !std::isfinite(dir_weight[d])) return report(SYNIM_ERR_INVALID_ARG, "synim_projection_matrix: negative weight");
    cudaStream_t s = static_cast<cudaStream_t>(stream);
    int dev = 0;
    POPT_CUDA(cudaGetDevice(&dev));
    if (dev < 0 || dev >= 64) return report(SYNIM_ERR_INVALID_ARG, "synim_projection_matrix: device index out of range");

    std::lock_guard<std::mutex> guard(g_libs_lock);   // handles are per device and bound to a stream per call
    if (!load_libs()) return report(SYNIM_ERR_UNSUPPORTED, "synim_projection_matrix: %s", g_libs.why);
    Libs &L = g_libs;
    if (!L.blas[dev]) POPT_LIB(L.blasCreate(&L.blas[dev]));
    if (!L.sol[dev]) POPT_LIB(L.solCreate(&L.sol[dev]));
    POPT_LIB(L.blasSetStream(L.blas[dev], s));
    POPT_LIB(L.solSetStream(L.sol[dev], s));

    AsyncMem mem;
    mem.s = s;
    float *a_dm = nullptr, *a_l = nullptr, *g = nullptr, *work = nullptr;
    int *info = nullptr;
    DirMap *d_maps = nullptr;
    POPT_CUDA(mem.get(reinterpret_cast<void **>(&a_dm), sizeof(float) * (size_t)K * (size_t)n_a));
    POPT_CUDA(mem.get(reinterpret_cast<void **>(&a_l), sizeof(float) * (size_t)K * (size_t)n_l));
    POPT_CUDA(mem.get(reinterpret_cast<void **>(&g), sizeof(float) * (size_t)n_a * (size_t)n_a));
    POPT_CUDA(mem.get(reinterpret_cast<void **>(&info), 2 * sizeof(int)));
    POPT_CUDA(mem.get(reinterpret_cast<void **>(&d_maps), sizeof(DirMap) * (size_t)n_dir * comps.size()));

    // (1) operands
    std::vector<DirMap> h_maps((size_t)n_dir * comps.size());
    for (size_t c = 0; c < comps.size(); ++c)
        for (int d = 0; d < n_dir; ++d) {
            DirMap &m = h_maps[c * n_dir + d];
            absolute_map(comps[c]->maps[d], mp, comps[c]->ny, comps[c]->nx, m.f);
            m.sw = (float)std::sqrt(dir_weight ? dir_weight[d] : 1.0);
        }
    // (pageable source: staged by the runtime before the call returns)
    POPT_CUDA(cudaMemcpyAsync(d_maps, h_maps.data(), sizeof(DirMap) * h_maps.size(), cudaMemcpyHostToDevice, s));
    long long col0 = 0;
    for (size_t c = 0; c < comps.size(); ++c) {
        const synim_component *q = comps[c];
        const bool is_layer = c + 1 == comps.size();
        if (q->n_modes == 0) continue;
        float *dst = is_layer ? a_l : a_dm + (size_t)K * (size_t)col0;
        note_launch();
        popt_operand_kernel<<<dim3((unsigned)((mp * mp + 255) / 256), (unsigned)n_dir, (unsigned)q->n_modes), 256, 0, s>>>(
            q->d_cube, q->ny, q->nx, d_maps + c * n_dir, d_pupil, mp, K, dst);
        POPT_CUDA(cudaGetLastError());
        if (!is_layer) col0 += q->n_modes;
    }
    // (2) G = A_dm^T A_dm (lower triangle) + lambda I;  C = A_dm^T A_l -> d_popt;  Cholesky;  solve in place
    const float one = 1.0f, zero = 0.0f;
    const int LOWER = 0, OP_N = 0, OP_T = 1;
    POPT_LIB(L.ssyrk(L.blas[dev], LOWER, OP_T, (int)n_a, (int)K, &one, a_dm, (int)K, &zero, g, (int)n_a));
    note_launch();
    popt_add_diagonal_kernel<<<(unsigned)((n_a + 255) / 256), 256, 0, s>>>(g, (int)n_a, (float)lambda);
    POPT_CUDA(cudaGetLastError());
    POPT_LIB(L.sgemm(L.blas[dev], OP_T, OP_N, (int)n_a, (int)n_l, (int)K, &one, a_dm, (int)K, a_l, (int)K, &zero, d_popt, (int)ld));
    int lwork = 0;
    POPT_LIB(L.potrfSize(L.sol[dev], LOWER, (int)n_a, g, (int)n_a, &lwork));
    POPT_CUDA(mem.get(reinterpret_cast<void **>(&work), sizeof(float) * (size_t)std::max(lwork, 1)));
    POPT_LIB(L.potrf(L.sol[dev], LOWER, (int)n_a, g, (int)n_a, work, lwork, info));
    POPT_LIB(L.potrs(L.sol[dev], LOWER, (int)n_a, (int)n_l, g, (int)n_a, d_popt, (int)ld, info + 1));
    int h_info[2] = {0, 0};
    POPT_CUDA(cudaMemcpyAsync(h_info, info, sizeof(h_info), cudaMemcpyDeviceToHost, s));
    POPT_CUDA(cudaStreamSynchronize(s));
    if (h_info[0] != 0)
        return report(SYNIM_ERR_INVALID_ARG, "synim_projection_matrix: P_DM^T P_DM + lambda I is not positive definite (Cholesky stopped at %d): "
                                             "raise lambda", h_info[0]);
    if (h_info[1] != 0) return report(SYNIM_ERR_CUDA, "synim_projection_matrix: triangular solve failed (%d)", h_info[1]);
    return SYNIM_OK;
}
