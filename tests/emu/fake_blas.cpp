// fake_blas.cpp -- TEST INFRASTRUCTURE (tests/emu/README.md): CPU stand-ins for the few cuBLAS / cuSOLVER entry points
// synim_popt.cu loads with dlopen, built as libcublas.so.12 / libcusolver.so.11 for the emulated library only.
#include <cmath>
#include <cstdlib>
extern "C" {
int cublasCreate_v2(void **h) { *h = malloc(8); return 0; }
int cublasSetStream_v2(void *, void *) { return 0; }
// C (n x n, lower) = alpha * A^T A + beta * C with A k x n column-major (trans = T)
int cublasSsyrk_v2(void *, int uplo, int trans, int n, int k, const float *alpha, const float *A, int lda, const float *beta, float *C, int ldc)
{
    if (uplo != 0 || trans != 1) return 7;
    for (int j = 0; j < n; ++j)
        for (int i = j; i < n; ++i) {
            double acc = 0;
            for (int q = 0; q < k; ++q) acc += (double)A[(size_t)i * lda + q] * A[(size_t)j * lda + q];
            C[(size_t)j * ldc + i] = (float)(*alpha * acc + (*beta != 0.f ? *beta * C[(size_t)j * ldc + i] : 0.0));
        }
    return 0;
}
// C (m x n) = alpha * A^T B + beta * C, A k x m, B k x n (transa = T, transb = N)
int cublasSgemm_v2(void *, int ta, int tb, int m, int n, int k, const float *alpha, const float *A, int lda, const float *B, int ldb,
                   const float *beta, float *C, int ldc)
{
    if (ta != 1 || tb != 0) return 7;
    for (int j = 0; j < n; ++j)
        for (int i = 0; i < m; ++i) {
            double acc = 0;
            for (int q = 0; q < k; ++q) acc += (double)A[(size_t)i * lda + q] * B[(size_t)j * ldb + q];
            C[(size_t)j * ldc + i] = (float)(*alpha * acc + (*beta != 0.f ? *beta * C[(size_t)j * ldc + i] : 0.0));
        }
    return 0;
}
int cusolverDnCreate(void **h) { *h = malloc(8); return 0; }
int cusolverDnSetStream(void *, void *) { return 0; }
int cusolverDnSpotrf_bufferSize(void *, int, int n, float *, int, int *lwork) { *lwork = n; return 0; }
int cusolverDnSpotrf(void *, int uplo, int n, float *A, int lda, float *, int, int *info)
{
    if (uplo != 0) return 7;
    *info = 0;
    for (int j = 0; j < n; ++j) {
        double d = A[(size_t)j * lda + j];
        for (int q = 0; q < j; ++q) d -= (double)A[(size_t)q * lda + j] * A[(size_t)q * lda + j];
        if (!(d > 0)) { *info = j + 1; return 0; }
        const float l = (float)std::sqrt(d);
        A[(size_t)j * lda + j] = l;
        for (int i = j + 1; i < n; ++i) {
            double v = A[(size_t)j * lda + i];
            for (int q = 0; q < j; ++q) v -= (double)A[(size_t)q * lda + i] * A[(size_t)q * lda + j];
            A[(size_t)j * lda + i] = (float)(v / l);
        }
    }
    return 0;
}
int cusolverDnSpotrs(void *, int uplo, int n, int nrhs, const float *A, int lda, float *B, int ldb, int *info)
{
    if (uplo != 0) return 7;
    *info = 0;
    for (int r = 0; r < nrhs; ++r) {
        float *b = B + (size_t)r * ldb;
        for (int i = 0; i < n; ++i) {   // L y = b
            double v = b[i];
            for (int q = 0; q < i; ++q) v -= (double)A[(size_t)q * lda + i] * b[q];
            b[i] = (float)(v / A[(size_t)i * lda + i]);
        }
        for (int i = n - 1; i >= 0; --i) {   // L^T x = y
            double v = b[i];
            for (int q = i + 1; q < n; ++q) v -= (double)A[(size_t)i * lda + q] * b[q];
            b[i] = (float)(v / A[(size_t)i * lda + i]);
        }
    }
    return 0;
}
}
