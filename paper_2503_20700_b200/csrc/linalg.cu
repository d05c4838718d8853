// Dense SVD of one sector matrix on the device (cuSOLVER gesvd: a library call), wrapped for
// row-major storage.  Row-major A [m x n] is column-major A^T [n x m]; gesvd needs rows >= cols, so for n >= m the
// factors of A^T are read back directly as (Vt, U), and for n < m the matrix is transposed first.
#include <cuda_runtime.h>
#include <cusolverDn.h>

#include <cstdlib>
#include <stdexcept>
#include <string>

#include "kernels.hpp"

namespace dmrg {

struct SvdWork {
    cusolverDnHandle_t h = nullptr;
    double* work = nullptr;
    int lwork = 0;
    double* scratch = nullptr;      // transposed input / outputs
    size_t scratch_n = 0;
    int* info = nullptr;
    gesvdjInfo_t jparams = nullptr; // one-sided Jacobi SVD: much faster than QR-iteration gesvd at sector sizes (<= ~1600)
    double* jwork = nullptr;
    int jlwork = 0;
    bool use_jacobi = true;
};

static void cs_check(cusolverStatus_t s, const char* what) {
    if (s != CUSOLVER_STATUS_SUCCESS) throw std::runtime_error(std::string(what) + ": cuSOLVER status " + std::to_string((int)s));
}
static void cu_check(cudaError_t e, const char* what) {
    if (e != cudaSuccess) throw std::runtime_error(std::string(what) + ": " + cudaGetErrorString(e));
}

SvdWork* svd_create(cudaStream_t st, bool jacobi) {
    SvdWork* w = new SvdWork();
    cs_check(cusolverDnCreate(&w->h), "cusolverDnCreate");
    cs_check(cusolverDnSetStream(w->h, st), "cusolverDnSetStream");
    cu_check(cudaMalloc(&w->info, sizeof(int)), "cudaMalloc");
    cs_check(cusolverDnCreateGesvdjInfo(&w->jparams), "CreateGesvdjInfo");
    cs_check(cusolverDnXgesvdjSetSortEig(w->jparams, 1), "gesvdj sort");
    cs_check(cusolverDnXgesvdjSetMaxSweeps(w->jparams, 100), "gesvdj sweeps");
    w->use_jacobi = jacobi;
    return w;
}
void svd_destroy(SvdWork* w) {
    if (!w) return;
    if (w->work) cudaFree(w->work);
    if (w->scratch) cudaFree(w->scratch);
    if (w->info) cudaFree(w->info);
    if (w->jwork) cudaFree(w->jwork);
    if (w->jparams) cusolverDnDestroyGesvdjInfo(w->jparams);
    if (w->h) cusolverDnDestroy(w->h);
    delete w;
}

// Jacobi path.  Row-major A [m x n] is column-major A^T (n x m) = U' S V'^T (economy, r = min(m, n)); then Vt = U'^T,
// which is U' (ld n) read row-major, and U = V', which is V' (column-major m x r) transposed once.
// Returns false when the sweeps did not converge (the caller falls back to gesvd on a saved copy).
static bool svd_jacobi(SvdWork* w, double* A, int m, int n, double* U, double* S, double* Vt, cudaStream_t st) {
    const int r = m < n ? m : n;
    const size_t need = (size_t)m * r + (size_t)m * n;
    if (need > w->scratch_n) {
        if (w->scratch) cudaFree(w->scratch);
        cu_check(cudaMalloc(&w->scratch, sizeof(double) * need), "cudaMalloc");
        w->scratch_n = need;
    }
    double* Vp = w->scratch;                      // V' column-major (m x r)
    double* Acopy = w->scratch + (size_t)m * r;   // gesvdj destroys its input: keep a copy for the fallback
    cu_check(cudaMemcpyAsync(Acopy, A, sizeof(double) * (size_t)m * n, cudaMemcpyDeviceToDevice, st), "svd copy");
    int lwork = 0;
    cs_check(cusolverDnDgesvdj_bufferSize(w->h, CUSOLVER_EIG_MODE_VECTOR, 1, n, m, A, n, S, Vt, n, Vp, m, &lwork, w->jparams),
             "gesvdj_bufferSize");
    if (lwork > w->jlwork) {
        if (w->jwork) cudaFree(w->jwork);
        cu_check(cudaMalloc(&w->jwork, sizeof(double) * (size_t)lwork), "cudaMalloc");
        w->jlwork = lwork;
    }
    cs_check(cusolverDnDgesvdj(w->h, CUSOLVER_EIG_MODE_VECTOR, 1, n, m, A, n, S, Vt, n, Vp, m, w->jwork, w->jlwork, w->info,
                               w->jparams), "gesvdj");
    int info = 0;
    cu_check(cudaMemcpyAsync(&info, w->info, sizeof(int), cudaMemcpyDeviceToHost, st), "gesvdj info");
    cu_check(cudaStreamSynchronize(st), "gesvdj");
    if (info != 0) {                              // not converged (info = r + 1) or bad argument: restore A
        cu_check(cudaMemcpyAsync(A, Acopy, sizeof(double) * (size_t)m * n, cudaMemcpyDeviceToDevice, st), "svd restore");
        return false;
    }
    launch_transpose(Vp, r, m, m, U, st);         // V' read row-major is [r x m]; U [m x r] is its transpose
    return true;
}

void svd_rowmajor(SvdWork* w, double* A, int m, int n, double* U, double* S, double* Vt, cudaStream_t st) {
    if (m <= 0 || n <= 0) return;
    if (w->use_jacobi && svd_jacobi(w, A, m, n, U, S, Vt, st)) return;
    const int big = m > n ? m : n, small = m > n ? n : m;     // column-major problem is big x small
    int lwork = 0;
    cs_check(cusolverDnDgesvd_bufferSize(w->h, big, small, &lwork), "gesvd_bufferSize");
    if (lwork > w->lwork) {
        if (w->work) cudaFree(w->work);
        cu_check(cudaMalloc(&w->work, sizeof(double) * (size_t)lwork), "cudaMalloc");
        w->lwork = lwork;
    }
    if (n >= m) {
        // column-major A^T (n x m) = U' S V'^T;  U' (ld n) read row-major is Vt [m x n];  V'^T (ld m) read row-major is U
        cs_check(cusolverDnDgesvd(w->h, 'S', 'S', n, m, A, n, S, Vt, n, U, m, w->work, w->lwork, nullptr, w->info), "gesvd");
    } else {
        const size_t need = (size_t)m * n * 2 + (size_t)n * n;
        if (need > w->scratch_n) {
            if (w->scratch) cudaFree(w->scratch);
            cu_check(cudaMalloc(&w->scratch, sizeof(double) * need), "cudaMalloc");
            w->scratch_n = need;
        }
        double* At = w->scratch;                 // row-major [n x m] = column-major A (m x n)
        double* Ut = At + (size_t)m * n;         // column-major U (m x n) = row-major U^T [n x m]
        double* V = Ut + (size_t)m * n;          // column-major V^T (n x n) = row-major V [n x n]
        launch_transpose(A, m, n, n, At, st);
        cs_check(cusolverDnDgesvd(w->h, 'S', 'S', m, n, At, m, S, Ut, m, V, n, w->work, w->lwork, nullptr, w->info), "gesvd");
        launch_transpose(Ut, n, m, m, U, st);    // U [m x n]
        launch_transpose(V, n, n, n, Vt, st);    // Vt [n x n]
    }
    int info = 0;
    cu_check(cudaMemcpyAsync(&info, w->info, sizeof(int), cudaMemcpyDeviceToHost, st), "gesvd info");
    cu_check(cudaStreamSynchronize(st), "gesvd");
    if (info != 0) throw std::runtime_error("gesvd did not converge (info " + std::to_string(info) + ")");
}

}  // namespace dmrg
