// Dense SVD of one sector matrix on the device (cuSOLVER gesvd: a library call), wrapped for
// row-major storage.  Row-major A [m x n] is column-major A^T [n x m]; gesvd needs rows >= cols, so for n >= m the
// factors of A^T are read back directly as (Vt, U), and for n < m the matrix is transposed first.
#include <cuda_runtime.h>
#include <cusolverDn.h>

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
};

static void cs_check(cusolverStatus_t s, const char* what) {
    if (s != CUSOLVER_STATUS_SUCCESS) throw std::runtime_error(std::string(what) + ": cuSOLVER status " + std::to_string((int)s));
}
static void cu_check(cudaError_t e, const char* what) {
    if (e != cudaSuccess) throw std::runtime_error(std::string(what) + ": " + cudaGetErrorString(e));
}

SvdWork* svd_create(cudaStream_t st) {
    SvdWork* w = new SvdWork();
    cs_check(cusolverDnCreate(&w->h), "cusolverDnCreate");
    cs_check(cusolverDnSetStream(w->h, st), "cusolverDnSetStream");
    cu_check(cudaMalloc(&w->info, sizeof(int)), "cudaMalloc");
    return w;
}
void svd_destroy(SvdWork* w) {
    if (!w) return;
    if (w->work) cudaFree(w->work);
    if (w->scratch) cudaFree(w->scratch);
    if (w->info) cudaFree(w->info);
    if (w->h) cusolverDnDestroy(w->h);
    delete w;
}

void svd_rowmajor(SvdWork* w, double* A, int m, int n, double* U, double* S, double* Vt, cudaStream_t st) {
    if (m <= 0 || n <= 0) return;
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
