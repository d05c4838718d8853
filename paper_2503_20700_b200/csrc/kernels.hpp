// Launchers of the sm_100a CUDA kernels (the only place tensor arithmetic happens).  Implemented in seg_gemm_tma.cu,
// seg_gemm.cu, vec_kernels.cu and linalg.cu (the integer block-map kernels are in heff_maps.cu / maps.hpp).  All pointers are device pointers unless a name ends in _host.
#pragma once
#include <cuda_runtime_api.h>

#include <cstdint>

namespace dmrg {

// ---- grouped, K-segmented FP64 GEMM on the FP64 tensor pipe (DMMA.8x8x4) -------------------------------------------
//   C_task[M x N] (+)= sum_{seg in task} alpha_seg * op(A_seg)[M x K_seg] * op(B_seg)[K_seg x N]
// One CTA owns one output tile of one task and walks the task's segment list (ownership by output tile: no
// atomics, deterministic summation order).  This single kernel executes every dense contraction of the path:
// H_eff psi (phase 1: T = O_L X or X O_R^T; phase 2: Y += sum_t c_t T_t O_R^T / O_L T_t, K-concatenated over
// terms), operator renormalisation, the integral-weighted linear combinations of operator stacks, the two-site
// tensor products and the RDM contractions.
enum : int { SEG_TRANS_A = 1,   // A stored [K x M] row-major (used transposed)
             SEG_TRANS_B = 2,   // B stored [N x K] row-major (used transposed); otherwise [K x N] row-major
             SEG_IDENT_B = 4 }; // B = identity: C += alpha * A, A stored [M x N] row-major
enum : int { TASK_ACCUM = 1 };  // C += ... instead of C = ...

struct Seg {
    const double* A;
    const double* B;
    int lda, ldb;
    int K;
    int flags;
    double alpha;
};
struct Task {
    double* C;
    int ldc, M, N;
    int seg_begin, seg_count;
    int flags;
    int ngemm;                  // segments [seg_begin, seg_begin + ngemm) are GEMM segments, the rest identity-B (set by finalize)
};
struct Tile {                   // output tile [m0, m0+mv) x [n0, n0+nv) of a task; m0, n0 multiples of 8, mv <= BM, nv <= BN
    int task, m0, n0, mv, nv;
};
constexpr int GEMM_BM = 64, GEMM_BN = 64, GEMM_BK = 16, GEMM_THREADS = 128, GEMM_STAGES = 4;

void launch_seg_gemm(const Task* tasks, const Seg* segs, const Tile* tiles, int ntiles, cudaStream_t st);
// Same contract, bulk-copy (TMA engine) fed, warp-specialised, persistent with a dynamic tile counter (seg_gemm_tma.cu).
// Needs every GEMM operand 16-byte aligned with an even leading dimension; `counter` is one device int of scratch.
void launch_seg_gemm_tma(const Task* tasks, const Seg* segs, const Tile* tiles, int ntiles, int* counter, cudaStream_t st);

// ---- vector kernels (Davidson; HBM-bound) ---------------------------------------------------------------------------
// out[j] = sum_i x[i] * Y[j*ldy + i], j < m  (deterministic two-stage reduction; out is a device array of m doubles)
// scratch: multi_dot_scratch() doubles owned by the caller (one per context: no process-global buffers)
int64_t multi_dot_scratch();
void launch_multi_dot(const double* x, const double* Y, int64_t ldy, int m, int64_t n, double* out, double* scratch,
                      cudaStream_t st);
constexpr int COMBINE_MAX = 32;
// out[i] = beta * out[i] + sum_{j<m} coef_host[j] * V[j*ldv + i],  m <= COMBINE_MAX
void launch_combine(double* out, double beta, const double* V, int64_t ldv, int m, const double* coef_host, int64_t n,
                    cudaStream_t st);
// t[i] = r[i] / clamp(diag[i] - theta), |denominator| floored at `floor` keeping its sign (reading S13)
void launch_precond(const double* r, const double* diag, double theta, double floor, double* t, int64_t n,
                    cudaStream_t st);
void launch_scale(double a, double* x, int64_t n, cudaStream_t st);

// diag(H_eff): for psi block b (rows x cols at off), d[off + i*cols + j] = sum_{items of b} c * ml[i*(ldl+1)] *
// mr[j*(ldr+1)] with a null ml / mr standing for the identity.
struct DiagItemK { const double* ml; int ldl; const double* mr; int ldr; double c; };
void launch_heff_diag(double* d, int nblocks, const int64_t* blk_off, const int* blk_rows, const int* blk_cols,
                      const int* item_ptr, const DiagItemK* items, cudaStream_t st);

// dst block b (at dst_off[b], row stride pad2(cols[b])) = src block b (at src_off[b], packed [rows x cols]); pads untouched
void launch_pad_blocks(double* dst, const double* src, int nblocks, const int64_t* dst_off, const int64_t* src_off,
                       const int* rows, const int* cols, cudaStream_t st);

// ---- small dense helpers ---------------------------------------------------------------------------------------------
// out[c*rows + r] = in[r*ld_in + c]   (out is [cols x rows] contiguous)
void launch_transpose(const double* in, int rows, int cols, int ld_in, double* out, cudaStream_t st);
// dst[r*ld_dst + c] = alpha * src[r*ld_src + c] * (row_scale ? row_scale[r] : 1) * (col_scale ? col_scale[c] : 1)
void launch_copy2d(double* dst, int ld_dst, const double* src, int ld_src, int rows, int cols, double alpha,
                   const double* row_scale, const double* col_scale, cudaStream_t st);
// RDM accumulation for few right-hand sides: E[r*ldE + c] = sum_k S[r*lds + k] * M[c*ldm + k], r < nrows, c < nc <= 8,
// k < K.  Streams every row of S (a stack of stored operators) once with coalesced 16-byte loads, warp-level shuffle
// reductions, fixed-order partial sums: HBM-bound (vec_kernels.cu).  S, M 16-byte aligned, lds, ldm even.
// scratch: stack_dots_scratch(nrows, nc, K) doubles.
int64_t stack_dots_scratch(int nrows, int nc, int64_t K, int64_t* span_out = nullptr, int* nspans_out = nullptr);
void launch_stack_dots(const double* S, int64_t lds, int nrows, const double* M, int64_t ldm, int nc, int64_t K, double* E,
                       int ldE, double* scratch, cudaStream_t st);

// ---- dense SVD of a row-major [m x n] matrix (cuSOLVER gesvd; library call) -----------------------
// U [m x r], S [r], Vt [r x n] row-major, r = min(m, n); A is destroyed.  work: opaque per-engine handle.
struct SvdWork;
SvdWork* svd_create(cudaStream_t st, bool jacobi);   // jacobi: gesvdj (gesvd fallback), else gesvd
void svd_destroy(SvdWork* w);
void svd_rowmajor(SvdWork* w, double* A, int m, int n, double* U, double* S, double* Vt, cudaStream_t st);

}  // namespace dmrg
