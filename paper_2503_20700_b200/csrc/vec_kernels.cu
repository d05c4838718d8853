// HBM-bound vector kernels of the Davidson driver and small dense helpers.
// Coalesced, 16-byte vectorised where alignment allows, warp-shuffle reductions, deterministic two-stage sums
// (fixed grid -> fixed partial-sum order; no floating-point atomics).
#include <cuda_runtime.h>

#include "kernels.hpp"

namespace dmrg {

namespace {

constexpr int RED_THREADS = 256;
constexpr int RED_BLOCKS = 592;     // 148 SMs x 4: one wave of resident CTAs

__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
    return v;
}
__device__ __forceinline__ double block_sum(double v, double* sh) {
    v = warp_sum(v);
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    if (lane == 0) sh[warp] = v;
    __syncthreads();
    double r = 0.0;
    if (warp == 0) {
        r = lane < (blockDim.x >> 5) ? sh[lane] : 0.0;
        r = warp_sum(r);
    }
    __syncthreads();
    return r;   // valid on thread 0
}

// partial[j * gridDim.x + b] = sum over this block's slice of x * Y_j
__global__ void __launch_bounds__(RED_THREADS) multi_dot_stage1(const double* __restrict__ x, const double* __restrict__ Y,
                                                                int64_t ldy, int m, int64_t n, double* __restrict__ partial) {
    __shared__ double sh[RED_THREADS / 32];
    const int64_t stride = (int64_t)gridDim.x * blockDim.x;
    for (int j = 0; j < m; ++j) {
        const double* y = Y + (int64_t)j * ldy;
        double acc = 0.0;
        for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += stride) acc += x[i] * y[i];
        acc = block_sum(acc, sh);
        if (threadIdx.x == 0) partial[(int64_t)j * gridDim.x + blockIdx.x] = acc;
    }
}
__global__ void __launch_bounds__(RED_THREADS) multi_dot_stage2(const double* __restrict__ partial, int nb, double* __restrict__ out) {
    __shared__ double sh[RED_THREADS / 32];
    const int j = blockIdx.x;
    double acc = 0.0;
    for (int i = threadIdx.x; i < nb; i += blockDim.x) acc += partial[(int64_t)j * nb + i];
    acc = block_sum(acc, sh);
    if (threadIdx.x == 0) out[j] = acc;
}

struct Coefs { double c[COMBINE_MAX]; };
__global__ void __launch_bounds__(256) combine_kernel(double* __restrict__ out, double beta, const double* __restrict__ V,
                                                      int64_t ldv, int m, Coefs cf, int64_t n) {
    const int64_t stride = (int64_t)gridDim.x * blockDim.x;
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += stride) {
        double s = beta == 0.0 ? 0.0 : beta * out[i];
        for (int j = 0; j < m; ++j) s += cf.c[j] * V[(int64_t)j * ldv + i];
        out[i] = s;
    }
}
__global__ void __launch_bounds__(256) precond_kernel(const double* __restrict__ r, const double* __restrict__ diag, double theta,
                                                      double floor_, double* __restrict__ t, int64_t n) {
    const int64_t stride = (int64_t)gridDim.x * blockDim.x;
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += stride) {
        double den = diag[i] - theta;
        if (fabs(den) < floor_) den = den < 0.0 ? -floor_ : floor_;
        t[i] = r[i] / den;
    }
}
__global__ void __launch_bounds__(256) scale_kernel(double a, double* __restrict__ x, int64_t n) {
    const int64_t stride = (int64_t)gridDim.x * blockDim.x;
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += stride) x[i] *= a;
}

// one CTA per psi block (grid-strided over blocks); the diagonals of the operator blocks are staged in registers per item
__global__ void __launch_bounds__(256) heff_diag_kernel(double* __restrict__ d, int nblocks, const int64_t* __restrict__ off,
                                                        const int* __restrict__ rows, const int* __restrict__ cols,
                                                        const int* __restrict__ ptr, const DiagItemK* __restrict__ items) {
    for (int b = blockIdx.x; b < nblocks; b += gridDim.x) {
        const int R = rows[b], Cc = cols[b];
        const int64_t total = (int64_t)R * Cc;
        for (int64_t e = threadIdx.x; e < total; e += blockDim.x) {
            const int i = (int)(e / Cc), j = (int)(e % Cc);
            double s = 0.0;
            for (int t = ptr[b]; t < ptr[b + 1]; ++t) {
                const DiagItemK it = items[t];
                const double l = it.ml ? it.ml[(size_t)i * (it.ldl + 1)] : 1.0;
                const double r = it.mr ? it.mr[(size_t)j * (it.ldr + 1)] : 1.0;
                s += it.c * l * r;
            }
            d[off[b] + e] = s;
        }
    }
}

// one CTA per block (grid-strided): packed [rows x cols] -> row stride pad2(cols)
__global__ void __launch_bounds__(256) pad_blocks_kernel(double* __restrict__ dst, const double* __restrict__ src, int nblocks,
                                                         const int64_t* __restrict__ doff, const int64_t* __restrict__ soff,
                                                         const int* __restrict__ rows, const int* __restrict__ cols) {
    for (int b = blockIdx.x; b < nblocks; b += gridDim.x) {
        const int R = rows[b], Cc = cols[b], ld = (Cc + 1) & ~1;
        const int64_t total = (int64_t)R * Cc;
        const double* s = src + soff[b];
        double* d = dst + doff[b];
        for (int64_t e = threadIdx.x; e < total; e += blockDim.x) {
            const int i = (int)(e / Cc), j = (int)(e % Cc);
            d[(size_t)i * ld + j] = s[e];
        }
    }
}

__global__ void transpose_kernel(const double* __restrict__ in, int rows, int cols, int ld, double* __restrict__ out) {
    __shared__ double tile[32][33];
    const int c0 = blockIdx.x * 32, r0 = blockIdx.y * 32;
    for (int j = threadIdx.y; j < 32; j += blockDim.y) {
        const int r = r0 + j, c = c0 + threadIdx.x;
        if (r < rows && c < cols) tile[j][threadIdx.x] = in[(size_t)r * ld + c];
    }
    __syncthreads();
    for (int j = threadIdx.y; j < 32; j += blockDim.y) {
        const int c = c0 + j, r = r0 + threadIdx.x;
        if (r < rows && c < cols) out[(size_t)c * rows + r] = tile[threadIdx.x][j];
    }
}
__global__ void __launch_bounds__(256) copy2d_kernel(double* __restrict__ dst, int ldd, const double* __restrict__ src, int lds,
                                                     int rows, int cols, double alpha, const double* __restrict__ rs,
                                                     const double* __restrict__ cs) {
    const int64_t total = (int64_t)rows * cols, stride = (int64_t)gridDim.x * blockDim.x;
    for (int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; e < total; e += stride) {
        const int r = (int)(e / cols), c = (int)(e % cols);
        dst[(size_t)r * ldd + c] = alpha * src[(size_t)r * lds + c] * (rs ? rs[r] : 1.0) * (cs ? cs[c] : 1.0);
    }
}

// RDM accumulation: one warp per block pair streams both blocks with coalesced loads and reduces with shuffles;
// pairs are sorted by target and each target is owned by exactly one contiguous run handled by one CTA pass, so
// out[target] is updated without atomics by the lane-0 thread of the first warp of the run's CTA.
__global__ void __launch_bounds__(256) block_dots_kernel(const DotPair* __restrict__ pairs, int npairs, double* __restrict__ partial) {
    const int warp = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, lane = threadIdx.x & 31;
    const int nwarps = (gridDim.x * blockDim.x) >> 5;
    for (int p = warp; p < npairs; p += nwarps) {
        const DotPair d = pairs[p];
        double acc = 0.0;
        if (d.lda == d.cols && d.ldb == d.cols) {
            const int64_t total = (int64_t)d.rows * d.cols;
            for (int64_t e = lane; e < total; e += 32) acc += d.A[e] * d.B[e];
        } else {
            for (int i = 0; i < d.rows; ++i)
                for (int j = lane; j < d.cols; j += 32) acc += d.A[(size_t)i * d.lda + j] * d.B[(size_t)i * d.ldb + j];
        }
        acc = warp_sum(acc);
        if (lane == 0) partial[p] = d.alpha * acc;
    }
}
// out[target] += sum of partial[p] over the pairs of that target, in pair order (one thread per target run)
__global__ void block_dots_reduce(const DotPair* __restrict__ pairs, int npairs, const double* __restrict__ partial,
                                  double* __restrict__ out) {
    const int p = blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= npairs) return;
    if (p > 0 && pairs[p - 1].target == pairs[p].target) return;     // not the head of a run
    const int tgt = pairs[p].target;
    double s = 0.0;
    for (int q = p; q < npairs && pairs[q].target == tgt; ++q) s += partial[q];
    out[tgt] += s;
}

int grid_for(int64_t n, int threads) {
    int64_t b = (n + threads - 1) / threads;
    if (b < 1) b = 1;
    if (b > RED_BLOCKS * 4) b = RED_BLOCKS * 4;
    return (int)b;
}

double* g_partial = nullptr;    // scratch of the two-stage reductions (COMBINE_MAX x RED_BLOCKS doubles)
double* g_pair_partial = nullptr;
size_t g_pair_cap = 0;

}  // namespace

void launch_multi_dot(const double* x, const double* Y, int64_t ldy, int m, int64_t n, double* out, cudaStream_t st) {
    if (m <= 0) return;
    if (!g_partial) cudaMalloc(&g_partial, sizeof(double) * 64 * RED_BLOCKS);
    int nb = grid_for(n, RED_THREADS);
    if (nb > RED_BLOCKS) nb = RED_BLOCKS;
    for (int j0 = 0; j0 < m; j0 += 64) {
        const int mm = m - j0 < 64 ? m - j0 : 64;
        multi_dot_stage1<<<nb, RED_THREADS, 0, st>>>(x, Y + (int64_t)j0 * ldy, ldy, mm, n, g_partial);
        multi_dot_stage2<<<mm, RED_THREADS, 0, st>>>(g_partial, nb, out + j0);
    }
}
void launch_combine(double* out, double beta, const double* V, int64_t ldv, int m, const double* coef_host, int64_t n,
                    cudaStream_t st) {
    Coefs cf;
    for (int j = 0; j < COMBINE_MAX; ++j) cf.c[j] = j < m ? coef_host[j] : 0.0;
    combine_kernel<<<grid_for(n, 256), 256, 0, st>>>(out, beta, V, ldv, m, cf, n);
}
void launch_precond(const double* r, const double* diag, double theta, double floor_, double* t, int64_t n, cudaStream_t st) {
    precond_kernel<<<grid_for(n, 256), 256, 0, st>>>(r, diag, theta, floor_, t, n);
}
void launch_scale(double a, double* x, int64_t n, cudaStream_t st) { scale_kernel<<<grid_for(n, 256), 256, 0, st>>>(a, x, n); }
void launch_heff_diag(double* d, int nblocks, const int64_t* off, const int* rows, const int* cols, const int* ptr,
                      const DiagItemK* items, cudaStream_t st) {
    if (nblocks <= 0) return;
    heff_diag_kernel<<<nblocks < 2368 ? nblocks : 2368, 256, 0, st>>>(d, nblocks, off, rows, cols, ptr, items);
}
void launch_pad_blocks(double* dst, const double* src, int nblocks, const int64_t* dst_off, const int64_t* src_off,
                       const int* rows, const int* cols, cudaStream_t st) {
    if (nblocks <= 0) return;
    pad_blocks_kernel<<<nblocks < 2368 ? nblocks : 2368, 256, 0, st>>>(dst, src, nblocks, dst_off, src_off, rows, cols);
}
void launch_transpose(const double* in, int rows, int cols, int ld, double* out, cudaStream_t st) {
    if (rows <= 0 || cols <= 0) return;
    dim3 grid((cols + 31) / 32, (rows + 31) / 32), block(32, 8);
    transpose_kernel<<<grid, block, 0, st>>>(in, rows, cols, ld, out);
}
void launch_copy2d(double* dst, int ldd, const double* src, int lds, int rows, int cols, double alpha, const double* rs,
                   const double* cs, cudaStream_t st) {
    if (rows <= 0 || cols <= 0) return;
    copy2d_kernel<<<grid_for((int64_t)rows * cols, 256), 256, 0, st>>>(dst, ldd, src, lds, rows, cols, alpha, rs, cs);
}
void launch_block_dots(const DotPair* pairs, int npairs, double* out, cudaStream_t st) {
    if (npairs <= 0) return;
    if ((size_t)npairs > g_pair_cap) {
        if (g_pair_partial) cudaFree(g_pair_partial);
        g_pair_cap = (size_t)npairs * 2;
        cudaMalloc(&g_pair_partial, sizeof(double) * g_pair_cap);
    }
    int blocks = (npairs + 7) / 8;
    if (blocks > RED_BLOCKS * 2) blocks = RED_BLOCKS * 2;
    block_dots_kernel<<<blocks, 256, 0, st>>>(pairs, npairs, g_pair_partial);
    block_dots_reduce<<<(npairs + 255) / 256, 256, 0, st>>>(pairs, npairs, g_pair_partial, out);
}

}  // namespace dmrg
