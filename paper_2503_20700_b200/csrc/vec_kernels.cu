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

// one CTA per psi block (grid-strided over blocks).  The diagonals of the operator blocks of a tile of items are
// gathered once into shared memory (R + C strided loads per item instead of two per element and item), then every
// element adds  c_t l_t[i] r_t[j]  in item order (the same summation order as a plain loop over the items).
constexpr int DIAG_SH = 6000;                      // doubles of staging: items per tile = DIAG_SH / (R + C), at most 16
__global__ void __launch_bounds__(256) heff_diag_kernel(double* __restrict__ d, int nblocks, const int64_t* __restrict__ off,
                                                        const int* __restrict__ rows, const int* __restrict__ cols,
                                                        const int* __restrict__ ptr, const DiagItemK* __restrict__ items) {
    __shared__ double sh[DIAG_SH];
    __shared__ double sc[16];
    for (int b = blockIdx.x; b < nblocks; b += gridDim.x) {
        const int R = rows[b], Cc = cols[b];
        const int64_t total = (int64_t)R * Cc;
        double* out = d + off[b];
        const int t0 = ptr[b], t1 = ptr[b + 1];
        if (t1 == t0) { for (int64_t e = threadIdx.x; e < total; e += blockDim.x) out[e] = 0.0; continue; }
        int DT = DIAG_SH / (R + Cc);
        if (DT > 16) DT = 16;
        if (DT < 1) {                              // a block too wide for the staging buffer: direct loop
            for (int64_t e = threadIdx.x; e < total; e += blockDim.x) {
                const int i = (int)(e / Cc), j = (int)(e % Cc);
                double s = 0.0;
                for (int t = t0; t < t1; ++t) {
                    const DiagItemK it = items[t];
                    const double l = it.ml ? it.ml[(size_t)i * (it.ldl + 1)] : 1.0;
                    const double r = it.mr ? it.mr[(size_t)j * (it.ldr + 1)] : 1.0;
                    s += it.c * l * r;
                }
                out[e] = s;
            }
            continue;
        }
        for (int tb = t0; tb < t1; tb += DT) {
            const int nt = min(DT, t1 - tb);
            __syncthreads();                       // previous tile (and previous block) fully consumed
            for (int q = threadIdx.x; q < nt * (R + Cc); q += blockDim.x) {
                const int t = q / (R + Cc), x = q % (R + Cc);
                const DiagItemK& it = items[tb + t];
                double v;
                if (x < R) v = it.ml ? it.ml[(size_t)x * (it.ldl + 1)] : 1.0;
                else       v = it.mr ? it.mr[(size_t)(x - R) * (it.ldr + 1)] : 1.0;
                sh[q] = v;
            }
            if (threadIdx.x < nt) sc[threadIdx.x] = items[tb + threadIdx.x].c;
            __syncthreads();
            for (int64_t e = threadIdx.x; e < total; e += blockDim.x) {
                const int i = (int)(e / Cc), j = (int)(e % Cc);
                double s = tb == t0 ? 0.0 : out[e];
                for (int t = 0; t < nt; ++t) s += sc[t] * sh[t * (R + Cc) + i] * sh[t * (R + Cc) + R + j];
                out[e] = s;
            }
        }
        __syncthreads();
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

// RDM accumulation for few right-hand sides:
//   E[r][c] = sum_k S[r][k] * M[c][k],   r < nrows (stored operators = rows of a stack), c < NC <= 8, k < K
// HBM-bound: every stored operator is streamed exactly once with coalesced 16-byte loads (one warp reads 512
// contiguous bytes of a row per instruction), the NC vectors M are staged chunk by chunk in shared memory and shared by
// the 32 rows of the CTA, each lane keeps 2 x NC running sums, and a warp-level shuffle reduction ends every K span.
// Partial sums of the K spans are added by a second kernel in span order (no atomics: bit-reproducible).
constexpr int SD_WARPS = 16, SD_KC = 1024;        // 16 warps = 32 rows per CTA; 1024 doubles of every M vector per chunk
template <int NC>
__global__ void __launch_bounds__(SD_WARPS * 32, 2) stack_dots_kernel(const double* __restrict__ S, int64_t lds, int nrows,
                                                                   const double* __restrict__ M, int64_t ldm, int nc, int64_t K,
                                                                   int64_t span, int nspans, double* __restrict__ partial) {
    extern __shared__ __align__(16) double sm[];          // [NC][SD_KC]
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int nrb = (nrows + 2 * SD_WARPS - 1) / (2 * SD_WARPS);
    for (int64_t item = blockIdx.x; item < (int64_t)nrb * nspans; item += gridDim.x) {
        const int rb = (int)(item % nrb), sp = (int)(item / nrb);
        const int r0 = rb * 2 * SD_WARPS + 2 * warp;        // this warp's row pair
        const bool v0 = r0 < nrows, v1 = r0 + 1 < nrows;
        const double* s0 = S + (size_t)r0 * lds;
        const double* s1 = s0 + lds;
        const int64_t kbeg = (int64_t)sp * span, kend = kbeg + span < K ? kbeg + span : K;
        double acc0[NC], acc1[NC];
#pragma unroll
        for (int c = 0; c < NC; ++c) acc0[c] = acc1[c] = 0.0;
        for (int64_t k0 = kbeg; k0 < kend; k0 += SD_KC) {
            __syncthreads();                                // previous chunk fully consumed
            for (int e = threadIdx.x * 2; e < NC * SD_KC; e += SD_WARPS * 64) {
                const int c = e / SD_KC, kk = e % SD_KC;
                double2 m = make_double2(0.0, 0.0);
                if (c < nc) {
                    const int64_t k = k0 + kk;
                    if (k + 1 < kend) m = *reinterpret_cast<const double2*>(M + (size_t)c * ldm + k);
                    else if (k < kend) m.x = M[(size_t)c * ldm + k];
                }
                *reinterpret_cast<double2*>(sm + e) = m;
            }
            __syncthreads();
#pragma unroll 4
            for (int kk = lane * 2; kk < SD_KC; kk += 64) {
                const int64_t k = k0 + kk;
                if (k >= kend) break;
                double2 a0 = make_double2(0.0, 0.0), a1 = make_double2(0.0, 0.0);
                if (k + 1 < kend) {
                    if (v0) a0 = *reinterpret_cast<const double2*>(s0 + k);
                    if (v1) a1 = *reinterpret_cast<const double2*>(s1 + k);
                } else {
                    if (v0) a0.x = s0[k];
                    if (v1) a1.x = s1[k];
                }
#pragma unroll
                for (int c = 0; c < NC; ++c) {
                    const double2 m = *reinterpret_cast<const double2*>(sm + c * SD_KC + kk);
                    acc0[c] = fma(a0.x, m.x, fma(a0.y, m.y, acc0[c]));
                    acc1[c] = fma(a1.x, m.x, fma(a1.y, m.y, acc1[c]));
                }
            }
        }
#pragma unroll
        for (int c = 0; c < NC; ++c) {
            const double t0 = warp_sum(acc0[c]), t1 = warp_sum(acc1[c]);
            if (lane == 0 && c < nc) {
                if (v0) partial[((size_t)sp * nrows + r0) * nc + c] = t0;
                if (v1) partial[((size_t)sp * nrows + r0 + 1) * nc + c] = t1;
            }
        }
    }
}
__global__ void stack_dots_reduce(const double* __restrict__ partial, int nrows, int nc, int nspans, double* __restrict__ E, int ldE) {
    const int idx = blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= nrows * nc) return;
    double s = 0.0;
    for (int sp = 0; sp < nspans; ++sp) s += partial[(size_t)sp * nrows * nc + idx];
    E[(size_t)(idx / nc) * ldE + idx % nc] = s;
}

int grid_for(int64_t n, int threads) {
    int64_t b = (n + threads - 1) / threads;
    if (b < 1) b = 1;
    if (b > RED_BLOCKS * 4) b = RED_BLOCKS * 4;
    return (int)b;
}

}  // namespace

int64_t multi_dot_scratch() { return (int64_t)64 * RED_BLOCKS; }
void launch_multi_dot(const double* x, const double* Y, int64_t ldy, int m, int64_t n, double* out, double* g_partial,
                      cudaStream_t st) {
    if (m <= 0) return;
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
int64_t stack_dots_scratch(int nrows, int nc, int64_t K, int64_t* span_out, int* nspans_out) {
    // K spans: enough work items (row blocks x spans) for ~8 per resident CTA, at least one chunk each
    const int nrb = (nrows + 2 * SD_WARPS - 1) / (2 * SD_WARPS);
    const int64_t nch = K > 0 ? (K + SD_KC - 1) / SD_KC : 1;   // K == 0: one empty span (E = 0)
    int64_t want = (148 * 2 * 8 + nrb - 1) / nrb;
    if (want < 1) want = 1;
    if (want > nch) want = nch;
    int64_t per = (nch + want - 1) / want;                  // chunks per span
    const int64_t span = per * SD_KC;
    const int nspans = K > 0 ? (int)((K + span - 1) / span) : 1;
    if (span_out) *span_out = span;
    if (nspans_out) *nspans_out = nspans;
    return (int64_t)nspans * nrows * nc;
}
void launch_stack_dots(const double* S, int64_t lds, int nrows, const double* M, int64_t ldm, int nc, int64_t K, double* E,
                       int ldE, double* scratch, cudaStream_t st) {
    if (nrows <= 0 || nc <= 0 || nc > 8) return;
    int64_t span = 0;
    int nspans = 0;
    stack_dots_scratch(nrows, nc, K, &span, &nspans);
    const int nrb = (nrows + 2 * SD_WARPS - 1) / (2 * SD_WARPS);
    const int64_t items = (int64_t)nrb * nspans;
    const int grid = (int)(items < 148 * 2 * 4 ? items : 148 * 2 * 4);
    const int NCt = nc <= 1 ? 1 : (nc <= 2 ? 2 : (nc <= 4 ? 4 : 8));
    const int smem = NCt * SD_KC * (int)sizeof(double);
    // the attribute is per device: set it on every launch (a cheap host-side call) instead of caching a process-wide flag
    if (NCt == 8) cudaFuncSetAttribute(stack_dots_kernel<8>, cudaFuncAttributeMaxDynamicSharedMemorySize, 8 * SD_KC * 8);
    if (K <= 0) { cudaMemsetAsync(scratch, 0, sizeof(double) * (size_t)nspans * nrows * nc, st); }
    else if (NCt == 1) stack_dots_kernel<1><<<grid, SD_WARPS * 32, smem, st>>>(S, lds, nrows, M, ldm, nc, K, span, nspans, scratch);
    else if (NCt == 2) stack_dots_kernel<2><<<grid, SD_WARPS * 32, smem, st>>>(S, lds, nrows, M, ldm, nc, K, span, nspans, scratch);
    else if (NCt == 4) stack_dots_kernel<4><<<grid, SD_WARPS * 32, smem, st>>>(S, lds, nrows, M, ldm, nc, K, span, nspans, scratch);
    else stack_dots_kernel<8><<<grid, SD_WARPS * 32, smem, st>>>(S, lds, nrows, M, ldm, nc, K, span, nspans, scratch);
    stack_dots_reduce<<<(nrows * nc + 255) / 256, 256, 0, st>>>(scratch, nrows, nc, nspans, E, ldE);
}

}  // namespace dmrg
