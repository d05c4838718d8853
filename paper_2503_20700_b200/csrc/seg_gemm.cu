// Grouped, K-segmented FP64 GEMM for sm_100a: see kernels.hpp.
//
// Pipeline: cp.async (LDGSTS, 16-byte, zero-filling ragged edges) -> 4-stage shared-memory ring -> register
// fragments -> DMMA.8x8x4 (mma.sync.aligned.m8n8k4.f64).  sm_100a has no FP64 kind in tcgen05/UMMA, so the warp-
// level DMMA is the only FP64 tensor path (hard part 2).  CTA tile 64x64, BK = 16, 4 warps
// (2x2), warp tile 32x32 = 4x4 DMMA tiles; shared strides 20 / 68 doubles (== 4 mod 16) make every fragment load
// conflict-free for both operand orientations, so transposed operands cost nothing extra.
#include "kernels.hpp"

#include <cuda_runtime.h>

namespace dmrg {

namespace {

constexpr int BM = GEMM_BM, BN = GEMM_BN, BK = GEMM_BK, NT = GEMM_THREADS, ST = GEMM_STAGES;
constexpr int LDK = BK + 4;        // stride of the [m][k] / [n][k] layouts (20)
constexpr int LDM = BM + 4;        // stride of the [k][m] / [k][n] layouts (68)
constexpr int PANEL = BM * LDK;    // 1280 doubles >= BK * LDM = 1088
constexpr int STAGE_DOUBLES = 2 * PANEL;

struct StageInfo {
    double alpha;
    int flags;   // SEG_TRANS_A | SEG_TRANS_B, bit 30 = valid
    int pad;
};

__device__ __forceinline__ void cp_async16(double* smem_dst, const double* gsrc, int bytes) {
    unsigned s = (unsigned)__cvta_generic_to_shared(smem_dst);
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;\n" ::"r"(s), "l"(gsrc), "r"(bytes) : "memory");
}
__device__ __forceinline__ void cp_async8(double* smem_dst, const double* gsrc, int bytes) {
    unsigned s = (unsigned)__cvta_generic_to_shared(smem_dst);
    asm volatile("cp.async.ca.shared.global [%0], [%1], 8, %2;\n" ::"r"(s), "l"(gsrc), "r"(bytes) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;\n" ::: "memory"); }
template <int N>
__device__ __forceinline__ void cp_async_wait() {
    asm volatile("cp.async.wait_group %0;\n" ::"n"(N) : "memory");
}

__device__ __forceinline__ void dmma(double& d0, double& d1, double a, double b) {
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n"
                 : "+d"(d0), "+d"(d1)
                 : "d"(a), "d"(b));
}

// Copy a ROWS x COLS panel of a row-major global matrix (row stride ld, `rv` valid rows, `cv` valid columns,
// everything else zero-filled) into shared memory with row stride STRIDE.
template <int ROWS, int COLS, int STRIDE>
__device__ __forceinline__ void load_panel(double* dst, const double* src, int ld, int rv, int cv, bool aligned,
                                           int tid) {
    if (aligned) {
        constexpr int CPR = COLS / 2;                 // 16-byte chunks per row
        constexpr int TOTAL = ROWS * CPR;
#pragma unroll
        for (int q0 = 0; q0 < TOTAL; q0 += NT) {
            int q = q0 + tid;
            int r = q / CPR, c = (q % CPR) * 2;
            int bytes = 0;
            if (r < rv) {
                int left = cv - c;
                bytes = left >= 2 ? 16 : (left == 1 ? 8 : 0);
            }
            const double* g = bytes ? src + (size_t)r * ld + c : src;
            cp_async16(dst + r * STRIDE + c, g, bytes);
        }
    } else {
        constexpr int TOTAL = ROWS * COLS;
#pragma unroll
        for (int q0 = 0; q0 < TOTAL; q0 += NT) {
            int q = q0 + tid;
            int r = q / COLS, c = q % COLS;
            int bytes = (r < rv && c < cv) ? 8 : 0;
            const double* g = bytes ? src + (size_t)r * ld + c : src;
            cp_async8(dst + r * STRIDE + c, g, bytes);
        }
    }
}

__global__ void __launch_bounds__(NT) seg_gemm_kernel(const Task* __restrict__ tasks, const Seg* __restrict__ segs,
                                                      const Tile* __restrict__ tiles, int ntiles) {
    extern __shared__ __align__(16) double smem[];
    __shared__ StageInfo info[ST];

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int wm = (warp >> 1) * 32, wn = (warp & 1) * 32;
    const int fr = lane >> 2, fc = lane & 3;          // fragment row (0..7) and k / column-pair index (0..3)

    for (int tile_id = blockIdx.x; tile_id < ntiles; tile_id += gridDim.x) {
        const Tile tl = tiles[tile_id];
        const Task tk = tasks[tl.task];
        const Seg* sg = segs + tk.seg_begin;
        const int nseg = tk.seg_count;
        const int m0 = tl.m0, n0 = tl.n0, mv = tl.mv, nv = tl.nv;

        double acc[4][4][2], tmp[4][4][2];
#pragma unroll
        for (int i = 0; i < 4; ++i)
#pragma unroll
            for (int j = 0; j < 4; ++j) acc[i][j][0] = acc[i][j][1] = tmp[i][j][0] = tmp[i][j][1] = 0.0;

        // ---- loader cursor --------------------------------------------------------------------------------
        int ls = 0, lk = 0;
        while (ls < nseg && (sg[ls].flags & SEG_IDENT_B)) ++ls;
        Seg cur;
        if (ls < nseg) cur = sg[ls];

        auto issue = [&](int stage) {
            if (ls < nseg) {
                double* As = smem + stage * STAGE_DOUBLES;
                double* Bs = As + PANEL;
                const int kv = min(BK, cur.K - lk);
                const bool al_a = ((((uintptr_t)cur.A) & 15) == 0) && ((cur.lda & 1) == 0);
                const bool al_b = ((((uintptr_t)cur.B) & 15) == 0) && ((cur.ldb & 1) == 0);
                if (cur.flags & SEG_TRANS_A)
                    load_panel<BK, BM, LDM>(As, cur.A + (size_t)lk * cur.lda + m0, cur.lda, kv, mv, al_a, tid);
                else
                    load_panel<BM, BK, LDK>(As, cur.A + (size_t)m0 * cur.lda + lk, cur.lda, mv, kv, al_a, tid);
                if (cur.flags & SEG_TRANS_B)
                    load_panel<BN, BK, LDK>(Bs, cur.B + (size_t)n0 * cur.ldb + lk, cur.ldb, nv, kv, al_b, tid);
                else
                    load_panel<BK, BN, LDM>(Bs, cur.B + (size_t)lk * cur.ldb + n0, cur.ldb, kv, nv, al_b, tid);
                if (tid == 0) {
                    info[stage].alpha = cur.alpha;
                    info[stage].flags = (cur.flags & 3) | (1 << 30);
                }
                lk += BK;
                if (lk >= cur.K) {
                    lk = 0;
                    ++ls;
                    while (ls < nseg && (sg[ls].flags & SEG_IDENT_B)) ++ls;
                    if (ls < nseg) cur = sg[ls];
                }
            } else if (tid == 0) {
                info[stage].flags = 0;
            }
            cp_async_commit();
        };

        __syncthreads();   // previous tile's readers of smem / info are done
#pragma unroll
        for (int s = 0; s < ST - 1; ++s) issue(s);

        double alpha_cur = 0.0;
        bool have = false;
        for (int step = 0;; ++step) {
            cp_async_wait<ST - 2>();
            __syncthreads();
            issue((step + ST - 1) % ST);
            const int stage = step % ST;
            const int fl = info[stage].flags;
            if (!(fl & (1 << 30))) break;
            const double al = info[stage].alpha;
            if (have && al != alpha_cur) {
#pragma unroll
                for (int i = 0; i < 4; ++i)
#pragma unroll
                    for (int j = 0; j < 4; ++j) {
                        acc[i][j][0] += alpha_cur * tmp[i][j][0];
                        acc[i][j][1] += alpha_cur * tmp[i][j][1];
                        tmp[i][j][0] = tmp[i][j][1] = 0.0;
                    }
            }
            alpha_cur = al;
            have = true;
            const double* As = smem + stage * STAGE_DOUBLES;
            const double* Bs = As + PANEL;
            // per-thread fragment base offsets and k-strides for the two possible layouts of each operand
            const int a_off = (fl & SEG_TRANS_A) ? (fc * LDM + wm + fr) : ((wm + fr) * LDK + fc);
            const int a_ks = (fl & SEG_TRANS_A) ? LDM : 1;         // stride per unit k
            const int a_ms = (fl & SEG_TRANS_A) ? 1 : LDK;         // stride per unit m
            const int b_off = (fl & SEG_TRANS_B) ? ((wn + fr) * LDK + fc) : (fc * LDM + wn + fr);
            const int b_ks = (fl & SEG_TRANS_B) ? 1 : LDM;
            const int b_ns = (fl & SEG_TRANS_B) ? LDK : 1;
#pragma unroll
            for (int kk = 0; kk < BK; kk += 4) {
                double a[4], b[4];
#pragma unroll
                for (int i = 0; i < 4; ++i) a[i] = As[a_off + kk * a_ks + 8 * i * a_ms];
#pragma unroll
                for (int j = 0; j < 4; ++j) b[j] = Bs[b_off + kk * b_ks + 8 * j * b_ns];
#pragma unroll
                for (int i = 0; i < 4; ++i)
#pragma unroll
                    for (int j = 0; j < 4; ++j) dmma(tmp[i][j][0], tmp[i][j][1], a[i], b[j]);
            }
        }
        cp_async_wait<0>();
        if (have) {
#pragma unroll
            for (int i = 0; i < 4; ++i)
#pragma unroll
                for (int j = 0; j < 4; ++j) {
                    acc[i][j][0] += alpha_cur * tmp[i][j][0];
                    acc[i][j][1] += alpha_cur * tmp[i][j][1];
                }
        }

        // ---- epilogue: identity-B segments, optional accumulate, store -----------------------------------------
        const bool accum = tk.flags & TASK_ACCUM;
        const bool al_c = ((((uintptr_t)tk.C) & 15) == 0) && ((tk.ldc & 1) == 0);
#pragma unroll
        for (int i = 0; i < 4; ++i) {
            const int row = m0 + wm + 8 * i + fr;
            if (row >= m0 + mv) continue;
#pragma unroll
            for (int j = 0; j < 4; ++j) {
                const int col = n0 + wn + 8 * j + 2 * fc;
                if (col >= n0 + nv) continue;
                double v0 = acc[i][j][0], v1 = acc[i][j][1];
                const bool two = (col + 1 < n0 + nv);
                for (int s = 0; s < nseg; ++s) {
                    if (!(sg[s].flags & SEG_IDENT_B)) continue;
                    const double* ap = sg[s].A + (size_t)row * sg[s].lda + col;
                    v0 += sg[s].alpha * ap[0];
                    if (two) v1 += sg[s].alpha * ap[1];
                }
                double* cp = tk.C + (size_t)row * tk.ldc + col;
                if (two && al_c) {
                    double2 o;
                    if (accum) {
                        o = *reinterpret_cast<double2*>(cp);
                        o.x += v0;
                        o.y += v1;
                    } else {
                        o.x = v0;
                        o.y = v1;
                    }
                    *reinterpret_cast<double2*>(cp) = o;
                } else {
                    cp[0] = accum ? cp[0] + v0 : v0;
                    if (two) cp[1] = accum ? cp[1] + v1 : v1;
                }
            }
        }
    }
}

}  // namespace

void launch_seg_gemm(const Task* d_tasks, const Seg* d_segs, const Tile* d_tiles, int ntiles, cudaStream_t stream) {
    if (ntiles <= 0) return;
    const int smem_bytes = ST * STAGE_DOUBLES * (int)sizeof(double);
    cudaFuncSetAttribute(seg_gemm_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_bytes);   // per device: not cached (test / fallback kernel)
    seg_gemm_kernel<<<ntiles, NT, smem_bytes, stream>>>(d_tasks, d_segs, d_tiles, ntiles);
}

}  // namespace dmrg
