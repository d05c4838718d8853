// Grouped, K-segmented FP64 GEMM for sm_100a, bulk-copy (TMA engine) fed and warp specialised: see kernels.hpp.
//
//   producer warp : walks the tile list (dynamic tile counter), each tile's segment list and K steps; for every
//                   pipeline stage it arms an mbarrier with the expected byte count and issues one
//                   cp.async.bulk (SASS UBLKCP) per panel row, global -> shared, completing on that mbarrier.
//   4 consumer warps (2x2, warp tile 32x32 = 4x4 DMMA.8x8x4): wait on the stage's "full" mbarrier, load register
//                   fragments from shared memory, issue mma.sync.m8n8k4.f64, release the stage on its "empty"
//                   mbarrier; no CTA-wide barrier in the main loop.  The ring runs across tile boundaries, so the
//                   next tile's panels are in flight while the consumers write the current tile's epilogue.
// sm_100a's tcgen05 / UMMA has no FP64 kind, so the warp-level DMMA is the FP64 tensor path.
// Requirements (checked on the host, else the cp.async kernel of seg_gemm.cu is used): every operand 16-byte
// aligned with an even leading dimension, so that a row piece of pad2(n) doubles is a legal bulk copy.  Ragged M / N
// edges need no zero fill (garbage rows / columns only reach outputs that are never stored); the ragged K tail is
// masked in registers.
#include "kernels.hpp"

#include <cuda_runtime.h>

#include <cstdint>

namespace dmrg {

namespace {

constexpr int BM = GEMM_BM, BN = GEMM_BN, BK = GEMM_BK;
constexpr int NCONS = 4;                       // consumer warps
constexpr int NT2 = (NCONS + 1) * 32;          // + one producer warp
constexpr int ST2 = 3;                         // pipeline stages (60 KB per CTA: three CTAs per SM)
constexpr int LDK = BK + 4;                    // row stride of the [m][k] / [n][k] layouts (160 B)
constexpr int LDM = BM + 4;                    // row stride of the [k][m] / [k][n] layouts (544 B)
constexpr int PANEL = BM * LDK;                // 1280 doubles >= BK * LDM = 1088
constexpr int STAGE_DOUBLES = 2 * PANEL;

enum : int { F_TA = 1, F_TB = 2, F_FIRST = 4, F_LAST = 8, F_COMPUTE = 16, F_STOP = 32 };

struct StageInfo {                             // written by the producer, read by the consumers
    double alpha;
    int flags, kv;
    // tile fields, valid when F_FIRST is set
    double* C;
    const Seg* ident;                          // identity-B segments of the task
    int ldc, M, N, m0, n0, tflags, nident, pad;
};

__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint64_t* bar, int count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;\n" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_arrive(uint64_t* bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];\n" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void mbar_arrive_expect_tx(uint64_t* bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;\n" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) {
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "WAIT_LOOP:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra WAIT_DONE;\n"
        "bra WAIT_LOOP;\n"
        "WAIT_DONE:\n"
        "}\n" ::"r"(smem_u32(bar)), "r"(parity) : "memory");
}
// one row piece, global -> shared, completion counted in bytes on the mbarrier (TMA engine, no tensor map needed)
__device__ __forceinline__ void bulk_g2s(double* dst, const double* src, uint32_t bytes, uint64_t* bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];\n" ::"r"(smem_u32(dst)),
                 "l"(src), "r"(bytes), "r"(smem_u32(bar))
                 : "memory");
}
// 16-byte Ampere-style async copy (LDGSTS) and its completion hook on an mbarrier: used for the operand orientations
// whose panel rows are only 128 bytes long, where one bulk copy per row would be bound by the TMA request rate
__device__ __forceinline__ void ldgsts16(double* dst, const double* src) {
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;\n" ::"r"(smem_u32(dst)), "l"(src) : "memory");
}
__device__ __forceinline__ void ldgsts_arrive_noinc(uint64_t* bar) {
    asm volatile("cp.async.mbarrier.arrive.noinc.shared::cta.b64 [%0];\n" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void dmma(double& d0, double& d1, double a, double b) {
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n"
                 : "+d"(d0), "+d"(d1)
                 : "d"(a), "d"(b));
}
__device__ __forceinline__ int pad2d(int n) { return (n + 1) & ~1; }


__global__ void __launch_bounds__(NT2, 3)
seg_gemm_tma_kernel(const Task* __restrict__ tasks, const Seg* __restrict__ segs, const Tile* __restrict__ tiles,
                    int ntiles, int* __restrict__ counter) {
    extern __shared__ __align__(128) double smem[];
    __shared__ __align__(8) uint64_t full_bar[ST2], empty_bar[ST2];
    __shared__ StageInfo info[ST2];

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    if (tid == 0) {
        for (int s = 0; s < ST2; ++s) { mbar_init(&full_bar[s], 33); mbar_init(&empty_bar[s], NCONS); }   // full: 32 LDGSTS hooks + 1 expect_tx
        asm volatile("fence.mbarrier_init.release.cluster;\n" ::: "memory");
    }
    __syncthreads();

    if (warp == NCONS) {
        // ===================================== producer warp ==========================================================
        uint32_t pstep = 0;
        for (;;) {
            int tile_id = 0;
            if (lane == 0) tile_id = atomicAdd(counter, 1);
            tile_id = __shfl_sync(0xffffffffu, tile_id, 0);
            const bool stop = tile_id >= ntiles;
            Tile tl;
            Task tk;
            const Seg* sg = nullptr;
            int m0 = 0, n0 = 0, mv = 0, nv = 0, lastseg = -1;
            if (!stop) {
                tl = tiles[tile_id];
                tk = tasks[tl.task];
                sg = segs + tk.seg_begin;
                m0 = tl.tm * BM; n0 = tl.tn * BN;
                mv = min(BM, tk.M - m0); nv = min(BN, tk.N - n0);
                lastseg = tk.ngemm - 1;
                while (lastseg >= 0 && sg[lastseg].K <= 0) --lastseg;
            }
            bool first = true;
            int s = 0, lk = 0;
            while (!stop && s <= lastseg && sg[s].K <= 0) ++s;
            do {                                              // one pipeline stage per iteration
                const int stage = pstep % ST2;
                mbar_wait(&empty_bar[stage], ((pstep / ST2) & 1) ^ 1);
                double* As = smem + stage * STAGE_DOUBLES;
                double* Bs = As + PANEL;
                const bool compute = !stop && s <= lastseg;
                Seg cur;
                int kv = 0, rowsA = 0, rowsB = 0;
                uint32_t bytesA = 0, bytesB = 0;
                bool last = true;
                if (compute) {
                    cur = sg[s];
                    kv = min(BK, cur.K - lk);
                    if (cur.flags & SEG_TRANS_A) { rowsA = kv; bytesA = (uint32_t)pad2d(mv) * 8u; }    // bulk rows [k][m]
                    if (!(cur.flags & SEG_TRANS_B)) { rowsB = kv; bytesB = (uint32_t)pad2d(nv) * 8u; } // bulk rows [k][n]
                    last = (s == lastseg) && (lk + BK >= cur.K);
                }
                if (lane == 0) {
                    StageInfo& in = info[stage];
                    in.alpha = compute ? cur.alpha : 0.0;
                    in.kv = kv;
                    in.flags = stop ? F_STOP
                                    : ((compute ? (F_COMPUTE | (cur.flags & 3)) : 0) | (first ? F_FIRST : 0) | (last ? F_LAST : 0));
                    if (first && !stop) {
                        in.C = tk.C; in.ident = sg + tk.ngemm; in.nident = tk.seg_count - tk.ngemm;
                        in.ldc = tk.ldc; in.M = tk.M; in.N = tk.N; in.m0 = m0; in.n0 = n0; in.tflags = tk.flags;
                    }
                    mbar_arrive_expect_tx(&full_bar[stage], (uint32_t)rowsA * bytesA + (uint32_t)rowsB * bytesB);
                }
                __syncwarp();
                if (compute) {
                    const int c2 = (lane & 7) * 2, r0 = lane >> 3;        // LDGSTS: this lane's 16-byte column chunk and first row
                    if (cur.flags & SEG_TRANS_A) {
                        const double* src = cur.A + (size_t)lk * cur.lda + m0;
                        for (int r = lane; r < rowsA; r += 32) bulk_g2s(As + r * LDM, src + (size_t)r * cur.lda, bytesA, &full_bar[stage]);
                    } else if (c2 < kv) {
                        const double* src = cur.A + (size_t)(m0 + r0) * cur.lda + lk + c2;
                        double* dst = As + r0 * LDK + c2;
                        const size_t step = (size_t)4 * cur.lda;
#pragma unroll 4
                        for (int r = r0; r < mv; r += 4) { ldgsts16(dst, src); dst += 4 * LDK; src += step; }
                    }
                    if (cur.flags & SEG_TRANS_B) {
                        if (c2 < kv) {
                            const double* src = cur.B + (size_t)(n0 + r0) * cur.ldb + lk + c2;
                            double* dst = Bs + r0 * LDK + c2;
                            const size_t step = (size_t)4 * cur.ldb;
#pragma unroll 4
                            for (int r = r0; r < nv; r += 4) { ldgsts16(dst, src); dst += 4 * LDK; src += step; }
                        }
                    } else {
                        const double* src = cur.B + (size_t)lk * cur.ldb + n0;
                        for (int r = lane; r < rowsB; r += 32) bulk_g2s(Bs + r * LDM, src + (size_t)r * cur.ldb, bytesB, &full_bar[stage]);
                    }
                    lk += BK;
                    if (lk >= cur.K) {
                        lk = 0;
                        ++s;
                        while (s <= lastseg && sg[s].K <= 0) ++s;
                    }
                }
                ldgsts_arrive_noinc(&full_bar[stage]);                // fires when this lane's LDGSTS of the stage have landed
                first = false;
                ++pstep;
            } while (!stop && s <= lastseg);
            if (stop) break;
        }
        return;
    }

    // ========================================= consumer warps ==========================================================
    const int wm = (warp >> 1) * 32, wn = (warp & 1) * 32;
    const int fr = lane >> 2, fc = lane & 3;              // fragment row (0..7) and k / column-pair index (0..3)
    double acc[4][4][2];
    double* tC = nullptr;
    const Seg* tident = nullptr;
    int tldc = 0, tM = 0, tN = 0, tm0 = 0, tn0 = 0, tflags = 0, tnident = 0;
    uint32_t cstep = 0;
    for (;; ++cstep) {
        const int stage = cstep % ST2;
        mbar_wait(&full_bar[stage], (cstep / ST2) & 1);
        const StageInfo& in = info[stage];
        const int fl = in.flags;
        if (fl & F_STOP) break;
        if (fl & F_FIRST) {
            tC = in.C; tident = in.ident; tnident = in.nident;
            tldc = in.ldc; tM = in.M; tN = in.N; tm0 = in.m0; tn0 = in.n0; tflags = in.tflags;
#pragma unroll
            for (int i = 0; i < 4; ++i)
#pragma unroll
                for (int j = 0; j < 4; ++j) acc[i][j][0] = acc[i][j][1] = 0.0;
        }
        if (fl & F_COMPUTE) {
            const double al = in.alpha;
            const int kv = in.kv;
            const double* As = smem + stage * STAGE_DOUBLES;
            const double* Bs = As + PANEL;
            const int a_off = (fl & F_TA) ? (fc * LDM + wm + fr) : ((wm + fr) * LDK + fc);
            const int a_ks = (fl & F_TA) ? LDM : 1;          // stride per unit k
            const int a_ms = (fl & F_TA) ? 1 : LDK;          // stride per unit m
            const int b_off = (fl & F_TB) ? ((wn + fr) * LDK + fc) : (fc * LDM + wn + fr);
            const int b_ks = (fl & F_TB) ? 1 : LDM;
            const int b_ns = (fl & F_TB) ? LDK : 1;
            if (kv == BK) {
#pragma unroll
                for (int kk = 0; kk < BK; kk += 4) {
                    double a[4], b[4];
#pragma unroll
                    for (int i = 0; i < 4; ++i) a[i] = al * As[a_off + kk * a_ks + 8 * i * a_ms];
#pragma unroll
                    for (int j = 0; j < 4; ++j) b[j] = Bs[b_off + kk * b_ks + 8 * j * b_ns];
#pragma unroll
                    for (int i = 0; i < 4; ++i)
#pragma unroll
                        for (int j = 0; j < 4; ++j) dmma(acc[i][j][0], acc[i][j][1], a[i], b[j]);
                }
            } else {                                         // ragged K tail: mask both fragments in registers
                for (int kk = 0; kk < kv; kk += 4) {
                    const bool ok = kk + fc < kv;
                    double a[4], b[4];
#pragma unroll
                    for (int i = 0; i < 4; ++i) { const double v = As[a_off + kk * a_ks + 8 * i * a_ms]; a[i] = ok ? al * v : 0.0; }
#pragma unroll
                    for (int j = 0; j < 4; ++j) { const double v = Bs[b_off + kk * b_ks + 8 * j * b_ns]; b[j] = ok ? v : 0.0; }
#pragma unroll
                    for (int i = 0; i < 4; ++i)
#pragma unroll
                        for (int j = 0; j < 4; ++j) dmma(acc[i][j][0], acc[i][j][1], a[i], b[j]);
                }
            }
        }
        __syncwarp();
        if (lane == 0) mbar_arrive(&empty_bar[stage]);       // this warp is done with the stage (data and info)
        if (fl & F_LAST) {
            // ---- epilogue: identity-B segments, optional accumulate, store ------------------------------------------
            const bool accum = tflags & TASK_ACCUM;
            const bool al_c = ((((uintptr_t)tC) & 15) == 0) && ((tldc & 1) == 0);
#pragma unroll
            for (int i = 0; i < 4; ++i) {
                const int row = tm0 + wm + 8 * i + fr;
                if (row >= tM) continue;
#pragma unroll
                for (int j = 0; j < 4; ++j) {
                    const int col = tn0 + wn + 8 * j + 2 * fc;
                    if (col >= tN) continue;
                    double v0 = acc[i][j][0], v1 = acc[i][j][1];
                    const bool two = (col + 1 < tN);
                    for (int s = 0; s < tnident; ++s) {
                        const double* ap = tident[s].A + (size_t)row * tident[s].lda + col;
                        v0 += tident[s].alpha * ap[0];
                        if (two) v1 += tident[s].alpha * ap[1];
                    }
                    double* cp = tC + (size_t)row * tldc + col;
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
}

}  // namespace

void launch_seg_gemm_tma(const Task* d_tasks, const Seg* d_segs, const Tile* d_tiles, int ntiles, int* d_counter,
                         cudaStream_t stream) {
    if (ntiles <= 0) return;
    static bool configured = false;
    static int grid_cap = 148 * 3;
    const int smem_bytes = ST2 * STAGE_DOUBLES * (int)sizeof(double);
    if (!configured) {
        cudaFuncSetAttribute(seg_gemm_tma_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_bytes);
        int dev = 0, sms = 148, per_sm = 3;
        cudaGetDevice(&dev);
        cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
        cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, seg_gemm_tma_kernel, NT2, smem_bytes);
        if (per_sm < 1) per_sm = 1;
        grid_cap = sms * per_sm;                            // persistent: one CTA per resident slot
        configured = true;
    }
    cudaMemsetAsync(d_counter, 0, sizeof(int), stream);
    const int grid = ntiles < grid_cap ? ntiles : grid_cap;
    seg_gemm_tma_kernel<<<grid, NT2, smem_bytes, stream>>>(d_tasks, d_segs, d_tiles, ntiles, d_counter);
}

}  // namespace dmrg
