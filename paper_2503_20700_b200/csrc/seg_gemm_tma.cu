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

#include <atomic>

#include <cstdint>

namespace dmrg {

namespace {

#ifndef TMA_BK
#define TMA_BK 16
#endif
#ifndef TMA_ST
#define TMA_ST 3
#endif
#ifndef TMA_CPS
#define TMA_CPS 3
#endif
constexpr int BM = GEMM_BM, BK = TMA_BK;      // CTA tile 64 x 64, K step of one pipeline stage
constexpr int NCONS = 4;                       // consumer warps
constexpr int NT2 = (NCONS + 1) * 32;          // + one producer warp
constexpr int ST2 = TMA_ST;                    // pipeline stages (BK 16: 20 KB each, 60 KB per CTA, three CTAs per SM)
constexpr int CPS = TMA_CPS;                   // resident CTAs per SM the register budget is cut for
constexpr int LDK = BK + 4;                    // row stride of the [m][k] / [n][k] layouts (160 B)
constexpr int LDM = BM + 4;                    // row stride of the [k][m] / [k][n] layouts (544 B)
constexpr int PANEL = (BM * LDK > BK * LDM) ? BM * LDK : BK * LDM;
constexpr int LCPR = BK / 2;                   // LDGSTS: 16-byte chunks per [m][k] panel row = lanes per row
constexpr int LRS = 32 / LCPR;                 // LDGSTS: panel rows covered by one warp instruction
constexpr int STAGE_DOUBLES = 2 * PANEL;

enum : int { F_TA = 1, F_TB = 2, F_FIRST = 4, F_LAST = 8, F_COMPUTE = 16, F_STOP = 32, F_RESCALE = 64 };

struct StageInfo {                             // written by the producer, read by the consumers
    double alpha;                              // alpha of the stage's segment: the accumulators are kept in units of it
    double ratio;                              // F_RESCALE: previous alpha / alpha, applied to the accumulators first
    int flags, kv;
    int tslot, pad;                            // slot of the tile in the tile ring, valid when F_FIRST is set
};
// Tile parameters live in a shared ring instead of consumer registers.  A tile occupies at least one stage and the
// producer runs at most ST2 stages ahead of the slowest consumer, so ST2 + 1 slots can never be overwritten early.
struct TileInfo {
    double* C;
    const Seg* ident;                          // identity-B segments of the task
    int ldc, mv, nv, m0, n0, tflags, nident, pad;   // output tile [m0, m0+mv) x [n0, n0+nv)
};
constexpr int NTR = ST2 + 1;

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


// One pipeline stage for a warp that owns NI x NJ fragments: fully unrolled, no predicated DMMA.  Every ragged tile
// shape gets its own straight-line DMMA sequence, so skipping fragments costs nothing in the instruction stream.
// FULL: all BK columns valid.  Otherwise the k-steps at or beyond kv are skipped (warp-uniform branch around whole
// steps) and the last partial step is masked in registers.
template <int NI, int NJ, bool FULL>
__device__ __forceinline__ void mma_stage(double (&acc)[4][4][2], const double* __restrict__ As,
                                          const double* __restrict__ Bs, int a_off, int a_ks, int a_ms, int b_off,
                                          int b_ks, int b_ns, int kv, int fc) {
#pragma unroll
    for (int kk = 0; kk < BK; kk += 4) {
        if (!FULL && kk >= kv) break;
        double a[NI], b[NJ];
#pragma unroll
        for (int i = 0; i < NI; ++i) a[i] = As[a_off + kk * a_ks + 8 * i * a_ms];
#pragma unroll
        for (int j = 0; j < NJ; ++j) b[j] = Bs[b_off + kk * b_ks + 8 * j * b_ns];
        if (!FULL && kk + fc >= kv) {
#pragma unroll
            for (int i = 0; i < NI; ++i) a[i] = 0.0;
#pragma unroll
            for (int j = 0; j < NJ; ++j) b[j] = 0.0;
        }
#pragma unroll
        for (int i = 0; i < NI; ++i)
#pragma unroll
            for (int j = 0; j < NJ; ++j) dmma(acc[i][j][0], acc[i][j][1], a[i], b[j]);
    }
}
template <int NI, bool FULL>
__device__ __forceinline__ void mma_stage_nj(int nj, double (&acc)[4][4][2], const double* As, const double* Bs,
                                             int a_off, int a_ks, int a_ms, int b_off, int b_ks, int b_ns, int kv, int fc) {
    switch (nj) {
        case 4: mma_stage<NI, 4, FULL>(acc, As, Bs, a_off, a_ks, a_ms, b_off, b_ks, b_ns, kv, fc); break;
        case 3: mma_stage<NI, 3, FULL>(acc, As, Bs, a_off, a_ks, a_ms, b_off, b_ks, b_ns, kv, fc); break;
        case 2: mma_stage<NI, 2, FULL>(acc, As, Bs, a_off, a_ks, a_ms, b_off, b_ks, b_ns, kv, fc); break;
        default: mma_stage<NI, 1, FULL>(acc, As, Bs, a_off, a_ks, a_ms, b_off, b_ks, b_ns, kv, fc); break;
    }
}
template <bool FULL>
__device__ __forceinline__ void mma_stage_ni(int ni, int nj, double (&acc)[4][4][2], const double* As,
                                             const double* Bs, int a_off, int a_ks, int a_ms, int b_off, int b_ks,
                                             int b_ns, int kv, int fc) {
    switch (ni) {
        case 4: mma_stage_nj<4, FULL>(nj, acc, As, Bs, a_off, a_ks, a_ms, b_off, b_ks, b_ns, kv, fc); break;
        case 3: mma_stage_nj<3, FULL>(nj, acc, As, Bs, a_off, a_ks, a_ms, b_off, b_ks, b_ns, kv, fc); break;
        case 2: mma_stage_nj<2, FULL>(nj, acc, As, Bs, a_off, a_ks, a_ms, b_off, b_ks, b_ns, kv, fc); break;
        default: mma_stage_nj<1, FULL>(nj, acc, As, Bs, a_off, a_ks, a_ms, b_off, b_ks, b_ns, kv, fc); break;
    }
}

__global__ void __launch_bounds__(NT2, CPS)
seg_gemm_tma_kernel(const Task* __restrict__ tasks, const Seg* __restrict__ segs, const Tile* __restrict__ tiles,
                    int ntiles, int* __restrict__ counter) {
    extern __shared__ __align__(128) double smem[];
    __shared__ __align__(8) uint64_t full_bar[ST2], empty_bar[ST2];
    __shared__ StageInfo info[ST2];
    __shared__ TileInfo tring[NTR];

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    if (tid == 0) {
        for (int s = 0; s < ST2; ++s) { mbar_init(&full_bar[s], 33); mbar_init(&empty_bar[s], NCONS); }   // full: 32 LDGSTS hooks + 1 expect_tx
        asm volatile("fence.mbarrier_init.release.cluster;\n" ::: "memory");
    }
    __syncthreads();

    if (warp == NCONS) {
        // ===================================== producer warp ==========================================================
        // Descriptor pipeline: the dependent chain  tile counter -> Tile -> Task -> first Seg  is spread over four
        // tiles (each load is issued one tile before its result is needed), and inside a tile the next Seg is loaded
        // while the current one is being streamed, so the producer never waits on descriptor latency in steady state.
        int pstage = 0;
        uint32_t pphase = 0;                                  // ring position and the parity of its round
        int tslot = 0;
        auto take = [&]() { int v = 0; if (lane == 0) v = atomicAdd(counter, 1); return v; };   // valid on lane 0
        Tile tl_d, tl_c, tl_b;
        Task tk_d, tk_c;
        Seg sg_d;
        int id_d, id_c, id_b, id_a;
        id_d = __shfl_sync(0xffffffffu, take(), 0);
        id_c = __shfl_sync(0xffffffffu, take(), 0);
        id_b = __shfl_sync(0xffffffffu, take(), 0);
        id_a = take();
        if (id_d < ntiles) { tl_d = tiles[id_d]; tk_d = tasks[tl_d.task]; if (tk_d.ngemm > 0) sg_d = segs[tk_d.seg_begin]; }
        if (id_c < ntiles) { tl_c = tiles[id_c]; tk_c = tasks[tl_c.task]; }
        if (id_b < ntiles) tl_b = tiles[id_b];
        for (;; tslot = (tslot + 1 == NTR) ? 0 : tslot + 1) {
            const bool stop = id_d >= ntiles;
            const Tile tl = tl_d;
            const Task tk = tk_d;
            Seg cur = sg_d, nxt;
            // advance the pipeline (every use below is of a load issued one tile ago)
            id_d = id_c; tl_d = tl_c; tk_d = tk_c;
            if (id_d < ntiles && tk_d.ngemm > 0) sg_d = segs[tk_d.seg_begin];
            id_c = id_b; tl_c = tl_b;
            if (id_c < ntiles) tk_c = tasks[tl_c.task];
            id_b = __shfl_sync(0xffffffffu, id_a, 0);
            if (id_b < ntiles) tl_b = tiles[id_b];
            if (!stop) id_a = take();
            const Seg* sg = nullptr;
            int m0 = 0, n0 = 0, mv = 0, nv = 0, lastseg = -1;
            if (!stop) {
                sg = segs + tk.seg_begin;
                m0 = tl.m0; n0 = tl.n0; mv = tl.mv; nv = tl.nv;
                lastseg = tk.ngemm - 1;                       // the host drops empty (K <= 0) GEMM segments
            }
            bool first = true;
            int s = 0, lk = 0;
            if (lastseg >= 1) nxt = sg[1];
            double ratio = 1.0;                               // != 1 on the first stage of a segment whose alpha differs
            bool rescale = false;
            // per-segment, per-lane copy state: source pointers of this lane's piece of the A / B panel of the next
            // stage and their per-stage advance, so that a stage costs pointer increments instead of index arithmetic
            const int c2 = (lane % LCPR) * 2, r0 = lane / LCPR;   // LDGSTS: this lane's 16-byte column chunk and first row
            const double* pa = nullptr;
            const double* pb = nullptr;
            size_t adv_a = 0, adv_b = 0, row_a = 0, row_b = 0;
            const uint32_t bytesA = (uint32_t)pad2d(mv) * 8u, bytesB = (uint32_t)pad2d(nv) * 8u;   // bulk row pieces
            auto seg_setup = [&]() {
                const size_t lda = (size_t)(uint32_t)cur.lda, ldb = (size_t)(uint32_t)cur.ldb;
                if (cur.flags & SEG_TRANS_A) { pa = cur.A + (uint32_t)m0 + (uint32_t)lane * lda; adv_a = BK * lda; }
                else { pa = cur.A + (uint32_t)(m0 + r0) * lda + (uint32_t)c2; adv_a = BK; row_a = LRS * lda; }
                if (cur.flags & SEG_TRANS_B) { pb = cur.B + (uint32_t)(n0 + r0) * ldb + (uint32_t)c2; adv_b = BK; row_b = LRS * ldb; }
                else { pb = cur.B + (uint32_t)n0 + (uint32_t)lane * ldb; adv_b = BK * ldb; }
            };
            if (!stop && lastseg >= 0) seg_setup();
            do {                                              // one pipeline stage per iteration
                mbar_wait(&empty_bar[pstage], pphase ^ 1);
                double* As = smem + pstage * STAGE_DOUBLES;
                double* Bs = As + PANEL;
                const bool compute = !stop && s <= lastseg;
                int kv = 0;
                uint32_t tx = 0;
                bool last = true;
                if (compute) {
                    kv = min(BK, cur.K - lk);
                    if (cur.flags & SEG_TRANS_A) tx += (uint32_t)kv * bytesA;      // bulk rows [k][m]
                    if (!(cur.flags & SEG_TRANS_B)) tx += (uint32_t)kv * bytesB;   // bulk rows [k][n]
                    last = (s == lastseg) && (lk + BK >= cur.K);
                }
                if (lane == 0) {
                    StageInfo& in = info[pstage];
                    in.alpha = compute ? cur.alpha : 0.0;
                    in.ratio = ratio;
                    in.kv = kv;
                    in.flags = stop ? F_STOP
                                    : ((compute ? (F_COMPUTE | (cur.flags & 3)) : 0) | (first ? F_FIRST : 0) | (last ? F_LAST : 0) |
                                       (rescale ? F_RESCALE : 0));
                    if (first && !stop) {
                        TileInfo& ti = tring[tslot];
                        ti.C = tk.C; ti.ident = sg + tk.ngemm; ti.nident = tk.seg_count - tk.ngemm;
                        ti.ldc = tk.ldc; ti.mv = mv; ti.nv = nv; ti.m0 = m0; ti.n0 = n0; ti.tflags = tk.flags;
                        in.tslot = tslot;
                    }
                    mbar_arrive_expect_tx(&full_bar[pstage], tx);
                }
                __syncwarp();
                if (compute) {
                    if (cur.flags & SEG_TRANS_A) {
                        if (lane < kv) bulk_g2s(As + lane * LDM, pa, bytesA, &full_bar[pstage]);   // BK <= 32: one row per lane
                    } else if (c2 < kv) {
                        const double* src = pa;
                        double* dst = As + r0 * LDK + c2;
#pragma unroll 4
                        for (int r = r0; r < mv; r += LRS) { ldgsts16(dst, src); dst += LRS * LDK; src += row_a; }
                    }
                    if (cur.flags & SEG_TRANS_B) {
                        if (c2 < kv) {
                            const double* src = pb;
                            double* dst = Bs + r0 * LDK + c2;
#pragma unroll 4
                            for (int r = r0; r < nv; r += LRS) { ldgsts16(dst, src); dst += LRS * LDK; src += row_b; }
                        }
                    } else {
                        if (lane < kv) bulk_g2s(Bs + lane * LDM, pb, bytesB, &full_bar[pstage]);
                    }
                    pa += adv_a; pb += adv_b;
                    lk += BK;
                    if (lk >= cur.K) {                                // next segment: already in registers
                        lk = 0;
                        ++s;
                        rescale = (s <= lastseg) && (nxt.alpha != cur.alpha);
                        if (rescale) ratio = cur.alpha / nxt.alpha;   // segments with alpha == 0 are dropped by the host
                        cur = nxt;
                        if (s <= lastseg) seg_setup();
                        if (s + 1 <= lastseg) nxt = sg[s + 1];
                    } else {
                        rescale = false;
                    }
                }
                ldgsts_arrive_noinc(&full_bar[pstage]);               // fires when this lane's LDGSTS of the stage have landed
                first = false;
                if (++pstage == ST2) { pstage = 0; pphase ^= 1; }
            } while (!stop && s <= lastseg);
            if (stop) break;
        }
        return;
    }

    // ========================================= consumer warps ==========================================================
    // The tile's ceil(mv/8) x ceil(nv/8) DMMA fragments are split evenly over the 2 x 2 warps (each at most 4 x 4);
    // fragments outside the tile are never issued, so ragged sector dimensions waste at most 7 rows / columns.
    const int fr = lane >> 2, fc = lane & 3;              // fragment row (0..7) and k / column-pair index (0..3)
    double acc[4][4][2];
    int cslot = 0;                                        // tile ring slot of the current tile
    int wm = 0, wn = 0, ni = 0, nj = 0;                   // this warp's fragment origin and counts within the tile
    uint32_t cstep = 0, rot = blockIdx.x;
    for (;; ++cstep) {
        const int stage = cstep % ST2;
        mbar_wait(&full_bar[stage], (cstep / ST2) & 1);
        const StageInfo& in = info[stage];
        const int fl = in.flags;
        if (fl & F_STOP) break;
        if (fl & F_FIRST) {
            cslot = in.tslot;
            const int tmv = tring[cslot].mv, tnv = tring[cslot].nv;
            const int fm = (tmv + 7) >> 3, fn = (tnv + 7) >> 3, hm = (fm + 1) >> 1, hn = (fn + 1) >> 1;
            // the quadrant a warp takes rotates from tile to tile: the heavier quadrants of ragged tiles visit every
            // warp (and with it every SM sub-partition's DMMA pipe) equally often
            const int role = (warp + (int)(rot++)) & 3;
            wm = (role >> 1) ? hm * 8 : 0; ni = (role >> 1) ? fm - hm : hm;
            wn = (role & 1) ? hn * 8 : 0;  nj = (role & 1) ? fn - hn : hn;
#pragma unroll
            for (int i = 0; i < 4; ++i)
#pragma unroll
                for (int j = 0; j < 4; ++j) acc[i][j][0] = acc[i][j][1] = 0.0;
        }
        const double al = in.alpha;                         // read before the stage is released
        if (fl & F_RESCALE) {                                // a new alpha: acc holds sum / alpha_prev -> sum / alpha
            const double r = in.ratio;
#pragma unroll
            for (int i = 0; i < 4; ++i)
#pragma unroll
                for (int j = 0; j < 4; ++j) { acc[i][j][0] *= r; acc[i][j][1] *= r; }
        }
        if (fl & F_COMPUTE) {
            const int kv = in.kv;
            const double* As = smem + stage * STAGE_DOUBLES;
            const double* Bs = As + PANEL;
            const int a_off = (fl & F_TA) ? (fc * LDM + wm + fr) : ((wm + fr) * LDK + fc);
            const int a_ks = (fl & F_TA) ? LDM : 1;          // stride per unit k
            const int a_ms = (fl & F_TA) ? 1 : LDK;          // stride per unit m
            const int b_off = (fl & F_TB) ? ((wn + fr) * LDK + fc) : (fc * LDM + wn + fr);
            const int b_ks = (fl & F_TB) ? 1 : LDM;
            const int b_ns = (fl & F_TB) ? LDK : 1;
            if (ni == 0 || nj == 0) {
                // nothing to do for this warp in this tile
            } else if (kv == BK) {
                mma_stage_ni<true>(ni, nj, acc, As, Bs, a_off, a_ks, a_ms, b_off, b_ks, b_ns, kv, fc);
            } else {                                         // ragged K tail of a segment
                mma_stage_ni<false>(ni, nj, acc, As, Bs, a_off, a_ks, a_ms, b_off, b_ks, b_ns, kv, fc);
            }
        }
        __syncwarp();
        if (lane == 0) mbar_arrive(&empty_bar[stage]);       // this warp is done with the stage (data and info)
        if (fl & F_LAST) {
            // ---- epilogue: identity-B segments, optional accumulate, store ------------------------------------------
            const TileInfo& ti = tring[cslot];
            double* const tC = ti.C;
            const Seg* const tident = ti.ident;
            const int tldc = ti.ldc, tnident = ti.nident, tm0 = ti.m0, tn0 = ti.n0, tmv = ti.mv, tnv = ti.nv;
            const bool accum = ti.tflags & TASK_ACCUM;
            const bool al_c = ((((uintptr_t)tC) & 15) == 0) && ((tldc & 1) == 0);
#pragma unroll
            for (int i = 0; i < 4; ++i) {
                const int row = tm0 + wm + 8 * i + fr;
                if (i >= ni || row >= tm0 + tmv) continue;
#pragma unroll
                for (int j = 0; j < 4; ++j) {
                    const int col = tn0 + wn + 8 * j + 2 * fc;
                    if (j >= nj || col >= tn0 + tnv) continue;
                    double v0 = al * acc[i][j][0], v1 = al * acc[i][j][1];
                    const bool two = (col + 1 < tn0 + tnv);
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
    // launch configuration cached per device (several contexts on several devices may live in one process)
    constexpr int MAX_DEV = 64;
    static std::atomic<int> grid_caps[MAX_DEV];
    const int smem_bytes = ST2 * STAGE_DOUBLES * (int)sizeof(double);
    int dev = 0;
    cudaGetDevice(&dev);
    int grid_cap = (dev >= 0 && dev < MAX_DEV) ? grid_caps[dev].load(std::memory_order_acquire) : 0;
    if (grid_cap == 0) {
        cudaFuncSetAttribute(seg_gemm_tma_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_bytes);
        int sms = 148, per_sm = 3;
        cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
        cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, seg_gemm_tma_kernel, NT2, smem_bytes);
        if (per_sm < 1) per_sm = 1;
        grid_cap = sms * per_sm;                            // persistent: one CTA per resident slot
        if (dev >= 0 && dev < MAX_DEV) grid_caps[dev].store(grid_cap, std::memory_order_release);
    }
    cudaMemsetAsync(d_counter, 0, sizeof(int), stream);
    const int grid = ntiles < grid_cap ? ntiles : grid_cap;
    seg_gemm_tma_kernel<<<grid, NT2, smem_bytes, stream>>>(d_tasks, d_segs, d_tiles, ntiles, d_counter);
}

}  // namespace dmrg
