// Device-built block maps of H_eff psi.
//
// Input: small tables uploaded once per bond - the psi block list, the sector tables of the two bond bases, the
// quantum-number maps of every operator class (in-sector -> out-sector, storage offset), the operator references
// and the symbolic term list (a few thousand entries).  Everything that scales as terms x blocks - which (term,
// psi block, site state) triples contribute, their Jordan-Wigner signs, which intermediates T = O_L X / X O_R^T are
// needed and where they live, the K-concatenated segment list of every output block, the tile lists sorted by cost,
// the diagonal items and the flop / byte accounting - is enumerated here by CUDA kernels, with prefix sums fixing the
// order, so the result is deterministic.  No arithmetic on tensor data happens in this file (integer work).
#include <thrust/execution_policy.h>
#include <thrust/functional.h>
#include <thrust/scan.h>
#include <thrust/sort.h>

#include <cstdint>

#include "maps.hpp"

namespace dmrg {

namespace {

__device__ __forceinline__ int pad2i(int d) { return (d + 1) & ~1; }

struct View { int out; const double* ptr; int ld; int trans; int rows, cols; int stored; };

// block of operator `op` of one side acting on in-sector `in` (device twin of op_block in block.cpp)
__device__ __forceinline__ bool op_view(const MapSide& sd, const MapOp& op, int in, View& v) {
    const int* out = sd.out + (size_t)op.cls * sd.nsec;
    const int* inv = sd.inv + (size_t)op.cls * sd.nsec;
    const int64_t* off = sd.off + (size_t)op.cls * sd.nsec;
    if (!op.trans) {
        const int o = out[in];
        if (o < 0) return false;
        v.out = o; v.ptr = op.base + off[in]; v.ld = pad2i(sd.dim[in]); v.trans = 0;
        v.rows = sd.dim[o]; v.cols = sd.dim[in]; v.stored = in;
    } else {
        const int j = inv[in];
        if (j < 0) return false;
        v.out = j; v.ptr = op.base + off[j]; v.ld = pad2i(sd.dim[j]); v.trans = 1;
        v.rows = sd.dim[j]; v.cols = sd.dim[in]; v.stored = j;
    }
    return true;
}

enum : int { C_NONE = 0, C_LONLY = 1, C_RONLY = 2, C_LFIRST = 3, C_RFIRST = 4 };
struct Contrib { int bo, kase; double c; View vl, vr; };

// contribution of (term ti, input psi block bi) to the output block with site state abo (the host loop body)
__device__ bool contrib(const MapCtx& cx, int ti, int bi, int abo, Contrib& o) {
    const MapTerm& t = cx.terms[ti];
    const MapBlock& in = cx.blocks[bi];
    const double dmv = cx.dm[(size_t)t.dm * 256 + abo * 16 + in.ab];
    if (dmv == 0.0) return false;
    int lo = in.l, ro = in.r;
    if (t.opL >= 0) { if (!op_view(cx.L, cx.opsL[t.opL], in.l, o.vl)) return false; lo = o.vl.out; }
    if (t.opR >= 0) { if (!op_view(cx.R, cx.opsR[t.opR], in.r, o.vr)) return false; ro = o.vr.out; }
    const int bo = cx.lookup[lo * 16 + abo];
    if (bo < 0 || cx.blocks[bo].r != ro) return false;
    const int nl = cx.nL[in.l];
    const double sgn = ((t.pd * nl + t.pr * (nl + cx.dotqn[in.ab])) & 1) ? -1.0 : 1.0;
    o.bo = bo;
    o.c = t.coef * dmv * sgn;
    if (t.opL < 0 && t.opR < 0) o.kase = C_NONE;
    else if (t.opL < 0) o.kase = C_RONLY;
    else if (t.opR < 0) o.kase = C_LONLY;
    else {
        const MapBlock& ob = cx.blocks[bo];
        const double dl = in.rows, dr = in.cols, dlo = ob.rows, dro = ob.cols;
        const double cost_l = 2.0 * dlo * dl * dr + 2.0 * dlo * dr * dro;
        const double cost_r = 2.0 * dl * dr * dro + 2.0 * dlo * dl * dro;
        o.kase = cost_l <= cost_r ? C_LFIRST : C_RFIRST;
    }
    return true;
}

// input block of term ti that can reach output block bo through site state ab_in, or -1
__device__ __forceinline__ int source_block(const MapCtx& cx, int ti, int bo, int ab_in) {
    const MapTerm& t = cx.terms[ti];
    const MapBlock& ob = cx.blocks[bo];
    int l_in = ob.l;
    if (t.opL >= 0) {
        const MapOp& op = cx.opsL[t.opL];
        l_in = op.trans ? cx.L.out[(size_t)op.cls * cx.L.nsec + ob.l] : cx.L.inv[(size_t)op.cls * cx.L.nsec + ob.l];
        if (l_in < 0) return -1;
    }
    return cx.lookup[l_in * 16 + ab_in];
}

__device__ __forceinline__ int64_t tkey(const MapCtx& cx, int side, int op, int bi) {
    return ((int64_t)(side ? cx.nopsL + op : op)) * cx.nblk + bi;
}

// ---- pass 0: per-term usage of intermediates (dedupe within the term only), flops, diagonal counts, touched operators
__global__ void k_term_usage(MapCtx cx, double* usage /*[nterm]*/, double* stats /*f_alg, ngemm_p2, b_ops*/,
                             int* diag_cnt /*[nblk*nterm]*/, unsigned char* touched) {
    const int64_t idx = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= (int64_t)cx.nterm * cx.nblk) return;
    const int ti = (int)(idx / cx.nblk), bi = (int)(idx % cx.nblk);
    double use = 0.0, falg = 0.0, ng = 0.0;
    bool usedL = false, usedR = false;
    for (int abo = 0; abo < 16; ++abo) {
        Contrib c;
        if (!contrib(cx, ti, bi, abo, c)) continue;
        const MapBlock& in = cx.blocks[bi];
        const MapBlock& ob = cx.blocks[c.bo];
        const double dl = in.rows, dr = in.cols, dlo = ob.rows, dro = ob.cols;
        if (c.bo == bi) diag_cnt[(size_t)bi * cx.nterm + ti] = 1;       // at most one site state maps a block to itself
        if (c.kase != C_NONE && c.kase != C_RONLY) touched[((size_t)cx.opsL[cx.terms[ti].opL].ref) * cx.L.nsec + c.vl.stored] = 1;
        if (c.kase != C_NONE && c.kase != C_LONLY) touched[(size_t)cx.nrefL * cx.L.nsec + ((size_t)cx.opsR[cx.terms[ti].opR].ref) * cx.R.nsec + c.vr.stored] = 1;
        if (c.kase == C_RONLY) { falg += 2.0 * dl * dr * dro; ng += 1; }
        else if (c.kase == C_LONLY) { falg += 2.0 * dlo * dl * dr; ng += 1; }
        else if (c.kase == C_LFIRST) {
            falg += 2.0 * dlo * dl * dr + 2.0 * dlo * dr * dro; ng += 1;
            if (!usedL) { usedL = true; use += (double)ob.rows * pad2i(in.cols); }
        } else if (c.kase == C_RFIRST) {
            falg += 2.0 * dl * dr * dro + 2.0 * dlo * dl * dro; ng += 1;
            if (!usedR) { usedR = true; use += (double)in.rows * pad2i(ob.cols); }
        }
    }
    if (use != 0.0) atomicAdd(&usage[ti], use);
    if (falg != 0.0) { atomicAdd(&stats[0], falg); atomicAdd(&stats[1], ng); }
}

__global__ void k_touched_bytes(MapCtx cx, const unsigned char* touched, double* stats) {
    const int64_t idx = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    const int64_t nl = (int64_t)cx.nrefL * cx.L.nsec, nr = (int64_t)cx.nrefR * cx.R.nsec;
    if (idx >= nl + nr || !touched[idx]) return;
    const bool left = idx < nl;
    const MapSide& sd = left ? cx.L : cx.R;
    const int64_t j = left ? idx : idx - nl;
    const int ref = (int)(j / sd.nsec), in = (int)(j % sd.nsec);
    const int cls = left ? cx.refclsL[ref] : cx.refclsR[ref];
    const int o = sd.out[(size_t)cls * sd.nsec + in];
    if (o >= 0) atomicAdd(&stats[2], 8.0 * sd.dim[o] * sd.dim[in]);
}

__global__ void k_diag_emit(MapCtx cx, const int* diag_pos, DiagItemK* items) {
    const int64_t idx = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= (int64_t)cx.nterm * cx.nblk) return;
    const int bi = (int)(idx / cx.nterm), ti = (int)(idx % cx.nterm);
    if (diag_pos[idx + 1] == diag_pos[idx]) return;
    Contrib c;
    if (!contrib(cx, ti, bi, cx.blocks[bi].ab, c)) return;
    DiagItemK it;
    it.ml = (c.kase == C_NONE || c.kase == C_RONLY) ? nullptr : c.vl.ptr;
    it.ldl = it.ml ? c.vl.ld : 0;
    it.mr = (c.kase == C_NONE || c.kase == C_LONLY) ? nullptr : c.vr.ptr;
    it.ldr = it.mr ? c.vr.ld : 0;
    it.c = c.c;
    items[diag_pos[idx]] = it;
}
__global__ void k_diag_ptr(int nblk, int nterm, const int* diag_pos, int* diag_ptr) {
    const int b = blockIdx.x * blockDim.x + threadIdx.x;
    if (b <= nblk) diag_ptr[b] = diag_pos[(size_t)b * nterm];
}

// ---- per chunk: which intermediates are needed ------------------------------------------------------------------------
__global__ void k_mark(MapCtx cx, int t0, int t1, unsigned char* need) {
    const int64_t idx = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= (int64_t)(t1 - t0) * cx.nblk) return;
    const int ti = t0 + (int)(idx / cx.nblk), bi = (int)(idx % cx.nblk);
    const MapTerm& t = cx.terms[ti];
    if (t.opL < 0 || t.opR < 0) return;
    for (int abo = 0; abo < 16; ++abo) {
        Contrib c;
        if (!contrib(cx, ti, bi, abo, c)) continue;
        if (c.kase == C_LFIRST) need[tkey(cx, 0, t.opL, bi)] = 1;
        else if (c.kase == C_RFIRST) need[tkey(cx, 1, t.opR, bi)] = 1;
    }
}
__global__ void k_tsize(MapCtx cx, const unsigned char* need, int64_t* tsize, int* tflag) {
    const int64_t key = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    const int64_t nkeys = (int64_t)(cx.nopsL + cx.nopsR) * cx.nblk;
    if (key > nkeys) return;
    if (key == nkeys) { tsize[key] = 0; tflag[key] = 0; return; }     // sentinel: scan totals
    int64_t sz = 0;
    if (need[key]) {
        const int u = (int)(key / cx.nblk), bi = (int)(key % cx.nblk);
        const MapBlock& in = cx.blocks[bi];
        View v;
        if (u < cx.nopsL) { op_view(cx.L, cx.opsL[u], in.l, v); sz = (int64_t)v.rows * pad2i(in.cols); }
        else { op_view(cx.R, cx.opsR[u - cx.nopsL], in.r, v); sz = (int64_t)in.rows * pad2i(v.rows); }
    }
    tsize[key] = sz;
    tflag[key] = sz > 0;
}
__global__ void k_emit_p1(MapCtx cx, const int64_t* toff, const int* trank, const int* tflag_src, double* Tbuf,
                          Task* tasks, Seg* segs, double* wK, double* flops) {
    const int64_t key = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    const int64_t nkeys = (int64_t)(cx.nopsL + cx.nopsR) * cx.nblk;
    if (key >= nkeys || trank[key + 1] == trank[key]) return;
    (void)tflag_src;
    const int u = (int)(key / cx.nblk), bi = (int)(key % cx.nblk);
    const MapBlock& in = cx.blocks[bi];
    const double* xin = cx.xpad + in.poff;
    const int xld = pad2i(in.cols);
    View v;
    Task t; Seg s;
    t.C = Tbuf + toff[key]; t.flags = 0; t.seg_begin = trank[key]; t.seg_count = 1; t.ngemm = 1;
    s.alpha = 1.0;
    if (u < cx.nopsL) {                                           // T = O_L X
        op_view(cx.L, cx.opsL[u], in.l, v);
        t.ldc = pad2i(in.cols); t.M = v.rows; t.N = in.cols;
        s.A = v.ptr; s.lda = v.ld; s.B = xin; s.ldb = xld; s.K = in.rows; s.flags = v.trans ? SEG_TRANS_A : 0;
    } else {                                                      // T = X O_R^T
        op_view(cx.R, cx.opsR[u - cx.nopsL], in.r, v);
        t.ldc = pad2i(v.rows); t.M = in.rows; t.N = v.rows;
        s.A = xin; s.lda = xld; s.B = v.ptr; s.ldb = v.ld; s.K = in.cols; s.flags = v.trans ? 0 : SEG_TRANS_B;
    }
    tasks[trank[key]] = t;
    segs[trank[key]] = s;
    wK[trank[key]] = (double)s.K;
    atomicAdd(flops, 2.0 * t.M * (double)t.N * s.K);
}

// ---- per chunk: segments of every output block, output-major so that a prefix sum groups them by task -----------------
// split-K of phase 2: the chunk's term range [0, ntc) is cut into S contiguous parts; part s starts at split_begin
__device__ __host__ __forceinline__ int split_begin(int s, int ntc, int S) { return (int)(((int64_t)ntc * s) / S); }
__device__ __forceinline__ int split_part(int rel, int ntc, int S) {
    int s = (int)(((int64_t)rel * S) / ntc);
    while (s + 1 < S && split_begin(s + 1, ntc, S) <= rel) ++s;
    while (s > 0 && split_begin(s, ntc, S) > rel) --s;
    return s;
}
template <bool EMIT>
__global__ void k_p2(MapCtx cx, int t0, int t1, int S, const int* pos, const int64_t* toff, double* Tbuf, int* cnt, Seg* segs,
                     double* wK, int* nident, double* flops) {
    const int ntc = t1 - t0;
    const int64_t idx = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= (int64_t)cx.nblk * ntc) return;
    const int bo = (int)(idx / ntc), ti = t0 + (int)(idx % ntc);
    const MapTerm& t = cx.terms[ti];
    const MapBlock& ob = cx.blocks[bo];
    int n = 0, w = EMIT ? pos[idx] : 0;
    double ksum = 0.0, fl = 0.0;
    int idn = 0;
    for (int ab = 0; ab < 16; ++ab) {
        if (cx.dm[(size_t)t.dm * 256 + ob.ab * 16 + ab] == 0.0) continue;
        const int bi = source_block(cx, ti, bo, ab);
        if (bi < 0) continue;
        Contrib c;
        if (!contrib(cx, ti, bi, ob.ab, c) || c.bo != bo) continue;
        ++n;
        if (!EMIT) continue;
        const MapBlock& in = cx.blocks[bi];
        const double* xin = cx.xpad + in.poff;
        const int xld = pad2i(in.cols);
        Seg s;
        s.alpha = c.c;
        if (c.kase == C_NONE) { s.A = xin; s.lda = xld; s.B = nullptr; s.ldb = 0; s.K = 0; s.flags = SEG_IDENT_B; ++idn; }
        else if (c.kase == C_RONLY) { s.A = xin; s.lda = xld; s.B = c.vr.ptr; s.ldb = c.vr.ld; s.K = in.cols; s.flags = c.vr.trans ? 0 : SEG_TRANS_B; }
        else if (c.kase == C_LONLY) { s.A = c.vl.ptr; s.lda = c.vl.ld; s.B = xin; s.ldb = xld; s.K = in.rows; s.flags = c.vl.trans ? SEG_TRANS_A : 0; }
        else if (c.kase == C_LFIRST) {
            s.A = Tbuf + toff[tkey(cx, 0, t.opL, bi)]; s.lda = xld;
            s.B = c.vr.ptr; s.ldb = c.vr.ld; s.K = in.cols; s.flags = c.vr.trans ? 0 : SEG_TRANS_B;
        } else {
            s.A = c.vl.ptr; s.lda = c.vl.ld;
            s.B = Tbuf + toff[tkey(cx, 1, t.opR, bi)]; s.ldb = pad2i(c.vr.rows); s.K = in.rows; s.flags = c.vl.trans ? SEG_TRANS_A : 0;
        }
        segs[w++] = s;
        ksum += s.K;
        fl += 2.0 * ob.rows * (double)ob.cols * s.K;
    }
    if (!EMIT) { cnt[idx] = n; return; }
    const int part = split_part(ti - t0, ntc, S);            // split-K: which part of the chunk's term range
    if (ksum != 0.0) { atomicAdd(&wK[(size_t)part * cx.nblk + bo], ksum); atomicAdd(flops, fl); }
    if (idn) atomicAdd(&nident[(size_t)part * cx.nblk + bo], idn);
}
// task (part s, block b): part 0 accumulates into y, parts >= 1 write partial sums to ypart (added to y by the
// reduce launch in part order, so the summation order stays fixed)
__global__ void k_tasks2(MapCtx cx, int ntc, int S, const int* pos, const int* nident, int accum, double* ypart,
                         int64_t nnz, Task* tasks) {
    const int idx = blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= cx.nblk * S) return;
    const int s = idx / cx.nblk, b = idx % cx.nblk;
    const MapBlock& ob = cx.blocks[b];
    Task t;
    t.C = s == 0 ? cx.y + ob.off : ypart + (size_t)(s - 1) * nnz + ob.off;
    t.ldc = ob.cols; t.M = ob.rows; t.N = ob.cols;
    const int a0 = split_begin(s, ntc, S), a1 = split_begin(s + 1, ntc, S);
    t.seg_begin = pos[(size_t)b * ntc + a0];
    t.seg_count = pos[(size_t)b * ntc + a1] - t.seg_begin;       // pos has nblk * ntc + 1 entries: a1 == ntc is the next block's start
    t.flags = (s == 0 && accum) ? TASK_ACCUM : 0; t.ngemm = t.seg_count - nident[idx];
    tasks[idx] = t;
}
// reduce launch: y block += sum_s ypart[s] block (identity-B segments only), built once per plan
__global__ void k_reduce(MapCtx cx, int S, const double* ypart, int64_t nnz, Task* tasks, Seg* segs) {
    const int b = blockIdx.x * blockDim.x + threadIdx.x;
    if (b >= cx.nblk) return;
    const MapBlock& ob = cx.blocks[b];
    Task t;
    t.C = cx.y + ob.off; t.ldc = ob.cols; t.M = ob.rows; t.N = ob.cols;
    t.seg_begin = b * (S - 1); t.seg_count = S - 1; t.flags = TASK_ACCUM; t.ngemm = 0;
    tasks[b] = t;
    for (int s = 1; s < S; ++s) {
        Seg g;
        g.A = ypart + (size_t)(s - 1) * nnz + ob.off; g.lda = ob.cols; g.B = nullptr; g.ldb = 0; g.K = 0;
        g.flags = SEG_IDENT_B; g.alpha = 1.0;
        segs[b * (S - 1) + s - 1] = g;
    }
}

// ---- tiles: even split at the 8-row fragment level (same rule as finalize in block.cpp), heaviest first ---------------
__device__ __forceinline__ void tile_split(int M, int N, int& pm, int& pn, int& nm, int& nn) {
    const int qm = (M + GEMM_BM - 1) / GEMM_BM, qn = (N + GEMM_BN - 1) / GEMM_BN;
    pm = min(GEMM_BM, (((M + qm - 1) / qm) + 7) & ~7);
    pn = min(GEMM_BN, (((N + qn - 1) / qn) + 7) & ~7);
    nm = (M + pm - 1) / pm; nn = (N + pn - 1) / pn;
}
__global__ void k_tile_count(const Task* tasks, int ntasks, int* cnt) {
    const int t = blockIdx.x * blockDim.x + threadIdx.x;
    if (t > ntasks) return;
    if (t == ntasks) { cnt[t] = 0; return; }
    int pm, pn, nm, nn;
    if (tasks[t].M <= 0 || tasks[t].N <= 0) { cnt[t] = 0; return; }
    tile_split(tasks[t].M, tasks[t].N, pm, pn, nm, nn);
    cnt[t] = nm * nn;
}
__global__ void k_tile_emit(const Task* tasks, int ntasks, const int* pos, const double* wK, Tile* tiles, double* weight) {
    const int t = blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= ntasks || pos[t + 1] == pos[t]) return;
    int pm, pn, nm, nn;
    const int M = tasks[t].M, N = tasks[t].N;
    tile_split(M, N, pm, pn, nm, nn);
    int w = pos[t];
    for (int m0 = 0; m0 < M; m0 += pm)
        for (int n0 = 0; n0 < N; n0 += pn) {
            const int mv = min(pm, M - m0), nv = min(pn, N - n0);
            Tile tl; tl.task = t; tl.m0 = m0; tl.n0 = n0; tl.mv = mv; tl.nv = nv;
            tiles[w] = tl;
            weight[w] = (wK[t] + 16.0) * ((mv + 7) / 8) * ((nv + 7) / 8);   // (a per-task key was tried: no gain)
            ++w;
        }
}

}  // namespace

namespace {

struct Scratch {                                     // frees its device allocations on scope exit
    MapAlloc alloc; void (*dealloc)(void*);
    std::vector<void*> held;
    Scratch(MapAlloc a, void (*d)(void*)) : alloc(a), dealloc(d) {}
    ~Scratch() { for (void* p : held) dealloc(p); }
    template <class T> T* get(size_t n, cudaStream_t st, bool zero) {
        T* p = (T*)alloc(std::max<size_t>(n, 1) * sizeof(T));
        held.push_back(p);
        if (zero) cudaMemsetAsync(p, 0, std::max<size_t>(n, 1) * sizeof(T), st);
        return p;
    }
};
inline unsigned nblocks(int64_t n, int bs) { return (unsigned)((n + bs - 1) / bs); }

// tiles of a task list, sorted by weight (heaviest first); tiles is allocated for the caller
int build_tiles(const Task* tasks, int ntasks, const double* wK, Tile** tiles_out, Scratch& sc, MapAlloc alloc,
                cudaStream_t st) {
    if (ntasks == 0) { *tiles_out = nullptr; return 0; }
    auto pol = thrust::cuda::par.on(st);
    int* cnt = sc.get<int>((size_t)ntasks + 1, st, false);
    k_tile_count<<<nblocks(ntasks + 1, 256), 256, 0, st>>>(tasks, ntasks, cnt);
    thrust::exclusive_scan(pol, cnt, cnt + ntasks + 1, cnt);
    int ntiles = 0;
    cudaMemcpyAsync(&ntiles, cnt + ntasks, sizeof(int), cudaMemcpyDeviceToHost, st);
    cudaStreamSynchronize(st);
    if (ntiles == 0) { *tiles_out = nullptr; return 0; }
    Tile* tiles = (Tile*)alloc((size_t)ntiles * sizeof(Tile));
    double* w = sc.get<double>((size_t)ntiles, st, false);
    k_tile_emit<<<nblocks(ntasks, 256), 256, 0, st>>>(tasks, ntasks, cnt, wK, tiles, w);
    thrust::stable_sort_by_key(pol, w, w + ntiles, tiles, thrust::greater<double>());
    *tiles_out = tiles;
    return ntiles;
}

}  // namespace

void maps_usage(const MapCtx& cx, std::vector<double>& usage_host, MapBuild& out, MapAlloc alloc, void (*dealloc)(void*),
                cudaStream_t st) {
    Scratch sc(alloc, dealloc);
    auto pol = thrust::cuda::par.on(st);
    const int64_t npair = (int64_t)cx.nterm * cx.nblk;
    double* usage = sc.get<double>((size_t)cx.nterm, st, true);
    double* stats = sc.get<double>(3, st, true);
    int* dcnt = sc.get<int>((size_t)npair + 1, st, true);
    const int64_t ntouch = (int64_t)cx.nrefL * cx.L.nsec + (int64_t)cx.nrefR * cx.R.nsec;
    unsigned char* touched = sc.get<unsigned char>((size_t)ntouch, st, true);
    if (npair > 0) {
        k_term_usage<<<nblocks(npair, 128), 128, 0, st>>>(cx, usage, stats, dcnt, touched);
        if (ntouch > 0) k_touched_bytes<<<nblocks(ntouch, 256), 256, 0, st>>>(cx, touched, stats);
        thrust::exclusive_scan(pol, dcnt, dcnt + npair + 1, dcnt);
    }
    int ndiag = 0;
    cudaMemcpyAsync(&ndiag, dcnt + npair, sizeof(int), cudaMemcpyDeviceToHost, st);
    double hs[3] = {0, 0, 0};
    cudaMemcpyAsync(hs, stats, sizeof hs, cudaMemcpyDeviceToHost, st);
    usage_host.assign((size_t)cx.nterm, 0.0);
    if (cx.nterm) cudaMemcpyAsync(usage_host.data(), usage, (size_t)cx.nterm * 8, cudaMemcpyDeviceToHost, st);
    cudaStreamSynchronize(st);
    out.f_alg = hs[0]; out.ngemm = hs[1]; out.b_ops = hs[2];
    out.ndiag = ndiag;
    out.diag_items = (DiagItemK*)alloc(std::max<size_t>(ndiag, 1) * sizeof(DiagItemK));
    out.diag_ptr = (int*)alloc(((size_t)cx.nblk + 1) * sizeof(int));
    if (npair > 0) k_diag_emit<<<nblocks(npair, 128), 128, 0, st>>>(cx, dcnt, out.diag_items);
    k_diag_ptr<<<nblocks(cx.nblk + 1, 256), 256, 0, st>>>(cx.nblk, cx.nterm, dcnt, out.diag_ptr);
    cudaStreamSynchronize(st);
}

void maps_reduce(const MapCtx& cx, int S, double* ypart, int64_t nnz, MapChunkOut& out, MapAlloc alloc,
                 void (*dealloc)(void*), cudaStream_t st) {
    Scratch sc(alloc, dealloc);
    out.ntasks2 = cx.nblk; out.nsegs2 = cx.nblk * (S - 1);
    out.tasks2 = (Task*)alloc(std::max<size_t>(cx.nblk, 1) * sizeof(Task));
    out.segs2 = (Seg*)alloc(std::max<size_t>(out.nsegs2, 1) * sizeof(Seg));
    k_reduce<<<nblocks(cx.nblk, 128), 128, 0, st>>>(cx, S, ypart, nnz, out.tasks2, out.segs2);
    double* w0 = sc.get<double>((size_t)cx.nblk, st, true);
    out.ntiles2 = build_tiles(out.tasks2, cx.nblk, w0, &out.tiles2, sc, alloc, st);
    cudaStreamSynchronize(st);
}

void maps_chunk(const MapCtx& cx, int t0, int t1, bool first_chunk, double* Tbuf, int S, double* ypart, int64_t nnz,
                MapChunkOut& out, MapAlloc alloc, void (*dealloc)(void*), cudaStream_t st) {
    Scratch sc(alloc, dealloc);
    auto pol = thrust::cuda::par.on(st);
    const int ntc = t1 - t0;
    const int64_t nkeys = (int64_t)(cx.nopsL + cx.nopsR) * cx.nblk;
    // ---- phase 1: distinct intermediates of the chunk ---------------------------------------------------------------------
    unsigned char* need = sc.get<unsigned char>((size_t)nkeys, st, true);
    int64_t* toff = sc.get<int64_t>((size_t)nkeys + 1, st, false);
    int* trank = sc.get<int>((size_t)nkeys + 1, st, false);
    if ((int64_t)ntc * cx.nblk > 0) k_mark<<<nblocks((int64_t)ntc * cx.nblk, 128), 128, 0, st>>>(cx, t0, t1, need);
    k_tsize<<<nblocks(nkeys + 1, 256), 256, 0, st>>>(cx, need, toff, trank);
    thrust::exclusive_scan(pol, toff, toff + nkeys + 1, toff);
    thrust::exclusive_scan(pol, trank, trank + nkeys + 1, trank);
    int64_t tdoubles = 0;
    int ntasks1 = 0;
    cudaMemcpyAsync(&tdoubles, toff + nkeys, 8, cudaMemcpyDeviceToHost, st);
    cudaMemcpyAsync(&ntasks1, trank + nkeys, 4, cudaMemcpyDeviceToHost, st);
    cudaStreamSynchronize(st);
    out.t_doubles = tdoubles;
    out.ntasks1 = out.nsegs1 = ntasks1;
    double* fl = sc.get<double>(2, st, true);
    if (ntasks1 > 0) {
        out.tasks1 = (Task*)alloc((size_t)ntasks1 * sizeof(Task));
        out.segs1 = (Seg*)alloc((size_t)ntasks1 * sizeof(Seg));
        double* wK1 = sc.get<double>((size_t)ntasks1, st, false);
        k_emit_p1<<<nblocks(nkeys, 256), 256, 0, st>>>(cx, toff, trank, nullptr, Tbuf, out.tasks1, out.segs1, wK1, fl);
        out.ntiles1 = build_tiles(out.tasks1, ntasks1, wK1, &out.tiles1, sc, alloc, st);
    }
    // ---- phase 2: one task per psi block, segments in (block, term) order ------------------------------------------------------
    const int64_t npair = (int64_t)cx.nblk * ntc;
    int* pos = sc.get<int>((size_t)npair + 1, st, true);
    if (npair > 0) k_p2<false><<<nblocks(npair, 128), 128, 0, st>>>(cx, t0, t1, S, nullptr, toff, Tbuf, pos, nullptr, nullptr, nullptr, nullptr);
    thrust::exclusive_scan(pol, pos, pos + npair + 1, pos);
    int nsegs2 = 0;
    cudaMemcpyAsync(&nsegs2, pos + npair, 4, cudaMemcpyDeviceToHost, st);
    cudaStreamSynchronize(st);
    out.nsegs2 = nsegs2;
    out.ntasks2 = cx.nblk * S;
    out.tasks2 = (Task*)alloc(std::max<size_t>((size_t)cx.nblk * S, 1) * sizeof(Task));
    out.segs2 = (Seg*)alloc(std::max<size_t>(nsegs2, 1) * sizeof(Seg));
    double* wK2 = sc.get<double>((size_t)cx.nblk * S, st, true);
    int* nident = sc.get<int>((size_t)cx.nblk * S, st, true);
    if (npair > 0) k_p2<true><<<nblocks(npair, 128), 128, 0, st>>>(cx, t0, t1, S, pos, toff, Tbuf, nullptr, out.segs2, wK2, nident, fl + 1);
    k_tasks2<<<nblocks((int64_t)cx.nblk * S, 256), 256, 0, st>>>(cx, ntc, S, pos, nident, first_chunk ? 0 : 1, ypart, nnz, out.tasks2);
    out.ntiles2 = build_tiles(out.tasks2, cx.nblk * S, wK2, &out.tiles2, sc, alloc, st);
    out.split = S;
    double hf[2] = {0, 0};
    cudaMemcpyAsync(hf, fl, sizeof hf, cudaMemcpyDeviceToHost, st);
    cudaStreamSynchronize(st);
    out.flops1 = hf[0]; out.flops2 = hf[1];
}

}  // namespace dmrg
