// 1- and 2-particle reduced density matrices of the current MPS (DESIGN.md 5.4 "RDM pass").
//   gamma_pq = <E_pq>                                  PAPER.md:91 (Eq. 9)
//   Gamma_pqrs = <sum_ss' a+_ps a+_rs' a_ss' a_qs>     PAPER.md:93 (Eq. 10) under readings S1/S2
//
// Half-chain partition.  Every spin-orbital element <a+_P a+_Q a_R a_S> (P<Q, S<R,
// Sz-conserving; the other orderings follow by antisymmetry) is evaluated once, at a one-site centre c chosen from the
// sorted sites s1 <= s2 <= s3 <= s4 of its four operators and kh = k/2:
//   s3 <  kh : c = s3   ("left rule")  - at most two operators left of the centre, both on sites < kh, at most one right
//   s3 >= kh : c = s2   ("right rule") - at most one operator left, at most two right, both on sites >= kh
// so a renormalised two-index operator A_PQ = a+_P a+_Q / B_PS = a+_P a_S is only ever needed for a pair of sites inside
// one half of the chain: O((k/2)^2) stored operators on the side that carries them instead of O(k^2), which is what
// lets the pass run BASELINE configs 4 and 5.  The pass is two sweeps of the centre:
//   left-rule pass   c = 0 .. kh-1 (centre moving right): left block with 1, a+_P, A, B (pairs of sites < kh), right
//                    blocks with a+_P only (all kept; built once from the right-canonical MPS);
//   (the centre then continues to k-1, keeping the left-orthonormal tensors and the left one-index blocks)
//   right-rule pass  c = k-1 .. 0 (centre moving left): right block with 1, a+_P, A, B (pairs of sites >= kh), left
//                    one-index blocks from the first pass; the 1-RDM strings a+_P a_S are evaluated here at the
//                    smaller of their two sites.
// At a centre every string is  <psi_c| Y (x) o_c (x) X |psi_c>  with X on the two-index ("stack") side and Y on the
// other; with  M_{Y,s',s} = sgn psi[s']^(T) Y psi[s]  contracted over the Y-side bond (two grouped FP64 GEMM launches
// for all (Y, s', s) of a centre), the value is  sum_{s',s} o[s',s] <X, M_{Y,s',s}>,  and the contraction of EVERY
// stored operator of one quantum-number class with all its M is one product  E = Stack [n_ops x nnz] . M^T [nnz x n_M]
// that streams each stored operator once per centre: the HBM-bound streaming kernel for n_M <= 8, split-K launches of
// the grouped DMMA GEMM otherwise.  E stays on the device until the centre is finished (one download per centre); the
// strings of the centre are then enumerated on the host with dense lookup tables and scattered into gamma / Gamma.
#include <algorithm>
#include <chrono>
#include <cmath>
#include <cstdlib>
#include <cstring>

#include <cuda_profiler_api.h>
#include <omp.h>

#include "core.hpp"

namespace dmrg {

namespace {

double now_s() { return std::chrono::duration<double>(std::chrono::steady_clock::now().time_since_epoch()).count(); }

struct OpTok { int P; int dag; };

// site-local matrices in the basis |0>, |dn>, |up>, |up dn> = a+_up a+_dn |0>  (reading S3)
struct M4 { double a[16]; };
M4 m4_eye() { M4 m; std::memset(&m, 0, sizeof m); for (int i = 0; i < 4; ++i) m.a[i * 5] = 1.0; return m; }
M4 m4_mul(const M4& x, const M4& y) {
    M4 r; std::memset(&r, 0, sizeof r);
    for (int i = 0; i < 4; ++i)
        for (int l = 0; l < 4; ++l) if (x.a[i * 4 + l] != 0.0)
            for (int j = 0; j < 4; ++j) r.a[i * 4 + j] += x.a[i * 4 + l] * y.a[l * 4 + j];
    return r;
}
M4 m4_site(int down, int dag) {
    M4 m; std::memset(&m, 0, sizeof m);
    if (!down) { m.a[0 * 4 + 2] = 1.0; m.a[1 * 4 + 3] = 1.0; }     // a_up
    else       { m.a[0 * 4 + 1] = 1.0; m.a[2 * 4 + 3] = -1.0; }    // a_dn
    if (dag) { M4 t; for (int i = 0; i < 4; ++i) for (int j = 0; j < 4; ++j) t.a[j * 4 + i] = m.a[i * 4 + j]; return t; }
    return m;
}

// Bump allocator over one device allocation made per dmrg_rdm12 call (thousands of short-lived intermediates per
// centre; a cudaMalloc / cudaFree pair each would synchronise the device every time).
struct Arena {
    DevVec<double> buf;
    size_t used = 0;
    std::vector<DevVec<double>> overflow;         // requests that do not fit fall back to their own allocation
    void init(size_t doubles) { buf.alloc(doubles); used = 0; }
    void reset() { used = 0; overflow.clear(); }
    double* get(size_t n) {
        n = (n + 1) & ~(size_t)1;                 // keep 16-byte alignment
        if (used + n <= buf.n) { double* p = buf.p + used; used += n; return p; }
        overflow.emplace_back();
        overflow.back().alloc(n);
        return overflow.back().p;
    }
};

struct Group {                      // all M vectors contracted with the stored operators of one (class, trans) of the stack side
    int cls = -1, trans = 0;
    std::vector<int> keys;          // (yid << 4) | (s_out * 4 + s_in), in column order
    std::vector<int> col;           // [yid * 16 + e] -> column or -1
    std::vector<int> stacks;        // stacks of the stack-side block whose rows are contracted with these columns
    std::vector<int64_t> eoff;      // per stack: offset of its E [n_ops x ncol] in the centre's E buffer
};
struct XOp { int stack, row, cls; };

struct Centre {
    int c = 0, k = 0, kh = 0;
    bool stack_left = true;         // the two-index ("stack") side X is the left block
    Block* XB = nullptr;
    Block* YB = nullptr;
    const SiteTensor* psi = nullptr;
    std::vector<Group> groups;
    std::vector<int> group_of;      // [cls * 2 + trans] -> group or -1
    std::vector<int64_t> eoff_of;   // [stack * 2 + trans] -> offset into E or -1
    int ny = 0;
    int64_t esize = 0;
    std::vector<XOp> xops;
    std::vector<int> xC, xA, xB;    // [P], [P * nso + Q], [P * nso + S] -> index into xops or -1
    int xI = -1;
    int part(int P) const { const int s = P >> 1; return s < c ? 0 : (s == c ? 1 : 2); }
};

void build_tables(Centre& cx) {
    const int nso = 2 * cx.k;
    Block& XB = *cx.XB;
    cx.xC.assign(nso, -1); cx.xA.assign((size_t)nso * nso, -1); cx.xB.assign((size_t)nso * nso, -1);
    for (const auto& kv : XB.ops) {
        const int kind = (int)(kv.first >> 24), a = (int)((kv.first >> 16) & 255), b = (int)((kv.first >> 8) & 255);
        const OpRef& r = kv.second;
        const int idx = (int)cx.xops.size();
        if (kind == K_I) cx.xI = idx;
        else if (kind == K_C) cx.xC[a] = idx;
        else if (kind == K_A) cx.xA[(size_t)a * nso + b] = idx;
        else if (kind == K_B) cx.xB[(size_t)a * nso + b] = idx;
        else continue;
        cx.xops.push_back({r.stack, r.row, r.cls});
    }
    // columns: every (Y, s_out, s_in) goes to the (class, trans) of the X operators that close the string
    const int g = XB.g();
    cx.ny = 1 + 2 * nso;
    cx.group_of.assign(XB.classes.size() * 2, -1);
    std::vector<int> yids(1, 0);
    for (int P : cx.YB->inside()) { yids.push_back(1 + 2 * P); yids.push_back(1 + 2 * P + 1); }
    for (int yid : yids) {
        int yn = 0, ys = 0;
        if (yid) { const int P = (yid - 1) >> 1, dag = (yid - 1) & 1; yn = dag ? 1 : -1; ys = dag ? spin_of(P) : -spin_of(P); }
        for (int e = 0; e < 16; ++e) {
            const int so = e >> 2, si = e & 3;
            const int dn = -(yn + SITE_QN[so] - SITE_QN[si]), ds = -(ys + SITE_QS[so] - SITE_QS[si]);
            if (dn < -2 || dn > 2) continue;
            const int trans = dn < 0 ? 1 : 0;
            const int sdn = trans ? -dn : dn, sds = trans ? -ds : ds;
            int cls = -1;
            for (size_t q = 0; q < XB.classes.size(); ++q)
                if (XB.classes[q].dn == g * sdn && XB.classes[q].ds == g * sds) { cls = (int)q; break; }
            if (cls < 0) continue;
            int& gi = cx.group_of[cls * 2 + trans];
            if (gi < 0) {
                gi = (int)cx.groups.size();
                cx.groups.emplace_back();
                cx.groups.back().cls = cls; cx.groups.back().trans = trans;
                cx.groups.back().col.assign((size_t)cx.ny * 16, -1);
            }
            Group& G = cx.groups[gi];
            G.col[(size_t)yid * 16 + e] = (int)G.keys.size();
            G.keys.push_back((yid << 4) | e);
        }
    }
    cx.eoff_of.assign(XB.stacks.size() * 2, -1);
    for (Group& G : cx.groups)
        for (size_t s = 0; s < XB.stacks.size(); ++s) {
            const Stack& st = XB.stacks[s];
            if (st.cls != G.cls || st.members.empty() || st.alloc < 0) continue;
            const bool ok = G.trans ? (st.kind == K_C || st.kind == K_A)
                                    : (st.kind == K_I || st.kind == K_C || st.kind == K_A || st.kind == K_B);
            if (!ok) continue;
            G.stacks.push_back((int)s);
            G.eoff.push_back(cx.esize);
            cx.eoff_of[s * 2 + G.trans] = cx.esize;
            cx.esize += (int64_t)st.members.size() * (int64_t)G.keys.size();
        }
}

struct Evaluator {
    Engine& eng;
    Arena arena;
    DevVec<double> Ebuf;
    double* Ehost = nullptr;
    size_t Ehost_n = 0;
    cudaEvent_t e0 = nullptr, e1 = nullptr, e2 = nullptr, e3 = nullptr;
    explicit Evaluator(Engine& e) : eng(e) {
        cuda_check(cudaEventCreate(&e0), "event"); cuda_check(cudaEventCreate(&e1), "event");
        cuda_check(cudaEventCreate(&e2), "event"); cuda_check(cudaEventCreate(&e3), "event");
    }
    ~Evaluator() {
        if (Ehost) cudaFreeHost(Ehost);
        cudaEventDestroy(e0); cudaEventDestroy(e1); cudaEventDestroy(e2); cudaEventDestroy(e3);
    }
    Evaluator(const Evaluator&) = delete;

    struct DotsCall { const double* S; int64_t ld; int nrows; const double* M; int nc; double* E; int ldE; double* scratch; };
    GemmBatch p1, p2, pe, pred;
    std::vector<DotsCall> dots;
    std::unordered_map<uint64_t, std::pair<double*, int>> tcache;      // (yid, psi block) -> (T, ld)

    void flush() {
        cudaStream_t st = eng.stream;
        eng.rdm_flops += p1.flops + p2.flops + pe.flops;
        run_once(p1, eng);
        run_once(p2, eng);
        // DMRG_B200_PROFILE_RDM=1 (diagnostics): open the profiler range around the accumulation launches only, so that
        // `ncu --profile-from-start off` lists exactly the E = Stack M^T kernels of the pass
        static const bool prof = [] { const char* g = std::getenv("DMRG_B200_PROFILE_RDM"); return g && g[0] == '1'; }();
        if (prof) cudaProfilerStart();
        if (!dots.empty()) {
            cudaEventRecord(e0, st);
            for (const DotsCall& d : dots) {
                launch_stack_dots(d.S, d.ld, d.nrows, d.M, d.ld, d.nc, d.ld, d.E, d.ldE, d.scratch, st);
                eng.launches += 2;
                eng.rdm_flops += 2.0 * d.nrows * (double)d.nc * (double)d.ld;
                eng.rdm_stream_bytes += 8.0 * ((double)d.nrows * d.ld + (double)d.nc * d.ld);
            }
            cudaEventRecord(e1, st);
        }
        const bool gem = !pe.empty();
        GemmLaunch le, lr;
        if (gem) {
            finalize(pe, le, eng);
            finalize(pred, lr, eng);
            cudaEventRecord(e2, st);
            run(le, eng);
            cudaEventRecord(e3, st);
            run(lr, eng);
        }
        cuda_check(cudaStreamSynchronize(st), "rdm accumulation");
        if (prof) cudaProfilerStop();
        float ms = 0.f;
        if (!dots.empty()) { cudaEventElapsedTime(&ms, e0, e1); eng.rdm_stream_ms += ms; }
        if (gem) { cudaEventElapsedTime(&ms, e2, e3); eng.rdm_gemm_ms += ms; }
        p1 = GemmBatch(); p2 = GemmBatch(); pe = GemmBatch(); pred = GemmBatch();
        dots.clear();
        tcache.clear();
        arena.reset();
    }

    // M vectors of columns [c0, c0 + nc) of group G (in the storage layout of the class) into Mbuf
    void build_columns(Centre& cx, const Group& G, int c0, int nc, double* Mbuf, const std::vector<int>& by_rs) {
        Block& XB = *cx.XB;
        Block& YB = *cx.YB;
        const SiteTensor& psi = *cx.psi;
        const OpClass& cls = XB.classes[G.cls];
        const int64_t ld = cls.ld;
        const int par_x = (cls.dn & 1) ? 1 : 0;
        for (int cc = 0; cc < nc; ++cc) {
            const int key = G.keys[c0 + cc];
            const int yid = key >> 4, s_out = (key & 15) >> 2, s_in = key & 3;
            const OpRef* yref = nullptr;
            bool ytrans = false;
            if (yid) { const int P = (yid - 1) >> 1, dag = (yid - 1) & 1; yref = &YB.get(L1(K_C, P)); ytrans = !dag; }
            const int par_y = yid ? 1 : 0, par_o = (SITE_QN[s_out] - SITE_QN[s_in]) & 1;
            double* mcol = Mbuf + (size_t)cc * ld;
            for (int a = 0; a < (int)XB.basis.size(); ++a) {
                const int b = cls.out[a];
                if (b < 0) continue;
                const int xk = G.trans ? b : a, xb = G.trans ? a : b;          // ket / bra sector of X as used
                const int db = XB.basis[b].d, da = XB.basis[a].d;
                if (cx.stack_left) {
                    // M[l', l] = sgn psi[(l', s')] Y psi[(l, s)]^T,  T = psi[(l, s)] Y^T
                    const SiteTensor::Blk* kb = psi.get(xk, s_in);
                    const SiteTensor::Blk* bb = psi.get(xb, s_out);
                    if (!kb || !bb) continue;
                    const double* tptr = kb->ptr;
                    int tld = kb->ld;
                    if (yref) {
                        OpBlockView v;
                        if (!op_block(YB, *yref, ytrans, kb->r, v) || v.out != bb->r) continue;
                        const uint64_t tk = ((uint64_t)yid << 32) | (uint64_t)(kb - psi.blocks.data());
                        auto it = tcache.find(tk);
                        if (it == tcache.end()) {
                            const int dro = YB.basis[v.out].d;
                            double* tp = arena.get((size_t)kb->rows * pad2(dro));
                            const int t1 = p1.add_task(tp, pad2(dro), kb->rows, dro, 0);
                            p1.add_seg(t1, kb->ptr, kb->ld, v.ptr, v.ld, kb->cols, v.trans ? 0 : SEG_TRANS_B, 1.0);
                            it = tcache.emplace(tk, std::make_pair(tp, pad2(dro))).first;
                        }
                        tptr = it->second.first; tld = it->second.second;
                    } else if (kb->r != bb->r) continue;
                    const int nl = XB.basis[xk].n;
                    const double sgn = ((par_y * (nl + SITE_QN[s_in]) + par_o * nl) & 1) ? -1.0 : 1.0;
                    const int t2 = p2.add_task(mcol + cls.off[a], pad2(da), db, da, 0);
                    if (!G.trans) p2.add_seg(t2, bb->ptr, bb->ld, tptr, tld, bb->cols, SEG_TRANS_B, sgn);   // psi' T^T
                    else          p2.add_seg(t2, tptr, tld, bb->ptr, bb->ld, bb->cols, SEG_TRANS_B, sgn);   // T psi'^T
                } else {
                    // M[r', r] = sgn psi[(l', s')]^T Y psi[(l, s)],  T = Y psi[(l, s)]
                    const int ki = by_rs[xk * 4 + s_in], bi = by_rs[xb * 4 + s_out];
                    if (ki < 0 || bi < 0) continue;
                    const SiteTensor::Blk* kb = &psi.blocks[ki];
                    const SiteTensor::Blk* bb = &psi.blocks[bi];
                    const double* tptr = kb->ptr;
                    int tld = kb->ld;
                    if (yref) {
                        OpBlockView v;
                        if (!op_block(YB, *yref, ytrans, kb->l, v) || v.out != bb->l) continue;
                        const uint64_t tk = ((uint64_t)yid << 32) | (uint64_t)ki;
                        auto it = tcache.find(tk);
                        if (it == tcache.end()) {
                            double* tp = arena.get((size_t)v.rows * kb->ld);
                            const int t1 = p1.add_task(tp, kb->ld, v.rows, kb->cols, 0);
                            p1.add_seg(t1, v.ptr, v.ld, kb->ptr, kb->ld, kb->rows, v.trans ? SEG_TRANS_A : 0, 1.0);
                            it = tcache.emplace(tk, std::make_pair(tp, kb->ld)).first;
                        }
                        tptr = it->second.first; tld = it->second.second;
                    } else if (kb->l != bb->l) continue;
                    const int nl = YB.basis[kb->l].n;
                    const double sgn = ((par_o * nl + par_x * (nl + SITE_QN[s_in])) & 1) ? -1.0 : 1.0;
                    const int t2 = p2.add_task(mcol + cls.off[a], pad2(da), db, da, 0);
                    if (!G.trans) p2.add_seg(t2, bb->ptr, bb->ld, tptr, tld, bb->rows, SEG_TRANS_A, sgn);   // psi'^T T   [r' x r]
                    else          p2.add_seg(t2, tptr, tld, bb->ptr, bb->ld, bb->rows, SEG_TRANS_A, sgn);   // T^T psi'   [r x r']
                }
            }
        }
    }

    // E of every (group, stack) of the centre -> Ehost
    void evaluate(Centre& cx) {
        cudaStream_t st = eng.stream;
        Block& XB = *cx.XB;
        const SiteTensor& psi = *cx.psi;
        if (cx.esize == 0) return;
        if ((size_t)cx.esize > Ebuf.n) Ebuf.alloc((size_t)cx.esize + (size_t)cx.esize / 4);
        cuda_check(cudaMemsetAsync(Ebuf.p, 0, (size_t)cx.esize * 8, st), "memset");
        std::vector<int> by_rs;
        if (!cx.stack_left) {
            by_rs.assign(XB.basis.size() * 4, -1);
            for (size_t j = 0; j < psi.blocks.size(); ++j) by_rs[psi.blocks[j].r * 4 + psi.blocks[j].s] = (int)j;
        }
        const int64_t cap = (int64_t)arena.buf.n;
        for (const Group& G : cx.groups) {
            const OpClass& cls = XB.classes[G.cls];
            const int ncol = (int)G.keys.size();
            if (cls.nnz == 0 || ncol == 0 || G.stacks.empty()) continue;
            const int64_t ld = cls.ld;
            const int chunk_cols = (int)std::max<int64_t>(1, std::min<int64_t>(ncol, (cap / 3) / ld));
            for (int c0 = 0; c0 < ncol; c0 += chunk_cols) {
                const int nc = std::min(chunk_cols, ncol - c0);
                if ((int64_t)arena.used + (int64_t)nc * ld > (cap * 2) / 3) flush();
                double* Mbuf = arena.get((size_t)nc * ld);
                cuda_check(cudaMemsetAsync(Mbuf, 0, (size_t)nc * ld * 8, st), "memset");
                build_columns(cx, G, c0, nc, Mbuf, by_rs);
                for (size_t si = 0; si < G.stacks.size(); ++si) {
                    const Stack& stk = XB.stacks[G.stacks[si]];
                    const int nrows = (int)stk.members.size();
                    double* Eout = Ebuf.p + G.eoff[si] + c0;
                    eng.rdm_bytes += 8.0 * ((double)nrows * ld + (double)nc * ld);
                    if (nc <= 8) {
                        // few right-hand sides: the HBM-bound streaming kernel (coalesced 16-byte loads of every stored
                        // operator, warp-level reductions, fixed-order partial sums) instead of the tensor-pipe GEMM
                        double* scratch = arena.get((size_t)stack_dots_scratch(nrows, nc, ld));
                        dots.push_back({stk.base, ld, nrows, Mbuf, nc, Eout, ncol, scratch});
                        continue;
                    }
                    const int tiles = ((nrows + GEMM_BM - 1) / GEMM_BM) * ((nc + GEMM_BN - 1) / GEMM_BN);
                    int64_t nsplit = std::max<int64_t>(1, ld / 32768);
                    if (tiles * nsplit < 1776) nsplit = std::max<int64_t>(nsplit, std::min<int64_t>((1776 + tiles - 1) / tiles, std::max<int64_t>(1, ld / 4096)));
                    int64_t kc = (ld + nsplit - 1) / nsplit;
                    kc = (kc + 15) & ~(int64_t)15;
                    nsplit = (ld + kc - 1) / kc;
                    if (nsplit == 1) {
                        const int t = pe.add_task(Eout, ncol, nrows, nc, 0);
                        pe.add_seg(t, stk.base, (int)ld, Mbuf, (int)ld, (int)ld, SEG_TRANS_B, 1.0);
                    } else {
                        double* part = arena.get((size_t)nsplit * nrows * pad2(nc));
                        const int tr = pred.add_task(Eout, ncol, nrows, nc, 0);
                        for (int p = 0; p < (int)nsplit; ++p) {
                            const int64_t k0 = (int64_t)p * kc, kk = std::min<int64_t>(kc, ld - k0);
                            double* pp = part + (size_t)p * nrows * pad2(nc);
                            const int t = pe.add_task(pp, pad2(nc), nrows, nc, 0);
                            pe.add_seg(t, stk.base + k0, (int)ld, Mbuf + k0, (int)ld, (int)kk, SEG_TRANS_B, 1.0);
                            pred.add_seg(tr, pp, pad2(nc), nullptr, 0, 0, SEG_IDENT_B, 1.0);
                        }
                    }
                }
            }
        }
        flush();
        if ((size_t)cx.esize > Ehost_n) {
            if (Ehost) cudaFreeHost(Ehost);
            Ehost = nullptr;
            Ehost_n = (size_t)cx.esize + (size_t)cx.esize / 4;
            cuda_check(cudaHostAlloc((void**)&Ehost, Ehost_n * 8, cudaHostAllocDefault), "pinned E buffer");
        }
        cuda_check(cudaMemcpyAsync(Ehost, Ebuf.p, (size_t)cx.esize * 8, cudaMemcpyDeviceToHost, st), "E download");
        cuda_check(cudaStreamSynchronize(st), "E download");
    }
};

// Host scatter of one centre: enumerate its strings, read their values from E, accumulate gamma / Gamma.
struct Scatter {
    Centre& cx;
    const double* E;
    double inv_nrm2;
    double* gamma;
    double* Gamma;
    size_t K1;
    int nso;
    std::vector<M4> omats;
    std::vector<int> ocode_of;      // dense over the code of the centre-operator product
    Scatter(Centre& c, const double* E_, double nrm2, double* g, double* G)
        : cx(c), E(E_), inv_nrm2(1.0 / nrm2), gamma(g), Gamma(G), K1((size_t)c.k), nso(2 * c.k), ocode_of(2048, -1) {}

    void add2(int A, int B, int C, int D, double v) {                 // Gamma^so_ABCD = <a+_A a+_B a_C a_D>
        if (spin_of(A) != spin_of(D) || spin_of(B) != spin_of(C)) return;
        Gamma[((((size_t)(A >> 1)) * K1 + (D >> 1)) * K1 + (B >> 1)) * K1 + (C >> 1)] += v;
    }
    // the string  prod ops  (creators first), already known to conserve N and 2Sz
    void string(const OpTok* ops, int n, const int* tgt) {
        int order[4], prt[4];
        for (int j = 0; j < n; ++j) { order[j] = j; prt[j] = cx.part(ops[j].P); }
        double sign = 1.0;
        for (int a = 0; a < n; ++a)                          // stable bubble sort into chain order, sign per swap
            for (int b = 0; b + 1 < n - a; ++b)
                if (prt[order[b]] > prt[order[b + 1]]) { std::swap(order[b], order[b + 1]); sign = -sign; }
        OpTok lo[4], co[4], ro[4];
        int nl = 0, nc = 0, nr = 0;
        for (int j = 0; j < n; ++j) {
            const OpTok& t = ops[order[j]];
            if (prt[order[j]] == 0) lo[nl++] = t; else if (prt[order[j]] == 1) co[nc++] = t; else ro[nr++] = t;
        }
        const OpTok* xo = cx.stack_left ? lo : ro;
        const OpTok* yo = cx.stack_left ? ro : lo;
        const int nx = cx.stack_left ? nl : nr, nyo = cx.stack_left ? nr : nl;
        if (nx > 2 || nyo > 1) throw std::logic_error("rdm: string does not belong to this centre");
        int xi = cx.xI, xtrans = 0;
        if (nx == 1) { xi = cx.xC[xo[0].P]; xtrans = xo[0].dag ? 0 : 1; }
        else if (nx == 2) {
            const int X = xo[0].P, Y = xo[1].P;
            if (xo[0].dag && xo[1].dag) { if (X < Y) xi = cx.xA[(size_t)X * nso + Y]; else { xi = cx.xA[(size_t)Y * nso + X]; sign = -sign; } }
            else if (!xo[0].dag && !xo[1].dag) {               // a_X a_Y = (a+_Y a+_X)^T
                xtrans = 1;
                if (Y < X) xi = cx.xA[(size_t)Y * nso + X]; else { xi = cx.xA[(size_t)X * nso + Y]; sign = -sign; }
            } else if (xo[0].dag && !xo[1].dag) xi = cx.xB[(size_t)X * nso + Y];
            else throw std::logic_error("rdm: annihilator before creator inside a block");
        }
        if (xi < 0) throw std::logic_error("rdm: stored operator missing on the stack side");
        const XOp& xr = cx.xops[xi];
        int code = nc;
        for (int j = 0; j < nc; ++j) code = code * 4 + ((co[j].P & 1) * 2 + co[j].dag);
        int oc = ocode_of[code];
        if (oc < 0) {
            M4 om = m4_eye();
            for (int j = 0; j < nc; ++j) om = m4_mul(om, m4_site(co[j].P & 1, co[j].dag));
            omats.push_back(om);
            oc = ocode_of[code] = (int)omats.size() - 1;
        }
        const int yid = nyo ? 1 + 2 * yo[0].P + yo[0].dag : 0;
        double v = 0.0;
        const int gi = cx.group_of[xr.cls * 2 + xtrans];
        if (gi >= 0) {
            const Group& G = cx.groups[gi];
            const int64_t eo = cx.eoff_of[(size_t)xr.stack * 2 + xtrans];
            if (eo >= 0) {
                const double* row = E + eo + (int64_t)xr.row * (int64_t)G.keys.size();
                const M4& om = omats[oc];
                for (int e = 0; e < 16; ++e)
                    if (om.a[e] != 0.0) { const int col = G.col[(size_t)yid * 16 + e]; if (col >= 0) v += om.a[e] * row[col]; }
            }
        }
        v *= sign * inv_nrm2;
        if (n == 2) gamma[(size_t)(tgt[0] >> 1) * K1 + (tgt[1] >> 1)] += v;
        else {
            const int P = tgt[0], Q = tgt[1], R = tgt[2], S = tgt[3];
            add2(P, Q, R, S, v); add2(Q, P, R, S, -v); add2(P, Q, S, R, -v); add2(Q, P, S, R, v);
        }
    }
    // four-operator strings whose operators fall into the given spin-orbital ranges of (left, centre, right) and whose
    // part counts satisfy ok(cnt)
    template <class OK>
    void four(const int* lo, const int* hi, OK ok) {
        for (int pP = 0; pP < 3; ++pP) for (int pQ = pP; pQ < 3; ++pQ)
        for (int pS = 0; pS < 3; ++pS) for (int pR = pS; pR < 3; ++pR) {
            const int pr[4] = {pP, pQ, pS, pR};
            int cnt[3] = {0, 0, 0};
            for (int j = 0; j < 4; ++j) cnt[pr[j]]++;
            if (!ok(cnt)) continue;
            for (int P = lo[pP]; P < hi[pP]; ++P)
                for (int Q = std::max(lo[pQ], P + 1); Q < hi[pQ]; ++Q)
                    for (int S = lo[pS]; S < hi[pS]; ++S)
                        for (int R = std::max(lo[pR], S + 1); R < hi[pR]; ++R) {
                            if (spin_of(P) + spin_of(Q) != spin_of(R) + spin_of(S)) continue;
                            const OpTok ops[4] = {{P, 1}, {Q, 1}, {R, 0}, {S, 0}};
                            const int tgt[4] = {P, Q, R, S};
                            string(ops, 4, tgt);
                        }
        }
    }
    void left_rule() {                                        // c = s3 < kh
        const int c = cx.c;
        const int lo[3] = {0, 2 * c, 2 * c + 2}, hi[3] = {2 * c, 2 * c + 2, nso};
        four(lo, hi, [](const int* cnt) { return cnt[2] <= 1 && cnt[1] + cnt[2] >= 2; });
    }
    void right_rule(bool want2) {                             // c = s2 and s3 >= kh;  1-RDM strings at their smaller site
        const int c = cx.c;
        for (int P = 2 * c; P < nso; ++P)
            for (int S = 2 * c; S < nso; ++S) {
                if (std::min(P >> 1, S >> 1) != c || ((P ^ S) & 1)) continue;
                const OpTok ops[2] = {{P, 1}, {S, 0}};
                const int tgt[4] = {P, S, -1, -1};
                string(ops, 2, tgt);
            }
        if (!want2) return;
        if (c >= cx.kh) {
            const int lo[3] = {0, 2 * c, 2 * c + 2}, hi[3] = {2 * c, 2 * c + 2, nso};
            four(lo, hi, [](const int* cnt) { return cnt[0] <= 1 && cnt[0] + cnt[1] >= 2; });
        } else {                                              // s3 >= kh > c: exactly two operators on sites >= kh
            const int lo[3] = {0, 2 * c, 2 * cx.kh}, hi[3] = {2 * c, 2 * c + 2, nso};
            four(lo, hi, [](const int* cnt) { return cnt[0] <= 1 && cnt[2] == 2; });
        }
    }
};

void clone_site(const SiteTensor& src, const Basis& bl, const Basis& br, SiteTensor& dst, Engine& eng) {
    make_site_tensor(dst, bl, br);
    if (dst.nnz != src.nnz) throw std::logic_error("rdm: site tensor layout mismatch");
    if (dst.nnz)
        cuda_check(cudaMemcpyAsync(dst.data.p, src.data.p, (size_t)dst.nnz * 8, cudaMemcpyDeviceToDevice, eng.stream), "clone");
    dst.gauge = src.gauge;
}

// psi (centre, site c) = A . Rm per right sector (SVD: A = U, Rm = S Vt); next = Rm . B_{c+1}
void move_centre_right(const SiteTensor& psi, const Basis& bl, const Basis& br, const SiteTensor& bnext,
                       const Basis& br2, SiteTensor& A, SiteTensor& next, Engine& eng) {
    cudaStream_t st = eng.stream;
    make_site_tensor(A, bl, br);
    make_site_tensor(next, br, br2);
    if (A.nnz) cuda_check(cudaMemsetAsync(A.data.p, 0, (size_t)A.nnz * 8, st), "memset");
    if (next.nnz) cuda_check(cudaMemsetAsync(next.data.p, 0, (size_t)next.nnz * 8, st), "memset");
    std::vector<DevVec<double>> rms(br.size());
    GemmBatch gb;
    // sector SVDs concurrently: a few host threads, each with its own stream and cuSOLVER handle (psi is complete: the
    // previous step ended synchronised)
    cuda_check(cudaStreamSynchronize(st), "rdm centre move");
    const int nthreads = eng.host_threads;
    eng.ensure_svd_pool(nthreads);
    std::string err;
    int64_t nlaunch = 0;
#pragma omp parallel for schedule(dynamic, 1) num_threads(nthreads) reduction(+ : nlaunch)
    for (int r = 0; r < (int)br.size(); ++r) {
        try {
            const int tid = omp_get_thread_num();
            cudaStream_t ts = eng.svd_streams[tid];
            cuda_check(cudaSetDevice(eng.opt.device_id), "cudaSetDevice");
            std::vector<const SiteTensor::Blk*> rows;
            int mrows = 0;
            for (const auto& b : psi.blocks) if (b.r == r) { rows.push_back(&b); mrows += b.rows; }
            const int n = br[r].d;
            if (mrows < n) throw Error(-2, "rdm12: rank-deficient centre (bond sector wider than its left space)");
            DevVec<double> buf, U, S, Vt;
            buf.alloc((size_t)mrows * n); U.alloc((size_t)mrows * n); S.alloc((size_t)n); Vt.alloc((size_t)n * n);
            int off = 0;
            for (const auto* b : rows) {
                launch_copy2d(buf.p + (size_t)off * n, n, b->ptr, b->ld, b->rows, n, 1.0, nullptr, nullptr, ts);
                nlaunch++;
                off += b->rows;
            }
            svd_rowmajor(eng.svd_pool[tid], buf.p, mrows, n, U.p, S.p, Vt.p, ts);
            off = 0;
            for (const auto* b : rows) {
                const SiteTensor::Blk* ab = A.get(b->l, b->s);
                launch_copy2d(ab->ptr, ab->ld, U.p + (size_t)off * n, n, b->rows, n, 1.0, nullptr, nullptr, ts);
                nlaunch++;
                off += b->rows;
            }
            rms[r].alloc((size_t)n * n);
            launch_copy2d(rms[r].p, n, Vt.p, n, n, n, 1.0, S.p, nullptr, ts);
            nlaunch++;
            cuda_check(cudaStreamSynchronize(ts), "rdm centre move");      // buf / U / S / Vt die here
        } catch (const std::exception& e) {
#pragma omp critical
            err = e.what();
        }
    }
    if (!err.empty()) throw Error(-2, err);
    eng.launches += nlaunch;
    for (int r = 0; r < (int)br.size(); ++r) {
        const int n = br[r].d;
        for (int s = 0; s < 4; ++s) {
            const SiteTensor::Blk* nb = next.get(r, s);
            if (!nb) continue;
            const SiteTensor::Blk* ob = bnext.get(r, s);
            if (!ob) throw std::logic_error("rdm: next-site block missing");
            const int t = gb.add_task(nb->ptr, nb->ld, nb->rows, nb->cols, 0);
            gb.add_seg(t, rms[r].p, n, ob->ptr, ob->ld, n, 0, 1.0);
        }
    }
    run_once(gb, eng);
    A.gauge = 'L';
    next.gauge = 'C';
}

// psi (centre, site c) = Lm . B per left sector (SVD: Lm = U S, B = Vt); prev = A_{c-1} . Lm
void move_centre_left(const SiteTensor& psi, const Basis& bl, const Basis& br, const SiteTensor& aprev,
                      const Basis& bl0, SiteTensor& B, SiteTensor& prev, Engine& eng) {
    cudaStream_t st = eng.stream;
    make_site_tensor(B, bl, br);
    make_site_tensor(prev, bl0, bl);
    if (B.nnz) cuda_check(cudaMemsetAsync(B.data.p, 0, (size_t)B.nnz * 8, st), "memset");
    if (prev.nnz) cuda_check(cudaMemsetAsync(prev.data.p, 0, (size_t)prev.nnz * 8, st), "memset");
    std::vector<DevVec<double>> lms(bl.size());
    GemmBatch gb;
    cuda_check(cudaStreamSynchronize(st), "rdm centre move");
    const int nthreads = eng.host_threads;
    eng.ensure_svd_pool(nthreads);
    std::string err;
    int64_t nlaunch = 0;
#pragma omp parallel for schedule(dynamic, 1) num_threads(nthreads) reduction(+ : nlaunch)
    for (int l = 0; l < (int)bl.size(); ++l) {
        try {
            const int tid = omp_get_thread_num();
            cudaStream_t ts = eng.svd_streams[tid];
            cuda_check(cudaSetDevice(eng.opt.device_id), "cudaSetDevice");
            std::vector<const SiteTensor::Blk*> cols;
            int ncols = 0;
            for (const auto& b : psi.blocks) if (b.l == l) { cols.push_back(&b); ncols += b.cols; }
            const int m = bl[l].d;
            if (ncols < m) throw Error(-2, "rdm12: rank-deficient centre (bond sector wider than its right space)");
            DevVec<double> buf, U, S, Vt;
            buf.alloc((size_t)m * ncols); U.alloc((size_t)m * m); S.alloc((size_t)m); Vt.alloc((size_t)m * ncols);
            int off = 0;
            for (const auto* b : cols) {
                launch_copy2d(buf.p + off, ncols, b->ptr, b->ld, m, b->cols, 1.0, nullptr, nullptr, ts);
                nlaunch++;
                off += b->cols;
            }
            svd_rowmajor(eng.svd_pool[tid], buf.p, m, ncols, U.p, S.p, Vt.p, ts);
            off = 0;
            for (const auto* b : cols) {
                const SiteTensor::Blk* bb = B.get(b->l, b->s);
                launch_copy2d(bb->ptr, bb->ld, Vt.p + off, ncols, m, b->cols, 1.0, nullptr, nullptr, ts);
                nlaunch++;
                off += b->cols;
            }
            lms[l].alloc((size_t)m * pad2(m));
            launch_copy2d(lms[l].p, pad2(m), U.p, m, m, m, 1.0, nullptr, S.p, ts);   // Lm = U diag(S)
            nlaunch++;
            cuda_check(cudaStreamSynchronize(ts), "rdm centre move");      // buf / U / S / Vt die here
        } catch (const std::exception& e) {
#pragma omp critical
            err = e.what();
        }
    }
    if (!err.empty()) throw Error(-2, err);
    eng.launches += nlaunch;
    for (int l = 0; l < (int)bl.size(); ++l) {
        const int m = bl[l].d;
        for (const auto& ab : aprev.blocks) {
            if (ab.r != l) continue;
            const SiteTensor::Blk* pb = prev.get(ab.l, ab.s);
            if (!pb) throw std::logic_error("rdm: previous-site block missing");
            const int t = gb.add_task(pb->ptr, pb->ld, pb->rows, pb->cols, 0);
            gb.add_seg(t, ab.ptr, ab.ld, lms[l].p, pad2(m), m, 0, 1.0);
        }
    }
    run_once(gb, eng);
    B.gauge = 'R';
    prev.gauge = 'C';
}

// write the identity operator into the (0,0)-class storage of label K_I on block b
void add_identity(Block& b, Engine& eng) {
    b.allocate(std::vector<Label>{L0(K_I)}, false);
    const OpRef& ref = b.get(L0(K_I));
    const OpClass& c = b.classes[ref.cls];
    int dmax = 1;
    for (const Sector& s : b.basis) dmax = std::max(dmax, s.d);
    std::vector<double> ones((size_t)dmax, 1.0);
    DevVec<double> d1;
    d1.upload(ones, eng.stream);
    for (int i = 0; i < (int)b.basis.size(); ++i) {
        const int d = b.basis[i].d, ld = pad2(d);
        cuda_check(cudaMemcpy2DAsync(ref.ptr + c.off[i], (size_t)(ld + 1) * 8, d1.p, 8, 8, d, cudaMemcpyDeviceToDevice,
                                     eng.stream), "identity");
    }
    cuda_check(cudaStreamSynchronize(eng.stream), "identity");
}

}  // namespace

void rdm12(Engine& eng, double* gamma, double* Gamma) {
    const double t_begin = now_s();
    const int k = eng.k;
    const int kh = (eng.opt.rdm_split >= 0 && eng.opt.rdm_split <= k) ? eng.opt.rdm_split : k / 2;   // partition point of the two rules
    const bool want2 = Gamma != nullptr;
    MPS& mps = eng.mps;
    for (int p = 1; p < k; ++p)
        if (mps.sites[p].gauge != 'R')
            throw Error(-2, "rdm12: the MPS must be right-canonical with its centre on site 0 (as imported or as left by dmrg_sweep)");
    eng.rdm_bytes = 0; eng.rdm_flops = 0; eng.rdm_stream_ms = 0; eng.rdm_gemm_ms = 0; eng.rdm_host_seconds = 0;
    eng.rdm_grow_seconds = 0; eng.rdm_stream_bytes = 0;
    Evaluator ev(eng);
    ev.arena.init((size_t)std::min<int64_t>(eng.t_capacity(), (int64_t)1 << 29));   // at most 4 GiB of intermediates at a time
    std::memset(gamma, 0, sizeof(double) * (size_t)k * k);
    if (want2) std::memset(Gamma, 0, sizeof(double) * (size_t)k * k * k * k);
    const int NOPAIR = 0;                                     // pair range [0, 0): one-index operators only

    // ---- right one-index blocks R_b (sites >= b) for the left-rule centres c = b - 1 < kh --------------------------------
    double tg = now_s();
    std::vector<std::unique_ptr<Block>> R1(k + 1);
    if (want2 && kh > 0) {
        R1[k].reset(new Block('R', k, k, mps.bonds[k], 'N'));
        for (int b = k; b >= 2; --b) {
            R1[b - 1] = grow_normal(*R1[b], eng.ham, mps.bonds[b - 1], mps.sites[b - 1], NOPAIR, NOPAIR, eng);
            if (b > kh) R1[b].reset();                        // centres c = b - 1 >= kh belong to the right-rule pass
        }
    }
    eng.rdm_grow_seconds += now_s() - tg;

    // ---- centre moving right: left-rule strings at c < kh; keep A_c and the left one-index blocks for the way back --------
    std::vector<std::unique_ptr<Block>> L1(k);                // L1[c]: sites < c, a+_P only
    std::vector<SiteTensor> Astore(k);
    L1[0].reset(new Block('L', 0, k, mps.bonds[0], 'N'));
    std::unique_ptr<Block> L2;                                // sites < c with 1, a+_P, A, B (pairs of sites < kh)
    if (want2 && kh > 0) { L2.reset(new Block('L', 0, k, mps.bonds[0], 'N')); add_identity(*L2, eng); }
    SiteTensor centre;
    clone_site(mps.sites[0], mps.bonds[0], mps.bonds[1], centre, eng);
    DevVec<double> scal;
    scal.alloc(1);
    launch_multi_dot(centre.data.p, centre.data.p, centre.nnz, 1, centre.nnz, scal.p, eng.red_scratch.p, eng.stream);
    eng.launches += 2;
    double nrm2 = 0.0;
    cuda_check(cudaMemcpyAsync(&nrm2, scal.p, 8, cudaMemcpyDeviceToHost, eng.stream), "norm");
    cuda_check(cudaStreamSynchronize(eng.stream), "norm");
    if (!(nrm2 > 0.0)) throw Error(-2, "rdm12: the MPS has zero norm");

    auto run_centre = [&](int c, bool stack_left, Block& XB, Block& YB, const SiteTensor& psi) {
        Centre cx;
        cx.c = c; cx.k = k; cx.kh = kh; cx.stack_left = stack_left; cx.XB = &XB; cx.YB = &YB; cx.psi = &psi;
        double th = now_s();
        build_tables(cx);
        eng.rdm_host_seconds += now_s() - th;
        ev.evaluate(cx);
        th = now_s();
        Scatter sc(cx, ev.Ehost, nrm2, gamma, Gamma);
        if (stack_left) sc.left_rule(); else sc.right_rule(want2);
        eng.rdm_host_seconds += now_s() - th;
    };

    for (int c = 0; c < k; ++c) {
        if (want2 && c < kh) run_centre(c, true, *L2, *R1[c + 1], centre);
        if (c == k - 1) break;
        tg = now_s();
        SiteTensor next;
        move_centre_right(centre, mps.bonds[c], mps.bonds[c + 1], mps.sites[c + 1], mps.bonds[c + 2], Astore[c], next, eng);
        L1[c + 1] = grow_normal(*L1[c], eng.ham, mps.bonds[c + 1], Astore[c], NOPAIR, NOPAIR, eng);
        if (L2) {
            if (c + 1 < kh) {
                std::unique_ptr<Block> Ln = grow_normal(*L2, eng.ham, mps.bonds[c + 1], Astore[c], 0, kh, eng);
                add_identity(*Ln, eng);
                L2 = std::move(Ln);
            } else L2.reset();
        }
        if (c + 1 < (int)R1.size()) R1[c + 1].reset();
        centre = std::move(next);
        eng.rdm_grow_seconds += now_s() - tg;
    }
    R1.clear();

    // ---- centre moving left: right-rule strings (and the 1-RDM) at every c ----------------------------------------------------
    std::unique_ptr<Block> R2(new Block('R', k, k, mps.bonds[k], 'N'));
    add_identity(*R2, eng);
    for (int c = k - 1; c >= 0; --c) {
        run_centre(c, false, *R2, *L1[c], centre);
        if (c == 0) break;
        tg = now_s();
        SiteTensor Bc, prev;
        move_centre_left(centre, mps.bonds[c], mps.bonds[c + 1], Astore[c - 1], mps.bonds[c - 1], Bc, prev, eng);
        std::unique_ptr<Block> Rn = want2 ? grow_normal(*R2, eng.ham, mps.bonds[c], Bc, kh, k, eng)
                                          : grow_normal(*R2, eng.ham, mps.bonds[c], Bc, NOPAIR, NOPAIR, eng);
        add_identity(*Rn, eng);
        R2 = std::move(Rn);
        L1[c].reset();
        Astore[c - 1] = SiteTensor();
        centre = std::move(prev);
        eng.rdm_grow_seconds += now_s() - tg;
    }
    eng.rdm_seconds = now_s() - t_begin;
}

}  // namespace dmrg
