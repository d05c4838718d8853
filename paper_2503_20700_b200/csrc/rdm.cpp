// 1- and 2-particle reduced density matrices of the current MPS.
//   gamma_pq = <E_pq>                                  PAPER.md:91 (Eq. 9)
//   Gamma_pqrs = <sum_ss' a+_ps a+_rs' a_ss' a_qs>     PAPER.md:93 (Eq. 10) under readings S1/S2
// A dedicated pass moves a one-site centre c = 0..k-1 through the chain.  Left blocks carry the renormalised NORMAL
// operators 1, a+_P, A_PQ = a+_P a+_Q, B_PS = a+_P a_S of the sites < c (grown by the fused blocking kernels), right
// blocks carry 1 and a+_P of the sites > c.  Every spin-orbital element <a+_P a+_Q a_R a_S> (P<Q, S<R) is evaluated
// once, at the centre c = second largest of its four sites (two-operator strings: at the larger site), as
//   <psi_c| X_L (x) o_c (x) Y_R |psi_c> = sum_{s',s} o[s',s]  < X , M_{Y,s',s} >,
//   M_{Y,s',s}[l',l] = sgn sum_{r',r} psi[(l',s')][:,r'] Y[r',r] psi[(l,s)][:,r]       (grouped FP64 GEMMs)
// and the contraction < X, M > of EVERY stored left operator X with every M of its quantum-number class is one
// tall-skinny product  E = Stack [n_ops x nnz] . M^T [nnz x n_M]  that streams each stored operator exactly once per
// centre (the HBM-bound accumulation of row a6), split over K with a fixed-order reduction (no atomics).
#include <algorithm>
#include <chrono>
#include <cmath>
#include <cstring>

#include "core.hpp"

namespace dmrg {

namespace {

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

// one string evaluated at a centre: value = coef * sum_{so,si} o[so,si] E[stack][row, col(cls, trans, yid, so, si)]
struct Rec {
    int stack, row, trans, yid;     // left factor (stack, row of the L block), right factor id
    int ocode;                      // index into the table of centre matrices
    double coef;
    int tgt[4];                     // spin orbitals (P, Q, R, S) or (P, S, -1, -1)
};

struct ColGroup {                   // all M vectors of one (class, trans)
    int cls, trans;
    std::vector<uint32_t> keys;     // (yid << 8) | (so << 4) | si, in column order
    std::unordered_map<uint32_t, int> index;
    int col(uint32_t key) {
        auto it = index.find(key);
        if (it != index.end()) return it->second;
        const int c = (int)keys.size();
        keys.push_back(key); index.emplace(key, c);
        return c;
    }
};

}  // namespace

}  // namespace dmrg

namespace dmrg {

static void clone_site(const SiteTensor& src, const Basis& bl, const Basis& br, SiteTensor& dst, Engine& eng) {
    make_site_tensor(dst, bl, br);
    if (dst.nnz != src.nnz) throw std::logic_error("rdm: site tensor layout mismatch");
    if (dst.nnz)
        cuda_check(cudaMemcpyAsync(dst.data.p, src.data.p, (size_t)dst.nnz * 8, cudaMemcpyDeviceToDevice, eng.stream), "clone");
    dst.gauge = src.gauge;
}

// psi (centre, site c) = A . Rm per right sector (SVD: A = U, Rm = S Vt); next = Rm . B_{c+1}
static void move_centre_right(const SiteTensor& psi, const Basis& bl, const Basis& br, const SiteTensor& bnext,
                              const Basis& br2, SiteTensor& A, SiteTensor& next, Engine& eng) {
    cudaStream_t st = eng.stream;
    make_site_tensor(A, bl, br);
    make_site_tensor(next, br, br2);
    if (A.nnz) cuda_check(cudaMemsetAsync(A.data.p, 0, (size_t)A.nnz * 8, st), "memset");
    if (next.nnz) cuda_check(cudaMemsetAsync(next.data.p, 0, (size_t)next.nnz * 8, st), "memset");
    std::vector<DevVec<double>> rms(br.size());
    GemmBatch gb;
    for (int r = 0; r < (int)br.size(); ++r) {
        std::vector<const SiteTensor::Blk*> rows;
        int mrows = 0;
        for (const auto& b : psi.blocks) if (b.r == r) { rows.push_back(&b); mrows += b.rows; }
        const int n = br[r].d;
        if (mrows < n) throw Error(-2, "rdm12: rank-deficient centre (bond sector wider than its left space)");
        DevVec<double> buf, U, S, Vt;
        buf.alloc((size_t)mrows * n); U.alloc((size_t)mrows * n); S.alloc((size_t)n); Vt.alloc((size_t)n * n);
        int off = 0;
        for (const auto* b : rows) {
            launch_copy2d(buf.p + (size_t)off * n, n, b->ptr, b->ld, b->rows, n, 1.0, nullptr, nullptr, st);
            eng.launches++;
            off += b->rows;
        }
        svd_rowmajor(eng.svd, buf.p, mrows, n, U.p, S.p, Vt.p, st);
        off = 0;
        for (const auto* b : rows) {
            const SiteTensor::Blk* ab = A.get(b->l, b->s);
            launch_copy2d(ab->ptr, ab->ld, U.p + (size_t)off * n, n, b->rows, n, 1.0, nullptr, nullptr, st);
            eng.launches++;
            off += b->rows;
        }
        rms[r].alloc((size_t)n * n);
        launch_copy2d(rms[r].p, n, Vt.p, n, n, n, 1.0, S.p, nullptr, st);
        eng.launches++;
        cuda_check(cudaStreamSynchronize(st), "rdm centre move");      // buf / U / S / Vt die here
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

// write the identity operator into the (0,0)-class storage of label K_I on block b
static void add_identity(Block& b, Engine& eng) {
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

}  // namespace dmrg

namespace dmrg {

namespace {

struct CentreCtx {
    int c, k;
    Block* L;
    Block* R;
    const SiteTensor* psi;
    std::vector<Rec> recs;
    std::vector<ColGroup> groups;
    std::map<std::pair<int, int>, int> group_of;          // (cls, trans) -> index into groups
    std::vector<M4> omats;
    std::unordered_map<uint32_t, int> ocode_of;
    int part(int P) const { const int s = P >> 1; return s < c ? 0 : (s == c ? 1 : 2); }
    int group(int cls, int trans) {
        auto key = std::make_pair(cls, trans);
        auto it = group_of.find(key);
        if (it != group_of.end()) return it->second;
        groups.emplace_back();
        groups.back().cls = cls; groups.back().trans = trans;
        group_of[key] = (int)groups.size() - 1;
        return (int)groups.size() - 1;
    }
    // register the string  prod ops  (creators first), already known to conserve N and 2Sz
    void add_string(const OpTok* ops, int n, const int* tgt) {
        int order[4], prt[4];
        for (int j = 0; j < n; ++j) { order[j] = j; prt[j] = part(ops[j].P); }
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
        if (nl > 2 || nr > 1) throw std::logic_error("rdm: string does not belong to this centre");
        Label xl = L0(K_I);
        int xtrans = 0;
        if (nl == 1) { xl = L1(K_C, lo[0].P); xtrans = lo[0].dag ? 0 : 1; }
        else if (nl == 2) {
            const int X = lo[0].P, Y = lo[1].P;
            if (lo[0].dag && lo[1].dag) { if (X < Y) xl = L2(K_A, X, Y); else { xl = L2(K_A, Y, X); sign = -sign; } }
            else if (!lo[0].dag && !lo[1].dag) {              // a_X a_Y = (a+_Y a+_X)^T
                xtrans = 1;
                if (Y < X) xl = L2(K_A, Y, X); else { xl = L2(K_A, X, Y); sign = -sign; }
            } else if (lo[0].dag && !lo[1].dag) xl = L2(K_B, X, Y);
            else throw std::logic_error("rdm: annihilator before creator inside the left block");
        }
        const OpRef& xr = L->get(xl);
        uint32_t code = (uint32_t)nc;
        M4 om = m4_eye();
        for (int j = 0; j < nc; ++j) {
            code = code * 4 + (uint32_t)((co[j].P & 1) * 2 + co[j].dag);
            om = m4_mul(om, m4_site(co[j].P & 1, co[j].dag));
        }
        auto oc = ocode_of.find(code);
        if (oc == ocode_of.end()) { omats.push_back(om); oc = ocode_of.emplace(code, (int)omats.size() - 1).first; }
        Rec r;
        r.stack = xr.stack; r.row = xr.row; r.trans = xtrans;
        r.yid = nr ? 1 + 2 * ro[0].P + ro[0].dag : 0;
        r.ocode = oc->second; r.coef = sign;
        for (int j = 0; j < 4; ++j) r.tgt[j] = tgt[j];
        ColGroup& g = groups[group(xr.cls, xtrans)];
        for (int e = 0; e < 16; ++e)
            if (om.a[e] != 0.0) g.col(((uint32_t)r.yid << 8) | (uint32_t)e);
        recs.push_back(r);
    }
};

void enumerate_strings(CentreCtx& cx, bool want2) {
    const int c = cx.c, nso = 2 * cx.k;
    const int lo[3] = {0, 2 * c, 2 * c + 2}, hi[3] = {2 * c, 2 * c + 2, nso};
    for (int P = 0; P < hi[1]; ++P)                          // a+_P a_S evaluated at the larger of the two sites
        for (int S = 0; S < hi[1]; ++S) {
            if (std::max(P >> 1, S >> 1) != c || ((P ^ S) & 1)) continue;
            const OpTok ops[2] = {{P, 1}, {S, 0}};
            const int tgt[4] = {P, S, -1, -1};
            cx.add_string(ops, 2, tgt);
        }
    if (!want2) return;
    for (int pP = 0; pP < 3; ++pP) for (int pQ = pP; pQ < 3; ++pQ)
    for (int pS = 0; pS < 3; ++pS) for (int pR = pS; pR < 3; ++pR) {
        const int pr[4] = {pP, pQ, pS, pR};
        int cnt[3] = {0, 0, 0};
        for (int j = 0; j < 4; ++j) cnt[pr[j]]++;
        if (cnt[2] > 1 || cnt[1] + cnt[2] < 2) continue;     // centre = second largest site of the string
        for (int P = lo[pP]; P < hi[pP]; ++P)
            for (int Q = std::max(lo[pQ], P + 1); Q < hi[pQ]; ++Q)
                for (int S = lo[pS]; S < hi[pS]; ++S)
                    for (int R = std::max(lo[pR], S + 1); R < hi[pR]; ++R) {
                        if (spin_of(P) + spin_of(Q) != spin_of(R) + spin_of(S)) continue;
                        const OpTok ops[4] = {{P, 1}, {Q, 1}, {R, 0}, {S, 0}};
                        const int tgt[4] = {P, Q, R, S};
                        cx.add_string(ops, 4, tgt);
                    }
    }
}

}  // namespace

}  // namespace dmrg

namespace dmrg {

namespace {

// Bump allocator over one device allocation made per dmrg_rdm12 call: the pass needs thousands of short-lived
// intermediates per centre, and a cudaMalloc / cudaFree pair each (the free synchronises the device) dominated its time.
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
Arena g_arena;

// E[stack][row * ncol + col] for every stack referenced by the records of each group
struct GroupResult { std::map<int, std::vector<double>> E; int ncol = 0; };

void evaluate_group(CentreCtx& cx, ColGroup& g, const std::vector<int>& stacks, GroupResult& out, Engine& eng) {
    Block& L = *cx.L;
    Block& R = *cx.R;
    const SiteTensor& psi = *cx.psi;
    const OpClass& cls = L.classes[g.cls];
    const int ncol = (int)g.keys.size();
    out.ncol = ncol;
    for (int s : stacks) out.E[s].assign((size_t)L.stacks[s].members.size() * ncol, 0.0);
    if (cls.nnz == 0 || ncol == 0) return;
    const int64_t ld = cls.ld;
    const int64_t cap = (int64_t)g_arena.buf.n;
    int chunk_cols = (int)std::max<int64_t>(1, std::min<int64_t>(ncol, (cap / 2) / ld));
    for (int c0 = 0; c0 < ncol; c0 += chunk_cols) {
        const int nc = std::min(chunk_cols, ncol - c0);
        g_arena.reset();
        struct { double* p; } Mbuf;
        Mbuf.p = g_arena.get((size_t)nc * ld);
        cuda_check(cudaMemsetAsync(Mbuf.p, 0, (size_t)nc * ld * 8, eng.stream), "memset");
        // ---- phase 1: T[(Y, l, si)] = psi[(l,si)] Y^T ; phase 2: M blocks ------------------------------------------------
        GemmBatch p1, p2;
        std::unordered_map<uint64_t, std::pair<double*, int>> tcache;       // (yid, l, si) -> (T, ld)
        for (int cc = 0; cc < nc; ++cc) {
            const uint32_t key = g.keys[c0 + cc];
            const int yid = (int)(key >> 8);
            const int s_out = (int)((key & 255) >> 2), s_in = (int)(key & 3);   // key & 255 = s_out * 4 + s_in
            const OpRef* yref = nullptr;
            bool ytrans = false;
            if (yid) { const int P = (yid - 1) >> 1, dag = (yid - 1) & 1; yref = &R.get(L1(K_C, P)); ytrans = !dag; }
            const int par_y = yid ? 1 : 0, par_o = (SITE_QN[s_out] - SITE_QN[s_in]) & 1;
            double* mcol = Mbuf.p + (size_t)cc * ld;
            for (int a = 0; a < (int)L.basis.size(); ++a) {
                const int b = cls.out[a];
                if (b < 0) continue;
                const int l = g.trans ? b : a, lp = g.trans ? a : b;       // ket sector l, bra sector l'
                const SiteTensor::Blk* kb = psi.get(l, s_in);
                const SiteTensor::Blk* bb = psi.get(lp, s_out);
                if (!kb || !bb) continue;
                const double* tptr = kb->ptr;
                int tld = kb->ld;
                if (yref) {
                    OpBlockView v;
                    if (!op_block(R, *yref, ytrans, kb->r, v) || v.out != bb->r) continue;
                    const uint64_t tk = ((uint64_t)yid << 24) | ((uint64_t)l << 4) | (uint64_t)s_in;
                    auto it = tcache.find(tk);
                    if (it == tcache.end()) {
                        const int dro = R.basis[v.out].d;
                        double* tp = g_arena.get((size_t)kb->rows * pad2(dro));
                        const int t1 = p1.add_task(tp, pad2(dro), kb->rows, dro, 0);
                        p1.add_seg(t1, kb->ptr, kb->ld, v.ptr, v.ld, kb->cols, v.trans ? 0 : SEG_TRANS_B, 1.0);
                        it = tcache.emplace(tk, std::make_pair(tp, pad2(dro))).first;
                    }
                    tptr = it->second.first; tld = it->second.second;
                } else if (kb->r != bb->r) continue;
                const int nl = L.basis[l].n;
                const double sgn = ((par_y * (nl + SITE_QN[s_in]) + par_o * nl) & 1) ? -1.0 : 1.0;
                const int db = L.basis[b].d, da = L.basis[a].d, K = bb->cols;
                const int t2 = p2.add_task(mcol + cls.off[a], pad2(da), db, da, 0);
                if (!g.trans) p2.add_seg(t2, bb->ptr, bb->ld, tptr, tld, K, SEG_TRANS_B, sgn);     // psi' T^T
                else          p2.add_seg(t2, tptr, tld, bb->ptr, bb->ld, K, SEG_TRANS_B, sgn);     // T psi'^T
            }
        }
        eng.rdm_flops += p1.flops + p2.flops;
        run_once(p1, eng);
        run_once(p2, eng);
        // ---- E = Stack . M^T, split over K with a fixed-order reduction -------------------------------------------------
        for (int s : stacks) {
            const Stack& stk = L.stacks[s];
            const int nrows = (int)stk.members.size();
            const int tiles = ((nrows + GEMM_BM - 1) / GEMM_BM) * ((nc + GEMM_BN - 1) / GEMM_BN);
            int nsplit = (int)std::max<int64_t>(1, std::min<int64_t>((592 + tiles - 1) / tiles, (ld + 2047) / 2048));
            int64_t kc = (ld + nsplit - 1) / nsplit;
            kc = (kc + 15) & ~(int64_t)15;
            nsplit = (int)((ld + kc - 1) / kc);
            struct { double* p; } part, Ed;
            part.p = nullptr;
            const size_t arena_mark = g_arena.used;
            Ed.p = g_arena.get((size_t)nrows * nc);
            if (nc <= 8) {
                // few right-hand sides: the HBM-bound streaming kernel (coalesced 16-byte loads of every stored operator,
                // warp-level reductions, fixed-order partial sums) instead of the tensor-pipe GEMM
                double* scratch = g_arena.get((size_t)stack_dots_scratch(nrows, nc, ld));
                cudaEvent_t e0, e1;
                cuda_check(cudaEventCreate(&e0), "event");
                cuda_check(cudaEventCreate(&e1), "event");
                cudaEventRecord(e0, eng.stream);
                launch_stack_dots(stk.base, ld, nrows, Mbuf.p, ld, nc, ld, Ed.p, nc, scratch, eng.stream);
                cudaEventRecord(e1, eng.stream);
                eng.launches += 2;
                eng.rdm_flops += 2.0 * nrows * (double)nc * (double)ld;
                eng.rdm_bytes += 8.0 * ((double)nrows * ld + (double)nc * ld);
                std::vector<double>& E = out.E[s];
                cuda_check(cudaMemcpy2DAsync(E.data() + c0, (size_t)ncol * 8, Ed.p, (size_t)nc * 8, (size_t)nc * 8, nrows,
                                             cudaMemcpyDeviceToHost, eng.stream), "E download");
                cuda_check(cudaStreamSynchronize(eng.stream), "E download");
                float ms = 0.f;
                cudaEventElapsedTime(&ms, e0, e1);
                eng.rdm_stream_ms += ms;
                cudaEventDestroy(e0);
                cudaEventDestroy(e1);
                g_arena.used = arena_mark;
                continue;
            }
            GemmBatch gb, red;
            if (nsplit == 1) {
                const int t = gb.add_task(Ed.p, nc, nrows, nc, 0);
                gb.add_seg(t, stk.base, (int)ld, Mbuf.p, (int)ld, (int)ld, SEG_TRANS_B, 1.0);
            } else {
                part.p = g_arena.get((size_t)nsplit * nrows * nc);
                const int tr = red.add_task(Ed.p, nc, nrows, nc, 0);
                for (int p = 0; p < nsplit; ++p) {
                    const int64_t k0 = (int64_t)p * kc, kk = std::min<int64_t>(kc, ld - k0);
                    double* pp = part.p + (size_t)p * nrows * nc;
                    const int t = gb.add_task(pp, nc, nrows, nc, 0);
                    gb.add_seg(t, stk.base + k0, (int)ld, Mbuf.p + k0, (int)ld, (int)kk, SEG_TRANS_B, 1.0);
                    red.add_seg(tr, pp, nc, nullptr, 0, 0, SEG_IDENT_B, 1.0);
                }
            }
            eng.rdm_flops += gb.flops;
            eng.rdm_bytes += 8.0 * ((double)nrows * ld + (double)nc * ld);
            eng.rdm_stream_ms += run_once_ms(gb, eng);
            run_once(red, eng);
            std::vector<double>& E = out.E[s];
            cuda_check(cudaMemcpy2DAsync(E.data() + c0, (size_t)ncol * 8, Ed.p, (size_t)nc * 8, (size_t)nc * 8, nrows,
                                         cudaMemcpyDeviceToHost, eng.stream), "E download");
            cuda_check(cudaStreamSynchronize(eng.stream), "E download");
            g_arena.used = arena_mark;                         // Ed / part of this stack are dead
        }
    }
}

}  // namespace

}  // namespace dmrg

namespace dmrg {

void rdm12(Engine& eng, double* gamma, double* Gamma) {
    const auto t0 = std::chrono::steady_clock::now();
    const int k = eng.k;
    const bool want2 = Gamma != nullptr;
    MPS& mps = eng.mps;
    for (int p = 1; p < k; ++p)
        if (mps.sites[p].gauge != 'R')
            throw Error(-2, "rdm12: the MPS must be right-canonical with its centre on site 0 (as imported or as left by dmrg_sweep)");
    eng.rdm_bytes = 0; eng.rdm_flops = 0; eng.rdm_stream_ms = 0;
    g_arena.init((size_t)std::min<int64_t>(eng.t_capacity(), (int64_t)1 << 29));   // at most 4 GiB of intermediates at a time
    struct ArenaRelease { ~ArenaRelease() { g_arena.overflow.clear(); g_arena.buf.release(); } } arena_release;
    std::memset(gamma, 0, sizeof(double) * (size_t)k * k);
    if (want2) std::memset(Gamma, 0, sizeof(double) * (size_t)k * k * k * k);
    // right blocks with the one-index operators of the sites > c
    std::vector<std::unique_ptr<Block>> Rn(k + 1);
    Rn[k].reset(new Block('R', k, k, mps.bonds[k], 'N'));
    for (int b = k; b >= 2; --b) Rn[b - 1] = grow_normal(*Rn[b], eng.ham, mps.bonds[b - 1], mps.sites[b - 1], false, eng);
    std::unique_ptr<Block> Lb(new Block('L', 0, k, mps.bonds[0], 'N'));
    add_identity(*Lb, eng);
    SiteTensor centre;
    clone_site(mps.sites[0], mps.bonds[0], mps.bonds[1], centre, eng);
    DevVec<double> scal;
    scal.alloc(1);
    launch_multi_dot(centre.data.p, centre.data.p, centre.nnz, 1, centre.nnz, scal.p, eng.stream);
    eng.launches += 2;
    double nrm2 = 0.0;
    cuda_check(cudaMemcpyAsync(&nrm2, scal.p, 8, cudaMemcpyDeviceToHost, eng.stream), "norm");
    cuda_check(cudaStreamSynchronize(eng.stream), "norm");
    if (!(nrm2 > 0.0)) throw Error(-2, "rdm12: the MPS has zero norm");
    const size_t K1 = (size_t)k;
    auto add2 = [&](int A, int B, int C, int D, double v) {           // Gamma^so_ABCD = <a+_A a+_B a_C a_D>
        if (spin_of(A) != spin_of(D) || spin_of(B) != spin_of(C)) return;
        Gamma[((((size_t)(A >> 1)) * K1 + (D >> 1)) * K1 + (B >> 1)) * K1 + (C >> 1)] += v;
    };
    for (int c = 0; c < k; ++c) {
        CentreCtx cx;
        cx.c = c; cx.k = k; cx.L = Lb.get(); cx.R = Rn[c + 1].get(); cx.psi = &centre;
        enumerate_strings(cx, want2);
        std::vector<std::vector<int>> stacks(cx.groups.size());
        for (const Rec& r : cx.recs) {
            std::vector<int>& v = stacks[cx.group(cx.L->stacks[r.stack].cls, r.trans)];
            if (std::find(v.begin(), v.end(), r.stack) == v.end()) v.push_back(r.stack);
        }
        std::vector<GroupResult> res(cx.groups.size());
        for (size_t g = 0; g < cx.groups.size(); ++g) evaluate_group(cx, cx.groups[g], stacks[g], res[g], eng);
        for (const Rec& r : cx.recs) {
            const int gi = cx.group(cx.L->stacks[r.stack].cls, r.trans);
            const ColGroup& g = cx.groups[gi];
            const std::vector<double>& E = res[gi].E.at(r.stack);
            const M4& om = cx.omats[r.ocode];
            double v = 0.0;
            for (int e = 0; e < 16; ++e)
                if (om.a[e] != 0.0) v += om.a[e] * E[(size_t)r.row * res[gi].ncol + g.index.at(((uint32_t)r.yid << 8) | (uint32_t)e)];
            v *= r.coef / nrm2;
            if (r.tgt[2] < 0) gamma[(size_t)(r.tgt[0] >> 1) * K1 + (r.tgt[1] >> 1)] += v;
            else {
                const int P = r.tgt[0], Q = r.tgt[1], R = r.tgt[2], S = r.tgt[3];
                add2(P, Q, R, S, v); add2(Q, P, R, S, -v); add2(P, Q, S, R, -v); add2(Q, P, S, R, v);
            }
        }
        if (c < k - 1) {
            SiteTensor A, next;
            move_centre_right(centre, mps.bonds[c], mps.bonds[c + 1], mps.sites[c + 1], mps.bonds[c + 2], A, next, eng);
            std::unique_ptr<Block> Ln = grow_normal(*Lb, eng.ham, mps.bonds[c + 1], A, want2, eng);
            add_identity(*Ln, eng);
            Lb = std::move(Ln);
            centre = std::move(next);
        }
    }
    eng.rdm_seconds = std::chrono::duration<double>(std::chrono::steady_clock::now() - t0).count();
}

}  // namespace dmrg
