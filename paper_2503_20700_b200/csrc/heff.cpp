// H_eff at a two-site bond: term list from the bipartition identity, block maps, and the two-phase grouped-GEMM plan
// (DESIGN.md "Algorithm" step 5 and "Kernels").
//
//   y[l', a'b', r'] = sum_t c_t sgn  O_L^t[l' <- l]  x[l, ab, r]  (O_R^t[r' <- r])^T  dm^t[a'b', ab]
//
// Phase 1 computes each distinct intermediate once: T = O_L X (shared by every term with that left factor and input
// block) or T = X O_R^T, whichever order needs fewer flops for the (term, block) pair.  Phase 2 gives every output
// block to one task that sums its contributions  Y += c T O_R^T  /  Y += c O_L T  as one K-concatenated GEMM: no
// atomics, fixed summation order.  Terms are processed in chunks bounded by the intermediate buffer.
//
// The descriptors (which triples contribute, signs, intermediates, segment lists, tiles, diagonal items, accounting)
// are enumerated on the device by heff_maps.cu from small uploaded tables (build_maps_device below); the host loop in
// build_heff is the reference builder kept for A/B tests (DMRG_B200_HOST_MAPS=1).  heff_apply runs the chunks as a
// two-stream pipeline with double-buffered intermediates and split-K partial sums.
#include <algorithm>
#include <cassert>
#include <cstdlib>

#include "core.hpp"
#include "maps.hpp"

namespace dmrg {

void psi_layout(const Basis& bl, const Basis& br, std::vector<PsiBlock>& layout, std::vector<int>& lookup,
                int64_t& nnz) {
    layout.clear();
    lookup.assign(bl.size() * 16, -1);
    nnz = 0;
    for (int l = 0; l < (int)bl.size(); ++l)
        for (int ab = 0; ab < 16; ++ab) {
            const int a = ab >> 2, b = ab & 3;
            const int r = find_sector(br, bl[l].n + SITE_QN[a] + SITE_QN[b], bl[l].s + SITE_QS[a] + SITE_QS[b]);
            if (r < 0) continue;
            lookup[l * 16 + ab] = (int)layout.size();
            layout.push_back({l, ab, r, bl[l].d, br[r].d, nnz, 0});
            nnz += (int64_t)bl[l].d * br[r].d;
        }
}

static std::vector<NTerm> heff_terms(const Ham& ham, Block& LB, Block& RB, const Dot& dot, Block*& Xout, Engine& eng) {
    Block* X = (LB.mode == 'N') ? &LB : &RB;
    Block* Y = (X == &LB) ? &RB : &LB;
    if (X->mode != 'N') throw std::logic_error("heff: neither block carries normal operators");
    if (!Y->inside().empty() && Y->mode != 'C') throw std::logic_error("heff: both blocks carry normal operators");
    Xout = X;
    const std::vector<int> Yin = Y->inside();
    make_temps(ham, *X, dot, Yin, eng);
    Gen gen(ham, block_info(*X), dot);
    auto yf = [&](const Label& l, bool tr) {
        Factor f; f.type = 0; f.side = Y->side; f.label = l; f.trans = tr;
        return f;
    };
    std::vector<int> A = X->inside();
    A.insert(A.end(), dot.so.begin(), dot.so.end());
    std::sort(A.begin(), A.end());
    // The term list in its fixed order: H_A, H_Y, G, G^+, B Q with G = a+_P^A S_P^Y, a+_P^Y S_P^A, A_PQ^A P_PQ^Y.  Each
    // entry of `jobs` yields a few terms; the host threads generate and normalise them (16 x 16 dot-matrix products per
    // term), the results are concatenated in job order, so the list does not depend on the number of threads.
    struct Job { int kind, a, b; };                            // 0: H_A, 1: H_Y, 2: cre(a) St_a^Y, 3: C_a^Y S(a), 4: A(a,b) Pt^Y, 5: B(a,b) Q^Y
    std::vector<Job> jobs;
    jobs.push_back({0, 0, 0});
    if (!Yin.empty()) {
        jobs.push_back({1, 0, 0});
        for (int P : A) jobs.push_back({2, P, 0});
        for (int P : Yin) jobs.push_back({3, P, 0});
        for (size_t a = 0; a < A.size(); ++a)
            for (size_t b = a + 1; b < A.size(); ++b) jobs.push_back({4, A[a], A[b]});
        for (int P : A)
            for (int S : A) jobs.push_back({5, P, S});
    }
    std::vector<std::vector<NTerm>> fwd(jobs.size()), adj(jobs.size());
    std::string err;
#pragma omp parallel for schedule(dynamic, 16) if (jobs.size() > 256)
    for (long j = 0; j < (long)jobs.size(); ++j) {
        try {
            const Job& jb = jobs[j];
            Expr e;
            bool hc = false;
            switch (jb.kind) {
                case 0: e = gen.H(); break;
                case 1: { Term t; t.f.push_back(yf(L0(K_H), false)); e.push_back(t); break; }
                case 2: for (Term t : gen.cre(jb.a)) { t.f.push_back(yf(L1(K_St, jb.a), true)); e.push_back(t); } hc = true; break;
                case 3:
                    for (const Term& sT : gen.S(jb.a)) {
                        Term t; t.coef = sT.coef; t.f.push_back(yf(L1(K_C, jb.a), false));
                        t.f.insert(t.f.end(), sT.f.begin(), sT.f.end());
                        e.push_back(t);
                    }
                    hc = true; break;
                case 4: for (Term t : gen.A(jb.a, jb.b)) { t.f.push_back(yf(L2(K_Pt, jb.a, jb.b), true)); e.push_back(t); } hc = true; break;
                default: for (Term t : gen.B(jb.a, jb.b)) { t.f.push_back(yf(L2(K_Q, jb.a, jb.b), false)); e.push_back(t); }
            }
            for (const Term& t : e) {
                fwd[j].push_back(normalise(t, "LdR", dot));
                if (hc) adj[j].push_back(normalise(adjoint(t), "LdR", dot));
            }
        } catch (const std::exception& ex) {
#pragma omp critical
            err = ex.what();
        }
    }
    if (!err.empty()) throw std::logic_error(err);
    std::vector<NTerm> out;
    auto append = [&](int kind, std::vector<std::vector<NTerm>>& src) {
        for (size_t j = 0; j < jobs.size(); ++j)
            if (jobs[j].kind == kind) for (NTerm& t : src[j]) out.push_back(std::move(t));
    };
    append(0, fwd); append(1, fwd);
    for (int kind : {2, 3, 4}) append(kind, fwd);
    for (int kind : {2, 3, 4}) append(kind, adj);
    append(5, fwd);
    return out;
}

int64_t Engine::t_capacity() const {
    if (opt.workspace_bytes > 0) return opt.workspace_bytes / 8;
    size_t free_b = 0, total_b = 0;
    if (cudaMemGetInfo(&free_b, &total_b) != cudaSuccess) return (int64_t)1 << 27;
    int64_t cap = (int64_t)(free_b / 8) / 4;                   // a quarter of what is free ...
    const int64_t hi = ws_cap > 0 ? ws_cap : (int64_t)3 << 30; // ... at most 24 GiB (6 GiB while the environment stack is checkpointed)
    const int64_t lo = (int64_t)1 << 24;
    return std::max(lo, std::min(cap, hi));
}

namespace {

template <class T>
T* upload_vec(const std::vector<T>& v, std::vector<void*>& keep, cudaStream_t st) {
    T* d = (T*)dev_alloc(std::max<size_t>(v.size(), 1) * sizeof(T));
    keep.push_back(d);
    if (!v.empty()) cuda_check(cudaMemcpyAsync(d, v.data(), v.size() * sizeof(T), cudaMemcpyHostToDevice, st), "upload");
    return d;
}

// flattened quantum-number maps of every operator class of a block
MapSide upload_side(const Block& B, std::vector<void*>& keep, cudaStream_t st) {
    const int nsec = (int)B.basis.size(), ncls = (int)B.classes.size();
    std::vector<int> out((size_t)ncls * nsec, -1), inv((size_t)ncls * nsec, -1), dim(nsec);
    std::vector<int64_t> off((size_t)ncls * nsec, 0);
    for (int c = 0; c < ncls; ++c)
        for (int a = 0; a < nsec; ++a) {
            out[(size_t)c * nsec + a] = B.classes[c].out[a];
            inv[(size_t)c * nsec + a] = B.classes[c].inv[a];
            off[(size_t)c * nsec + a] = B.classes[c].off[a];
        }
    for (int a = 0; a < nsec; ++a) dim[a] = B.basis[a].d;
    MapSide sd;
    sd.out = upload_vec(out, keep, st); sd.inv = upload_vec(inv, keep, st); sd.off = upload_vec(off, keep, st);
    sd.dim = upload_vec(dim, keep, st); sd.nsec = nsec; sd.pad = 0;
    return sd;
}

void adopt(GemmLaunch& l, Task* tasks, int nt, Seg* segs, int ns, Tile* tiles, int ntiles, double flops) {
    l.tasks.p = tasks; l.tasks.n = (size_t)nt;
    l.segs.p = segs; l.segs.n = (size_t)ns;
    l.tiles.p = tiles; l.tiles.n = (size_t)ntiles;
    l.ntiles = ntiles; l.flops = flops; l.aligned = true;     // every operand of H_eff psi is 16-byte aligned with an even ld
    if (!l.counter.p) l.counter.alloc(1);
}

}  // namespace

// Device-built block maps: the host uploads O(terms + classes x sectors) integers, the kernels of
// heff_maps.cu enumerate everything that scales as terms x blocks.
static void build_maps_device(HeffPlan& p, const std::vector<NTerm>& terms, Block& LB, Block& RB, const Dot& dot,
                              Engine& eng) {
    cudaStream_t st = eng.stream;
    std::vector<void*> keep;                                   // tables only needed while building
    struct Guard { std::vector<void*>& k; ~Guard() { for (void* q : k) dev_free(q); } } guard{keep};
    const int nblk = (int)p.layout.size();
    // ---- tables ----------------------------------------------------------------------------------------------------------
    std::vector<MapBlock> blocks(nblk);
    for (int b = 0; b < nblk; ++b) {
        const PsiBlock& q = p.layout[b];
        blocks[b] = {q.l, q.ab, q.r, q.rows, q.cols, 0, q.off, q.poff};
    }
    std::vector<MapOp> opsL, opsR;
    std::vector<int> refclsL, refclsR;
    std::unordered_map<uint64_t, int> idxL, idxR, refL, refR;
    auto op_index = [&](Block& B, const Label& lab, bool trans, std::vector<MapOp>& ops, std::vector<int>& refcls,
                        std::unordered_map<uint64_t, int>& idx, std::unordered_map<uint64_t, int>& ref) {
        const uint64_t k1 = (uint64_t)lab.key() * 2 + (trans ? 1 : 0);
        auto it = idx.find(k1);
        if (it != idx.end()) return it->second;
        const OpRef& r = B.get(lab);
        auto ir = ref.find(lab.key());
        if (ir == ref.end()) { ir = ref.emplace(lab.key(), (int)refcls.size()).first; refcls.push_back(r.cls); }
        ops.push_back({r.ptr, r.cls, trans ? 1 : 0, ir->second, 0});
        idx.emplace(k1, (int)ops.size() - 1);
        return (int)ops.size() - 1;
    };
    std::vector<double> dmtab;
    std::map<std::vector<double>, int> dmidx;
    std::vector<MapTerm> mt, mt_ident;
    for (const NTerm& nt : terms) {
        if (nt.coef == 0.0) continue;
        MapTerm t;
        t.opL = nt.hasL ? op_index(LB, nt.L, nt.transL, opsL, refclsL, idxL, refL) : -1;
        t.opR = nt.hasR ? op_index(RB, nt.R, nt.transR, opsR, refclsR, idxR, refR) : -1;
        auto id = dmidx.find(nt.dm.a);
        if (id == dmidx.end()) {
            id = dmidx.emplace(nt.dm.a, (int)dmidx.size()).first;
            dmtab.insert(dmtab.end(), nt.dm.a.begin(), nt.dm.a.end());
        }
        t.dm = id->second;
        t.pd = dot.parity(nt.dm); t.pr = nt.hasR ? KIND_PAR[nt.R.kind] : 0; t.pad = 0; t.coef = nt.coef;
        (t.opL < 0 && t.opR < 0 ? mt_ident : mt).push_back(t);
    }
    mt.insert(mt.end(), mt_ident.begin(), mt_ident.end());     // operator-free terms last: their segments close every task
    std::vector<int> nL(LB.basis.size());
    for (size_t l = 0; l < LB.basis.size(); ++l) nL[l] = LB.basis[l].n;
    MapCtx cx;
    cx.blocks = upload_vec(blocks, keep, st); cx.lookup = upload_vec(p.lookup, keep, st);
    cx.terms = upload_vec(mt, keep, st); cx.dm = upload_vec(dmtab, keep, st);
    cx.opsL = upload_vec(opsL, keep, st); cx.opsR = upload_vec(opsR, keep, st);
    cx.refclsL = upload_vec(refclsL, keep, st); cx.refclsR = upload_vec(refclsR, keep, st);
    cx.nL = upload_vec(nL, keep, st); cx.dotqn = upload_vec(dot.qn, keep, st);
    cx.L = upload_side(LB, keep, st); cx.R = upload_side(RB, keep, st);
    cx.nblk = nblk; cx.nterm = (int)mt.size(); cx.nopsL = (int)opsL.size(); cx.nopsR = (int)opsR.size();
    cx.nrefL = (int)refclsL.size(); cx.nrefR = (int)refclsR.size();
    cx.xpad = p.xpad.p; cx.y = p.ybuf.p;
    // ---- pass A: accounting, diagonal, per-term intermediate usage -> chunks ---------------------------------------------------
    MapBuild mb;
    std::vector<double> usage;
    maps_usage(cx, usage, mb, dev_alloc, dev_free, st);
    p.diag_items.p = mb.diag_items; p.diag_items.n = (size_t)std::max(mb.ndiag, 1);
    p.diag_ptr.p = mb.diag_ptr; p.diag_ptr.n = (size_t)nblk + 1;
    const int64_t cap = eng.t_capacity();
    std::vector<int> cbegin(1, 0);
    double used = 0.0, t_max = 0.0;
    for (int t = 0; t < cx.nterm; ++t) {
        if (used > (double)(cap / 2)) { cbegin.push_back(t); used = 0.0; }
        used += usage[t];
        t_max = std::max(t_max, used);
    }
    cbegin.push_back(cx.nterm);
    const int nc = (int)cbegin.size() - 1;
    const size_t tsz = (size_t)std::max<double>(t_max, 2.0);
    p.T.alloc(tsz);
    cuda_check(cudaMemsetAsync(p.T.p, 0, tsz * 8, st), "memset");     // finite pads
    if (nc > 1) { p.T2.alloc(tsz); cuda_check(cudaMemsetAsync(p.T2.p, 0, tsz * 8, st), "memset"); }
    // split-K of phase 2: with few output tiles (small / medium bond dimensions) one tile per CTA slot leaves most of the
    // machine idle in the last wave, so each output block's term range is cut into S parts summed in fixed order
    int64_t base_tiles = 0;
    for (int b = 0; b < nblk; ++b)
        base_tiles += (int64_t)((p.layout[b].rows + GEMM_BM - 1) / GEMM_BM) * ((p.layout[b].cols + GEMM_BN - 1) / GEMM_BN);
    int S = 1;
    {
        int dev = 0, sms = 148;
        cudaGetDevice(&dev);
        cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
        // measured on B200: H_eff psi keeps improving up to ~50 tiles per resident CTA slot (config 4: S = 1 / 2 / 6 / 12
        // -> 25.2 / 25.9 / 26.3 / 26.5 TFLOP/s; config 3: S = 1 / 6 / 16 -> 9.0 / 12.5 / 13.6): shorter K ranges also keep
        // the tiles of one output block closer together in time, which helps the L2 hit rate of their shared panels
        const int64_t target = (int64_t)sms * 3 * 64;
        if (base_tiles > 0) S = (int)std::min<int64_t>(16, std::max<int64_t>(1, (target + base_tiles - 1) / base_tiles));
        if (eng.opt.split_k > 0) S = std::min(64, eng.opt.split_k);
    }
    p.split = S;
    if (S > 1) p.ypart.alloc((size_t)(S - 1) * (size_t)std::max<int64_t>(p.nnz, 1));
    // ---- pass B: descriptors of every chunk ------------------------------------------------------------------------------------
    p.chunks.resize(nc);
    p.ev_p1.resize(nc); p.ev_p2.resize(nc);
    double ngemm = mb.ngemm;
    for (int c = 0; c < nc; ++c) {
        MapChunkOut o;
        maps_chunk(cx, cbegin[c], cbegin[c + 1], c == 0, (c & 1) ? p.T2.p : p.T.p, S, p.ypart.p, p.nnz, o, dev_alloc, dev_free, st);
        if ((size_t)o.t_doubles > tsz) throw std::logic_error("heff: intermediate buffer bound violated");
        adopt(p.chunks[c].p1, o.tasks1, o.ntasks1, o.segs1, o.nsegs1, o.tiles1, o.ntiles1, o.flops1);
        adopt(p.chunks[c].p2, o.tasks2, o.ntasks2, o.segs2, o.nsegs2, o.tiles2, o.ntiles2, o.flops2);
        p.f_exec += o.flops1 + o.flops2;
        ngemm += o.ntasks1;
        cuda_check(cudaEventCreateWithFlags(&p.ev_p1[c], cudaEventDisableTiming), "event");
        cuda_check(cudaEventCreateWithFlags(&p.ev_p2[c], cudaEventDisableTiming), "event");
    }
    cuda_check(cudaEventCreateWithFlags(&p.ev_in, cudaEventDisableTiming), "event");
    if (S > 1) {
        MapChunkOut r;
        maps_reduce(cx, S, p.ypart.p, p.nnz, r, dev_alloc, dev_free, st);
        adopt(p.reduce, r.tasks2, r.ntasks2, r.segs2, r.nsegs2, r.tiles2, r.ntiles2, 0.0);
    }
    p.f_alg = mb.f_alg; p.ngemm = (int64_t)ngemm;
    p.b_alg = mb.b_ops + 16.0 * (double)p.nnz;
    // block tables for the diagonal / padding kernels
    std::vector<int> rows(nblk), cols(nblk);
    std::vector<int64_t> offs(nblk), poffs(nblk);
    for (int b = 0; b < nblk; ++b) { rows[b] = p.layout[b].rows; cols[b] = p.layout[b].cols; offs[b] = p.layout[b].off; poffs[b] = p.layout[b].poff; }
    p.blk_poff.upload(poffs, st); p.blk_rows.upload(rows, st); p.blk_cols.upload(cols, st); p.blk_off.upload(offs, st);
    cuda_check(cudaStreamSynchronize(st), "heff maps");
    cuda_check(cudaGetLastError(), "heff maps kernels");
}

std::unique_ptr<HeffPlan> build_heff(const Ham& ham, Block& LB, Block& RB, int i, Engine& eng) {
    std::unique_ptr<HeffPlan> pp(new HeffPlan());
    HeffPlan& p = *pp;
    p.bond = i;
    psi_layout(LB.basis, RB.basis, p.layout, p.lookup, p.nnz);
    Dot dot(&ham, std::vector<int>{i, i + 1});
    const std::vector<NTerm> terms = heff_terms(ham, LB, RB, dot, p.X, eng);
    p.nterms = (int64_t)terms.size();
    p.xbuf.alloc((size_t)p.nnz);
    p.ybuf.alloc((size_t)p.nnz);
    const int nblk = (int)p.layout.size();
    for (PsiBlock& b : p.layout) { b.poff = p.nnz_pad; p.nnz_pad += (int64_t)b.rows * pad2(b.cols); }
    p.xpad.alloc((size_t)std::max<int64_t>(p.nnz_pad, 2));
    cuda_check(cudaMemsetAsync(p.xpad.p, 0, (size_t)std::max<int64_t>(p.nnz_pad, 2) * 8, eng.stream), "memset");

    if (!eng.host_maps) {                                      // block maps built on the device (heff_maps.cu)
        build_maps_device(p, terms, LB, RB, dot, eng);
        return pp;
    }
    // ---- host reference builder (DMRG_B200_HOST_MAPS=1; A/B testing of the device builder) ----------------------------
    // enumerate contributions term by term, chunked by the intermediate buffer
    const int64_t cap = eng.t_capacity();
    int64_t t_max = 0;
    struct ChunkBuild { GemmBatch p1, p2; std::vector<int> task_of; };
    std::vector<ChunkBuild> builds;
    std::vector<std::vector<DiagItem>> diag(nblk);
    std::unordered_map<uint64_t, char> touched;                // operator blocks referenced (for b_alg)
    double b_ops = 0.0;
    auto new_chunk = [&]() {
        builds.emplace_back();
        ChunkBuild& cb = builds.back();
        cb.task_of.assign(nblk, -1);
        if (builds.size() == 1)                                // the first chunk initialises every output block
            for (int b = 0; b < nblk; ++b)
                cb.task_of[b] = cb.p2.add_task(p.ybuf.p + p.layout[b].off, p.layout[b].cols, p.layout[b].rows,
                                               p.layout[b].cols, 0);
    };
    new_chunk();
    int64_t used = 0;
    std::unordered_map<uint64_t, int64_t> tcache;              // (side, op, trans, in block) -> offset into T
    // T is allocated after planning (its size is only known then): record where its offsets must be patched in
    struct Patch { int chunk; size_t index; int64_t off; };
    std::vector<Patch> patchA, patchB, patchC;                 // p2 seg A / p2 seg B / p1 task C

    for (size_t ti = 0; ti < terms.size(); ++ti) {
        const NTerm& nt = terms[ti];
        const OpRef* opL = nt.hasL ? &LB.get(nt.L) : nullptr;
        const OpRef* opR = nt.hasR ? &RB.get(nt.R) : nullptr;
        const int pd = dot.parity(nt.dm), pr = nt.hasR ? KIND_PAR[nt.R.kind] : 0;
        if (used > cap / 2) { new_chunk(); used = 0; tcache.clear(); }
        ChunkBuild& cb = builds.back();
        const int chunk = (int)builds.size() - 1;
        for (int bi = 0; bi < nblk; ++bi) {
            const PsiBlock& in = p.layout[bi];
            OpBlockView vl, vr;
            int lo = in.l, ro = in.r;
            if (opL) { if (!op_block(LB, *opL, nt.transL, in.l, vl)) continue; lo = vl.out; }
            if (opR) { if (!op_block(RB, *opR, nt.transR, in.r, vr)) continue; ro = vr.out; }
            const int nl = LB.basis[in.l].n;
            const double sgn = ((pd * nl + pr * (nl + dot.qn[in.ab])) & 1) ? -1.0 : 1.0;
            for (int abo = 0; abo < 16; ++abo) {
                const double dmv = nt.dm(abo, in.ab);
                if (dmv == 0.0) continue;
                const int bo = p.lookup[lo * 16 + abo];
                if (bo < 0 || p.layout[bo].r != ro) continue;
                const PsiBlock& out = p.layout[bo];
                const double c = nt.coef * dmv * sgn;
                const double dl = in.rows, dr = in.cols, dlo = out.rows, dro = out.cols;
                if (cb.task_of[bo] < 0)
                    cb.task_of[bo] = cb.p2.add_task(p.ybuf.p + out.off, out.cols, out.rows, out.cols, TASK_ACCUM);
                const int t2 = cb.task_of[bo];
                const double* xin = p.xpad.p + in.poff;        // padded copy of x: every GEMM operand is aligned
                const int xld = pad2(in.cols);
                if (opL && opR && bo == bi)
                    diag[bi].push_back({vl.ptr, vl.ld, vr.ptr, vr.ld, c});
                else if (opL && !opR && bo == bi) diag[bi].push_back({vl.ptr, vl.ld, nullptr, 0, c});
                else if (!opL && opR && bo == bi) diag[bi].push_back({nullptr, 0, vr.ptr, vr.ld, c});
                else if (!opL && !opR && bo == bi) diag[bi].push_back({nullptr, 0, nullptr, 0, c});
                if (opL) { uint64_t k = ((uint64_t)(uintptr_t)vl.ptr); if (!touched.count(k)) { touched[k] = 1; b_ops += 8.0 * dlo * dl; } }
                if (opR) { uint64_t k = ((uint64_t)(uintptr_t)vr.ptr); if (!touched.count(k)) { touched[k] = 1; b_ops += 8.0 * dro * dr; } }
                if (!opL && !opR) {                            // c * X
                    cb.p2.add_seg(t2, xin, xld, nullptr, 0, 0, SEG_IDENT_B, c);
                    continue;
                }
                if (!opL) {                                    // Y += c X O_R^T
                    cb.p2.add_seg(t2, xin, xld, vr.ptr, vr.ld, in.cols, vr.trans ? 0 : SEG_TRANS_B, c);
                    p.f_alg += 2.0 * dl * dr * dro; p.ngemm += 1;
                    continue;
                }
                if (!opR) {                                    // Y += c O_L X
                    cb.p2.add_seg(t2, vl.ptr, vl.ld, xin, xld, in.rows, vl.trans ? SEG_TRANS_A : 0, c);
                    p.f_alg += 2.0 * dlo * dl * dr; p.ngemm += 1;
                    continue;
                }
                const double cost_l = 2.0 * dlo * dl * dr + 2.0 * dlo * dr * dro;   // (O_L X) O_R^T
                const double cost_r = 2.0 * dl * dr * dro + 2.0 * dlo * dl * dro;   // O_L (X O_R^T)
                p.f_alg += std::min(cost_l, cost_r);
                const bool lfirst = cost_l <= cost_r;
                const OpBlockView& v1 = lfirst ? vl : vr;
                const uint64_t key = ((uint64_t)(uintptr_t)v1.ptr) * 2 + (lfirst ? 0 : 1);
                const uint64_t key2 = key * 1315423911ull + (uint64_t)bi * 2654435761ull;
                auto it = tcache.find(key2);
                const int trows = lfirst ? out.rows : in.rows, tcols = lfirst ? in.cols : out.cols;
                const int tld = pad2(tcols);
                if (it == tcache.end()) {
                    const int64_t toff = used;
                    used += (int64_t)trows * tld;
                    t_max = std::max(t_max, used);
                    const int t1 = cb.p1.add_task(nullptr, tld, trows, tcols, 0);
                    patchC.push_back({chunk, (size_t)t1, toff});
                    if (lfirst) cb.p1.add_seg(t1, vl.ptr, vl.ld, xin, xld, in.rows, vl.trans ? SEG_TRANS_A : 0, 1.0);
                    else        cb.p1.add_seg(t1, xin, xld, vr.ptr, vr.ld, in.cols, vr.trans ? 0 : SEG_TRANS_B, 1.0);
                    p.ngemm += 1;
                    it = tcache.emplace(key2, toff).first;
                }
                const int64_t toff = it->second;
                if (lfirst) {                                  // Y += c T O_R^T
                    cb.p2.add_seg(t2, nullptr, tld, vr.ptr, vr.ld, in.cols, vr.trans ? 0 : SEG_TRANS_B, c);
                    patchA.push_back({chunk, cb.p2.segs.size() - 1, toff});
                } else {                                       // Y += c O_L T
                    cb.p2.add_seg(t2, vl.ptr, vl.ld, nullptr, tld, in.rows, vl.trans ? SEG_TRANS_A : 0, c);
                    patchB.push_back({chunk, cb.p2.segs.size() - 1, toff});
                }
                p.ngemm += 1;
            }
        }
    }
    // ---- materialise: allocate T, patch offsets into addresses, upload ------------------------------------------------
    // two buffers: even chunks use T, odd chunks T2, so phase 1 of chunk c+1 can run beside phase 2 of chunk c
    const size_t tsz = (size_t)std::max<int64_t>(t_max, 2);
    p.T.alloc(tsz);
    cuda_check(cudaMemsetAsync(p.T.p, 0, tsz * 8, eng.stream), "memset");   // finite pads
    if (builds.size() > 1) {
        p.T2.alloc(tsz);
        cuda_check(cudaMemsetAsync(p.T2.p, 0, tsz * 8, eng.stream), "memset");
    }
    auto tbase = [&](int chunk) { return (chunk & 1) ? p.T2.p : p.T.p; };
    for (auto& pc : patchC) builds[pc.chunk].p1.tasks[pc.index].C = tbase(pc.chunk) + pc.off;
    for (auto& pa : patchA) builds[pa.chunk].p2.segs[pa.index].A = tbase(pa.chunk) + pa.off;
    for (auto& pb : patchB) builds[pb.chunk].p2.segs[pb.index].B = tbase(pb.chunk) + pb.off;
    p.ev_p1.resize(builds.size());
    p.ev_p2.resize(builds.size());
    for (size_t c = 0; c < builds.size(); ++c) {
        cuda_check(cudaEventCreateWithFlags(&p.ev_p1[c], cudaEventDisableTiming), "event");
        cuda_check(cudaEventCreateWithFlags(&p.ev_p2[c], cudaEventDisableTiming), "event");
    }
    cuda_check(cudaEventCreateWithFlags(&p.ev_in, cudaEventDisableTiming), "event");
    p.chunks.resize(builds.size());
    for (size_t c = 0; c < builds.size(); ++c) {
        p.f_exec += builds[c].p1.flops + builds[c].p2.flops;
        finalize(builds[c].p1, p.chunks[c].p1, eng);
        finalize(builds[c].p2, p.chunks[c].p2, eng);
    }
    p.b_alg = b_ops + 16.0 * (double)p.nnz;
    // ---- diagonal items -----------------------------------------------------------------------------------------------
    std::vector<DiagItem> items;
    std::vector<int> ptr(nblk + 1, 0), rows(nblk), cols(nblk);
    std::vector<int64_t> offs(nblk);
    for (int b = 0; b < nblk; ++b) {
        items.insert(items.end(), diag[b].begin(), diag[b].end());
        ptr[b + 1] = (int)items.size();
        rows[b] = p.layout[b].rows; cols[b] = p.layout[b].cols; offs[b] = p.layout[b].off;
    }
    std::vector<int64_t> poffs(nblk);
    for (int b = 0; b < nblk; ++b) poffs[b] = p.layout[b].poff;
    p.blk_poff.upload(poffs, eng.stream);
    p.diag_items.upload(items, eng.stream);
    p.diag_ptr.upload(ptr, eng.stream);
    p.blk_rows.upload(rows, eng.stream);
    p.blk_cols.upload(cols, eng.stream);
    p.blk_off.upload(offs, eng.stream);
    cuda_check(cudaStreamSynchronize(eng.stream), "heff plan upload");
    return pp;
}

void heff_apply(HeffPlan& p, const double* x_dev, double* y_dev, Engine& eng) {
    // x (packed exchange layout) -> padded, aligned copy read by the GEMM kernel
    launch_pad_blocks(p.xpad.p, x_dev, (int)p.layout.size(), p.blk_poff.p, p.blk_off.p, p.blk_rows.p, p.blk_cols.p, eng.stream);
    eng.launches++;
    // Software pipeline over the chunks on two streams: phase 1 (T = O X) of chunk c+1 fills the SMs that the tail of
    // phase 2 (Y += T O^T) of chunk c leaves idle.  Phase 2 launches stay in chunk order on one stream, so the
    // accumulation order into y is fixed (bit-reproducible); T is double buffered (chunk parity).
    const int nc = (int)p.chunks.size();
    if (nc == 1 || eng.trace) {
        for (auto& c : p.chunks) { run(c.p1, eng); run(c.p2, eng); if (p.split > 1) run(p.reduce, eng); }
    } else {
        cuda_check(cudaEventRecord(p.ev_in, eng.stream), "event record");
        cuda_check(cudaStreamWaitEvent(eng.stream2, p.ev_in, 0), "stream wait");
        for (int c = 0; c < nc; ++c) {
            if (c >= 2) cuda_check(cudaStreamWaitEvent(eng.stream, p.ev_p2[c - 2], 0), "stream wait");   // T buffer free
            run(p.chunks[c].p1, eng, eng.stream);
            cuda_check(cudaEventRecord(p.ev_p1[c], eng.stream), "event record");
            cuda_check(cudaStreamWaitEvent(eng.stream2, p.ev_p1[c], 0), "stream wait");
            run(p.chunks[c].p2, eng, eng.stream2);
            if (p.split > 1) run(p.reduce, eng, eng.stream2);
            cuda_check(cudaEventRecord(p.ev_p2[c], eng.stream2), "event record");
        }
        cuda_check(cudaStreamWaitEvent(eng.stream, p.ev_p2[nc - 1], 0), "stream wait");
    }
    if (y_dev != p.ybuf.p)
        cuda_check(cudaMemcpyAsync(y_dev, p.ybuf.p, (size_t)p.nnz * 8, cudaMemcpyDeviceToDevice, eng.stream), "y copy");
}

void heff_diag(HeffPlan& p, double* d_dev, Engine& eng) {
    launch_heff_diag(d_dev, (int)p.layout.size(), p.blk_off.p, p.blk_rows.p, p.blk_cols.p, p.diag_ptr.p,
                     p.diag_items.p, eng.stream);
    eng.launches++;
}

}  // namespace dmrg
