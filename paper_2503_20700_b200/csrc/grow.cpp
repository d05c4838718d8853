// Operator renormalisation (blocking), SURVEY.md 8(a) row a5 / DESIGN.md "Algorithm" step 3:
//   X' = sum_{s',s} A[s']^T ( sum_j c_j O_j (x) o_j[s',s] ) A[s]      (left block; B ... B^T for a right block)
// The enlarged operator is never materialised: phase 1 forms the half-rotated pieces
//   tmp[(o,s'), m] = sum_{j,s,i} c_j o_j[s',s] sgn  O_j[o<-i] A[(i,s) -> m]      (K-concatenated over pieces)
// and phase 2 contracts them with the bra tensor, out[m' <- m] = sum_{(o,s')} A[(o,s') -> m']^T tmp[(o,s'), m];
// both phases are launches of the grouped FP64 GEMM kernel over all new operators of a chunk.
#include <algorithm>
#include <cassert>
#include <chrono>
#include <cstdio>

#include "core.hpp"

namespace dmrg {

void Block::drop_kind(int kind) {
    for (auto it = ops.begin(); it != ops.end();)
        if ((int)(it->first >> 24) == kind) it = ops.erase(it);
        else ++it;
}

std::unique_ptr<Block> empty_block(char side, int k, const MPS& mps) {
    const int b = side == 'L' ? 0 : k;
    return std::unique_ptr<Block>(new Block(side, b, k, mps.bonds[b], 'N'));
}

// ---------------------------------------------------------------------------------------------------------------
// temporaries on X: complementary two-index operators touching the dot (N mode only) and the one-index
// combinations U, V that enter the growth of S_P
// ---------------------------------------------------------------------------------------------------------------
void make_temps(const Ham& ham, Block& X, const Dot& dot, const std::vector<int>& far, Engine& eng) {
    const std::vector<int> Xin = X.inside();
    if (Xin.empty()) return;
    std::vector<int> pool = dot.so;
    pool.insert(pool.end(), far.begin(), far.end());
    std::sort(pool.begin(), pool.end());
    // destinations first (cheap), then the integral-weighted source lists on the host threads: at k = 82 that is ~10^7
    // lookups of (pq|rs) per bond.  Dense (stack, row) tables of the stored A / B / C operators replace the label lookups.
    const int nso = 2 * X.k;
    struct Src { int stack, row; };
    std::vector<Src> tA((size_t)nso * nso, Src{-1, -1}), tB((size_t)nso * nso, Src{-1, -1}), tC(nso, Src{-1, -1});
    for (const auto& kv : X.ops) {
        const int kind = (int)(kv.first >> 24), a = (int)((kv.first >> 16) & 255), b = (int)((kv.first >> 8) & 255);
        if (kind == K_A) tA[(size_t)a * nso + b] = {kv.second.stack, kv.second.row};
        else if (kind == K_B) tB[(size_t)a * nso + b] = {kv.second.stack, kv.second.row};
        else if (kind == K_C) tC[a] = {kv.second.stack, kv.second.row};
    }
    auto shift = [](const Label& x, int& a, int& b) { op_shift(x, a, b); };
    std::vector<LinSpec> specs;
    if (X.mode == 'N') {
        for (size_t a = 0; a < pool.size(); ++a)
            for (size_t b = a + 1; b < pool.size(); ++b) {
                if (!dot.has(pool[a]) && !dot.has(pool[b])) continue;
                LinSpec s; s.dst = L2(K_Pt, pool[a], pool[b]);   // (P_PQ)^T = -sum_{R<S} w_PQRS A_RS
                specs.push_back(s);
            }
        for (int P : pool)
            for (int S : pool) {
                if (!dot.has(P) && !dot.has(S)) continue;
                LinSpec s; s.dst = L2(K_Q, P, S);              // Q_PS = sum_{QR} w_PQRS B_QR
                specs.push_back(s);
            }
    }
    const size_t n_two = specs.size();
    for (int P : far) {
        for (size_t a = 0; a < dot.so.size(); ++a)
            for (size_t b = a + 1; b < dot.so.size(); ++b) { LinSpec s; s.dst = L3(K_U, P, dot.so[a], dot.so[b]); specs.push_back(s); }   // U_{P;RS} = sum_Q w_PQRS a+_Q
        for (int Q : dot.so)
            for (int R : dot.so) { LinSpec s; s.dst = L3(K_V, P, Q, R); specs.push_back(s); }                                                // V_{P;QR} = sum_S w_PQRS a+_S
    }
#pragma omp parallel for schedule(dynamic, 8) if (specs.size() > 64)
    for (long j = 0; j < (long)specs.size(); ++j) {
        LinSpec& s = specs[j];
        int dn, ds, sn, ss;
        shift(s.dst, dn, ds);
        if (s.dst.kind == K_Pt) {
            const int P = s.dst.a, Q = s.dst.b;
            for (size_t i = 0; i < Xin.size(); ++i)
                for (size_t q = i + 1; q < Xin.size(); ++q) {
                    const Label src = L2(K_A, Xin[i], Xin[q]);
                    shift(src, sn, ss);
                    if (sn != dn || ss != ds) continue;
                    const Src t = tA[(size_t)Xin[i] * nso + Xin[q]];
                    s.items.push_back({-ham.w(P, Q, Xin[i], Xin[q]), src, t.stack, t.row});
                }
        } else if (s.dst.kind == K_Q) {
            const int P = s.dst.a, S = s.dst.b;
            for (int Q : Xin)
                for (int R : Xin) {
                    const Label src = L2(K_B, Q, R);
                    shift(src, sn, ss);
                    if (sn != dn || ss != ds) continue;
                    const Src t = tB[(size_t)Q * nso + R];
                    s.items.push_back({ham.w(P, Q, R, S), src, t.stack, t.row});
                }
        } else if (s.dst.kind == K_U) {
            const int P = s.dst.a, R = s.dst.b, S = s.dst.c;
            for (int Q : Xin) { const double w = ham.w(P, Q, R, S); if (w != 0.0) s.items.push_back({w, L1(K_C, Q), tC[Q].stack, tC[Q].row}); }
        } else {
            const int P = s.dst.a, Q = s.dst.b, R = s.dst.c;
            for (int S : Xin) { const double w = ham.w(P, Q, R, S); if (w != 0.0) s.items.push_back({w, L1(K_C, S), tC[S].stack, tC[S].row}); }
        }
    }
    // one-index combinations without any source are not stored (their absence is how the generator skips them)
    std::vector<LinSpec> kept;
    kept.reserve(specs.size());
    for (size_t j = 0; j < specs.size(); ++j)
        if (j < n_two || !specs[j].items.empty()) kept.push_back(std::move(specs[j]));
    std::vector<Label> labels;
    for (const LinSpec& s : kept) labels.push_back(s.dst);
    X.allocate(labels, true);
    lincomb(X, kept, false, eng);
}

// ---------------------------------------------------------------------------------------------------------------
// rotation of a list of enlarged-operator expressions into the new basis
// ---------------------------------------------------------------------------------------------------------------
struct NewOp { Label label; Expr expr; };

// Descriptors of ONE new operator, built by one host thread: T pointers are relative to offset 0 of the workspace and
// task indices are local; merge() below rebases both into the launch-wide batches.
struct OpPlan {
    GemmBatch p1, p2;
    std::vector<int> tsegs;                        // phase-2 segments whose B operand is a workspace buffer
    int64_t used = 0;
};

static void plan_op(Block& X, const Dot& dot, const SiteTensor& tensor, Block& nb, const NewOp& no, int64_t cap,
                    OpPlan& out) {
    double* const tbase = nullptr;                         // workspace addresses are offsets until merge() rebases them
    const bool left = X.side == 'L';
    const char* chain = left ? "Ld" : "dR";
    const int nnew = (int)nb.basis.size();
    GemmBatch& p1 = out.p1;
    GemmBatch& p2 = out.p2;
    int64_t& used = out.used;
    // new-basis sector reached from X-sector i by adding (left) / removing (right) site state s
    auto new_sector = [&](int i, int s) {
        const Sector& q = X.basis[i];
        return left ? find_sector(nb.basis, q.n + SITE_QN[s], q.s + SITE_QS[s])
                    : find_sector(nb.basis, q.n - SITE_QN[s], q.s - SITE_QS[s]);
    };
    auto tensor_block = [&](int xsec, int s, int newsec) -> const SiteTensor::Blk* {
        if (newsec < 0) return nullptr;
        return left ? tensor.get(xsec, s) : tensor.get(newsec, s);
    };
    const OpRef& ref = nb.get(no.label);
    const OpClass& nc = nb.classes[ref.cls];
    std::vector<int> p2task(nnew, -1);
    auto out_task = [&](int mi) {
        if (p2task[mi] < 0)
            p2task[mi] = p2.add_task(ref.ptr + nc.off[mi], pad2(nb.basis[mi].d), nb.basis[nc.out[mi]].d,
                                     nb.basis[mi].d, 0);
        return p2task[mi];
    };
    for (int mi = 0; mi < nnew; ++mi)
        if (nc.out[mi] >= 0) out_task(mi);                 // every block is written (zero if nothing feeds it)
    std::unordered_map<int64_t, std::pair<int, double*>> tmps;   // (o, so, mi) -> (phase-1 task, buffer)
    for (const Term& term : no.expr) {
        const NTerm nt = normalise(term, chain, dot);
        const bool has_op = left ? nt.hasL : nt.hasR;
        const Label& lab = left ? nt.L : nt.R;
        const bool tr = left ? nt.transL : nt.transR;
        const OpRef* op = has_op ? &X.get(lab) : nullptr;
        const int po = has_op ? KIND_PAR[lab.kind] : 0;
        const int pm = dot.parity(nt.dm);
        for (int so = 0; so < 4; ++so)
            for (int si = 0; si < 4; ++si) {
                const double dmv = nt.dm(so, si);
                if (dmv == 0.0) continue;
                for (int i = 0; i < (int)X.basis.size(); ++i) {
                    OpBlockView v;
                    int o = i;
                    if (op) { if (!op_block(X, *op, tr, i, v)) continue; o = v.out; }
                    const int mi = new_sector(i, si), mo = new_sector(o, so);
                    const SiteTensor::Blk* ti = tensor_block(i, si, mi);
                    const SiteTensor::Blk* to = tensor_block(o, so, mo);
                    if (!ti || !to) continue;
                    if (nc.out[mi] != mo) throw std::logic_error("rotate: quantum numbers do not close");
                    const double sgn = left ? ((pm && (X.basis[i].n & 1)) ? -1.0 : 1.0)
                                            : ((po && (SITE_QN[si] & 1)) ? -1.0 : 1.0);
                    const double alpha = nt.coef * dmv * sgn;
                    const int di = X.basis[i].d, dO = X.basis[o].d, dmi = nb.basis[mi].d;
                    if (!op) {                             // identity block factor: straight into phase 2
                        if (left) p2.add_seg(out_task(mi), to->ptr, to->ld, ti->ptr, ti->ld, di, SEG_TRANS_A, alpha);
                        else      p2.add_seg(out_task(mi), to->ptr, to->ld, ti->ptr, ti->ld, di, SEG_TRANS_B, alpha);
                        continue;
                    }
                    const int64_t key = ((int64_t)o * 4 + so) * nnew + mi;
                    auto it = tmps.find(key);
                    if (it == tmps.end()) {
                        const int64_t sz = (int64_t)dO * pad2(dmi);
                        if (used + sz > cap) throw Error(-3, "renormalisation workspace too small");
                        double* buf = tbase + used;
                        used += sz;
                        const int t1 = p1.add_task(buf, pad2(dmi), dO, dmi, 0);
                        it = tmps.emplace(key, std::make_pair(t1, buf)).first;
                        // phase 2: out[mo <- mi] += to^T tmp (left) / to tmp (right)
                        if (left) p2.add_seg(out_task(mi), to->ptr, to->ld, buf, pad2(dmi), dO, SEG_TRANS_A, 1.0);
                        else      p2.add_seg(out_task(mi), to->ptr, to->ld, buf, pad2(dmi), dO, 0, 1.0);
                        out.tsegs.push_back((int)p2.segs.size() - 1);
                    }
                    int fl = v.trans ? SEG_TRANS_A : 0;
                    if (!left) fl |= SEG_TRANS_B;          // ti stored [d_m x d_i]
                    p1.add_seg(it->second.first, v.ptr, v.ld, ti->ptr, ti->ld, di, fl, alpha);
                }
            }
    }
}

// append the plans [j0, j1) to the launch-wide batches in list order: task indices shifted, workspace offsets turned into
// addresses (plan j starts at base + toff[j]).  Sizes are prefix-summed first, then the copies run on the host threads.
static void merge_range(GemmBatch& p1, GemmBatch& p2, const std::vector<OpPlan>& plans, size_t j0, size_t j1,
                        const std::vector<int64_t>& toff, double* base) {
    const size_t n = j1 - j0;
    std::vector<size_t> t1(n + 1, 0), s1(n + 1, 0), t2(n + 1, 0), s2(n + 1, 0);
    for (size_t j = 0; j < n; ++j) {
        const OpPlan& pl = plans[j0 + j];
        t1[j + 1] = t1[j] + pl.p1.tasks.size(); s1[j + 1] = s1[j] + pl.p1.segs.size();
        t2[j + 1] = t2[j] + pl.p2.tasks.size(); s2[j + 1] = s2[j] + pl.p2.segs.size();
        p1.flops += pl.p1.flops; p2.flops += pl.p2.flops;
    }
    p1.tasks.resize(t1[n]); p1.segs.resize(s1[n]); p1.seg_task.resize(s1[n]);
    p2.tasks.resize(t2[n]); p2.segs.resize(s2[n]); p2.seg_task.resize(s2[n]);
#pragma omp parallel for schedule(dynamic, 8) if (n > 32)
    for (long j = 0; j < (long)n; ++j) {
        const OpPlan& pl = plans[j0 + j];
        double* tb = base + toff[j0 + j];
        for (size_t q = 0; q < pl.p1.tasks.size(); ++q) {
            Task t = pl.p1.tasks[q];
            t.C = tb + (t.C - (double*)nullptr);
            p1.tasks[t1[j] + q] = t;
        }
        for (size_t q = 0; q < pl.p1.segs.size(); ++q) {
            p1.segs[s1[j] + q] = pl.p1.segs[q];
            p1.seg_task[s1[j] + q] = (int)t1[j] + pl.p1.seg_task[q];
        }
        for (size_t q = 0; q < pl.p2.tasks.size(); ++q) p2.tasks[t2[j] + q] = pl.p2.tasks[q];
        for (size_t q = 0; q < pl.p2.segs.size(); ++q) {
            p2.segs[s2[j] + q] = pl.p2.segs[q];
            p2.seg_task[s2[j] + q] = (int)t2[j] + pl.p2.seg_task[q];
        }
        for (int q : pl.tsegs) { Seg& sg = p2.segs[s2[j] + q]; sg.B = tb + (sg.B - (const double*)nullptr); }
    }
}

static void rotate_batch(Block& X, const Dot& dot, const SiteTensor& tensor, Block& nb, const std::vector<NewOp>& list,
                         bool temp, Engine& eng) {
    std::vector<Label> labels;
    for (const NewOp& o : list) labels.push_back(o.label);
    nb.allocate(labels, temp);
    const int64_t cap = eng.t_capacity();
    // The integer descriptors of the new operators are independent of each other: host threads plan them (workspace
    // addresses as offsets from zero), then the plans are appended in list order, so the launches do not depend on the
    // number of threads.  The workspace is sized by what the plans need (at most `cap`: then in several flushes).
    std::vector<OpPlan> plans(list.size());
    std::string err;
    int err_code = 0;
    const auto tp0 = std::chrono::steady_clock::now();
#pragma omp parallel for schedule(dynamic, 4) if (list.size() > 32)
    for (long j = 0; j < (long)list.size(); ++j) {
        try {
            plan_op(X, dot, tensor, nb, list[j], cap, plans[j]);
        } catch (const Error& e) {
#pragma omp critical
            { err = e.what(); err_code = e.code; }
        } catch (const std::exception& e) {
#pragma omp critical
            { err = e.what(); err_code = -2; }
        }
    }
    if (err_code) { if (err_code == -3) throw Error(-3, err); throw std::logic_error(err); }
    const auto tp1 = std::chrono::steady_clock::now();
    int64_t total = 0;
    for (const OpPlan& pl : plans) total += pl.used;
    DevVec<double> tmp;
    tmp.alloc((size_t)std::max<int64_t>(2, std::min(total, cap)));
    GemmBatch p1, p2;
    int64_t used = 0;
    double t_run = 0.0;
    auto flush = [&]() {
        const auto a = std::chrono::steady_clock::now();
        run_once(p1, eng);
        run_once(p2, eng);
        t_run += std::chrono::duration<double>(std::chrono::steady_clock::now() - a).count();
        used = 0;
    };
    // flush groups: consecutive plans whose workspace fits (one group when everything fits)
    std::vector<int64_t> toff(plans.size(), 0);
    size_t j = 0;
    while (j < plans.size()) {
        const size_t g0 = j;
        used = 0;
        while (j < plans.size()) {
            if (used + plans[j].used > cap) break;            // does not fit: the group closes before plan j
            toff[j] = used;
            used += plans[j].used;
            ++j;
            if (total > cap && used > cap / 2) break;         // several flushes: close at half the workspace
        }
        if (j == g0) throw Error(-3, "renormalisation workspace too small");
        merge_range(p1, p2, plans, g0, j, toff, tmp.p);
        for (size_t q = g0; q < j; ++q) plans[q] = OpPlan();
        flush();
    }
    if (eng.trace) {
        const double all = std::chrono::duration<double>(std::chrono::steady_clock::now() - tp0).count();
        const double plan = std::chrono::duration<double>(tp1 - tp0).count();
        std::fprintf(stderr, "[dmrg trace] rotate_batch ops=%zu plan=%.4f merge=%.4f finalize+run=%.4f s\n", list.size(), plan,
                     all - plan - t_run, t_run);
    }
}

// symbolic expressions of a list of new operators, generated by the host threads (the generator is read-only)
enum OpWhat : int { W_H, W_CRE, W_ST, W_A, W_B, W_COPY };
struct OpSpec { Label label; int what; };
static std::vector<NewOp> make_ops(const std::vector<OpSpec>& specs, const Gen& gen) {
    std::vector<NewOp> out(specs.size());
#pragma omp parallel for schedule(dynamic, 16) if (specs.size() > 256)
    for (long j = 0; j < (long)specs.size(); ++j) {
        const Label& l = specs[j].label;
        NewOp& o = out[j];
        o.label = l;
        switch (specs[j].what) {
            case W_H: o.expr = gen.H(); break;
            case W_CRE: o.expr = gen.cre(l.a); break;
            case W_ST: for (const Term& t : gen.S(l.a)) o.expr.push_back(adjoint(t)); break;
            case W_A: o.expr = gen.A(l.a, l.b); break;
            case W_B: o.expr = gen.B(l.a, l.b); break;
            default: { Term t; t.f.push_back(gen.bf(l)); o.expr.push_back(t); }
        }
    }
    return out;
}

static bool same_shift(const Label& x, const Label& y) {
    int a, b, c, d;
    op_shift(x, a, b); op_shift(y, c, d);
    return a == c && b == d;
}

std::unique_ptr<Block> grow(Block& X, const Ham& ham, const MPS& mps, char new_mode, Engine& eng) {
    const bool left = X.side == 'L';
    const int p = left ? X.b : X.b - 1, nbond = left ? X.b + 1 : X.b - 1;
    const SiteTensor& tensor = mps.sites[p];
    Dot dot(&ham, std::vector<int>{p});
    std::unique_ptr<Block> nbp(new Block(X.side, nbond, X.k, mps.bonds[nbond], new_mode));
    Block& nb = *nbp;
    const std::vector<int> inside = nb.inside(), outside = nb.outside();
    make_temps(ham, X, dot, outside, eng);
    Gen gen(ham, block_info(X), dot);
    std::vector<OpSpec> list;
    list.push_back({L0(K_H), W_H});
    for (int P : inside) list.push_back({L1(K_C, P), W_CRE});
    for (int P : outside) list.push_back({L1(K_St, P), W_ST});
    if (X.mode == 'N') {
        std::vector<OpSpec> two;
        for (size_t a = 0; a < inside.size(); ++a) {
            for (size_t b = a + 1; b < inside.size(); ++b) two.push_back({L2(K_A, inside[a], inside[b]), W_A});
            for (int S : inside) two.push_back({L2(K_B, inside[a], S), W_B});
        }
        if (new_mode == 'N') {
            list.insert(list.end(), two.begin(), two.end());
            rotate_batch(X, dot, tensor, nb, make_ops(list, gen), false, eng);
        } else {                                               // grow the normal operators, then convert
            rotate_batch(X, dot, tensor, nb, make_ops(list, gen), false, eng);
            rotate_batch(X, dot, tensor, nb, make_ops(two, gen), true, eng);
            std::vector<LinSpec> specs;
            for (size_t a = 0; a < outside.size(); ++a) {
                for (size_t b = a + 1; b < outside.size(); ++b) {
                    LinSpec s; s.dst = L2(K_Pt, outside[a], outside[b]);
                    for (size_t i = 0; i < inside.size(); ++i)
                        for (size_t j = i + 1; j < inside.size(); ++j) {
                            const Label src = L2(K_A, inside[i], inside[j]);
                            if (same_shift(src, s.dst)) s.items.push_back({-ham.w(outside[a], outside[b], inside[i], inside[j]), src});
                        }
                    specs.push_back(s);
                }
                for (int S : outside) {
                    LinSpec s; s.dst = L2(K_Q, outside[a], S);
                    for (int Q : inside)
                        for (int R : inside) {
                            const Label src = L2(K_B, Q, R);
                            if (same_shift(src, s.dst)) s.items.push_back({ham.w(outside[a], Q, R, S), src});
                        }
                    specs.push_back(s);
                }
            }
            std::vector<Label> labels;
            for (const LinSpec& s : specs) labels.push_back(s.dst);
            nb.allocate(labels, false);
            lincomb(nb, specs, false, eng);
            nb.drop_temps();
        }
    } else {
        if (new_mode != 'C') throw std::logic_error("grow: complementary -> normal is not supported");
        std::vector<char> in_x(2 * X.k, 0);
        for (int P : X.inside()) in_x[P] = 1;
        std::vector<OpSpec> mixed;                             // new normal operators with one index on the new site
        for (size_t a = 0; a < inside.size(); ++a) {
            for (size_t b = a + 1; b < inside.size(); ++b)
                if (!(in_x[inside[a]] && in_x[inside[b]])) mixed.push_back({L2(K_A, inside[a], inside[b]), W_A});
            for (int S : inside)
                if (!(in_x[inside[a]] && in_x[S])) mixed.push_back({L2(K_B, inside[a], S), W_B});
        }
        std::vector<LinSpec> specs;
        for (size_t a = 0; a < outside.size(); ++a) {
            for (size_t b = a + 1; b < outside.size(); ++b) {
                const Label l = L2(K_Pt, outside[a], outside[b]);
                list.push_back({l, W_COPY});
                LinSpec s; s.dst = l;
                for (const OpSpec& m : mixed)
                    if (m.label.kind == K_A && same_shift(m.label, l))
                        s.items.push_back({-ham.w(outside[a], outside[b], m.label.a, m.label.b), m.label});
                specs.push_back(s);
            }
            for (int S : outside) {
                const Label l = L2(K_Q, outside[a], S);
                list.push_back({l, W_COPY});
                LinSpec s; s.dst = l;
                for (const OpSpec& m : mixed)
                    if (m.label.kind == K_B && same_shift(m.label, l))
                        s.items.push_back({ham.w(outside[a], m.label.a, m.label.b, S), m.label});
                specs.push_back(s);
            }
        }
        rotate_batch(X, dot, tensor, nb, make_ops(list, gen), false, eng);
        rotate_batch(X, dot, tensor, nb, make_ops(mixed, gen), true, eng);
        lincomb(nb, specs, true, eng);
        nb.drop_temps();
    }
    X.drop_temps();
    return nbp;
}

std::unique_ptr<Block> grow_normal(Block& X, const Ham& ham, const Basis& new_basis, const SiteTensor& tensor,
                                   int pair_lo, int pair_hi, Engine& eng) {
    const bool left = X.side == 'L';
    const int p = left ? X.b : X.b - 1, nbond = left ? X.b + 1 : X.b - 1;
    Dot dot(&ham, std::vector<int>{p});
    std::unique_ptr<Block> nbp(new Block(X.side, nbond, X.k, new_basis, 'N'));
    Gen gen(ham, block_info(X), dot);
    const std::vector<int> inside = nbp->inside();
    auto paired = [&](int P) { const int s = P >> 1; return s >= pair_lo && s < pair_hi; };
    std::vector<OpSpec> list;
    for (size_t a = 0; a < inside.size(); ++a) {
        list.push_back({L1(K_C, inside[a]), W_CRE});
        if (!paired(inside[a])) continue;
        for (size_t b = a + 1; b < inside.size(); ++b)
            if (paired(inside[b])) list.push_back({L2(K_A, inside[a], inside[b]), W_A});
        for (int S : inside)
            if (paired(S)) list.push_back({L2(K_B, inside[a], S), W_B});
    }
    rotate_batch(X, dot, tensor, *nbp, make_ops(list, gen), false, eng);
    return nbp;
}

}  // namespace dmrg
