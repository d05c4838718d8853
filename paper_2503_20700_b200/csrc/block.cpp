// Device-resident block operators: storage, launch-descriptor plumbing, linear combinations, blocking (grow).
#include <algorithm>
#include <cassert>
#include <chrono>
#include <cmath>
#include <cstdio>
#include <cstring>
#include <mutex>

#include "core.hpp"

namespace dmrg {

// ---------------------------------------------------------------------------------------------------------------
// device memory and descriptors
// ---------------------------------------------------------------------------------------------------------------
int64_t g_device_bytes = 0;
static std::unordered_map<void*, size_t> g_sizes;
static std::mutex g_alloc_mutex;                           // allocations also come from the host threads of split_theta

void cuda_check(cudaError_t e, const char* what) {
    if (e != cudaSuccess) throw Error(-4, std::string(what) + ": " + cudaGetErrorString(e));
}
void* dev_alloc(size_t bytes) {
    void* p = nullptr;
    if (bytes == 0) return nullptr;
    cudaError_t e = cudaMalloc(&p, bytes);
    if (e == cudaErrorMemoryAllocation) { cudaGetLastError(); throw Error(-3, "out of device memory"); }
    cuda_check(e, "cudaMalloc");
    std::lock_guard<std::mutex> lock(g_alloc_mutex);
    g_sizes[p] = bytes;
    g_device_bytes += (int64_t)bytes;
    return p;
}
void dev_free(void* p) {
    if (!p) return;
    {
        std::lock_guard<std::mutex> lock(g_alloc_mutex);
        auto it = g_sizes.find(p);
        if (it != g_sizes.end()) { g_device_bytes -= (int64_t)it->second; g_sizes.erase(it); }
    }
    cudaFree(p);
}

void* PinnedBuf::get(size_t n) {
    if (n <= bytes) return p;
    if (p) cudaFreeHost(p);
    p = nullptr;
    bytes = n + n / 2 + 4096;
    if (cudaHostAlloc(&p, bytes, cudaHostAllocDefault) != cudaSuccess) {
        cudaGetLastError();
        p = nullptr; bytes = 0;
        throw Error(-3, "pinned host memory exhausted (descriptor staging)");
    }
    return p;
}
PinnedBuf::~PinnedBuf() { if (p) cudaFreeHost(p); }

int find_sector(const Basis& b, int n, int s) {
    int lo = 0, hi = (int)b.size() - 1;
    while (lo <= hi) {
        const int mid = (lo + hi) / 2;
        if (b[mid].n == n && b[mid].s == s) return mid;
        if (b[mid].n < n || (b[mid].n == n && b[mid].s < s)) lo = mid + 1;
        else hi = mid - 1;
    }
    return -1;
}

void make_site_tensor(SiteTensor& t, const Basis& bl, const Basis& br) {
    t.blocks.clear();
    t.lookup.assign(bl.size() * 4, -1);
    int64_t off = 0;
    std::vector<int64_t> offs;
    for (int l = 0; l < (int)bl.size(); ++l)
        for (int s = 0; s < 4; ++s) {
            const int r = find_sector(br, bl[l].n + SITE_QN[s], bl[l].s + SITE_QS[s]);
            if (r < 0) continue;
            t.lookup[l * 4 + s] = (int)t.blocks.size();
            t.blocks.push_back({l, s, r, bl[l].d, br[r].d, pad2(br[r].d), nullptr});
            offs.push_back(off);
            off += (int64_t)bl[l].d * pad2(br[r].d);          // even leading dimension: 16-byte aligned rows
        }
    t.data.alloc((size_t)off);
    t.nnz = off;
    for (size_t j = 0; j < t.blocks.size(); ++j) t.blocks[j].ptr = t.data.p + offs[j];
}

int GemmBatch::add_task(double* C, int ldc, int M, int N, int flags) {
    Task t;
    t.C = C; t.ldc = ldc; t.M = M; t.N = N; t.seg_begin = 0; t.seg_count = 0; t.flags = flags; t.ngemm = 0;
    tasks.push_back(t);
    return (int)tasks.size() - 1;
}
void GemmBatch::add_seg(int task, const double* A, int lda, const double* B, int ldb, int K, int flags,
                        double alpha) {
    Seg s;
    s.A = A; s.B = B; s.lda = lda; s.ldb = ldb; s.K = K; s.flags = flags; s.alpha = alpha;
    segs.push_back(s);
    seg_task.push_back(task);
    if (!(flags & SEG_IDENT_B)) flops += 2.0 * tasks[task].M * (double)tasks[task].N * K;
}

void finalize(GemmBatch& b, GemmLaunch& out, Engine& eng) {
    const int nt = (int)b.tasks.size();
    const size_t ns = b.segs.size();
    // Order within a task: GEMM segments first, sorted by alpha (stable), identity-B segments last.  Empty products
    // (K <= 0 or alpha == 0) are dropped.  Equal alphas adjacent let the bulk-copy kernel keep its accumulators in
    // units of the current alpha and rescale them only when alpha changes (no per-fragment multiply in the main loop).
    // Counting sort of the segments by task (stable), then one small sort per task - tasks in parallel on the host.
    FinalizeScratch& fs = eng.fin;
    std::vector<int>& off = fs.off;
    off.assign((size_t)nt + 1, 0);
    for (size_t j = 0; j < ns; ++j) {
        const Seg& sg = b.segs[j];
        if (!(sg.flags & SEG_IDENT_B) && (sg.K <= 0 || sg.alpha == 0.0)) continue;
        off[(size_t)b.seg_task[j] + 1]++;
    }
    for (int t = 0; t < nt; ++t) off[t + 1] += off[t];
    std::vector<int>& idx = fs.idx;
    std::vector<int>& fill = fs.fill;
    idx.resize((size_t)off[nt]);
    fill.assign(off.begin(), off.end() - 1);
    for (size_t j = 0; j < ns; ++j) {
        const Seg& sg = b.segs[j];
        if (!(sg.flags & SEG_IDENT_B) && (sg.K <= 0 || sg.alpha == 0.0)) continue;
        idx[(size_t)fill[b.seg_task[j]]++] = (int)j;
    }
    const size_t nsorted = (size_t)off[nt];
    Seg* sorted = (Seg*)fs.segs.get(std::max<size_t>(nsorted, 1) * sizeof(Seg));
    std::vector<double>& weight = fs.weight;
    std::vector<int>& ntile = fs.ntile;
    weight.assign(nt, 0.0);
    ntile.assign((size_t)nt + 1, 0);
    int aligned_i = 1;
#pragma omp parallel for schedule(static, 256) reduction(&& : aligned_i) if (nt > 4096)
    for (int t = 0; t < nt; ++t) {
        int* v0 = idx.data() + off[t];
        int* v1 = idx.data() + off[t + 1];
        std::stable_sort(v0, v1, [&](int x, int y) {
            const bool ix = b.segs[x].flags & SEG_IDENT_B, iy = b.segs[y].flags & SEG_IDENT_B;
            if (ix != iy) return iy;
            if (ix) return false;
            return b.segs[x].alpha < b.segs[y].alpha;
        });
        Task& tk = b.tasks[t];
        tk.seg_begin = off[t];
        tk.seg_count = off[t + 1] - off[t];
        tk.ngemm = 0;
        double w = 0.0;
        bool al = true;
        for (int* q = v0; q != v1; ++q) {
            const Seg& sg = b.segs[*q];
            sorted[(size_t)(q - idx.data())] = sg;
            w += sg.K;
            if (sg.flags & SEG_IDENT_B) continue;
            tk.ngemm++;
            // bulk-copy kernel: 16-byte aligned operands, even leading dimensions; a transposed / row operand is read
            // in pieces of pad2(extent) doubles, so the leading dimension must cover them
            if ((((uintptr_t)sg.A) & 15) || (((uintptr_t)sg.B) & 15) || (sg.lda & 1) || (sg.ldb & 1)) al = false;
            const int needA = (sg.flags & SEG_TRANS_A) ? pad2(tk.M) : pad2(sg.K);
            const int needB = (sg.flags & SEG_TRANS_B) ? pad2(sg.K) : pad2(tk.N);
            if (sg.lda < needA || sg.ldb < needB) al = false;
        }
        weight[t] = w;
        aligned_i = aligned_i && al;
        if (tk.M > 0 && tk.N > 0) {
            const int nm = (tk.M + GEMM_BM - 1) / GEMM_BM, nn = (tk.N + GEMM_BN - 1) / GEMM_BN;
            const int pm = std::min(GEMM_BM, (((tk.M + nm - 1) / nm) + 7) & ~7), pn = std::min(GEMM_BN, (((tk.N + nn - 1) / nn) + 7) & ~7);
            ntile[(size_t)t + 1] = ((tk.M + pm - 1) / pm) * ((tk.N + pn - 1) / pn);
        }
    }
    out.aligned = aligned_i != 0;
    // tiles: even split of each extent into ceil(extent / 64) pieces rounded up to the 8-row DMMA fragment (the kernel
    // skips fragments outside [mv x nv], so the padding waste is at the 8 level, not the 64 level); heaviest first
    // (weight = K extent x DMMA fragments of the tile) so that the persistent kernel's dynamic tile counter ends the
    // launch on short tiles
    for (int t = 0; t < nt; ++t) ntile[(size_t)t + 1] += ntile[t];
    const size_t ntl = (size_t)ntile[nt];
    std::vector<Tile>& raw = fs.raw;
    std::vector<double>& tw = fs.tw;
    raw.resize(ntl);
    tw.resize(ntl);
#pragma omp parallel for schedule(static, 256) if (nt > 4096)
    for (int t = 0; t < nt; ++t) {
        const Task& tk = b.tasks[t];
        if (tk.M <= 0 || tk.N <= 0) continue;
        const int nm = (tk.M + GEMM_BM - 1) / GEMM_BM, nn = (tk.N + GEMM_BN - 1) / GEMM_BN;
        const int pm = std::min(GEMM_BM, (((tk.M + nm - 1) / nm) + 7) & ~7), pn = std::min(GEMM_BN, (((tk.N + nn - 1) / nn) + 7) & ~7);
        size_t q = (size_t)ntile[t];
        for (int m0 = 0; m0 < tk.M; m0 += pm)
            for (int n0 = 0; n0 < tk.N; n0 += pn) {
                const int mv = std::min(pm, tk.M - m0), nv = std::min(pn, tk.N - n0);
                raw[q] = {t, m0, n0, mv, nv};
                tw[q] = (weight[t] + 16.0) * ((mv + 7) / 8) * ((nv + 7) / 8);
                ++q;
            }
    }
    if (eng.trace) {                                           // flop and stage histogram by fragments of the busiest warp
        double hf[17] = {0}, hs[17] = {0}, tf = 0, ts = 0;
        for (size_t j = 0; j < raw.size(); ++j) {
            const int fm = (raw[j].mv + 7) / 8, fn = (raw[j].nv + 7) / 8, c = ((fm + 1) / 2) * ((fn + 1) / 2);
            const double kk = weight[raw[j].task];
            hf[c] += 2.0 * kk * raw[j].mv * raw[j].nv; tf += 2.0 * kk * raw[j].mv * raw[j].nv;
            hs[c] += kk / 16.0; ts += kk / 16.0;
        }
        std::fprintf(stderr, "[dmrg trace] tiles=%zu flops%%/stages%% by max warp fragments:", raw.size());
        for (int c = 1; c <= 16; ++c)
            if (hs[c] > 0) std::fprintf(stderr, " %d:%.1f/%.1f", c, 100.0 * hf[c] / tf, 100.0 * hs[c] / ts);
        std::fprintf(stderr, "\n");
    }
    // stable counting sort by weight, heaviest first, on 1/16-octave buckets (the order only balances the load: results do
    // not depend on it, every tile is owned by one CTA and its summation order is the segment order)
    constexpr int NB = 1024;
    std::vector<int>& bucket = fs.bucket;
    std::vector<size_t>& hist = fs.hist;
    bucket.resize(ntl);
    hist.assign(NB + 1, 0);
    for (size_t j = 0; j < ntl; ++j) {
        int q = (int)(std::log2(std::max(tw[j], 1.0)) * 16.0);
        q = NB - 1 - std::min(NB - 1, std::max(0, q));          // heavy tiles -> low bucket
        bucket[j] = q;
        hist[(size_t)q + 1]++;
    }
    for (int q = 0; q < NB; ++q) hist[(size_t)q + 1] += hist[q];
    Tile* tiles = (Tile*)fs.tiles.get(std::max<size_t>(ntl, 1) * sizeof(Tile));
    for (size_t j = 0; j < ntl; ++j) tiles[hist[bucket[j]]++] = raw[j];
    Task* ptasks = (Task*)fs.tasks.get(std::max<size_t>((size_t)nt, 1) * sizeof(Task));
    std::memcpy(ptasks, b.tasks.data(), (size_t)nt * sizeof(Task));
    out.tasks.upload_raw(ptasks, (size_t)nt, eng.stream);
    out.segs.upload_raw(sorted, nsorted, eng.stream);
    out.tiles.upload_raw(tiles, ntl, eng.stream);
    if (!out.counter.p) out.counter.alloc(1);
    out.ntiles = (int)ntl;
    out.flops = b.flops;
    cuda_check(cudaStreamSynchronize(eng.stream), "descriptor upload");   // host vectors die after this call
}
void run(const GemmLaunch& l, Engine& eng, cudaStream_t st) {
    if (l.ntiles == 0) return;
    if (!st) st = eng.stream;
    cudaEvent_t e0 = nullptr, e1 = nullptr;
    if (eng.trace) {                                           // DMRG_B200_TRACE=1: per-launch device time on stderr
        cudaEventCreate(&e0); cudaEventCreate(&e1);
        cudaEventRecord(e0, st);
    }
    if (l.aligned && !eng.force_generic_gemm)
        launch_seg_gemm_tma(l.tasks.p, l.segs.p, l.tiles.p, l.ntiles, l.counter.p, st);
    else
        launch_seg_gemm(l.tasks.p, l.segs.p, l.tiles.p, l.ntiles, st);
    eng.launches++;
    eng.flops_total += l.flops;
    if (eng.trace) {
        cudaEventRecord(e1, st);
        cudaEventSynchronize(e1);
        float ms = 0.f;
        cudaEventElapsedTime(&ms, e0, e1);
        std::fprintf(stderr, "[dmrg trace] gemm %s tiles=%d tasks=%zu segs=%zu flops=%.4e ms=%.3f tflops=%.2f\n",
                     l.aligned ? "tma" : "generic", l.ntiles, l.tasks.n, l.segs.n, l.flops, ms, l.flops / (ms * 1e-3) / 1e12);
        cudaEventDestroy(e0); cudaEventDestroy(e1);
    }
}
void run_once(GemmBatch& b, Engine& eng) {
    if (b.tasks.empty()) return;
    GemmLaunch l;
    const auto t0 = std::chrono::steady_clock::now();
    finalize(b, l, eng);
    if (eng.trace)
        std::fprintf(stderr, "[dmrg trace] finalize tasks=%zu segs=%zu host=%.4f s\n", b.tasks.size(), b.segs.size(),
                     std::chrono::duration<double>(std::chrono::steady_clock::now() - t0).count());
    run(l, eng);
    cuda_check(cudaStreamSynchronize(eng.stream), "grouped GEMM");
    b = GemmBatch();
}
double run_once_ms(GemmBatch& b, Engine& eng) {
    if (b.tasks.empty()) return 0.0;
    GemmLaunch l;
    finalize(b, l, eng);
    cudaEvent_t e0, e1;
    cuda_check(cudaEventCreate(&e0), "event");
    cuda_check(cudaEventCreate(&e1), "event");
    cudaEventRecord(e0, eng.stream);
    run(l, eng);
    cudaEventRecord(e1, eng.stream);
    cuda_check(cudaStreamSynchronize(eng.stream), "grouped GEMM");
    float ms = 0.f;
    cudaEventElapsedTime(&ms, e0, e1);
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    b = GemmBatch();
    return (double)ms;
}

// ---------------------------------------------------------------------------------------------------------------
// Block
// ---------------------------------------------------------------------------------------------------------------
Block::Block(char side_, int b_, int k_, const Basis& basis_, char mode_)
    : side(side_), b(b_), k(k_), mode(mode_), basis(basis_) {}
Block::~Block() {
    if (spill_done) { cudaEventSynchronize(spill_done); cudaEventDestroy(spill_done); }
    for (BlockAlloc& a : allocs) {
        if (a.dev) dev_free(a.dev);
        if (a.host && pool) pool->put(a.host);
    }
    for (void* p : temp_allocs) dev_free(p);
}

// ---------------------------------------------------------------------------------------------------------------
// pinned host pool and spill / restore of a block's storage
// ---------------------------------------------------------------------------------------------------------------
double* HostPool::get(size_t doubles) {
    int best = -1;
    for (size_t j = 0; j < regions.size(); ++j)              // best fit among free regions that are not wastefully large
        if (!regions[j].used && regions[j].doubles >= doubles && regions[j].doubles <= doubles + doubles / 2 + 1024 &&
            (best < 0 || regions[j].doubles < regions[best].doubles)) best = (int)j;
    if (best >= 0) { regions[best].used = true; return regions[best].p; }
    void* p = nullptr;
    const cudaError_t e = cudaHostAlloc(&p, std::max<size_t>(doubles, 1) * sizeof(double), cudaHostAllocDefault);
    if (e != cudaSuccess) {
        cudaGetLastError();
        for (size_t j = 0; j < regions.size();)               // give back the free regions and retry once
            if (!regions[j].used) { cudaFreeHost(regions[j].p); bytes -= (int64_t)regions[j].doubles * 8; regions.erase(regions.begin() + j); }
            else ++j;
        if (cudaHostAlloc(&p, std::max<size_t>(doubles, 1) * sizeof(double), cudaHostAllocDefault) != cudaSuccess) {
            cudaGetLastError();
            throw Error(-3, "pinned host memory exhausted while spilling an environment block");
        }
    }
    regions.push_back({(double*)p, doubles, true});
    bytes += (int64_t)doubles * 8;
    return (double*)p;
}
void HostPool::put(double* p) {
    for (Region& r : regions) if (r.p == p) { r.used = false; return; }
}
void HostPool::clear() {
    for (Region& r : regions) cudaFreeHost(r.p);
    regions.clear();
    bytes = 0;
}

void Block::spill(HostPool& hp, cudaStream_t copy_stream) {
    if (spilled) return;
    if (!temp_allocs.empty()) throw std::logic_error("Block::spill: temporaries alive");
    pool = &hp;
    for (BlockAlloc& a : allocs) {
        if (!a.dev) continue;
        a.host = hp.get(a.doubles);
        cuda_check(cudaMemcpyAsync(a.host, a.dev, a.doubles * sizeof(double), cudaMemcpyDeviceToHost, copy_stream), "spill");
    }
    if (!spill_done) cuda_check(cudaEventCreateWithFlags(&spill_done, cudaEventDisableTiming), "event");
    cuda_check(cudaEventRecord(spill_done, copy_stream), "event record");
    spilled = true;
}
void Block::finish_spill() {
    if (!spilled) return;
    if (spill_done) cuda_check(cudaEventSynchronize(spill_done), "spill wait");
    for (BlockAlloc& a : allocs)
        if (a.dev && a.host) { dev_free(a.dev); a.dev = nullptr; }
}
void Block::restore(cudaStream_t st) {
    if (!spilled) return;
    if (spill_done) cuda_check(cudaEventSynchronize(spill_done), "spill wait");
    for (BlockAlloc& a : allocs) {
        if (!a.host) continue;
        if (!a.dev) {
            a.dev = (double*)dev_alloc(a.doubles * sizeof(double));
            cuda_check(cudaMemcpyAsync(a.dev, a.host, a.doubles * sizeof(double), cudaMemcpyHostToDevice, st), "restore");
        }
    }
    cuda_check(cudaStreamSynchronize(st), "restore");
    for (BlockAlloc& a : allocs)
        if (a.host) { pool->put(a.host); a.host = nullptr; }
    for (Stack& stk : stacks) {                                // device addresses changed: re-derive every pointer
        if (stk.alloc < 0) continue;
        stk.base = allocs[stk.alloc].dev ? allocs[stk.alloc].dev + stk.alloc_off : nullptr;
        const int64_t ld = classes[stk.cls].ld;
        for (size_t r = 0; r < stk.members.size(); ++r) {
            auto it = ops.find(stk.members[r].key());
            if (it != ops.end() && it->second.stack == (int)(&stk - stacks.data()))
                it->second.ptr = stk.base ? stk.base + (int64_t)r * ld : nullptr;
        }
    }
    spilled = false;
}
std::vector<int> Block::inside() const {
    std::vector<int> v;
    if (side == 'L') for (int P = 0; P < 2 * b; ++P) v.push_back(P);
    else for (int P = 2 * b; P < 2 * k; ++P) v.push_back(P);
    return v;
}
std::vector<int> Block::outside() const {
    std::vector<int> v;
    if (side == 'L') for (int P = 2 * b; P < 2 * k; ++P) v.push_back(P);
    else for (int P = 0; P < 2 * b; ++P) v.push_back(P);
    return v;
}
const OpRef& Block::get(const Label& l) const {
    auto it = ops.find(l.key());
    if (it == ops.end()) {
        char buf[96];
        std::snprintf(buf, sizeof buf, "operator (%d,%d,%d,%d) missing on block %c%d", l.kind, l.a, l.b, l.c, side, b);
        throw std::logic_error(buf);
    }
    return it->second;
}
int Block::class_of(int dn, int ds) {
    for (size_t c = 0; c < classes.size(); ++c)
        if (classes[c].dn == dn && classes[c].ds == ds) return (int)c;
    OpClass oc;
    oc.dn = dn; oc.ds = ds;
    const int ns = (int)basis.size();
    oc.out.assign(ns, -1); oc.inv.assign(ns, -1); oc.off.assign(ns, 0);
    int64_t off = 0;
    for (int i = 0; i < ns; ++i) {
        const int o = find_sector(basis, basis[i].n + dn, basis[i].s + ds);
        if (o < 0) continue;
        oc.out[i] = o; oc.inv[o] = i; oc.off[i] = off;
        off += (int64_t)basis[o].d * pad2(basis[i].d);         // even leading dimension: 16-byte aligned rows
    }
    oc.nnz = off; oc.ld = off;
    classes.push_back(oc);
    return (int)classes.size() - 1;
}
int Block::label_class(const Label& l) {
    int dn, ds;
    op_shift(l, dn, ds);
    return class_of(g() * dn, g() * ds);
}
void Block::allocate(const std::vector<Label>& labels, bool temp) {
    std::map<std::pair<int, int>, int> group;                  // (kind, class) -> new stack index
    const size_t first = stacks.size();
    for (const Label& l : labels) {
        if (has(l)) throw std::logic_error("Block::allocate: operator exists");
        const int cls = label_class(l);
        auto key = std::make_pair(l.kind, cls);
        auto it = group.find(key);
        if (it == group.end()) {
            Stack s; s.kind = l.kind; s.cls = cls;
            stacks.push_back(s);
            it = group.emplace(key, (int)stacks.size() - 1).first;
        }
        Stack& st = stacks[it->second];
        OpRef r; r.cls = cls; r.stack = it->second; r.row = (int)st.members.size();
        st.members.push_back(l);
        ops[l.key()] = r;
        if (temp) temp_keys.push_back(l.key());
    }
    int64_t total = 0;
    for (size_t s = first; s < stacks.size(); ++s) total += (int64_t)stacks[s].members.size() * classes[stacks[s].cls].ld;
    if (spilled) throw std::logic_error("Block::allocate on a spilled block");
    double* base = (double*)dev_alloc((size_t)total * sizeof(double));
    int alloc_idx = -1;
    if (base) {
        if (temp) temp_allocs.push_back(base);
        else { BlockAlloc a; a.dev = base; a.doubles = (size_t)total; allocs.push_back(a); alloc_idx = (int)allocs.size() - 1; }
        cuda_check(cudaMemset(base, 0, (size_t)total * sizeof(double)), "memset");   // padding stays finite
    }
    if (!temp) bytes_ += total * 8;
    int64_t off = 0;
    for (size_t s = first; s < stacks.size(); ++s) {
        Stack& st = stacks[s];
        st.alloc = alloc_idx; st.alloc_off = off;
        st.base = base ? base + off : nullptr;
        const int64_t ld = classes[st.cls].ld;
        for (size_t r = 0; r < st.members.size(); ++r) ops[st.members[r].key()].ptr = st.base ? st.base + (int64_t)r * ld : nullptr;
        off += (int64_t)st.members.size() * ld;
    }
}
void Block::drop_temps() {
    for (uint32_t key : temp_keys) ops.erase(key);
    temp_keys.clear();
    for (void* p : temp_allocs) dev_free(p);
    temp_allocs.clear();
}
int64_t Block::bytes() const { return bytes_; }

bool op_block(const Block& blk, const OpRef& op, bool trans, int in, OpBlockView& v) {
    const OpClass& c = blk.classes[op.cls];
    if (!trans) {
        const int o = c.out[in];
        if (o < 0) return false;
        v.out = o; v.ptr = op.ptr + c.off[in]; v.ld = pad2(blk.basis[in].d); v.trans = false;
        v.rows = blk.basis[o].d; v.cols = blk.basis[in].d;
    } else {
        const int j = c.inv[in];                               // stored block j -> in ; transposed maps in -> j
        if (j < 0) return false;
        v.out = j; v.ptr = op.ptr + c.off[j]; v.ld = pad2(blk.basis[j].d); v.trans = true;
        v.rows = blk.basis[j].d; v.cols = blk.basis[in].d;
    }
    return true;
}

static bool block_has_op(const void* blk, const Label& l) { return ((const Block*)blk)->has(l); }
BlockInfo block_info(const Block& b) {
    BlockInfo bi;
    bi.side = b.side; bi.inside = b.inside(); bi.has_op = block_has_op; bi.blk = &b;
    return bi;
}

// ---------------------------------------------------------------------------------------------------------------
// linear combinations of operator stacks as GEMMs:  Dst[n_dst x nnz] (+)= W[n_dst x n_src] Src[n_src x nnz]
// ---------------------------------------------------------------------------------------------------------------
void lincomb(Block& blk, const std::vector<LinSpec>& specs, bool accumulate, Engine& eng) {
    std::map<int, std::vector<const LinSpec*>> by_stack;       // dst stack -> specs
    for (const LinSpec& s : specs) by_stack[blk.get(s.dst).stack].push_back(&s);
    GemmBatch batch;
    std::vector<DevVec<double>> keep;
    for (auto& kv : by_stack) {
        const Stack& ds = blk.stacks[kv.first];
        const OpClass& cls = blk.classes[ds.cls];
        int src_stack = -1;
        for (const LinSpec* s : kv.second)
            for (const LinItem& it : s->items) {
                const int st = it.stack >= 0 ? it.stack : blk.get(it.src).stack;
                if (src_stack >= 0 && st != src_stack) throw std::logic_error("lincomb: sources span two stacks");
                src_stack = st;
            }
        const int n_dst = (int)ds.members.size();
        if (!accumulate && (int)kv.second.size() != n_dst) throw std::logic_error("lincomb: partial overwrite");
        if (cls.nnz == 0) continue;
        if (src_stack < 0) {                                   // nothing to add
            if (!accumulate) cuda_check(cudaMemsetAsync(ds.base, 0, (size_t)n_dst * cls.ld * 8, eng.stream), "memset");
            continue;
        }
        const Stack& ss = blk.stacks[src_stack];
        if (ss.cls != ds.cls) throw std::logic_error("lincomb: class mismatch");
        const int n_src = (int)ss.members.size();
        const int ldw = pad2(n_src);                           // even leading dimension: bulk-copy kernel eligible
        std::vector<double> W((size_t)n_dst * ldw, 0.0);
        for (const LinSpec* s : kv.second) {
            const int r = blk.get(s->dst).row;
            for (const LinItem& it : s->items) W[(size_t)r * ldw + (it.row >= 0 ? it.row : blk.get(it.src).row)] += it.coef;
        }
        keep.emplace_back();
        keep.back().upload(W, eng.stream);
        cuda_check(cudaStreamSynchronize(eng.stream), "lincomb upload");
        // the row length can exceed the int range of Task::N only beyond 2^31 doubles per operator: not reachable
        const int t = batch.add_task(ds.base, (int)cls.ld, n_dst, (int)cls.nnz, accumulate ? TASK_ACCUM : 0);
        batch.add_seg(t, keep.back().p, ldw, ss.base, (int)cls.ld, n_src, 0, 1.0);
    }
    run_once(batch, eng);
}

}  // namespace dmrg
