// C ABI of include/dmrg_b200.h: argument checking, host<->device marshalling, exception -> status translation.
#include <algorithm>
#include <cmath>
#include <cstdlib>
#include <cstring>

#include <omp.h>

#include "../../include/dmrg_b200.h"
#include "core.hpp"

using namespace dmrg;

struct dmrg_ctx {
    Engine eng;
};

namespace dmrg {

void Engine::ensure_left(int i) {
    if (L.find(0) == L.end()) L[0] = empty_block('L', k, mps);
    for (int b = 0; b < i; ++b) {
        if (L.find(b + 1) != L.end()) continue;
        L[b + 1] = grow(*L[b], ham, mps, mode_L(b + 1), *this);
        if (!keep_env_stack && b > 0) L.erase(b);
    }
}
void Engine::ensure_right(int j) {
    if (R.find(k) == R.end()) R[k] = empty_block('R', k, mps);
    for (int b = k; b > j; --b) {
        if (R.find(b - 1) != R.end()) continue;
        R[b - 1] = grow(*R[b], ham, mps, mode_R(b - 1), *this);
        if (!keep_env_stack && b < k) R.erase(b);
    }
}
void Engine::prepare_bond(int i) {
    plan.reset();
    ensure_left(i);
    ensure_right(i + 2);
    plan = build_heff(ham, *L[i], *R[i + 2], i, *this);
}
HeffPlan::~HeffPlan() {
    if (X) X->drop_temps();
    for (cudaEvent_t e : ev_p1) cudaEventDestroy(e);
    for (cudaEvent_t e : ev_p2) cudaEventDestroy(e);
    if (ev_in) cudaEventDestroy(ev_in);
}

}  // namespace dmrg

#define API_BEGIN(ctx)                                   \
    if (!(ctx)) return DMRG_EINVAL;                      \
    Engine& eng = (ctx)->eng;                            \
    try {                                                \
        cuda_check(cudaSetDevice(eng.opt.device_id), "cudaSetDevice");
#define API_END                                          \
    }                                                    \
    catch (const Error& e) { eng.last_error = e.what(); return e.code; }                 \
    catch (const std::bad_alloc&) { eng.last_error = "host memory exhausted"; return DMRG_ENOMEM; } \
    catch (const std::exception& e) { eng.last_error = e.what(); return DMRG_ESTATE; }

static int fail(Engine& eng, int code, const char* msg) {
    eng.last_error = msg;
    return code;
}

extern "C" {

void dmrg_default_options(dmrg_options* o) {
    if (!o) return;
    Options d;
    o->davidson_tol = d.davidson_tol;
    o->davidson_max_iter = d.davidson_max_iter;
    o->davidson_max_subspace = d.davidson_max_subspace;
    o->sv_floor = d.sv_floor;
    o->cluster_rel_gap = d.cluster_rel_gap;
    o->device_id = 0;
    o->keep_env_stack = 1;
    o->workspace_bytes = 0;
    o->hbm_budget_bytes = 0; o->host_budget_bytes = 0; o->host_spill = 0; o->env_stride = 0;
    o->dbss_eps = 0.0; o->dbss_dmin = 0; o->split_k = 0; o->svd_qr = 0; o->host_maps = 0; o->generic_gemm = 0;
    o->eigensolver = 0; o->rdm_split = -1; o->env_stride2 = 0;
}

int dmrg_create(dmrg_ctx** out, int k, int n_elec, int two_sz, const double* h, const double* eri,
                const dmrg_options* opt) {
    if (!out || !h || !eri) return DMRG_EINVAL;
    *out = nullptr;
    if (k < 1 || k > 120 || n_elec < 0 || n_elec > 2 * k) return DMRG_EINVAL;
    if (((n_elec + two_sz) & 1) != 0) return DMRG_EINVAL;
    const int na = (n_elec + two_sz) / 2, nb = (n_elec - two_sz) / 2;
    if (na < 0 || nb < 0 || na > k || nb > k) return DMRG_EINVAL;
    for (int p = 0; p < k; ++p)
        for (int q = 0; q < p; ++q)
            if (std::fabs(h[p * k + q] - h[q * k + p]) > 1e-12) return DMRG_EINVAL;
    dmrg_ctx* ctx = nullptr;
    try {
        ctx = new dmrg_ctx();
        Engine& eng = ctx->eng;
        if (opt) {
            eng.opt.davidson_tol = opt->davidson_tol;
            eng.opt.davidson_max_iter = opt->davidson_max_iter;
            eng.opt.davidson_max_subspace = opt->davidson_max_subspace;
            eng.opt.sv_floor = opt->sv_floor;
            eng.opt.cluster_rel_gap = opt->cluster_rel_gap;
            eng.opt.device_id = opt->device_id;
            eng.opt.workspace_bytes = opt->workspace_bytes;
            eng.keep_env_stack = opt->keep_env_stack != 0;
            eng.opt.hbm_budget_bytes = opt->hbm_budget_bytes; eng.opt.host_budget_bytes = opt->host_budget_bytes;
            eng.opt.host_spill = opt->host_spill; eng.opt.env_stride = opt->env_stride;
            eng.opt.dbss_eps = opt->dbss_eps; eng.opt.dbss_dmin = opt->dbss_dmin;
            eng.opt.split_k = opt->split_k; eng.opt.svd_qr = opt->svd_qr;
            eng.host_maps = opt->host_maps != 0; eng.force_generic_gemm = opt->generic_gemm != 0;
            eng.opt.eigensolver = opt->eigensolver; eng.opt.rdm_split = opt->rdm_split; eng.opt.env_stride2 = opt->env_stride2;
        }
        if (eng.opt.davidson_max_subspace < 2 || eng.opt.davidson_max_subspace > COMBINE_MAX ||
            eng.opt.davidson_max_iter < 1 || !(eng.opt.davidson_tol > 0) || eng.opt.env_stride < 0 ||
            eng.opt.split_k < 0 || eng.opt.split_k > 64 || eng.opt.dbss_eps < 0 || eng.opt.dbss_dmin < 0 ||
            eng.opt.hbm_budget_bytes < 0 || eng.opt.host_budget_bytes < 0 || eng.opt.eigensolver < 0 ||
            eng.opt.eigensolver > 1) { delete ctx; return DMRG_EINVAL; }
        int ndev = 0;
        if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev <= eng.opt.device_id) { delete ctx; return DMRG_ECUDA; }
        cuda_check(cudaSetDevice(eng.opt.device_id), "cudaSetDevice");
        cuda_check(cudaStreamCreateWithFlags(&eng.stream, cudaStreamNonBlocking), "cudaStreamCreate");
        cuda_check(cudaStreamCreateWithFlags(&eng.stream2, cudaStreamNonBlocking), "cudaStreamCreate");
        cuda_check(cudaStreamCreateWithFlags(&eng.copy_stream, cudaStreamNonBlocking), "cudaStreamCreate");
        eng.k = k; eng.n_elec = n_elec; eng.two_sz = two_sz;
        eng.bsw = (k >= 3) ? (k - 3) / 2 : -1;
        eng.ham.k = k;
        eng.ham.h.assign(h, h + (size_t)k * k);
        eng.ham.eri.assign(eri, eri + (size_t)k * k * k * k);
        eng.host_threads = std::max(1, std::min(8, omp_get_num_procs()));
        if (const char* g = std::getenv("DMRG_B200_HOST_THREADS")) eng.host_threads = std::max(1, std::min(64, std::atoi(g)));   // diagnostics: A/B of the host team size
        omp_set_num_threads(eng.host_threads);
        eng.svd = svd_create(eng.stream, eng.opt.svd_qr == 0);
        eng.red_scratch.alloc((size_t)multi_dot_scratch());
        { const char* g = std::getenv("DMRG_B200_TRACE"); eng.trace = g && g[0] == '1'; }   // diagnostics only: per-launch times on stderr
    } catch (...) {
        delete ctx;
        return DMRG_ECUDA;
    }
    *out = ctx;
    return DMRG_OK;
}

int dmrg_destroy(dmrg_ctx* ctx) {
    if (!ctx) return DMRG_EINVAL;
    Engine& eng = ctx->eng;
    cudaSetDevice(eng.opt.device_id);
    eng.invalidate();
    eng.host_pool.clear();
    eng.red_scratch.release();
    eng.mps.sites.clear();
    if (eng.svd) svd_destroy(eng.svd);
    for (SvdWork* w : eng.svd_pool) svd_destroy(w);
    for (cudaStream_t ts : eng.svd_streams) cudaStreamDestroy(ts);
    if (eng.stream) cudaStreamDestroy(eng.stream);
    if (eng.stream2) cudaStreamDestroy(eng.stream2);
    if (eng.copy_stream) cudaStreamDestroy(eng.copy_stream);
    delete ctx;
    return DMRG_OK;
}

const char* dmrg_last_error(const dmrg_ctx* ctx) { return ctx ? ctx->eng.last_error.c_str() : "null context"; }
int64_t dmrg_launch_count(const dmrg_ctx* ctx) { return ctx ? ctx->eng.launches : 0; }
double dmrg_flops_total(const dmrg_ctx* ctx) { return ctx ? ctx->eng.flops_total : 0.0; }
int64_t dmrg_device_bytes(const dmrg_ctx*) { return g_device_bytes; }

int dmrg_mps_import(dmrg_ctx* ctx, const dmrg_mps_blob* b) {
    API_BEGIN(ctx)
    if (!b || !b->bond_ptr || !b->sec_n || !b->sec_2sz || !b->sec_dim || !b->blk_ptr || !b->blk_l || !b->blk_s ||
        !b->blk_off || !b->data || !b->gauge)
        return fail(eng, DMRG_EINVAL, "mps_import: null array");
    const int k = eng.k;
    if (b->k != k || b->n_elec != eng.n_elec || b->two_sz != eng.two_sz)
        return fail(eng, DMRG_EINVAL, "mps_import: k / n_elec / two_sz differ from the context");
    MPS m;
    m.k = k; m.n_elec = eng.n_elec; m.two_sz = eng.two_sz;
    m.bonds.resize(k + 1);
    for (int bd = 0; bd <= k; ++bd) {
        for (int j = b->bond_ptr[bd]; j < b->bond_ptr[bd + 1]; ++j) {
            Sector s{b->sec_n[j], b->sec_2sz[j], b->sec_dim[j]};
            if (s.d < 1) return fail(eng, DMRG_EINVAL, "mps_import: sector of dimension < 1");
            if (!m.bonds[bd].empty()) {
                const Sector& pr = m.bonds[bd].back();
                if (!(pr.n < s.n || (pr.n == s.n && pr.s < s.s))) return fail(eng, DMRG_EINVAL, "mps_import: sectors not sorted");
            }
            m.bonds[bd].push_back(s);
        }
        if (m.bonds[bd].empty()) return fail(eng, DMRG_EINVAL, "mps_import: empty bond");
    }
    if (m.bonds[0].size() != 1 || m.bonds[0][0].n != 0 || m.bonds[0][0].s != 0 || m.bonds[0][0].d != 1 ||
        m.bonds[k].size() != 1 || m.bonds[k][0].n != eng.n_elec || m.bonds[k][0].s != eng.two_sz || m.bonds[k][0].d != 1)
        return fail(eng, DMRG_EINVAL, "mps_import: boundary bonds must be {(0,0,1)} and {(n_elec,two_sz,1)}");
    m.sites.resize(k);
    for (int p = 0; p < k; ++p) {
        SiteTensor& t = m.sites[p];
        make_site_tensor(t, m.bonds[p], m.bonds[p + 1]);
        t.gauge = (char)b->gauge[p];
        if (t.gauge != 'L' && t.gauge != 'R' && t.gauge != 'C') return fail(eng, DMRG_EINVAL, "mps_import: bad gauge flag");
        if (t.nnz) cuda_check(cudaMemsetAsync(t.data.p, 0, (size_t)t.nnz * 8, eng.stream), "memset");
        std::vector<char> seen(t.blocks.size(), 0);
        for (int j = b->blk_ptr[p]; j < b->blk_ptr[p + 1]; ++j) {
            const int l = b->blk_l[j], s = b->blk_s[j];
            if (l < 0 || l >= (int)m.bonds[p].size() || s < 0 || s > 3) return fail(eng, DMRG_EINVAL, "mps_import: bad block index");
            const int idx = t.lookup[l * 4 + s];
            if (idx < 0) return fail(eng, DMRG_EINVAL, "mps_import: block whose right sector does not exist");
            const SiteTensor::Blk& bk = t.blocks[idx];
            seen[idx] = 1;
            cuda_check(cudaMemcpy2DAsync(bk.ptr, (size_t)bk.ld * 8, b->data + b->blk_off[j], (size_t)bk.cols * 8,
                                         (size_t)bk.cols * 8, bk.rows, cudaMemcpyHostToDevice, eng.stream), "mps upload");
        }
    }
    cuda_check(cudaStreamSynchronize(eng.stream), "mps upload");
    eng.invalidate();
    eng.mps = std::move(m);
    eng.have_mps = true;
    return DMRG_OK;
    API_END
}

int dmrg_mps_export(dmrg_ctx* ctx, dmrg_mps_blob* b) {
    API_BEGIN(ctx)
    if (!b) return fail(eng, DMRG_EINVAL, "mps_export: null blob");
    if (!eng.have_mps) return fail(eng, DMRG_ESTATE, "mps_export: no MPS");
    const MPS& m = eng.mps;
    int64_t ns = 0, nb = 0, nd = 0;
    for (auto& bd : m.bonds) ns += (int64_t)bd.size();
    for (auto& t : m.sites)
        for (auto& bk : t.blocks) { nb++; nd += (int64_t)bk.rows * bk.cols; }
    b->k = m.k; b->n_elec = m.n_elec; b->two_sz = m.two_sz;
    if (!b->data) { b->n_sectors = ns; b->n_blocks = nb; b->n_data = nd; return DMRG_OK; }
    if (b->n_sectors < ns || b->n_blocks < nb || b->n_data < nd) return fail(eng, DMRG_EINVAL, "mps_export: arrays too small");
    int32_t* bond_ptr = (int32_t*)b->bond_ptr; int32_t* sn = (int32_t*)b->sec_n; int32_t* ss = (int32_t*)b->sec_2sz;
    int32_t* sd = (int32_t*)b->sec_dim; int32_t* blk_ptr = (int32_t*)b->blk_ptr; int32_t* bl = (int32_t*)b->blk_l;
    int32_t* bs = (int32_t*)b->blk_s; int64_t* bo = (int64_t*)b->blk_off; double* data = (double*)b->data;
    uint8_t* gauge = (uint8_t*)b->gauge;
    int j = 0;
    bond_ptr[0] = 0;
    for (int bd = 0; bd <= m.k; ++bd) {
        for (const Sector& s : m.bonds[bd]) { sn[j] = s.n; ss[j] = s.s; sd[j] = s.d; ++j; }
        bond_ptr[bd + 1] = j;
    }
    j = 0;
    int64_t off = 0;
    blk_ptr[0] = 0;
    for (int p = 0; p < m.k; ++p) {
        for (const auto& bk : m.sites[p].blocks) {
            bl[j] = bk.l; bs[j] = bk.s; bo[j] = off;
            cuda_check(cudaMemcpy2DAsync(data + off, (size_t)bk.cols * 8, bk.ptr, (size_t)bk.ld * 8, (size_t)bk.cols * 8,
                                         bk.rows, cudaMemcpyDeviceToHost, eng.stream), "mps download");
            off += (int64_t)bk.rows * bk.cols;
            ++j;
        }
        blk_ptr[p + 1] = j;
        gauge[p] = (uint8_t)m.sites[p].gauge;
    }
    cuda_check(cudaStreamSynchronize(eng.stream), "mps download");
    b->n_sectors = ns; b->n_blocks = nb; b->n_data = nd;
    return DMRG_OK;
    API_END
}

int dmrg_prepare_bond(dmrg_ctx* ctx, int i) {
    API_BEGIN(ctx)
    if (!eng.have_mps) return fail(eng, DMRG_ESTATE, "prepare_bond: import an MPS first");
    if (i < 0 || i > eng.k - 2) return fail(eng, DMRG_EINVAL, "prepare_bond: bond out of range");
    if (eng.sweep_ready) eng.invalidate();                     // left blocks of a finished sweep are stale
    eng.prepare_bond(i);
    return DMRG_OK;
    API_END
}

static int need_plan(Engine& eng, int i) {
    if (!eng.plan || eng.plan->bond != i) return fail(eng, DMRG_ESTATE, "bond not prepared (call dmrg_prepare_bond)");
    return DMRG_OK;
}

int dmrg_heff_layout(dmrg_ctx* ctx, int i, int64_t* nnz, int32_t* nblocks, dmrg_block* blocks) {
    API_BEGIN(ctx)
    if (int rc = need_plan(eng, i)) return rc;
    const HeffPlan& p = *eng.plan;
    if (nnz) *nnz = p.nnz;
    if (nblocks) *nblocks = (int32_t)p.layout.size();
    if (blocks)
        for (size_t j = 0; j < p.layout.size(); ++j) {
            const PsiBlock& b = p.layout[j];
            blocks[j].l_idx = b.l; blocks[j].s_i = b.ab >> 2; blocks[j].s_j = b.ab & 3; blocks[j].r_idx = b.r;
            blocks[j].rows = b.rows; blocks[j].cols = b.cols; blocks[j].offset = b.off;
        }
    return DMRG_OK;
    API_END
}

int dmrg_heff_apply(dmrg_ctx* ctx, int i, const double* x, double* y, int where, void* cuda_stream) {
    API_BEGIN(ctx)
    if (int rc = need_plan(eng, i)) return rc;
    if (!x || !y) return fail(eng, DMRG_EINVAL, "heff_apply: null vector");
    HeffPlan& p = *eng.plan;
    const size_t bytes = (size_t)p.nnz * 8;
    if (where == DMRG_HOST) {
        cuda_check(cudaMemcpyAsync(p.xbuf.p, x, bytes, cudaMemcpyHostToDevice, eng.stream), "x upload");
        heff_apply(p, p.xbuf.p, p.ybuf.p, eng);
        cuda_check(cudaMemcpyAsync(y, p.ybuf.p, bytes, cudaMemcpyDeviceToHost, eng.stream), "y download");
        cuda_check(cudaStreamSynchronize(eng.stream), "heff_apply");
    } else if (where == DMRG_DEVICE) {
        // order the library stream after the caller's stream and back (events), so device buffers are used in place
        cudaStream_t cs = (cudaStream_t)cuda_stream;
        cudaEvent_t ev;
        cuda_check(cudaEventCreateWithFlags(&ev, cudaEventDisableTiming), "event");
        cuda_check(cudaEventRecord(ev, cs), "event record");
        cuda_check(cudaStreamWaitEvent(eng.stream, ev, 0), "stream wait");
        heff_apply(p, x, y, eng);
        cuda_check(cudaEventRecord(ev, eng.stream), "event record");
        cuda_check(cudaStreamWaitEvent(cs, ev, 0), "stream wait");
        cuda_check(cudaEventDestroy(ev), "event destroy");
    } else return fail(eng, DMRG_EINVAL, "heff_apply: bad `where`");
    return DMRG_OK;
    API_END
}

int dmrg_heff_diag(dmrg_ctx* ctx, int i, double* d, int where, void* cuda_stream) {
    API_BEGIN(ctx)
    if (int rc = need_plan(eng, i)) return rc;
    if (!d) return fail(eng, DMRG_EINVAL, "heff_diag: null vector");
    HeffPlan& p = *eng.plan;
    if (where == DMRG_HOST) {
        heff_diag(p, p.ybuf.p, eng);
        cuda_check(cudaMemcpyAsync(d, p.ybuf.p, (size_t)p.nnz * 8, cudaMemcpyDeviceToHost, eng.stream), "diag download");
        cuda_check(cudaStreamSynchronize(eng.stream), "heff_diag");
    } else if (where == DMRG_DEVICE) {
        // same ordering as dmrg_heff_apply: the library stream starts after the caller's pending work on `d` and the
        // caller's stream continues after the kernel; asynchronous
        cudaStream_t cs = (cudaStream_t)cuda_stream;
        cudaEvent_t ev;
        cuda_check(cudaEventCreateWithFlags(&ev, cudaEventDisableTiming), "event");
        cuda_check(cudaEventRecord(ev, cs), "event record");
        cuda_check(cudaStreamWaitEvent(eng.stream, ev, 0), "stream wait");
        heff_diag(p, d, eng);
        cuda_check(cudaEventRecord(ev, eng.stream), "event record");
        cuda_check(cudaStreamWaitEvent(cs, ev, 0), "stream wait");
        cuda_check(cudaEventDestroy(ev), "event destroy");
    } else return fail(eng, DMRG_EINVAL, "heff_diag: bad `where`");
    return DMRG_OK;
    API_END
}

int dmrg_heff_stats(dmrg_ctx* ctx, int i, double* f_alg, double* f_exec, double* b_alg, int64_t* nterms, int64_t* ngemm) {
    API_BEGIN(ctx)
    if (int rc = need_plan(eng, i)) return rc;
    const HeffPlan& p = *eng.plan;
    if (f_alg) *f_alg = p.f_alg;
    if (f_exec) *f_exec = p.f_exec;
    if (b_alg) *b_alg = p.b_alg;
    if (nterms) *nterms = p.nterms;
    if (ngemm) *ngemm = p.ngemm;
    return DMRG_OK;
    API_END
}

static int run_sweep(Engine& eng, int D, dmrg_sweep_result* result, dmrg_bond_record* records) {
    if (!eng.have_mps) return fail(eng, DMRG_ESTATE, "sweep: import an MPS first");
    if (D < 1) return fail(eng, DMRG_EINVAL, "sweep: D < 1");
    if (eng.k < 2) return fail(eng, DMRG_EINVAL, "sweep: needs at least two sites");
    if (!eng.sweep_ready)
        for (int p = 0; p < eng.k; ++p)
            if (eng.mps.sites[p].gauge == 'L') return fail(eng, DMRG_ESTATE, "sweep: the MPS must be right-canonical");
    std::vector<BondRecord> recs;
    double seconds = 0.0;
    int warnings = 0;
    try {
        warnings = sweep(eng, D, recs, seconds);
    } catch (...) {
        eng.invalidate();                                      // a half-finished sweep leaves no usable environments
        throw;
    }
    if (result) {
        result->energy_last = recs.back().energy;
        result->energy_min = recs[0].energy;
        for (const BondRecord& r : recs) result->energy_min = std::min(result->energy_min, r.energy);
        result->seconds = seconds;
        result->n_records = (int32_t)recs.size();
        result->warnings = warnings;
    }
    if (records)
        for (size_t j = 0; j < recs.size(); ++j) {
            const BondRecord& r = recs[j];
            dmrg_bond_record& o = records[j];
            o.bond = r.bond; o.forward = r.forward; o.energy = r.energy; o.residual = r.residual; o.trunc_err = r.trunc_err;
            o.n_matvec = r.n_matvec; o.kept = r.kept; o.nsectors = r.nsectors; o.converged = r.converged; o.nnz = r.nnz;
            o.f_alg = r.f_alg; o.seconds = r.seconds; o.seconds_matvec = r.seconds_matvec;
        }
    return warnings ? DMRG_ENOCONV : DMRG_OK;
}

int dmrg_sweep(dmrg_ctx* ctx, int D, dmrg_sweep_result* result, dmrg_bond_record* records) {
    API_BEGIN(ctx)
    return run_sweep(eng, D, result, records);
    API_END
}

int dmrg_solve(dmrg_ctx* ctx, int D, double eps_sweep, int max_sweeps, int32_t* n_sweeps, double* energies,
               dmrg_sweep_result* last, dmrg_bond_record* last_records) {
    API_BEGIN(ctx)
    if (!(eps_sweep > 0.0) || max_sweeps < 1 || !n_sweeps) return fail(eng, DMRG_EINVAL, "solve: bad eps_sweep / max_sweeps / n_sweeps");
    *n_sweeps = 0;
    std::vector<double> e;
    dmrg_sweep_result res;
    int rc = DMRG_OK;
    bool met = false;
    while ((int)e.size() < max_sweeps) {
        rc = run_sweep(eng, D, &res, last_records);
        if (rc < 0) return rc;
        e.push_back(res.energy_last);
        if (energies) energies[e.size() - 1] = res.energy_last;
        *n_sweeps = (int32_t)e.size();
        const size_t s = e.size();
        if (s >= 3 && std::fabs(e[s - 2] - e[s - 3]) < eps_sweep && std::fabs(e[s - 1] - e[s - 2]) < eps_sweep) { met = true; break; }
    }
    if (last) *last = res;
    return (!met || rc == DMRG_ENOCONV) ? DMRG_ENOCONV : DMRG_OK;
    API_END
}

int dmrg_sweep_stats(dmrg_ctx* ctx, dmrg_sweep_stats_t* out) {
    API_BEGIN(ctx)
    if (!out) return fail(eng, DMRG_EINVAL, "sweep_stats: null output");
    out->seconds_environments = eng.t_env; out->seconds_restore = eng.t_restore; out->seconds_regrow = eng.t_regrow;
    out->seconds_spill_wait = eng.t_spill_wait; out->seconds_maps = eng.t_plan; out->seconds_davidson = eng.t_davidson;
    out->seconds_matvec = eng.t_matvec; out->seconds_split = eng.t_split; out->seconds_renormalise = eng.t_grow;
    out->bytes_spilled = eng.spill_bytes; out->bytes_restored = eng.restore_bytes;
    out->peak_device_bytes = eng.env_peak_bytes; out->host_pool_bytes = eng.host_pool.bytes;
    out->est_stack_bytes = eng.env_est_total; out->est_max_block_bytes = eng.env_est_max;
    out->env_stride = eng.env_stride; out->host_spill = eng.env_spill ? 1 : 0; out->env_stride2 = eng.env_stride2; out->reserved = 0;
    return DMRG_OK;
    API_END
}

int dmrg_rdm12(dmrg_ctx* ctx, double* gamma, double* Gamma, int where, void* cuda_stream) {
    API_BEGIN(ctx)
    if (!eng.have_mps) return fail(eng, DMRG_ESTATE, "rdm12: import an MPS first");
    if (!gamma) return fail(eng, DMRG_EINVAL, "rdm12: null gamma");
    const size_t k = (size_t)eng.k;
    if (where == DMRG_HOST) {
        rdm12(eng, gamma, Gamma);
    } else if (where == DMRG_DEVICE) {
        // the pass runs on the library stream and ends synchronised; the results are then written to the caller's
        // buffers on the caller's stream (ordered after its pending work on them), and the call returns when they are there
        cudaStream_t cs = (cudaStream_t)cuda_stream;
        std::vector<double> g(k * k), G(Gamma ? k * k * k * k : 0);
        rdm12(eng, g.data(), Gamma ? G.data() : nullptr);
        cuda_check(cudaMemcpyAsync(gamma, g.data(), g.size() * 8, cudaMemcpyHostToDevice, cs), "gamma upload");
        if (Gamma) cuda_check(cudaMemcpyAsync(Gamma, G.data(), G.size() * 8, cudaMemcpyHostToDevice, cs), "Gamma upload");
        cuda_check(cudaStreamSynchronize(cs), "rdm12 upload");
    } else return fail(eng, DMRG_EINVAL, "rdm12: bad `where`");
    return DMRG_OK;
    API_END
}

int dmrg_rdm_stats(dmrg_ctx* ctx, dmrg_rdm_stats_t* out) {
    API_BEGIN(ctx)
    if (!out) return fail(eng, DMRG_EINVAL, "rdm_stats: null output");
    out->seconds = eng.rdm_seconds; out->seconds_host = eng.rdm_host_seconds; out->seconds_renormalise = eng.rdm_grow_seconds;
    out->bytes_streamed = eng.rdm_bytes; out->flops = eng.rdm_flops;
    out->stream_bytes = eng.rdm_stream_bytes; out->stream_seconds = eng.rdm_stream_ms * 1e-3;
    out->gemm_seconds = eng.rdm_gemm_ms * 1e-3;
    return DMRG_OK;
    API_END
}

int dmrg_stack_dots(const double* S, int64_t lds, int nrows, const double* M, int64_t ldm, int nc, int64_t K, double* E,
                    int ldE, double* ms, void* cuda_stream) {
    if (!S || !M || !E || nrows < 1 || nc < 1 || nc > 8 || K < 0 || (lds & 1) || (ldm & 1) || ldE < nc) return DMRG_EINVAL;
    if ((((uintptr_t)S) & 15) || (((uintptr_t)M) & 15)) return DMRG_EINVAL;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    double* scratch = nullptr;
    const int64_t need = stack_dots_scratch(nrows, nc, K);
    if (cudaMalloc(&scratch, sizeof(double) * (size_t)std::max<int64_t>(need, 1)) != cudaSuccess) { cudaGetLastError(); return DMRG_ENOMEM; }
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0); cudaEventCreate(&e1);
    cudaEventRecord(e0, st);
    launch_stack_dots(S, lds, nrows, M, ldm, nc, K, E, ldE, scratch, st);
    cudaEventRecord(e1, st);
    const cudaError_t err = cudaStreamSynchronize(st);
    float t = 0.f;
    cudaEventElapsedTime(&t, e0, e1);
    if (ms) *ms = t;
    cudaEventDestroy(e0); cudaEventDestroy(e1);
    cudaFree(scratch);
    return (err == cudaSuccess && cudaGetLastError() == cudaSuccess) ? DMRG_OK : DMRG_ECUDA;
}

int dmrg_grouped_gemm(int ntasks, const int64_t* c_ptr, const int32_t* ldc, const int32_t* m, const int32_t* n,
                      const int32_t* seg_begin, const int32_t* seg_count, const int32_t* task_flags, int nsegs,
                      const int64_t* a_ptr, const int64_t* b_ptr, const int32_t* lda, const int32_t* ldb,
                      const int32_t* kk, const int32_t* seg_flags, const double* alpha, int generic_kernel,
                      double* kernel_ms, void* cuda_stream) {
    if (ntasks < 0 || nsegs < 0) return DMRG_EINVAL;
    try {
        Engine tmp;                                            // only the stream and the launch counter are used
        tmp.stream = (cudaStream_t)cuda_stream;
        tmp.force_generic_gemm = generic_kernel != 0;
        GemmBatch b;
        for (int t = 0; t < ntasks; ++t) {
            if (seg_begin[t] < 0 || seg_count[t] < 0 || seg_begin[t] + seg_count[t] > nsegs) return DMRG_EINVAL;
            b.add_task((double*)(uintptr_t)c_ptr[t], ldc[t], m[t], n[t], task_flags[t]);
            for (int s = seg_begin[t]; s < seg_begin[t] + seg_count[t]; ++s)
                b.add_seg(t, (const double*)(uintptr_t)a_ptr[s], lda[s], (const double*)(uintptr_t)b_ptr[s], ldb[s], kk[s],
                          seg_flags[s], alpha[s]);
        }
        if (!b.tasks.empty()) {
            GemmLaunch l;
            finalize(b, l, tmp);
            cudaEvent_t e0, e1;
            cuda_check(cudaEventCreate(&e0), "event");
            cuda_check(cudaEventCreate(&e1), "event");
            cudaEventRecord(e0, tmp.stream);
            run(l, tmp);
            cudaEventRecord(e1, tmp.stream);
            cuda_check(cudaStreamSynchronize(tmp.stream), "grouped GEMM");
            float ms = 0.f;
            cudaEventElapsedTime(&ms, e0, e1);
            if (kernel_ms) *kernel_ms = ms;
            cudaEventDestroy(e0);
            cudaEventDestroy(e1);
        }
    } catch (const Error& e) { return e.code; }
    catch (...) { return DMRG_ECUDA; }
    return DMRG_OK;
}

}  // extern "C"
