// Davidson driver, decomposition + truncation, and the two-site sweep (DESIGN.md
// "Algorithm" step 4 and readings S12-S18).  Vectors live on the device; the host sees O(subspace) scalars per
// iteration and the singular values of each bond.
#include <algorithm>
#include <chrono>
#include <cstdio>
#include <cstdlib>
#include <cmath>

#include <omp.h>

#include "core.hpp"

namespace dmrg {

// ---------------------------------------------------------------------------------------------------------------
// tiny symmetric eigenproblem of the Rayleigh-Ritz step (host, cyclic Jacobi; m <= 32)
// ---------------------------------------------------------------------------------------------------------------
static void jacobi_eigh(std::vector<double> a, int m, std::vector<double>& w, std::vector<double>& v) {
    v.assign((size_t)m * m, 0.0);
    for (int i = 0; i < m; ++i) v[(size_t)i * m + i] = 1.0;
    double prev_off = 1e300;
    for (int sweep = 0; sweep < 100; ++sweep) {
        double off = 0.0, diag = 0.0;
        for (int i = 0; i < m; ++i)
            for (int j = 0; j < m; ++j) (i == j ? diag : off) += a[(size_t)i * m + j] * a[(size_t)i * m + j];
        if (off <= 1e-32 * (diag + off) || off == 0.0) break;
        // rounding floor: the off-diagonal norm of an m x m matrix cannot go below ~m eps ||a||; once it is there and has
        // stopped shrinking, further sweeps only burn host time (they were ~1 ms per Davidson iteration at m = 20)
        if (off <= 1e-26 * (diag + off) && off >= 0.25 * prev_off) break;
        prev_off = off;
        for (int p = 0; p < m; ++p)
            for (int q = p + 1; q < m; ++q) {
                const double apq = a[(size_t)p * m + q];
                if (apq == 0.0) continue;
                const double zeta = (a[(size_t)q * m + q] - a[(size_t)p * m + p]) / (2.0 * apq);
                const double t = (zeta >= 0 ? 1.0 : -1.0) / (std::fabs(zeta) + std::sqrt(1.0 + zeta * zeta));
                const double c = 1.0 / std::sqrt(1.0 + t * t), s = c * t;
                for (int r = 0; r < m; ++r) {
                    const double x = a[(size_t)r * m + p], y = a[(size_t)r * m + q];
                    a[(size_t)r * m + p] = c * x - s * y; a[(size_t)r * m + q] = s * x + c * y;
                }
                for (int r = 0; r < m; ++r) {
                    const double x = a[(size_t)p * m + r], y = a[(size_t)q * m + r];
                    a[(size_t)p * m + r] = c * x - s * y; a[(size_t)q * m + r] = s * x + c * y;
                }
                for (int r = 0; r < m; ++r) {
                    const double x = v[(size_t)r * m + p], y = v[(size_t)r * m + q];
                    v[(size_t)r * m + p] = c * x - s * y; v[(size_t)r * m + q] = s * x + c * y;
                }
            }
    }
    w.resize(m);
    for (int i = 0; i < m; ++i) w[i] = a[(size_t)i * m + i];
}

// ---------------------------------------------------------------------------------------------------------------
// Davidson (reading S13): single root, diagonal preconditioner, twice-applied Gram-Schmidt, restart
// ---------------------------------------------------------------------------------------------------------------
DavidsonResult davidson(HeffPlan& p, double* x_dev, Engine& eng) {
    const int64_t n = p.nnz;
    const int maxsub = eng.opt.davidson_max_subspace;
    cudaStream_t st = eng.stream;
    DevVec<double> V, W, diag, r, scal;
    V.alloc((size_t)maxsub * n); W.alloc((size_t)maxsub * n); diag.alloc((size_t)n); r.alloc((size_t)n);
    scal.alloc(COMBINE_MAX + 2);
    std::vector<double> hs((size_t)COMBINE_MAX + 2);
    auto dots = [&](const double* x, const double* Y, int m) {          // -> hs[0..m)
        launch_multi_dot(x, Y, n, m, n, scal.p, eng.red_scratch.p, st);
        eng.launches += 2;
        cuda_check(cudaMemcpyAsync(hs.data(), scal.p, sizeof(double) * m, cudaMemcpyDeviceToHost, st), "dots");
        cuda_check(cudaStreamSynchronize(st), "dots");
    };
    cudaEvent_t e0, e1;
    cuda_check(cudaEventCreate(&e0), "event"); cuda_check(cudaEventCreate(&e1), "event");
    double ms_matvec = 0.0;
    auto matvec = [&](const double* v, double* w) {
        cuda_check(cudaEventRecord(e0, st), "event");
        heff_apply(p, v, w, eng);
        cuda_check(cudaEventRecord(e1, st), "event");
        cuda_check(cudaEventSynchronize(e1), "event");
        float ms = 0.f;
        cuda_check(cudaEventElapsedTime(&ms, e0, e1), "event");
        ms_matvec += ms;
    };
    heff_diag(p, diag.p, eng);
    dots(x_dev, x_dev, 1);
    if (!(hs[0] > 0.0)) throw Error(-2, "davidson: zero initial guess");
    cuda_check(cudaMemcpyAsync(V.p, x_dev, (size_t)n * 8, cudaMemcpyDeviceToDevice, st), "copy");
    launch_scale(1.0 / std::sqrt(hs[0]), V.p, n, st); eng.launches++;
    matvec(V.p, W.p);
    int m = 1, nmv = 1;
    std::vector<double> H((size_t)maxsub * maxsub, 0.0);
    dots(W.p, V.p, 1);
    H[0] = hs[0];
    DavidsonResult res{0.0, 1e300, 0, false, 0.0};
    std::vector<double> w, s, coef(COMBINE_MAX);
    for (int iter = 0; iter < eng.opt.davidson_max_iter; ++iter) {
        std::vector<double> hm((size_t)m * m);
        for (int i = 0; i < m; ++i)
            for (int j = 0; j < m; ++j) hm[(size_t)i * m + j] = H[(size_t)i * maxsub + j];
        jacobi_eigh(hm, m, w, s);
        int lo = 0;
        for (int i = 1; i < m; ++i) if (w[i] < w[lo]) lo = i;
        const double theta = w[lo];
        for (int i = 0; i < m; ++i) coef[i] = s[(size_t)i * m + lo];
        // r = sum s_i W_i - theta sum s_i V_i
        launch_combine(r.p, 0.0, W.p, n, m, coef.data(), n, st);
        std::vector<double> c2(m);
        for (int i = 0; i < m; ++i) c2[i] = -theta * coef[i];
        launch_combine(r.p, 1.0, V.p, n, m, c2.data(), n, st);
        eng.launches += 2;
        dots(r.p, r.p, 1);
        const double rn = std::sqrt(hs[0]);
        res.theta = theta; res.residual = rn; res.n_matvec = nmv;
        const bool done = rn <= eng.opt.davidson_tol;
        if (done || iter + 1 == eng.opt.davidson_max_iter) {
            res.converged = done;
            launch_combine(x_dev, 0.0, V.p, n, m, coef.data(), n, st); eng.launches++;
            dots(x_dev, x_dev, 1);
            launch_scale(1.0 / std::sqrt(hs[0]), x_dev, n, st); eng.launches++;
            break;
        }
        // preconditioned correction (into r)
        launch_precond(r.p, diag.p, theta, 1e-8, r.p, n, st); eng.launches++;
        if (m >= maxsub) {                                                  // restart with the Ritz pair
            DevVec<double> u, hu;
            u.alloc((size_t)n); hu.alloc((size_t)n);
            launch_combine(u.p, 0.0, V.p, n, m, coef.data(), n, st);
            launch_combine(hu.p, 0.0, W.p, n, m, coef.data(), n, st);
            eng.launches += 2;
            dots(u.p, u.p, 1);
            const double inv = 1.0 / std::sqrt(hs[0]);
            launch_scale(inv, u.p, n, st); launch_scale(inv, hu.p, n, st); eng.launches += 2;
            cuda_check(cudaMemcpyAsync(V.p, u.p, (size_t)n * 8, cudaMemcpyDeviceToDevice, st), "copy");
            cuda_check(cudaMemcpyAsync(W.p, hu.p, (size_t)n * 8, cudaMemcpyDeviceToDevice, st), "copy");
            cuda_check(cudaStreamSynchronize(st), "restart");
            m = 1;
            dots(W.p, V.p, 1);
            H[0] = hs[0];
        }
        for (int gs = 0; gs < 2; ++gs) {                                    // t -= V (V^T t), twice
            dots(r.p, V.p, m);
            std::vector<double> c(m);
            for (int i = 0; i < m; ++i) c[i] = -hs[i];
            launch_combine(r.p, 1.0, V.p, n, m, c.data(), n, st); eng.launches++;
        }
        dots(r.p, r.p, 1);
        const double nt = std::sqrt(hs[0]);
        if (nt < 1e-14) {                                                   // subspace exhausted
            launch_combine(x_dev, 0.0, V.p, n, m, coef.data(), n, st); eng.launches++;
            dots(x_dev, x_dev, 1);
            launch_scale(1.0 / std::sqrt(hs[0]), x_dev, n, st); eng.launches++;
            break;
        }
        double* vnew = V.p + (size_t)m * n;
        double* wnew = W.p + (size_t)m * n;
        cuda_check(cudaMemcpyAsync(vnew, r.p, (size_t)n * 8, cudaMemcpyDeviceToDevice, st), "copy");
        launch_scale(1.0 / nt, vnew, n, st); eng.launches++;
        matvec(vnew, wnew);
        ++nmv;
        dots(wnew, V.p, m + 1);                                             // new column of V^T W
        for (int i = 0; i <= m; ++i) { H[(size_t)i * maxsub + m] = hs[i]; H[(size_t)m * maxsub + i] = hs[i]; }
        ++m;
    }
    cuda_check(cudaStreamSynchronize(st), "davidson");
    cudaEventDestroy(e0); cudaEventDestroy(e1);
    res.n_matvec = nmv;
    res.seconds_matvec = ms_matvec * 1e-3;
    return res;
}

// ---------------------------------------------------------------------------------------------------------------
// Lanczos (PAPER.md:179 names it beside Davidson; reading S33): full re-orthogonalisation (twice) against the stored
// Krylov vectors, Rayleigh-Ritz on the tridiagonal matrix, residual norm beta_{m+1} |s_m|, restart from the Ritz vector
// ---------------------------------------------------------------------------------------------------------------
DavidsonResult lanczos(HeffPlan& p, double* x_dev, Engine& eng) {
    const int64_t n = p.nnz;
    const int maxsub = eng.opt.davidson_max_subspace;
    cudaStream_t st = eng.stream;
    DevVec<double> V, w, scal;
    V.alloc((size_t)maxsub * n); w.alloc((size_t)n);
    scal.alloc(COMBINE_MAX + 2);
    std::vector<double> hs((size_t)COMBINE_MAX + 2);
    auto dots = [&](const double* x, const double* Y, int m) {          // -> hs[0..m)
        launch_multi_dot(x, Y, n, m, n, scal.p, eng.red_scratch.p, st);
        eng.launches += 2;
        cuda_check(cudaMemcpyAsync(hs.data(), scal.p, sizeof(double) * m, cudaMemcpyDeviceToHost, st), "dots");
        cuda_check(cudaStreamSynchronize(st), "dots");
    };
    cudaEvent_t e0, e1;
    cuda_check(cudaEventCreate(&e0), "event"); cuda_check(cudaEventCreate(&e1), "event");
    double ms_matvec = 0.0;
    auto matvec = [&](const double* v, double* y) {
        cuda_check(cudaEventRecord(e0, st), "event");
        heff_apply(p, v, y, eng);
        cuda_check(cudaEventRecord(e1, st), "event");
        cuda_check(cudaEventSynchronize(e1), "event");
        float ms = 0.f;
        cuda_check(cudaEventElapsedTime(&ms, e0, e1), "event");
        ms_matvec += ms;
    };
    dots(x_dev, x_dev, 1);
    if (!(hs[0] > 0.0)) throw Error(-2, "lanczos: zero initial guess");
    cuda_check(cudaMemcpyAsync(V.p, x_dev, (size_t)n * 8, cudaMemcpyDeviceToDevice, st), "copy");
    launch_scale(1.0 / std::sqrt(hs[0]), V.p, n, st); eng.launches++;
    int m = 1, nmv = 0;
    std::vector<double> alphas, betas, ev, es, coef(COMBINE_MAX);
    DavidsonResult res{0.0, 1e300, 0, false, 0.0};
    for (int iter = 0; iter < eng.opt.davidson_max_iter; ++iter) {
        double* vlast = V.p + (size_t)(m - 1) * n;
        matvec(vlast, w.p);
        ++nmv;
        dots(w.p, vlast, 1);
        alphas.push_back(hs[0]);
        if (m > 1) { const double c[2] = {-betas.back(), -alphas.back()}; launch_combine(w.p, 1.0, V.p + (size_t)(m - 2) * n, n, 2, c, n, st); }
        else { const double c[1] = {-alphas.back()}; launch_combine(w.p, 1.0, vlast, n, 1, c, n, st); }
        eng.launches++;
        for (int gs = 0; gs < 2; ++gs) {
            dots(w.p, V.p, m);
            std::vector<double> c(m);
            for (int i = 0; i < m; ++i) c[i] = -hs[i];
            launch_combine(w.p, 1.0, V.p, n, m, c.data(), n, st); eng.launches++;
        }
        dots(w.p, w.p, 1);
        const double beta = std::sqrt(std::max(hs[0], 0.0));
        std::vector<double> T((size_t)m * m, 0.0);
        for (int i = 0; i < m; ++i) {
            T[(size_t)i * m + i] = alphas[i];
            if (i + 1 < m) { T[(size_t)i * m + i + 1] = betas[i]; T[(size_t)(i + 1) * m + i] = betas[i]; }
        }
        jacobi_eigh(T, m, ev, es);
        int lo = 0;
        for (int i = 1; i < m; ++i) if (ev[i] < ev[lo]) lo = i;
        for (int i = 0; i < m; ++i) coef[i] = es[(size_t)i * m + lo];
        const double rn = std::fabs(beta * coef[m - 1]);
        res.theta = ev[lo]; res.residual = rn; res.n_matvec = nmv;
        const bool done = rn <= eng.opt.davidson_tol;
        if (done || beta < 1e-14 || iter + 1 == eng.opt.davidson_max_iter) {
            res.converged = done;
            launch_combine(x_dev, 0.0, V.p, n, m, coef.data(), n, st); eng.launches++;
            dots(x_dev, x_dev, 1);
            launch_scale(1.0 / std::sqrt(hs[0]), x_dev, n, st); eng.launches++;
            break;
        }
        if (m >= maxsub) {                                                  // restart from the Ritz vector
            launch_combine(w.p, 0.0, V.p, n, m, coef.data(), n, st); eng.launches++;
            dots(w.p, w.p, 1);
            cuda_check(cudaMemcpyAsync(V.p, w.p, (size_t)n * 8, cudaMemcpyDeviceToDevice, st), "copy");
            launch_scale(1.0 / std::sqrt(hs[0]), V.p, n, st); eng.launches++;
            m = 1; alphas.clear(); betas.clear();
            continue;
        }
        betas.push_back(beta);
        cuda_check(cudaMemcpyAsync(V.p + (size_t)m * n, w.p, (size_t)n * 8, cudaMemcpyDeviceToDevice, st), "copy");
        launch_scale(1.0 / beta, V.p + (size_t)m * n, n, st); eng.launches++;
        ++m;
    }
    cuda_check(cudaStreamSynchronize(st), "lanczos");
    cudaEventDestroy(e0); cudaEventDestroy(e1);
    res.n_matvec = nmv;
    res.seconds_matvec = ms_matvec * 1e-3;
    return res;
}

// ---------------------------------------------------------------------------------------------------------------
// theta[l, a, b, r] = sum_m T_i[(l,a)][:, m] T_{i+1}[(m,b)][m, :]      (prediction of the next guess, reading S16)
// ---------------------------------------------------------------------------------------------------------------
void two_site_tensor(const MPS& mps, int i, const HeffPlan& p, double* theta_dev, Engine& eng) {
    GemmBatch b;
    const SiteTensor& ta = mps.sites[i];
    const SiteTensor& tb = mps.sites[i + 1];
    for (const PsiBlock& blk : p.layout) {
        const int t = b.add_task(theta_dev + blk.off, blk.cols, blk.rows, blk.cols, 0);
        const SiteTensor::Blk* x = ta.get(blk.l, blk.ab >> 2);
        if (!x) continue;
        const SiteTensor::Blk* y = tb.get(x->r, blk.ab & 3);
        if (!y) continue;
        b.add_seg(t, x->ptr, x->ld, y->ptr, y->ld, x->cols, 0, 1.0);
    }
    run_once(b, eng);
}

// ---------------------------------------------------------------------------------------------------------------
// SVD per enlarged-left sector and global top-D selection that never cuts a near-degenerate cluster (reading S14)
// ---------------------------------------------------------------------------------------------------------------
void split_theta(MPS& mps, int i, const HeffPlan& p, const double* theta, int D, bool forward, Engine& eng,
                 double& trunc_err, int& kept, int& nsectors) {
    cudaStream_t st = eng.stream;
    const Basis& bl = mps.bonds[i];
    const Basis& br = mps.bonds[i + 2];
    struct Sec {
        int n, s;
        std::vector<std::pair<int, int>> rows, cols;          // (l, a) and (b, r)
        std::vector<int> roff, coff;
        int nr = 0, nc = 0, rk = 0;
        DevVec<double> M, U, S, Vt;
        std::vector<double> sv;
        int keep = 0;
    };
    std::map<std::pair<int, int>, Sec> secs;
    for (const PsiBlock& b : p.layout) {
        const int a = b.ab >> 2, bb = b.ab & 3;
        const auto q = std::make_pair(bl[b.l].n + SITE_QN[a], bl[b.l].s + SITE_QS[a]);
        Sec& sc = secs[q];
        sc.n = q.first; sc.s = q.second;
        if (std::find(sc.rows.begin(), sc.rows.end(), std::make_pair(b.l, a)) == sc.rows.end()) sc.rows.push_back({b.l, a});
        if (std::find(sc.cols.begin(), sc.cols.end(), std::make_pair(bb, b.r)) == sc.cols.end()) sc.cols.push_back({bb, b.r});
    }
    // norm of theta (the kept state is rescaled to unit norm afterwards)
    DevVec<double> scal;
    scal.alloc(1);
    launch_multi_dot(theta, theta, p.nnz, 1, p.nnz, scal.p, eng.red_scratch.p, st); eng.launches += 2;
    double nrm2 = 0.0;
    cuda_check(cudaMemcpyAsync(&nrm2, scal.p, 8, cudaMemcpyDeviceToHost, st), "norm");
    cuda_check(cudaStreamSynchronize(st), "norm");
    const double inv_nrm = 1.0 / std::sqrt(nrm2);
    struct PoolItem { double sv; int sec, j; };
    std::vector<PoolItem> pool;
    std::vector<Sec*> order;
    for (auto& kv : secs) {                                    // std::map iterates in ascending (n, s)
        Sec& sc = kv.second;
        std::sort(sc.rows.begin(), sc.rows.end());
        std::sort(sc.cols.begin(), sc.cols.end());
        for (auto& rc : sc.rows) { sc.roff.push_back(sc.nr); sc.nr += bl[rc.first].d; }
        for (auto& cc : sc.cols) { sc.coff.push_back(sc.nc); sc.nc += br[cc.second].d; }
        sc.rk = std::min(sc.nr, sc.nc);
        order.push_back(&sc);
    }
    // The sector SVDs are independent and individually too small to fill the device: a few host threads run them
    // concurrently, each on its own stream and cuSOLVER handle (theta is complete: Davidson ended synchronised).
    // Largest sectors first.
    const int nthreads = eng.host_threads;
    eng.ensure_svd_pool(nthreads);
    std::vector<int> by_size(order.size());
    for (size_t j = 0; j < order.size(); ++j) by_size[j] = (int)j;
    std::stable_sort(by_size.begin(), by_size.end(), [&](int x, int y) {
        return (double)order[x]->nr * order[x]->nc * order[x]->rk > (double)order[y]->nr * order[y]->nc * order[y]->rk; });
    std::string err;
    int64_t nlaunch = 0;
#pragma omp parallel for schedule(dynamic, 1) num_threads(nthreads) reduction(+ : nlaunch)
    for (long jj = 0; jj < (long)by_size.size(); ++jj) {
        try {
            const int tid = omp_get_thread_num();
            cudaStream_t ts = eng.svd_streams[tid];
            cuda_check(cudaSetDevice(eng.opt.device_id), "cudaSetDevice");
            Sec& sc = *order[by_size[jj]];
            sc.M.alloc((size_t)sc.nr * sc.nc);
            cuda_check(cudaMemsetAsync(sc.M.p, 0, (size_t)sc.nr * sc.nc * 8, ts), "memset");
            for (size_t ri = 0; ri < sc.rows.size(); ++ri)
                for (size_t ci = 0; ci < sc.cols.size(); ++ci) {
                    const int ix = p.lookup[sc.rows[ri].first * 16 + sc.rows[ri].second * 4 + sc.cols[ci].first];
                    if (ix < 0 || p.layout[ix].r != sc.cols[ci].second) continue;
                    const PsiBlock& b = p.layout[ix];
                    launch_copy2d(sc.M.p + (size_t)sc.roff[ri] * sc.nc + sc.coff[ci], sc.nc, theta + b.off, b.cols, b.rows,
                                  b.cols, inv_nrm, nullptr, nullptr, ts);
                    nlaunch++;
                }
            sc.U.alloc((size_t)sc.nr * sc.rk); sc.S.alloc((size_t)sc.rk); sc.Vt.alloc((size_t)sc.rk * sc.nc);
            svd_rowmajor(eng.svd_pool[tid], sc.M.p, sc.nr, sc.nc, sc.U.p, sc.S.p, sc.Vt.p, ts);
            sc.sv.resize(sc.rk);
            cuda_check(cudaMemcpyAsync(sc.sv.data(), sc.S.p, (size_t)sc.rk * 8, cudaMemcpyDeviceToHost, ts), "sv");
            cuda_check(cudaStreamSynchronize(ts), "sv");
            sc.M.release();
        } catch (const std::exception& e) {
#pragma omp critical
            err = e.what();
        }
    }
    if (!err.empty()) throw Error(-4, "split: " + err);
    eng.launches += nlaunch;
    for (size_t j = 0; j < order.size(); ++j)
        for (int q = 0; q < order[j]->rk; ++q) pool.push_back({order[j]->sv[q], (int)j, q});
    std::vector<int> idx(pool.size());
    for (size_t t = 0; t < idx.size(); ++t) idx[t] = (int)t;
    std::stable_sort(idx.begin(), idx.end(), [&](int x, int y) { return pool[x].sv > pool[y].sv; });
    int count = 0;
    for (int t : idx) if (pool[t].sv > eng.opt.sv_floor) ++count;
    // kept states: fixed D (reading S14) or dynamic block state selection (reading S32: the
    // fewest states with discarded weight <= dbss_eps, clamped to [dbss_dmin, D]); a cut never splits a near-degenerate
    // cluster - under DBSS it moves up to the end of the cluster when the cap allows, otherwise (and for fixed D) down
    const int cap = std::min(D, count);
    auto inside = [&](int mm) { return mm > 0 && mm < count && pool[idx[mm]].sv >= (1.0 - eng.opt.cluster_rel_gap) * pool[idx[mm - 1]].sv; };
    int m = cap;
    bool chosen = false;
    if (eng.opt.dbss_eps > 0.0) {
        double kw = 0.0;
        m = 0;
        while (m < count && 1.0 - kw > eng.opt.dbss_eps) { kw += pool[idx[m]].sv * pool[idx[m]].sv; ++m; }
        m = std::min(std::max(m, eng.opt.dbss_dmin), cap);
        int up = m;
        while (inside(up)) ++up;
        if (up <= cap) { m = up; chosen = true; }
    }
    if (!chosen) {
        const int m0 = m;
        while (inside(m)) --m;
        if (m == 0) m = m0;
    }
    if (m == 0) throw Error(-2, "split: the two-site state has no singular value above the floor");
    double kept_w = 0.0;
    for (int t = 0; t < m; ++t) { kept_w += pool[idx[t]].sv * pool[idx[t]].sv; order[pool[idx[t]].sec]->keep++; }
    trunc_err = std::max(0.0, 1.0 - kept_w);
    const double scale = 1.0 / std::sqrt(kept_w);
    kept = m;
    Basis mid;
    for (Sec* sc : order) if (sc->keep > 0) mid.push_back({sc->n, sc->s, sc->keep});
    nsectors = (int)mid.size();
    // new site tensors
    SiteTensor A, B;
    make_site_tensor(A, bl, mid);
    make_site_tensor(B, mid, br);
    if (A.nnz) cuda_check(cudaMemsetAsync(A.data.p, 0, (size_t)A.nnz * 8, st), "memset");
    if (B.nnz) cuda_check(cudaMemsetAsync(B.data.p, 0, (size_t)B.nnz * 8, st), "memset");
    for (Sec* sc : order) {
        if (sc->keep == 0) continue;
        const int mi = find_sector(mid, sc->n, sc->s);
        const int nk = sc->keep;
        for (size_t ri = 0; ri < sc->rows.size(); ++ri) {
            const SiteTensor::Blk* blk = A.get(sc->rows[ri].first, sc->rows[ri].second);
            if (!blk || blk->r != mi) throw std::logic_error("split: A block missing");
            launch_copy2d(blk->ptr, blk->ld, sc->U.p + (size_t)sc->roff[ri] * sc->rk, sc->rk, blk->rows, nk,
                          forward ? 1.0 : scale, nullptr, forward ? nullptr : sc->S.p, st);
            eng.launches++;
        }
        for (size_t ci = 0; ci < sc->cols.size(); ++ci) {
            const SiteTensor::Blk* blk = B.get(mi, sc->cols[ci].first);
            if (!blk || blk->r != sc->cols[ci].second) throw std::logic_error("split: B block missing");
            launch_copy2d(blk->ptr, blk->ld, sc->Vt.p + sc->coff[ci], sc->nc, nk, blk->cols, forward ? scale : 1.0,
                          forward ? sc->S.p : nullptr, nullptr, st);
            eng.launches++;
        }
    }
    cuda_check(cudaStreamSynchronize(st), "split");
    A.gauge = forward ? 'L' : 'C';
    B.gauge = forward ? 'C' : 'R';
    mps.bonds[i + 1] = mid;
    mps.sites[i] = std::move(A);
    mps.sites[i + 1] = std::move(B);
}

// ---------------------------------------------------------------------------------------------------------------
// Environment-stack memory path (SURVEY.md 7 hard part 5; BASELINE configs 4 and 5: "block-sparse operator storage
// sized to fit 180 GB HBM").  A pass consumes the blocks of one side in the order the previous pass produced them
// reversed, so only every env_stride-th block (a checkpoint) is kept; when the pass enters the segment between two
// checkpoints, its blocks are recomputed from the checkpoint with the unchanged site tensors (one extra blocking step
// per block and pass - renormalisation is a few percent of a sweep).  Checkpoints may additionally be spilled to
// pinned host memory with an asynchronous copy on a separate stream and fetched back when their segment is entered.
// ---------------------------------------------------------------------------------------------------------------
void Engine::ensure_svd_pool(int n) {
    while ((int)svd_pool.size() < n) {
        cudaStream_t ts = nullptr;
        cuda_check(cudaStreamCreateWithFlags(&ts, cudaStreamNonBlocking), "cudaStreamCreate");
        svd_streams.push_back(ts);
        svd_pool.push_back(svd_create(ts, opt.svd_qr == 0));
    }
}

static double wall() { return std::chrono::duration<double>(std::chrono::steady_clock::now().time_since_epoch()).count(); }

static int64_t g_device_bytes_env(const Engine& eng) {         // device bytes held by environment blocks right now
    int64_t b = 0;
    for (const auto& kv : eng.L) if (!kv.second->spilled) b += kv.second->bytes();
    for (const auto& kv : eng.R) if (!kv.second->spilled) b += kv.second->bytes();
    return b;
}
static void erase_block(Engine& eng, std::map<int, std::unique_ptr<Block>>& side, std::map<int, std::unique_ptr<Block>>::iterator& it) {
    for (size_t j = 0; j < eng.pending_spills.size(); ++j)
        if (eng.pending_spills[j] == it->second.get()) { eng.pending_spills.erase(eng.pending_spills.begin() + j); break; }
    it = side.erase(it);
}

void Engine::plan_env_policy(int D) {
    // estimate of every left block's bytes at bond dimension D from the current sector structure
    std::vector<double> est(k + 1, 0.0);
    double total = 0.0, bmax = 0.0;
    for (int b = 0; b <= k; ++b) {
        double sumsq = 0.0, dcur = 0.0;
        for (const Sector& q : mps.bonds[b]) { sumsq += (double)q.d * q.d; dcur += q.d; }
        // exact Schmidt bound of the bond, evaluated in log space (4^b overflows a double only beyond k ~ 500)
        const double lg4 = std::log2(4.0) * std::min(b, k - b);
        const double cap = lg4 < 40 ? std::min((double)D, std::pow(2.0, lg4)) : (double)D;
        if (dcur < cap && dcur > 0) sumsq *= (cap / dcur) * (cap / dcur);
        const double nin = 2.0 * std::min(b, k - b), nall = 2.0 * k;
        const double nops = nin * (nin - 1) / 2 + nin * nin + nall + 1;
        est[b] = 8.0 * nops * sumsq;
        total += est[b];
        bmax = std::max(bmax, est[b]);
    }
    env_est_total = (int64_t)total; env_est_max = (int64_t)bmax;
    size_t free_b = 0, total_b = 0;
    cuda_check(cudaMemGetInfo(&free_b, &total_b), "cudaMemGetInfo");
    // what is free now also has to hold the intermediates of H_eff psi and of the blocking step (two T buffers, capped at
    // 6 GiB each once the stack is checkpointed), the Davidson subspace and allocator slack
    const double avail = (double)free_b + (double)g_device_bytes_env(*this);
    const double budget = opt.hbm_budget_bytes > 0 ? (double)opt.hbm_budget_bytes : std::max(0.55 * avail, 0.8 * avail - 20.0 * (double)(1ull << 30));
    const double host_budget = opt.host_budget_bytes > 0 ? (double)opt.host_budget_bytes : 64.0 * (double)(1ull << 30);
    env_spill = false;
    env_stride = 1;
    env_stride2 = 1;
    ws_cap = 0;
    if (opt.env_stride > 0) { env_stride = opt.env_stride; env_stride2 = std::max(1, opt.env_stride2); env_spill = opt.host_spill != 0; return; }
    // everything resident only with headroom for the two full-size (24 GiB) T buffers of H_eff psi
    if (total <= (opt.hbm_budget_bytes > 0 ? budget : budget - 24.0 * (double)(1ull << 30))) return;
    // Peak device bytes of the environment blocks over a whole sweep for checkpoint spacing s, second-level spacing q
    // (1 = keep the whole segment) and checkpoints on the host or not: the resident sets of need_left / need_right /
    // retire_* replayed on the per-bond estimates.
    auto simulate = [&](int sp, int q, bool spill, double& host) {
        auto ck = [&](int b) { return b == 0 || b == k || b % sp == 0; };
        host = 0.0;
        double cks = 0.0;
        for (int c = 1; c < k; ++c) if (ck(c)) cks += est[c];
        if (spill) host = 1.7 * cks;      // measured: the pinned pool peaks at 1.65-1.8 x one side's checkpoints (both sides at the turn-around, best-fit slack)
        double peak = 0.0;
        for (int i = 0; i <= k - 2; ++i) {
            // forward pass: left side produces, right side is consumed
            double left = est[i] + est[i + 1], right = 0.0;
            if (spill) { if (i - 1 > 0 && ck(i - 1)) left += est[i - 1]; }             // spill copy still in flight
            else for (int c = 1; c < i; ++c) if (ck(c)) left += est[c];
            {
                const int b = i + 2;
                int c = b;
                while (!ck(c)) ++c;
                const int kb = (b / q + 1) * q;
                for (int j = b; j <= c; ++j) if (j == c || j % q == 0 || j < kb) right += est[j];
                if (!spill) for (int c2 = c + 1; c2 < k; ++c2) if (ck(c2)) right += est[c2];
            }
            peak = std::max(peak, left + right);
            // backward pass: right side produces, left side is consumed
            right = est[i + 2] + est[i + 1];
            left = 0.0;
            if (spill) { if (i + 3 < k && ck(i + 3)) right += est[i + 3]; }
            else for (int c = i + 3; c < k; ++c) if (ck(c)) right += est[c];
            {
                const int b = i;
                int c = b;
                while (!ck(c)) --c;
                const int ka = b > 0 ? ((b - 1) / q) * q : 0;
                for (int j = c; j <= b; ++j) if (j == c || j % q == 0 || j > ka) left += est[j];
                if (!spill) for (int c2 = 1; c2 < c; ++c2) if (ck(c2)) left += est[c2];
            }
            peak = std::max(peak, left + right);
        }
        return peak;
    };
    // cheapest feasible setting: cost = fraction of blocks recomputed per pass (second level: again) + a small charge for
    // the host round trips
    int bs = 0, bq = 1;
    bool bspill = false;
    double bcost = 0.0, bpeak = 0.0;
    for (int spill = 0; spill <= (opt.host_spill ? 1 : 0); ++spill)
        for (int sp = 1; sp <= std::min(k, 24); ++sp)
            for (int q = 1; q < std::max(2, sp); ++q) {
                if (sp == 1 && !spill) continue;                      // everything resident: already ruled out above
                double host = 0.0;
                const double peak = simulate(sp, q, spill != 0, host);
                if (peak > budget || host > host_budget) continue;
                const double r1 = (double)(sp - 1) / sp;
                const double cost = r1 + (q > 1 ? r1 * (q - 1) / q : 0.0) + (spill ? 0.3 / sp : 0.0);
                if (!bs || cost < bcost - 1e-12 || (cost < bcost + 1e-12 && peak < bpeak)) { bs = sp; bq = q; bspill = spill != 0; bcost = cost; bpeak = peak; }
            }
    if (!bs)
        throw Error(-3, opt.host_spill ? "environment stack does not fit the device and host budgets even with two checkpoint levels"
                                       : "environment stack does not fit the device even with recomputation: set host_spill = 1");
    env_stride = bs; env_stride2 = bq; env_spill = bspill;
    if (opt.workspace_bytes == 0) ws_cap = (int64_t)6 << 27;          // 6 GiB of doubles per T buffer while memory is tight
}

void Engine::finish_spills() {
    const double t0 = wall();
    for (Block* b : pending_spills) b->finish_spill();
    pending_spills.clear();
    t_spill_wait += wall() - t0;
}

static bool is_checkpoint(const Engine& eng, int b) { return b == 0 || b == eng.k || b % eng.env_stride == 0; }

void Engine::retire_left(int b) {
    auto it = L.find(b);
    if (it == L.end() || b == 0) return;
    if (!is_checkpoint(*this, b)) { erase_block(*this, L, it); return; }
    if (env_spill && !it->second->spilled) {
        spill_bytes += (double)it->second->bytes();
        it->second->spill(host_pool, copy_stream);
        pending_spills.push_back(it->second.get());
    }
}
void Engine::retire_right(int b) {
    auto it = R.find(b);
    if (it == R.end() || b == k) return;
    if (!is_checkpoint(*this, b)) { erase_block(*this, R, it); return; }
    if (env_spill && !it->second->spilled) {
        spill_bytes += (double)it->second->bytes();
        it->second->spill(host_pool, copy_stream);
        pending_spills.push_back(it->second.get());
    }
}
static void make_resident(Engine& eng, Block& blk) {
    if (!blk.spilled) return;
    const double t0 = wall();
    for (size_t j = 0; j < eng.pending_spills.size(); ++j)
        if (eng.pending_spills[j] == &blk) { eng.pending_spills.erase(eng.pending_spills.begin() + j); break; }
    eng.restore_bytes += (double)blk.bytes();
    blk.restore(eng.stream);
    eng.t_restore += wall() - t0;
}
Block& Engine::need_left(int b) {
    auto it = L.find(b);
    if (it != L.end()) { make_resident(*this, *it->second); return *it->second; }
    int c = b;
    while (c > 0 && L.find(c) == L.end()) --c;                        // nearest checkpoint below
    if (L.find(c) == L.end()) L[0] = empty_block('L', k, mps);
    make_resident(*this, *L.at(c));
    const double t0 = wall();
    // second checkpoint level (env_stride2 > 1): of the blocks between the checkpoint and the target only every
    // env_stride2-th one and the target's own sub-segment stay; the rest is erased as soon as it has produced its
    // successor and is recomputed from the nearest kept block when the pass gets there
    const int s2 = std::max(1, env_stride2);
    const int keep_above = ((b - 1) / s2) * s2;                       // sub-segment of the target: (keep_above, b]
    for (int j = c; j < b; ++j) {
        L[j + 1] = grow(*L.at(j), ham, mps, mode_L(j + 1), *this);
        if (j != c && j % s2 != 0 && j <= keep_above) L.erase(j);
    }
    t_regrow += wall() - t0;
    return *L.at(b);
}
Block& Engine::need_right(int b) {
    auto it = R.find(b);
    if (it != R.end()) { make_resident(*this, *it->second); return *it->second; }
    int c = b;
    while (c < k && R.find(c) == R.end()) ++c;
    if (R.find(c) == R.end()) R[k] = empty_block('R', k, mps);
    make_resident(*this, *R.at(c));
    const double t0 = wall();
    const int s2 = std::max(1, env_stride2);
    const int keep_below = (b / s2 + 1) * s2;                         // sub-segment of the target: [b, keep_below)
    for (int j = c; j > b; --j) {
        R[j - 1] = grow(*R.at(j), ham, mps, mode_R(j - 1), *this);
        if (j != c && j % s2 != 0 && j >= keep_below) R.erase(j);
    }
    t_regrow += wall() - t0;
    return *R.at(b);
}
void Engine::build_right_stack() {
    if (R.find(k) == R.end()) R[k] = empty_block('R', k, mps);
    for (int b = k; b > 2; --b) {
        finish_spills();
        R[b - 1] = grow(*R.at(b), ham, mps, mode_R(b - 1), *this);
        retire_right(b);
    }
}
static void track_peak(Engine& eng) { eng.env_peak_bytes = std::max(eng.env_peak_bytes, g_device_bytes); }

// ---------------------------------------------------------------------------------------------------------------
// one sweep: forward pass over bonds 0..k-2, backward pass k-2..0 (reading S12)
// ---------------------------------------------------------------------------------------------------------------
static BondRecord optimise(Engine& eng, int i, int D, bool forward) {
    typedef std::chrono::steady_clock clk;
    auto secs = [](clk::time_point a, clk::time_point b) { return std::chrono::duration<double>(b - a).count(); };
    const auto t0 = clk::now();
    eng.plan.reset();
    eng.finish_spills();                                       // device copies of blocks spilled during the previous step
    Block& LB = eng.need_left(i);
    Block& RB = eng.need_right(i + 2);
    const auto t0b = clk::now();
    eng.plan = build_heff(eng.ham, LB, RB, i, eng);
    HeffPlan& p = *eng.plan;
    const auto t1 = clk::now();
    DevVec<double> theta;
    theta.alloc((size_t)p.nnz);
    two_site_tensor(eng.mps, i, p, theta.p, eng);
    const DavidsonResult dr = eng.opt.eigensolver == 1 ? lanczos(p, theta.p, eng) : davidson(p, theta.p, eng);
    const auto t2 = clk::now();
    BondRecord rec;
    rec.bond = i; rec.forward = forward ? 1 : 0;
    rec.energy = dr.theta; rec.residual = dr.residual; rec.n_matvec = dr.n_matvec; rec.converged = dr.converged ? 1 : 0;
    rec.nnz = p.nnz; rec.f_alg = p.f_alg; rec.seconds_matvec = dr.seconds_matvec;
    split_theta(eng.mps, i, p, theta.p, D, forward, eng, rec.trunc_err, rec.kept, rec.nsectors);
    const auto t3 = clk::now();
    eng.plan.reset();                                          // releases the temporaries before the block grows
    track_peak(eng);
    if (forward) {
        // blocks of the right stack up to bond i+2 are consumed (the backward pass rebuilds them); L_i has produced
        // L_{i+1} and stays only as a checkpoint
        for (auto it = eng.R.begin(); it != eng.R.end();)
            if (it->first <= i + 2 && it->first < eng.k) erase_block(eng, eng.R, it); else ++it;
        eng.L[i + 1] = grow(LB, eng.ham, eng.mps, eng.mode_L(i + 1), eng);
        if (i < eng.k - 2) eng.retire_left(i);                 // the backward pass starts at this bond: keep L_{k-2}
    } else {
        for (auto it = eng.L.begin(); it != eng.L.end();)      // L_i is consumed, every L_b with b > i is stale
            if (it->first >= i && it->first > 0) erase_block(eng, eng.L, it); else ++it;
        if (i > 0) {                                           // R_1 is never used; the next forward pass starts from R_2
            eng.R[i + 1] = grow(RB, eng.ham, eng.mps, eng.mode_R(i + 1), eng);
            eng.retire_right(i + 2);
        }
    }
    track_peak(eng);
    const auto t4 = clk::now();
    rec.seconds = secs(t0, t4);
    eng.t_env += secs(t0, t0b);
    eng.t_plan += secs(t0b, t1); eng.t_davidson += secs(t1, t2); eng.t_split += secs(t2, t3); eng.t_grow += secs(t3, t4);
    eng.t_matvec += dr.seconds_matvec;
    return rec;
}

int sweep(Engine& eng, int D, std::vector<BondRecord>& recs, double& seconds) {
    const auto t0 = std::chrono::steady_clock::now();
    const int k = eng.k;
    eng.t_plan = eng.t_davidson = eng.t_split = eng.t_grow = eng.t_matvec = eng.t_env = 0.0;
    eng.t_spill_wait = eng.t_restore = eng.t_regrow = eng.spill_bytes = eng.restore_bytes = 0.0;
    eng.env_peak_bytes = 0;
    if (!eng.sweep_ready || D != eng.env_D) {
        const bool rebuild = !eng.sweep_ready;
        if (rebuild) eng.invalidate();
        eng.plan_env_policy(D);
        eng.env_D = D;
        if (rebuild) {
            eng.keep_env_stack = true;
            eng.L[0] = empty_block('L', k, eng.mps);
            const double tb = wall();
            eng.build_right_stack();
            eng.t_env += wall() - tb;
            eng.sweep_ready = true;
        }
    }
    recs.clear();
    for (int i = 0; i <= k - 2; ++i) recs.push_back(optimise(eng, i, D, true));
    for (int i = k - 2; i >= 0; --i) recs.push_back(optimise(eng, i, D, false));
    seconds = std::chrono::duration<double>(std::chrono::steady_clock::now() - t0).count();
    if (eng.trace || std::getenv("DMRG_B200_TIMERS"))
        std::fprintf(stderr, "[dmrg trace] sweep D=%d: %.2f s = environments (restore %.2f, regrow %.2f, spill wait %.2f) %.2f + plan (block maps) %.2f + davidson %.2f (matvec %.2f) + svd/split %.2f + renormalise %.2f; stride %d spill %d peak %.1f GB\n",
                     D, seconds, eng.t_restore, eng.t_regrow, eng.t_spill_wait, eng.t_env, eng.t_plan, eng.t_davidson, eng.t_matvec, eng.t_split, eng.t_grow,
                     eng.env_stride, (int)eng.env_spill, eng.env_peak_bytes / 1e9);
    int warnings = 0;
    for (const BondRecord& r : recs) if (!r.converged) ++warnings;
    return warnings;
}

}  // namespace dmrg
