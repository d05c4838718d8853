"""Pins for oracle tier 2 (plain block-sparse DMRG) against tier 1 (brute-force FCI) and invariants.
DESIGN.md C5: H_eff x vs P^T H P x at every bond; untruncated sweeps vs FCI energy and RDMs; RDM invariants."""
import numpy as np
import pytest

from oracle import fci, dmrg
from synth import random_dense, random_mps, make_config, full_sector_dims


@pytest.mark.parametrize("k,n,s2,D,bonds", [
    (4, 4, 0, 8, None), (5, 5, 1, 10, None), (6, 8, 0, 12, None), (6, 3, -1, 12, None),
    (8, 8, 0, 16, (0, 3, 6)),                                           # k = 8: both ends and the middle
    pytest.param(10, 10, 0, 20, (4,), marks=pytest.mark.slow)])        # k = 10 (FCI dimension 63504), mid-chain
def test_heff_vs_bruteforce_every_bond(k, n, s2, D, bonds):
    h, eri = random_dense(k, 40 + k)
    ham = dmrg.Ham(h, eri)
    sp = fci.FCISpace(k, n, s2)
    for i in (range(k - 1) if bonds is None else bonds):
        mps = random_mps(k, n, s2, D, seed=70 + i, gauge="LR:%d" % i)
        L = dmrg.build_left(mps, ham, i)[-1]
        R = dmrg.build_right(mps, ham, i + 2)[i + 2]
        for side in ("L", "R"):
            H = dmrg.Heff(L, R, ham, i, normal_side=side)
            lay, nnz = fci.heff_layout(mps, i)
            assert nnz == H.nnz and [tuple(b) for b in lay] == [tuple(b) for b in H.layout]
            x = np.random.default_rng(i).normal(size=nnz)
            y = H.apply(x)
            yb = fci.heff_apply_bruteforce(mps, i, h, eri, x, sp)
            assert np.linalg.norm(y - yb) <= 1e-13 * np.linalg.norm(yb)


def test_heff_symmetric_and_diagonal():
    k, n, s2 = 6, 6, 0
    h, eri = random_dense(k, 3)
    ham = dmrg.Ham(h, eri)
    i = 2
    mps = random_mps(k, n, s2, 6, seed=1, gauge="LR:%d" % i)
    H = dmrg.Heff(dmrg.build_left(mps, ham, i)[-1], dmrg.build_right(mps, ham, i + 2)[i + 2], ham, i)
    M = np.stack([H.apply(e) for e in np.eye(H.nnz)], axis=1)
    assert np.abs(M - M.T).max() < 1e-12
    assert np.abs(np.diag(M) - H.diagonal()).max() < 1e-12


def test_davidson_against_dense_eigh():
    rng = np.random.default_rng(5)
    n = 200
    M = rng.normal(size=(n, n))
    M = M + M.T + np.diag(np.arange(n) * 2.0)
    w = np.linalg.eigvalsh(M)
    th, u, nmv, rn, ok = dmrg.davidson(lambda v: M @ v, np.diag(M).copy(), rng.normal(size=n), tol=1e-10,
                                       max_iter=300)
    assert ok and abs(th - w[0]) < 1e-10 and np.linalg.norm(M @ u - th * u) < 1e-9


def test_truncation_never_splits_a_degenerate_cluster():
    # one left sector (dim 1 bond 0), theta = diag-like with singular values 0.8, 0.5, 0.5(degenerate), 0.1:
    # D = 2 would cut through the 0.5 doublet -> rule keeps 1 (reading S14)
    bonds_l = [(0, 0, 4)]
    bonds_r = [(0, 0, 4)]
    sv = np.array([0.8, 0.5, 0.5 * (1 - 1e-9), 0.1])
    sv = sv / np.linalg.norm(sv)
    rng = np.random.default_rng(0)
    U, _ = np.linalg.qr(rng.normal(size=(4, 4)))
    V, _ = np.linalg.qr(rng.normal(size=(4, 4)))
    theta = {(0, 0, 0): U @ np.diag(sv) @ V.T}
    mid, A, B, trunc, kept = dmrg.split_theta(theta, bonds_l, bonds_r, 2, "fwd")
    assert kept == 1 and mid == [(0, 0, 1)]
    assert abs(trunc - (1 - sv[0] ** 2)) < 1e-12
    mid, A, B, trunc, kept = dmrg.split_theta(theta, bonds_l, bonds_r, 3, "fwd")
    assert kept == 3 and abs(trunc - sv[3] ** 2) < 1e-12
    assert np.abs(A[(0, 0)].T @ A[(0, 0)] - np.eye(3)).max() < 1e-12       # left-orthonormal
    assert abs(np.sum(B[(0, 0)] ** 2) - 1.0) < 1e-12                        # kept state renormalised


@pytest.mark.parametrize("k,n,s2", [(5, 5, 1), (6, 6, 0)])
def test_untruncated_sweep_reaches_fci_energy_and_rdms(k, n, s2):
    h, eri = random_dense(k, 11 + k, scale=0.25)
    sp = fci.FCISpace(k, n, s2)
    e0, c0 = sp.ground_state(h, eri)
    mps = random_mps(k, n, s2, 8, seed=2, gauge="R")
    eng = dmrg.SweepEngine(h, eri, mps, davidson_tol=1e-11, davidson_max_iter=300)
    for _ in range(3):
        r = eng.sweep(10 ** 6)
    assert abs(r["energy_last"] - e0) < 1e-10
    g, G = dmrg.rdm12(h, eri, eng.mps)
    gf, Gf = sp.rdm12(c0)
    assert np.abs(g - gf).max() < 1e-8 and np.abs(G - Gf).max() < 1e-8     # eigenvector accuracy ~ sqrt-free 1e-10/gap
    assert abs(np.einsum("pq,pq", h, g) + 0.5 * np.einsum("pqrs,pqrs", eri, G) - e0) < 1e-10


def test_truncated_sweep_variational_and_rdm_energy_of_final_mps():
    k, n, s2, D = 6, 6, 0, 10
    h, eri = random_dense(k, 17, scale=0.25)
    sp = fci.FCISpace(k, n, s2)
    e0, _ = sp.ground_state(h, eri)
    mps = random_mps(k, n, s2, D, seed=2, gauge="R")
    eng = dmrg.SweepEngine(h, eri, mps, davidson_tol=1e-10, davidson_max_iter=300)
    for _ in range(2):
        r = eng.sweep(D)
    assert all(b["energy"] >= e0 - 1e-10 for b in r["bonds"])
    assert max(sum(d for _, _, d in bb) for bb in eng.mps["bonds"]) <= D
    c = fci.mps_to_ci(eng.mps, sp)
    assert abs(np.linalg.norm(c) - 1.0) < 1e-10
    e_mps = c @ sp.apply_h(h, eri, c)
    g, G = dmrg.rdm12(h, eri, eng.mps)
    assert abs(np.einsum("pq,pq", h, g) + 0.5 * np.einsum("pqrs,pqrs", eri, G) - e_mps) < 1e-10     # reading S20
    gf, Gf = sp.rdm12(c)
    assert np.abs(g - gf).max() < 1e-11 and np.abs(G - Gf).max() < 1e-11


def test_rdm_invariants_random_mps():
    k, n, s2 = 7, 9, 1
    h, eri = random_dense(k, 1)
    mps = random_mps(k, n, s2, 14, seed=8, gauge="R")
    g, G = dmrg.rdm12(h, eri, mps)
    assert abs(np.trace(g) - n) < 1e-11
    assert np.abs(np.einsum("pqrr->pq", G) - (n - 1) * g).max() < 1e-11
    assert np.abs(G - G.transpose(2, 3, 0, 1)).max() < 1e-11
    assert np.abs(G - G.transpose(1, 0, 3, 2)).max() < 1e-11
    assert np.abs(g - g.T).max() < 1e-12


@pytest.mark.slow
def test_config1_untruncated_sweep_vs_fci():
    cfg = make_config(1)
    k = cfg["k"]
    mps = random_mps(k, cfg["n_elec"], 0, 64, seed=cfg["seed"] + 1000, gauge="R")
    eng = dmrg.SweepEngine(cfg["h"], cfg["eri"], mps, davidson_tol=1e-10)
    for _ in range(3):
        r = eng.sweep(1024)
    assert abs(r["energy_last"] + cfg["e_core"] - (-0.8822829988)) < 1e-8


def test_select_kept_fixed_D_and_dbss_on_synthetic_spectra():
    """Pins of the truncation rule (readings S14, S32) on spectra where the answer is known by
    hand: the kept count follows eps_TR, clamps at D_min / D_max, and never splits a near-degenerate cluster."""
    sel = dmrg.select_kept
    # geometric spectrum sigma_t^2 = w0 r^t, normalised: discarded weight after m states is r^m exactly
    r = 0.5
    sv = np.sqrt((1 - r) * r ** np.arange(80))
    sv = list(sv / np.sqrt(np.sum(sv ** 2)))
    for eps, want in [(0.3, 2), (0.2, 3), (1e-3, 10), (1e-6, 20)]:          # r^m <= eps  <=>  m >= log(eps) / log(r)
        assert sel(sv, 1000, dbss_eps=eps) == want
    assert sel(sv, 1000, dbss_eps=1e-3, dbss_dmin=16) == 16                  # clamps at D_min
    assert sel(sv, 7, dbss_eps=1e-3) == 7                                    # clamps at D_max
    assert sel(sv, 7, dbss_eps=1e-3, dbss_dmin=16) == 7                      # D_max wins over D_min
    assert sel(sv, 12) == 12 and sel(sv, 1000) == 66                         # fixed D; sigma_t = 0.5^((t+1)/2) <= 1e-10 dropped
    # clusters: doublets (sigma_{2j} = sigma_{2j+1}), as the Sz partners of a spin multiplet
    w = np.repeat(0.5 ** np.arange(10), 2)
    d = list(np.sqrt(w / w.sum()))
    assert sel(d, 5) == 4 and sel(d, 6) == 6 and sel(d, 1) == 1              # fixed D: cut moves down, never to zero
    disc = lambda m: 1.0 - sum(x * x for x in d[:m])
    m = sel(d, 100, dbss_eps=disc(3) * 0.999)                                # target needs 4 states -> exactly a boundary
    assert m == 4
    m = sel(d, 100, dbss_eps=disc(3) * 1.001)                                # 3 states would do: inside a doublet -> up to 4
    assert m == 4 and disc(m) <= disc(3)
    assert sel(d, 3, dbss_eps=disc(3) * 1.001) == 2                          # cannot go up (D_max = 3): moves down
    assert sel(d, 100, dbss_eps=0.9, dbss_dmin=5) == 6                       # D_min inside a doublet -> up


def test_dbss_sweep_truncation_error_below_target():
    """A DBSS sweep of the oracle keeps, at every bond, a truncation error <= eps_TR unless the bond sits at D_max, and
    at least D_min states where the bond allows it; its energy lies between the D_min and the D_max fixed-D energies."""
    k, n, s2 = 6, 6, 0
    h, eri = random_dense(k, 5)
    mps = random_mps(k, n, s2, 24, seed=3, gauge="R")
    eps, dmin, dmax = 1e-6, 6, 40
    eng = dmrg.SweepEngine(h, eri, mps, davidson_tol=1e-10, dbss_eps=eps, dbss_dmin=dmin)
    for _ in range(3):
        r = eng.sweep(dmax)
    full = full_sector_dims(k, n, s2)
    for b in r["bonds"]:
        cap = min(dmax, sum(full[b["bond"] + 1].values()))
        assert b["kept"] <= dmax
        assert b["trunc_err"] <= eps * (1 + 1e-9) or b["kept"] >= cap - 3       # within a cluster of the cap
        assert b["kept"] >= min(dmin, cap) - 3
    lo = dmrg.SweepEngine(h, eri, mps, davidson_tol=1e-10)
    hi = dmrg.SweepEngine(h, eri, mps, davidson_tol=1e-10)
    for _ in range(3):
        e_lo, e_hi = lo.sweep(dmin)["energy_last"], hi.sweep(dmax)["energy_last"]
    assert e_hi - 1e-9 <= r["energy_last"] <= e_lo + 1e-9


def _jw_dense(k):
    """Dense Jordan-Wigner annihilators a_P on the 4^k Fock space, site 0 slowest, local order (|0>,|dn>,|up>,|up dn>),
    spin orbital P = 2p + [dn]: a_P = F x ... x F x a_local x 1 x ... x 1 (F = (-1)^N of the sites before p)."""
    F = np.diag([1.0, -1.0, -1.0, 1.0])
    out = []
    for P in range(2 * k):
        m = np.ones((1, 1))
        for q in range(k):
            m = np.kron(m, F if q < P // 2 else (dmrg.site_ann(P) if q == P // 2 else np.eye(4)))
        out.append(m)
    return out


def test_block_operators_are_projected_jordan_wigner_matrices():
    """Operator identities against dense Jordan-Wigner matrices (k = 3): every stored operator of a renormalised left
    block equals V^T O V, with O the dense operator built from its DEFINITION (C3 step 1: a+_P, A_PQ = a+_P a+_Q,
    B_PS = a+_P a_S, H_X, S_P^X) on the block's own Fock space and V the isometry the site tensors define (Eq. 14)."""
    k, n, s2, nb = 3, 3, 1, 2
    h, eri = random_dense(k, 11)
    ham = dmrg.Ham(h, eri)
    mps = random_mps(k, n, s2, 16, seed=4, gauge="L")
    blk = dmrg.build_left(mps, ham, nb)[-1]
    # isometry V [4^nb, dim(bond nb)]: V[(s0 s1), (sector, alpha)] = (A0[s0] A1[s1])[0, alpha]
    cols = []
    for ri, (N, S, d) in enumerate(blk.basis):
        V = np.zeros((4 ** nb, d))
        for s0 in range(4):
            for s1 in range(4):
                t0 = mps["tensors"][0].get((0, s0))
                if t0 is None:
                    continue
                n1, z1 = dmrg.SITE_Q[s0]
                mid = [j for j, (a, b, _) in enumerate(mps["bonds"][1]) if (a, b) == (n1, z1)]
                if not mid:
                    continue
                t1 = mps["tensors"][1].get((mid[0], s1))
                if t1 is None or (n1 + dmrg.SITE_Q[s1][0], z1 + dmrg.SITE_Q[s1][1]) != (N, S):
                    continue
                V[s0 * 4 + s1] = (t0 @ t1)[0]
        cols.append(V)
    a = _jw_dense(nb)                                                   # operators of the block's own sites
    ad = [m.T for m in a]
    inside = list(range(2 * nb))

    def check(op, dense):
        for i, (N, S, d) in enumerate(blk.basis):
            for o in range(len(blk.basis)):
                ref = cols[o].T @ dense @ cols[i]
                if i in op.blocks and op.blocks[i][0] == o:
                    assert np.abs(op.blocks[i][1] - ref).max() < 1e-12
                else:
                    assert np.abs(ref).max() < 1e-12

    for P in inside:
        check(blk.ops[("C", P)], ad[P])
        for Q in inside:
            if P < Q:
                check(blk.ops[("A", P, Q)], ad[P] @ ad[Q])
            check(blk.ops[("B", P, Q)], ad[P] @ a[Q])
    Hd = sum(ham.t(P, Q) * ad[P] @ a[Q] for P in inside for Q in inside)
    Hd = Hd + 0.5 * sum(ham.v(P, Q, R, S) * ad[P] @ ad[Q] @ a[R] @ a[S]
                        for P in inside for Q in inside for R in inside for S in inside)
    check(blk.ops[("H",)], Hd)
    for P in range(2 * nb, 2 * k):                                      # S_P^X for P outside, by definition
        Sd = sum(0.5 * ham.t(P, Q) * a[Q] for Q in inside)
        Sd = Sd + sum(ham.v(P, Q, R, S) * ad[Q] @ a[R] @ a[S] for Q in inside for R in inside for S in inside)
        check(blk.ops[("S", P)], Sd)


def test_lanczos_against_dense_eigh_and_davidson():
    """Lanczos reaches the lowest eigenpair of a dense symmetric matrix (numpy eigh), through restarts,
    and agrees with Davidson on an H_eff."""
    rng = np.random.default_rng(8)
    n = 300
    M = rng.normal(size=(n, n))
    M = M + M.T + np.diag(np.arange(n) * 1.5)
    w = np.linalg.eigvalsh(M)
    for sub in (40, 8):                                                  # without and with restarts
        th, u, nmv, rn, ok = dmrg.lanczos(lambda v: M @ v, rng.normal(size=n), tol=1e-10, max_iter=2000, max_subspace=sub)
        assert ok and abs(th - w[0]) < 1e-10 and np.linalg.norm(M @ u - th * u) < 1e-9
    k, n_e, s2, i = 6, 6, 0, 2
    h, eri = random_dense(k, 3)
    ham = dmrg.Ham(h, eri)
    mps = random_mps(k, n_e, s2, 8, seed=1, gauge="LR:%d" % i)
    H = dmrg.Heff(dmrg.build_left(mps, ham, i)[-1], dmrg.build_right(mps, ham, i + 2)[i + 2], ham, i)
    x0 = rng.normal(size=H.nnz)
    t1 = dmrg.lanczos(H.apply, x0, tol=1e-11, max_iter=500)
    t2 = dmrg.davidson(H.apply, H.diagonal(), x0, tol=1e-11, max_iter=500)
    assert t1[4] and t2[4] and abs(t1[0] - t2[0]) < 1e-10 and abs(abs(t1[1] @ t2[1]) - 1.0) < 1e-9


def test_sweep_stopping_rule():
    """eps_sweep rule (reading S34) on hand-made energy sequences, and inside SweepEngine.solve."""
    conv = dmrg.sweeps_converged
    assert not conv([-1.0, -1.0], 1e-3)                                  # needs three sweeps
    assert conv([-1.0, -1.0004, -1.0007], 1e-3)
    assert not conv([-1.0, -1.002, -1.0021], 1e-3)                       # first difference too large
    assert not conv([-1.0, -1.0001, -1.002], 1e-3)                       # second difference too large
    assert conv([-0.5, -1.0, -1.0004, -1.0007], 1e-3)                    # only the last three count
    k, n, s2 = 6, 6, 0
    h, eri = random_dense(k, 9)
    mps = random_mps(k, n, s2, 16, seed=2, gauge="R")
    eng = dmrg.SweepEngine(h, eri, mps, davidson_tol=1e-9)
    out = eng.solve(16, 1e-6, 12)
    e = [r["energy_last"] for r in out]
    assert 3 <= len(e) < 12 and conv(e, 1e-6) and not any(conv(e[:j], 1e-6) for j in range(len(e)))
