"""Parity at BASELINE.json's own sizes.
configs[1] (coronene CAS(24,24), D = 512) and configs[2] (Fe-S-like CAS(30,20), D = 1024): H_eff psi and diag(H_eff)
vs the oracle, element by element, on environments each side builds itself ("dual gauge": one left-orthonormal and one
right-orthonormal seeded MPS on the same sector plan serve every bond).  configs[3] (circumcoronene CAS(54,54),
D = 4096, the launch configuration bench.py times): the oracle cannot build these environments in bounded time, so the
full-size check is by properties that hold at any size - symmetry <p|H x> = <H p|x>, linearity, determinism - and by
the flop/byte accounting identities."""
import numpy as np
import pytest

from oracle import dmrg as odmrg
from synth import random_mps, mps_to_blob_arrays, make_config, bond_sector_plan

pytestmark = pytest.mark.gpu
TOL = 1e-11


def _dual_gauge(cfg, D, seed):
    k, n = cfg["k"], cfg["n_elec"]
    plan = bond_sector_plan(k, n, 0, D)
    A = random_mps(k, n, 0, D, seed=seed, gauge="L", plan=plan)
    B = random_mps(k, n, 0, D, seed=seed + 1, gauge="R", plan=plan)
    return A, B


def _mixed(A, B, i):
    k = A["k"]
    return dict(k=k, n_elec=A["n_elec"], two_sz=A["two_sz"], bonds=A["bonds"],
                tensors=[A["tensors"][p] if p < i else B["tensors"][p] for p in range(k)],
                gauge=["L" if p < i else "R" for p in range(k)])


def _compare(lib, cfg, D, bonds, seed):
    k, n = cfg["k"], cfg["n_elec"]
    A, B = _dual_gauge(cfg, D, seed)
    assert A["bonds"] == B["bonds"]
    oham = odmrg.Ham(cfg["h"], cfg["eri"])
    oL = odmrg.build_left(A, oham, max(bonds))
    oR = odmrg.build_right(B, oham, min(bonds) + 2)
    ctx = lib.dmrg_create(k, n, 0, cfg["h"], cfg["eri"], keep_env_stack=0)
    try:
        for i in bonds:
            lib.dmrg_mps_import(ctx, mps_to_blob_arrays(_mixed(A, B, i)), k, n, 0)
            lib.dmrg_prepare_bond(ctx, i)
            nnz, lay = lib.dmrg_heff_layout(ctx, i)
            H = odmrg.Heff(oL[i], oR[i + 2], oham, i)
            assert nnz == H.nnz and [tuple(b) for b in lay] == [tuple(b) for b in H.layout]
            x = np.random.default_rng(1000 + i).normal(size=nnz)
            x /= np.linalg.norm(x)
            y = np.zeros(nnz)
            lib.dmrg_heff_apply(ctx, i, x, y)
            y0 = H.apply(x)
            assert np.linalg.norm(y - y0) <= TOL * np.linalg.norm(y0)
            d = np.zeros(nnz)
            lib.dmrg_heff_diag(ctx, i, d)
            assert np.abs(d - H.diagonal()).max() <= 1e-11 * max(1.0, np.abs(d).max())
            st = lib.dmrg_heff_stats(ctx, i)
            assert 0 < st["f_exec"] <= st["f_alg"] and st["b_alg"] >= 16.0 * nnz
    finally:
        lib.dmrg_destroy(ctx)


def test_config2_coronene_D512_heff_vs_oracle(lib):
    _compare(lib, make_config(2), 512, [0, 6, 10, 11, 12, 22], seed=2001)   # full D: ends, around the N/C switch, between


def test_config2_coronene_every_bond_heff_vs_oracle(lib):
    _compare(lib, make_config(2), 128, list(range(0, 23)), seed=2003)             # EVERY two-site bond


def test_config3_fes_D1024_midbond_heff_vs_oracle(lib):
    cfg = make_config(3)
    _compare(lib, cfg, 1024, [cfg["k"] // 2 - 1], seed=3001)


def test_config4_D4096_full_size_properties(lib):
    """The exact launch configuration of bench.py (config 4, D = 4096, mid-chain bond 26)."""
    import torch
    cfg = make_config(4)
    k, n, D = cfg["k"], cfg["n_elec"], cfg["D"]
    i = k // 2 - 1
    mps = random_mps(k, n, 0, D, seed=cfg["seed"] + 1000, gauge="LR:%d" % i)
    ctx = lib.dmrg_create(k, n, 0, cfg["h"], cfg["eri"], keep_env_stack=0)
    try:
        lib.dmrg_mps_import(ctx, mps_to_blob_arrays(mps), k, n, 0)
        lib.dmrg_prepare_bond(ctx, i)
        nnz, lay = lib.dmrg_heff_layout(ctx, i)
        assert nnz == sum(b[4] * b[5] for b in lay) and lay[-1][6] + lay[-1][4] * lay[-1][5] == nnz
        g = torch.Generator(device="cpu").manual_seed(7)
        x = torch.randn(nnz, dtype=torch.float64, generator=g).cuda()
        p = torch.randn(nnz, dtype=torch.float64, generator=g).cuda()
        x /= x.norm()
        p /= p.norm()
        y, q, z, y2 = (torch.empty_like(x) for _ in range(4))
        lib.dmrg_heff_apply(ctx, i, x, y)
        lib.dmrg_heff_apply(ctx, i, p, q)
        lib.dmrg_heff_apply(ctx, i, 0.5 * x - 2.0 * p, z)
        lib.dmrg_heff_apply(ctx, i, x, y2)
        torch.cuda.synchronize()
        assert torch.isfinite(y).all() and float(y.norm()) > 0
        assert torch.equal(y, y2)                                        # fixed summation order: bit-reproducible
        assert abs(float(p @ y) - float(q @ x)) <= 1e-11 * float(y.norm())
        assert float((z - (0.5 * y - 2.0 * q)).norm()) <= 1e-12 * float(z.norm())
        d = torch.empty_like(x)
        lib.dmrg_heff_diag(ctx, i, d)
        torch.cuda.synchronize()
        # <e_j|H|e_j> = diag_j on sampled unit vectors (each costs one full application)
        for j in (0, nnz // 3, nnz - 1):
            e = torch.zeros_like(x)
            e[j] = 1.0
            lib.dmrg_heff_apply(ctx, i, e, z)
            torch.cuda.synchronize()
            assert abs(float(z[j]) - float(d[j])) <= 1e-11 * max(1.0, abs(float(d[j])))
        st = lib.dmrg_heff_stats(ctx, i)
        assert 0 < st["f_exec"] <= st["f_alg"] and st["nterms"] > 6000
    finally:
        lib.dmrg_destroy(ctx)


def test_config5_D1024_properties(lib):
    """configs[4] (82-site PAH-like chain of fused hexagons, CAS(82,82)) at a reduced bond dimension: the oracle cannot
    reach it in bounded time (reading S27), so the check is by properties that hold at any size - symmetry,
    linearity, bit-reproducibility, <e_j|H|e_j> = diag_j - on the device-built block maps of a 13 000-term bond."""
    import torch
    cfg = make_config(5)
    k, n, D = cfg["k"], cfg["n_elec"], 1024
    i = k // 2 - 1
    mps = random_mps(k, n, 0, D, seed=cfg["seed"] + 1000, gauge="LR:%d" % i)
    ctx = lib.dmrg_create(k, n, 0, cfg["h"], cfg["eri"], keep_env_stack=0)
    try:
        lib.dmrg_mps_import(ctx, mps_to_blob_arrays(mps), k, n, 0)
        lib.dmrg_prepare_bond(ctx, i)
        nnz, lay = lib.dmrg_heff_layout(ctx, i)
        assert nnz == sum(b[4] * b[5] for b in lay)
        g = torch.Generator(device="cpu").manual_seed(11)
        x = torch.randn(nnz, dtype=torch.float64, generator=g).cuda()
        p = torch.randn(nnz, dtype=torch.float64, generator=g).cuda()
        x /= x.norm()
        p /= p.norm()
        y, q, z, y2 = (torch.empty_like(x) for _ in range(4))
        lib.dmrg_heff_apply(ctx, i, x, y)
        lib.dmrg_heff_apply(ctx, i, p, q)
        lib.dmrg_heff_apply(ctx, i, 0.5 * x - 2.0 * p, z)
        lib.dmrg_heff_apply(ctx, i, x, y2)
        torch.cuda.synchronize()
        assert torch.isfinite(y).all() and float(y.norm()) > 0
        assert torch.equal(y, y2)
        assert abs(float(p @ y) - float(q @ x)) <= 1e-11 * float(y.norm())
        assert float((z - (0.5 * y - 2.0 * q)).norm()) <= 1e-12 * float(z.norm())
        d = torch.empty_like(x)
        lib.dmrg_heff_diag(ctx, i, d)
        torch.cuda.synchronize()
        for j in (1, nnz // 2, nnz - 2):
            e = torch.zeros_like(x)
            e[j] = 1.0
            lib.dmrg_heff_apply(ctx, i, e, z)
            torch.cuda.synchronize()
            assert abs(float(z[j]) - float(d[j])) <= 1e-11 * max(1.0, abs(float(d[j])))
        st = lib.dmrg_heff_stats(ctx, i)
        assert 0 < st["f_exec"] <= st["f_alg"] and st["nterms"] > 13000
    finally:
        lib.dmrg_destroy(ctx)


def test_config4_reduced_D_sweep_memory_path_and_rdm(lib):
    """BASELINE config 4 (k = 54) at D = 96: one sweep with every environment block resident against the same sweep
    under a device budget that forces checkpoints, recomputation and the pinned-host spill (bit-identical), then the
    RDM pass on the swept MPS: E_RDM = <Psi|H|Psi> must equal the last Davidson Rayleigh quotient up to the truncation of
    the final bond (reading S20), Tr gamma = N, partial trace."""
    cfg = make_config(4)
    k, n, D = cfg["k"], cfg["n_elec"], 96
    mps = random_mps(k, n, 0, D, seed=cfg["seed"] + 1000, gauge="R")
    out = []
    for run in (0, 1):
        # second run: budgets derived from the library's own estimate of the first (stack / 3 on the host, six blocks on
        # the device), so the automatic policy must choose checkpoints, recomputation and the spill
        opts = dict(env_stride=1) if run == 0 else dict(host_spill=1, hbm_budget_bytes=6 * out[0][1]["est_max_block_bytes"],
                                                        host_budget_bytes=out[0][1]["est_stack_bytes"] // 3)
        ctx = lib.dmrg_create(k, n, 0, cfg["h"], cfg["eri"], davidson_max_iter=6, **opts)
        try:
            lib.dmrg_mps_import(ctx, mps_to_blob_arrays(mps), k, n, 0)
            r = lib.dmrg_sweep(ctx, D, k)
            st = lib.dmrg_sweep_stats(ctx)
            g, G = lib.dmrg_rdm12(ctx, k, True) if not out else (None, None)
            out.append((r, st, g, G))
        finally:
            lib.dmrg_destroy(ctx)
    (ra, sa, g, G), (rb, sb, _, _) = out
    assert sa["env_stride"] == 1 and sa["host_spill"] == 0
    assert sb["env_stride"] > 1 and sb["seconds_regrow"] > 0           # the automatic policy had to checkpoint ...
    assert sb["host_spill"] == 1 and sb["bytes_spilled"] > 0           # ... and, with these budgets, to spill
    assert sb["peak_device_bytes"] < sa["peak_device_bytes"]
    assert [b["energy"] for b in ra["bonds"]] == [b["energy"] for b in rb["bonds"]]
    assert [b["kept"] for b in ra["bonds"]] == [b["kept"] for b in rb["bonds"]]
    assert abs(np.trace(g) - n) <= 1e-9
    assert np.abs(np.einsum("pqrr->pq", G) - (n - 1) * g).max() <= 1e-8
    e_rdm = np.einsum("pq,pq->", cfg["h"], g) + 0.5 * np.einsum("pqrs,pqrs->", cfg["eri"], G)
    last = ra["bonds"][-1]
    assert abs(e_rdm - last["energy"]) <= 1e-6 + 10 * last["trunc_err"]   # Davidson capped at 6 iterations: Rayleigh quotient of the kept state
