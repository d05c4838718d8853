"""Parity of the device two-site sweep (Davidson + SVD truncation + fused renormalisation) with the CPU oracle on
the same imported MPS.  Tolerance (BASELINE.json north_star): sweep energies <= 1e-8 Eh; parity runs use the
Davidson tolerance 1e-10 of reading S13 so the converged eigenpair does not depend on the iteration path."""
import numpy as np
import pytest

from oracle import dmrg as odmrg
from oracle import fci as ofci
from synth import random_dense, random_mps, mps_to_blob_arrays, make_config

pytestmark = pytest.mark.gpu
TOL_E = 1e-8


def _run_both(lib, h, eri, k, n, s2, D, nsweeps, seed, Dinit=None):
    mps = random_mps(k, n, s2, Dinit or D, seed=seed, gauge="R")
    ctx = lib.dmrg_create(k, n, s2, h, eri, davidson_tol=1e-10)
    eng = odmrg.SweepEngine(h, eri, mps, davidson_tol=1e-10)
    out = []
    try:
        lib.dmrg_mps_import(ctx, mps_to_blob_arrays(mps), k, n, s2)
        for _ in range(nsweeps):
            g = lib.dmrg_sweep(ctx, D, k)
            o = eng.sweep(D)
            out.append((g, o))
    finally:
        lib.dmrg_destroy(ctx)
    return out


@pytest.mark.parametrize("k,n,s2,D", [(4, 4, 0, 16), (6, 6, 0, 12), (6, 7, 1, 16), (8, 8, 0, 24)])
def test_sweep_energies_match_oracle(lib, k, n, s2, D):
    h, eri = random_dense(k, 90 + k)
    for (g, o) in _run_both(lib, h, eri, k, n, s2, D, 2, seed=17 + k):
        assert abs(g["energy_last"] - o["energy_last"]) <= TOL_E
        assert abs(g["energy_min"] - o["energy_min"]) <= TOL_E
        for rg, ro in zip(g["bonds"], o["bonds"]):
            assert rg["bond"] == ro["bond"] and rg["kept"] == ro["kept"] and rg["nsectors"] == ro["nsectors"]
            assert abs(rg["energy"] - ro["energy"]) <= TOL_E
            assert abs(rg["trunc_err"] - ro["trunc_err"]) <= 1e-9


def test_untruncated_sweep_reaches_fci(lib):
    """At full bond dimension the device sweep converges to the brute-force FCI ground energy."""
    k, n, s2 = 6, 6, 0
    h, eri = random_dense(k, 123)
    space = ofci.FCISpace(k, n, s2)
    e_fci = space.ground_state(h, eri)[0]
    mps = random_mps(k, n, s2, 8, seed=5, gauge="R")
    ctx = lib.dmrg_create(k, n, s2, h, eri, davidson_tol=1e-10)
    try:
        lib.dmrg_mps_import(ctx, mps_to_blob_arrays(mps), k, n, s2)
        e = None
        for _ in range(4):
            e = lib.dmrg_sweep(ctx, 4096, k)["energy_last"]
        assert abs(e - e_fci) <= 1e-9
    finally:
        lib.dmrg_destroy(ctx)


# BASELINE config 1 at D = 64, 4 sweeps (reading S11: D = 64 is truncated): per-bond parity with the oracle is in
# tests/test_gpu_golden.py::test_sweep_vs_golden[sweep_cfg1_D64.json] (stored oracle result; the live oracle took 2 min here).


def _golden():
    import os
    vals = {}
    for line in open(os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", "config1_fci.txt")):
        if not line.startswith("#"):
            key, rest = line.split(None, 1)
            vals[key] = [float(x) for x in rest.split()]
    return vals


def test_config1_untruncated_reaches_golden_fci(lib):
    """BASELINE config 1 with no truncation (reading S11: the exact mid-chain rank is 1024, so D >= 1024): energy vs
    the brute-force FCI value of tests/golden/config1_fci.txt to 1e-8 Eh, natural occupations of the device 1-RDM."""
    gold = _golden()
    cfg = make_config(1)
    k, n = cfg["k"], cfg["n_elec"]
    mps = random_mps(k, n, 0, 64, seed=cfg["seed"] + 1000, gauge="R")
    ctx = lib.dmrg_create(k, n, 0, cfg["h"], cfg["eri"], davidson_tol=1e-9)
    try:
        lib.dmrg_mps_import(ctx, mps_to_blob_arrays(mps), k, n, 0)
        for _ in range(5):
            r = lib.dmrg_sweep(ctx, 2048, k)
        g, G = lib.dmrg_rdm12(ctx, k, True)
    finally:
        lib.dmrg_destroy(ctx)
    assert abs(r["energy_last"] - gold["e_el_fci"][0]) <= 1e-8
    occ = np.sort(np.linalg.eigvalsh(g))[::-1]
    assert np.abs(occ - np.array(gold["natural_occupations"])).max() <= 1e-6
    e_rdm = np.einsum("pq,pq->", cfg["h"], g) + 0.5 * np.einsum("pqrs,pqrs->", cfg["eri"], G)
    assert abs(e_rdm - gold["e_el_fci"][0]) <= 1e-8


@pytest.mark.parametrize("opts", [dict(env_stride=3), dict(env_stride=2, host_spill=1), dict(env_stride=1, host_spill=1),
                                  dict(env_stride=4, host_spill=1), dict(env_stride=6, env_stride2=2, host_spill=1),
                                  dict(env_stride=9, env_stride2=3)])
def test_sweep_env_checkpoints_and_host_spill_are_bit_identical(lib, opts):
    """Environment-stack memory path: keeping only every env_stride-th block (the others recomputed when
    a pass reaches them) and spilling the checkpoints to pinned host memory must not change a single bit of a sweep,
    and must lower the peak device footprint."""
    k, n, s2, D = 10, 10, 0, 48
    h, eri = random_dense(k, 311)
    mps = random_mps(k, n, s2, D, seed=41, gauge="R")
    runs = []
    for o in (dict(env_stride=1), opts):
        ctx = lib.dmrg_create(k, n, s2, h, eri, davidson_tol=1e-10, **o)
        try:
            lib.dmrg_mps_import(ctx, mps_to_blob_arrays(mps), k, n, s2)
            base = lib.dmrg_device_bytes(ctx)
            recs = [lib.dmrg_sweep(ctx, D, k) for _ in range(2)]
            runs.append((recs, lib.dmrg_sweep_stats(ctx), base))
        finally:
            lib.dmrg_destroy(ctx)
    (ra, sa, ba), (rb, sb, bb) = runs
    for x, y in zip(ra, rb):
        assert x["energy_last"] == y["energy_last"] and x["energy_min"] == y["energy_min"]
        for bx, by in zip(x["bonds"], y["bonds"]):
            assert bx["energy"] == by["energy"] and bx["kept"] == by["kept"] and bx["trunc_err"] == by["trunc_err"]
    assert sb["env_stride"] == opts["env_stride"] and sb["host_spill"] == opts.get("host_spill", 0)
    assert sb["peak_device_bytes"] - bb < sa["peak_device_bytes"] - ba
    if opts.get("host_spill"):
        assert sb["bytes_spilled"] > 0 and sb["bytes_restored"] > 0 and sb["host_pool_bytes"] > 0
    else:
        assert sb["seconds_regrow"] > 0


def test_sweep_releases_consumed_environments(lib):
    """With every block kept (env_stride = 1) a pass still frees what it has consumed: at the turn-around only one
    operator stack is resident, so the peak is far below two stacks (round-1 behaviour)."""
    k, n, s2, D = 12, 12, 0, 64
    h, eri = random_dense(k, 77)
    mps = random_mps(k, n, s2, D, seed=9, gauge="R")
    ctx = lib.dmrg_create(k, n, s2, h, eri, env_stride=1)
    try:
        lib.dmrg_mps_import(ctx, mps_to_blob_arrays(mps), k, n, s2)
        base = lib.dmrg_device_bytes(ctx)
        lib.dmrg_sweep(ctx, D, k)
        after_first = lib.dmrg_device_bytes(ctx) - base           # = the right stack R_2 .. R_k
        lib.dmrg_sweep(ctx, D, k)
        st = lib.dmrg_sweep_stats(ctx)
        assert st["peak_device_bytes"] - base < 1.6 * after_first
    finally:
        lib.dmrg_destroy(ctx)


@pytest.mark.parametrize("k,n,s2,eps,dmin,dmax", [(6, 6, 0, 1e-6, 6, 40), (8, 8, 0, 1e-5, 10, 32), (8, 9, 1, 1e-4, 4, 64)])
def test_dbss_sweep_matches_oracle(lib, k, n, s2, eps, dmin, dmax):
    """Dynamic block state selection (reading S32): kept states per bond, truncation error and
    energies of DBSS sweeps, device vs oracle."""
    h, eri = random_dense(k, 400 + k)
    mps = random_mps(k, n, s2, 16, seed=55 + k, gauge="R")
    ctx = lib.dmrg_create(k, n, s2, h, eri, davidson_tol=1e-10, dbss_eps=eps, dbss_dmin=dmin)
    eng = odmrg.SweepEngine(h, eri, mps, davidson_tol=1e-10, dbss_eps=eps, dbss_dmin=dmin)
    try:
        lib.dmrg_mps_import(ctx, mps_to_blob_arrays(mps), k, n, s2)
        kept = set()
        for _ in range(2):
            g, o = lib.dmrg_sweep(ctx, dmax, k), eng.sweep(dmax)
            assert abs(g["energy_last"] - o["energy_last"]) <= TOL_E
            for rg, ro in zip(g["bonds"], o["bonds"]):
                assert rg["kept"] == ro["kept"] and rg["nsectors"] == ro["nsectors"]
                assert abs(rg["energy"] - ro["energy"]) <= TOL_E and abs(rg["trunc_err"] - ro["trunc_err"]) <= 1e-9
                kept.add(rg["kept"])
        assert len(kept) > 2                                      # the bond dimension really varies along the chain
    finally:
        lib.dmrg_destroy(ctx)


@pytest.mark.parametrize("k,n,s2,D", [(6, 6, 0, 12), (7, 8, 2, 16)])
def test_lanczos_sweep_matches_oracle(lib, k, n, s2, D):
    """Lanczos as the local eigensolver (reading S33): converged to 1e-10 it reaches the same eigenpairs as
    the oracle's Lanczos (and Davidson), so the whole sweep agrees."""
    h, eri = random_dense(k, 500 + k)
    mps = random_mps(k, n, s2, D, seed=7 + k, gauge="R")
    ctx = lib.dmrg_create(k, n, s2, h, eri, davidson_tol=1e-10, eigensolver=1, davidson_max_iter=400)
    eng = odmrg.SweepEngine(h, eri, mps, davidson_tol=1e-10, eigensolver="lanczos", davidson_max_iter=400)
    dav = odmrg.SweepEngine(h, eri, mps, davidson_tol=1e-10)
    try:
        lib.dmrg_mps_import(ctx, mps_to_blob_arrays(mps), k, n, s2)
        for _ in range(2):
            g, o, d = lib.dmrg_sweep(ctx, D, k), eng.sweep(D), dav.sweep(D)
            assert g["status"] == 0
            assert abs(g["energy_last"] - o["energy_last"]) <= TOL_E and abs(g["energy_last"] - d["energy_last"]) <= TOL_E
            for rg, ro in zip(g["bonds"], o["bonds"]):
                assert rg["kept"] == ro["kept"] and abs(rg["energy"] - ro["energy"]) <= TOL_E
    finally:
        lib.dmrg_destroy(ctx)


def test_solve_stops_by_eps_sweep_like_the_oracle(lib):
    """dmrg_solve: the eps_sweep rule of PAPER.md:179 (reading S34) stops after the same number of sweeps as the oracle's
    SweepEngine.solve, at the same energy."""
    k, n, s2, D = 5, 5, 1, 8
    h, eri = random_dense(k, 640)
    mps = random_mps(k, n, s2, D, seed=12, gauge="R")
    ctx = lib.dmrg_create(k, n, s2, h, eri, davidson_tol=1e-10)
    try:
        lib.dmrg_mps_import(ctx, mps_to_blob_arrays(mps), k, n, s2)
        r = lib.dmrg_solve(ctx, D, k, 1e-5, 15)
    finally:
        lib.dmrg_destroy(ctx)
    out = odmrg.SweepEngine(h, eri, mps, davidson_tol=1e-10).solve(D, 1e-5, 15)
    assert r["status"] == 0 and r["n_sweeps"] == len(out) and 3 <= len(out) < 15
    assert np.abs(r["energies"] - np.array([o["energy_last"] for o in out])).max() <= TOL_E
    assert abs(r["last"]["energy_last"] - out[-1]["energy_last"]) <= TOL_E
