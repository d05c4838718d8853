"""Parity of the device RDM pass (dmrg_rdm12) with the CPU oracle, element by element, plus the invariants of
BASELINE.json north_star: Tr gamma = N, sum_r Gamma_pqrr = (N-1) gamma_pq, symmetries, and
E = sum h gamma + 1/2 sum (pq|rs) Gamma.  Tolerance: RDM max-abs error <= 1e-10."""
import numpy as np
import pytest

from oracle import dmrg as odmrg
from oracle import fci as ofci
from synth import random_dense, random_mps, mps_to_blob_arrays, blob_arrays_to_mps, make_config

pytestmark = pytest.mark.gpu
TOL = 1e-10


def _invariants(g, G, n):
    k = g.shape[0]
    assert abs(np.trace(g) - n) <= 1e-9
    assert np.abs(g - g.T).max() <= 1e-10
    assert np.abs(np.einsum("pqrr->pq", G) - (n - 1) * g).max() <= 1e-9
    assert abs(np.einsum("pprr->", G) - n * (n - 1)) <= 1e-8
    assert np.abs(G - G.transpose(2, 3, 0, 1)).max() <= 1e-10
    assert np.abs(G - G.transpose(1, 0, 3, 2)).max() <= 1e-10
    w = np.linalg.eigvalsh(g)
    assert w.min() >= -1e-9 and w.max() <= 2 + 1e-9 and k > 0


@pytest.mark.parametrize("k,n,s2,D", [(2, 2, 0, 4), (3, 3, 1, 6), (4, 4, 0, 8), (5, 6, 0, 12), (6, 6, 0, 16),
                                      (6, 7, 1, 12), (6, 3, -1, 10), (8, 8, 0, 20)])
def test_rdm12_random_mps_vs_oracle(lib, k, n, s2, D):
    h, eri = random_dense(k, 300 + k)
    mps = random_mps(k, n, s2, D, seed=31 + k, gauge="R")
    for key in list(mps["tensors"][0].keys()):                      # an unnormalised centre must not matter
        mps["tensors"][0][key] = 1.7 * mps["tensors"][0][key]
    g0, G0 = odmrg.rdm12(h, eri, mps, True)
    ctx = lib.dmrg_create(k, n, s2, h, eri)
    try:
        lib.dmrg_mps_import(ctx, mps_to_blob_arrays(mps), k, n, s2)
        g, G = lib.dmrg_rdm12(ctx, k, True)
        g1, _ = lib.dmrg_rdm12(ctx, k, False)                       # 1-RDM only path; repeated calls allowed
    finally:
        lib.dmrg_destroy(ctx)
    assert np.abs(g - g0).max() <= TOL and np.abs(G - G0).max() <= TOL and np.abs(g1 - g0).max() <= TOL
    _invariants(g, G, n)


def test_rdm12_after_sweep_energy_and_fci(lib):
    """After untruncated sweeps the RDMs equal the brute-force FCI RDMs and reproduce the energy (S20)."""
    k, n, s2 = 6, 6, 0
    h, eri = random_dense(k, 77)
    space = ofci.FCISpace(k, n, s2)
    e_fci, c = space.ground_state(h, eri)
    gf, Gf = space.rdm12(c)
    mps = random_mps(k, n, s2, 8, seed=9, gauge="R")
    ctx = lib.dmrg_create(k, n, s2, h, eri, davidson_tol=1e-11)
    try:
        lib.dmrg_mps_import(ctx, mps_to_blob_arrays(mps), k, n, s2)
        for _ in range(4):
            e = lib.dmrg_sweep(ctx, 4096, k)["energy_last"]
        g, G = lib.dmrg_rdm12(ctx, k, True)
    finally:
        lib.dmrg_destroy(ctx)
    assert abs(e - e_fci) <= 1e-9
    assert np.abs(g - gf).max() <= 1e-7 and np.abs(G - Gf).max() <= 1e-7     # state converged to ~1e-11 in energy
    e_rdm = np.einsum("pq,pq->", h, g) + 0.5 * np.einsum("pqrs,pqrs->", eri, G)
    assert abs(e_rdm - e_fci) <= 1e-9
    _invariants(g, G, n)


def test_rdm12_config1_truncated_sweep_vs_oracle(lib):
    """BASELINE config 1 at D = 64: RDMs of the GPU's final MPS vs the oracle's RDM pass on that same MPS."""
    cfg = make_config(1)
    k, n = cfg["k"], cfg["n_elec"]
    mps = random_mps(k, n, 0, 64, seed=cfg["seed"] + 1000, gauge="R")
    ctx = lib.dmrg_create(k, n, 0, cfg["h"], cfg["eri"])
    try:
        lib.dmrg_mps_import(ctx, mps_to_blob_arrays(mps), k, n, 0)
        for _ in range(2):
            r = lib.dmrg_sweep(ctx, 64, k)
        g, G = lib.dmrg_rdm12(ctx, k, True)
        arrs, n2, s2 = lib.dmrg_mps_export(ctx, k)
    finally:
        lib.dmrg_destroy(ctx)
    final = blob_arrays_to_mps(k, n, 0, *arrs)
    g0, G0 = odmrg.rdm12(cfg["h"], cfg["eri"], final, True)
    assert np.abs(g - g0).max() <= TOL and np.abs(G - G0).max() <= TOL
    _invariants(g, G, n)
    e_rdm = np.einsum("pq,pq->", cfg["h"], g) + 0.5 * np.einsum("pqrs,pqrs->", cfg["eri"], G)
    assert e_rdm >= r["energy_min"] - 1e-9                           # <Psi|H|Psi> of the truncated MPS (reading S20)


@pytest.mark.parametrize("nrows,nc,K", [(1, 1, 1), (5, 3, 77), (33, 8, 1025), (64, 2, 4096 + 3), (70, 5, 2 * 1024 * 9 + 1), (3, 8, 0)])
def test_stack_dots_kernel_matches_definition(lib, nrows, nc, K):
    """RDM accumulation kernel for few right-hand sides against its definition E = S M^T (numpy, FP64): ragged row
    counts, K tails (odd, below / above one chunk, several spans), every template width."""
    import torch
    rng = np.random.default_rng(nrows * 1000 + nc)
    lds = K + (K & 1) + 2
    ldm = K + (K & 1) + 4
    S = rng.normal(size=(nrows, lds))
    M = rng.normal(size=(nc, ldm))
    Sd, Md = torch.tensor(S, device="cuda"), torch.tensor(M, device="cuda")
    ldE = nc + 1
    Ed = torch.full((nrows, ldE), 7.0, dtype=torch.float64, device="cuda")
    ms = lib.dmrg_stack_dots(Sd.data_ptr(), lds, nrows, Md.data_ptr(), ldm, nc, K, Ed.data_ptr(), ldE,
                             torch.cuda.current_stream().cuda_stream)
    torch.cuda.synchronize()
    assert ms >= 0.0
    E = Ed.cpu().numpy()
    ref = S[:, :K] @ M[:, :K].T
    assert np.abs(E[:, :nc] - ref).max() <= 1e-12 * max(1.0, np.abs(ref).max()) * max(1.0, np.sqrt(K))
    assert np.all(E[:, nc:] == 7.0)


@pytest.mark.parametrize("cid,D", [(2, 12), (3, 12)])
def test_rdm12_config_geometries_small_D_vs_oracle(lib, cid, D):
    """1-/2-RDM element by element against the oracle on the Hamiltonians and chain lengths of BASELINE configs 2
    (coronene, k = 24) and 3 (Fe-S-like, k = 20, N = 30 > k), at a bond dimension the plain oracle pass finishes in
    about a minute (the full D = 512 / 1024 oracle pass would take hours; the GPU pass at full D is checked by its
    invariants in bench.py and test_rdm12_after_sweep_energy_and_fci)."""
    cfg = make_config(cid)
    k, n = cfg["k"], cfg["n_elec"]
    mps = random_mps(k, n, 0, D, seed=900 + cid, gauge="R")
    g0, G0 = odmrg.rdm12(cfg["h"], cfg["eri"], mps, True)
    ctx = lib.dmrg_create(k, n, 0, cfg["h"], cfg["eri"])
    try:
        lib.dmrg_mps_import(ctx, mps_to_blob_arrays(mps), k, n, 0)
        g, G = lib.dmrg_rdm12(ctx, k, True)
    finally:
        lib.dmrg_destroy(ctx)
    assert np.abs(g - g0).max() <= TOL and np.abs(G - G0).max() <= TOL
    _invariants(g, G, n)


@pytest.mark.parametrize("k,n,s2,D", [(6, 6, 0, 12), (7, 8, 2, 16), (8, 7, 1, 20)])
def test_rdm12_partition_point_does_not_matter_and_matches_oracle(lib, k, n, s2, D):
    """Half-chain partition: every partition point kh = 0 (right rule only: c = s2, two-index operators on
    the right - the oracle's order), k (left rule only: c = s3, on the left - the round-1 order) and everything between
    gives the oracle's RDMs."""
    h, eri = random_dense(k, 700 + k)
    mps = random_mps(k, n, s2, D, seed=80 + k, gauge="R")
    g0, G0 = odmrg.rdm12(h, eri, mps, True)
    for kh in [0, 1, k // 2, k - 1, k, -1]:
        ctx = lib.dmrg_create(k, n, s2, h, eri, rdm_split=kh)
        try:
            lib.dmrg_mps_import(ctx, mps_to_blob_arrays(mps), k, n, s2)
            g, G = lib.dmrg_rdm12(ctx, k, True)
        finally:
            lib.dmrg_destroy(ctx)
        assert np.abs(g - g0).max() <= TOL and np.abs(G - G0).max() <= TOL, kh


def test_rdm12_config4_chain_partition_points_agree(lib):
    """BASELINE config 4 (k = 54, the 9 279-term Hamiltonian) at reduced D: the pass with the partition in the middle
    (the one that scales) against the two one-sided evaluation orders, which the oracle tests above pin; invariants."""
    cfg = make_config(4)
    k, n, D = cfg["k"], cfg["n_elec"], 48
    mps = random_mps(k, n, 0, D, seed=4321, gauge="R")
    res = []
    for kh in (-1, 0, k):
        ctx = lib.dmrg_create(k, n, 0, cfg["h"], cfg["eri"], rdm_split=kh)
        try:
            lib.dmrg_mps_import(ctx, mps_to_blob_arrays(mps), k, n, 0)
            res.append(lib.dmrg_rdm12(ctx, k, True))
        finally:
            lib.dmrg_destroy(ctx)
    (g, G) = res[0]
    for (g1, G1) in res[1:]:
        assert np.abs(g - g1).max() <= TOL and np.abs(G - G1).max() <= TOL
    _invariants(g, G, n)


def test_rdm12_and_diag_into_device_buffers_on_the_callers_stream(lib):
    """`where = DMRG_DEVICE`: dmrg_rdm12 and dmrg_heff_diag write into caller device buffers on the caller's stream
    (ordered after its pending work) and agree with the host-buffer results."""
    import torch
    k, n, s2, D = 6, 6, 0, 12
    h, eri = random_dense(k, 31)
    mps = random_mps(k, n, s2, D, seed=14, gauge="R")
    ctx = lib.dmrg_create(k, n, s2, h, eri)
    try:
        lib.dmrg_mps_import(ctx, mps_to_blob_arrays(mps), k, n, s2)
        g0, G0 = lib.dmrg_rdm12(ctx, k, True)
        st = torch.cuda.Stream()
        with torch.cuda.stream(st):
            gd = torch.full((k, k), 7.0, dtype=torch.float64, device="cuda")      # pending work on the buffers
            Gd = torch.full((k, k, k, k), 7.0, dtype=torch.float64, device="cuda")
            lib.dmrg_rdm12(ctx, k, True, out=(gd, Gd))
            g1, G1 = gd.cpu().numpy(), Gd.cpu().numpy()
        assert np.array_equal(g0, g1) and np.array_equal(G0, G1)
        i = 2
        lib.dmrg_mps_import(ctx, mps_to_blob_arrays(random_mps(k, n, s2, D, seed=15, gauge="LR:%d" % i)), k, n, s2)
        lib.dmrg_prepare_bond(ctx, i)
        nnz, _ = lib.dmrg_heff_layout(ctx, i)
        dh = np.zeros(nnz)
        lib.dmrg_heff_diag(ctx, i, dh)
        with torch.cuda.stream(st):
            dd = torch.full((nnz,), 3.0, dtype=torch.float64, device="cuda")
            lib.dmrg_heff_diag(ctx, i, dd)
            d1 = dd.cpu().numpy()
        assert np.array_equal(dh, d1)
    finally:
        lib.dmrg_destroy(ctx)
