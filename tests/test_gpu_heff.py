"""Parity of the CUDA path with the CPU oracle, element by element on the same seeded inputs:
environments built by the fused renormalisation kernels, then y = H_eff x and diag(H_eff) at EVERY two-site bond.
Tolerance (BASELINE.json north_star): relative L2 error <= 1e-11."""
import numpy as np
import pytest

from oracle import dmrg as odmrg
from synth import random_dense, random_mps, mps_to_blob_arrays, make_config

pytestmark = pytest.mark.gpu
TOL = 1e-11


def _check_bond(P, ctx, mps, oham, i, seed):
    P.dmrg_prepare_bond(ctx, i)
    nnz, lay = P.dmrg_heff_layout(ctx, i)
    oL = odmrg.build_left(mps, oham, i)[-1]
    oR = odmrg.build_right(mps, oham, i + 2)[i + 2]
    H = odmrg.Heff(oL, oR, oham, i)
    assert nnz == H.nnz and [tuple(b) for b in lay] == [tuple(b) for b in H.layout]
    x = np.random.default_rng(seed).normal(size=nnz)
    x /= np.linalg.norm(x)
    y = np.zeros(nnz)
    P.dmrg_heff_apply(ctx, i, x, y)
    y0 = H.apply(x)
    assert np.linalg.norm(y - y0) <= TOL * np.linalg.norm(y0)
    d = np.zeros(nnz)
    P.dmrg_heff_diag(ctx, i, d)
    assert np.abs(d - H.diagonal()).max() <= 1e-11 * max(1.0, np.abs(d).max())
    return x, y


@pytest.mark.parametrize("k,n,s2,D", [(2, 2, 0, 4), (3, 3, 1, 6), (4, 4, 0, 8), (6, 6, 0, 10), (6, 7, 1, 12),
                                      (7, 6, 0, 10), (6, 3, -1, 12), (8, 10, 0, 40)])
def test_heff_every_bond_vs_oracle(lib, k, n, s2, D):
    h, eri = random_dense(k, 40 + k)
    oham = odmrg.Ham(h, eri)
    ctx = lib.dmrg_create(k, n, s2, h, eri)
    try:
        for i in range(k - 1):
            mps = random_mps(k, n, s2, D, seed=70 + i, gauge="LR:%d" % i)
            lib.dmrg_mps_import(ctx, mps_to_blob_arrays(mps), k, n, s2)
            _check_bond(lib, ctx, mps, oham, i, i)
    finally:
        lib.dmrg_destroy(ctx)


def test_heff_device_buffers_and_symmetry(lib):
    """Device-resident x / y on torch's stream; <phi|H psi> = <H phi|psi>; linearity; chunked T buffer = unchunked."""
    import torch
    k, n, s2, D, i = 8, 8, 0, 48, 3
    h, eri = random_dense(k, 5)
    mps = random_mps(k, n, s2, D, seed=3, gauge="LR:%d" % i)
    outs = []
    for ws in (0, 1 << 17):                                         # automatic, and a 128 KiB cap that forces many chunks
        ctx = lib.dmrg_create(k, n, s2, h, eri, workspace_bytes=ws)
        try:
            lib.dmrg_mps_import(ctx, mps_to_blob_arrays(mps), k, n, s2)
            lib.dmrg_prepare_bond(ctx, i)
            nnz, _ = lib.dmrg_heff_layout(ctx, i)
            g = torch.Generator(device="cpu").manual_seed(1)
            x = torch.randn(nnz, dtype=torch.float64, generator=g).cuda()
            p = torch.randn(nnz, dtype=torch.float64, generator=g).cuda()
            y, q, z = torch.empty_like(x), torch.empty_like(x), torch.empty_like(x)
            lib.dmrg_heff_apply(ctx, i, x, y)
            lib.dmrg_heff_apply(ctx, i, p, q)
            lib.dmrg_heff_apply(ctx, i, 2.0 * x - 3.0 * p, z)
            torch.cuda.synchronize()
            assert abs(float(p @ y) - float(q @ x)) <= 1e-11 * float(y.norm() * p.norm())
            assert float((z - (2.0 * y - 3.0 * q)).norm()) <= 1e-12 * float(z.norm())
            yh = np.zeros(nnz)
            lib.dmrg_heff_apply(ctx, i, x.cpu().numpy(), yh)
            assert np.array_equal(yh, y.cpu().numpy())              # host and device entry: bit-identical
            outs.append(yh)
        finally:
            lib.dmrg_destroy(ctx)
    assert np.linalg.norm(outs[0] - outs[1]) <= 1e-13 * np.linalg.norm(outs[0])


def test_heff_config1_naphthalene_every_bond(lib):
    """BASELINE config 1 (PPP naphthalene, CAS(10,10), rotated dense ERI) at D=64: every bond vs the oracle."""
    cfg = make_config(1)
    k, n = cfg["k"], cfg["n_elec"]
    oham = odmrg.Ham(cfg["h"], cfg["eri"])
    ctx = lib.dmrg_create(k, n, 0, cfg["h"], cfg["eri"])
    try:
        for i in range(k - 1):
            mps = random_mps(k, n, 0, 64, seed=cfg["seed"] + 1000 + i, gauge="LR:%d" % i)
            lib.dmrg_mps_import(ctx, mps_to_blob_arrays(mps), k, n, 0)
            _check_bond(lib, ctx, mps, oham, i, 100 + i)
    finally:
        lib.dmrg_destroy(ctx)
