"""Device-built block maps against the host reference builder of the same library: the layout,
the flop / byte accounting and the diagonal must agree exactly, H_eff x to rounding (the two builders order the
K-concatenated segments differently), and both must match the oracle (tests/test_gpu_heff.py covers the default path)."""
import numpy as np
import pytest

from synth import random_dense, random_mps, mps_to_blob_arrays

pytestmark = pytest.mark.gpu


def _run(lib, host_maps, k, n, s2, D, i, h, eri, mps, x):
    ctx = lib.dmrg_create(k, n, s2, h, eri, workspace_bytes=1 << 22, host_maps=1 if host_maps else 0)   # small workspace: several chunks
    try:
        lib.dmrg_mps_import(ctx, mps_to_blob_arrays(mps), k, n, s2)
        lib.dmrg_prepare_bond(ctx, i)
        nnz, lay = lib.dmrg_heff_layout(ctx, i)
        y = np.zeros(nnz)
        lib.dmrg_heff_apply(ctx, i, x[:nnz], y)
        d = np.zeros(nnz)
        lib.dmrg_heff_diag(ctx, i, d)
        return nnz, lay, y, d, lib.dmrg_heff_stats(ctx, i)
    finally:
        lib.dmrg_destroy(ctx)


@pytest.mark.parametrize("k,n,s2,D,seed", [(8, 8, 0, 40, 5), (10, 9, 1, 64, 6), (12, 14, 0, 96, 7), (6, 4, 2, 16, 8)])
def test_device_maps_match_host_maps(lib, k, n, s2, D, seed):
    h, eri = random_dense(k, seed)
    x = np.random.default_rng(seed).normal(size=1 << 22)
    for i in sorted({0, 1, k // 2 - 1, k - 3, k - 2}):
        mps = random_mps(k, n, s2, D, seed=seed + 10, gauge="LR:%d" % i)
        nd, lay_d, y_d, d_d, st_d = _run(lib, False, k, n, s2, D, i, h, eri, mps, x)
        nh, lay_h, y_h, d_h, st_h = _run(lib, True, k, n, s2, D, i, h, eri, mps, x)
        assert nd == nh and [tuple(b) for b in lay_d] == [tuple(b) for b in lay_h]
        assert st_d["f_alg"] == st_h["f_alg"] and st_d["b_alg"] == st_h["b_alg"] and st_d["nterms"] == st_h["nterms"]
        assert st_d["f_exec"] <= st_d["f_alg"]
        scale = max(1.0, np.abs(y_h).max())
        assert np.abs(y_d - y_h).max() <= 1e-12 * scale
        assert np.abs(d_d - d_h).max() <= 1e-12 * max(1.0, np.abs(d_h).max())
