"""Kernel-level parity: the grouped, K-segmented FP64 DMMA GEMM against its plain definition
C_t = sum_s alpha_s op(A_s) op(B_s) evaluated with numpy in FP64 (ragged sizes, all operand orientations)."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu


def _case(lib, rng, shapes, accumulate, generic=False, aligned=False):
    import torch
    dev = torch.device("cuda:0")
    tasks, segs, keep, expect = [], [], [], []
    for (M, N, ks) in shapes:
        ldc = N + (0 if aligned else int(rng.integers(0, 3)))
        c0 = rng.normal(size=(M, ldc))
        Cd = torch.tensor(c0, device=dev)
        keep.append(Cd)
        ref = c0[:, :N].copy() if accumulate else np.zeros((M, N))
        sb = len(segs)
        for K in ks:
            fl = int(rng.integers(0, 4))
            ident = (K == 0)
            alpha = float(rng.normal())
            if ident:
                a = rng.normal(size=(M, N + 1))
                Ad = torch.tensor(a, device=dev)
                keep.append(Ad)
                segs.append(dict(A=Ad.data_ptr(), B=0, lda=N + 1, ldb=0, K=0, flags=4, alpha=alpha))
                ref += alpha * a[:, :N]
                continue
            pa, pb = int(rng.integers(0, 2)), int(rng.integers(0, 2))
            if aligned:                                           # even leading dimensions covering pad2(extent): bulk-copy kernel eligible
                pa, pb = (M if (fl & 1) else K) % 2 + 2, (K if (fl & 2) else N) % 2 + 2
            a = rng.normal(size=(K, M + pa)) if (fl & 1) else rng.normal(size=(M, K + pa))
            b = rng.normal(size=(N, K + pb)) if (fl & 2) else rng.normal(size=(K, N + pb))
            Ad, Bd = torch.tensor(a, device=dev), torch.tensor(b, device=dev)
            keep += [Ad, Bd]
            opa = a[:, :M].T if (fl & 1) else a[:, :K]
            opb = b[:, :K].T if (fl & 2) else b[:, :N]
            ref += alpha * (opa @ opb)
            segs.append(dict(A=Ad.data_ptr(), B=Bd.data_ptr(), lda=a.shape[1], ldb=b.shape[1], K=K, flags=fl, alpha=alpha))
        tasks.append(dict(C=Cd.data_ptr(), ldc=ldc, M=M, N=N, seg_begin=sb, seg_count=len(segs) - sb,
                          flags=1 if accumulate else 0))
        expect.append((Cd, ref, c0, N))
    torch.cuda.synchronize()
    ms = lib.dmrg_grouped_gemm(tasks, segs, torch.cuda.current_stream().cuda_stream, generic=generic)
    torch.cuda.synchronize()
    assert ms > 0.0
    for (Cd, ref, c0, N) in expect:
        got = Cd.cpu().numpy()
        scale = max(1.0, np.abs(ref).max())
        assert np.abs(got[:, :N] - ref).max() <= 1e-12 * scale * 50
        assert np.array_equal(got[:, N:], c0[:, N:])              # padding columns untouched


@pytest.mark.parametrize("accumulate", [False, True])
def test_grouped_gemm_ragged(lib, accumulate):
    rng = np.random.default_rng(7)
    shapes = [(1, 1, [1]), (7, 5, [3, 9]), (64, 64, [16]), (65, 63, [17, 0, 31]), (130, 70, [5, 64, 1, 33]),
              (33, 200, [129]), (200, 37, [2, 2, 2, 0]), (64, 128, []), (3, 3, [0])]
    _case(lib, rng, shapes, accumulate)


def test_grouped_gemm_many_segments_spanning_tiles(lib):
    rng = np.random.default_rng(11)
    shapes = [(150, 170, [int(k) for k in rng.integers(1, 90, size=40)]), (257, 129, [300, 7, 64])]
    _case(lib, rng, shapes, False)


@pytest.mark.parametrize("generic", [False, True])
def test_grouped_gemm_aligned_operands_both_kernels(lib, generic):
    """16-byte aligned operands with even leading dimensions: the bulk-copy (TMA engine) kernel, and the cp.async kernel
    forced on the same problem."""
    rng = np.random.default_rng(23)
    shapes = [(64, 64, [16, 48]), (150, 170, [int(k) for k in rng.integers(1, 90, size=12)]), (9, 300, [77, 0, 5]), (257, 129, [300, 7])]
    _case(lib, rng, shapes, False, generic=generic, aligned=True)
    _case(lib, rng, shapes, True, generic=generic, aligned=True)


def test_probe_and_counters(lib):
    """The bench-only probe library returns plausible ceilings (DMMA within 50-110 % of the nominal 37.2 TFLOP/s of a
    B200); dmrg_flops_total counts unpadded flops."""
    import torch
    r = lib.dmrg_fp64_probe(0, iters=4000, ctas_per_sm=3, reps=2)
    assert 0.5 * 37.2 <= r["tflops"] <= 1.1 * 37.2 and r["ms"] > 0
    r1 = lib.dmrg_fp64_probe(1, iters=4000, ctas_per_sm=3, reps=2)
    assert 5.0 <= r1["tflops"] <= 1.1 * 37.2
    with pytest.raises(lib.binding.DmrgError):
        lib.dmrg_fp64_probe(7)
    from synth import random_dense, random_mps, mps_to_blob_arrays
    k, n = 6, 6
    h, eri = random_dense(k, 1)
    ctx = lib.dmrg_create(k, n, 0, h, eri)
    try:
        assert lib.dmrg_flops_total(ctx) == 0.0
        lib.dmrg_mps_import(ctx, mps_to_blob_arrays(random_mps(k, n, 0, 12, seed=2, gauge="LR:2")), k, n, 0)
        lib.dmrg_prepare_bond(ctx, 2)
        f0 = lib.dmrg_flops_total(ctx)
        assert f0 > 0.0
        nnz, _ = lib.dmrg_heff_layout(ctx, 2)
        x = np.ones(nnz)
        y = np.zeros(nnz)
        lib.dmrg_heff_apply(ctx, 2, x, y)
        st = lib.dmrg_heff_stats(ctx, 2)
        assert lib.dmrg_flops_total(ctx) - f0 == st["f_exec"]
    finally:
        lib.dmrg_destroy(ctx)
    torch.cuda.synchronize()
