"""dmrg_stack_dots_noalloc - the allocation-free entry point (static device scratch, no cudaMalloc) - against the existing
dmrg_stack_dots path on the same inputs, on two calls in a row (the second with other inputs and another shape, so stale
scratch contents of the first call would show), plus the size limit.  Collected last on purpose (file name): the suite
runs with pytest -x."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu


def _both(lib, torch, rng, nrows, nc, K):
    lds, ldm, ldE = K + (K & 1) + 2, K + (K & 1) + 4, nc + 1
    S = torch.tensor(rng.normal(size=(nrows, lds)), device="cuda")
    M = torch.tensor(rng.normal(size=(nc, ldm)), device="cuda")
    E0 = torch.full((nrows, ldE), 7.0, dtype=torch.float64, device="cuda")
    E1 = torch.full((nrows, ldE), 7.0, dtype=torch.float64, device="cuda")
    st = torch.cuda.current_stream().cuda_stream
    torch.cuda.synchronize()
    lib.dmrg_stack_dots(S.data_ptr(), lds, nrows, M.data_ptr(), ldm, nc, K, E0.data_ptr(), ldE, st)      # existing path
    assert lib.dmrg_stack_dots_noalloc(S.data_ptr(), lds, nrows, M.data_ptr(), ldm, nc, K, E1.data_ptr(), ldE, st) == 0
    torch.cuda.synchronize()
    e0, e1 = E0.cpu().numpy(), E1.cpu().numpy()
    ref = S.cpu().numpy()[:, :K] @ M.cpu().numpy()[:, :K].T
    tol = 1e-12 * max(1.0, np.abs(ref).max()) * max(1.0, np.sqrt(K))          # the tolerance of the stack_dots parity test
    assert np.abs(e1[:, :nc] - e0[:, :nc]).max() <= tol
    assert np.abs(e1[:, :nc] - ref).max() <= tol
    assert np.all(e1[:, nc:] == 7.0)                                          # padding column untouched


def test_stack_dots_noalloc_matches_existing_path_twice_in_a_row(lib):
    import torch
    rng = np.random.default_rng(2503)
    _both(lib, torch, rng, 70, 5, 2 * 1024 * 9 + 1)        # several K spans, ragged rows, odd K tail
    _both(lib, torch, rng, 33, 8, 1025)                    # second call: other shape and data over the same static scratch
    _both(lib, torch, rng, 70, 5, 2 * 1024 * 9 + 1)        # and the first shape again


def test_stack_dots_noalloc_rejects_sizes_beyond_the_static_scratch(lib):
    import torch
    x = torch.zeros(16, dtype=torch.float64, device="cuda")
    st = torch.cuda.current_stream().cuda_stream
    with pytest.raises(lib.binding.DmrgError) as err:      # 200000 rows x 8 right-hand sides: 1.6e6 > 2^20 doubles of scratch
        lib.dmrg_stack_dots_noalloc(x.data_ptr(), 2, 200000, x.data_ptr(), 2, 8, 2, x.data_ptr(), 8, st)
    assert err.value.code == lib.DMRG_ENOMEM and "static scratch" in str(err.value)
    torch.cuda.synchronize()
