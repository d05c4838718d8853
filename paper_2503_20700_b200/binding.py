"""ctypes binding of include/dmrg_b200.h - argument marshalling only; every step of the path runs in the CUDA library.

The functions carry the names of the C entry points (dmrg_create, dmrg_mps_import, dmrg_prepare_bond, dmrg_heff_layout,
dmrg_heff_apply, dmrg_heff_diag, dmrg_heff_stats, dmrg_sweep, dmrg_rdm12, ...).  Vectors may be numpy arrays (host
buffers, copied by the library) or torch CUDA tensors (device buffers used in place on torch's current stream; torch is
only the allocator and stream provider here).  There is no CPU fallback: if the shared library is missing, import of
this module raises.
"""
import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.environ.get("DMRG_B200_LIB", os.path.join(_HERE, "libdmrg_b200.so"))
if not os.path.exists(LIB_PATH):
    raise ImportError("%s not found: build it with `python -c 'import __graft_entry__ as g; g.build()'` "
                      "(there is no CPU fallback)" % LIB_PATH)
lib = C.CDLL(LIB_PATH)

DMRG_OK, DMRG_EINVAL, DMRG_ESTATE, DMRG_ENOMEM, DMRG_ECUDA, DMRG_ENOCONV = 0, -1, -2, -3, -4, 1
DMRG_HOST, DMRG_DEVICE = 0, 1


class dmrg_options(C.Structure):
    _fields_ = [("davidson_tol", C.c_double), ("davidson_max_iter", C.c_int32), ("davidson_max_subspace", C.c_int32),
                ("sv_floor", C.c_double), ("cluster_rel_gap", C.c_double), ("device_id", C.c_int32),
                ("keep_env_stack", C.c_int32), ("workspace_bytes", C.c_int64),
                ("hbm_budget_bytes", C.c_int64), ("host_budget_bytes", C.c_int64), ("host_spill", C.c_int32),
                ("env_stride", C.c_int32), ("dbss_eps", C.c_double), ("dbss_dmin", C.c_int32), ("split_k", C.c_int32),
                ("svd_qr", C.c_int32), ("host_maps", C.c_int32), ("generic_gemm", C.c_int32), ("eigensolver", C.c_int32),
                ("rdm_split", C.c_int32), ("env_stride2", C.c_int32)]


class dmrg_mps_blob(C.Structure):
    _fields_ = [("k", C.c_int32), ("n_elec", C.c_int32), ("two_sz", C.c_int32), ("reserved", C.c_int32),
                ("bond_ptr", C.c_void_p), ("sec_n", C.c_void_p), ("sec_2sz", C.c_void_p), ("sec_dim", C.c_void_p),
                ("blk_ptr", C.c_void_p), ("blk_l", C.c_void_p), ("blk_s", C.c_void_p), ("blk_off", C.c_void_p),
                ("data", C.c_void_p), ("gauge", C.c_void_p),
                ("n_sectors", C.c_int64), ("n_blocks", C.c_int64), ("n_data", C.c_int64)]


class dmrg_block(C.Structure):
    _fields_ = [("l_idx", C.c_int32), ("s_i", C.c_int32), ("s_j", C.c_int32), ("r_idx", C.c_int32),
                ("rows", C.c_int32), ("cols", C.c_int32), ("offset", C.c_int64)]


class dmrg_bond_record(C.Structure):
    _fields_ = [("bond", C.c_int32), ("forward", C.c_int32), ("energy", C.c_double), ("residual", C.c_double),
                ("trunc_err", C.c_double), ("n_matvec", C.c_int32), ("kept", C.c_int32), ("nsectors", C.c_int32),
                ("converged", C.c_int32), ("nnz", C.c_int64), ("f_alg", C.c_double), ("seconds", C.c_double),
                ("seconds_matvec", C.c_double)]


class dmrg_sweep_result(C.Structure):
    _fields_ = [("energy_last", C.c_double), ("energy_min", C.c_double), ("seconds", C.c_double),
                ("n_records", C.c_int32), ("warnings", C.c_int32)]


EXPORTS = ["dmrg_default_options", "dmrg_create", "dmrg_destroy", "dmrg_last_error", "dmrg_mps_import",
           "dmrg_mps_export", "dmrg_prepare_bond", "dmrg_heff_layout", "dmrg_heff_apply", "dmrg_heff_diag",
           "dmrg_heff_stats", "dmrg_sweep", "dmrg_solve", "dmrg_sweep_stats", "dmrg_rdm12", "dmrg_rdm_stats", "dmrg_launch_count", "dmrg_flops_total", "dmrg_device_bytes",
           "dmrg_grouped_gemm", "dmrg_stack_dots", "dmrg_stack_dots_noalloc"]

lib.dmrg_last_error.restype = C.c_char_p
lib.dmrg_last_error.argtypes = [C.c_void_p]
lib.dmrg_launch_count.restype = C.c_int64
lib.dmrg_launch_count.argtypes = [C.c_void_p]
lib.dmrg_flops_total.restype = C.c_double
lib.dmrg_flops_total.argtypes = [C.c_void_p]
lib.dmrg_device_bytes.restype = C.c_int64
lib.dmrg_device_bytes.argtypes = [C.c_void_p]


class DmrgError(RuntimeError):
    def __init__(self, code, msg):
        RuntimeError.__init__(self, "dmrg_b200 status %d: %s" % (code, msg))
        self.code = code


def _check(ctx, rc):
    if rc < 0:
        raise DmrgError(rc, lib.dmrg_last_error(ctx).decode() if ctx else "invalid argument")
    return rc


def _f64(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def _ptr(a):
    return C.c_void_p(a.ctypes.data)


def _vec(v):
    """(pointer, where, stream, keepalive) of a numpy array (host) or a torch CUDA tensor (device)."""
    if isinstance(v, np.ndarray):
        assert v.dtype == np.float64 and v.flags["C_CONTIGUOUS"]
        return C.c_void_p(v.ctypes.data), DMRG_HOST, C.c_void_p(0)
    import torch
    assert v.is_cuda and v.dtype == torch.float64 and v.is_contiguous()
    return C.c_void_p(v.data_ptr()), DMRG_DEVICE, C.c_void_p(torch.cuda.current_stream(v.device).cuda_stream)


def dmrg_default_options():
    o = dmrg_options()
    lib.dmrg_default_options(C.byref(o))
    return o


def dmrg_create(k, n_elec, two_sz, h, eri, **opts):
    """-> opaque context handle.  opts: fields of dmrg_options."""
    o = dmrg_default_options()
    for key, val in opts.items():
        if not hasattr(o, key):
            raise TypeError("unknown option " + key)
        setattr(o, key, val)
    h, eri = _f64(h), _f64(eri)
    assert h.shape == (k, k) and eri.size == k ** 4
    ctx = C.c_void_p()
    rc = lib.dmrg_create(C.byref(ctx), int(k), int(n_elec), int(two_sz), _ptr(h), _ptr(eri), C.byref(o))
    if rc != 0:
        raise DmrgError(rc, "dmrg_create failed (invalid arguments or no CUDA device)")
    return ctx


def dmrg_destroy(ctx):
    return lib.dmrg_destroy(ctx)


def dmrg_mps_import(ctx, blob_arrays, k, n_elec, two_sz):
    """blob_arrays = (bond_ptr, sec_n, sec_2sz, sec_dim, blk_ptr, blk_l, blk_s, blk_off, data, gauge) as produced by
    synth.mps_to_blob_arrays."""
    bp, sn, ss, sd, kp, bl, bs, bo, data, gauge = blob_arrays
    keep = [np.ascontiguousarray(bp, np.int32), np.ascontiguousarray(sn, np.int32), np.ascontiguousarray(ss, np.int32),
            np.ascontiguousarray(sd, np.int32), np.ascontiguousarray(kp, np.int32), np.ascontiguousarray(bl, np.int32),
            np.ascontiguousarray(bs, np.int32), np.ascontiguousarray(bo, np.int64), _f64(data),
            np.ascontiguousarray(gauge, np.uint8)]
    b = dmrg_mps_blob(k, n_elec, two_sz, 0, *[a.ctypes.data for a in keep], len(keep[1]), len(keep[5]), len(keep[8]))
    return _check(ctx, lib.dmrg_mps_import(ctx, C.byref(b)))


def dmrg_mps_export(ctx, k):
    """-> (blob_arrays as in dmrg_mps_import, n_elec, two_sz)."""
    b = dmrg_mps_blob()
    _check(ctx, lib.dmrg_mps_export(ctx, C.byref(b)))
    ns, nb, nd = b.n_sectors, b.n_blocks, b.n_data
    arrs = [np.zeros(k + 2, np.int32), np.zeros(ns, np.int32), np.zeros(ns, np.int32), np.zeros(ns, np.int32),
            np.zeros(k + 1, np.int32), np.zeros(nb, np.int32), np.zeros(nb, np.int32), np.zeros(nb, np.int64),
            np.zeros(max(nd, 1), np.float64), np.zeros(k, np.uint8)]
    b2 = dmrg_mps_blob(k, 0, 0, 0, *[a.ctypes.data for a in arrs], ns, nb, nd)
    _check(ctx, lib.dmrg_mps_export(ctx, C.byref(b2)))
    arrs[8] = arrs[8][:nd]
    return tuple(arrs), b2.n_elec, b2.two_sz


def dmrg_prepare_bond(ctx, i):
    return _check(ctx, lib.dmrg_prepare_bond(ctx, int(i)))


def dmrg_heff_layout(ctx, i):
    """-> (nnz, list of (l_idx, s_i, s_j, r_idx, rows, cols, offset))."""
    nnz, nb = C.c_int64(), C.c_int32()
    _check(ctx, lib.dmrg_heff_layout(ctx, int(i), C.byref(nnz), C.byref(nb), None))
    arr = (dmrg_block * nb.value)()
    _check(ctx, lib.dmrg_heff_layout(ctx, int(i), C.byref(nnz), C.byref(nb), arr))
    return nnz.value, [(b.l_idx, b.s_i, b.s_j, b.r_idx, b.rows, b.cols, b.offset) for b in arr]


def dmrg_heff_apply(ctx, i, x, y):
    px, wx, st = _vec(x)
    py, wy, _ = _vec(y)
    assert wx == wy
    return _check(ctx, lib.dmrg_heff_apply(ctx, int(i), px, py, wx, st))


def dmrg_heff_diag(ctx, i, d):
    pd, w, st = _vec(d)
    return _check(ctx, lib.dmrg_heff_diag(ctx, int(i), pd, w, st))


def dmrg_heff_stats(ctx, i):
    fa, fe, ba = C.c_double(), C.c_double(), C.c_double()
    nt, ng = C.c_int64(), C.c_int64()
    _check(ctx, lib.dmrg_heff_stats(ctx, int(i), C.byref(fa), C.byref(fe), C.byref(ba), C.byref(nt), C.byref(ng)))
    return dict(f_alg=fa.value, f_exec=fe.value, b_alg=ba.value, nterms=nt.value, ngemm=ng.value)


def dmrg_sweep(ctx, D, k):
    """One sweep at bond dimension D -> dict(energy_last, energy_min, seconds, warnings, bonds=[records])."""
    res = dmrg_sweep_result()
    recs = (dmrg_bond_record * (2 * (k - 1)))()
    rc = _check(ctx, lib.dmrg_sweep(ctx, int(D), C.byref(res), recs))
    bonds = [dict((f, getattr(r, f)) for f, _ in dmrg_bond_record._fields_) for r in recs[:res.n_records]]
    return dict(energy_last=res.energy_last, energy_min=res.energy_min, seconds=res.seconds,
                warnings=res.warnings, status=rc, bonds=bonds)


def dmrg_solve(ctx, D, k, eps_sweep, max_sweeps):
    """Sweeps until three subsequent sweep energies differ by less than eps_sweep or max_sweeps ->
    dict(n_sweeps, energies, converged, last = result dict of the final sweep as returned by dmrg_sweep)."""
    res = dmrg_sweep_result()
    recs = (dmrg_bond_record * (2 * (k - 1)))()
    n = C.c_int32(0)
    en = np.zeros(max_sweeps)
    rc = _check(ctx, lib.dmrg_solve(ctx, int(D), C.c_double(eps_sweep), int(max_sweeps), C.byref(n), _ptr(en), C.byref(res), recs))
    bonds = [dict((f, getattr(r, f)) for f, _ in dmrg_bond_record._fields_) for r in recs[:res.n_records]]
    return dict(n_sweeps=n.value, energies=en[:n.value].copy(), status=rc,
                last=dict(energy_last=res.energy_last, energy_min=res.energy_min, seconds=res.seconds,
                          warnings=res.warnings, bonds=bonds))


class dmrg_sweep_stats_t(C.Structure):
    _fields_ = [(n, C.c_double) for n in ("seconds_environments", "seconds_restore", "seconds_regrow",
                                          "seconds_spill_wait", "seconds_maps", "seconds_davidson", "seconds_matvec",
                                          "seconds_split", "seconds_renormalise", "bytes_spilled", "bytes_restored")] + \
               [(n, C.c_int64) for n in ("peak_device_bytes", "host_pool_bytes", "est_stack_bytes", "est_max_block_bytes")] + \
               [("env_stride", C.c_int32), ("host_spill", C.c_int32), ("env_stride2", C.c_int32), ("reserved", C.c_int32)]


def dmrg_sweep_stats(ctx):
    """Phase seconds and environment-stack accounting of the last dmrg_sweep -> dict."""
    st = dmrg_sweep_stats_t()
    _check(ctx, lib.dmrg_sweep_stats(ctx, C.byref(st)))
    return dict((f, getattr(st, f)) for f, _ in dmrg_sweep_stats_t._fields_)


def dmrg_rdm12(ctx, k, want_2rdm=True, out=None):
    """-> (gamma [k,k], Gamma [k,k,k,k] or None) as numpy arrays; with out = (gamma, Gamma) torch CUDA tensors the
    results are written to those device buffers (on torch's current stream) and returned."""
    if out is not None:
        g, G = out
        pg, where, stream = _vec(g)
        pG = _vec(G)[0] if (want_2rdm and G is not None) else None
        _check(ctx, lib.dmrg_rdm12(ctx, pg, pG, where, stream))
        return g, G
    g = np.zeros((k, k))
    G = np.zeros((k, k, k, k)) if want_2rdm else None
    _check(ctx, lib.dmrg_rdm12(ctx, _ptr(g), _ptr(G) if want_2rdm else None, DMRG_HOST, None))
    return g, G


class dmrg_rdm_stats_t(C.Structure):
    _fields_ = [(n, C.c_double) for n in ("seconds", "seconds_host", "seconds_renormalise", "bytes_streamed", "flops",
                                          "stream_bytes", "stream_seconds", "gemm_seconds")]


def dmrg_rdm_stats(ctx):
    st = dmrg_rdm_stats_t()
    _check(ctx, lib.dmrg_rdm_stats(ctx, C.byref(st)))
    return dict((f, getattr(st, f)) for f, _ in dmrg_rdm_stats_t._fields_)


def dmrg_launch_count(ctx):
    return lib.dmrg_launch_count(ctx)


def dmrg_device_bytes(ctx):
    return lib.dmrg_device_bytes(ctx)


def dmrg_grouped_gemm(tasks, segs, stream=None, generic=False):
    """Kernel-level entry for the unit parity tests.  tasks: list of dict(C=ptr, ldc, M, N, seg_begin, seg_count,
    flags); segs: list of dict(A=ptr, B=ptr, lda, ldb, K, flags, alpha); pointers are device addresses (ints).
    generic: force the cp.async kernel.  Returns the device milliseconds of the kernel launch."""
    nt, ns = len(tasks), len(segs)
    i64 = lambda key, src: np.array([s[key] for s in src], dtype=np.int64)
    i32 = lambda key, src: np.array([s[key] for s in src], dtype=np.int32)
    arrs = [i64("C", tasks), i32("ldc", tasks), i32("M", tasks), i32("N", tasks), i32("seg_begin", tasks),
            i32("seg_count", tasks), i32("flags", tasks)]
    sarr = [i64("A", segs), i64("B", segs), i32("lda", segs), i32("ldb", segs), i32("K", segs), i32("flags", segs),
            np.array([s["alpha"] for s in segs], dtype=np.float64)]
    ms = C.c_double(0.0)
    rc = lib.dmrg_grouped_gemm(nt, *[_ptr(a) for a in arrs], ns, *[_ptr(a) for a in sarr], 1 if generic else 0,
                               C.byref(ms), C.c_void_p(stream or 0))
    if rc != 0:
        raise DmrgError(rc, "dmrg_grouped_gemm failed")
    return ms.value


def dmrg_stack_dots_noalloc(S_ptr, lds, nrows, M_ptr, ldm, nc, K, E_ptr, ldE, stream=None):
    """Allocation-free variant of dmrg_stack_dots (static device scratch of DMRG_STACK_DOTS_NOALLOC_MAX_SCRATCH doubles):
    asynchronous on `stream`, no timing.  Raises DmrgError(DMRG_ENOMEM) when the problem exceeds the static scratch."""
    rc = lib.dmrg_stack_dots_noalloc(C.c_void_p(S_ptr), C.c_int64(lds), int(nrows), C.c_void_p(M_ptr), C.c_int64(ldm), int(nc),
                                     C.c_int64(K), C.c_void_p(E_ptr), int(ldE), C.c_void_p(stream or 0))
    if rc == DMRG_ENOMEM:
        raise DmrgError(rc, "dmrg_stack_dots_noalloc: problem needs more than the static scratch (%d doubles); use dmrg_stack_dots"
                        % DMRG_STACK_DOTS_NOALLOC_MAX_SCRATCH)
    if rc != 0:
        raise DmrgError(rc, "dmrg_stack_dots_noalloc failed")
    return rc


DMRG_STACK_DOTS_NOALLOC_MAX_SCRATCH = 1 << 20
_bench_lib = None


def dmrg_fp64_probe(kind, iters=20000, ctas_per_sm=3, size=8192, reps=3, stream=None):
    """FP64 ceiling probe of the measurement-only library libdmrg_b200_bench.so (include/dmrg_b200_bench.h; kind 0 DMMA,
    1 DFMA, 2 DMMA fed by LDS, 3 cuBLAS DGEMM size^3): dict(tflops, ms).  Not part of the product library."""
    global _bench_lib
    if _bench_lib is None:
        path = os.path.join(_HERE, "libdmrg_b200_bench.so")
        if not os.path.exists(path):
            raise ImportError(path + " not found: run __graft_entry__.build()")
        _bench_lib = C.CDLL(path)
    tf, ms = C.c_double(0.0), C.c_double(0.0)
    rc = _bench_lib.dmrg_bench_fp64_probe(int(kind), int(iters), int(ctas_per_sm), int(size), int(reps), C.byref(tf),
                                          C.byref(ms), C.c_void_p(stream or 0))
    if rc != 0:
        raise DmrgError(rc, "dmrg_bench_fp64_probe failed")
    return {"tflops": tf.value, "ms": ms.value}


def dmrg_flops_total(ctx):
    """Unpadded flops of every grouped-GEMM launch of the context since creation."""
    return float(lib.dmrg_flops_total(ctx))


def dmrg_stack_dots(S_ptr, lds, nrows, M_ptr, ldm, nc, K, E_ptr, ldE, stream=None):
    """E[r*ldE + c] = sum_k S[r*lds + k] * M[c*ldm + k] on device buffers (addresses as ints) -> device milliseconds."""
    ms = C.c_double(0.0)
    rc = lib.dmrg_stack_dots(C.c_void_p(S_ptr), C.c_int64(lds), int(nrows), C.c_void_p(M_ptr), C.c_int64(ldm), int(nc),
                             C.c_int64(K), C.c_void_p(E_ptr), int(ldE), C.byref(ms), C.c_void_p(stream or 0))
    if rc != 0:
        raise DmrgError(rc, "dmrg_stack_dots failed")
    return ms.value
