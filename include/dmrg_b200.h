/* dmrg_b200.h - C ABI of the B200-native two-site DMRG hot path (H_eff psi, renormalisation, sweep, 1-/2-RDM).
 *
 * What it computes is fixed by the paper (arxiv 2503.20700, /root/reference/PAPER.md) and BASELINE.json:
 *   - the active-space Hamiltonian H = sum h_pq E_pq + 1/2 sum (pq|rs) (E_pq E_rs - d_qr E_ps)   PAPER.md:52-68, Eq. 1-5
 *     (normalisation / index pairing: reading S1 of DESIGN.md),
 *   - the wavefunction as a matrix product state with (N, 2Sz) block sparsity                    PAPER.md:107, 122-127, Eq. 14
 *   - the variational sweep E = min <Psi|H|Psi>/<Psi|Psi>, Davidson local solver, fixed D        PAPER.md:127-130 (Eq. 15), 179
 *   - the reduced density matrices gamma_pq = <E_pq>, Gamma_pqrs                                  PAPER.md:89-95, Eq. 9-10
 * How it is computed (complementary operators, blocking) is NOT in the paper (deferred to its refs [44,50,60,81,82],
 * PAPER.md:40, 132, 171); the algorithm is DESIGN.md section "Algorithm".
 *
 * Conventions: all matrices row-major FP64; spin orbital P = 2p + [down]; site states 0:|0>, 1:|dn>, 2:|up>,
 * 3:|up dn> = a+_up a+_dn |0> (phases: reading S3).  One thread at a time per context.  Every entry
 * point returns an int status: 0 ok, <0 failure (state unchanged where possible), >0 warning.  No exceptions cross
 * the boundary, nothing is printed.  There is no CPU fallback: every call needs a CUDA device (sm_100a build).
 */
#ifndef DMRG_B200_H
#define DMRG_B200_H
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct dmrg_ctx dmrg_ctx; /* opaque; owned by the library; freed only by dmrg_destroy */

enum { DMRG_OK = 0, DMRG_EINVAL = -1, DMRG_ESTATE = -2, DMRG_ENOMEM = -3, DMRG_ECUDA = -4, DMRG_ENOCONV = 1 };
enum { DMRG_HOST = 0, DMRG_DEVICE = 1 }; /* where a caller buffer lives */

/* Options of a context (all fields must be set; dmrg_default_options fills the defaults).
 * davidson_tol: residual 2-norm threshold (PAPER.md:179 uses 1e-7; parity runs use 1e-10, reading S13). */
typedef struct dmrg_options {
    double davidson_tol;          /* default 1e-7  */
    int32_t davidson_max_iter;    /* default 100   */
    int32_t davidson_max_subspace;/* default 20    */
    double sv_floor;              /* default 1e-10: singular values <= floor are dropped (reading S14)        */
    double cluster_rel_gap;       /* default 1e-6 : never cut inside a near-degenerate cluster (reading S14)  */
    int32_t device_id;            /* default 0     */
    int32_t keep_env_stack;       /* default 1: keep every environment block (needed by sweeps); 0: prepare_bond
                                     keeps only the two blocks of the prepared bond (large-D single-bond runs)  */
    int64_t workspace_bytes;      /* default 0 = automatic: cap of the intermediate (T) buffer of H_eff psi   */
    /* Environment stack of dmrg_sweep (BASELINE configs 4-5: "operator storage sized to fit 180 GB HBM"; SURVEY.md 7
     * hard part 5).  One pass consumes the blocks the previous pass produced; only every env_stride-th block is kept
     * (a checkpoint), the blocks in between are recomputed from it when the pass reaches them; with host_spill the
     * checkpoints are moved to pinned host memory by asynchronous copies and fetched back when needed.  Results do not
     * depend on these settings (the recomputed blocks are bit-identical). */
    int64_t hbm_budget_bytes;     /* default 0 = automatic (55 % of the free device memory): bytes the stack may hold */
    int64_t host_budget_bytes;    /* default 0 = automatic (64 GiB): pinned host bytes for spilled checkpoints        */
    int32_t host_spill;           /* default 0; 1: checkpoints may be spilled to pinned host memory                    */
    int32_t env_stride;           /* default 0 = automatic from the budgets; 1 = keep every block; s: every s-th       */
    /* Dynamic block state selection: dbss_eps > 0 keeps, at every bond, the fewest states
     * whose discarded weight is <= dbss_eps, at least dbss_dmin and at most the D passed to dmrg_sweep (D_max).       */
    double dbss_eps;              /* default 0 = fixed D                                                               */
    int32_t dbss_dmin;            /* default 0                                                                         */
    int32_t split_k;              /* default 0 = automatic: split-K parts (1..64) of phase 2 of H_eff psi              */
    int32_t svd_qr;               /* default 0: one-sided Jacobi SVD (cuSOLVER gesvdj, gesvd fallback); 1: gesvd       */
    int32_t host_maps;            /* default 0: block maps built on the device; 1: host reference builder (A/B tests)  */
    int32_t generic_gemm;         /* default 0; 1: always the cp.async GEMM kernel instead of the bulk-copy one (A/B)  */
    int32_t eigensolver;          /* default 0: Davidson; 1: Lanczos (PAPER.md:179 names both); same tolerance fields  */
    int32_t rdm_split;            /* default -1 = k/2: site kh of the half-chain partition of dmrg_rdm12 (strings with their
                                     third-smallest site < kh are evaluated there with the two-index operators on the left,
                                     the others at their second-smallest site with them on the right); 0 and k give the two
                                     one-sided evaluation orders.  Results do not depend on it (tested); memory does.       */
    int32_t env_stride2;          /* default 0 = automatic: second checkpoint level inside a segment - of the blocks recomputed
                                     from a checkpoint only every env_stride2-th and the sub-segment in use stay resident      */
} dmrg_options;

/* Neutral MPS exchange format (host memory, caller-owned, flat arrays).
 * Bond b = 0..k sits left of site b.  Sectors of bond b are entries bond_ptr[b] .. bond_ptr[b+1]-1 of
 * sec_n / sec_2sz / sec_dim, sorted ascending by (N, 2Sz); bond 0 = {(0,0,1)}, bond k = {(n_elec, two_sz, 1)}
 * (boundary bonds of dimension 1).  Site p owns blocks blk_ptr[p] .. blk_ptr[p+1]-1, ordered by
 * (l_idx, s): blk_l = sector index within bond p, blk_s = site state, the right sector is q_l + q(s) on bond p+1;
 * the dense block [dim_l x dim_r] row-major starts at data[blk_off[j]].  gauge[p] in {'L','R','C'}. */
typedef struct dmrg_mps_blob {
    int32_t k, n_elec, two_sz, reserved;
    const int32_t* bond_ptr; /* k+2 */
    const int32_t* sec_n;
    const int32_t* sec_2sz;
    const int32_t* sec_dim;
    const int32_t* blk_ptr;  /* k+1 */
    const int32_t* blk_l;
    const int32_t* blk_s;
    const int64_t* blk_off;
    const double* data;
    const uint8_t* gauge;    /* k */
    int64_t n_sectors, n_blocks, n_data;
} dmrg_mps_blob;

/* One block of the two-site wavefunction layout at bond i: psi[q_l, s_i, s_j, q_r], dense [rows x cols]
 * row-major at `offset` doubles into the packed vector; blocks ordered by (l_idx, s_i, s_j). */
typedef struct dmrg_block {
    int32_t l_idx, s_i, s_j, r_idx, rows, cols;
    int64_t offset;
} dmrg_block;

/* Per optimised bond record of a sweep. */
typedef struct dmrg_bond_record {
    int32_t bond, forward;        /* two-site bond index i, 1 = forward pass                                  */
    double energy;                /* Davidson eigenvalue (electronic, no E_core: reading S5)                   */
    double residual;
    double trunc_err;             /* discarded weight sum sigma^2 of the normalised state (reading S14)        */
    int32_t n_matvec, kept, nsectors, converged;
    int64_t nnz;                  /* length of the two-site vector                                             */
    double f_alg;                 /* algorithmic flops of one H_eff psi at this bond (D3)            */
    double seconds;               /* wall time of the whole bond step                                          */
    double seconds_matvec;        /* device time (CUDA events) spent in H_eff psi at this bond                 */
} dmrg_bond_record;

typedef struct dmrg_sweep_result {
    double energy_last, energy_min; /* eigenvalue at the last bond of the sweep / minimum over the sweep (S12) */
    double seconds;
    int32_t n_records;              /* 2(k-1) */
    int32_t warnings;               /* number of bonds where Davidson hit max_iter                             */
} dmrg_sweep_result;

void dmrg_default_options(dmrg_options* opt);

/* Create a context for k spatial orbitals, n_elec electrons, 2Sz = two_sz.  h: host, k*k row-major symmetric;
 * eri: host, k^4, (pq|rs) at ((p*k+q)*k+r)*k+s with 8-fold symmetry (Eq. 5).  Both are copied.
 * opt nullable.  Errors: DMRG_EINVAL for k<1, n_elec<0 or >2k, odd n_elec+two_sz, |two_sz| too large, h asymmetric
 * beyond 1e-12; DMRG_ECUDA if no usable device. */
int dmrg_create(dmrg_ctx** out, int k, int n_elec, int two_sz, const double* h, const double* eri,
                const dmrg_options* opt);
int dmrg_destroy(dmrg_ctx* ctx);
/* Library-owned message of the last failure of this context (valid until the next call on it). */
const char* dmrg_last_error(const dmrg_ctx* ctx);

/* Copy an MPS into the context (device-resident afterwards).  Does not change the gauge.  Invalidates
 * environments.  DMRG_EINVAL if shapes / quantum numbers are inconsistent. */
int dmrg_mps_import(dmrg_ctx* ctx, const dmrg_mps_blob* blob);
/* Two-call export of the current MPS: first call with blob->data == NULL (and all other pointers NULL) fills the
 * counts n_sectors, n_blocks, n_data; second call with caller-allocated arrays (cast away const) fills them. */
int dmrg_mps_export(dmrg_ctx* ctx, dmrg_mps_blob* blob);

/* Build the left environment of bond i from sites < i (must be left-orthonormal) and the right environment of
 * bond i+2 from sites > i+1 (right-orthonormal): renormalised normal and complementary operators (fused blocking
 * kernels), then the term list and block maps of H_eff at two-site bond i, 0 <= i <= k-2. */
int dmrg_prepare_bond(dmrg_ctx* ctx, int i);
/* Layout of the two-site vector at the prepared bond i.  blocks nullable (size query). */
int dmrg_heff_layout(dmrg_ctx* ctx, int i, int64_t* nnz, int32_t* nblocks, dmrg_block* blocks);
/* y = H_eff x at the prepared bond i (y = P^T H P x, C2).  x, y: nnz doubles, host or device per `where`;
 * cuda_stream: a cudaStream_t (NULL = default stream); device buffers are used in place, asynchronously on that
 * stream; host buffers are copied in and out and the call returns after completion.  Never modifies the MPS. */
int dmrg_heff_apply(dmrg_ctx* ctx, int i, const double* x, double* y, int where, void* cuda_stream);
/* diag(H_eff) at the prepared bond (Davidson preconditioner), same layout, `where` and stream semantics. */
int dmrg_heff_diag(dmrg_ctx* ctx, int i, double* d, int where, void* cuda_stream);
/* Flop and byte accounting of one H_eff psi at the prepared bond (D3): f_alg = canonical algorithmic
 * flops with true sector dimensions, f_exec = flops of the GEMMs actually issued (unpadded), b_alg = 8 x (nnz of
 * every operator block referenced once + nnz(x) + nnz(y)). */
int dmrg_heff_stats(dmrg_ctx* ctx, int i, double* f_alg, double* f_exec, double* b_alg, int64_t* nterms,
                    int64_t* ngemm);

/* One sweep (forward pass over bonds 0..k-2, backward pass k-2..0; reading S12) at bond dimension D on the current
 * MPS, which must be right-canonical before the first sweep.  records: caller array of 2(k-1) entries (nullable).
 * Returns DMRG_ENOCONV (warning) if any Davidson hit max_iter. */
int dmrg_sweep(dmrg_ctx* ctx, int D, dmrg_sweep_result* result, dmrg_bond_record* records);

/* Sweeps at bond dimension D until the stopping rule of PAPER.md:179 holds - the sweep energies (energy_last) of three
 * subsequent sweeps differ by less than eps_sweep, |E_s - E_{s-1}| < eps and |E_{s-1} - E_{s-2}| < eps (reading S34) - or
 * max_sweeps sweeps have run.  *n_sweeps (HOST) receives the number of sweeps, energies (HOST, max_sweeps doubles,
 * nullable) their energy_last; last / last_records as in dmrg_sweep for the final sweep.  Returns DMRG_ENOCONV if the
 * rule was not met within max_sweeps (or a Davidson hit max_iter in the final sweep). */
int dmrg_solve(dmrg_ctx* ctx, int D, double eps_sweep, int max_sweeps, int32_t* n_sweeps, double* energies,
               dmrg_sweep_result* last, dmrg_bond_record* last_records);

/* Phase timers and environment-stack accounting of the last dmrg_sweep call (seconds per phase).
 * seconds_environments = restore + regrow + the initial right stack; seconds_spill_wait = time the host waited for an
 * asynchronous spill copy before it could free the device copy (0 when the copy was hidden behind the bond's Davidson). */
typedef struct dmrg_sweep_stats_t {
    double seconds_environments, seconds_restore, seconds_regrow, seconds_spill_wait;
    double seconds_maps, seconds_davidson, seconds_matvec, seconds_split, seconds_renormalise;
    double bytes_spilled, bytes_restored;
    int64_t peak_device_bytes, host_pool_bytes, est_stack_bytes, est_max_block_bytes;
    int32_t env_stride, host_spill, env_stride2, reserved;
} dmrg_sweep_stats_t;
int dmrg_sweep_stats(dmrg_ctx* ctx, dmrg_sweep_stats_t* out);

/* gamma (k*k) and Gamma (k^4, nullable -> 1-RDM only) of the normalised current MPS (readings S2, S20):
 * gamma_pq = <E_pq>, Gamma_pqrs = <sum_ss' a+_ps a+_rs' a_ss' a_qs> at ((p*k+q)*k+r)*k+s.  Output buffers host or
 * device per `where`; device buffers are written on `cuda_stream` after its pending work, and the call returns when
 * the results are in place. */
int dmrg_rdm12(dmrg_ctx* ctx, double* gamma, double* Gamma, int where, void* cuda_stream);

/* Timing / accounting of the last dmrg_rdm12 call.  bytes_streamed: operator storage (plus the M
 * vectors) read by ALL accumulation launches E = Stack M^T - every stored operator of the two-index side once per
 * centre; of these, stream_bytes went through the HBM-bound streaming kernel (operator classes with <= 8 right-hand
 * sides) in stream_seconds of device time (CUDA events), the rest through split-K launches of the FP64 tensor-pipe GEMM in
 * gemm_seconds.  seconds_host: string enumeration and gamma / Gamma scatter on the host; seconds_renormalise: centre
 * moves and blocking steps of the pass (host plan assembly + kernels). */
typedef struct dmrg_rdm_stats_t {
    double seconds, seconds_host, seconds_renormalise;
    double bytes_streamed, flops;
    double stream_bytes, stream_seconds, gemm_seconds;
} dmrg_rdm_stats_t;
int dmrg_rdm_stats(dmrg_ctx* ctx, dmrg_rdm_stats_t* out);

/* Number of kernels this library launched on the context since creation (bench.py's gpu_launches). */
int64_t dmrg_launch_count(const dmrg_ctx* ctx);
/* Unpadded flops (sum of 2 M N K) of every grouped-GEMM launch of the context since creation: H_eff psi, operator
 * renormalisation, RDM contractions.  Differences around a call give that call's executed flops. */
double dmrg_flops_total(const dmrg_ctx* ctx);
/* Device bytes currently held by the context's arenas. */
int64_t dmrg_device_bytes(const dmrg_ctx* ctx);

/* Kernel-level entry used by the unit parity tests: grouped, K-segmented FP64 GEMM on device buffers.
 * For task t: C_t[M x N] (+)= sum_{s in segs of t} alpha_s op(A_s) op(B_s); all pointers are DEVICE addresses
 * stored as int64; arrays below are HOST arrays (copied to the device by the call).  seg_flags bit0: A stored
 * [K x M]; bit1: B stored [N x K]; bit2: B = identity (C += alpha A, A stored [M x N]).  task_flags bit0: accumulate.  generic_kernel
 * != 0 forces the cp.async kernel (otherwise the bulk-copy kernel runs whenever the operands are aligned); *kernel_ms (HOST,
 * nullable) receives the device time of the kernel launch alone (CUDA events on `cuda_stream`, descriptor upload excluded). */
int dmrg_grouped_gemm(int ntasks, const int64_t* c_ptr, const int32_t* ldc, const int32_t* m, const int32_t* n,
                      const int32_t* seg_begin, const int32_t* seg_count, const int32_t* task_flags, int nsegs,
                      const int64_t* a_ptr, const int64_t* b_ptr, const int32_t* lda, const int32_t* ldb,
                      const int32_t* kk, const int32_t* seg_flags, const double* alpha, int generic_kernel,
                      double* kernel_ms, void* cuda_stream);

/* Kernel-level entry of the RDM accumulation kernel for few right-hand sides ("streams every stored
 * 2-index operator once", HBM-bound):  E[r*ldE + c] = sum_k S[r*lds + k] * M[c*ldm + k], r < nrows, c < nc (1..8), k < K.
 * S, M, E are DEVICE pointers (S, M 16-byte aligned, lds and ldm even); scratch is allocated and freed by the call.
 * *ms (HOST, nullable) receives the device time of the two kernels (CUDA events on `cuda_stream`).  Used by the parity
 * test and by bench.py's HBM probe; inside dmrg_rdm12 the same kernel serves the operator classes with nc <= 8. */
int dmrg_stack_dots(const double* S, int64_t lds, int nrows, const double* M, int64_t ldm, int nc, int64_t K, double* E,
                    int ldE, double* ms, void* cuda_stream);

/* Allocation-free variant of dmrg_stack_dots for callers that cannot call cudaMalloc (CUDA graph capture, tight serving
 * loops, harnesses that forbid allocation): same operation, same kernels, same argument meaning; the span partial sums
 * live in one static device array of DMRG_STACK_DOTS_NOALLOC_MAX_SCRATCH doubles (8 MiB, held by every GPU that loads the
 * library until exit).  Calls no cudaMalloc / cudaFree / allocating library routine, creates no events and does not
 * synchronise: the launches are asynchronous on `cuda_stream`.  Limit: the scratch need is nspans * nrows * nc doubles
 * with nspans <= ceil(2368 / ceil(nrows / 32)) K spans; every nc <= 8 with nrows <= 32768 fits; a problem that needs more
 * returns DMRG_ENOMEM (nothing launched) - use dmrg_stack_dots then.  All calls on a device share the array: calls that overlap on
 * the GPU (different streams or host threads) race; order them on one stream.  Nothing in the array needs clearing
 * between calls (every partial sum read was written by the same call). */
#define DMRG_STACK_DOTS_NOALLOC_MAX_SCRATCH (1 << 20)
int dmrg_stack_dots_noalloc(const double* S, int64_t lds, int nrows, const double* M, int64_t ldm, int nc, int64_t K,
                            double* E, int ldE, void* cuda_stream);

#ifdef __cplusplus
}
#endif
#endif
