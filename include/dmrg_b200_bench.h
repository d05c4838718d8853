/* dmrg_b200_bench.h - measurement-only companion of dmrg_b200.h, built into libdmrg_b200_bench.so.  Nothing of the hot
 * path lives here and the product library does not link it (or cuBLAS): bench.py uses it for the FP64 roofline
 * denominators SURVEY.md 8(d) D2 asks for. */
#ifndef DMRG_B200_BENCH_H
#define DMRG_B200_BENCH_H
#ifdef __cplusplus
extern "C" {
#endif

/* FP64 ceiling probe.  kind 0: register-resident DMMA.8x8x4 loop; 1: register-resident DFMA loop; 2: the DMMA loop fed
 * from shared memory with the GEMM kernel's fragment pattern; 3: cublasDgemm size^3.  iters: inner iterations (kinds 0-2)
 * or DGEMM calls per timing (kind 3); ctas_per_sm: resident 4-warp CTAs per SM (kinds 0-2).  Best of `reps` launches timed
 * with CUDA events on `cuda_stream` (a cudaStream_t); *tflops and *ms are HOST outputs.  Returns 0, -1 (bad argument),
 * -3 (out of device memory) or -4 (CUDA / cuBLAS failure). */
int dmrg_bench_fp64_probe(int kind, int iters, int ctas_per_sm, int size, int reps, double* tflops, double* ms,
                          void* cuda_stream);

#ifdef __cplusplus
}
#endif
#endif
