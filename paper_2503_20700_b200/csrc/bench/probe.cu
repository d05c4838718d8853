// FP64 ceiling probes for the roofline denominator:
// register-resident DMMA.8x8x4 and DFMA issue-rate loops, the same DMMA loop fed from shared memory with the
// fragment pattern of the grouped GEMM kernel, and cuBLAS DGEMM on a square problem.  Measurement only: built into the
// separate library libdmrg_b200_bench.so (include/dmrg_b200_bench.h); the product library neither contains nor links it.
#include <cublas_v2.h>
#include <cuda_runtime.h>

#include <cstdint>

#include "../../../include/dmrg_b200_bench.h"

namespace dmrg {

namespace {

constexpr int GEMM_BM = 64, GEMM_BN = 64, GEMM_BK = 16;   // tile shape of the product GEMM kernel (stated here: no shared header)

__device__ __forceinline__ void dmma_p(double& d0, double& d1, double a, double b) {
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n"
                 : "+d"(d0), "+d"(d1)
                 : "d"(a), "d"(b));
}

// 16 independent accumulator fragments per warp, 4 + 4 operand registers: the register shape of the GEMM consumer
__global__ void __launch_bounds__(128) probe_dmma(int iters, double* sink) {
    double acc[4][4][2];
    double a[4], b[4];
    for (int i = 0; i < 4; ++i) {
        a[i] = 1.0 + 1e-9 * (threadIdx.x + i);
        b[i] = 1.0 - 1e-9 * (threadIdx.x + 4 * i);
        for (int j = 0; j < 4; ++j) acc[i][j][0] = acc[i][j][1] = 0.0;
    }
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int i = 0; i < 4; ++i)
#pragma unroll
            for (int j = 0; j < 4; ++j) dmma_p(acc[i][j][0], acc[i][j][1], a[i], b[j]);
    }
    double s = 0.0;
    for (int i = 0; i < 4; ++i)
        for (int j = 0; j < 4; ++j) s += acc[i][j][0] + acc[i][j][1];
    if (s == 12345.678) sink[0] = s;
}

__global__ void __launch_bounds__(128) probe_dfma(int iters, double* sink) {
    double acc[32];
    const double a = 1.0 + 1e-9 * threadIdx.x, b = 1e-9 * threadIdx.x;
    for (int i = 0; i < 32; ++i) acc[i] = i;
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int i = 0; i < 32; ++i) acc[i] = fma(acc[i], a, b);
    }
    double s = 0.0;
    for (int i = 0; i < 32; ++i) s += acc[i];
    if (s == 12345.678) sink[0] = s;
}

// the consumer inner loop of seg_gemm_tma_kernel on a resident shared-memory stage: 8 LDS.64 per 16 DMMA
__global__ void __launch_bounds__(128) probe_dmma_lds(int iters, double* sink) {
    constexpr int LDK = GEMM_BK + 4;
    __shared__ double As[GEMM_BM * LDK], Bs[GEMM_BN * LDK];
    for (int i = threadIdx.x; i < GEMM_BM * LDK; i += blockDim.x) { As[i] = 1.0 + 1e-9 * i; Bs[i] = 1.0 - 1e-9 * i; }
    __syncthreads();
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int wm = (warp >> 1) * 32, wn = (warp & 1) * 32, fr = lane >> 2, fc = lane & 3;
    double acc[4][4][2];
    for (int i = 0; i < 4; ++i)
        for (int j = 0; j < 4; ++j) acc[i][j][0] = acc[i][j][1] = 0.0;
    const int a_off = (wm + fr) * LDK + fc, b_off = (wn + fr) * LDK + fc;
    for (int it = 0; it < iters; ++it) {
        const int kk = (it * 4) & (GEMM_BK - 1);
        double a[4], b[4];
#pragma unroll
        for (int i = 0; i < 4; ++i) a[i] = As[a_off + kk + 8 * i * LDK];
#pragma unroll
        for (int j = 0; j < 4; ++j) b[j] = Bs[b_off + kk + 8 * j * LDK];
#pragma unroll
        for (int i = 0; i < 4; ++i)
#pragma unroll
            for (int j = 0; j < 4; ++j) dmma_p(acc[i][j][0], acc[i][j][1], a[i], b[j]);
    }
    double s = 0.0;
    for (int i = 0; i < 4; ++i)
        for (int j = 0; j < 4; ++j) s += acc[i][j][0] + acc[i][j][1];
    if (s == 12345.678) sink[0] = s;
}

}  // namespace

// kind 0: DMMA registers only; 1: DFMA; 2: DMMA fed by LDS; 3: cuBLAS DGEMM n x n x n (iters = repetitions, n = size)
// ctas_per_sm resident CTAs of 4 warps.  Returns 0 on success; tflops and ms of the best of `reps` timed launches.
static int fp64_probe(int kind, int iters, int ctas_per_sm, int size, int reps, double* tflops, double* ms, cudaStream_t st) {
    int dev = 0, sms = 148;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0);
    cudaEventCreate(&e1);
    double best = 1e30, flops = 0.0;
    if (kind == 3) {
        const int64_t n = size;
        double *A = nullptr, *B = nullptr, *Cm = nullptr;
        if (cudaMalloc(&A, n * n * 8) || cudaMalloc(&B, n * n * 8) || cudaMalloc(&Cm, n * n * 8)) return -3;
        cudaMemsetAsync(A, 0, n * n * 8, st);
        cudaMemsetAsync(B, 0, n * n * 8, st);
        cublasHandle_t h;
        if (cublasCreate(&h) != CUBLAS_STATUS_SUCCESS) return -4;
        cublasSetStream(h, st);
        const double one = 1.0, zero = 0.0;
        flops = 2.0 * n * n * n * iters;
        for (int r = 0; r < reps + 1; ++r) {
            cudaEventRecord(e0, st);
            for (int it = 0; it < iters; ++it)
                cublasDgemm(h, CUBLAS_OP_N, CUBLAS_OP_N, (int)n, (int)n, (int)n, &one, A, (int)n, B, (int)n, &zero, Cm, (int)n);
            cudaEventRecord(e1, st);
            cudaEventSynchronize(e1);
            float t = 0;
            cudaEventElapsedTime(&t, e0, e1);
            if (r > 0 && t < best) best = t;
        }
        cublasDestroy(h);
        cudaFree(A); cudaFree(B); cudaFree(Cm);
    } else {
        double* sink = nullptr;
        if (cudaMalloc(&sink, 8)) return -3;
        const int grid = sms * ctas_per_sm;
        // per CTA: 4 warps; DMMA kinds: 16 DMMA x 512 flop per warp per iteration; DFMA: 32 x 32 lanes x 2 flop
        flops = (kind == 1 ? 32.0 * 32 * 2 : 16.0 * 512) * 4.0 * (double)grid * (double)iters;
        for (int r = 0; r < reps + 1; ++r) {
            cudaEventRecord(e0, st);
            if (kind == 0) probe_dmma<<<grid, 128, 0, st>>>(iters, sink);
            else if (kind == 1) probe_dfma<<<grid, 128, 0, st>>>(iters, sink);
            else probe_dmma_lds<<<grid, 128, 0, st>>>(iters, sink);
            cudaEventRecord(e1, st);
            cudaEventSynchronize(e1);
            float t = 0;
            cudaEventElapsedTime(&t, e0, e1);
            if (r > 0 && t < best) best = t;
        }
        cudaFree(sink);
    }
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    if (cudaGetLastError() != cudaSuccess) return -4;
    *ms = best;
    *tflops = flops / (best * 1e-3) / 1e12;
    return 0;
}

}  // namespace dmrg

extern "C" int dmrg_bench_fp64_probe(int kind, int iters, int ctas_per_sm, int size, int reps, double* tflops, double* ms,
                                     void* cuda_stream) {
    if (kind < 0 || kind > 3 || iters < 1 || reps < 1 || !tflops || !ms) return -1;
    if (kind < 3 && (ctas_per_sm < 1 || ctas_per_sm > 16)) return -1;
    if (kind == 3 && (size < 1 || size > 32768)) return -1;
    const int rc = dmrg::fp64_probe(kind, iters, ctas_per_sm, size, reps, tflops, ms, (cudaStream_t)cuda_stream);
    return rc == 0 ? 0 : (rc == -3 ? -3 : -4);
}
