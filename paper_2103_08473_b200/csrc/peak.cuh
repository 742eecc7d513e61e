// FP64 tensor-pipe yardstick: register-resident DMMA.8x8x4 issue loop (no memory traffic).  Its rate is the
// denominator of every "fraction of FP64 peak" the benchmark reports.
#pragma once
#include "gemm_dmma.cuh"

__global__ void __launch_bounds__(512) dmma_peak_kernel(double* out, int iters, double a0, double b0)
{
    double c[8][2];
#pragma unroll
    for (int i = 0; i < 8; i++) { c[i][0] = 0.0; c[i][1] = 0.0; }
    const double a = a0 + threadIdx.x, b = b0;
    for (int it = 0; it < iters; it++) {
#pragma unroll
        for (int i = 0; i < 8; i++) dmma884(c[i][0], c[i][1], a, b);
    }
    double s = 0.0;
#pragma unroll
    for (int i = 0; i < 8; i++) s += c[i][0] + c[i][1];
    if (s == 123.456) out[0] = s;   // keep the loop alive without a store in the common case
}

// runs ~`launches` launches of ~1 ms each; returns the best-launch rate in TFLOP/s (512 flop per warp-level DMMA)
static int measure_fp64_peak(cudaStream_t st, double* scratch, int launches, double* tflops)
{
    int dev = 0, nsm = 0;
    CCSD_CUDA_TRY(cudaGetDevice(&dev));
    CCSD_CUDA_TRY(cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, dev));
    cudaEvent_t e0, e1;
    CCSD_CUDA_TRY(cudaEventCreate(&e0));
    CCSD_CUDA_TRY(cudaEventCreate(&e1));
    const int iters = 40000;
    dmma_peak_kernel<<<nsm, 512, 0, st>>>(scratch, 1000, 1.0, 1e-3);
    double best = 0.0;
    for (int r = 0; r < launches; r++) {
        cudaEventRecord(e0, st);
        dmma_peak_kernel<<<nsm, 512, 0, st>>>(scratch, iters, 1.0, 1e-3);
        cudaEventRecord(e1, st);
        CCSD_CUDA_TRY(cudaEventSynchronize(e1));
        float ms = 0.f;
        cudaEventElapsedTime(&ms, e0, e1);
        double tf = 16.0 * 8 * (double)iters * 512.0 * nsm / (ms * 1e-3) * 1e-12;
        if (tf > best) best = tf;
        count_launches(1);
    }
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    *tflops = best;
    return CCSD_OK;
}
