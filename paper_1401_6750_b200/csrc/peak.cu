// peak.cu -- measured fp32 FMA peak of the device (the ALU roofline denominator of the contraction kernel).
//
// "B200 ALU peaks ... are not verified here -- measure with an FMA microbenchmark ... before quoting
// an ALU roofline".  The contraction kernel (contract_tma.cu) is bound by the fp32 FMA pipe, not by HBM, so bench.py
// divides its achieved FLOP/s by the number this kernel measures in the same run, on the same box, under the same
// clocks: every thread runs `iters` rounds of 16 independent dependent-chain FMAs (mode 0: scalar FFMA, mode 1: packed
// FFMA2 on (re, im) register pairs -- the instruction the contraction and the fp32 Dslash use), 2 flop per FMA lane.
#include "kernels.h"
#include "contract.cuh"

template <int MODE>
__global__ void __launch_bounds__(256) fma_peak_kernel(float* __restrict__ out, int iters, float a, float b) {
    float acc[16];
#pragma unroll
    for (int i = 0; i < 16; i++) acc[i] = (float)(threadIdx.x + i) * 1e-3f;
    if (MODE == 0) {
        for (int it = 0; it < iters; it++) {
#pragma unroll
            for (int i = 0; i < 16; i++) acc[i] = fmaf(acc[i], a, b);
        }
    } else {
        typedef P2<float>::T T2;
        T2 p[8];
#pragma unroll
        for (int i = 0; i < 8; i++) p[i] = P2<float>::make(acc[2 * i], acc[2 * i + 1]);
        const T2 bb = P2<float>::make(b, b);
        for (int it = 0; it < iters; it++) {
#pragma unroll
            for (int i = 0; i < 8; i++) p[i] = P2<float>::fma_s(a, p[i], bb);
        }
#pragma unroll
        for (int i = 0; i < 8; i++) P2<float>::get(p[i], acc[2 * i], acc[2 * i + 1]);
    }
    float s = 0.f;
#pragma unroll
    for (int i = 0; i < 16; i++) s += acc[i];
    if (s == 123.456f) out[blockIdx.x * blockDim.x + threadIdx.x] = s;      // never true: keeps the chains alive
}

extern "C" tm_status tm_fma_peak(tm_ctx* ctx, int mode, int iters, double* tflops, void* stream) {
    if (!ctx || !tflops || iters < 1 || (mode != 0 && mode != 1)) return tm_fail(ctx, TM_EARG, "tm_fma_peak: bad argument");
    cudaStream_t st = (cudaStream_t)stream;
    TM_CUDA(ctx, cudaSetDevice(ctx->device));
    float* sink;
    const unsigned grid = (unsigned)ctx->sm_count * 8;
    TM_TRY(tm_ws(ctx, WS_API_C, (size_t)grid * 256 * sizeof(float), (void**)&sink));
    cudaEvent_t e0 = ctx->ev[2], e1 = ctx->ev[3];
    float best = 0.f;
    for (int rep = 0; rep < 4; rep++) {          // first repetition warms up; best of the rest
        TM_CUDA(ctx, cudaEventRecord(e0, st));
        if (mode == 0) fma_peak_kernel<0><<<grid, 256, 0, st>>>(sink, iters, 1.0000001f, 1e-9f);
        else           fma_peak_kernel<1><<<grid, 256, 0, st>>>(sink, iters, 1.0000001f, 1e-9f);
        TM_LAUNCH_CHECK(ctx, "fma_peak_kernel");
        TM_CUDA(ctx, cudaEventRecord(e1, st));
        TM_CUDA(ctx, cudaEventSynchronize(e1));
        float ms = 0.f;
        cudaEventElapsedTime(&ms, e0, e1);
        if (rep > 0 && (best == 0.f || ms < best)) best = ms;
    }
    *tflops = 2.0 * 16.0 * (double)iters * (double)grid * 256.0 / ((double)best * 1e-3) / 1e12;
    return TM_OK;
}
