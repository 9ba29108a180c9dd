// qp_peaks.cu -- measured arithmetic peaks of the device the library runs on (include/qp.h qp_measure_peaks).
//
// SURVEY.md 8(d) asks for the roofline denominators to be MEASURED ("measure it with a MUFU.EX2 micro-benchmark at
// the sustained clock, as was done for HBM"; "report the FP32-pipe bound beside it"). The pair kernels issue packed
// fp32 (FFMA2) for two thirds of their arithmetic and one MUFU per cell, and they are bound by issue slots rather
// than by either pipe, so three rates matter: scalar FFMA (= the warp-instruction issue rate
// when nothing else limits it), FFMA2 in scalar-equivalent FMAs, and MUFU. Each kernel runs 148 x 32 warps' worth of
// independent dependency chains long enough (a few ms) for the sustained clock to settle; rates are per second, so no
// clock has to be assumed.
#include <cuda_runtime.h>

#include "qp.h"

namespace qp {

constexpr int kPeakChains = 16;   // independent chains per thread: enough to cover the pipe latency at 8+ warps per scheduler

__global__ void k_peak_ffma(float* out, float a, float b, int iters) {
    float x[kPeakChains];
#pragma unroll
    for (int i = 0; i < kPeakChains; ++i) x[i] = threadIdx.x * 0.001f + i;
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int i = 0; i < kPeakChains; ++i) x[i] = fmaf(x[i], a, b);
    }
    float s = 0.f;
#pragma unroll
    for (int i = 0; i < kPeakChains; ++i) s += x[i];
    out[blockIdx.x * blockDim.x + threadIdx.x] = s;
}

__global__ void k_peak_ffma2(float* out, float a, float b, int iters) {
    unsigned long long x[kPeakChains / 2], aa, bb;
#pragma unroll
    for (int i = 0; i < kPeakChains / 2; ++i)
        asm("mov.b64 %0, {%1, %2};" : "=l"(x[i]) : "f"(threadIdx.x * 0.001f + i), "f"(i + 0.5f));
    asm("mov.b64 %0, {%1, %1};" : "=l"(aa) : "f"(a));
    asm("mov.b64 %0, {%1, %1};" : "=l"(bb) : "f"(b));
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int i = 0; i < kPeakChains / 2; ++i) asm volatile("fma.rn.f32x2 %0, %0, %1, %2;" : "+l"(x[i]) : "l"(aa), "l"(bb));
    }
    float s = 0.f;
#pragma unroll
    for (int i = 0; i < kPeakChains / 2; ++i) {
        float lo, hi;
        asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(x[i]));
        s += lo + hi;
    }
    out[blockIdx.x * blockDim.x + threadIdx.x] = s;
}

__global__ void k_peak_mufu(float* out, float a, int iters) {
    float x[kPeakChains];
#pragma unroll
    for (int i = 0; i < kPeakChains; ++i) x[i] = a + threadIdx.x * 0.001f + i;
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int i = 0; i < kPeakChains; ++i) asm volatile("sqrt.approx.ftz.f32 %0, %0;" : "+f"(x[i]));   // the pair kernels' MUFU
    }
    float s = 0.f;
#pragma unroll
    for (int i = 0; i < kPeakChains; ++i) s += x[i];
    out[blockIdx.x * blockDim.x + threadIdx.x] = s;
}

}  // namespace qp

using namespace qp;

extern "C" int qp_measure_peaks(qp_peaks* out, void* d_scratch, size_t scratch_bytes, void* cuda_stream) {
    if (!out || !d_scratch) return QP_ERR_INVALID_ARG;
    int dev, sms;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess)
        return QP_ERR_CUDA;
    const int threads = 1024;   // 32 warps per SM: 8 per scheduler
    if (scratch_bytes < (size_t)sms * threads * 4) return QP_ERR_WORKSPACE_TOO_SMALL;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    cudaEvent_t e0, e1;
    if (cudaEventCreate(&e0) != cudaSuccess || cudaEventCreate(&e1) != cudaSuccess) return QP_ERR_CUDA;
    float* o = (float*)d_scratch;
    const int iters = 40000;
    double rate[3] = {0, 0, 0};
    for (int which = 0; which < 3; ++which) {
        float best = 1e30f;
        for (int rep = 0; rep < 3; ++rep) {   // the first repetition warms the clocks up
            cudaEventRecord(e0, st);
            if (which == 0) k_peak_ffma<<<sms, threads, 0, st>>>(o, 0.999f, 0.001f, iters);
            else if (which == 1) k_peak_ffma2<<<sms, threads, 0, st>>>(o, 0.999f, 0.001f, iters);
            else k_peak_mufu<<<sms, threads, 0, st>>>(o, 1.5f, iters / 4);
            cudaEventRecord(e1, st);
            if (cudaEventSynchronize(e1) != cudaSuccess) return QP_ERR_CUDA;
            float ms;
            cudaEventElapsedTime(&ms, e0, e1);
            if (rep > 0 && ms < best) best = ms;
        }
        const double ops = (double)sms * threads * kPeakChains * (which == 2 ? iters / 4 : iters);
        rate[which] = ops / (best * 1e-3);
    }
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    out->sms = sms;
    out->ffma_per_s = rate[0];
    out->ffma2_fma_per_s = rate[1];
    out->mufu_per_s = rate[2];
    out->warp_instr_per_s = rate[0] / 32.0;
    return cudaGetLastError() == cudaSuccess ? QP_OK : QP_ERR_CUDA;
}
