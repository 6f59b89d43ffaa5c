// shg_diag.cu -- bench-side equipment, built into libshg_diag.so (NOT part of libshg): the measured fp32 pipe peak that
// bench.py uses as the denominator of its "alu" roofline.  Nothing of the method is in here.
#include "../../include/shg_diag.h"

#include <cuda_runtime.h>

namespace {

#define CU(call)                                          \
    do {                                                  \
        cudaError_t e__ = (call);                         \
        if (e__ != cudaSuccess) return SHG_DIAG_ECUDA;    \
    } while (0)

// fp32 pipe peak: 16 independent FFMA chains per thread, nothing else in the loop
__global__ void __launch_bounds__(512, 1) k_fp32_peak(float* out, const float* in, int iters) {
    float a[16];
    const float b = in[threadIdx.x & 31], c = in[32 + (threadIdx.x & 31)];
#pragma unroll
    for (int i = 0; i < 16; ++i) a[i] = in[i] + (float)threadIdx.x;
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int i = 0; i < 16; ++i) a[i] = fmaf(a[i], b, c);
    }
    float s = 0.f;
#pragma unroll
    for (int i = 0; i < 16; ++i) s += a[i];
    out[blockIdx.x * blockDim.x + threadIdx.x] = s;
}

// the same with three DISTINCT register operands per FFMA (no operand reuse between neighbouring instructions): what
// a transform butterfly or an RK4 stage looks like to the register file
__global__ void __launch_bounds__(512, 1) k_fp32_peak_distinct(float* out, const float* in, int iters) {
    float a[16], b[16], c[16];
#pragma unroll
    for (int i = 0; i < 16; ++i) {
        a[i] = in[i] + (float)threadIdx.x;
        b[i] = in[16 + i] + 1.0f;
        c[i] = in[32 + i];
    }
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int i = 0; i < 16; ++i) a[i] = fmaf(a[i], b[i], c[i]);
    }
    float s = 0.f;
#pragma unroll
    for (int i = 0; i < 16; ++i) s += a[i];
    out[blockIdx.x * blockDim.x + threadIdx.x] = s;
}

}  // namespace

static int measure_fp32(double* tflops, bool distinct);

extern "C" int shg_measure_fp32_peak(double* tflops) { return measure_fp32(tflops, false); }
extern "C" int shg_measure_fp32_peak_distinct(double* tflops) { return measure_fp32(tflops, true); }

static int measure_fp32(double* tflops, bool distinct) {
    if (!tflops) return SHG_DIAG_EINVAL;
    int dev = 0, sms = 0;
    CU(cudaGetDevice(&dev));
    CU(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
    float *out = nullptr, *in = nullptr;
    CU(cudaMalloc((void**)&out, sizeof(float) * (size_t)sms * 512));
    CU(cudaMalloc((void**)&in, 4096));
    CU(cudaMemset(in, 0, 4096));
    cudaEvent_t e0, e1;
    CU(cudaEventCreate(&e0));
    CU(cudaEventCreate(&e1));
    const int iters = 20000;
    float best = 0.f;
    for (int rep = 0; rep < 4; ++rep) {        // first repetition warms up
        CU(cudaEventRecord(e0, nullptr));
        if (distinct) k_fp32_peak_distinct<<<sms, 512>>>(out, in, iters);
        else k_fp32_peak<<<sms, 512>>>(out, in, iters);
        CU(cudaEventRecord(e1, nullptr));
        CU(cudaEventSynchronize(e1));
        float ms = 0.f;
        CU(cudaEventElapsedTime(&ms, e0, e1));
        if (rep > 0 && (best == 0.f || ms < best)) best = ms;
    }
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    cudaFree(out);
    cudaFree(in);
    *tflops = 2.0 * 16.0 * (double)iters * 512.0 * (double)sms / ((double)best * 1e-3) / 1e12;
    return SHG_DIAG_OK;
}

