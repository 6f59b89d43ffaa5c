// fft_issue_rate.cu -- probe (not part of libshg): at what rate does an SM run the line transform of libshg when
// nothing else is in the way (no global memory, no barriers), and which warps share a scheduler?
//
//   part 1: W warps per CTA (one CTA per SM) run warp_fft<N> / fft_reg<32> / table_mul_s back to back on register
//           data; prints SM clocks per call and per line-holding warp of a scheduler.  Two warps per scheduler
//           already reach the throughput of four (the transforms are bound by the scheduler's fp32 pipe and
//           register-file bandwidth, not by latency), and 14 warps (4, 4, 3, 3 per scheduler: a 1024 x 1024
//           simulation's seven rows per SM) take exactly as long as 16.
//   part 2: fft_reg<32> on chosen subsets of the 16 warps: warps w and w + 4 share a scheduler (w % 4), warps
//           w .. w + 3 do not.
// Figures quoted in profiles/r02b_summary.md and DESIGN.md 12 come from this program.
//   nvcc -gencode arch=compute_100a,code=sm_100a -O3 -std=c++17 --expt-relaxed-constexpr -o fft_issue_rate fft_issue_rate.cu
#include <cstdio>
#include <cuda_runtime.h>
#include "../../paper_2410_04994_b200/csrc/shg_device.cuh"
using namespace shg;

template <int N, int MODE>
__global__ void __launch_bounds__(512, 1) k_rate(int iters, unsigned mask, const float4* tw, long long* out, float2* sink) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    using GE = Geo<N>;
    constexpr int R = GE::R, M = GE::M, G = GE::G, NP = GE::NP;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const float4* tws = load_twiddles<N>(smem_raw, tw);
    float4* stab = reinterpret_cast<float4*>(smem_raw + GE::CTA_SMEM);
    for (int i = threadIdx.x; i < 4 * N; i += blockDim.x) stab[i] = tw[i % N];
    __syncthreads();
    const int g = lane / M, m = lane % M;
    float2* own = reinterpret_cast<float2*>(smem_raw) + (size_t)warp * (G * NP) + g * NP;
    float2 v[R];
#pragma unroll
    for (int q = 0; q < R; ++q) v[q] = make_float2(1e-3f * (lane + q), 1e-3f * (warp - q));
    __syncthreads();
    const long long t0 = clock64();
    if ((mask >> warp) & 1) {
        for (int it = 0; it < iters; ++it) {
            if (MODE == 0) warp_fft<N, true>(v, own, tws, m);
            else if (MODE == 1) fft_reg<R, false, true>(v);
            else table_mul_s<R, M, true, false>(v, (unsigned)__cvta_generic_to_shared(stab + m), std::make_integer_sequence<int, R>{});
#pragma unroll
            for (int q = 0; q < R; ++q) { v[q].x *= 1e-3f; v[q].y *= 1e-3f; }      // (keeps the values finite)
        }
    }
    const long long t1 = clock64();
    if (lane == 0) out[blockIdx.x * 16 + warp] = t1 - t0;
    float2 s = make_float2(0.f, 0.f);
#pragma unroll
    for (int q = 0; q < R; ++q) { s.x += v[q].x; s.y += v[q].y; }
    sink[blockIdx.x * blockDim.x + threadIdx.x] = s;
}

static int g_fail = 0;

template <int N, int MODE>
void run(const char* name, unsigned mask, int sms, const float4* tw, long long* out, float2* sink, double* per_warp) {
    using GE = Geo<N>;
    const int smem = GE::CTA_SMEM_TAB, iters = 100;
    cudaFuncSetAttribute(k_rate<N, MODE>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
    for (int rep = 0; rep < 2; ++rep) {
        k_rate<N, MODE><<<sms, 512, smem>>>(iters, mask, tw, out, sink);
        if (cudaDeviceSynchronize() != cudaSuccess) { printf("%s: CUDA error\n", name); g_fail = 1; return; }
    }
    static long long h[256 * 16];
    cudaMemcpy(h, out, sizeof(long long) * sms * 16, cudaMemcpyDeviceToHost);
    for (int w = 0; w < 16; ++w) {
        double mean = 0;
        for (int c = 0; c < sms; ++c) mean += (double)h[c * 16 + w];
        per_warp[w] = mean / sms / iters;
    }
}

int main() {
    int sms = 0;
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, 0);
    if (sms <= 0 || sms > 256) { printf("no device\n"); return 1; }
    float4* tw; long long* out; float2* sink;
    cudaMalloc(&tw, 4096 * 16); cudaMalloc(&out, sizeof(long long) * sms * 16); cudaMalloc(&sink, sizeof(float2) * sms * 512);
    static float4 h[4096];
    for (int i = 0; i < 4096; ++i) h[i] = make_float4(0.9f, 0.1f, 1e-9f, 1e-9f);
    cudaMemcpy(tw, h, sizeof(h), cudaMemcpyHostToDevice);
    double pw[16];
    printf("part 1: SM clocks per call, W warps per CTA (clocks of warp 0; 'per warp of a scheduler' = clocks / (W / 4))\n");
    const int Ws[5] = {4, 8, 12, 14, 16};
    double t16 = 0, t14 = 0, t8 = 0;
    for (int wi = 0; wi < 5; ++wi) {
        const unsigned mask = (1u << Ws[wi]) - 1u;
        run<1024, 0>("warp_fft<1024>", mask, sms, tw, out, sink, pw);
        printf("rate warp_fft<1024>   W=%2d: %6.0f  (%6.0f per warp of a scheduler)\n", Ws[wi], pw[0], pw[0] / (Ws[wi] / 4.0));
        if (Ws[wi] == 16) t16 = pw[0];
        if (Ws[wi] == 14) t14 = pw[0];
        if (Ws[wi] == 8) t8 = pw[0];
    }
    for (int wi = 0; wi < 5; ++wi) {
        const unsigned mask = (1u << Ws[wi]) - 1u;
        run<1024, 1>("fft_reg<32>", mask, sms, tw, out, sink, pw);
        printf("rate fft_reg<32>      W=%2d: %6.0f  (%6.0f per warp of a scheduler)\n", Ws[wi], pw[0], pw[0] / (Ws[wi] / 4.0));
    }
    for (int wi = 0; wi < 5; ++wi) {
        const unsigned mask = (1u << Ws[wi]) - 1u;
        run<1024, 2>("table_mul_s<32>", mask, sms, tw, out, sink, pw);
        printf("rate table_mul_s<32>  W=%2d: %6.0f  (%6.0f per warp of a scheduler)\n", Ws[wi], pw[0], pw[0] / (Ws[wi] / 4.0));
    }
    run<256, 0>("warp_fft<256>", 0xFFFFu, sms, tw, out, sink, pw);
    printf("rate warp_fft<256>    W=16: %6.0f  (two lines per warp)\n", pw[0]);
    run<128, 0>("warp_fft<128>", 0xFFFFu, sms, tw, out, sink, pw);
    printf("rate warp_fft<128>    W=16: %6.0f  (four lines per warp)\n", pw[0]);
    printf("check: 14 warps take as long as 16 (%.3f), 16 warps twice as long as 8 (%.3f)\n", t14 / t16, t16 / t8);
    if (t14 / t16 < 0.97 || t14 / t16 > 1.03 || t16 / t8 < 1.8 || t16 / t8 > 2.2) g_fail = 1;

    printf("part 2: fft_reg<32> on subsets of the warps (mask: bit w = warp w runs), clocks per call of each running warp\n");
    const unsigned masks[] = {0x1, 0x3, 0x5, 0x9, 0xF, 0x11, 0x101, 0x1111, 0x3333, 0x3FFF, 0xFFFF};
    double solo = 0, same = 0, other = 0;
    for (unsigned mk : masks) {
        run<1024, 1>("fft_reg<32>", mk, sms, tw, out, sink, pw);
        printf("map mask %04x:", mk);
        for (int w = 0; w < 16; ++w) if ((mk >> w) & 1) printf(" w%d=%.0f", w, pw[w]);
        printf("\n");
        if (mk == 0x1) solo = pw[0];
        if (mk == 0x11) same = pw[0];
        if (mk == 0xF) other = pw[0];
    }
    printf("check: warps 0 and 4 share a scheduler (%.2fx a lone warp), warps 0..3 do not (%.2fx)\n", same / solo, other / solo);
    if (same / solo < 1.7 || other / solo > 1.15) g_fail = 1;
    printf(g_fail ? "PROBE FAILED\n" : "probe ok\n");
    return g_fail;
}
