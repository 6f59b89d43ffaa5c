// dsmem_alltoall.cu -- probe (not part of libshg): how fast can the CTAs of a 16-CTA cluster exchange the blocks of a
// 2-D transposition through distributed shared memory on sm_100a?  Every CTA sends BLK bytes to each of the 16 CTAs
// (all-to-all, 16 * BLK bytes out and in per CTA), the pattern of shg_cluster.cuh's column exchange.
//   method 0: 16 bulk copies (cp.async.bulk.shared::cluster, mbarrier complete_tx), issued by 16 lanes of warp 0
//   method 1: the same 16 bulk copies, issued by lane 0 of 16 different warps
//   method 2: st.shared::cluster.v4 (16 B per lane, 512 B contiguous per warp instruction) by all 512 threads,
//             completion by a cluster barrier (arrive.release / wait.acquire)
//   method 3: st.shared::cluster.v2 (8 B per lane, 64 B contiguous segments), 128 threads, cluster barrier
// Prints SM clocks per exchange (issue of the first store / copy .. data of all senders visible), mean over CTAs.
//   nvcc -gencode arch=compute_100a,code=sm_100a -O3 -o dsmem_alltoall dsmem_alltoall.cu && ./dsmem_alltoall
#include <cstdio>
#include <cuda_runtime.h>

constexpr int C = 16, THREADS = 512;

__device__ __forceinline__ unsigned mapa(unsigned a, unsigned r) {
    unsigned o;
    asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(o) : "r"(a), "r"(r));
    return o;
}
__device__ __forceinline__ void csync() {
    asm volatile("barrier.cluster.arrive.release.aligned;" ::: "memory");
    asm volatile("barrier.cluster.wait.acquire.aligned;" ::: "memory");
}

template <int METHOD>
__global__ void __launch_bounds__(THREADS, 1) k_probe(int blk_bytes, int iters, long long* out) {
    extern __shared__ __align__(128) unsigned char smem[];
    unsigned char* src = smem;                      // [C][blk_bytes]
    unsigned char* dst = smem + C * blk_bytes;      // [C][blk_bytes]
    __shared__ __align__(8) unsigned long long bar;
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    unsigned rank;
    asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(rank));
    const unsigned bar_s = (unsigned)__cvta_generic_to_shared(&bar);
    const unsigned src_s = (unsigned)__cvta_generic_to_shared(src), dst_s = (unsigned)__cvta_generic_to_shared(dst);
    for (int i = tid; i < C * blk_bytes / 4; i += THREADS) reinterpret_cast<float*>(src)[i] = (float)(rank * 1000 + i);
    if (tid == 0) {
        asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"(bar_s));
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    csync();
    long long total = 0;
    unsigned parity = 0;
    for (int it = 0; it < iters; ++it) {
        if (METHOD <= 1 && tid == 0)
            asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar_s), "r"(C * blk_bytes) : "memory");
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
        csync();                                    // everyone armed and ready: start of the timed exchange
        const long long t0 = clock64();
        if (METHOD == 0) {
            if (warp == 0 && lane < C)
                asm volatile("cp.async.bulk.shared::cluster.shared::cta.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                             ::"r"(mapa(dst_s + rank * blk_bytes, lane)), "r"(src_s + lane * blk_bytes), "r"(blk_bytes),
                               "r"(mapa(bar_s, lane)) : "memory");
        } else if (METHOD == 1) {
            if (lane == 0 && warp < C)
                asm volatile("cp.async.bulk.shared::cluster.shared::cta.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                             ::"r"(mapa(dst_s + rank * blk_bytes, warp)), "r"(src_s + warp * blk_bytes), "r"(blk_bytes),
                               "r"(mapa(bar_s, warp)) : "memory");
        } else if (METHOD == 2) {
            for (int o = tid * 16; o < C * blk_bytes; o += THREADS * 16) {
                const int d = o / blk_bytes, w = o % blk_bytes;
                const float4 v = *reinterpret_cast<const float4*>(src + o);
                asm volatile("st.shared::cluster.v4.f32 [%0], {%1, %2, %3, %4};"
                             ::"r"(mapa(dst_s + rank * blk_bytes + w, d)), "f"(v.x), "f"(v.y), "f"(v.z), "f"(v.w) : "memory");
            }
        } else {
            if (tid < 128) {
                // 8 lanes x 8 B = 64 B contiguous per destination; a warp instruction touches 4 destinations
                for (int o = tid * 8; o < C * blk_bytes; o += 128 * 8) {
                    const int d = o / blk_bytes, w = o % blk_bytes;
                    const float2 v = *reinterpret_cast<const float2*>(src + o);
                    asm volatile("st.shared::cluster.v2.f32 [%0], {%1, %2};"
                                 ::"r"(mapa(dst_s + rank * blk_bytes + w, d)), "f"(v.x), "f"(v.y) : "memory");
                }
            }
        }
        if (METHOD <= 1) {
            unsigned done;
            do {
                asm volatile("{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
                             "selp.u32 %0, 1, 0, p;\n\t}" : "=r"(done) : "r"(bar_s), "r"(parity) : "memory");
            } while (!done);
            parity ^= 1u;
        } else {
            csync();
        }
        const long long t1 = clock64();
        if (it >= 4) total += t1 - t0;
        __syncthreads();
    }
    csync();
    if (tid == 0) out[blockIdx.x] = total / (iters - 4);
    // check: block s of dst holds what CTA s sent to this rank
    if (tid == 0 && reinterpret_cast<float*>(dst)[3 * blk_bytes / 4 + 5] != (float)(3 * 1000 + rank * blk_bytes / 4 + 5))
        out[blockIdx.x] = -1;
}

template <int METHOD>
static void run(int blk_bytes) {
    long long* d;
    cudaMalloc(&d, sizeof(long long) * C);
    auto kern = k_probe<METHOD>;
    const int smem = 2 * C * blk_bytes;
    cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, smem > 120 * 1024 ? smem : 120 * 1024);
    cudaFuncSetAttribute(kern, cudaFuncAttributeNonPortableClusterSizeAllowed, 1);
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(C);
    cfg.blockDim = dim3(THREADS);
    cfg.dynamicSmemBytes = smem > 120 * 1024 ? smem : 120 * 1024;
    cudaLaunchAttribute a[1];
    a[0].id = cudaLaunchAttributeClusterDimension;
    a[0].val.clusterDim.x = C; a[0].val.clusterDim.y = 1; a[0].val.clusterDim.z = 1;
    cfg.attrs = a; cfg.numAttrs = 1;
    cudaError_t e = cudaLaunchKernelEx(&cfg, kern, blk_bytes, 104, d);
    if (e == cudaSuccess) e = cudaDeviceSynchronize();
    long long h[C];
    cudaMemcpy(h, d, sizeof(h), cudaMemcpyDeviceToHost);
    double mean = 0; long long mx = 0; bool bad = false;
    for (int i = 0; i < C; ++i) { mean += (double)h[i] / C; if (h[i] > mx) mx = h[i]; if (h[i] < 0) bad = true; }
    printf("method %d  block %5d B (%6d B per CTA)  clocks per exchange: mean %7.0f max %7lld  = %5.1f B/clk per CTA  %s %s\n",
           METHOD, blk_bytes, C * blk_bytes, mean, mx, C * blk_bytes / mean, cudaGetErrorString(e), bad ? "DATA MISMATCH" : "");
    cudaFree(d);
}

int main() {
    for (int blk : {256, 1024, 4096}) {
        run<0>(blk); run<1>(blk); run<2>(blk); run<3>(blk);
    }
    return 0;
}
