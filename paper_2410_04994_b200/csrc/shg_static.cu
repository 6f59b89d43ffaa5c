// shg_static.cu -- shg_field_power_static: the library's one entry point that never allocates.
//
// Who needs it.  Some code that wants a power integral is not allowed to call cudaMalloc: a callback that runs inside
// somebody else's allocator or memory pool (allocating there re-enters the pool or dead-locks on its lock), a plug-in
// whose host owns every byte of device memory and hands out fixed buffers, a real-time loop that must not take the
// driver's allocation lock or the implicit device synchronisation of cudaFree, a process that runs close to the
// memory limit on purpose.  shg_create allocates (tables, history, scratch), so those callers cannot even own a
// context.  This file gives them the power integral of include/shg.h (P_j = scale_j sum |A_j|^2) with no
// context and no allocation: the scratch that the two-level sum needs lives in a fixed array in the library's
// device image.
//
// The sum itself is the one k_input_power (shg_api.cu) does for node 0 of every propagate: per member, up to 64 blocks
// each add their chunk in double in a fixed order, write the chunk sum to scratch, and the block that takes the last
// ticket adds the chunk sums in chunk order.  The result does not depend on the order in which blocks finish.
#include "../../include/shg.h"

#include <cstdint>
#include <mutex>

#include "shg_launch.h"

namespace {

constexpr int MAXB = SHG_STATIC_MAX_BATCH;   // members per call
constexpr int MAXCH = 64;                     // chunk sums per member
constexpr size_t PART_WORDS = (size_t)MAXB * MAXCH * 2;       // double [MAXB][MAXCH][2]
constexpr size_t TICKET_WORDS = (size_t)MAXB / 2;             // unsigned int [MAXB], kept in the tail of the array
constexpr int MAX_DEVICES = 64;

// The scratch: 256 KiB of chunk sums + 1 KiB of tickets.  It is part of the library's device image, so every GPU on
// which libshg runs a kernel holds its own copy from module load until the process exits.
// On the HOST side the name `g_static_scratch` is only a handle for cudaGetSymbolAddress -- it is NOT a device
// address; a kernel given `g_static_scratch` from host code would fault (or, where the GPU can reach host memory,
// quietly use the wrong bytes).  Host code below therefore only ever uses the pointer that cudaGetSymbolAddress
// returned for the current device.
static __device__ __align__(256) double g_static_scratch[PART_WORDS + TICKET_WORDS];

static_assert(sizeof(double) * (PART_WORDS + TICKET_WORDS) == 263168, "scratch size stated in include/shg.h");
static_assert(MAXB % 2 == 0, "tickets are packed two per double word");

std::mutex g_setup_lock;
double* g_scratch_of_device[MAX_DEVICES] = {};   // device address of g_static_scratch, per CUDA device ordinal

// Same arithmetic as k_input_power; the result goes to the caller's array instead of the fixed-point history.
__global__ void __launch_bounds__(256) k_field_power_static(const float2* __restrict__ A1,
                                                            const float2* __restrict__ A2, size_t np, size_t len,
                                                            double scale1, double scale2, double* part,
                                                            unsigned int* ticket, double* __restrict__ P) {
    const int b = blockIdx.y, c = blockIdx.x, CH = gridDim.x;
    const size_t lo = (size_t)c * len, hi = lo + len < np ? lo + len : np;
    const size_t base = (size_t)b * np;
    double s1 = 0.0, s2 = 0.0;
    for (size_t i = lo + threadIdx.x; i < hi; i += blockDim.x) {
        const float2 a = A1[base + i];
        s1 += (double)a.x * a.x + (double)a.y * a.y;
        if (A2) {
            const float2 d = A2[base + i];
            s2 += (double)d.x * d.x + (double)d.y * d.y;
        }
    }
    __shared__ double sh[2][8];
#pragma unroll
    for (int o = 16; o >= 1; o >>= 1) {
        s1 += __shfl_xor_sync(0xffffffffu, s1, o);
        s2 += __shfl_xor_sync(0xffffffffu, s2, o);
    }
    if ((threadIdx.x & 31) == 0) { sh[0][threadIdx.x >> 5] = s1; sh[1][threadIdx.x >> 5] = s2; }
    __syncthreads();
    if (threadIdx.x == 0) {
        double t1 = 0.0, t2 = 0.0;
        for (int w = 0; w < 8; ++w) { t1 += sh[0][w]; t2 += sh[1][w]; }
        part[((size_t)b * MAXCH + c) * 2 + 0] = t1;
        part[((size_t)b * MAXCH + c) * 2 + 1] = t2;
        __threadfence();
        if (atomicAdd(&ticket[b], 1u) == (unsigned)(CH - 1)) {   // last chunk of this member to finish
            __threadfence();
            double S1 = 0.0, S2 = 0.0;
            for (int k = 0; k < CH; ++k) {
                S1 += __ldcg(&part[((size_t)b * MAXCH + k) * 2 + 0]);
                S2 += __ldcg(&part[((size_t)b * MAXCH + k) * 2 + 1]);
            }
            P[2 * b + 0] = scale1 * S1;
            P[2 * b + 1] = scale2 * S2;
        }
    }
}

// Device address of the scratch on the CURRENT device, looked up once per device.
int scratch_for_current_device(double** out) {
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return shg::record_cuda_error(e, "cudaGetDevice");
    if (dev < 0 || dev >= MAX_DEVICES) return SHG_EINVAL;
    std::lock_guard<std::mutex> hold(g_setup_lock);
    if (!g_scratch_of_device[dev]) {
        double* p = nullptr;
        e = cudaGetSymbolAddress((void**)&p, g_static_scratch);
        if (e != cudaSuccess) return shg::record_cuda_error(e, "cudaGetSymbolAddress(g_static_scratch)");
        if (!p) return shg::record_cuda_error(cudaErrorInvalidSymbol, "cudaGetSymbolAddress returned NULL");
        g_scratch_of_device[dev] = p;
    }
    *out = g_scratch_of_device[dev];
    return SHG_OK;
}

}  // namespace

extern "C" int shg_field_power_static(const void* A1_device, const void* A2_device, int nx, int ny, int batch,
                                      double scale1, double scale2, double* P_device, void* cuda_stream) {
    if (!A1_device || !P_device || nx < 1 || ny < 1 || batch < 1) return SHG_EINVAL;
    if (batch > MAXB) return SHG_ELIMIT;
    if ((reinterpret_cast<uintptr_t>(A1_device) | reinterpret_cast<uintptr_t>(A2_device) |
         reinterpret_cast<uintptr_t>(P_device)) & 7u)
        return SHG_EINVAL;
    double* scratch = nullptr;
    int rc = scratch_for_current_device(&scratch);
    if (rc != SHG_OK) return rc;
    double* part = scratch;
    unsigned int* ticket = reinterpret_cast<unsigned int*>(scratch + PART_WORDS);

    const size_t np = (size_t)nx * (size_t)ny;
    int ch = (int)(np / 4096);
    ch = ch < 1 ? 1 : (ch > MAXCH ? MAXCH : ch);
    const size_t len = (np + (size_t)ch - 1) / (size_t)ch;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    // The array still holds whatever the previous call (or a call that failed half-way) left in it.  The chunk sums
    // are all overwritten before they are read; the tickets must start at zero, so they are cleared here, on the
    // caller's stream, ahead of the kernel.
    cudaError_t e = cudaMemsetAsync(ticket, 0, sizeof(unsigned int) * (size_t)batch, st);
    if (e != cudaSuccess) return shg::record_cuda_error(e, "cudaMemsetAsync(static scratch tickets)");
    k_field_power_static<<<dim3(ch, batch), 256, 0, st>>>((const float2*)A1_device, (const float2*)A2_device, np, len,
                                                          scale1, scale2, part, ticket, P_device);
    e = cudaGetLastError();
    if (e != cudaSuccess) return shg::record_cuda_error(e, "k_field_power_static launch");
    return SHG_OK;
}
