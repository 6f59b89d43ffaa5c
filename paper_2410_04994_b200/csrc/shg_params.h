// shg_params.h -- plain structs passed from the host side of libshg to its kernels.
#pragma once

#include <cuda_runtime.h>
#include <stdint.h>

namespace shg {

// Per-member constants (device copy).  "P:n" = PAPER.md line n.
struct MemberDev {
    float kap1dz, kap2dz;      // kappa_j * dz                                   (P:72-73 with G2)
    float g1dz, g2dz;          // (beta_j / 2) (eps0 c n_j / 2) dz                (G5)
    float dz;
    float gT;                  // ddk_dT
    float Tpm_hi, Tpm_lo;      // T_pm = hi + lo
    float dk0;
    double dk_uniform;         // dk0 + ddk_dT (T_uniform - T_pm), used when nzt == 0
    double dzd;
    float qa1, qb1, qa2, qb2;  // heat source of Eq. 8 per |A_j|^2: q = s1 (qa1 + qb1 s1) + s2 (qa2 + qb2 s2), s_j = |A_j|^2
};

struct Params {
    int nx, ny, nz, nzt, batch;
    int n_begin, n_end;        // z-steps [n_begin, n_end) of this launch of a persistent kernel (normally 0, nz; a host
                               // temperature array that is still being uploaded is consumed range by range, shg_api.cu)
    int ny_log2;               // ny = 1 << ny_log2 (every supported line length is a power of two)
    int flat_rows;             // 1: sparse launch, the persistent kernel spreads the nonlinear step over the CTA (row_pass_flat)
    int scheme;                // 0: L/2 - N - L/2 with merged half-steps; 1: the paper's N/2 - L - N/2 (SHG_OPT_SCHEME)
    int acquire_fence;         // acquire side of the device-wide barrier (SHG_OPT_ACQUIRE_FENCE): 0 none (L2-only loads),
                               // 1 gpu-scope fence after the poll, 2 the successful poll is an ld.acquire.gpu
    int pipeline;              // 1: batched run in the software-pipelined persistent kernel (k_persist_pipe)
    int tab_smem;              // 1: the propagator tables hx / hy of member 0 are staged in shared memory (batch == 1)
    int rec_every, nrec;       // power history: nodes n with n % rec_every == 0, and node nz (slot nrec), are recorded
    unsigned long long spin_limit;   // device-wide barrier: SM clocks before a timeout is declared (0 = wait forever)
    int row_slots, col_teams;  // slots (warps / warp pairs) and teams per CTA that take items (<= Geo limits)
    float2* A[2];              // working / output fields [batch][ny][nx]
    const float2* Ain[2];      // inputs (Ain[1] may be null)
    const float* T;            // [members][nzt][ny][nx] or null
    int T_per_member;
    float* phi;                // [batch][ny][nx]
    const float4* twx;         // [nx]  exp(-2 pi i e/nx) as (hi.re, hi.im, lo.re, lo.im)
    const float4* twy;         // [ny]
    const float4* hx[2];       // [0]=full step dz, [1]=half step: [batch][2][nx]
    const float4* hy[2];       // [batch][2][ny], includes 1/(nx ny)
    const MemberDev* mem;      // [batch]
    const float4* ucoef;       // nzt == 0: [nz][3] coupling coefficients of every z-step, shared by all members (shg_device.cuh), else null
    long long* hfix;           // [batch][nrec+1][2] power sums in fixed point: sum over points of rint(|A_j|^2 * pfix[b])
    const float* pfix;         // [batch] the member's fixed-point scale 2^e (k_input_power), see shg_device.cuh "power sums"
    float* Q;                  // optional heat-source output [batch][nq][ny][nx] (shg_set_heat_output), else null
    const int* qmap;           // [nz]: plane of Q that samples z-step n, or -1
    int nq;
    unsigned int* barrier;     // grid barrier counter (persistent kernel); [2..5]: the four counters of k_persist_pipe
    int* status;               // device status word (barrier timeout)
    long long* trace;          // optional phase timeline of the persistent kernel (SHG_OPT_TRACE), else null:
    int trace_steps;           //   [trace_steps][grid][2 barriers][4] = {clock64 CTA done, clock64 grid done, globaltimer, smid}
    int trace_grid;            //   CTAs that record (cluster kernel: [trace_steps][trace_grid][8] phase stamps, shg_cluster.cuh)
};

enum RowMode { ROW_FIRST = 0, ROW_MID = 1, ROW_FINAL = 2 };

// A0/(1+i tau0) and 1/(w0^2 (1+i tau0)) of one member, for the Gaussian pump of Eq. 5-6.
struct GaussDev { float ar, ai, qr, qi, dx, dy; };

}  // namespace shg
