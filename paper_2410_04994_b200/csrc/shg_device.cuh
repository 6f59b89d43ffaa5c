// shg_device.cuh -- device side of libshg: the warp-level 1-D FFT, the fused row pass
// (FFT_x -> temperature/phase -> RK4 -> power -> FFT_x -> propagator) and column pass
// (FFT_y -> propagator -> FFT_y), the per-pass kernels and the persistent whole-run kernel.
//
// One line of length N = R * M is held by M lanes (R values per lane, G = 32/M lines per warp).
// Decomposition  n = M n1 + n2 (lane n2 = m holds n1 = 0..R-1),  k = k1 + R k2:
//   X[k1 + R k2] = sum_{n2} W_M^{n2 k2} [ W_N^{n2 k1} sum_{n1} W_R^{n1 k1} x[M n1 + n2] ]
// stage A: radix-R in registers; twiddle W_N^{k1 m}; one transpose through shared memory (padded line,
// pitch M + 1: conflict free); stage B: R/M radix-M FFTs in registers.  Input and output are both "strided": lane m holds
// elements m + M q, q = 0..R-1 -- which is also the coalesced global layout.
//
// Only the FORWARD transform exists in the code (one instance keeps the z-loop inside the instruction
// cache).  Inverse transforms are taken as conj(F(conj(.))) with every conjugation folded into a neighbour:
//   column pass:  F_y -> * hy, conjugated (free) -> F_y -> store            [global holds conj(field)]
//   row pass:     load -> F_x -> conj (free, operand negation) -> RK4 -> F_x -> * hx -> store
// so between a column pass and the next row pass global memory holds the complex conjugate of the field in
// (k_x, y) representation.  DESIGN.md §5.
//
// The two fields of a row are transformed by different lane groups (or, at N = 1024, by the two warps of a
// pair) and meet for the nonlinear step through shared memory.  To make the two sides symmetric the SH row
// is handled rotated by N/2 in real space (its spectrum is then modulated by (-1)^k, which commutes with
// every linear operation of the step): the lane that holds FH elements e, e + N/2 in registers q, q + R/2
// has an SH partner lane that holds e + N/2, e in the same registers, so each side integrates "own lower
// half, partner's upper half".  DESIGN.md §5.3.
#pragma once

#include <cuda_runtime.h>
#include <stdint.h>

#include "fft_reg.cuh"
#include "shg_params.h"

namespace shg {

template <int N> struct FftCfg;
template <> struct FftCfg<64>   { static constexpr int R = 8,  M = 8;  };
template <> struct FftCfg<128>  { static constexpr int R = 16, M = 8;  };
template <> struct FftCfg<256>  { static constexpr int R = 16, M = 16; };
template <> struct FftCfg<512>  { static constexpr int R = 32, M = 16; };
template <> struct FftCfg<1024> { static constexpr int R = 32, M = 32; };

template <int N> struct Geo {
    static constexpr int R = FftCfg<N>::R, M = FftCfg<N>::M;
    static constexpr int G = 32 / M;                       // lines per warp
    static constexpr int Q = R / M;                        // radix-M transforms per lane in stage B
    static constexpr int MP = M + 1;                       // padded pitch of the in-line transpose
    static constexpr int LP = R * MP;                      // float2 slots one line needs (>= N)
    // line pitch in shared memory (float2): with M = 8 two lines share a 16-lane wavefront and must start
    // 16 banks apart (pitch = 8 mod 16)
    static constexpr int NP = (M == 8) ? ((LP + 7) / 16 * 16 + 8) : LP;
    static constexpr int WARP_SMEM = G * NP * 8;           // one warp's lines
    static constexpr int WARPS = 16;
    static constexpr int THREADS = WARPS * 32;
    // row pass: one item = HG rows x both fields (one warp), or one row handled by a warp pair (G == 1)
    static constexpr int HG = (G >= 2) ? G / 2 : 1;
    static constexpr int ROW_SLOTS = (G >= 2) ? WARPS : WARPS / 2;
    // column pass: a team of TW warps stages a strip of SC adjacent columns (64 B per row) in shared memory
    // The strip is stored column by column, one line of pitch CP per column; CP = 2 mod 16 makes the
    // staging stores (8 columns x 2 rows per 16-lane wavefront) conflict free.
    static constexpr int SC = 8;                           // strip columns
    static constexpr int CP = (LP + 13) / 16 * 16 + 2;     // column line pitch (float2), >= LP
    static constexpr int TW = SC / G;                      // warps per team
    static constexpr int TEAMS = WARPS / TW;
    static constexpr int STRIP_SMEM = SC * CP * 8;
    static constexpr int ROW_SMEM = WARPS * WARP_SMEM, COL_SMEM = TEAMS * STRIP_SMEM;
    static constexpr int WORK_SMEM = ROW_SMEM > COL_SMEM ? ROW_SMEM : COL_SMEM;
    static constexpr int TW_SMEM = N * 16;                 // twiddles [R][M] as float4 (hi.re, hi.im, lo.re, lo.im)
    static constexpr int CTA_SMEM = WORK_SMEM + TW_SMEM;
    // persistent kernel of a single simulation: the propagator tables hx, hy of both fields staged in shared memory
    static constexpr int TAB_SMEM = 4 * N * 16;            // [hx f=0][hx f=1][hy f=0][hy f=1], N float4 each
    static constexpr int CTA_SMEM_TAB = CTA_SMEM + TAB_SMEM;
    // pipelined kernel (k_persist_pipe): no CTA-wide barrier separates a row pass from a column pass, so a team's strip
    // must alias only the line regions of the team's own warps: one region per team, TEAM_SMEM bytes
    static constexpr int TEAM_SMEM = ((TW * WARP_SMEM > STRIP_SMEM ? TW * WARP_SMEM : STRIP_SMEM) + 15) / 16 * 16;
    static constexpr int PIPE_WORK_SMEM = TEAMS * TEAM_SMEM;
    static constexpr int PIPE_SMEM = PIPE_WORK_SMEM + TW_SMEM;
    static_assert(PIPE_SMEM <= 227 * 1024 && (TEAM_SMEM - TW * WARP_SMEM) % 8 == 0, "pipelined kernel: shared memory");
    // ... and, where it fits (N <= 256), one staging buffer per team ([N][SC] dense) that the NEXT strip is copied into
    // asynchronously while this one is transformed.  (The same for the lines of a row item was measured slower:
    // stream256 271 us per z-step against 255 with the strips alone -- it costs 64 KB of L1, through which the
    // batched kernels read their propagator tables, and the row items' 8-byte loads were not the problem.)
    static constexpr bool STAGE_COL = (N <= 256);
    static constexpr int COL_STAGE_SMEM = STAGE_COL ? TEAMS * N * SC * 8 : 0;
    static constexpr int PIPE_SMEM_STG = PIPE_SMEM + COL_STAGE_SMEM;
    static_assert(PIPE_SMEM_STG <= 227 * 1024, "pipelined kernel: staging buffers");
    static_assert(CTA_SMEM_TAB <= 227 * 1024, "shared memory budget");
    static_assert(WARPS % TW == 0 && WARPS % 2 == 0, "team / pair layout");
    static_assert(TEAMS + 1 <= 16 && WARPS / 2 + 1 <= 16, "named barrier ids");
};

__device__ __forceinline__ float2 ldcg2(const float2* p) { return __ldcg(p); }
__device__ __forceinline__ void stcg2(float2* p, float2 v) { __stcg(p, v); }

__device__ __forceinline__ void named_barrier(int id, int nthreads) {
    asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(nthreads) : "memory");
}

// 16-byte asynchronous copy global -> shared (LDGSTS, L2 only), completion with cp.async.wait_all
__device__ __forceinline__ void cp_async16(float2* dst_smem, const float2* src) {
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;"
                 ::"r"((unsigned)__cvta_generic_to_shared(dst_smem)), "l"(src) : "memory");
}
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_all;" ::: "memory"); }

// Table loads whose address carries a (numerically void) dependency on an earlier result.  Without it ptxas
// hoists all R twiddle / propagator loads (4 registers each) far above their use and spills the line data
// to make room; chaining load k to product k - TABLE_DEPTH keeps TABLE_DEPTH loads in flight.  One LOP3 each.
// Measured on cfg5 (us per z-step): depth 4: 40.2, 6: 39.0, 8: 39.1, 12: 36.6, 16: 36.7, 20: 38.7, 31 (no chain): 40.7
// (spills return); the propagator tables are the sensitive ones (twiddles 6..16 with tables at 12-14: 36.6-37.8).
// Re-measured at the end of round 2 (radix-2^2 butterflies, packed RK4; -DSHG_TWIDDLE_DEPTH=d), cfg5 / cfg4 / stream256 /
// stream1024: 4: 35.7 / 25.2 / 256 / 426, 8: 33.8 / 24.5 / 252 / 425, 10: 34.0 / 24.5 / 253 / 422, 12: 34.0 / 24.8 /
// 252 / 421, 16: 34.2 / 24.5 / 251, 20: 34.1 / 24.4 / 250 -- flat within 1 % from 8 on; 12 stays.
#ifndef SHG_TABLE_DEPTH
#define SHG_TABLE_DEPTH 12
#endif
#ifndef SHG_TWIDDLE_DEPTH
#define SHG_TWIDDLE_DEPTH 12
#endif
constexpr int TABLE_DEPTH = SHG_TABLE_DEPTH;      // global propagator tables (L1 latency)
constexpr int TWIDDLE_DEPTH = SHG_TWIDDLE_DEPTH;  // shared-memory twiddles (and shared-memory propagator tables)

template <int BYTE_OFF>
__device__ __forceinline__ float4 lds128_after(unsigned saddr, float dep) {
    unsigned a;
    asm("lop3.b32 %0, %1, %2, 0, 0xF8;" : "=r"(a) : "r"(saddr), "r"(__float_as_uint(dep)));   // a | (dep & 0)
    float4 w;
    asm("ld.shared.v4.f32 {%0, %1, %2, %3}, [%4+%5];"
        : "=f"(w.x), "=f"(w.y), "=f"(w.z), "=f"(w.w) : "r"(a), "n"(BYTE_OFF));
    return w;
}

__device__ __forceinline__ const float4* ptr_after(const float4* p, float dep) {
    unsigned lo, hi;
    asm("mov.b64 {%0, %1}, %2;" : "=r"(lo), "=r"(hi) : "l"(p));
    asm("lop3.b32 %0, %0, %1, 0, 0xF8;" : "+r"(lo) : "r"(__float_as_uint(dep)));
    const float4* r;
    asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "r"(lo), "r"(hi));
    return r;
}

// Pull one line group's table (N float4 = N/8 lines of 128 B) into L1: the device-wide barrier's fence
// invalidates L1 every pass, and the chained table loads below would otherwise each pay an L2 round trip.
template <int R, int M>
__device__ __forceinline__ void table_prefetch(const float4* __restrict__ tab, int m) {
    constexpr int LINES = R * M / 8, PER_LANE = (LINES + M - 1) / M;
#pragma unroll
    for (int i = 0; i < PER_LANE; ++i) {
        const int line = m + M * i;
        if (LINES % M == 0 || line < LINES)
            asm volatile("prefetch.global.L1 [%0];" ::"l"(tab + 8 * line));
    }
}

// v[q] *= table[M q] for q = 0..R-1 (table already offset by the lane), loads chained TABLE_DEPTH deep
template <int R, int M, bool PREC, bool CONJ_OUT>
__device__ __forceinline__ void table_mul(float2 (&v)[R], const float4* __restrict__ tab) {
#pragma unroll
    for (int q = 0; q < R; ++q) {
        const float dep = (q >= TABLE_DEPTH) ? v[q - TABLE_DEPTH].x : v[q].x;
        const float2 w = cmul_hl<false, PREC>(v[q], __ldg(ptr_after(tab, dep) + M * q));
        v[q] = CONJ_OUT ? make_float2(w.x, -w.y) : w;
    }
}

// same from a table in shared memory (stab_saddr: shared-window address of this lane's first entry)
template <int R, int M, bool PREC, bool CONJ_OUT, int Q>
__device__ __forceinline__ void table_mul_s_one(float2 (&v)[R], unsigned stab_saddr) {
    const float dep = (Q >= TWIDDLE_DEPTH) ? v[Q - TWIDDLE_DEPTH].x : v[Q].x;
    const float2 w = cmul_hl<false, PREC>(v[Q], lds128_after<Q * M * 16>(stab_saddr, dep));
    v[Q] = CONJ_OUT ? make_float2(w.x, -w.y) : w;
}
template <int R, int M, bool PREC, bool CONJ_OUT, int... Q>
__device__ __forceinline__ void table_mul_s(float2 (&v)[R], unsigned stab_saddr, std::integer_sequence<int, Q...>) {
    (table_mul_s_one<R, M, PREC, CONJ_OUT, Q>(v, stab_saddr), ...);
}

template <int N, bool PREC, int K1>
__device__ __forceinline__ void twiddle_one(float2 (&v)[FftCfg<N>::R], unsigned tws_saddr) {
    constexpr int M = FftCfg<N>::M;
    const float dep = (K1 > TWIDDLE_DEPTH) ? v[K1 - TWIDDLE_DEPTH].x : v[K1].x;
    v[K1] = cmul_hl<false, PREC>(v[K1], lds128_after<K1 * M * 16>(tws_saddr, dep));
}

template <int N, bool PREC, int... K>
__device__ __forceinline__ void twiddle_all(float2 (&v)[FftCfg<N>::R], unsigned tws_saddr,
                                            std::integer_sequence<int, K...>) {
    (twiddle_one<N, PREC, K + 1>(v, tws_saddr), ...);
}

// ------------------------------------------------------------------------------------------------
// Forward transform of one line per M-lane group; v in/out in strided layout (lane m holds m + M q).
// line: this group's line in shared memory (Geo<N>::LP slots; the transpose is padded, so every address is
// a per-lane base plus a compile-time offset and every access is conflict free).  tws: twiddles
// W_N^{k1 m} at [k1 * M + m] (lanes read consecutive entries).
// ------------------------------------------------------------------------------------------------
template <int N, bool PREC>
__device__ __forceinline__ void warp_fft(float2 (&v)[FftCfg<N>::R], float2* __restrict__ line,
                                         const float4* __restrict__ tws, int m) {
    constexpr int R = FftCfg<N>::R, M = FftCfg<N>::M, Q = R / M, MP = M + 1;
    const unsigned tws_saddr = (unsigned)__cvta_generic_to_shared(tws + m);
    float2* wr = line + m;            // transpose: value (k1, lane m) goes to slot k1 * MP + m ...
    float2* rd = line + m * MP;       // ... and lane m collects row k1 = m (+ M i): slots k1 * MP + n2
    if constexpr (Q == 1) {
        // both stages are the same radix: one copy of the butterfly code, executed twice
#pragma unroll 1
        for (int s = 0; s < 2; ++s) {
            fft_reg<R, false, PREC>(v);
            if (s == 0) {
                twiddle_all<N, PREC>(v, tws_saddr, std::make_integer_sequence<int, R - 1>{});
#pragma unroll
                for (int k1 = 0; k1 < R; ++k1) wr[k1 * MP] = v[k1];
                __syncwarp();
#pragma unroll
                for (int n2 = 0; n2 < M; ++n2) v[n2] = rd[n2];
                __syncwarp();
            }
        }
    } else {
        fft_reg<R, false, PREC>(v);
        twiddle_all<N, PREC>(v, tws_saddr, std::make_integer_sequence<int, R - 1>{});
#pragma unroll
        for (int k1 = 0; k1 < R; ++k1) wr[k1 * MP] = v[k1];
        __syncwarp();
#pragma unroll
        for (int i = 0; i < Q; ++i) {
            float2 u[M];
#pragma unroll
            for (int n2 = 0; n2 < M; ++n2) u[n2] = rd[i * M * MP + n2];
            fft_reg<M, false, PREC>(u);
#pragma unroll
            for (int k2 = 0; k2 < M; ++k2) v[i + Q * k2] = u[k2];
        }
        __syncwarp();
    }
}

__device__ __forceinline__ float warp_sum(float x) {
#pragma unroll
    for (int o = 16; o >= 1; o >>= 1) x += __shfl_xor_sync(0xffffffffu, x, o);
    return x;
}

// ---- power sums, order independent ---------------------------------------------------------
// sum |A_j|^2 over a member's points is accumulated in 64-bit FIXED POINT: every point's |A_j|^2 (fp32) is scaled
// by the member's power-of-two scale pfix = 2^e (exact) and rounded to an integer once; integers add
// associatively, so the result does not depend on which warp, CTA, launch scheme or kernel summed which points,
// nor on the arrival order of the atomics: the power history is bit-reproducible and identical between the
// persistent, per-pass, sparse and cluster kernels.  k_input_power picks e so that the input's total sum maps to
// [2^55, 2^56): 7 bits of headroom (power does not grow, alpha, beta >= 0; a deliberately unstable RK4 step, e.g.
// nz = 1 at kW powers, may gain a factor ~10) and a resolution of 2^-56 of the input per point.
__device__ __forceinline__ long long to_fix(float s, float scale) { return __float2ll_rn(s * scale); }

__device__ __forceinline__ long long warp_sum_ll(long long x) {
#pragma unroll
    for (int o = 16; o >= 1; o >>= 1) x += __shfl_xor_sync(0xffffffffu, x, o);
    return x;
}

__device__ __forceinline__ void fix_add(long long* dst, long long v) {
    atomicAdd(reinterpret_cast<unsigned long long*>(dst), (unsigned long long)v);
}

// history slot of step node `node` (0..nz), or -1 when that node is not recorded (shg_grid.record_every)
__device__ __forceinline__ int rec_slot(const Params& P, int node) {
    if (P.rec_every == 1) return node;
    if (node == P.nz) return P.nrec;
    return (node % P.rec_every == 0) ? node / P.rec_every : -1;
}

// phase reduced to [-pi, pi]
__device__ __forceinline__ float wrap_2pi(float p) {
    constexpr float TWO_PI_HI = 6.2831854820251465f;          // fl32(2 pi)
    constexpr float TWO_PI_LO = -1.7484555314695172e-07f;     // 2 pi - fl32(2 pi)
    float k = rintf(p * 0.15915494309189535f);
    p = fmaf(-k, TWO_PI_HI, p);
    return fmaf(-k, TWO_PI_LO, p);
}

// Coefficients of the nonlinear right-hand side for one sampled phase:
//   dA1 = p * U1 - g1 |A1|^2 A1,  p = A2 conj(A1),  U1 = i kappa1 dz e^{-i phi} = kappa1 dz (s, c)
//   dA2 = q * U2 - g2 |A2|^2 A2,  q = A1^2,         U2 = i kappa2 dz e^{+i phi} = kappa2 dz (-s, c)
struct PhaseCoef { float u1x, u1y, u2x, u2y; };

__device__ __forceinline__ PhaseCoef phase_coef(float c, float s, float k1, float k2) {
    PhaseCoef pc;
    pc.u1x = k1 * s; pc.u1y = k1 * c;
    pc.u2x = -k2 * s; pc.u2y = k2 * c;
    return pc;
}

// Uniform temperature (nzt == 0): phi(z) = dk z exactly (Eq. 3 with constant dk), so z-step n has the same three
// sampled phases at every point.  They are reduced mod 2 pi in double and evaluated once per step into
// the table ucoef[n][3] = {CA, CM, CB} as (u1x, u1y, u2x, u2y) (k_uniform_coefs, built with the other tables; one
// table for all members: kappa_j dz, dz and dk depend on the crystal and T_uniform only, not on a member's window):
// the kernels read 48 bytes per item instead of repeating ~500 double-precision instructions.
__device__ __forceinline__ void uniform_coefs(const MemberDev& mb, int n, PhaseCoef& CA, PhaseCoef& CM, PhaseCoef& CB) {
    const double TWO_PI = 6.283185307179586476925286766559;
    double pa = mb.dk_uniform * ((double)n * mb.dzd);
    double pm = mb.dk_uniform * (((double)n + 0.5) * mb.dzd);
    double pb = mb.dk_uniform * (((double)n + 1.0) * mb.dzd);
    pa -= TWO_PI * rint(pa / TWO_PI);
    pm -= TWO_PI * rint(pm / TWO_PI);
    pb -= TWO_PI * rint(pb / TWO_PI);
    float ca, sa, cm, sm, cb, sb;
    sincosf((float)pa, &sa, &ca);
    sincosf((float)pm, &sm, &cm);
    sincosf((float)pb, &sb, &cb);
    CA = phase_coef(ca, sa, mb.kap1dz, mb.kap2dz);
    CM = phase_coef(cm, sm, mb.kap1dz, mb.kap2dz);
    CB = phase_coef(cb, sb, mb.kap1dz, mb.kap2dz);
}

__device__ __forceinline__ void load_uniform_coefs(const Params& P, int b, int n, PhaseCoef& CA, PhaseCoef& CM, PhaseCoef& CB) {
    const float4* uc = P.ucoef + (size_t)n * 3;        // the same for every member b (crystal and T_uniform only)
    const float4 a = __ldg(uc), c = __ldg(uc + 1), d = __ldg(uc + 2);
    CA.u1x = a.x; CA.u1y = a.y; CA.u2x = a.z; CA.u2y = a.w;
    CM.u1x = c.x; CM.u1y = c.y; CM.u2x = c.z; CM.u2y = c.w;
    CB.u1x = d.x; CB.u1y = d.y; CB.u2x = d.z; CB.u2y = d.w;
}

// dz * N(A) of P:72-73 (Eq. 2) / P:138-145 (Eq. 11) for one point (two-photon terms always evaluated;
// g1 = g2 = 0 switches them off).
__device__ __forceinline__ void nl_rhs(float2 a1, float2 a2, const PhaseCoef& pc, float g1, float g2,
                                       float2& d1, float2& d2) {
    float px = fmaf(a2.x, a1.x, a2.y * a1.y);            // A2 conj(A1)
    float py = fmaf(a2.y, a1.x, -a2.x * a1.y);
    float qx = fmaf(a1.x, a1.x, -a1.y * a1.y);           // A1^2
    float qy = (2.0f * a1.x) * a1.y;
    d1.x = fmaf(px, pc.u1x, -py * pc.u1y);
    d1.y = fmaf(px, pc.u1y, py * pc.u1x);
    d2.x = fmaf(qx, pc.u2x, -qy * pc.u2y);
    d2.y = fmaf(qx, pc.u2y, qy * pc.u2x);
    // (two-photon terms: g_j is the same for every point of a member, so the branches are warp-uniform; a term
    // that is switched off -- beta_1 = 0 in every BASELINE config -- costs a predicate instead of five operations)
    if (g1 != 0.f) {
        float t1 = -g1 * fmaf(a1.x, a1.x, a1.y * a1.y);
        d1.x = fmaf(t1, a1.x, d1.x); d1.y = fmaf(t1, a1.y, d1.y);
    }
    if (g2 != 0.f) {
        float t2 = -g2 * fmaf(a2.x, a2.x, a2.y * a2.y);
        d2.x = fmaf(t2, a2.x, d2.x); d2.y = fmaf(t2, a2.y, d2.y);
    }
}

// One classical RK4 step of length dz; the phase is sampled at z_n, z_n + dz/2, z_n + dz (G8).
__device__ __forceinline__ void rk4_point(float2& a1, float2& a2, const PhaseCoef& ca, const PhaseCoef& cm,
                                          const PhaseCoef& cb, float g1, float g2) {
    float2 k1a, k1b, k2a, k2b, k3a, k3b, k4a, k4b;
    nl_rhs(a1, a2, ca, g1, g2, k1a, k1b);
    nl_rhs(make_float2(fmaf(0.5f, k1a.x, a1.x), fmaf(0.5f, k1a.y, a1.y)),
           make_float2(fmaf(0.5f, k1b.x, a2.x), fmaf(0.5f, k1b.y, a2.y)), cm, g1, g2, k2a, k2b);
    nl_rhs(make_float2(fmaf(0.5f, k2a.x, a1.x), fmaf(0.5f, k2a.y, a1.y)),
           make_float2(fmaf(0.5f, k2b.x, a2.x), fmaf(0.5f, k2b.y, a2.y)), cm, g1, g2, k3a, k3b);
    nl_rhs(make_float2(a1.x + k3a.x, a1.y + k3a.y), make_float2(a2.x + k3b.x, a2.y + k3b.y), cb, g1, g2,
           k4a, k4b);
    // a += (k1 + 2 (k2 + k3) + k4) / 6, every rounding spelled out (the packed twin rk4_point2 repeats them)
    constexpr float S = 1.0f / 6.0f;
    a1.x = fmaf(S, fmaf(2.0f, k2a.x + k3a.x, k1a.x) + k4a.x, a1.x);
    a1.y = fmaf(S, fmaf(2.0f, k2a.y + k3a.y, k1a.y) + k4a.y, a1.y);
    a2.x = fmaf(S, fmaf(2.0f, k2b.x + k3b.x, k1b.x) + k4b.x, a2.x);
    a2.y = fmaf(S, fmaf(2.0f, k2b.y + k3b.y, k1b.y) + k4b.y, a2.y);
}

// ---- the same for TWO points at once in Blackwell's packed fp32x2 instructions (FFMA2 / FMUL2 / FADD2) ----------
// A float2 here is NOT a complex number but one real quantity of two points (.x = point q, .y = point q + 1).  The
// nonlinear step is bound by instruction issue (232 instructions per point, 174 of them fp32 arithmetic, at 0.84 per
// clock with four warps per scheduler: profiles/r02b_summary.md 3); a packed instruction does the arithmetic of both
// points in one issue slot.  Every operation is the one of the scalar code above, in the same order, so both give
// the same bits.  What made an earlier attempt useless (+186 MOVs to form the pairs) was the complex
// (re, im) layout of the line in shared memory; row_item now writes the line "split" for the nonlinear step --
// (re_q, re_q+1) and (im_q, im_q+1) as two 8-byte records -- so that the pairs arrive as pairs.
struct PhaseCoef2 { float2 u1x, u1y, u2x, u2y; };
__device__ __forceinline__ float2 bc2(float a) { return make_float2(a, a); }
__device__ __forceinline__ float2 ng2(float2 a) { return make_float2(-a.x, -a.y); }

__device__ __forceinline__ PhaseCoef2 phase_coef2(float2 c, float2 s, float k1, float k2) {
    PhaseCoef2 pc;
    pc.u1x = __fmul2_rn(bc2(k1), s); pc.u1y = __fmul2_rn(bc2(k1), c);
    pc.u2x = __fmul2_rn(bc2(-k2), s); pc.u2y = __fmul2_rn(bc2(k2), c);
    return pc;
}
__device__ __forceinline__ PhaseCoef2 phase_coef2(const PhaseCoef& p) {
    PhaseCoef2 pc;
    pc.u1x = bc2(p.u1x); pc.u1y = bc2(p.u1y); pc.u2x = bc2(p.u2x); pc.u2y = bc2(p.u2y);
    return pc;
}

__device__ __forceinline__ void nl_rhs2(float2 a1x, float2 a1y, float2 a2x, float2 a2y, const PhaseCoef2& pc, float g1,
                                        float g2, float2& d1x, float2& d1y, float2& d2x, float2& d2y) {
    const float2 px = __ffma2_rn(a2x, a1x, __fmul2_rn(a2y, a1y));            // A2 conj(A1)
    const float2 py = __ffma2_rn(a2y, a1x, __fmul2_rn(ng2(a2x), a1y));
    const float2 qx = __ffma2_rn(a1x, a1x, __fmul2_rn(ng2(a1y), a1y));       // A1^2
    const float2 qy = __fmul2_rn(__fmul2_rn(bc2(2.0f), a1x), a1y);
    d1x = __ffma2_rn(px, pc.u1x, __fmul2_rn(ng2(py), pc.u1y));
    d1y = __ffma2_rn(px, pc.u1y, __fmul2_rn(py, pc.u1x));
    d2x = __ffma2_rn(qx, pc.u2x, __fmul2_rn(ng2(qy), pc.u2y));
    d2y = __ffma2_rn(qx, pc.u2y, __fmul2_rn(qy, pc.u2x));
    if (g1 != 0.f) {
        const float2 t1 = __fmul2_rn(bc2(-g1), __ffma2_rn(a1x, a1x, __fmul2_rn(a1y, a1y)));
        d1x = __ffma2_rn(t1, a1x, d1x); d1y = __ffma2_rn(t1, a1y, d1y);
    }
    if (g2 != 0.f) {
        const float2 t2 = __fmul2_rn(bc2(-g2), __ffma2_rn(a2x, a2x, __fmul2_rn(a2y, a2y)));
        d2x = __ffma2_rn(t2, a2x, d2x); d2y = __ffma2_rn(t2, a2y, d2y);
    }
}

__device__ __forceinline__ void rk4_point2(float2& a1x, float2& a1y, float2& a2x, float2& a2y, const PhaseCoef2& ca,
                                           const PhaseCoef2& cm, const PhaseCoef2& cb, float g1, float g2) {
    float2 k1ax, k1ay, k1bx, k1by, k2ax, k2ay, k2bx, k2by, k3ax, k3ay, k3bx, k3by, k4ax, k4ay, k4bx, k4by;
    const float2 h = bc2(0.5f), two = bc2(2.0f), S = bc2(1.0f / 6.0f);
    nl_rhs2(a1x, a1y, a2x, a2y, ca, g1, g2, k1ax, k1ay, k1bx, k1by);
    nl_rhs2(__ffma2_rn(h, k1ax, a1x), __ffma2_rn(h, k1ay, a1y), __ffma2_rn(h, k1bx, a2x), __ffma2_rn(h, k1by, a2y), cm,
            g1, g2, k2ax, k2ay, k2bx, k2by);
    nl_rhs2(__ffma2_rn(h, k2ax, a1x), __ffma2_rn(h, k2ay, a1y), __ffma2_rn(h, k2bx, a2x), __ffma2_rn(h, k2by, a2y), cm,
            g1, g2, k3ax, k3ay, k3bx, k3by);
    nl_rhs2(__fadd2_rn(a1x, k3ax), __fadd2_rn(a1y, k3ay), __fadd2_rn(a2x, k3bx), __fadd2_rn(a2y, k3by), cb, g1, g2,
            k4ax, k4ay, k4bx, k4by);
    a1x = __ffma2_rn(S, __fadd2_rn(__ffma2_rn(two, __fadd2_rn(k2ax, k3ax), k1ax), k4ax), a1x);
    a1y = __ffma2_rn(S, __fadd2_rn(__ffma2_rn(two, __fadd2_rn(k2ay, k3ay), k1ay), k4ay), a1y);
    a2x = __ffma2_rn(S, __fadd2_rn(__ffma2_rn(two, __fadd2_rn(k2bx, k3bx), k1bx), k4bx), a2x);
    a2y = __ffma2_rn(S, __fadd2_rn(__ffma2_rn(two, __fadd2_rn(k2by, k3by), k1by), k4by), a2y);
}

// Raw operands of one point's phase update: the (up to) two temperature planes around z_n and around
// z_{n+1}, and the running phase.  Loaded one RK4 iteration ahead of their use (software pipeline).
struct TPoint { float a0, a1, b0, b1, ph; };

__device__ __forceinline__ TPoint t_load(const float* __restrict__ Ta, const float* __restrict__ Tn, size_t plane,
                                         size_t idx, bool two_a, bool two_b, const float* __restrict__ phi_q) {
    TPoint t;
    t.a0 = __ldg(Ta + idx);
    t.a1 = two_a ? __ldg(Ta + plane + idx) : 0.f;
    t.b0 = __ldg(Tn + idx);
    t.b1 = two_b ? __ldg(Tn + plane + idx) : 0.f;
    t.ph = __ldcg(phi_q);
    return t;
}

// Temperature rise T - T_pm from a plane pair (k, k+1) with weight f  (G15).
__device__ __forceinline__ float dT_lerp(float t0, float t1, float f, bool two, float Thi, float Tlo) {
    float a = (t0 - Thi) - Tlo;
    if (two) {
        float b = (t1 - Thi) - Tlo;
        a = fmaf(f, b - a, a);
    }
    return a;
}

__device__ __forceinline__ float2 dT_lerp2(float2 t0, float2 t1, float f, bool two, float Thi, float Tlo) {
    float2 a = __fadd2_rn(__fadd2_rn(t0, bc2(-Thi)), bc2(-Tlo));
    if (two) {
        const float2 b = __fadd2_rn(__fadd2_rn(t1, bc2(-Thi)), bc2(-Tlo));
        a = __ffma2_rn(bc2(f), __fadd2_rn(b, ng2(a)), a);
    }
    return a;
}
__device__ __forceinline__ float2 wrap_2pi2(float2 p) {
    constexpr float TWO_PI_HI = 6.2831854820251465f, TWO_PI_LO = -1.7484555314695172e-07f;
    const float2 t = __fmul2_rn(p, bc2(0.15915494309189535f));
    const float2 k = make_float2(rintf(t.x), rintf(t.y));
    p = __ffma2_rn(ng2(k), bc2(TWO_PI_HI), p);
    return __ffma2_rn(ng2(k), bc2(TWO_PI_LO), p);
}

// Which T planes serve step node n: k = min(floor(n (nzt-1)/nz), nzt-2), f = frac.
struct TNode { int k; float f; bool two; };
__device__ __forceinline__ TNode t_node(int n, int nz, int nzt) {
    TNode t;
    if (nzt <= 1) { t.k = 0; t.f = 0.f; t.two = false; return t; }
    long long num = (long long)n * (nzt - 1);
    int k = (int)(num / nz);
    int rem = (int)(num - (long long)k * nz);
    if (k > nzt - 2) { k = nzt - 2; rem = nz; }
    t.k = k; t.f = (float)rem / (float)nz; t.two = (rem != 0);
    return t;
}

// Scalars that are the same for every item of a CTA's pass.  Computing them per item costs two 64-bit and one
// 32-bit integer division (~400 instructions) at the head of every row item, where all warps of the CTA execute them
// at the same time right after a device-wide barrier and nothing else can be issued (measured on cfg5 with per-warp
// clock stamps: ~2.5 K of the row pass's 39.5 K clocks).  They live in shared memory instead: the ranges are fixed
// for the run, the step's entries are written by ONE thread while it waits at the barrier before the pass.
struct StepCtx {
    int row_lo, row_hi, col_lo, col_hi;    // cta_range of the row items / column strips
    TNode ta, tb;                          // temperature planes of step nodes n and n + 1 (G15)
    int slot;                              // rec_slot(n + 1): history slot of P_j(z_{n+1}), -1 = not recorded
};

__device__ __forceinline__ void cta_range(int U, int& lo, int& hi);
template <int NX> __host__ __device__ inline int row_items(int batch, int ny);
template <int NY> __host__ __device__ inline int col_items(int batch, int nx);

template <int NX> __device__ __forceinline__ void ctx_rows(const Params& P, StepCtx& sc) {
    cta_range(row_items<NX>(P.batch, P.ny), sc.row_lo, sc.row_hi);
}
template <int NY> __device__ __forceinline__ void ctx_cols(const Params& P, StepCtx& sc) {
    cta_range(col_items<NY>(P.batch, P.nx), sc.col_lo, sc.col_hi);
}
__device__ __forceinline__ void ctx_step(const Params& P, StepCtx& sc, int n) {
    sc.ta = t_node(n, P.nz, P.nzt);
    sc.tb = t_node(n + 1, P.nz, P.nzt);
    sc.slot = rec_slot(P, n + 1);
}

// ------------------------------------------------------------------------------------------------
// Row pass, one item = HG rows x both fields.  Lane group g of the warp holds one line: field f, row r.
// (G == 1: the item is one row and the two warps of a pair hold its two fields.)
//   ROW_FIRST : A_in (real space) -> P_j(0) -> F_x -> * hx                          -> A
//   ROW_MID   : A -> F_x -> conj -> [T -> dk -> phi] -> RK4 -> P_j(z_{n+1}) -> F_x -> * hx -> A
//   ROW_FINAL : A -> F_x -> conj -> A (output, real space)
// smem_cta: base of the per-warp line regions.  hsel: 0 = full-step tables, 1 = half-step tables.
// ------------------------------------------------------------------------------------------------
// HEAT: also write the heat source of Eq. 8 (a separate instantiation: the common path carries none of it).
// TS: the hx tables are read from shared memory (stab: [2][NX] float4, single simulation) instead of global / L1.
template <int NX, int MODE, bool PREC, bool HEAT = false, bool TS = false>
__device__ __forceinline__ void row_item(const Params& P, const StepCtx& sc, int item, int n, int hsel, float2* smem_cta,
                                         const float4* __restrict__ tws, int warp, int lane,
                                         const float4* __restrict__ stab = nullptr,
                                         unsigned long long* s_pow = nullptr) {
    using GE = Geo<NX>;
    constexpr int R = GE::R, M = GE::M, G = GE::G, NP = GE::NP, HG = GE::HG, H = R / 2;
    const int g = lane / M, m = lane % M;
    const int f = (G >= 2) ? g / HG : (warp & 1);
    const int r = (G >= 2) ? g % HG : 0;
    const int row = item * HG + r;                            // over [batch * ny]
    const int b = (item * HG) >> P.ny_log2;                   // (ny is a power of two)
    const int y = row - (b << P.ny_log2);
    const size_t rbase = (size_t)row * NX;
    float2* own = smem_cta + (size_t)warp * (G * NP) + g * NP;
    float2* par = (G >= 2) ? smem_cta + (size_t)warp * (G * NP) + (g ^ HG) * NP
                           : smem_cta + (size_t)(warp ^ 1) * (G * NP);
    const MemberDev& mb = P.mem[b];
    const int rot = f ? NX / 2 : 0;                           // the SH row lives rotated by N/2 in real space
    float2 v[R];

    if constexpr (MODE == ROW_FIRST) {
        const float2* src = f ? P.Ain[1] : P.Ain[0];
        if (src) {
#pragma unroll
            for (int q = 0; q < R; ++q) v[q] = src[rbase + ((M * q + m + rot) & (NX - 1))];
        } else {
#pragma unroll
            for (int q = 0; q < R; ++q) v[q] = make_float2(0.f, 0.f);
        }
        // (P_j(0) is taken from the input by k_input_power, which also fixes the member's fixed-point scale)
        warp_fft<NX, PREC>(v, own, tws, m);
        table_mul<R, M, PREC, false>(v, P.hx[hsel] + ((size_t)b * 2 + f) * NX + m);
        float2* dst = (f ? P.A[1] : P.A[0]) + rbase;
#pragma unroll
        for (int q = 0; q < R; ++q) stcg2(dst + M * q + m, v[q]);
        return;
    }

    if constexpr (MODE == ROW_FINAL) {
        float2* A = (f ? P.A[1] : P.A[0]) + rbase;
#pragma unroll
        for (int q = 0; q < R; ++q) v[q] = ldcg2(A + M * q + m);
        warp_fft<NX, PREC>(v, own, tws, m);
#pragma unroll
        for (int q = 0; q < R; ++q) stcg2(A + ((M * q + m + rot) & (NX - 1)), make_float2(v[q].x, -v[q].y));
        return;
    }

    if constexpr (MODE == ROW_MID) {
        float2* A = (f ? P.A[1] : P.A[0]) + rbase;
        const float4* hx = P.hx[hsel] + ((size_t)b * 2 + f) * NX;
#pragma unroll
        for (int q = 0; q < R; ++q) v[q] = ldcg2(A + M * q + m);
        if constexpr (!TS) table_prefetch<R, M>(hx, m);
        if (P.nzt == 0) asm volatile("prefetch.global.L1 [%0];" ::"l"(P.ucoef + (size_t)n * 3));
        // temperature / phase operands of the first RK4 point are requested before the transform (when
        // registers allow), those of the second right after it; inside the loop two points ahead
        const size_t plane = (size_t)P.ny * NX;
        const size_t pbase = (size_t)y * NX + rot + m;
        const TNode ta = sc.ta, tb = sc.tb;
        const float* Ta = nullptr;
        const float* Tn = nullptr;
        float* phi = nullptr;
        TPoint cur{}, nxt{};
        if (P.nzt != 0) {
            const float* Tb = P.T + (P.T_per_member ? (size_t)b * P.nzt * plane : 0);
            Ta = Tb + (size_t)ta.k * plane;
            Tn = Tb + (size_t)tb.k * plane;
            phi = P.phi + (size_t)b * plane + pbase;
            if constexpr (R < 32) cur = t_load(Ta, Tn, plane, pbase, ta.two, tb.two, phi);
        }
        warp_fft<NX, PREC>(v, own, tws, m);
        if (P.nzt != 0) {
            // (a 32-value line leaves no registers to carry operands across the transform)
            if constexpr (R >= 32) cur = t_load(Ta, Tn, plane, pbase, ta.two, tb.two, phi);
            nxt = t_load(Ta, Tn, plane, pbase + M, ta.two, tb.two, phi + M);
        }
        // conj(field), rotated for f = 1, goes to shared memory: register q <-> element M q + m (+ N/2).
        // PK (no heat output): "split" image for the packed two-point RK4 -- slot M q + m holds (re_q, re_q+1) and
        // slot M (q + 1) + m holds (im_q, im_q+1) for even q, instead of the complex values of points q and q + 1
        // (not for 1024-point rows with global tables, where the packed loop makes ptxas spill: stream1024 +1 %)
        constexpr bool PK = !HEAT && (TS || G >= 2);
        if constexpr (PK) {
#pragma unroll
            for (int q = 0; q < R; q += 2) {
                own[M * q + m] = make_float2(v[q].x, v[q + 1].x);
                own[M * (q + 1) + m] = make_float2(v[q].y, v[q + 1].y);
            }
        } else {
#pragma unroll
            for (int q = 0; q < R; ++q) own[M * q + m] = v[q];
        }
        if constexpr (G >= 2) __syncwarp(); else named_barrier(1 + (warp >> 1), 64);

        // ---- nonlinear step on elements e = M q + m + f N/2, q < R/2: own lower half, partner's upper half.
        // p1 / p2 address A1 / A2 of this lane's points whichever side it is on (no value selects).
        float2* p1 = (f ? par + M * H : own) + m;
        float2* p2 = (f ? own : par + M * H) + m;
        const float k1dz = mb.kap1dz, k2dz = mb.kap2dz, g1 = mb.g1dz, g2 = mb.g2dz;
        const int slot = sc.slot;                             // warp-uniform: is P_j(z_{n+1}) recorded?
        const float fsc = P.pfix[b];
        long long s1 = 0, s2 = 0;
        // Heat source of Eq. 8 for the plane that samples this z-step, if any (warp-uniform): half of
        // q on the fields before the nonlinear step now, the other half after it (G27).  Only nq of the nz
        // steps come here, so the two extra sweeps over the line in shared memory stay off the common path.
        float* qrow = nullptr;
        if constexpr (HEAT) {
            const int kq = P.qmap[n];
            if (kq >= 0) qrow = P.Q + (((size_t)b * P.nq + kq) * P.ny + y) * NX + rot + m;
        }
        auto heat_half = [&](bool first) {
#pragma unroll 4
            for (int q = 0; q < H; ++q) {
                const float2 a1 = p1[M * q], a2 = p2[M * q];
                const float i1 = fmaf(a1.x, a1.x, a1.y * a1.y), i2 = fmaf(a2.x, a2.x, a2.y * a2.y);
                const float h = 0.5f * fmaf(i1, fmaf(mb.qb1, i1, mb.qa1), i2 * fmaf(mb.qb2, i2, mb.qa2));
                if (first) qrow[M * q] = h; else qrow[M * q] += h;
            }
        };
        if constexpr (HEAT) { if (qrow) heat_half(true); }
        if constexpr (PK) {
          // ---- two points per iteration in packed fp32x2 (rk4_point2): .x = point q, .y = point q + 1
          auto finish2 = [&](int q, float2 a1x, float2 a1y, float2 a2x, float2 a2y) {
              if (slot >= 0) {
                  const float2 i1 = __fmul2_rn(__ffma2_rn(a1x, a1x, __fmul2_rn(a1y, a1y)), bc2(fsc));
                  const float2 i2 = __fmul2_rn(__ffma2_rn(a2x, a2x, __fmul2_rn(a2y, a2y)), bc2(fsc));
                  s1 += __float2ll_rn(i1.x) + __float2ll_rn(i1.y);
                  s2 += __float2ll_rn(i2.x) + __float2ll_rn(i2.y);
              }
              p1[M * q] = a1x; p1[M * (q + 1)] = a1y;
              p2[M * q] = a2x; p2[M * (q + 1)] = a2y;
          };
          if (P.nzt == 0) {
            // uniform temperature: the step's coefficients from the table (warp-uniform 48-byte read)
            PhaseCoef CA, CM, CB;
            load_uniform_coefs(P, b, n, CA, CM, CB);
            const PhaseCoef2 A2c = phase_coef2(CA), M2c = phase_coef2(CM), B2c = phase_coef2(CB);
#pragma unroll 1
            for (int q = 0; q < H; q += 2) {
                float2 a1x = p1[M * q], a1y = ng2(p1[M * (q + 1)]);
                float2 a2x = p2[M * q], a2y = ng2(p2[M * (q + 1)]);
                rk4_point2(a1x, a1y, a2x, a2y, A2c, M2c, B2c, g1, g2);
                finish2(q, a1x, a1y, a2x, a2y);
            }
          } else {
            const float hdz = 0.5f * mb.dz, e8 = 0.125f * mb.dz;
            const float gT = mb.gT, dk0 = mb.dk0, Thi = mb.Tpm_hi, Tlo = mb.Tpm_lo;
#pragma unroll 1
            for (int q = 0; q < H; q += 2) {
                // consume the operands of points q, q + 1 (requested two points earlier), request those of q + 2, q + 3
                const TPoint t0 = cur, t1 = nxt;
                const int qa = (q + 2 < H) ? q + 2 : H - 1, qb = (q + 3 < H) ? q + 3 : H - 1;   // clamped tail
                cur = t_load(Ta, Tn, plane, pbase + M * qa, ta.two, tb.two, phi + M * qa);
                nxt = t_load(Ta, Tn, plane, pbase + M * qb, ta.two, tb.two, phi + M * qb);
                const float2 dTa = dT_lerp2(make_float2(t0.a0, t1.a0), make_float2(t0.a1, t1.a1), ta.f, ta.two, Thi, Tlo);
                const float2 dTb = dT_lerp2(make_float2(t0.b0, t1.b0), make_float2(t0.b1, t1.b1), tb.f, tb.two, Thi, Tlo);
                const float2 dka = __ffma2_rn(bc2(gT), dTa, bc2(dk0)), dkb = __ffma2_rn(bc2(gT), dTb, bc2(dk0));
                const float2 ph = make_float2(t0.ph, t1.ph);
                const float2 phm = __ffma2_rn(bc2(e8), __ffma2_rn(bc2(3.0f), dka, dkb), ph);   // phi_n + dz (3 dk_n + dk_{n+1})/8
                const float2 phb = __ffma2_rn(bc2(hdz), __fadd2_rn(dka, dkb), ph);             // phi_n + dz (dk_n + dk_{n+1})/2
                float2 ca, sa, cm, sm, cb, sb;
                __sincosf(ph.x, &sa.x, &ca.x);   __sincosf(ph.y, &sa.y, &ca.y);
                __sincosf(phm.x, &sm.x, &cm.x);  __sincosf(phm.y, &sm.y, &cm.y);
                __sincosf(phb.x, &sb.x, &cb.x);  __sincosf(phb.y, &sb.y, &cb.y);
                const float2 pw = wrap_2pi2(phb);
                __stcg(phi + M * q, pw.x);
                __stcg(phi + M * (q + 1), pw.y);
                const PhaseCoef2 CA = phase_coef2(ca, sa, k1dz, k2dz), CM = phase_coef2(cm, sm, k1dz, k2dz),
                                 CB = phase_coef2(cb, sb, k1dz, k2dz);
                float2 a1x = p1[M * q], a1y = ng2(p1[M * (q + 1)]);
                float2 a2x = p2[M * q], a2y = ng2(p2[M * (q + 1)]);
                rk4_point2(a1x, a1y, a2x, a2y, CA, CM, CB, g1, g2);
                finish2(q, a1x, a1y, a2x, a2y);
            }
          }
        } else if (P.nzt == 0) {
            // uniform temperature: the step's coefficients from the table (warp-uniform 48-byte read)
            PhaseCoef CA, CM, CB;
            load_uniform_coefs(P, b, n, CA, CM, CB);
#pragma unroll 2
            for (int q = 0; q < H; ++q) {
                float2 a1 = p1[M * q], a2 = p2[M * q];
                a1.y = -a1.y; a2.y = -a2.y;
                rk4_point(a1, a2, CA, CM, CB, g1, g2);
                if (slot >= 0) {
                    s1 += to_fix(fmaf(a1.x, a1.x, a1.y * a1.y), fsc);
                    s2 += to_fix(fmaf(a2.x, a2.x, a2.y * a2.y), fsc);
                }
                p1[M * q] = a1;
                p2[M * q] = a2;
            }
        } else {
            const float hdz = 0.5f * mb.dz, e8 = 0.125f * mb.dz;
            const float gT = mb.gT, dk0 = mb.dk0, Thi = mb.Tpm_hi, Tlo = mb.Tpm_lo;
            // one point: consume operands tp (requested two points earlier), request those of point q + 2
            auto point = [&](int q, TPoint& tp) {
                const float a0 = tp.a0, a1v = tp.a1, b0 = tp.b0, b1 = tp.b1, ph = tp.ph;
                const int qn = (q + 2 < H) ? q + 2 : H - 1;          // clamped: the tail re-reads, never branches
                tp = t_load(Ta, Tn, plane, pbase + M * qn, ta.two, tb.two, phi + M * qn);
                float dTa = dT_lerp(a0, a1v, ta.f, ta.two, Thi, Tlo);
                float dTb = dT_lerp(b0, b1, tb.f, tb.two, Thi, Tlo);
                float dka = fmaf(gT, dTa, dk0), dkb = fmaf(gT, dTb, dk0);
                float phm = fmaf(e8, fmaf(3.0f, dka, dkb), ph);        // phi_n + dz (3 dk_n + dk_{n+1})/8
                float phb = fmaf(hdz, dka + dkb, ph);                  // phi_n + dz (dk_n + dk_{n+1})/2
                float ca, sa, cm, sm, cb, sb;
                __sincosf(ph, &sa, &ca);
                __sincosf(phm, &sm, &cm);
                __sincosf(phb, &sb, &cb);
                __stcg(phi + M * q, wrap_2pi(phb));
                const PhaseCoef CA = phase_coef(ca, sa, k1dz, k2dz), CM = phase_coef(cm, sm, k1dz, k2dz),
                                CB = phase_coef(cb, sb, k1dz, k2dz);
                float2 a1 = p1[M * q], a2 = p2[M * q];
                a1.y = -a1.y; a2.y = -a2.y;
                rk4_point(a1, a2, CA, CM, CB, g1, g2);
                if (slot >= 0) {
                    s1 += to_fix(fmaf(a1.x, a1.x, a1.y * a1.y), fsc);
                    s2 += to_fix(fmaf(a2.x, a2.x, a2.y * a2.y), fsc);
                }
                p1[M * q] = a1;
                p2[M * q] = a2;
            };
#pragma unroll 1
            for (int q = 0; q < H; q += 2) {
                point(q, cur);
                point(q + 1, nxt);
            }
        }
        if constexpr (HEAT) { if (qrow) heat_half(false); }
        if (slot >= 0) {
            s1 = warp_sum_ll(s1); s2 = warp_sum_ll(s2);
            if (lane == 0) {
                if (s_pow) {
                    // single simulation: the CTA's sums meet in shared memory; one global atomic per CTA, field
                    // and step (flush_powers) instead of one per warp on the same two history words
                    atomicAdd(s_pow + 0, (unsigned long long)s1);
                    atomicAdd(s_pow + 1, (unsigned long long)s2);
                } else {
                    long long* hst = P.hfix + ((long long)b * (P.nrec + 1) + slot) * 2;
                    fix_add(hst + 0, s1);
                    fix_add(hst + 1, s2);
                }
            }
        }
        if constexpr (G >= 2) __syncwarp(); else named_barrier(1 + (warp >> 1), 64);
        if constexpr (PK) {
#pragma unroll
            for (int q = 0; q < R; q += 2) {
                const float2 re = own[M * q + m], im = own[M * (q + 1) + m];
                v[q] = make_float2(re.x, im.x);
                v[q + 1] = make_float2(re.y, im.y);
            }
        } else {
#pragma unroll
            for (int q = 0; q < R; ++q) v[q] = own[M * q + m];
        }
        __syncwarp();
        warp_fft<NX, PREC>(v, own, tws, m);
        if constexpr (TS)
            table_mul_s<R, M, PREC, false>(v, (unsigned)__cvta_generic_to_shared(stab + f * NX + m),
                                           std::make_integer_sequence<int, R>{});
        else
            table_mul<R, M, PREC, false>(v, hx + m);
#pragma unroll
        for (int q = 0; q < R; ++q) stcg2(A + M * q + m, v[q]);
    }
}

// ------------------------------------------------------------------------------------------------
// The paper's own ordering, Eq. 14-15:  N(dz/2) - L(dz) - N(dz/2)  per z-step (SHG_OPT_SCHEME = 1).
// Two consecutive nonlinear half-steps meet in real space, so the row pass between the linear steps of z-step
// n and n + 1 takes the second half of step n, records P_j(z_{n+1}) at the true node, and takes the first half
// of step n + 1:
//   ROW_FIRST : A_in -> P_j(0) -> N(dz/2) [step 0, first half] -> F_x -> * hx(dz)                     -> A
//   ROW_MID   : A -> F_x -> conj -> N(dz/2) [step n, second] -> P_j(z_{n+1}) -> N(dz/2) [step n+1, first]
//                 -> F_x -> * hx(dz)                                                                  -> A
//   ROW_FINAL : A -> F_x -> conj -> N(dz/2) [step nz-1, second] -> P_j(L)                             -> A_out
// The linear step is always a full dz (tables index 0); the column pass is the one of the merged scheme.
// Phases inside a step (G15, dk linear in z):  phi(z_n + s) = phi_n + s dk_n + s^2 (dk_{n+1} - dk_n)/(2 dz),
// sampled at s = 0, dz/4, dz/2 (first half) and dz/2, 3dz/4, dz (second half): RK4 of length dz/2 (G8).
// A variant, not the benchmarked path: no software pipelining of the temperature loads.
// ------------------------------------------------------------------------------------------------
// Temperature rise at step node j for the point at idx (G15)
__device__ __forceinline__ float dT_at_node(const float* __restrict__ Tb, size_t plane, size_t idx, const TNode& t,
                                            float Thi, float Tlo) {
    const float* p = Tb + (size_t)t.k * plane + idx;
    const float t0 = __ldg(p);
    const float t1 = t.two ? __ldg(p + plane) : 0.f;
    return dT_lerp(t0, t1, t.f, t.two, Thi, Tlo);
}

// phase reduced to [-pi, pi] in double, returned as float (uniform temperature: phi = dk z exactly)
__device__ __forceinline__ float wrapped_phase(double p) {
    const double TWO_PI = 6.283185307179586476925286766559;
    return (float)(p - TWO_PI * rint(p / TWO_PI));
}

template <int NX, int MODE, bool PREC>
__device__ __forceinline__ void row_item_paper(const Params& P, int item, int n, float2* smem_cta,
                                               const float4* __restrict__ tws, int warp, int lane) {
    using GE = Geo<NX>;
    constexpr int R = GE::R, M = GE::M, G = GE::G, NP = GE::NP, HG = GE::HG, H = R / 2;
    const int g = lane / M, m = lane % M;
    const int f = (G >= 2) ? g / HG : (warp & 1);
    const int r = (G >= 2) ? g % HG : 0;
    const int row = item * HG + r;
    const int b = (item * HG) / P.ny;
    const int y = row - b * P.ny;
    const size_t rbase = (size_t)row * NX;
    float2* own = smem_cta + (size_t)warp * (G * NP) + g * NP;
    float2* par = (G >= 2) ? smem_cta + (size_t)warp * (G * NP) + (g ^ HG) * NP
                           : smem_cta + (size_t)(warp ^ 1) * (G * NP);
    const MemberDev& mb = P.mem[b];
    const int rot = f ? NX / 2 : 0;
    float2 v[R];

    if constexpr (MODE == ROW_FIRST) {
        const float2* src = f ? P.Ain[1] : P.Ain[0];
        if (src) {
#pragma unroll
            for (int q = 0; q < R; ++q) v[q] = src[rbase + ((M * q + m + rot) & (NX - 1))];
        } else {
#pragma unroll
            for (int q = 0; q < R; ++q) v[q] = make_float2(0.f, 0.f);
        }
    } else {
        float2* A = (f ? P.A[1] : P.A[0]) + rbase;
#pragma unroll
        for (int q = 0; q < R; ++q) v[q] = ldcg2(A + M * q + m);
        warp_fft<NX, PREC>(v, own, tws, m);             // inverse along x of the previous linear step (conj trick)
    }
    // the line meets its partner field in shared memory (MID / FINAL: conj(field) is stored)
#pragma unroll
    for (int q = 0; q < R; ++q) own[M * q + m] = v[q];
    if constexpr (G >= 2) __syncwarp(); else named_barrier(1 + (warp >> 1), 64);

    // ---- nonlinear half-steps on elements e = M q + m + f N/2, q < R/2 (own lower half, partner's upper half)
    float2* p1 = (f ? par + M * H : own) + m;
    float2* p2 = (f ? own : par + M * H) + m;
    constexpr bool DO_SECOND = (MODE != ROW_FIRST);     // second half of z-step n
    constexpr bool DO_FIRST = (MODE != ROW_FINAL);      // first half of z-step n1
    const int n1 = (MODE == ROW_FIRST) ? 0 : n + 1;
    const float k1h = 0.5f * mb.kap1dz, k2h = 0.5f * mb.kap2dz, g1h = 0.5f * mb.g1dz, g2h = 0.5f * mb.g2dz;
    const int slot = DO_SECOND ? rec_slot(P, n + 1) : -1;
    const float fsc = P.pfix[b];
    long long s1 = 0, s2 = 0;
    if (P.nzt == 0) {
        // uniform temperature: phi(z) = dk z exactly, all sampled phases are warp-uniform
        PhaseCoef S[3], F[3];
        const double z0 = (double)n * mb.dzd, z1 = (double)n1 * mb.dzd;
        const double zs[3] = {z0 + 0.5 * mb.dzd, z0 + 0.75 * mb.dzd, z0 + mb.dzd};
        const double zf[3] = {z1, z1 + 0.25 * mb.dzd, z1 + 0.5 * mb.dzd};
#pragma unroll
        for (int i = 0; i < 3; ++i) {
            float c, sn;
            if (DO_SECOND) { sincosf(wrapped_phase(mb.dk_uniform * zs[i]), &sn, &c); S[i] = phase_coef(c, sn, k1h, k2h); }
            if (DO_FIRST) { sincosf(wrapped_phase(mb.dk_uniform * zf[i]), &sn, &c); F[i] = phase_coef(c, sn, k1h, k2h); }
        }
#pragma unroll 1
        for (int q = 0; q < H; ++q) {
            float2 a1 = p1[M * q], a2 = p2[M * q];
            if (MODE != ROW_FIRST) { a1.y = -a1.y; a2.y = -a2.y; }
            if (DO_SECOND) {
                rk4_point(a1, a2, S[0], S[1], S[2], g1h, g2h);
                if (slot >= 0) {
                    s1 += to_fix(fmaf(a1.x, a1.x, a1.y * a1.y), fsc);
                    s2 += to_fix(fmaf(a2.x, a2.x, a2.y * a2.y), fsc);
                }
            }
            if (DO_FIRST) rk4_point(a1, a2, F[0], F[1], F[2], g1h, g2h);
            p1[M * q] = a1;
            p2[M * q] = a2;
        }
    } else {
        const size_t plane = (size_t)P.ny * NX;
        const size_t pbase = (size_t)y * NX + rot + m;
        const float* Tb = P.T + (P.T_per_member ? (size_t)b * P.nzt * plane : 0);
        float* phi = P.phi + (size_t)b * plane + pbase;
        const TNode tn0 = t_node(n, P.nz, P.nzt), tn1 = t_node(n1, P.nz, P.nzt), tn2 = t_node(n1 + 1, P.nz, P.nzt);
        const float dz = mb.dz, gT = mb.gT, dk0c = mb.dk0, Thi = mb.Tpm_hi, Tlo = mb.Tpm_lo;
        auto half = [&](float2& a1, float2& a2, float pa, float pm, float pb) {
            float ca, sa, cm, sm, cb, sb;
            __sincosf(pa, &sa, &ca);
            __sincosf(pm, &sm, &cm);
            __sincosf(pb, &sb, &cb);
            rk4_point(a1, a2, phase_coef(ca, sa, k1h, k2h), phase_coef(cm, sm, k1h, k2h),
                      phase_coef(cb, sb, k1h, k2h), g1h, g2h);
        };
#pragma unroll 1
        for (int q = 0; q < H; ++q) {
            const size_t idx = pbase + (size_t)(M * q);
            float2 a1 = p1[M * q], a2 = p2[M * q];
            if (MODE != ROW_FIRST) { a1.y = -a1.y; a2.y = -a2.y; }
            float ph = __ldcg(phi + M * q);                                  // phi at node n (MID, FINAL) / 0 (FIRST)
            float dkA = fmaf(gT, dT_at_node(Tb, plane, idx, tn1, Thi, Tlo), dk0c);   // dk at node n1
            if (DO_SECOND) {
                const float dk0 = fmaf(gT, dT_at_node(Tb, plane, idx, tn0, Thi, Tlo), dk0c);   // node n; dkA = node n+1
                const float pa = fmaf(0.125f * dz, fmaf(3.0f, dk0, dkA), ph);
                const float pm = fmaf(0.03125f * dz, fmaf(15.0f, dk0, 9.0f * dkA), ph);
                const float pb = fmaf(0.5f * dz, dk0 + dkA, ph);
                half(a1, a2, pa, pm, pb);
                if (slot >= 0) {
                    s1 += to_fix(fmaf(a1.x, a1.x, a1.y * a1.y), fsc);
                    s2 += to_fix(fmaf(a2.x, a2.x, a2.y * a2.y), fsc);
                }
                ph = wrap_2pi(pb);
                __stcg(phi + M * q, ph);                                     // phi at node n + 1
            }
            if (DO_FIRST) {
                const float dkB = fmaf(gT, dT_at_node(Tb, plane, idx, tn2, Thi, Tlo), dk0c);   // node n1 + 1
                const float pm = fmaf(0.03125f * dz, fmaf(7.0f, dkA, dkB), ph);
                const float pb = fmaf(0.125f * dz, fmaf(3.0f, dkA, dkB), ph);
                half(a1, a2, ph, pm, pb);
            }
            p1[M * q] = a1;
            p2[M * q] = a2;
        }
    }
    // ---- powers at the true nodes (no Parseval factor: the fields are in real space at z_{n+1})
    if (slot >= 0) {
        s1 = warp_sum_ll(s1); s2 = warp_sum_ll(s2);
        if (lane == 0) {
            long long* hst = P.hfix + ((long long)b * (P.nrec + 1) + slot) * 2;
            fix_add(hst + 0, s1);
            fix_add(hst + 1, s2);
        }
    }
    if constexpr (G >= 2) __syncwarp(); else named_barrier(1 + (warp >> 1), 64);
#pragma unroll
    for (int q = 0; q < R; ++q) v[q] = own[M * q + m];
    if constexpr (MODE == ROW_FINAL) {
        float2* A = (f ? P.A[1] : P.A[0]) + rbase;
#pragma unroll
        for (int q = 0; q < R; ++q) stcg2(A + ((M * q + m + rot) & (NX - 1)), v[q]);
    } else {
        __syncwarp();
        warp_fft<NX, PREC>(v, own, tws, m);
        table_mul<R, M, PREC, false>(v, P.hx[0] + ((size_t)b * 2 + f) * NX + m);
        float2* dst = (f ? P.A[1] : P.A[0]) + rbase;
#pragma unroll
        for (int q = 0; q < R; ++q) stcg2(dst + M * q + m, v[q]);
    }
}
// ------------------------------------------------------------------------------------------------
// Forward transform of SC = 8 adjacent columns by a team of TW = M/4 warps ("tile" layout).  Thread
// (c, t) -- lane = 8 j + c, t = 4 (warp rank in team) + j -- holds, for column c, the elements t + M q,
// q = 0..R-1, in v[q]: the same strided layout in and out as warp_fft, but the M residues of a column sit
// in M different (c, t) threads spread over the team instead of in the M lanes of one warp.  Hence
//   * a load / store of v[q] touches 4 consecutive rows x 64 contiguous bytes: the strip needs no staging;
//   * the twiddle W_N^{t k1} depends on the lane only through j: a 128-bit table read is a 4-address
//     broadcast (one wavefront instead of four);
//   * the one transpose goes through the strip's shared-memory tile with two team barriers.
// col: the strip's tile, one padded line of pitch CP per column (conflict free for both access patterns:
// CP = 2 mod 16, M + 1 odd).
// ------------------------------------------------------------------------------------------------
template <int N, bool PREC>
__device__ __forceinline__ void tile_fft(float2 (&v)[FftCfg<N>::R], float2* __restrict__ colline,
                                         const float4* __restrict__ tws, int t, int bar_id) {
    constexpr int R = FftCfg<N>::R, M = FftCfg<N>::M, Q = R / M, MP = M + 1, TT = Geo<N>::TW * 32;
    const unsigned tws_saddr = (unsigned)__cvta_generic_to_shared(tws + t);
    float2* wr = colline + t;            // value (k1, residue t) goes to slot k1 * MP + t ...
    float2* rd = colline + t * MP;       // ... and thread t collects row k1 = t (+ M i): slots k1 * MP + n2
    if constexpr (Q == 1) {
#pragma unroll 1
        for (int s = 0; s < 2; ++s) {
            fft_reg<R, false, PREC>(v);
            if (s == 0) {
                twiddle_all<N, PREC>(v, tws_saddr, std::make_integer_sequence<int, R - 1>{});
                named_barrier(bar_id, TT);              // every reader of the previous exchange is done
#pragma unroll
                for (int k1 = 0; k1 < R; ++k1) wr[k1 * MP] = v[k1];
                named_barrier(bar_id, TT);
#pragma unroll
                for (int n2 = 0; n2 < M; ++n2) v[n2] = rd[n2];
            }
        }
    } else {
        fft_reg<R, false, PREC>(v);
        twiddle_all<N, PREC>(v, tws_saddr, std::make_integer_sequence<int, R - 1>{});
        named_barrier(bar_id, TT);
#pragma unroll
        for (int k1 = 0; k1 < R; ++k1) wr[k1 * MP] = v[k1];
        named_barrier(bar_id, TT);
#pragma unroll
        for (int i = 0; i < Q; ++i) {
            float2 u[M];
#pragma unroll
            for (int n2 = 0; n2 < M; ++n2) u[n2] = rd[i * M * MP + n2];
            fft_reg<M, false, PREC>(u);
#pragma unroll
            for (int k2 = 0; k2 < M; ++k2) v[i + Q * k2] = u[k2];
        }
    }
}

// ------------------------------------------------------------------------------------------------
// Column pass, one item = a strip of SC = 8 adjacent columns of one field of one member, handled by a team
// of TW warps:  load (4 rows x 64 B per warp instruction) -> F_y -> * hy (includes 1/(nx ny)), conjugated
// -> F_y -> store to the same addresses.
// ------------------------------------------------------------------------------------------------
// NXC: the row length when it is known at compile time (square grids in the persistent kernel: every
// load / store is then one base register plus an immediate), 0 = take P.nx.
// The strip of column item `item` ([NY] rows x 64 B) into a team's staging buffer [NY][SC], asynchronously.
template <int NY, int NXC>
__device__ __forceinline__ void col_prefetch(const Params& P, int item, float2* cstg, int trank, int lane) {
    using GE = Geo<NY>;
    const int nx = NXC ? NXC : P.nx;
    const int spf = nx / GE::SC;
    const int bf = item / spf;
    const float2* A = P.A[bf & 1] + (size_t)(bf >> 1) * NY * nx + (item - bf * spf) * GE::SC;
#pragma unroll
    for (int c = trank * 32 + lane; c < 4 * NY; c += GE::TW * 32)
        cp_async16(cstg + (c >> 2) * GE::SC + 2 * (c & 3), A + (size_t)(c >> 2) * nx + 2 * (c & 3));
}

template <int NY, bool PREC, int NXC, bool TS = false, bool STG = false>
__device__ __forceinline__ void col_item(const Params& P, int item, int hsel, float2* strip,
                                         const float4* __restrict__ tws, int trank, int bar_id, int lane,
                                         const float4* __restrict__ stab = nullptr, float2* cstg = nullptr,
                                         int next = -1) {
    using GE = Geo<NY>;
    constexpr int R = GE::R, M = GE::M, SC = GE::SC, CP = GE::CP;
    static_assert(SC == 8 && GE::TW * 4 == M, "tile layout: 8 columns x 4 residues per warp");
    const int nx = NXC ? NXC : P.nx;
    const int strips_per_field = nx / SC;
    const int bf = item / strips_per_field;                   // b*2 + f
    const int c0 = (item - bf * strips_per_field) * SC;
    const int c = lane & 7, t = trank * 4 + (lane >> 3);
    float2* A = P.A[bf & 1] + (size_t)(bf >> 1) * NY * nx + c0 + c + (size_t)t * nx;
    const size_t gstep = (size_t)M * nx;
    const float4* h = P.hy[hsel] + (size_t)bf * NY;
    float2* colline = strip + c * CP;
    float2 v[R];

    if constexpr (STG) {
        // the strip was copied into the team's staging buffer one item earlier (all threads of the team); the copy of
        // strip `next` (< 0: none) is issued as soon as this one is in registers, so its L2 / HBM latency runs under
        // this strip's transforms
        cp_async_wait_all();
        named_barrier(bar_id, GE::TW * 32);
#pragma unroll
        for (int q = 0; q < R; ++q) v[q] = cstg[(t + M * q) * SC + c];
        named_barrier(bar_id, GE::TW * 32);
        if (next >= 0) col_prefetch<NY, NXC>(P, next, cstg, trank, lane);
    } else {
#pragma unroll
        for (int q = 0; q < R; ++q) v[q] = ldcg2(A + q * gstep);
    }
    if constexpr (!TS) table_prefetch<R, M>(h, t);
    tile_fft<NY, PREC>(v, colline, tws, t, bar_id);
    if constexpr (TS)      // (single simulation: bf is the field; the hy tables follow the two hx tables)
        table_mul_s<R, M, PREC, true>(v, (unsigned)__cvta_generic_to_shared(stab + (2 + bf) * NY + t),
                                      std::make_integer_sequence<int, R>{});
    else
        table_mul<R, M, PREC, true>(v, h + t);
    tile_fft<NY, PREC>(v, colline, tws, t, bar_id);
    if constexpr (NXC == 0) {
        // runtime stride: recompute the addresses instead of keeping R pointers alive across the transforms
        asm volatile("" : "+l"(A));
        float2* a = A;
#pragma unroll
        for (int q = 0; q < R; ++q) { stcg2(a, v[q]); a += gstep; }
    } else {
#pragma unroll
        for (int q = 0; q < R; ++q) stcg2(A + q * gstep, v[q]);
    }
}

template <int NX> __host__ __device__ inline int row_items(int batch, int ny) { return batch * ny / Geo<NX>::HG; }
template <int NY> __host__ __device__ inline int col_items(int batch, int nx) { return batch * 2 * (nx / Geo<NY>::SC); }

// Balanced static schedule: CTA c owns items [U c / grid, U (c+1) / grid); inside the CTA they go round
// robin to the slots (warps, warp pairs or teams), so the four schedulers of an SM differ by <= 1 item.
__device__ __forceinline__ void cta_range(int U, int& lo, int& hi) {
    lo = (int)(((long long)U * blockIdx.x) / gridDim.x);
    hi = (int)(((long long)U * (blockIdx.x + 1)) / gridDim.x);
}

template <int N>
__device__ __forceinline__ const float4* load_twiddles(unsigned char* smem_raw, const float4* __restrict__ tw) {
    float4* tws = reinterpret_cast<float4*>(smem_raw + Geo<N>::WORK_SMEM);
    for (int i = threadIdx.x; i < N; i += blockDim.x) tws[i] = tw[i];
    __syncthreads();
    return tws;
}

template <int NX, int MODE, bool PREC, bool HEAT = false, bool TS = false>
__device__ __forceinline__ void row_pass(const Params& P, const StepCtx& sc, int n, int hsel, float2* smem_cta,
                                         const float4* __restrict__ tws, int warp, int lane,
                                         const float4* __restrict__ stab = nullptr,
                                         unsigned long long* s_pow = nullptr) {
    using GE = Geo<NX>;
    const int lo = sc.row_lo, hi = sc.row_hi;
    const int slot = (GE::G >= 2) ? warp : (warp >> 1);
    if (slot >= P.row_slots) return;
    for (int it = lo + slot; it < hi; it += P.row_slots)
        row_item<NX, MODE, PREC, HEAT, TS>(P, sc, it, n, hsel, smem_cta, tws, warp, lane, stab, s_pow);
}

// single simulation (batch == 1): the CTA's shared power sums of node n + 1 go to the history (after a CTA barrier)
__device__ __forceinline__ void flush_powers(const Params& P, const StepCtx& sc, unsigned long long* s_pow) {
    __syncthreads();
    if (threadIdx.x < 2) {
        const int slot = sc.slot;
        if (slot >= 0) fix_add(P.hfix + (long long)slot * 2 + threadIdx.x, (long long)s_pow[threadIdx.x]);
        s_pow[threadIdx.x] = 0ull;
    }
}

// ------------------------------------------------------------------------------------------------
// Row pass of a z-step for SPARSE launches: a CTA owns at most one item per slot and at most half of its warps
// have one (single small simulations: cfg1-cfg3 give an SM one or two rows).  The transforms stay with the
// warps that own the rows, but the nonlinear step of the CTA's rows is dealt point by point to all 512 threads
// (one or two points per thread instead of R/2 per lane of one warp): the RK4 chain, half of a row item's
// latency, leaves the critical path.  Same per-point arithmetic as row_item<ROW_MID>: bit-identical fields.
//   phase A  owners: load -> F_x -> line to shared memory          | __syncthreads
//   phase B  everyone: T / phase / RK4 on the CTA's points, power sums (fixed point) to the history | __syncthreads
//   phase C  owners: F_x -> * hx -> store
// ------------------------------------------------------------------------------------------------
template <int NX, bool PREC>
__device__ __forceinline__ void row_pass_flat(const Params& P, const StepCtx& sc, int n, int hsel, float2* smem_cta,
                                              const float4* __restrict__ tws, int warp, int lane,
                                              unsigned long long* s_acc) {
    using GE = Geo<NX>;
    constexpr int R = GE::R, M = GE::M, G = GE::G, NP = GE::NP, HG = GE::HG;
    const int lo = sc.row_lo, hi = sc.row_hi;
    const int nitems = hi - lo;                               // <= ROW_SLOTS (the host selects this pass only then)
    const int slot = (G >= 2) ? warp : (warp >> 1);
    const bool has = slot < nitems;
    const int g = lane / M, m = lane % M;
    const int f = (G >= 2) ? g / HG : (warp & 1);
    const int r = (G >= 2) ? g % HG : 0;
    float2* own = smem_cta + (size_t)warp * (G * NP) + g * NP;
    float2 v[R];
    float2* A = nullptr;
    const float4* hx = nullptr;
    // (read last in phase C of the previous step, two device-wide barriers ago)
    if (threadIdx.x < 2 * GE::ROW_SLOTS * HG) s_acc[threadIdx.x] = 0ull;
    if (has) {
        const int item = lo + slot;
        const int b = (item * HG) >> P.ny_log2;
        A = (f ? P.A[1] : P.A[0]) + (size_t)(item * HG + r) * NX;
        hx = P.hx[hsel] + ((size_t)b * 2 + f) * NX;
#pragma unroll
        for (int q = 0; q < R; ++q) v[q] = ldcg2(A + M * q + m);
        table_prefetch<R, M>(hx, m);
        warp_fft<NX, PREC>(v, own, tws, m);
#pragma unroll
        for (int q = 0; q < R; ++q) own[M * q + m] = v[q];     // conj(field), SH rotated by N/2
    }
    __syncthreads();

    // ---- phase B: point idx = ((local item) * HG + row in item) * NX + e; a warp's 32 points share a row
    const int total = nitems * HG * NX;
    const size_t plane = (size_t)P.ny * NX;
    const TNode ta = sc.ta, tb = sc.tb;
    const int rslot = sc.slot;
    for (int idx = threadIdx.x; idx < total; idx += GE::THREADS) {
        const int li = idx / (HG * NX), rr = (idx / NX) % HG, e = idx % NX;
        float2* l1;
        float2* l2;
        if constexpr (G >= 2) {
            l1 = smem_cta + (size_t)li * (G * NP) + rr * NP;             // group (f = 0, rr)
            l2 = smem_cta + (size_t)li * (G * NP) + (HG + rr) * NP;      // group (f = 1, rr)
        } else {
            l1 = smem_cta + (size_t)(2 * li) * NP;
            l2 = smem_cta + (size_t)(2 * li + 1) * NP;
        }
        float2* q1 = l1 + e;
        float2* q2 = l2 + ((e + NX / 2) & (NX - 1));
        const int row = (lo + li) * HG + rr;
        const int b = row >> P.ny_log2, y = row - (b << P.ny_log2);
        const MemberDev& mb = P.mem[b];
        const float k1dz = mb.kap1dz, k2dz = mb.kap2dz;
        PhaseCoef CA, CM, CB;
        if (P.nzt == 0) {
            load_uniform_coefs(P, b, n, CA, CM, CB);
        } else {
            float ca, sa, cm, sm, cb, sb;
            const float* Tb = P.T + (P.T_per_member ? (size_t)b * P.nzt * plane : 0);
            const size_t pidx = (size_t)y * NX + e;
            float* phi = P.phi + (size_t)b * plane + pidx;
            const TPoint tp = t_load(Tb + (size_t)ta.k * plane, Tb + (size_t)tb.k * plane, plane, pidx, ta.two, tb.two, phi);
            const float dTa = dT_lerp(tp.a0, tp.a1, ta.f, ta.two, mb.Tpm_hi, mb.Tpm_lo);
            const float dTb = dT_lerp(tp.b0, tp.b1, tb.f, tb.two, mb.Tpm_hi, mb.Tpm_lo);
            const float dka = fmaf(mb.gT, dTa, mb.dk0), dkb = fmaf(mb.gT, dTb, mb.dk0);
            const float phm = fmaf(0.125f * mb.dz, fmaf(3.0f, dka, dkb), tp.ph);
            const float phb = fmaf(0.5f * mb.dz, dka + dkb, tp.ph);
            __sincosf(tp.ph, &sa, &ca);
            __sincosf(phm, &sm, &cm);
            __sincosf(phb, &sb, &cb);
            __stcg(phi, wrap_2pi(phb));
            CA = phase_coef(ca, sa, k1dz, k2dz);
            CM = phase_coef(cm, sm, k1dz, k2dz);
            CB = phase_coef(cb, sb, k1dz, k2dz);
        }
        float2 a1 = *q1, a2 = *q2;
        a1.y = -a1.y; a2.y = -a2.y;
        rk4_point(a1, a2, CA, CM, CB, mb.g1dz, mb.g2dz);
        *q1 = a1;
        *q2 = a2;
        // a warp's 32 points share a row: fixed-point warp sums into the row's shared accumulators
        if (rslot >= 0) {
            const float fsc = P.pfix[b];
            const long long w1 = warp_sum_ll(to_fix(fmaf(a1.x, a1.x, a1.y * a1.y), fsc));
            const long long w2 = warp_sum_ll(to_fix(fmaf(a2.x, a2.x, a2.y * a2.y), fsc));
            if (lane == 0) {
                atomicAdd(&s_acc[(li * HG + rr) * 2 + 0], (unsigned long long)w1);
                atomicAdd(&s_acc[(li * HG + rr) * 2 + 1], (unsigned long long)w2);
            }
        }
    }
    __syncthreads();

    // ---- phase C: one thread per (row, field) adds the row's sum to the history (2 global atomics per row instead
    // of 2 per warp: they all hit the member's two history words, and the barrier's release waits for them)
    if ((int)threadIdx.x < nitems * HG * 2) {
        const int slot = rslot;
        if (slot >= 0) {
            const int row = lo * HG + (int)threadIdx.x / 2, fld = threadIdx.x & 1;
            const int b = row >> P.ny_log2;
            fix_add(P.hfix + ((long long)b * (P.nrec + 1) + slot) * 2 + fld, (long long)s_acc[threadIdx.x]);
        }
    }
    if (has) {
#pragma unroll
        for (int q = 0; q < R; ++q) v[q] = own[M * q + m];
        __syncwarp();
        warp_fft<NX, PREC>(v, own, tws, m);
        table_mul<R, M, PREC, false>(v, hx + m);
#pragma unroll
        for (int q = 0; q < R; ++q) stcg2(A + M * q + m, v[q]);
    }
}

template <int NX, int MODE, bool PREC>
__device__ __forceinline__ void row_pass_paper(const Params& P, int n, float2* smem_cta,
                                               const float4* __restrict__ tws, int warp, int lane) {
    using GE = Geo<NX>;
    int lo, hi;
    cta_range(row_items<NX>(P.batch, P.ny), lo, hi);
    const int slot = (GE::G >= 2) ? warp : (warp >> 1);
    if (slot >= P.row_slots) return;
    for (int it = lo + slot; it < hi; it += P.row_slots)
        row_item_paper<NX, MODE, PREC>(P, it, n, smem_cta, tws, warp, lane);
}

// CS: the team stages its next strip asynchronously while it transforms this one (cstg_cta: the staging buffers,
// [TEAMS][NY][SC]; see col_item)
template <int NY, bool PREC, int NXC, bool TS = false, bool CS = false>
__device__ __forceinline__ void col_pass(const Params& P, const StepCtx& sc, int hsel, float2* smem_cta,
                                         const float4* __restrict__ tws, int warp, int lane,
                                         const float4* __restrict__ stab = nullptr, float2* cstg_cta = nullptr) {
    using GE = Geo<NY>;
    const int lo = sc.col_lo, hi = sc.col_hi;
    const int team = warp / GE::TW, trank = warp % GE::TW;
    float2* strip = smem_cta + (size_t)team * (GE::SC * GE::CP);
    if (team >= P.col_teams) return;
    if constexpr (CS) {
        float2* cstg = cstg_cta + (size_t)team * (NY * GE::SC);
        int it = lo + team;
        if (it < hi) col_prefetch<NY, NXC>(P, it, cstg, trank, lane);
        for (; it < hi; it += P.col_teams)
            col_item<NY, PREC, NXC, TS, true>(P, it, hsel, strip, tws, trank, 1 + team, lane, stab, cstg,
                                              it + P.col_teams < hi ? it + P.col_teams : -1);
    } else {
        for (int it = lo + team; it < hi; it += P.col_teams)
            col_item<NY, PREC, NXC, TS>(P, it, hsel, strip, tws, trank, 1 + team, lane, stab);
    }
}

// ------------------------------------------------------------------------------------------------
// Per-pass kernels (two launches per z-step; any nx, ny)
// ------------------------------------------------------------------------------------------------
template <int NX, int MODE, bool PREC, bool HEAT = false>
__global__ void __launch_bounds__(Geo<NX>::THREADS, 1) k_row(Params P, int n, int hsel) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    __shared__ unsigned long long s_pow[2];
    __shared__ StepCtx sc;
    if (threadIdx.x < 2) s_pow[threadIdx.x] = 0ull;
    if (threadIdx.x == 32) { ctx_rows<NX>(P, sc); ctx_step(P, sc, n); }
    const float4* tws = load_twiddles<NX>(smem_raw, P.twx);
    unsigned long long* sp = (MODE == ROW_MID && P.batch == 1) ? s_pow : nullptr;
    row_pass<NX, MODE, PREC, HEAT>(P, sc, n, hsel, reinterpret_cast<float2*>(smem_raw), tws, warp, lane, nullptr, sp);
    if (sp) flush_powers(P, sc, sp);
}

template <int NX, int MODE, bool PREC>
__global__ void __launch_bounds__(Geo<NX>::THREADS, 1) k_row_paper(Params P, int n) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const float4* tws = load_twiddles<NX>(smem_raw, P.twx);
    row_pass_paper<NX, MODE, PREC>(P, n, reinterpret_cast<float2*>(smem_raw), tws, warp, lane);
}

template <int NY, bool PREC>
__global__ void __launch_bounds__(Geo<NY>::THREADS, 1) k_col(Params P, int hsel) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    __shared__ StepCtx sc;
    if (threadIdx.x == 32) ctx_cols<NY>(P, sc);
    const float4* tws = load_twiddles<NY>(smem_raw, P.twy);
    col_pass<NY, PREC, 0>(P, sc, hsel, reinterpret_cast<float2*>(smem_raw), tws, warp, lane);
}

// ------------------------------------------------------------------------------------------------
// Persistent whole-run kernel (square grids): the z-loop runs on the device; the only device-wide
// dependency is one barrier between a row pass and a column pass (a 2-D FFT needs every row before any
// column).  Launched cooperatively (all CTAs co-resident), one CTA per SM.
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ unsigned int ld_relaxed_u32(const unsigned int* p) {
    unsigned int v;
    asm volatile("ld.relaxed.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}

__device__ __forceinline__ unsigned int ld_acquire_u32(const unsigned int* p) {
    unsigned int v;
    asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}

// Monotonic-counter barrier: instance k is complete when the counter reaches (k+1) * gridDim.x.
// Arrive = one release reduction (orders the whole CTA's stores, which thread 0 observed through
// bar.sync, before the increment; no value returned, so no round trip), poll = relaxed loads (one L2 round
// trip per poll; the timeout / status checks only every 32nd).  A bounded spin turns a lost CTA into an
// error status instead of a hung GPU.
// sc_next (barrier after a column pass): the polling thread fills in the step entries of z-step n + 1 between its
// arrival and its first poll (every warp of the CTA is past its last read of the old entries: the opening
// bar.sync), the closing bar.sync publishes them.
__device__ __forceinline__ bool grid_barrier(const Params& P, unsigned int& epoch, int n, int which,
                                             StepCtx* sc_next = nullptr) {
    __shared__ int ok;
    __syncthreads();
    if (threadIdx.x == 0) {
        const long long t_cta = clock64();
        epoch += 1;
        const unsigned int target = epoch * gridDim.x;
        asm volatile("red.release.gpu.global.add.u32 [%0], %1;" ::"l"(P.barrier), "r"(1u) : "memory");
        if (sc_next != nullptr && n + 1 < P.n_end) ctx_step(P, *sc_next, n + 1);
        int good = 1;
        if (ld_relaxed_u32(P.barrier) < target) {
            const long long t0 = clock64();
            int spins = 0;
            while (ld_relaxed_u32(P.barrier) < target) {
                // (the timeout / status checks cost an L2 round trip: not in every poll)
                if (((++spins) & 31) == 0) {
                    if (P.spin_limit != 0 && (unsigned long long)(clock64() - t0) > P.spin_limit) {
                        good = 0; atomicExch(P.status, 1); break;
                    }
                    if (*((volatile int*)P.status) != 0) { good = 0; break; }
                }
            }
        }
        // Acquire side (SHG_OPT_ACQUIRE_FENCE).  The last arrival's red.release ordered that CTA's stores before
        // the increment this thread has now observed; the acquire that pairs with it is
        //   2 (default): one more load of the counter, ld.acquire.gpu -- it reads a value >= target, i.e. from the
        //      release sequence of every arrival; the bar.sync below carries the ordering to the rest of the CTA
        //      (causality order is transitive over CTA barriers);
        //   1: a gpu-scope fence.acq_rel after the relaxed poll (same guarantee, a full MEMBAR);
        //   0: nothing -- relies on every mutable global array (fields, phi) being read with ld.global.cg
        //      (SASS LDG.STRONG.GPU: served by L2, never by L1) and on L1 holding only read-only data; outside the
        //      PTX memory model, kept for measurements (bit-identical results in all three modes).
        if (P.acquire_fence == 2) (void)ld_acquire_u32(P.barrier);
        else if (P.acquire_fence == 1) asm volatile("fence.acq_rel.gpu;" ::: "memory");
        ok = good;
        if (P.trace != nullptr && n < P.trace_steps) {
            long long* t = P.trace + (((size_t)n * gridDim.x + blockIdx.x) * 2 + which) * 4;
            unsigned long long gt;
            unsigned int smid;
            asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(gt));
            asm volatile("mov.u32 %0, %%smid;" : "=r"(smid));
            t[0] = t_cta; t[1] = clock64(); t[2] = (long long)gt; t[3] = (long long)smid;
        }
    }
    __syncthreads();
    return ok != 0;
}

// TS (single simulation): hx / hy of both fields live in shared memory for the whole run -- 16 B per point and
// pass that otherwise go through L1 beside the field and temperature streams (ncu, round 1: 35 % L1 hit rate,
// long_scoreboard on the hx load the top stall of the second row transform).
template <int N, bool PREC, bool HEAT = false, bool TS = false>
__global__ void __launch_bounds__(Geo<N>::THREADS, 1) k_persist(Params P) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const float4* tws = load_twiddles<N>(smem_raw, P.twx);   // twx == twy on a square grid
    float2* smem_cta = reinterpret_cast<float2*>(smem_raw);
    float4* stab = reinterpret_cast<float4*>(smem_raw + Geo<N>::CTA_SMEM);
    auto stage_tables = [&](int hs) {
        if constexpr (TS) {
            for (int i = threadIdx.x; i < 2 * N; i += blockDim.x) {
                stab[i] = P.hx[hs][i];
                stab[2 * N + i] = P.hy[hs][i];
            }
            __syncthreads();
        }
    };
    __shared__ unsigned long long s_pow[2];
    __shared__ StepCtx sc;
    if (threadIdx.x < 2) s_pow[threadIdx.x] = 0ull;
    if (threadIdx.x == 32) { ctx_rows<N>(P, sc); ctx_cols<N>(P, sc); ctx_step(P, sc, P.n_begin); }
    unsigned long long* sp = (P.batch == 1) ? s_pow : nullptr;
    __syncthreads();
    stage_tables(P.n_begin == P.nz - 1 ? 1 : 0);
    unsigned int epoch = 0;
#pragma unroll 1
    for (int n = P.n_begin; n < P.n_end; ++n) {
        const int hsel = (n == P.nz - 1) ? 1 : 0;
        if (hsel == 1 && n > P.n_begin) stage_tables(1);     // (every warp passed the barrier's closing bar.sync)
        row_pass<N, ROW_MID, PREC, HEAT, TS>(P, sc, n, hsel, smem_cta, tws, warp, lane, stab, sp);
        if (sp) flush_powers(P, sc, sp);
        if (!grid_barrier(P, epoch, n, 0)) return;
        // (batched runs, N <= 256: a team's next strip is staged under the transforms of this one)
        constexpr bool CS = !TS && !HEAT && Geo<N>::STAGE_COL;
        col_pass<N, PREC, N, TS, CS>(P, sc, hsel, smem_cta, tws, warp, lane, stab,
                                     reinterpret_cast<float2*>(smem_raw + Geo<N>::CTA_SMEM));
        if (!grid_barrier(P, epoch, n, 1, &sc)) return;
    }
}

// Persistent kernel for sparse launches (see row_pass_flat).
template <int N, bool PREC>
__global__ void __launch_bounds__(Geo<N>::THREADS, 1) k_persist_flat(Params P) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    __shared__ unsigned long long s_acc[2 * Geo<N>::ROW_SLOTS * Geo<N>::HG];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    __shared__ StepCtx sc;
    if (threadIdx.x == 32) { ctx_rows<N>(P, sc); ctx_cols<N>(P, sc); ctx_step(P, sc, P.n_begin); }
    const float4* tws = load_twiddles<N>(smem_raw, P.twx);
    float2* smem_cta = reinterpret_cast<float2*>(smem_raw);
    unsigned int epoch = 0;
#pragma unroll 1
    for (int n = P.n_begin; n < P.n_end; ++n) {
        const int hsel = (n == P.nz - 1) ? 1 : 0;
        row_pass_flat<N, PREC>(P, sc, n, hsel, smem_cta, tws, warp, lane, s_acc);
        if (!grid_barrier(P, epoch, n, 0)) return;
        col_pass<N, PREC, N>(P, sc, hsel, smem_cta, tws, warp, lane);
        if (!grid_barrier(P, epoch, n, 1, &sc)) return;
    }
}

// ------------------------------------------------------------------------------------------------
// Persistent kernel for BATCHED runs (batch >= 2), software pipelined over two groups of members.
//
// The members of a batch are independent simulations (the paper sweeps parameters by running one simulation
// per process); only the rows and columns of ONE member depend on each other.  k_persist nevertheless stops the
// whole device twice per z-step: ncu on cfg4 (64 x 128 x 128) shows 27 % of the warp-time parked at barriers -- the
// ~1.9 K clocks of the barrier itself plus the skew between CTAs and between the warps of a CTA, in a pass of only
// 3.5 items per warp.  Here the members are split into two groups with their own device-wide barriers, and every
// barrier is SPLIT-PHASE: a warp arrives when its items of a phase are done and waits only before the first
// access that needs the other CTAs' results -- one whole phase of the other group later:
//
//     wait C0 | rows of group 0 | arrive R0 | wait C1 | rows of group 1 | arrive R1 |
//     wait R0 | cols of group 0 | arrive C0 | wait R1 | cols of group 1 | arrive C1 |      (one z-step)
//
// so a barrier is normally complete when a warp asks, and neither its latency nor the skew stops anything.  There
// is no CTA-wide barrier either: warps, warp pairs and teams run through the phases on their own.
//   arrive: __syncwarp, lane 0 adds 1 to the CTA's shared counter of that barrier (atom.acq_rel.cta); the warp that
//           completes the CTA's count adds 1 to the device counter (red.release.gpu) -- cumulativity makes every
//           warp's stores visible with it.
//   wait:   lane 0 looks at the CTA's cached copy of the device counter (ld.acquire.cta, shared memory), else polls
//           the device counter (relaxed, then one ld.acquire.gpu) and publishes the value (atom.max.release.cta);
//           __syncwarp carries the ordering to the warp.
// Shared memory: one region per team (Geo::TEAM_SMEM) holds the lines of the team's warps in a row phase and the
// team's strip in a column phase.  Items are dealt to the slots round robin CONTINUING from phase to phase, so the
// per-warp work of a z-step stays even although a phase has only a few items per slot.
// Same device code per item as k_persist / k_row / k_col: bit-identical fields and powers.
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ unsigned ld_acquire_cta_shared(unsigned saddr) {
    unsigned v;
    asm volatile("ld.acquire.cta.shared.u32 %0, [%1];" : "=r"(v) : "r"(saddr) : "memory");
    return v;
}

// counters: gcnt[k] device-wide (one arrival per CTA and instance), s_cnt[k] / s_seen[k] per CTA
__device__ __forceinline__ void pipe_arrive(unsigned int* gcnt, unsigned int* s_cnt, int lane) {
    __syncwarp();
    if (lane == 0) {
        unsigned old;
        asm volatile("atom.acq_rel.cta.shared.add.u32 %0, [%1], 1;"
                     : "=r"(old) : "r"((unsigned)__cvta_generic_to_shared(s_cnt)) : "memory");
        // (an instance's arrivals begin only after the previous instance of the same barrier completed)
        if ((old + 1) % (blockDim.x >> 5) == 0)
            asm volatile("red.release.gpu.global.add.u32 [%0], %1;" ::"l"(gcnt), "r"(1u) : "memory");
    }
}

// (a wait that times out raises the status word and lets the warp run on with invalid data: every warp keeps the
// same control flow, so no team or pair barrier is left hanging, and every later wait gives up at its first check)
__device__ __forceinline__ void pipe_wait(const Params& P, const unsigned int* gcnt, unsigned int* s_seen,
                                          unsigned int target, int lane) {
    if (lane == 0) {
        int good = 1;
        const unsigned sa = (unsigned)__cvta_generic_to_shared(s_seen);
        if (ld_acquire_cta_shared(sa) < target) {
            unsigned v = ld_relaxed_u32(gcnt);
            if (v < target) {
                const long long t0 = clock64();
                int spins = 0;
                while ((v = ld_relaxed_u32(gcnt)) < target) {
                    if (((spins++) & 31) == 0) {
                        if (P.spin_limit != 0 && (unsigned long long)(clock64() - t0) > P.spin_limit) {
                            good = 0; atomicExch(P.status, 1); break;
                        }
                        if (*((volatile int*)P.status) != 0) { good = 0; break; }
                    }
                }
            }
            if (good) {
                v = ld_acquire_u32(gcnt);
                asm volatile("atom.release.cta.shared.max.u32 %0, [%1], %2;" : "=r"(v) : "r"(sa), "r"(v) : "memory");
            }
        }
    }
    __syncwarp();                                   // carries the ordering to the other lanes
}

template <int N, bool PREC>
__global__ void __launch_bounds__(Geo<N>::THREADS, 1) k_persist_pipe(Params P) {
    using GE = Geo<N>;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    __shared__ unsigned int s_cnt[4], s_seen[4];
    __shared__ int s_rng[2][4];                              // per group: row lo, row hi, col lo, col hi
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    float4* twsw = reinterpret_cast<float4*>(smem_raw + GE::PIPE_WORK_SMEM);
    for (int i = threadIdx.x; i < N; i += blockDim.x) twsw[i] = P.twx[i];     // twx == twy on a square grid
    if (threadIdx.x < 4) { s_cnt[threadIdx.x] = 0u; s_seen[threadIdx.x] = 0u; }
    const int B0 = (P.batch + 1) / 2;                        // members of group 0; group 1 takes the rest
    if (threadIdx.x < 2) {
        const int g = threadIdx.x;
        const int m0 = g ? B0 : 0, m1 = g ? P.batch : B0;
        const int rpm = P.ny / GE::HG, cpm = 2 * (N / GE::SC);                // row items / strips per member
        int lo, hi;
        cta_range((m1 - m0) * rpm, lo, hi);
        s_rng[g][0] = m0 * rpm + lo; s_rng[g][1] = m0 * rpm + hi;
        cta_range((m1 - m0) * cpm, lo, hi);
        s_rng[g][2] = m0 * cpm + lo; s_rng[g][3] = m0 * cpm + hi;
    }
    __syncthreads();
    const float4* tws = twsw;
    const int team = warp / GE::TW, trank = warp % GE::TW;
    // row items address their lines as base + warp * WARP_SMEM: shift the base so that they fall into the team's region
    float2* row_base = reinterpret_cast<float2*>(smem_raw + (size_t)team * (GE::TEAM_SMEM - GE::TW * GE::WARP_SMEM));
    float2* strip = reinterpret_cast<float2*>(smem_raw + (size_t)team * GE::TEAM_SMEM);
    constexpr bool CSTG = GE::STAGE_COL;
    float2* cstg = reinterpret_cast<float2*>(smem_raw + GE::PIPE_SMEM) + (size_t)team * (N * GE::SC);
    const int rslot = (GE::G >= 2) ? warp : (warp >> 1);
    // named barriers: warp pairs of a row phase use 1 + pair (G == 1), teams of a column phase 9 + team then
    // (pairs and teams of different phases run at the same time)
    const int bar_id = (GE::G == 1 ? 9 : 1) + team;
    static_assert(GE::G == 1 ? GE::TEAMS <= 7 : GE::TEAMS <= 15, "named barrier ids");
    // barriers: 0 = R0, 1 = R1 (rows of group g done), 2 = C0, 3 = C1 (columns of group g done)
    unsigned int* gcnt = P.barrier + 2;
    // where the round-robin deal of each kind of item stands (continues over phases and z-steps)
    int rdeal = 0, cdeal = 0;
    StepCtx sc;
#pragma unroll 1
    for (int n = 0; n < P.nz; ++n) {
        const int hsel = (n == P.nz - 1) ? 1 : 0;
        sc.ta = t_node(n, P.nz, P.nzt);
        sc.tb = t_node(n + 1, P.nz, P.nzt);
        sc.slot = rec_slot(P, n + 1);
#pragma unroll 1
        for (int g = 0; g < 2; ++g) {
            // the columns of this group's previous z-step are complete everywhere (n = 0: the launch boundary)
            if (n > 0) pipe_wait(P, gcnt + 2 + g, &s_seen[2 + g], (unsigned)n * gridDim.x, lane);
            const int lo = s_rng[g][0], hi = s_rng[g][1];
            // item lo + i goes to slot (rdeal + i) % ROW_SLOTS
            for (int i = (rslot - rdeal % GE::ROW_SLOTS + GE::ROW_SLOTS) % GE::ROW_SLOTS; lo + i < hi; i += GE::ROW_SLOTS)
                row_item<N, ROW_MID, PREC>(P, sc, lo + i, n, hsel, row_base, tws, warp, lane);
            rdeal += hi - lo;
            pipe_arrive(gcnt + g, &s_cnt[g], lane);
        }
#pragma unroll 1
        for (int g = 0; g < 2; ++g) {
            pipe_wait(P, gcnt + g, &s_seen[g], (unsigned)(n + 1) * gridDim.x, lane);
            const int lo = s_rng[g][2], hi = s_rng[g][3];
            bool any = false;
            int i = (team - cdeal % GE::TEAMS + GE::TEAMS) % GE::TEAMS;
            if constexpr (CSTG) { if (lo + i < hi) col_prefetch<N, N>(P, lo + i, cstg, trank, lane); }
            for (; lo + i < hi; i += GE::TEAMS) {
                col_item<N, PREC, N, false, CSTG>(P, lo + i, hsel, strip, tws, trank, bar_id, lane, nullptr, cstg,
                                                 lo + i + GE::TEAMS < hi ? lo + i + GE::TEAMS : -1);
                any = true;
            }
            // the team's region turns into line buffers again: every warp of the team is done reading the strip
            if (any) named_barrier(bar_id, GE::TW * 32);
            cdeal += hi - lo;
            pipe_arrive(gcnt + 2 + g, &s_cnt[2 + g], lane);
        }
    }
}

// The paper's ordering (SHG_OPT_SCHEME = 1): the loop body is "second half of step n, first half of step n + 1",
// then the linear step of step n + 1 along y; n = 0 .. nz - 2 (ROW_FIRST / ROW_FINAL take the outer half-steps).
template <int N, bool PREC>
__global__ void __launch_bounds__(Geo<N>::THREADS, 1) k_persist_paper(Params P) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    __shared__ StepCtx sc;
    if (threadIdx.x == 32) ctx_cols<N>(P, sc);
    const float4* tws = load_twiddles<N>(smem_raw, P.twx);
    float2* smem_cta = reinterpret_cast<float2*>(smem_raw);
    unsigned int epoch = 0;
#pragma unroll 1
    for (int n = 0; n < P.nz - 1; ++n) {
        row_pass_paper<N, ROW_MID, PREC>(P, n, smem_cta, tws, warp, lane);
        if (!grid_barrier(P, epoch, n, 0)) return;
        col_pass<N, PREC, N>(P, sc, 0, smem_cta, tws, warp, lane);
        if (!grid_barrier(P, epoch, n, 1)) return;
    }
}

}  // namespace shg
