// shg_device.cuh -- device side of libshg: warp-autonomous 1-D FFTs, the fused row pass
// (inverse FFT_x -> temperature/phase -> RK4 -> power -> forward FFT_x -> propagator) and column pass
// (FFT_y -> propagator -> inverse FFT_y), the per-pass kernels and the persistent whole-run kernel.
//
// Decomposition of one line of length N = R * M (R values per thread, M threads per line, G = 32/M lines
// per warp):  n = M n1 + n2 (thread n2 = m holds n1 = 0..R-1),  k = k1 + R k2:
//   X[k1 + R k2] = sum_{n2} W_M^{n2 k2} [ W_N^{n2 k1} sum_{n1} W_R^{n1 k1} x[M n1 + n2] ]
// stage A: radix-R in registers; twiddle W_N^{k1 m}; one transpose through shared memory (XOR-swizzled,
// conflict free); stage B: R/M radix-M FFTs in registers.  Input and output are both in the "strided"
// layout: thread m holds elements m + M q, q = 0..R-1 -- which is also the coalesced global layout.
// A warp never synchronises with another warp inside a pass.
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
    static constexpr int G = 32 / M;                     // lines per warp
    static constexpr int NP = N + (M == 8 ? 8 : 0);      // padded line pitch in shared memory (float2)
    static constexpr int LINE_BYTES = NP * 8;
    static constexpr int WARP_SMEM = 2 * G * LINE_BYTES; // scratch + park
    static constexpr int WARPS = (N >= 512) ? 12 : 16;
    static constexpr int THREADS = WARPS * 32;
    static constexpr int CTA_SMEM = WARPS * WARP_SMEM;
    // column pass: columns per warp unit (staged two at a time when a warp holds a single line)
    static constexpr int CW = (G >= 2) ? G : 2;
};

__device__ __forceinline__ float2 ldcg2(const float2* p) { return __ldcg(p); }
__device__ __forceinline__ void stcg2(float2* p, float2 v) { __stcg(p, v); }

// ------------------------------------------------------------------------------------------------
// One line transform per M-lane group; v in/out in strided layout (thread m holds m + M q).
// scr: this group's shared-memory line (NP float2).  tw: inter-stage twiddles W_N^e, e < N.
// ------------------------------------------------------------------------------------------------
template <int N, bool INV, bool PREC>
__device__ __forceinline__ void warp_fft(float2 (&v)[FftCfg<N>::R], float2* __restrict__ scr,
                                         const float4* __restrict__ tw, int m) {
    constexpr int R = FftCfg<N>::R, M = FftCfg<N>::M, Q = R / M;
    fft_reg<R, INV, PREC>(v);
#pragma unroll
    for (int k1 = 1; k1 < R; ++k1) {
        float4 w = tw[k1 * m];
        v[k1] = cmul_hl<INV, PREC>(v[k1], w);
    }
#pragma unroll
    for (int k1 = 0; k1 < R; ++k1) scr[k1 * M + (m ^ (k1 & (M - 1)))] = v[k1];
    __syncwarp();
#pragma unroll
    for (int i = 0; i < Q; ++i) {
        float2 u[M];
        const int k1 = m + M * i;
#pragma unroll
        for (int n2 = 0; n2 < M; ++n2) u[n2] = scr[k1 * M + (n2 ^ m)];
        fft_reg<M, INV, PREC>(u);
#pragma unroll
        for (int k2 = 0; k2 < M; ++k2) v[i + Q * k2] = u[k2];
    }
    __syncwarp();
}

__device__ __forceinline__ float warp_sum(float x) {
#pragma unroll
    for (int o = 16; o >= 1; o >>= 1) x += __shfl_xor_sync(0xffffffffu, x, o);
    return x;
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

// dz * N(A) of P:72-73 (Eq. 2) / P:138-145 (Eq. 11) for one point.
template <bool TPA>
__device__ __forceinline__ void nl_rhs(float2 a1, float2 a2, const PhaseCoef& pc, float g1, float g2,
                                       float2& d1, float2& d2) {
    float px = fmaf(a2.x, a1.x, a2.y * a1.y);            // A2 conj(A1)
    float py = fmaf(a2.y, a1.x, -a2.x * a1.y);
    float qx = fmaf(a1.x, a1.x, -a1.y * a1.y);           // A1^2
    float qy = 2.0f * a1.x * a1.y;
    d1.x = fmaf(px, pc.u1x, -py * pc.u1y);
    d1.y = fmaf(px, pc.u1y, py * pc.u1x);
    d2.x = fmaf(qx, pc.u2x, -qy * pc.u2y);
    d2.y = fmaf(qx, pc.u2y, qy * pc.u2x);
    if constexpr (TPA) {
        float t1 = -g1 * fmaf(a1.x, a1.x, a1.y * a1.y);
        float t2 = -g2 * fmaf(a2.x, a2.x, a2.y * a2.y);
        d1.x = fmaf(t1, a1.x, d1.x); d1.y = fmaf(t1, a1.y, d1.y);
        d2.x = fmaf(t2, a2.x, d2.x); d2.y = fmaf(t2, a2.y, d2.y);
    }
}

// One classical RK4 step of length dz; the phase is sampled at z_n, z_n + dz/2, z_n + dz (G8).
template <bool TPA>
__device__ __forceinline__ void rk4_point(float2& a1, float2& a2, const PhaseCoef& ca, const PhaseCoef& cm,
                                          const PhaseCoef& cb, float g1, float g2) {
    float2 k1a, k1b, k2a, k2b, k3a, k3b, k4a, k4b;
    nl_rhs<TPA>(a1, a2, ca, g1, g2, k1a, k1b);
    nl_rhs<TPA>(make_float2(fmaf(0.5f, k1a.x, a1.x), fmaf(0.5f, k1a.y, a1.y)),
                make_float2(fmaf(0.5f, k1b.x, a2.x), fmaf(0.5f, k1b.y, a2.y)), cm, g1, g2, k2a, k2b);
    nl_rhs<TPA>(make_float2(fmaf(0.5f, k2a.x, a1.x), fmaf(0.5f, k2a.y, a1.y)),
                make_float2(fmaf(0.5f, k2b.x, a2.x), fmaf(0.5f, k2b.y, a2.y)), cm, g1, g2, k3a, k3b);
    nl_rhs<TPA>(make_float2(a1.x + k3a.x, a1.y + k3a.y), make_float2(a2.x + k3b.x, a2.y + k3b.y), cb, g1, g2,
                k4a, k4b);
    constexpr float S = 1.0f / 6.0f;
    a1.x += S * (k1a.x + 2.0f * (k2a.x + k3a.x) + k4a.x);
    a1.y += S * (k1a.y + 2.0f * (k2a.y + k3a.y) + k4a.y);
    a2.x += S * (k1b.x + 2.0f * (k2b.x + k3b.x) + k4b.x);
    a2.y += S * (k1b.y + 2.0f * (k2b.y + k3b.y) + k4b.y);
}

// Temperature rise T - T_pm at one point of plane pair (k, k+1) with weight f  (G15).
__device__ __forceinline__ float dT_lerp(const float* __restrict__ T0, size_t plane, size_t idx, float f,
                                         bool two, float Thi, float Tlo) {
    float a = (__ldg(T0 + idx) - Thi) - Tlo;
    if (two) {
        float b = (__ldg(T0 + plane + idx) - Thi) - Tlo;
        a = fmaf(f, b - a, a);
    }
    return a;
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

// ------------------------------------------------------------------------------------------------
// Row pass for one warp unit = G consecutive rows of one member, both fields.
//   ROW_FIRST : A_in (real space) -> P_j(0) -> FFT_x -> * hx            -> A
//   ROW_MID   : A -> inverse FFT_x -> [T -> dk -> phi] -> RK4 -> P_j(z_{n+1}) -> FFT_x -> * hx -> A
//   ROW_FINAL : A -> inverse FFT_x -> A (output, real space)
// hsel: 0 = full-step tables, 1 = half-step tables.  n = step index (ROW_MID).
// ------------------------------------------------------------------------------------------------
template <int NX, int MODE, bool PREC>
__device__ __forceinline__ void row_unit(const Params& P, int unit, int n, int hsel, float2* smem_warp,
                                         const float4* __restrict__ twx, int lane) {
    using GE = Geo<NX>;
    constexpr int R = GE::R, M = GE::M, G = GE::G, NP = GE::NP;
    const int g = lane / M, m = lane % M;
    const int rows_per_member = P.ny;
    const int row0 = unit * G;                       // global row index over [batch*ny]
    const int b = row0 / rows_per_member;
    const int y = row0 - b * rows_per_member + g;
    const size_t rbase = ((size_t)b * P.ny + y) * NX;
    float2* scr = smem_warp + g * NP;
    float2* park = smem_warp + (G + g) * NP;
    const MemberDev& mb = P.mem[b];
    float2 v[R];

    if constexpr (MODE == ROW_FIRST) {
        float s[2] = {0.f, 0.f};
#pragma unroll
        for (int f = 0; f < 2; ++f) {
            const float2* src = P.Ain[f];
            if (src) {
#pragma unroll
                for (int q = 0; q < R; ++q) v[q] = src[rbase + M * q + m];
            } else {
#pragma unroll
                for (int q = 0; q < R; ++q) v[q] = make_float2(0.f, 0.f);
            }
#pragma unroll
            for (int q = 0; q < R; ++q) s[f] += fmaf(v[q].x, v[q].x, v[q].y * v[q].y);
            warp_fft<NX, false, PREC>(v, scr, twx, m);
            const float4* h = P.hx[hsel] + ((size_t)b * 2 + f) * NX;
#pragma unroll
            for (int q = 0; q < R; ++q) {
                v[q] = cmul_hl<false, PREC>(v[q], __ldg(h + M * q + m));
                stcg2(P.A[f] + rbase + M * q + m, v[q]);
            }
        }
        float s0 = warp_sum(s[0]), s1 = warp_sum(s[1]);
        if (lane == 0) {
            double* hst = P.hist + (size_t)b * (P.nz + 1) * 2;
            atomicAdd(hst + 0, (double)s0 * mb.pscale_in[0]);
            atomicAdd(hst + 1, (double)s1 * mb.pscale_in[1]);
        }
        return;
    }

    if constexpr (MODE == ROW_FINAL) {
#pragma unroll
        for (int f = 0; f < 2; ++f) {
#pragma unroll
            for (int q = 0; q < R; ++q) v[q] = ldcg2(P.A[f] + rbase + M * q + m);
            warp_fft<NX, true, PREC>(v, scr, twx, m);
#pragma unroll
            for (int q = 0; q < R; ++q) stcg2(P.A[f] + rbase + M * q + m, v[q]);
        }
        return;
    }

    if constexpr (MODE == ROW_MID) {
        // ---- field 1: inverse FFT_x, park in shared memory
#pragma unroll
        for (int q = 0; q < R; ++q) v[q] = ldcg2(P.A[0] + rbase + M * q + m);
        warp_fft<NX, true, PREC>(v, scr, twx, m);
#pragma unroll
        for (int q = 0; q < R; ++q) park[M * q + m] = v[q];
        // ---- field 2: inverse FFT_x, stays in registers
#pragma unroll
        for (int q = 0; q < R; ++q) v[q] = ldcg2(P.A[1] + rbase + M * q + m);
        warp_fft<NX, true, PREC>(v, scr, twx, m);

        // ---- nonlinear step
        const float k1dz = mb.kap1dz, k2dz = mb.kap2dz, g1 = mb.g1dz, g2 = mb.g2dz;
        const bool tpa = (g1 != 0.f) || (g2 != 0.f);
        float s1 = 0.f, s2 = 0.f;
        if (P.nzt == 0) {
            // uniform temperature: phi(z) = dk z exactly; three sampled phases per step, warp-uniform
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
            const PhaseCoef A = phase_coef(ca, sa, k1dz, k2dz), Mi = phase_coef(cm, sm, k1dz, k2dz),
                            B = phase_coef(cb, sb, k1dz, k2dz);
#pragma unroll
            for (int q = 0; q < R; ++q) {
                float2 a1 = park[M * q + m], a2 = v[q];
                if (tpa) rk4_point<true>(a1, a2, A, Mi, B, g1, g2);
                else     rk4_point<false>(a1, a2, A, Mi, B, g1, g2);
                s1 += fmaf(a1.x, a1.x, a1.y * a1.y);
                s2 += fmaf(a2.x, a2.x, a2.y * a2.y);
                park[M * q + m] = a1; v[q] = a2;
            }
        } else {
            const size_t plane = (size_t)P.ny * NX;
            const float* Tb = P.T + (P.T_per_member ? (size_t)b * P.nzt * plane : 0);
            const TNode ta = t_node(n, P.nz, P.nzt), tb = t_node(n + 1, P.nz, P.nzt);
            const float* Ta = Tb + (size_t)ta.k * plane;
            const float* Tn = Tb + (size_t)tb.k * plane;
            const float hdz = 0.5f * mb.dz, e8 = 0.125f * mb.dz;
            float* phi = P.phi + (size_t)b * plane;
            const size_t pbase = (size_t)y * NX;
#pragma unroll
            for (int q = 0; q < R; ++q) {
                const size_t idx = pbase + M * q + m;
                float dTa = dT_lerp(Ta, plane, idx, ta.f, ta.two, mb.Tpm_hi, mb.Tpm_lo);
                float dTb = dT_lerp(Tn, plane, idx, tb.f, tb.two, mb.Tpm_hi, mb.Tpm_lo);
                float dka = fmaf(mb.gT, dTa, mb.dk0), dkb = fmaf(mb.gT, dTb, mb.dk0);
                float ph = __ldcg(phi + idx);
                float phm = fmaf(e8, fmaf(3.0f, dka, dkb), ph);        // phi_n + dz (3 dk_n + dk_{n+1})/8
                float phb = fmaf(hdz, dka + dkb, ph);                  // phi_n + dz (dk_n + dk_{n+1})/2
                float ca, sa, cm, sm, cb, sb;
                __sincosf(ph, &sa, &ca);
                __sincosf(phm, &sm, &cm);
                __sincosf(phb, &sb, &cb);
                __stcg(phi + idx, wrap_2pi(phb));
                const PhaseCoef A = phase_coef(ca, sa, k1dz, k2dz), Mi = phase_coef(cm, sm, k1dz, k2dz),
                                B = phase_coef(cb, sb, k1dz, k2dz);
                float2 a1 = park[M * q + m], a2 = v[q];
                if (tpa) rk4_point<true>(a1, a2, A, Mi, B, g1, g2);
                else     rk4_point<false>(a1, a2, A, Mi, B, g1, g2);
                s1 += fmaf(a1.x, a1.x, a1.y * a1.y);
                s2 += fmaf(a2.x, a2.x, a2.y * a2.y);
                park[M * q + m] = a1; v[q] = a2;
            }
        }
        s1 = warp_sum(s1); s2 = warp_sum(s2);
        if (lane == 0) {
            double* hst = P.hist + ((size_t)b * (P.nz + 1) + (n + 1)) * 2;
            atomicAdd(hst + 0, (double)s1 * mb.pscale_step[0]);
            atomicAdd(hst + 1, (double)s2 * mb.pscale_step[1]);
        }
        // ---- field 2 forward FFT_x, propagator, store
        {
            warp_fft<NX, false, PREC>(v, scr, twx, m);
            const float4* h = P.hx[hsel] + ((size_t)b * 2 + 1) * NX;
#pragma unroll
            for (int q = 0; q < R; ++q)
                stcg2(P.A[1] + rbase + M * q + m, cmul_hl<false, PREC>(v[q], __ldg(h + M * q + m)));
        }
        // ---- field 1
        {
#pragma unroll
            for (int q = 0; q < R; ++q) v[q] = park[M * q + m];
            warp_fft<NX, false, PREC>(v, scr, twx, m);
            const float4* h = P.hx[hsel] + ((size_t)b * 2 + 0) * NX;
#pragma unroll
            for (int q = 0; q < R; ++q)
                stcg2(P.A[0] + rbase + M * q + m, cmul_hl<false, PREC>(v[q], __ldg(h + M * q + m)));
        }
    }
}

// ------------------------------------------------------------------------------------------------
// Column pass for one warp unit = CW adjacent columns of one field of one member:
//   FFT_y -> * hy (includes 1/(nx ny)) -> inverse FFT_y, in place.
// ------------------------------------------------------------------------------------------------
template <int NY, bool PREC>
__device__ __forceinline__ void col_unit(const Params& P, int unit, int hsel, float2* smem_warp,
                                         const float4* __restrict__ twy, int lane) {
    using GE = Geo<NY>;
    constexpr int R = GE::R, M = GE::M, G = GE::G, NP = GE::NP, CW = GE::CW;
    const int nx = P.nx;
    const int units_per_field = nx / CW;
    const int bf = unit / units_per_field;           // b*2 + f
    const int c0 = (unit - bf * units_per_field) * CW;
    const int b = bf >> 1, f = bf & 1;
    float2* A = P.A[f] + (size_t)b * NY * nx;
    const float4* h = P.hy[hsel] + (size_t)bf * NY;
    float2 v[R];

    if constexpr (G >= 2) {
        const int g = lane / M, m = lane % M;
        float2* scr = smem_warp + g * NP;
        float2* col = A + c0 + g;
#pragma unroll
        for (int q = 0; q < R; ++q) v[q] = ldcg2(col + (size_t)(M * q + m) * nx);
        warp_fft<NY, false, PREC>(v, scr, twy, m);
#pragma unroll
        for (int q = 0; q < R; ++q) v[q] = cmul_hl<false, PREC>(v[q], __ldg(h + M * q + m));
        warp_fft<NY, true, PREC>(v, scr, twy, m);
#pragma unroll
        for (int q = 0; q < R; ++q) stcg2(col + (size_t)(M * q + m) * nx, v[q]);
    } else {
        // one line per warp (NY = 1024): stage two adjacent columns (16 B per row) through shared memory
        static_assert(G >= 2 || CW == 2, "staged path handles two columns");
        const int m = lane;
        float2* c_a = smem_warp;             // column c0   [NY]
        float2* c_b = smem_warp + NP;        // column c0+1 [NY]
        const float4* src = reinterpret_cast<const float4*>(A + c0);
        const size_t pitch4 = (size_t)nx / 2;    // row pitch in float4
#pragma unroll
        for (int q0 = 0; q0 < R; q0 += 8) {
            float4 t[8];
#pragma unroll
            for (int j = 0; j < 8; ++j) t[j] = __ldcg(src + (size_t)(M * (q0 + j) + m) * pitch4);
#pragma unroll
            for (int j = 0; j < 8; ++j) {
                c_a[M * (q0 + j) + m] = make_float2(t[j].x, t[j].y);
                c_b[M * (q0 + j) + m] = make_float2(t[j].z, t[j].w);
            }
        }
        __syncwarp();
#pragma unroll 1
        for (int c = 0; c < 2; ++c) {
            float2* cc = c ? c_b : c_a;
#pragma unroll
            for (int q = 0; q < R; ++q) v[q] = cc[M * q + m];
            __syncwarp();
            warp_fft<NY, false, PREC>(v, cc, twy, m);
#pragma unroll
            for (int q = 0; q < R; ++q) v[q] = cmul_hl<false, PREC>(v[q], __ldg(h + M * q + m));
            warp_fft<NY, true, PREC>(v, cc, twy, m);
#pragma unroll
            for (int q = 0; q < R; ++q) cc[M * q + m] = v[q];
        }
        __syncwarp();
        float4* dst = reinterpret_cast<float4*>(A + c0);
#pragma unroll
        for (int q = 0; q < R; ++q) {
            float2 a = c_a[M * q + m], bb = c_b[M * q + m];
            __stcg(dst + (size_t)(M * q + m) * pitch4, make_float4(a.x, a.y, bb.x, bb.y));
        }
        __syncwarp();
    }
}

template <int NX> __host__ __device__ inline int row_units(int batch, int ny) { return batch * ny / Geo<NX>::G; }
template <int NY> __host__ __device__ inline int col_units(int batch, int nx) { return batch * 2 * nx / Geo<NY>::CW; }

// ------------------------------------------------------------------------------------------------
// Per-pass kernels (two launches per z-step; any nx, ny)
// ------------------------------------------------------------------------------------------------
template <int NX, int MODE, bool PREC>
__global__ void __launch_bounds__(Geo<NX>::THREADS, 1) k_row(Params P, int n, int hsel) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    float2* smem_warp = reinterpret_cast<float2*>(smem_raw + (size_t)warp * Geo<NX>::WARP_SMEM);
    const int U = row_units<NX>(P.batch, P.ny);
    for (int u = blockIdx.x + gridDim.x * warp; u < U; u += gridDim.x * Geo<NX>::WARPS)
        row_unit<NX, MODE, PREC>(P, u, n, hsel, smem_warp, P.twx, lane);
}

template <int NY, bool PREC>
__global__ void __launch_bounds__(Geo<NY>::THREADS, 1) k_col(Params P, int hsel) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    float2* smem_warp = reinterpret_cast<float2*>(smem_raw + (size_t)warp * Geo<NY>::WARP_SMEM);
    const int U = col_units<NY>(P.batch, P.nx);
    for (int u = blockIdx.x + gridDim.x * warp; u < U; u += gridDim.x * Geo<NY>::WARPS)
        col_unit<NY, PREC>(P, u, hsel, smem_warp, P.twy, lane);
}

// ------------------------------------------------------------------------------------------------
// Persistent whole-run kernel (square grids): the z-loop runs on the device; the only device-wide
// dependency is one barrier between a row pass and a column pass (a 2-D FFT needs every row before any
// column).  Launched cooperatively (all CTAs co-resident), one CTA per SM.
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ unsigned int ld_acquire_u32(const unsigned int* p) {
    unsigned int v;
    asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}

// Monotonic-counter barrier: instance k is complete when the counter reaches (k+1) * gridDim.x.
// A bounded spin turns a lost CTA into an error status instead of a hung GPU.
__device__ __forceinline__ bool grid_barrier(const Params& P, unsigned int& epoch) {
    __shared__ int ok;
    __syncthreads();
    if (threadIdx.x == 0) {
        epoch += 1;
        const unsigned int target = epoch * gridDim.x;
        __threadfence();
        atomicAdd(P.barrier, 1u);
        int good = 1;
        long long t0 = clock64();
        while (ld_acquire_u32(P.barrier) < target) {
            if (clock64() - t0 > 4000000000LL) { good = 0; atomicExch(P.status, 1); break; }
            if (*((volatile int*)P.status) != 0) { good = 0; break; }
        }
        __threadfence();
        ok = good;
    }
    __syncthreads();
    return ok != 0;
}

template <int N, bool PREC>
__global__ void __launch_bounds__(Geo<N>::THREADS, 1) k_persist(Params P) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    float2* smem_warp = reinterpret_cast<float2*>(smem_raw + (size_t)warp * Geo<N>::WARP_SMEM);
    float4* tw_s = reinterpret_cast<float4*>(smem_raw + Geo<N>::CTA_SMEM);   // [N] twiddles (twx == twy)
    for (int i = threadIdx.x; i < N; i += blockDim.x) tw_s[i] = P.twx[i];
    __syncthreads();
    const int UR = row_units<N>(P.batch, P.ny), UC = col_units<N>(P.batch, P.nx);
    unsigned int epoch = 0;
    for (int n = 0; n < P.nz; ++n) {
        const int hsel = (n == P.nz - 1) ? 1 : 0;
        for (int u = blockIdx.x + gridDim.x * warp; u < UR; u += gridDim.x * Geo<N>::WARPS)
            row_unit<N, ROW_MID, PREC>(P, u, n, hsel, smem_warp, tw_s, lane);
        if (!grid_barrier(P, epoch)) return;
        for (int u = blockIdx.x + gridDim.x * warp; u < UC; u += gridDim.x * Geo<N>::WARPS)
            col_unit<N, PREC>(P, u, hsel, smem_warp, tw_s, lane);
        if (!grid_barrier(P, epoch)) return;
    }
}

}  // namespace shg
