// fft_reg.cuh -- register-resident radix-R complex FFTs (R = 2..32) and the hi+lo constant multiply.
//
// Everything here is compile-time indexed (templates + fold expressions), so the R complex values of a
// thread live in registers and every internal twiddle is an immediate.
//
// Why hi+lo constants: the SSFM applies the SAME transform and propagator thousands of times, so an
// fp32-rounded constant is a FIXED perturbation of the per-step operator and its error grows linearly
// with the step count.  Each reused constant w is held as W = fl32(w), w' = fl32(w - W)
// and the small product v*w' is put in the FMA ADDEND of the large one, so it is added before the large
// product is rounded:  v*w ~= fma(v, W, v*w').  (fl(v*W) + fl(v*w') as two rounded products would discard it.)
#pragma once

#include <cuda_runtime.h>
#include <utility>

namespace shg {

// cos(2 pi e / 32), e = 0..8, to 20 digits.
__host__ __device__ constexpr double cos32_table(int e) {
    constexpr double t[9] = {1.0,
                             0.98078528040323044913,
                             0.92387953251128675613,
                             0.83146961230254523708,
                             0.70710678118654752440,
                             0.55557023301960222474,
                             0.38268343236508977173,
                             0.19509032201612826785,
                             0.0};
    return t[e];
}
// cos / sin of 2 pi e / 32 for e = 0..15
__host__ __device__ constexpr double cos32(int e) { return e <= 8 ? cos32_table(e) : -cos32_table(16 - e); }
__host__ __device__ constexpr double sin32(int e) { return e <= 8 ? cos32_table(8 - e) : cos32_table(e - 8); }

__host__ __device__ constexpr float hi_of(double x) { return (float)x; }
__host__ __device__ constexpr float lo_of(double x) { return (float)(x - (double)(float)x); }

// t * c for a compile-time real constant c = C + c'
template <bool PREC>
__device__ __forceinline__ float mul_const(float t, float C, float c_lo) {
    if constexpr (PREC) return fmaf(t, C, t * c_lo);
    else return t * C;
}

// v * (W + w') for a complex constant; w4 = (W.re, W.im, w'.re, w'.im).  CONJ multiplies by conj(w).
// Operand order matters: the OUTERMOST fma of each component carries the product with W.re, so that for the
// near-unity constants of a small-angle propagator (W.re == 1.0f exactly when the angle is < 2.4e-4) the
// dominant term v * W.re is rounded once, together with everything else.  With v.y * W.re in an inner fma
// the correction below half an ulp of v.y is dropped EVERY time (v.y * 1.0f is exact: no dither), a bias of
// ~theta^2 per multiply that showed up as +7e-9 per z-step of power gain over 10^4 steps.
template <bool CONJ, bool PREC>
__device__ __forceinline__ float2 cmul_hl(float2 v, float Wr, float Wi, float wr, float wi) {
    float2 r;
    if constexpr (!CONJ) {
        if constexpr (PREC) {
            r.x = fmaf(v.x, Wr, fmaf(-v.y, Wi, fmaf(v.x, wr, -v.y * wi)));
            r.y = fmaf(v.y, Wr, fmaf(v.x, Wi, fmaf(v.x, wi, v.y * wr)));
        } else {
            r.x = fmaf(v.x, Wr, -v.y * Wi);
            r.y = fmaf(v.y, Wr, v.x * Wi);
        }
    } else {
        if constexpr (PREC) {
            r.x = fmaf(v.x, Wr, fmaf(v.y, Wi, fmaf(v.x, wr, v.y * wi)));
            r.y = fmaf(v.y, Wr, fmaf(-v.x, Wi, fmaf(v.y, wr, -v.x * wi)));
        } else {
            r.x = fmaf(v.x, Wr, v.y * Wi);
            r.y = fmaf(v.y, Wr, -v.x * Wi);
        }
    }
    return r;
}

template <bool CONJ, bool PREC>
__device__ __forceinline__ float2 cmul_hl(float2 v, float4 w) {
    return cmul_hl<CONJ, PREC>(v, w.x, w.y, w.z, w.w);
}

// d * exp(-/+ 2 pi i E / 32)   (INV: + sign), E = 0..15 compile time
template <int E, bool INV, bool PREC>
__device__ __forceinline__ float2 twmul32(float2 d) {
    if constexpr (E == 0) {
        return d;
    } else if constexpr (E == 8) {           // -i (fwd) / +i (inv)
        return INV ? make_float2(-d.y, d.x) : make_float2(d.y, -d.x);
    } else if constexpr (E == 4) {           // (1 -/+ i)/sqrt2
        constexpr float C = hi_of(cos32(4)), c = lo_of(cos32(4));
        float a = INV ? d.x - d.y : d.x + d.y;
        float b = INV ? d.x + d.y : d.y - d.x;
        return make_float2(mul_const<PREC>(a, C, c), mul_const<PREC>(b, C, c));
    } else if constexpr (E == 12) {          // (-1 -/+ i)/sqrt2
        constexpr float C = hi_of(cos32(4)), c = lo_of(cos32(4));
        float a = INV ? -(d.x + d.y) : d.y - d.x;
        float b = INV ? d.x - d.y : -(d.x + d.y);
        return make_float2(mul_const<PREC>(a, C, c), mul_const<PREC>(b, C, c));
    } else {
        // w = cos - i sin (fwd); conj for inverse
        constexpr float Wr = hi_of(cos32(E)), wr = lo_of(cos32(E));
        constexpr float Wi = hi_of(-sin32(E)), wi = lo_of(-sin32(E));
        return cmul_hl<INV, PREC>(d, Wr, Wi, wr, wi);
    }
}

// ---- radix-2^2 arrangement of the radix-2 butterflies ----------------------------------------------------------
// The plain decimation-in-frequency network (round 1) multiplies by W_{2 SPAN}^k after EVERY stage (32 points: 20 general
// and 14 eighth-root twiddles).  Moving the twiddles of two consecutive stages behind the second one (He &
// Torkelson's radix-2^2: the first stage of a pair keeps only the factor -i on the upper half of its differences,
// the second stage none, then the outputs of the length-4S block are multiplied by W_{4S}^{k j}, j = 0, 2, 1, 3 for its
// four quarters) leaves the butterfly topology and the bit-reversed output order unchanged and needs 16 general + 12
// eighth-root twiddles per 32 points (16 points: 4 + 4 instead of 4 + 6).  The transforms run at the fp32 pipe's
// throughput (measured by a stand-alone issue-rate probe, profiles/r02b_fft_issue_rate.txt), so the saved operations
// are saved time.

// d * W_32^E (fwd; conj for INV) for E = 0..31: E >= 16 is the negative of E - 16 (folded into the constants)
template <int E, bool INV, bool PREC>
__device__ __forceinline__ float2 twmul32x(float2 d) {
    if constexpr (E < 16) {
        return twmul32<E, INV, PREC>(d);
    } else if constexpr ((E - 16) % 4 == 0) {
        const float2 r = twmul32<E - 16, INV, PREC>(d);
        return make_float2(-r.x, -r.y);
    } else {
        constexpr float Wr = hi_of(-cos32(E - 16)), wr = lo_of(-cos32(E - 16));
        constexpr float Wi = hi_of(sin32(E - 16)), wi = lo_of(sin32(E - 16));
        return cmul_hl<INV, PREC>(d, Wr, Wi, wr, wi);
    }
}

// (a, b) -> a + b and (a - b) * W_32^E
template <int R, int I0, int I1, int E, bool INV, bool PREC>
__device__ __forceinline__ void bfly_tw(float2 (&v)[R]) {
    const float2 a = v[I0], b = v[I1];
    v[I0] = __fadd2_rn(a, b);
    if constexpr (E % 16 == 8) v[I1] = twmul32x<E, INV, PREC>(make_float2(a.x - b.x, a.y - b.y));   // (+-i swaps re and im, which a register pair cannot do for free: scalar)
    else v[I1] = twmul32x<E, INV, PREC>(__fadd2_rn(a, make_float2(-b.x, -b.y)));
}
// (a, b) -> (a + b) * W_32^E0 and (a - b) * W_32^E1
template <int R, int I0, int I1, int E0, int E1, bool INV, bool PREC>
__device__ __forceinline__ void bfly_tw2(float2 (&v)[R]) {
    const float2 a = v[I0], b = v[I1];
    v[I0] = twmul32x<E0, INV, PREC>(__fadd2_rn(a, b));
    if constexpr (E1 % 16 == 8) v[I1] = twmul32x<E1, INV, PREC>(make_float2(a.x - b.x, a.y - b.y));
    else v[I1] = twmul32x<E1, INV, PREC>(__fadd2_rn(a, make_float2(-b.x, -b.y)));
}

template <int R, int BASE, int LEN, bool INV, bool PREC, int... K>
__device__ __forceinline__ void r22_stage_a(float2 (&v)[R], std::integer_sequence<int, K...>) {
    constexpr int S = LEN / 4;
    (bfly_tw<R, BASE + K, BASE + K + 2 * S, (K >= S ? 8 : 0), INV, PREC>(v), ...);        // K = 0 .. 2S-1
}
template <int R, int BASE, int LEN, bool INV, bool PREC, int... K>
__device__ __forceinline__ void r22_stage_b(float2 (&v)[R], std::integer_sequence<int, K...>) {
    constexpr int S = LEN / 4, U = 32 / LEN;                                              // W_LEN = W_32^U
    (bfly_tw<R, BASE + K, BASE + K + S, 2 * K * U, INV, PREC>(v), ...);                   // quarters j = 0, 2
    (bfly_tw2<R, BASE + 2 * S + K, BASE + 3 * S + K, K * U, 3 * K * U, INV, PREC>(v), ...);   // quarters j = 1, 3
}

template <int R, int BASE, int LEN, bool INV, bool PREC>
__device__ __forceinline__ void r22(float2 (&v)[R]) {
    if constexpr (LEN == 2) {
        bfly_tw<R, BASE, BASE + 1, 0, INV, PREC>(v);
    } else if constexpr (LEN >= 4) {
        constexpr int S = LEN / 4;
        r22_stage_a<R, BASE, LEN, INV, PREC>(v, std::make_integer_sequence<int, 2 * S>{});
        r22_stage_b<R, BASE, LEN, INV, PREC>(v, std::make_integer_sequence<int, S>{});
        r22<R, BASE, S, INV, PREC>(v);
        r22<R, BASE + S, S, INV, PREC>(v);
        r22<R, BASE + 2 * S, S, INV, PREC>(v);
        r22<R, BASE + 3 * S, S, INV, PREC>(v);
    }
}

__host__ __device__ constexpr int bitrev(int i, int n) {
    int r = 0;
    for (int b = 1; b < n; b <<= 1) { r = (r << 1) | (i & 1); i >>= 1; }
    return r;
}

template <int R, int I>
__device__ __forceinline__ void brev_swap(float2 (&v)[R]) {
    constexpr int j = bitrev(I, R);
    if constexpr (I < j) { float2 t = v[I]; v[I] = v[j]; v[j] = t; }
}

template <int R, int... I>
__device__ __forceinline__ void brev_all(float2 (&v)[R], std::integer_sequence<int, I...>) {
    (brev_swap<R, I>(v), ...);
}

// In-place length-R DFT of v[0..R-1], natural order in and out.
//   forward: V[k] = sum_n v[n] e^{-2 pi i n k / R};  INV: e^{+...}, unnormalised.
template <int R, bool INV, bool PREC>
__device__ __forceinline__ void fft_reg(float2 (&v)[R]) {
    static_assert(R == 2 || R == 4 || R == 8 || R == 16 || R == 32, "radix");
    r22<R, 0, R, INV, PREC>(v);
    brev_all<R>(v, std::make_integer_sequence<int, R>{});
}

}  // namespace shg
