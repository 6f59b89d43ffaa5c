// shg_cluster.cuh -- the whole propagate of ONE small simulation in one thread-block cluster (nx = ny <= 256).
//
// The large-grid kernels (shg_device.cuh) keep the fields in global memory / L2 and meet at two device-wide
// barriers per z-step; a single 64 x 64 .. 128 x 128 simulation gives an SM one or two rows, so it runs at the
// latency of those barriers and of the L2 round trips (round 1: 6.7 / 8.7 us per z-step).  Here the field state of
// a member (N^2 x 16 B: 64 KB .. 1 MB) lives in the DISTRIBUTED SHARED MEMORY of a cluster of C CTAs for the whole
// run (the step is "dominated by the 2DFT" -- so keep the 2-D transform on chip):
//
//   CTA `rank` owns rows    y  = rank NR .. rank NR + NR - 1   (row pass:    F_x^-1 -> T/phase -> RK4 -> F_x * hx)
//             and columns   kx = rank NR .. rank NR + NR - 1   (column pass: F_y * hy -> F_y^-1),      NR = N / C
//   rowbuf [2][NR][N]   the CTA's rows    in (kx, y) representation, written by the column owners (DSMEM stores)
//   colbuf [2][N][NR]   the CTA's columns in (kx, y) representation, written by the row owners    (DSMEM stores)
//
// One z-step = row pass -> push to the column owners -> cluster barrier -> column pass -> push to the row owners
// -> cluster barrier.  Nothing of the field state touches global memory between the input load and the output
// store; per step only the temperature plane is read (phi and dk(z_n) stay in registers: a thread integrates the
// same points in every step) and two fixed-point power sums per CTA are added to the history.  The barrier is
// split (arrive.release ... wait.acquire) and the field-independent part of the nonlinear step (T -> dk -> phi ->
// three sincos -> coupling coefficients, Eq. 3) is computed in its shadow.
//
// Arithmetic: the same warp_fft / cmul_hl / rk4_point, conjugation trick and N/2-rotated SH row as the other
// kernels, applied to the same values in the same order -- fields and power history are bit-identical to the
// per-pass and persistent kernels (tests/test_gpu_parity.py).  DESIGN.md §5.7.
#pragma once

#include "shg_device.cuh"

namespace shg {

template <int N, int C> struct CGeo {
    using GE = Geo<N>;
    static constexpr int R = GE::R, M = GE::M, G = GE::G, HG = GE::HG, NP = GE::NP;
    static constexpr int NR = N / C;                       // rows (row pass) / columns (column pass) per CTA
    static constexpr int LINES = 2 * NR;                   // lines per pass: both fields
    static constexpr int FW = LINES / G;                   // warps that hold lines
    static constexpr int POINTS = NR * N;                  // grid points whose nonlinear step the CTA takes
    static constexpr int THREADS = POINTS >= 512 ? 512 : POINTS;
    static constexpr int WARPS = THREADS / 32;
    static constexpr int PT = POINTS / THREADS;            // points per thread
    static constexpr int KP = PT <= 2 ? PT : 1;            // points whose coefficients are precomputed in the barrier shadow
    static constexpr int BUF = 2 * NR * N;                 // float2 slots of rowbuf and of colbuf
    static constexpr int SCR = FW * G * NP;                // float2 slots of the transform scratch / real-space lines
    static constexpr int SMEM = (2 * BUF + SCR) * 8 + N * 16 + 4 * N * 16;
    static_assert(G >= 2 && NR % HG == 0 && NR % G == 0 && FW <= WARPS && FW >= 1, "line -> warp mapping");
    static_assert(POINTS % THREADS == 0 && SMEM <= 227 * 1024, "cluster kernel geometry");
};

__device__ __forceinline__ unsigned cluster_ctarank() {
    unsigned r;
    asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(r));
    return r;
}
__device__ __forceinline__ void cluster_arrive() { asm volatile("barrier.cluster.arrive.release.aligned;" ::: "memory"); }
__device__ __forceinline__ void cluster_wait() { asm volatile("barrier.cluster.wait.acquire.aligned;" ::: "memory"); }

// store to the shared memory of CTA `rank` of the cluster at the address that `saddr` has in this CTA
__device__ __forceinline__ void st_dsmem(unsigned saddr, unsigned rank, float2 v) {
    unsigned ra;
    asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(ra) : "r"(saddr), "r"(rank));
    asm volatile("st.shared::cluster.v2.f32 [%0], {%1, %2};" ::"r"(ra), "f"(v.x), "f"(v.y) : "memory");
}

template <int N, int C, bool PREC>
__global__ void __launch_bounds__(CGeo<N, C>::THREADS, 1) k_cluster(Params P) {
    using CG = CGeo<N, C>;
    constexpr int R = CG::R, M = CG::M, G = CG::G, HG = CG::HG, NP = CG::NP, NR = CG::NR, FW = CG::FW;
    constexpr int PT = CG::PT, KP = CG::KP, THREADS = CG::THREADS;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    float2* rowbuf = reinterpret_cast<float2*>(smem_raw);            // [2][NR][N]
    float2* colbuf = rowbuf + CG::BUF;                               // [2][N][NR]
    float2* scr = colbuf + CG::BUF;                                  // [FW][G][NP]
    float4* tws = reinterpret_cast<float4*>(scr + CG::SCR);          // [N] twiddles
    float4* stab = tws + N;                                          // hx f=0, hx f=1, hy f=0, hy f=1: [N] each
    __shared__ unsigned long long s_pow[2];

    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int g = lane / M, m = lane % M;
    const int rank = (int)cluster_ctarank();
    const int b = blockIdx.x / C;                                    // one cluster per member
    const MemberDev& mb = P.mem[b];
    const bool owner = warp < FW;

    // row pass: lane group g of warp w holds field rf of the CTA's row rr (global row ry)
    const int rf = g / HG, rr = warp * HG + g % HG, ry = rank * NR + rr;
    const int rot = rf ? N / 2 : 0;                                  // the SH row lives rotated by N/2 in real space
    float2* own = scr + warp * (G * NP) + g * NP;
    // column pass: lane group g of warp w holds column ccl (global kx = rank NR + ccl) of field cf
    const int cline = warp * G + g, cf = cline / NR, ccl = cline % NR;

    // SHG_OPT_TRACE: 8 SM-clock stamps per z-step and CTA (thread 0): step start, end of phases A, B, C (pushes
    // issued), first barrier passed, column pass done (pushes issued), second barrier passed; [7] = SM id
    long long* trc = nullptr;
    auto stamp = [&](int i) { if (trc) trc[i] = clock64(); };
    for (int i = tid; i < N; i += THREADS) tws[i] = P.twx[i];
    if (tid < 2) s_pow[tid] = 0ull;
    auto stage_tables = [&](int hs) {                                // hs: 0 = full step dz, 1 = half step
        const float4* hx = P.hx[hs] + (size_t)b * 2 * N;
        const float4* hy = P.hy[hs] + (size_t)b * 2 * N;
        for (int i = tid; i < 2 * N; i += THREADS) { stab[i] = hx[i]; stab[2 * N + i] = hy[i]; }
        __syncthreads();
    };
    stage_tables(1);

    const unsigned colbuf_s = (unsigned)__cvta_generic_to_shared(colbuf);
    const unsigned rowbuf_s = (unsigned)__cvta_generic_to_shared(rowbuf);
    // spectrum element kx = M q + m of row (rf, ry) -> colbuf[rf][ry][kx % NR] of CTA kx / NR
    auto push_to_columns = [&](const float2 (&v)[R]) {
#pragma unroll
        for (int q = 0; q < R; ++q) {
            const int kx = M * q + m;
            st_dsmem(colbuf_s + (unsigned)(((rf * N + ry) * NR + kx % NR) * 8), (unsigned)(kx / NR), v[q]);
        }
    };
    // element y = M q + m of column (cf, rank NR + ccl) -> rowbuf[cf][y % NR][kx] of CTA y / NR
    auto push_to_rows = [&](const float2 (&v)[R]) {
#pragma unroll
        for (int q = 0; q < R; ++q) {
            const int y = M * q + m;
            st_dsmem(rowbuf_s + (unsigned)(((cf * NR + y % NR) * N + rank * NR + ccl) * 8), (unsigned)(y / NR), v[q]);
        }
    };
    // F_y -> * hy (includes 1/(nx ny)), conjugated -> F_y on the CTA's columns, result to the row owners
    auto column_pass = [&]() {
        if (owner) {
            float2 v[R];
#pragma unroll
            for (int q = 0; q < R; ++q) v[q] = colbuf[(cf * N + M * q + m) * NR + ccl];
            warp_fft<N, PREC>(v, own, tws, m);
            table_mul_s<R, M, PREC, true>(v, (unsigned)__cvta_generic_to_shared(stab + (2 + cf) * N + m),
                                          std::make_integer_sequence<int, R>{});
            warp_fft<N, PREC>(v, own, tws, m);
            push_to_rows(v);
        }
    };

    // ---- the points whose nonlinear step this thread takes (the same in every z-step): idx = tid + k THREADS
    const size_t plane = (size_t)N * N;
    const float* Tb = (P.nzt != 0) ? P.T + (P.T_per_member ? (size_t)b * P.nzt * plane : 0) : nullptr;
    const float k1dz = mb.kap1dz, k2dz = mb.kap2dz, g1 = mb.g1dz, g2 = mb.g2dz;
    const float fsc = P.pfix[b];
    float phi[PT], dkn[PT], tq0[PT], tq1[PT];                       // phi(z_n), dk(z_n), raw T of the next node
    PhaseCoef CA[KP], CM[KP], CB[KP];
#pragma unroll
    for (int k = 0; k < PT; ++k) { phi[k] = 0.f; dkn[k] = 0.f; tq0[k] = 0.f; tq1[k] = 0.f; }
    auto point_row = [&](int k) {                                    // local row of point k
        const int idx = tid + k * THREADS;
        return (idx / (HG * N)) * HG + (idx / N) % HG;
    };
    // raw temperature of step node `node` at this thread's points (G15: one or two planes)
    auto load_T = [&](int node) {
        const TNode t = t_node(node, P.nz, P.nzt);
#pragma unroll
        for (int k = 0; k < PT; ++k) {
            const int e = (tid + k * THREADS) % N;
            const float* p = Tb + (size_t)t.k * plane + (size_t)(rank * NR + point_row(k)) * N + e;
            tq0[k] = __ldg(p);
            tq1[k] = t.two ? __ldg(p + plane) : 0.f;
        }
    };
    auto dk_of = [&](int node, int k) {
        const TNode t = t_node(node, P.nz, P.nzt);
        return fmaf(mb.gT, dT_lerp(tq0[k], tq1[k], t.f, t.two, mb.Tpm_hi, mb.Tpm_lo), mb.dk0);
    };
    // coupling coefficients of z-step n at point k from phi_n, dk_n, dk_{n+1}; advances phi and dk to node n+1
    auto coefs_of_point = [&](int k, float dkb, PhaseCoef& ca_, PhaseCoef& cm_, PhaseCoef& cb_) {
        const float ph = phi[k], dka = dkn[k];
        const float phm = fmaf(0.125f * mb.dz, fmaf(3.0f, dka, dkb), ph);      // phi_n + dz (3 dk_n + dk_{n+1})/8
        const float phb = fmaf(0.5f * mb.dz, dka + dkb, ph);                   // phi_n + dz (dk_n + dk_{n+1})/2
        float ca, sa, cm, sm, cb, sb;
        __sincosf(ph, &sa, &ca);
        __sincosf(phm, &sm, &cm);
        __sincosf(phb, &sb, &cb);
        phi[k] = wrap_2pi(phb);
        dkn[k] = dkb;
        ca_ = phase_coef(ca, sa, k1dz, k2dz);
        cm_ = phase_coef(cm, sm, k1dz, k2dz);
        cb_ = phase_coef(cb, sb, k1dz, k2dz);
    };
    // what can be done for z-step n before its fields exist (runs in the shadow of a cluster barrier)
    auto prepare_step = [&](int n) {
        if (P.nzt == 0) {
            // uniform temperature: phi(z) = dk z exactly, the same three phases at every point
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
            CA[0] = phase_coef(ca, sa, k1dz, k2dz);
            CM[0] = phase_coef(cm, sm, k1dz, k2dz);
            CB[0] = phase_coef(cb, sb, k1dz, k2dz);
        } else if constexpr (PT <= 2) {
#pragma unroll
            for (int k = 0; k < PT; ++k) coefs_of_point(k, dk_of(n + 1, k), CA[k], CM[k], CB[k]);
        }
    };

    // ---- opening linear half-step along x on the input (order L/2 - N - L/2), pushed to the column owners
    if (owner) {
        float2 v[R];
        const float2* src = rf ? P.Ain[1] : P.Ain[0];
        const size_t rbase = ((size_t)b * N + ry) * N;
        if (src) {
#pragma unroll
            for (int q = 0; q < R; ++q) v[q] = src[rbase + ((M * q + m + rot) & (N - 1))];
        } else {
#pragma unroll
            for (int q = 0; q < R; ++q) v[q] = make_float2(0.f, 0.f);
        }
        warp_fft<N, PREC>(v, own, tws, m);
        table_mul_s<R, M, PREC, false>(v, (unsigned)__cvta_generic_to_shared(stab + rf * N + m),
                                       std::make_integer_sequence<int, R>{});
        push_to_columns(v);
    }
    cluster_arrive();
    if (P.nzt != 0) {                                                // dk at node 0, raw T of node 1
        load_T(0);
#pragma unroll
        for (int k = 0; k < PT; ++k) dkn[k] = dk_of(0, k);
        load_T(1);
    }
    cluster_wait();
    column_pass();                                                   // ... and along y
    cluster_arrive();
    prepare_step(0);
    cluster_wait();
    if (P.nz > 1) stage_tables(0);

#pragma unroll 1
    for (int n = 0; n < P.nz; ++n) {
        const int hsel = (n == P.nz - 1) ? 1 : 0;                    // the last step closes with a half-step
        if (hsel && P.nz > 1) stage_tables(1);
        trc = (P.trace != nullptr && n < P.trace_steps && tid == 0 && (int)blockIdx.x < P.trace_grid)
                  ? P.trace + ((size_t)n * P.trace_grid + blockIdx.x) * 8 : nullptr;
        if (trc) { unsigned smid; asm volatile("mov.u32 %0, %%smid;" : "=r"(smid)); trc[7] = (long long)smid; }
        stamp(0);
        // ---- phase A (line owners): F_x^-1 of the previous linear step (conj trick), line to shared memory
        if (owner) {
            float2 v[R];
#pragma unroll
            for (int q = 0; q < R; ++q) v[q] = rowbuf[(rf * NR + rr) * N + M * q + m];
            warp_fft<N, PREC>(v, own, tws, m);
#pragma unroll
            for (int q = 0; q < R; ++q) own[M * q + m] = v[q];        // conj(field), SH rotated by N/2
        }
        __syncthreads();
        stamp(1);
        // ---- phase B (everyone): one RK4 step of Eq. 2 per point, power sums
        const int slot = rec_slot(P, n + 1);
        long long s1 = 0, s2 = 0;
#pragma unroll
        for (int k = 0; k < PT; ++k) {
            const int idx = tid + k * THREADS;
            const int li = idx / (HG * N), rw = (idx / N) % HG, e = idx % N;
            float2* q1 = scr + li * (G * NP) + rw * NP + e;
            float2* q2 = scr + li * (G * NP) + (HG + rw) * NP + ((e + N / 2) & (N - 1));
            PhaseCoef ca_, cm_, cb_;
            if (P.nzt == 0) { ca_ = CA[0]; cm_ = CM[0]; cb_ = CB[0]; }
            else if constexpr (PT <= 2) { ca_ = CA[k]; cm_ = CM[k]; cb_ = CB[k]; }
            else coefs_of_point(k, dk_of(n + 1, k), ca_, cm_, cb_);
            float2 a1 = *q1, a2 = *q2;
            a1.y = -a1.y; a2.y = -a2.y;
            rk4_point(a1, a2, ca_, cm_, cb_, g1, g2);
            *q1 = a1;
            *q2 = a2;
            if (slot >= 0) {
                s1 += to_fix(fmaf(a1.x, a1.x, a1.y * a1.y), fsc);
                s2 += to_fix(fmaf(a2.x, a2.x, a2.y * a2.y), fsc);
            }
        }
        if (slot >= 0) {
            s1 = warp_sum_ll(s1); s2 = warp_sum_ll(s2);
            if (lane == 0) {
                atomicAdd(&s_pow[0], (unsigned long long)s1);
                atomicAdd(&s_pow[1], (unsigned long long)s2);
            }
        }
        __syncthreads();
        stamp(2);
        if (slot >= 0 && tid < 2) {
            fix_add(P.hfix + ((size_t)b * (P.nrec + 1) + slot) * 2 + tid, (long long)s_pow[tid]);
            s_pow[tid] = 0ull;
        }
        // ---- phase C (line owners): F_x -> * hx -> column owners
        if (owner) {
            float2 v[R];
#pragma unroll
            for (int q = 0; q < R; ++q) v[q] = own[M * q + m];
            __syncwarp();
            warp_fft<N, PREC>(v, own, tws, m);
            table_mul_s<R, M, PREC, false>(v, (unsigned)__cvta_generic_to_shared(stab + rf * N + m),
                                           std::make_integer_sequence<int, R>{});
            push_to_columns(v);
        }
        stamp(3);
        cluster_arrive();
        if (P.nzt != 0 && n + 2 <= P.nz) load_T(n + 2);              // raw T for dk(z_{n+2}), used after the column pass
        cluster_wait();
        stamp(4);
        column_pass();
        stamp(5);
        cluster_arrive();
        if (n + 1 < P.nz) prepare_step(n + 1);
        cluster_wait();
        stamp(6);
    }

    // ---- back to real space along x, output (the SH row un-rotated)
    if (owner) {
        float2 v[R];
#pragma unroll
        for (int q = 0; q < R; ++q) v[q] = rowbuf[(rf * NR + rr) * N + M * q + m];
        warp_fft<N, PREC>(v, own, tws, m);
        float2* dst = (rf ? P.A[1] : P.A[0]) + ((size_t)b * N + ry) * N;
#pragma unroll
        for (int q = 0; q < R; ++q) dst[(M * q + m + rot) & (N - 1)] = make_float2(v[q].x, -v[q].y);
    }
}

}  // namespace shg
