// shg_cluster.cuh -- the whole propagate of ONE small simulation in one thread-block cluster (nx = ny <= 128).
//
// The large-grid kernels (shg_device.cuh) keep the fields in global memory / L2 and meet at two device-wide
// barriers per z-step; a single 64 x 64 .. 128 x 128 simulation gives an SM one or two rows, so it runs at the
// latency of those barriers and of the L2 round trips (round 1: 6.7 / 8.7 us per z-step).  Here the field state of
// a member (N^2 x 16 B: 64 KB / 256 KB) lives in the DISTRIBUTED SHARED MEMORY of a cluster of C CTAs for the whole
// run (the step is "dominated by the 2DFT" -- so keep the 2-D transform on chip):
//
//   CTA `rank` owns rows    y  = rank NR .. rank NR + NR - 1   (row pass:    F_x^-1 -> T/phase -> RK4 -> F_x * hx)
//             and columns   kx = rank NR .. rank NR + NR - 1   (column pass: F_y * hy -> F_y^-1),      NR = N / C
//   rowbuf [C][2][NR][NR]   block s = the CTA's rows    x the columns of CTA s, sent by CTA s after its column pass
//   colbuf [C][2][NR][NR]   block s = the rows of CTA s x the CTA's columns,    sent by CTA s after its row pass
//
// The 2-D transform's transposition is an all-to-all between the CTAs: a pass writes its result destination-major
// into a staging buffer ([C][2][NR][NR]) and one lane per destination issues ONE bulk asynchronous copy
// (cp.async.bulk.shared::cluster, SASS UBLKCP) of the contiguous 2 NR^2 x 8 B block into the destination's buffer;
// the copy engine signals the DESTINATION's mbarrier (complete_tx), and the receiver waits on that mbarrier for
// the bytes of all C senders.  There is no cluster barrier in the z-loop: every buffer reuse is ordered by the
// data flow itself (a CTA can only produce the next pass's blocks after it has received all blocks of this pass,
// which every sender produced after consuming what it had received before -- DESIGN.md 5.7).
//
// Nothing of the field state touches global memory between the input load and the output store; per step only the
// temperature plane is read (phi and dk(z_n) stay in registers: a thread integrates the same points in every
// step) and two fixed-point power sums per CTA are added to the history.  The field-independent part of the
// nonlinear step (T -> dk -> phi -> three sincos -> coupling coefficients, Eq. 3) is computed while the
// blocks are in flight.
//
// Arithmetic: the same warp_fft / cmul_hl / rk4_point, conjugation trick and N/2-rotated SH row as the other
// kernels.  At N = 64 they are applied to the same values in the same order: fields and power history are
// bit-identical to the per-pass and persistent kernels.  At N = 128 the line transform (CFft<128> below) sums in
// another order: fields and history agree with the other kernels to fp32 rounding (rel. L2 < 2e-6), not bit for bit
// (tests/test_gpu_parity.py checks both statements).
#pragma once

#include "shg_device.cuh"

namespace shg {

// ---- the line transform of the cluster kernel ----------------------------------------------------------------
// A line of N points is held by ML lanes with RV values each; register q of lane l holds element ein(q, l) on
// input and element eout(q, l) on output (every consumer addresses by element, so the two need not agree).
//   N = 64 : warp_fft<64> as in the other kernels (8 lanes x 8 values, 4 lines per warp).
//   N = 128: the other kernels' warp_fft<128> gives a lane 16 values; here a pass has only 16 lines per CTA, i.e.
//            4 busy warps that each run a ~560-instruction stream at the latency of a lone warp.  The cluster
//            kernel therefore spreads a line over 16 lanes x 8 values (8 busy warps, streams half as long):
//            128 = 8 x 16 by the four-step scheme, the 16-point transforms across lanes as 8 (registers) x 2
//            (one shuffle).  Same hi+lo constants; not the same summation order as warp_fft<128>, so for N = 128
//            the cluster kernel agrees with the other kernels to rounding, not bit for bit.
template <int N> struct CFft;

template <> struct CFft<64> {
    static constexpr int RV = 8, ML = 8, GL = 4, NPL = Geo<64>::NP, TW = 64;   // TW: float4 entries of the twiddle table
    __device__ static __forceinline__ int ein(int q, int l) { return l + 8 * q; }
    __device__ static __forceinline__ int eout(int q, int l) { return l + 8 * q; }
    __device__ static __forceinline__ int tab_lane(int l) { return l; }        // eout(q, l) = tab_lane(l) + 8 q
    __device__ static __forceinline__ void load_tw(float4* tws, const float4* __restrict__ twx, int tid, int nthreads) {
        for (int i = tid; i < 64; i += nthreads) tws[i] = twx[i];
    }
    template <bool PREC>
    __device__ static __forceinline__ void run(float2 (&v)[8], float2* line, const float4* tws, int l) {
        warp_fft<64, PREC>(v, line, tws, l);
    }
};

template <> struct CFft<128> {
    static constexpr int RV = 8, ML = 16, GL = 2, TP = 18, NPL = 152, TW = 144;  // TP: pitch of the transposition (4 k1 + 2 c: conflict free)
    static_assert(NPL >= 8 * TP && NPL >= 128, "line scratch");
    __device__ static __forceinline__ int ein(int q, int l) { return l + 16 * q; }
    // lane l = 2 k1 + c ends with X[k1 + 8 ka + 64 c], ka = register index
    __device__ static __forceinline__ int eout(int q, int l) { return (l >> 1) + 8 * q + 64 * (l & 1); }
    __device__ static __forceinline__ int tab_lane(int l) { return (l >> 1) + 64 * (l & 1); }
    // tws[k1 * 16 + l] = W_128^{l k1} (k1 < 8, l < 16); tws[128 + c * 8 + ka] = W_16^{c ka}.  twx is the table of
    // warp_fft<128>: twx[a * 8 + b] = W_128^{a b}, a < 16, b < 8.
    __device__ static __forceinline__ void load_tw(float4* tws, const float4* __restrict__ twx, int tid, int nthreads) {
        for (int i = tid; i < 128; i += nthreads) tws[i] = twx[(i & 15) * 8 + (i >> 4)];
        for (int i = tid; i < 16; i += nthreads) tws[128 + i] = (i < 8) ? make_float4(1.f, 0.f, 0.f, 0.f) : twx[64 + (i - 8)];
    }
    // X[k1 + 8 k2] = sum_{n2} W_16^{n2 k2} [ W_128^{n2 k1} sum_{n1} W_8^{n1 k1} x[16 n1 + n2] ],  n2 = lane;
    // the 16-point sums with n2 = 2 j + c, k2 = ka + 8 kb:  sum_c (-1)^{c kb} W_16^{c ka} sum_j W_8^{j ka} z[2 j + c]
    template <bool PREC>
    __device__ static __forceinline__ void run(float2 (&v)[8], float2* line, const float4* tws, int l) {
        fft_reg<8, false, PREC>(v);
#pragma unroll
        for (int k1 = 1; k1 < 8; ++k1) v[k1] = cmul_hl<false, PREC>(v[k1], tws[k1 * 16 + l]);
#pragma unroll
        for (int k1 = 0; k1 < 8; ++k1) line[k1 * TP + l] = v[k1];
        __syncwarp();
        const int k1r = l >> 1, c = l & 1;
#pragma unroll
        for (int j = 0; j < 8; ++j) v[j] = line[k1r * TP + c + 2 * j];
        __syncwarp();
        fft_reg<8, false, PREC>(v);
#pragma unroll
        for (int ka = 1; ka < 8; ++ka) v[ka] = cmul_hl<false, PREC>(v[ka], tws[128 + c * 8 + ka]);
#pragma unroll
        for (int ka = 0; ka < 8; ++ka) {
            const float px = __shfl_xor_sync(0xffffffffu, v[ka].x, 1), py = __shfl_xor_sync(0xffffffffu, v[ka].y, 1);
            v[ka] = c ? make_float2(px - v[ka].x, py - v[ka].y) : make_float2(v[ka].x + px, v[ka].y + py);
        }
    }
};

template <int N, int C> struct CGeo {
    using F = CFft<N>;
    static constexpr int R = F::RV, M = F::ML, G = F::GL, HG = G / 2, NP = F::NPL;
    static constexpr int NR = N / C;                       // rows (row pass) / columns (column pass) per CTA
    static constexpr int LINES = 2 * NR;                   // lines per pass: both fields
    static constexpr int FW = LINES / G;                   // warps that hold lines ("owners")
    static constexpr int POINTS = NR * N;                  // grid points whose nonlinear step the CTA takes
    static constexpr int THREADS = POINTS >= 512 ? 512 : POINTS;
    static constexpr int WARPS = THREADS / 32;
    static constexpr int PT = POINTS / THREADS;            // points per thread
    static constexpr int KP = PT <= 2 ? PT : 1;            // points whose coefficients are precomputed ahead of the fields
    static constexpr int BLK = 2 * NR * NR;                // float2 slots of one (sender, receiver) block
    static constexpr int BUF = C * BLK;                    // float2 slots of rowbuf, colbuf and of each staging buffer
    static constexpr int SCR = FW * G * NP;                // float2 slots of the transform scratch / real-space lines
    static constexpr int SMEM = (4 * BUF + SCR) * 8 + F::TW * 16 + 4 * N * 16;
    static_assert(G >= 2 && NR % HG == 0 && NR % G == 0 && FW < WARPS && FW >= 1 && C <= 32, "line -> warp mapping");
    static_assert(POINTS % THREADS == 0 && (BLK * 8) % 16 == 0 && SMEM <= 227 * 1024, "cluster kernel geometry");
};

__device__ __forceinline__ unsigned cluster_ctarank() {
    unsigned r;
    asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(r));
    return r;
}
__device__ __forceinline__ void cluster_sync_all() {
    asm volatile("barrier.cluster.arrive.release.aligned;" ::: "memory");
    asm volatile("barrier.cluster.wait.acquire.aligned;" ::: "memory");
}
// shared::cluster address of `saddr` (a shared::cta address of this CTA) in CTA `rank`
__device__ __forceinline__ unsigned map_to_rank(unsigned saddr, unsigned rank) {
    unsigned ra;
    asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(ra) : "r"(saddr), "r"(rank));
    return ra;
}
__device__ __forceinline__ void mbar_init(unsigned bar, unsigned count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
// one arrival + `bytes` expected from the copy engine for the current phase
__device__ __forceinline__ void mbar_arm(unsigned bar, unsigned bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned bar, unsigned parity) {
    unsigned done;
    do {
        asm volatile("{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
                     "selp.u32 %0, 1, 0, p;\n\t}" : "=r"(done) : "r"(bar), "r"(parity) : "memory");
    } while (!done);
}
// bulk copy shared::cta -> shared memory of another CTA of the cluster; completes on that CTA's mbarrier
__device__ __forceinline__ void bulk_copy_to_rank(unsigned dst_cluster, unsigned src_cta, unsigned bytes, unsigned bar_cluster) {
    asm volatile("cp.async.bulk.shared::cluster.shared::cta.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(dst_cluster), "r"(src_cta), "r"(bytes), "r"(bar_cluster) : "memory");
}

template <int N, int C, bool PREC>
__global__ void __launch_bounds__(CGeo<N, C>::THREADS, 1) k_cluster(Params P) {
    using CG = CGeo<N, C>;
    using F = CFft<N>;
    constexpr int R = CG::R, M = CG::M, G = CG::G, HG = CG::HG, NP = CG::NP, NR = CG::NR, FW = CG::FW;
    constexpr int PT = CG::PT, KP = CG::KP, THREADS = CG::THREADS, WARPS = CG::WARPS, BLK = CG::BLK;
    constexpr unsigned BUF_BYTES = CG::BUF * 8, BLK_BYTES = BLK * 8;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    float2* rowbuf = reinterpret_cast<float2*>(smem_raw);            // [C][2][NR][NR] received after a column pass
    float2* colbuf = rowbuf + CG::BUF;                               // [C][2][NR][NR] received after a row pass
    float2* xrow = colbuf + CG::BUF;                                 // staging of a row pass's result    (-> colbuf)
    float2* xcol = xrow + CG::BUF;                                   // staging of a column pass's result (-> rowbuf)
    float2* scr = xcol + CG::BUF;                                    // [FW][G][NP]
    float4* tws = reinterpret_cast<float4*>(scr + CG::SCR);          // twiddles of the line transform
    float4* stab = tws + F::TW;                                      // hx f=0, hx f=1, hy f=0, hy f=1: [N] each
    __shared__ __align__(8) unsigned long long s_bar[2];             // mbarriers: [0] colbuf full, [1] rowbuf full
    __shared__ long long s_part[WARPS][2];                           // per-warp power sums of the current step
    __shared__ float s_coef[12];                                     // uniform temperature: the step's coefficients

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

    // SHG_OPT_TRACE: 8 SM-clock stamps per z-step and CTA (thread 0): step start, row blocks received + F_x^-1
    // done, RK4 done, F_x + hx + blocks sent, column blocks received, column pass done + blocks sent, coefficients
    // of the next step done; [7] = SM id
    long long* trc = nullptr;
    auto stamp = [&](int i) { if (trc) trc[i] = clock64(); };
    const unsigned bar_col = (unsigned)__cvta_generic_to_shared(&s_bar[0]);
    const unsigned bar_row = (unsigned)__cvta_generic_to_shared(&s_bar[1]);
    unsigned par_col = 0, par_row = 0;                               // phase parities of the next wait
    if (tid == 0) {
        mbar_init(bar_col, 1);
        mbar_init(bar_row, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        mbar_arm(bar_col, BUF_BYTES);
        mbar_arm(bar_row, BUF_BYTES);
    }

    F::load_tw(tws, P.twx, tid, THREADS);
    auto stage_tables = [&](int hs) {                                // hs: 0 = full step dz, 1 = half step
        const float4* hx = P.hx[hs] + (size_t)b * 2 * N;
        const float4* hy = P.hy[hs] + (size_t)b * 2 * N;
        for (int i = tid; i < 2 * N; i += THREADS) { stab[i] = hx[i]; stab[2 * N + i] = hy[i]; }
        __syncthreads();
    };
    stage_tables(1);
    cluster_sync_all();                                              // every CTA's mbarriers exist before any copy is sent

    // Send the C blocks of a staging buffer: block d goes to slot `rank` of CTA d's receive buffer.  Called by ALL
    // warps once the owner warps have written the staging buffer (their generic-proxy writes fenced towards the async
    // proxy).  A warp issues its bulk copies one lane after the other (~60 clocks each: 16 copies from one warp
    // cost ~1000 clocks, measured by a stand-alone probe: profiles/r02a_summary.md 7), so the C copies are spread over all warps of the CTA.
    auto send_blocks = [&](float2* xbuf, float2* recv, unsigned bar) {
        if (owner) asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
        __syncthreads();
        constexpr int PER_WARP = (C + WARPS - 1) / WARPS;
        const int d = warp * PER_WARP + lane;
        if (lane < PER_WARP && d < C) {
            const unsigned src = (unsigned)__cvta_generic_to_shared(xbuf + d * BLK);
            const unsigned dst = map_to_rank((unsigned)__cvta_generic_to_shared(recv + rank * BLK), (unsigned)d);
            bulk_copy_to_rank(dst, src, BLK_BYTES, map_to_rank(bar, (unsigned)d));
        }
    };
    // wait for the blocks of all C senders, then (thread 0) arm the barrier for its next phase
    auto receive = [&](unsigned bar, unsigned& parity) {
        mbar_wait(bar, parity);
        parity ^= 1u;
        if (tid == 0) mbar_arm(bar, BUF_BYTES);
    };
    // spectrum element kx = M q + m of row (rf, rr): block of column owner kx / NR, [rf][rr][kx % NR]
    auto stage_row_result = [&](const float2 (&v)[R]) {
#pragma unroll
        for (int q = 0; q < R; ++q) {
            const int kx = F::eout(q, m);
            xrow[(((kx / NR) * 2 + rf) * NR + rr) * NR + kx % NR] = v[q];
        }
    };
    // registers in eout order -> registers in ein order (a no-op where the two agree), through the line scratch
    auto relayout = [&](float2 (&v)[R]) {
        if constexpr (N != 64) {
#pragma unroll
            for (int q = 0; q < R; ++q) own[F::eout(q, m)] = v[q];
            __syncwarp();
#pragma unroll
            for (int q = 0; q < R; ++q) v[q] = own[F::ein(q, m)];
            __syncwarp();
        }
    };
    // F_y -> * hy (includes 1/(nx ny)), conjugated -> F_y on the CTA's columns; element y = M q + m of column
    // (cf, ccl) goes to the block of row owner y / NR, [cf][y % NR][ccl]
    auto column_pass = [&]() {
        if (owner) {
            receive(bar_col, par_col);
            stamp(4);
            float2 v[R];
#pragma unroll
            for (int q = 0; q < R; ++q) {
                const int y = F::ein(q, m);
                v[q] = colbuf[(((y / NR) * 2 + cf) * NR + y % NR) * NR + ccl];
            }
            F::template run<PREC>(v, own, tws, m);
            table_mul_s<R, 8, PREC, true>(v, (unsigned)__cvta_generic_to_shared(stab + (2 + cf) * N + F::tab_lane(m)),
                                          std::make_integer_sequence<int, R>{});
            // (the second transform reads its input in ein order: bring the line into that order through the scratch)
            relayout(v);
            F::template run<PREC>(v, own, tws, m);
#pragma unroll
            for (int q = 0; q < R; ++q) {
                const int y = F::eout(q, m);
                xcol[(((y / NR) * 2 + cf) * NR + y % NR) * NR + ccl] = v[q];
            }
        }
        send_blocks(xcol, rowbuf, bar_row);
    };
    // the CTA's row (rf, rr) from the blocks of the column owners: element kx = M q + m
    auto load_row = [&](float2 (&v)[R]) {
#pragma unroll
        for (int q = 0; q < R; ++q) {
            const int kx = F::ein(q, m);
            v[q] = rowbuf[(((kx / NR) * 2 + rf) * NR + rr) * NR + kx % NR];
        }
    };

    // ---- the points whose nonlinear step this thread takes (the same in every z-step): idx = tid + k THREADS
    const size_t plane = (size_t)N * N;
    const float* Tb = (P.nzt != 0) ? P.T + (P.T_per_member ? (size_t)b * P.nzt * plane : 0) : nullptr;
    const float k1dz = mb.kap1dz, k2dz = mb.kap2dz, g1 = mb.g1dz, g2 = mb.g2dz;
    const float fsc = P.pfix[b];
    float phi[PT], dkn[PT], tq0[PT], tq1[PT];                       // phi(z_n), dk(z_n), raw T of the next node
    PhaseCoef CA[KP], CM[KP], CB[KP];
    // PT == 2 (128 x 128): the thread's two points are integrated together in packed fp32x2 (rk4_point2: the same
    // operations in the same order as the scalar code, see shg_device.cuh), their coefficients kept as pairs
    constexpr bool PK2 = (PT == 2);
    PhaseCoef2 CA2{}, CM2{}, CB2{};
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
    // What z-step n needs besides its fields, computed while the blocks of the previous pass are in flight.
    // Uniform temperature: phi(z) = dk z exactly, the same three phases at every point -- ONE lane (of a warp that
    // holds no lines) fetches the step's twelve coefficients from the table and leaves them in shared memory.
    auto prepare_step = [&](int n) {
        if (P.nzt == 0) {
            if (tid == THREADS - 32) {
                PhaseCoef a, c, d;
                load_uniform_coefs(P, b, n, a, c, d);
                s_coef[0] = a.u1x; s_coef[1] = a.u1y; s_coef[2] = a.u2x; s_coef[3] = a.u2y;
                s_coef[4] = c.u1x; s_coef[5] = c.u1y; s_coef[6] = c.u2x; s_coef[7] = c.u2y;
                s_coef[8] = d.u1x; s_coef[9] = d.u1y; s_coef[10] = d.u2x; s_coef[11] = d.u2y;
            }
        } else if constexpr (PK2) {
            // both points at once (coefs_of_point, operation for operation, on pairs)
            const TNode t = t_node(n + 1, P.nz, P.nzt);
            const float2 dkb = __ffma2_rn(bc2(mb.gT), dT_lerp2(make_float2(tq0[0], tq0[PT - 1]), make_float2(tq1[0], tq1[PT - 1]),
                                                                 t.f, t.two, mb.Tpm_hi, mb.Tpm_lo), bc2(mb.dk0));
            const float2 ph = make_float2(phi[0], phi[PT - 1]), dka = make_float2(dkn[0], dkn[PT - 1]);
            const float2 phm = __ffma2_rn(bc2(0.125f * mb.dz), __ffma2_rn(bc2(3.0f), dka, dkb), ph);
            const float2 phb = __ffma2_rn(bc2(0.5f * mb.dz), __fadd2_rn(dka, dkb), ph);
            float2 ca, sa, cm, sm, cb, sb;
            __sincosf(ph.x, &sa.x, &ca.x);   __sincosf(ph.y, &sa.y, &ca.y);
            __sincosf(phm.x, &sm.x, &cm.x);  __sincosf(phm.y, &sm.y, &cm.y);
            __sincosf(phb.x, &sb.x, &cb.x);  __sincosf(phb.y, &sb.y, &cb.y);
            const float2 pw = wrap_2pi2(phb);
            phi[0] = pw.x; phi[PT - 1] = pw.y;
            dkn[0] = dkb.x; dkn[PT - 1] = dkb.y;
            CA2 = phase_coef2(ca, sa, k1dz, k2dz);
            CM2 = phase_coef2(cm, sm, k1dz, k2dz);
            CB2 = phase_coef2(cb, sb, k1dz, k2dz);
        } else if constexpr (PT <= 2) {
#pragma unroll
            for (int k = 0; k < PT; ++k) coefs_of_point(k, dk_of(n + 1, k), CA[k], CM[k], CB[k]);
        }
    };

    // ---- opening linear half-step along x on the input (order L/2 - N - L/2), sent to the column owners
    if (owner) {
        float2 v[R];
        const float2* src = rf ? P.Ain[1] : P.Ain[0];
        const size_t rbase = ((size_t)b * N + ry) * N;
        if (src) {
#pragma unroll
            for (int q = 0; q < R; ++q) v[q] = src[rbase + ((F::ein(q, m) + rot) & (N - 1))];
        } else {
#pragma unroll
            for (int q = 0; q < R; ++q) v[q] = make_float2(0.f, 0.f);
        }
        F::template run<PREC>(v, own, tws, m);
        table_mul_s<R, 8, PREC, false>(v, (unsigned)__cvta_generic_to_shared(stab + rf * N + F::tab_lane(m)),
                                       std::make_integer_sequence<int, R>{});
        stage_row_result(v);
    }
    send_blocks(xrow, colbuf, bar_col);
    if (P.nzt != 0) {                                                // dk at node 0, raw T of node 1
        load_T(0);
#pragma unroll
        for (int k = 0; k < PT; ++k) dkn[k] = dk_of(0, k);
        load_T(1);
    }
    column_pass();                                                   // ... and along y
    prepare_step(0);
    // the half-step tables are replaced by the full-step ones once every owner warp is done with them
    if (P.nz > 1) { __syncthreads(); stage_tables(0); }

#pragma unroll 1
    for (int n = 0; n < P.nz; ++n) {
        const int hsel = (n == P.nz - 1) ? 1 : 0;                    // the last step closes with a half-step
        if (hsel && P.nz > 1) { __syncthreads(); stage_tables(1); }
        trc = (P.trace != nullptr && n < P.trace_steps && tid == 0 && (int)blockIdx.x < P.trace_grid)
                  ? P.trace + ((size_t)n * P.trace_grid + blockIdx.x) * 8 : nullptr;
        if (trc) { unsigned smid; asm volatile("mov.u32 %0, %%smid;" : "=r"(smid)); trc[7] = (long long)smid; }
        stamp(0);
        // ---- phase A (line owners): F_x^-1 of the previous linear step (conj trick), line to shared memory
        if (owner) {
            receive(bar_row, par_row);
            float2 v[R];
            load_row(v);
            F::template run<PREC>(v, own, tws, m);
#pragma unroll
            for (int q = 0; q < R; ++q) own[F::eout(q, m)] = v[q];    // conj(field), SH rotated by N/2
        }
        __syncthreads();
        stamp(1);
        // ---- phase B (everyone): one RK4 step of Eq. 2 per point, power sums
        const int slot = rec_slot(P, n + 1);
        long long s1 = 0, s2 = 0;
        if constexpr (PK2) {
            float2* q1[2];
            float2* q2[2];
#pragma unroll
            for (int k = 0; k < 2; ++k) {
                const int idx = tid + k * THREADS;
                const int li = idx / (HG * N), rw = (idx / N) % HG, e = idx % N;
                q1[k] = scr + li * (G * NP) + rw * NP + e;
                q2[k] = scr + li * (G * NP) + (HG + rw) * NP + ((e + N / 2) & (N - 1));
            }
            if (P.nzt == 0) {
                CA2.u1x = bc2(s_coef[0]); CA2.u1y = bc2(s_coef[1]); CA2.u2x = bc2(s_coef[2]); CA2.u2y = bc2(s_coef[3]);
                CM2.u1x = bc2(s_coef[4]); CM2.u1y = bc2(s_coef[5]); CM2.u2x = bc2(s_coef[6]); CM2.u2y = bc2(s_coef[7]);
                CB2.u1x = bc2(s_coef[8]); CB2.u1y = bc2(s_coef[9]); CB2.u2x = bc2(s_coef[10]); CB2.u2y = bc2(s_coef[11]);
            }
            const float2 u0 = *q1[0], u1 = *q1[1], w0 = *q2[0], w1 = *q2[1];
            float2 a1x = make_float2(u0.x, u1.x), a1y = make_float2(-u0.y, -u1.y);
            float2 a2x = make_float2(w0.x, w1.x), a2y = make_float2(-w0.y, -w1.y);
            rk4_point2(a1x, a1y, a2x, a2y, CA2, CM2, CB2, g1, g2);
            *q1[0] = make_float2(a1x.x, a1y.x); *q1[1] = make_float2(a1x.y, a1y.y);
            *q2[0] = make_float2(a2x.x, a2y.x); *q2[1] = make_float2(a2x.y, a2y.y);
            if (slot >= 0) {
                const float2 i1 = __fmul2_rn(__ffma2_rn(a1x, a1x, __fmul2_rn(a1y, a1y)), bc2(fsc));
                const float2 i2 = __fmul2_rn(__ffma2_rn(a2x, a2x, __fmul2_rn(a2y, a2y)), bc2(fsc));
                s1 = __float2ll_rn(i1.x) + __float2ll_rn(i1.y);
                s2 = __float2ll_rn(i2.x) + __float2ll_rn(i2.y);
            }
        } else {
#pragma unroll
        for (int k = 0; k < PT; ++k) {
            const int idx = tid + k * THREADS;
            const int li = idx / (HG * N), rw = (idx / N) % HG, e = idx % N;
            float2* q1 = scr + li * (G * NP) + rw * NP + e;
            float2* q2 = scr + li * (G * NP) + (HG + rw) * NP + ((e + N / 2) & (N - 1));
            PhaseCoef ca_, cm_, cb_;
            if (P.nzt == 0) {
                ca_.u1x = s_coef[0]; ca_.u1y = s_coef[1]; ca_.u2x = s_coef[2]; ca_.u2y = s_coef[3];
                cm_.u1x = s_coef[4]; cm_.u1y = s_coef[5]; cm_.u2x = s_coef[6]; cm_.u2y = s_coef[7];
                cb_.u1x = s_coef[8]; cb_.u1y = s_coef[9]; cb_.u2x = s_coef[10]; cb_.u2y = s_coef[11];
            }
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
        }
        if (slot >= 0) {
            s1 = warp_sum_ll(s1); s2 = warp_sum_ll(s2);
            if (lane == 0) { s_part[warp][0] = s1; s_part[warp][1] = s2; }
        }
        __syncthreads();
        stamp(2);
        if (slot >= 0 && tid >= THREADS - 2) {                       // (a warp that holds no lines)
            const int fld = tid & 1;
            long long t = 0;
#pragma unroll
            for (int w = 0; w < WARPS; ++w) t += s_part[w][fld];
            fix_add(P.hfix + ((size_t)b * (P.nrec + 1) + slot) * 2 + fld, t);
        }
        // ---- phase C (line owners): F_x -> * hx -> column owners
        if (owner) {
            float2 v[R];
#pragma unroll
            for (int q = 0; q < R; ++q) v[q] = own[F::ein(q, m)];
            __syncwarp();
            F::template run<PREC>(v, own, tws, m);
            table_mul_s<R, 8, PREC, false>(v, (unsigned)__cvta_generic_to_shared(stab + rf * N + F::tab_lane(m)),
                                           std::make_integer_sequence<int, R>{});
            stage_row_result(v);
        }
        send_blocks(xrow, colbuf, bar_col);
        stamp(3);
        if (P.nzt != 0 && n + 2 <= P.nz) load_T(n + 2);              // raw T for dk(z_{n+2}), used after the column pass
        column_pass();
        stamp(5);
        if (n + 1 < P.nz) prepare_step(n + 1);
        stamp(6);
    }

    // ---- back to real space along x, output (the SH row un-rotated)
    if (owner) {
        receive(bar_row, par_row);
        float2 v[R];
        load_row(v);
        F::template run<PREC>(v, own, tws, m);
        float2* dst = (rf ? P.A[1] : P.A[0]) + ((size_t)b * N + ry) * N;
#pragma unroll
        for (int q = 0; q < R; ++q) dst[(F::eout(q, m) + rot) & (N - 1)] = make_float2(v[q].x, -v[q].y);
    }
    // no CTA leaves while a copy into its shared memory, or a signal on its mbarrier, may still be on its way
    cluster_sync_all();
}

}  // namespace shg
