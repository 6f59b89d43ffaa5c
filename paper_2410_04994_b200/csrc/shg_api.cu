// shg_api.cu -- host side of libshg: the C ABI of include/shg.h.  Builds the constant tables in fp64 and
// splits them into fp32 hi+lo pairs, owns the device state, and enqueues the kernels of shg_device.cuh.
// There is no CPU fallback: every entry point that computes needs a CUDA device.
#include "../../include/shg.h"

#include <cmath>
#include <cstdio>
#include <cstring>
#include <new>
#include <string>
#include <vector>

#include "shg_device.cuh"   // uniform_coefs (k_uniform_coefs); no kernel template is instantiated here
#include "shg_launch.h"
#include "shg_params.h"

namespace {

constexpr double PI = 3.14159265358979323846264338327950288;
constexpr double EPS0 = 8.8541878128e-12;   // F/m
constexpr double C0 = 299792458.0;          // m/s

thread_local std::string g_cuda_msg = "no CUDA error recorded";

int cuda_fail(cudaError_t e, const char* what) {
    g_cuda_msg = std::string(what) + ": " + cudaGetErrorString(e);
    return SHG_ECUDA;
}
#define CU(call)                                              \
    do {                                                      \
        cudaError_t e__ = (call);                             \
        if (e__ != cudaSuccess) return cuda_fail(e__, #call); \
    } while (0)

struct Launchers {
    cudaError_t (*row)(const shg::Params&, int, int, int, bool, int, cudaStream_t);
    cudaError_t (*col)(const shg::Params&, int, bool, int, cudaStream_t);
    cudaError_t (*persist)(const shg::Params&, bool, int, cudaStream_t);
    cudaError_t (*cluster)(const shg::Params&, int, bool, int*, cudaStream_t);
    shg::LaunchInfo (*info)();
};

bool launchers_for(int n, Launchers* L) {
    switch (n) {
#define SHG_CASE(N)                                                                                         \
    case N:                                                                                                 \
        *L = Launchers{shg::launch_row_##N, shg::launch_col_##N, shg::launch_persist_##N, shg::launch_cluster_##N, \
                       shg::launch_info_##N};                                                                \
        return true;
        SHG_CASE(64)
        SHG_CASE(128)
        SHG_CASE(256)
        SHG_CASE(512)
        SHG_CASE(1024)
#undef SHG_CASE
        default:
            return false;
    }
}

float4 split4(double re, double im) {
    float hr = (float)re, hi = (float)im;
    return make_float4(hr, hi, (float)(re - (double)hr), (float)(im - (double)hi));
}

__global__ void k_gaussian(float2* A, const shg::GaussDev* gd, int nx, int ny, int batch) {
    size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x;
    size_t np = (size_t)nx * ny;
    if (i >= np * batch) return;
    int b = (int)(i / np);
    size_t r = i - (size_t)b * np;
    int iy = (int)(r / nx), ix = (int)(r - (size_t)iy * nx);
    shg::GaussDev g = gd[b];
    float x = (ix - nx / 2) * g.dx, y = (iy - ny / 2) * g.dy;
    float r2 = x * x + y * y;
    float er = -r2 * g.qr, ei = -r2 * g.qi;
    float mag = expf(er), c, s;
    sincosf(ei, &s, &c);
    A[i] = make_float2(mag * (g.ar * c - g.ai * s), mag * (g.ar * s + g.ai * c));
}

// P_j(0) and the member's fixed-point scale (shg_device.cuh, "power sums").  Grid (chunks, batch): every block sums
// |A_1|^2 and |A_2|^2 over its chunk of the member's input in double, in a fixed order; the last block to finish
// (ticket counter) adds the chunk sums in chunk order -- deterministic -- and writes
//   pfix[b] = 2^e with (S_1 + S_2) 2^e in [2^55, 2^56),   hfix[b][0][j] = rint(S_j 2^e).
__global__ void __launch_bounds__(256) k_input_power(const float2* __restrict__ A1, const float2* __restrict__ A2,
                                                     size_t np, int nrec, double* part, unsigned int* ticket,
                                                     float* pfix, long long* hfix) {
    const int b = blockIdx.y, c = blockIdx.x, CH = gridDim.x;
    const size_t len = np / CH, base = (size_t)b * np + (size_t)c * len;
    double s1 = 0.0, s2 = 0.0;
    for (size_t i = threadIdx.x; i < len; i += blockDim.x) {
        const float2 a = A1[base + i];
        s1 += (double)a.x * a.x + (double)a.y * a.y;
        if (A2) {
            const float2 d = A2[base + i];
            s2 += (double)d.x * d.x + (double)d.y * d.y;
        }
    }
    __shared__ double sh[2][8];
    __shared__ bool last;
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
        part[((size_t)b * CH + c) * 2 + 0] = t1;
        part[((size_t)b * CH + c) * 2 + 1] = t2;
        __threadfence();
        last = (atomicAdd(&ticket[b], 1u) == (unsigned)(CH - 1));
        if (last) {
            __threadfence();
            double S1 = 0.0, S2 = 0.0;
            for (int k = 0; k < CH; ++k) {
                S1 += __ldcg(&part[((size_t)b * CH + k) * 2 + 0]);
                S2 += __ldcg(&part[((size_t)b * CH + k) * 2 + 1]);
            }
            const double S = S1 + S2;
            int e = 0;
            if (S > 0.0 && S < 1e300) {
                e = 55 - ilogb(S);
                e = e > 120 ? 120 : (e < -120 ? -120 : e);
            }
            pfix[b] = ldexpf(1.0f, e);
            hfix[(size_t)b * (nrec + 1) * 2 + 0] = llrint(ldexp(S1, e));
            hfix[(size_t)b * (nrec + 1) * 2 + 1] = llrint(ldexp(S2, e));
            ticket[b] = 0;
        }
    }
}

// nzt == 0: coupling coefficients of every z-step, see shg_device.cuh: uniform_coefs.  One table for all members (the
// quantities that enter are the crystal's and T_uniform, identical in every MemberDev): member 0's scalars are used.
__global__ void k_uniform_coefs(const shg::MemberDev* mem, float4* ucoef, int nz) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= nz) return;
    const int n = i;
    shg::PhaseCoef a, c, d;
    shg::uniform_coefs(mem[0], n, a, c, d);
    ucoef[(size_t)i * 3 + 0] = make_float4(a.u1x, a.u1y, a.u2x, a.u2y);
    ucoef[(size_t)i * 3 + 1] = make_float4(c.u1x, c.u1y, c.u2x, c.u2y);
    ucoef[(size_t)i * 3 + 2] = make_float4(d.u1x, d.u1y, d.u2x, d.u2y);
}

// A new uniform temperature changes one scalar per member, dk_uniform = dk0 + ddk_dT (T_uniform - T_pm) (Eq. 3):
// written on the propagate's stream, so that a sweep over T_uniform needs neither a host copy nor a host wait.
__global__ void k_set_dk_uniform(shg::MemberDev* mem, int batch, double dk) {
    const int b = blockIdx.x * blockDim.x + threadIdx.x;
    if (b < batch) mem[b].dk_uniform = dk;
}

}  // namespace

struct shg_ctx {
    shg_grid g{};
    shg_crystal c{};
    std::vector<shg_beam> beams;
    int device = 0;
    int sm_count = 0;
    bool persistent = true;
    bool precise = true;
    int acquire_fence = 2;
    int tables_smem = 1;
    int cluster_mode = 1;                 // SHG_OPT_CLUSTER: 0 never, 1 auto, 8 / 16 that cluster size whenever possible
    int pipeline = 1;                     // SHG_OPT_PIPELINE
    unsigned long long spin_limit = 4000000000ULL;
    int rec_every = 1, nrec = 0;
    bool undepleted = false;
    int scheme = 0;
    bool tables_dirty = true;
    bool uniform_dirty = false;           // only T_uniform changed since the tables were built (k_set_dk_uniform)

    Launchers Lx{}, Ly{};

    // device state
    float4* d_twx = nullptr;
    float4* d_twy = nullptr;
    float4* d_hx[2] = {nullptr, nullptr};
    float4* d_hy[2] = {nullptr, nullptr};
    shg::MemberDev* d_mem = nullptr;
    shg::GaussDev* d_gauss = nullptr;
    float4* d_ucoef = nullptr;           // nzt == 0: [nz][3] coupling coefficients per z-step, shared by all members
    float* d_phi = nullptr;
    long long* d_hfix = nullptr;         // [batch][nrec+1][2] fixed-point power sums
    float* d_pfix = nullptr;             // [batch] fixed-point scale 2^e of each member
    double* d_inpart = nullptr;          // k_input_power chunk sums [batch][64][2]
    unsigned int* d_ticket = nullptr;    // [batch]
    std::vector<double> pscale_in, pscale_step;   // [batch][2] (eps0 c n_j/2) dx dy, and times exp(-alpha_j dz/2)
    unsigned int* d_barrier = nullptr;   // [0] barrier counter, [1] status word, [2..5] counters of the pipelined kernel
    float* d_T_owned = nullptr;
    float* d_Q = nullptr;              // borrowed heat-source output (shg_set_heat_output)
    int nq = 0;
    int* d_qmap = nullptr;             // [nz] z-step -> plane of Q, or -1
    size_t T_owned_bytes = 0;
    float2* d_stage[2] = {nullptr, nullptr};
    long long* d_trace = nullptr;
    int trace_steps = 0;        // steps recorded per propagate (0 = tracing off)
    int trace_grid = 0;         // CTAs of the last traced launch

    const float* d_T = nullptr;
    double T_uniform = 0.0;
    int T_per_member = 0;
    bool T_set = false;
    // A host temperature array is uploaded in chunks of planes on the library's own copy stream, one event per chunk,
    // so that the persistent kernel can start on the first planes while the rest is still on its way
    // (shg_set_temperature_host / shg_propagate).  up_chunks == 0: nothing pending, d_T is complete.
    cudaStream_t copy_stream = nullptr;
    cudaEvent_t guard_ev = nullptr;
    std::vector<cudaEvent_t> up_ev;
    int up_chunks = 0;                   // chunks of the current upload
    std::vector<int> up_end;             // planes [0, up_end[c]) are on the device when chunk c has arrived
    const float* up_host = nullptr;      // deferred upload: the host array that the next propagate copies, chunk by chunk,
                                         // AFTER its own field uploads (the copy engine serves its queue in order)

    bool timing = false;
    cudaEvent_t ev[2] = {nullptr, nullptr};
    bool ev_recorded = false;

    cudaStream_t last_stream = nullptr;
    int last_batch = 0;
    int last_launches = 0;
    int last_cluster = 0;               // cluster size of the last propagate (0: batched kernels)
    int last_kernel = 0;                // shg_last_kernel
    bool hist_valid = false;
    int last_scheme = 0;
    std::vector<double> hist_host;       // [batch][nrec+1][2], W
    std::vector<long long> hfix_host;
    std::vector<float> pfix_host;
};

namespace {

size_t np_of(const shg_ctx* ctx) { return (size_t)ctx->g.nx * ctx->g.ny; }

// Tables that depend on the crystal, the grid, each member's window and the uniform temperature.
int upload_tables(shg_ctx* ctx) {
    const shg_grid& g = ctx->g;
    const shg_crystal& c = ctx->c;
    const int B = g.batch;
    const double dz = c.L / g.nz;
    const double k[2] = {2.0 * PI * c.n1 / c.lambda1, 2.0 * PI * c.n2 / (0.5 * c.lambda1)};
    const double alpha[2] = {c.alpha1, c.alpha2};
    const double beta[2] = {c.beta1, c.beta2};
    const double nj[2] = {c.n1, c.n2};
    const double tanrho[2] = {std::tan(c.rho1), std::tan(c.rho2)};
    const bool prec = ctx->precise;
    auto mk = [&](double re, double im) {
        float4 w = split4(re, im);
        if (!prec) { w.z = 0.f; w.w = 0.f; }
        return w;
    };

    // inter-stage twiddles W_N^{k1 m} = exp(-2 pi i k1 m / N), N = R M, stored [k1][m] so that the M lanes of a
    // line read consecutive entries
    for (int axis = 0; axis < 2; ++axis) {
        const int n = axis ? g.ny : g.nx;
        const shg::LaunchInfo li = axis ? ctx->Ly.info() : ctx->Lx.info();
        std::vector<float4> tw(n);
        for (int k1 = 0; k1 < li.fft_r; ++k1)
            for (int m = 0; m < li.fft_m; ++m) {
                double a = -2.0 * PI * (double)((long long)k1 * m % n) / (double)n;
                tw[(size_t)k1 * li.fft_m + m] = mk(std::cos(a), std::sin(a));
            }
        CU(cudaMemcpy(axis ? ctx->d_twy : ctx->d_twx, tw.data(), sizeof(float4) * n, cudaMemcpyHostToDevice));
    }

    // separable propagator: hx_j[m] = exp(-i kx_m^2 h/(2 k_j) - alpha_j h/4), same in y, times 1/(nx ny)
    // in the y table (P:346-352 Eq. A.4-A.5; sign per G3).  h = dz (index 0) and dz/2 (index 1).
    for (int hs = 0; hs < 2; ++hs) {
        const double h = hs ? 0.5 * dz : dz;
        for (int axis = 0; axis < 2; ++axis) {
            const int n = axis ? g.ny : g.nx;
            const double scale = axis ? 1.0 / ((double)g.nx * (double)g.ny) : 1.0;
            std::vector<float4> tab((size_t)B * 2 * n);
            for (int b = 0; b < B; ++b) {
                const double len = axis ? ctx->beams[b].ly : ctx->beams[b].lx;
                for (int f = 0; f < 2; ++f)
                    for (int m = 0; m < n; ++m) {
                        const int ms = (m < n / 2) ? m : m - n;
                        const double kk = 2.0 * PI * (double)ms / len;
                        // diffraction; along x also the walk-off term tan(rho) dA/dx of P:387 (G21)
                        const double ang = -kk * kk * h / (2.0 * k[f]) - (axis ? 0.0 : kk * tanrho[f] * h);
                        const double mag = std::exp(-0.25 * alpha[f] * h) * scale;
                        tab[((size_t)b * 2 + f) * n + m] = mk(mag * std::cos(ang), mag * std::sin(ang));
                    }
            }
            CU(cudaMemcpy(axis ? ctx->d_hy[hs] : ctx->d_hx[hs], tab.data(), sizeof(float4) * tab.size(),
                          cudaMemcpyHostToDevice));
        }
    }

    // per-member scalars
    std::vector<shg::MemberDev> mem(B);
    std::vector<shg::GaussDev> gs(B);
    const double kappa1 = 2.0 * PI * c.d_eff / (c.n1 * c.lambda1);
    const double kappa2 = 2.0 * PI * c.d_eff / (c.n2 * c.lambda1);     // P:73 with G2
    for (int b = 0; b < B; ++b) {
        shg::MemberDev& m = mem[b];
        const shg_beam& bm = ctx->beams[b];
        m.kap1dz = ctx->undepleted ? 0.f : (float)(kappa1 * dz);     // undepleted pump
        m.kap2dz = (float)(kappa2 * dz);
        m.g1dz = (float)(0.5 * beta[0] * 0.5 * EPS0 * C0 * nj[0] * dz);
        m.g2dz = (float)(0.5 * beta[1] * 0.5 * EPS0 * C0 * nj[1] * dz);
        m.dz = (float)dz;
        m.dzd = dz;
        m.gT = (float)c.ddk_dT;
        m.Tpm_hi = (float)c.T_pm;
        m.Tpm_lo = (float)(c.T_pm - (double)m.Tpm_hi);
        m.dk0 = (float)c.dk0;
        m.dk_uniform = c.dk0 + c.ddk_dT * (ctx->T_uniform - c.T_pm);
        {   // heat source per |A_j|^2 (Eq. 8 with I_j = c_j |A_j|^2, c_j = eps0 c n_j / 2)
            const double c1 = 0.5 * EPS0 * C0 * nj[0], c2 = 0.5 * EPS0 * C0 * nj[1];
            m.qa1 = (float)(alpha[0] * c1); m.qb1 = (float)(beta[0] * c1 * c1);
            m.qa2 = (float)(alpha[1] * c2); m.qb2 = (float)(beta[1] * c2 * c2);
        }
        const double dxdy = (bm.lx / g.nx) * (bm.ly / g.ny);
        for (int f = 0; f < 2; ++f) {
            ctx->pscale_in[(size_t)b * 2 + f] = 0.5 * EPS0 * C0 * nj[f] * dxdy;
            // Parseval: the sum taken right after the nonlinear step, times exp(-alpha_j dz/2), is the power
            // after the closing half-step
            ctx->pscale_step[(size_t)b * 2 + f] = std::exp(-0.5 * alpha[f] * dz) * ctx->pscale_in[(size_t)b * 2 + f];
        }
        // Eq. 5 at z = 0: tau0 = -focus_z / zR; |A0|^2 = 4P/(eps0 c n1 pi w0^2) (G17)
        shg::GaussDev& gd = gs[b];
        if (bm.w0 > 0.0) {
            const double zR = 0.5 * bm.w0 * bm.w0 * k[0];
            const double tau0 = -bm.focus_z / zR;
            const double A0 = std::sqrt(4.0 * bm.P / (EPS0 * C0 * c.n1 * PI * bm.w0 * bm.w0));
            const double den = 1.0 + tau0 * tau0;
            gd.ar = (float)(A0 / den);
            gd.ai = (float)(-A0 * tau0 / den);
            gd.qr = (float)(1.0 / (bm.w0 * bm.w0 * den));
            gd.qi = (float)(-tau0 / (bm.w0 * bm.w0 * den));
        } else {
            gd.ar = gd.ai = gd.qr = gd.qi = 0.f;
        }
        gd.dx = (float)(bm.lx / g.nx);
        gd.dy = (float)(bm.ly / g.ny);
    }
    CU(cudaMemcpy(ctx->d_mem, mem.data(), sizeof(shg::MemberDev) * B, cudaMemcpyHostToDevice));
    CU(cudaMemcpy(ctx->d_gauss, gs.data(), sizeof(shg::GaussDev) * B, cudaMemcpyHostToDevice));
    if (ctx->d_ucoef) {
        k_uniform_coefs<<<(g.nz + 127) / 128, 128>>>(ctx->d_mem, ctx->d_ucoef, g.nz);
        CU(cudaGetLastError());
        CU(cudaStreamSynchronize(nullptr));
    }
    ctx->tables_dirty = false;
    ctx->uniform_dirty = false;
    return SHG_OK;
}

void free_ctx(shg_ctx* ctx) {
    if (!ctx) return;
    cudaFree(ctx->d_twx);
    cudaFree(ctx->d_twy);
    for (int i = 0; i < 2; ++i) {
        cudaFree(ctx->d_hx[i]);
        cudaFree(ctx->d_hy[i]);
        cudaFree(ctx->d_stage[i]);
    }
    cudaFree(ctx->d_mem);
    cudaFree(ctx->d_gauss);
    cudaFree(ctx->d_ucoef);
    cudaFree(ctx->d_phi);
    cudaFree(ctx->d_hfix);
    cudaFree(ctx->d_pfix);
    cudaFree(ctx->d_inpart);
    cudaFree(ctx->d_ticket);
    cudaFree(ctx->d_barrier);
    cudaFree(ctx->d_T_owned);
    cudaFree(ctx->d_qmap);
    cudaFree(ctx->d_trace);
    for (int i = 0; i < 2; ++i)
        if (ctx->ev[i]) cudaEventDestroy(ctx->ev[i]);
    for (cudaEvent_t e : ctx->up_ev) cudaEventDestroy(e);
    if (ctx->guard_ev) cudaEventDestroy(ctx->guard_ev);
    if (ctx->copy_stream) cudaStreamDestroy(ctx->copy_stream);
    delete ctx;
}

// The persistent kernel needs every CTA co-resident (cooperative launch).  When the device cannot grant that
// (SMs taken by another context, MPS / MIG slices, cooperative launch unsupported) the z-loop falls back to
// two ordinary launches per z-step -- the same device code, bit-identical fields.
bool coop_unavailable(cudaError_t e) {
    if (e == cudaErrorCooperativeLaunchTooLarge || e == cudaErrorLaunchOutOfResources || e == cudaErrorNotSupported) {
        cudaGetLastError();      // clear the sticky-free launch error
        return true;
    }
    return false;
}

bool aligned16(const void* p) { return (reinterpret_cast<uintptr_t>(p) & 15u) == 0; }

}  // namespace

int shg::record_cuda_error(cudaError_t e, const char* what) { return cuda_fail(e, what); }

extern "C" {

const char* shg_strerror(int code) {
    switch (code) {
        case SHG_OK: return "ok";
        case SHG_EINVAL: return "invalid argument (NULL / out of range / unsupported grid size)";
        case SHG_ESTATE: return "call made in the wrong state (temperature not set, or power requested before a propagate)";
        case SHG_ECUDA: return g_cuda_msg.c_str();
        case SHG_ENOMEM: return "allocation failed";
        case SHG_ELIMIT:
            return "size beyond the fixed capacity of an entry point that works in static scratch "
                   "(shg_field_power_static: at most SHG_STATIC_MAX_BATCH = 256 members per call)";
        default: return "unknown error code";
    }
}

int shg_create(const shg_grid* grid, const shg_crystal* crystal, const shg_beam* beams, shg_ctx** out) {
    if (!grid || !crystal || !beams || !out) return SHG_EINVAL;
    *out = nullptr;
    Launchers Lx, Ly;
    if (!launchers_for(grid->nx, &Lx) || !launchers_for(grid->ny, &Ly)) return SHG_EINVAL;
    if (grid->nz < 1 || grid->nzt < 0 || grid->batch < 1 || grid->record_every < 0) return SHG_EINVAL;
    if (crystal->alpha1 < 0 || crystal->alpha2 < 0 || crystal->beta1 < 0 || crystal->beta2 < 0) return SHG_EINVAL;
    if (!(crystal->L > 0) || !(crystal->lambda1 > 0) || !(crystal->n1 > 0) || !(crystal->n2 > 0)) return SHG_EINVAL;
    for (int b = 0; b < grid->batch; ++b)
        if (!(beams[b].lx > 0) || !(beams[b].ly > 0)) return SHG_EINVAL;
    if ((long long)grid->batch * grid->ny > (1LL << 30)) return SHG_EINVAL;

    int dev = 0;
    CU(cudaGetDevice(&dev));
    shg_ctx* ctx = new (std::nothrow) shg_ctx();
    if (!ctx) return SHG_ENOMEM;
    ctx->g = *grid;
    ctx->c = *crystal;
    ctx->beams.assign(beams, beams + grid->batch);
    ctx->Lx = Lx;
    ctx->Ly = Ly;
    ctx->device = dev;
    ctx->T_uniform = crystal->T_pm;
    ctx->T_set = (grid->nzt == 0);
    ctx->rec_every = grid->record_every < 1 ? 1 : (grid->record_every > grid->nz ? grid->nz : grid->record_every);
    ctx->nrec = (grid->nz + ctx->rec_every - 1) / ctx->rec_every;
    ctx->pscale_in.assign((size_t)grid->batch * 2, 0.0);
    ctx->pscale_step.assign((size_t)grid->batch * 2, 0.0);
    cudaError_t e = cudaDeviceGetAttribute(&ctx->sm_count, cudaDevAttrMultiProcessorCount, dev);
    if (e != cudaSuccess) { free_ctx(ctx); return cuda_fail(e, "cudaDeviceGetAttribute"); }

    const int B = grid->batch;
    const size_t np = (size_t)grid->nx * grid->ny;
    bool ok = true;
    auto alloc = [&](void** p, size_t bytes) {
        if (!ok) return;
        cudaError_t e2 = cudaMalloc(p, bytes);
        if (e2 != cudaSuccess) { ok = false; cuda_fail(e2, "cudaMalloc"); }
    };
    alloc((void**)&ctx->d_twx, sizeof(float4) * grid->nx);
    alloc((void**)&ctx->d_twy, sizeof(float4) * grid->ny);
    for (int hs = 0; hs < 2; ++hs) {
        alloc((void**)&ctx->d_hx[hs], sizeof(float4) * (size_t)B * 2 * grid->nx);
        alloc((void**)&ctx->d_hy[hs], sizeof(float4) * (size_t)B * 2 * grid->ny);
    }
    alloc((void**)&ctx->d_mem, sizeof(shg::MemberDev) * B);
    alloc((void**)&ctx->d_gauss, sizeof(shg::GaussDev) * B);
    if (grid->nzt > 0) alloc((void**)&ctx->d_phi, sizeof(float) * (size_t)B * np);
    else alloc((void**)&ctx->d_ucoef, sizeof(float4) * (size_t)grid->nz * 3);
    alloc((void**)&ctx->d_hfix, sizeof(long long) * (size_t)B * (ctx->nrec + 1) * 2);
    alloc((void**)&ctx->d_pfix, sizeof(float) * B);
    alloc((void**)&ctx->d_inpart, sizeof(double) * (size_t)B * 64 * 2);
    alloc((void**)&ctx->d_ticket, sizeof(unsigned int) * B);
    alloc((void**)&ctx->d_barrier, 8 * sizeof(unsigned int));
    if (!ok) { free_ctx(ctx); return SHG_ECUDA; }
    e = cudaMemset(ctx->d_ticket, 0, sizeof(unsigned int) * B);
    if (e != cudaSuccess) { free_ctx(ctx); return cuda_fail(e, "cudaMemset"); }
    // the status word [1] is cleared here and by the call that reports it, never by a propagate (it is sticky)
    e = cudaMemset(ctx->d_barrier, 0, 8 * sizeof(unsigned int));
    if (e != cudaSuccess) { free_ctx(ctx); return cuda_fail(e, "cudaMemset"); }
    ctx->hist_host.assign((size_t)B * (ctx->nrec + 1) * 2, 0.0);
    ctx->hfix_host.assign((size_t)B * (ctx->nrec + 1) * 2, 0);
    ctx->pfix_host.assign((size_t)B, 1.0f);
    int rc = upload_tables(ctx);
    if (rc != SHG_OK) { free_ctx(ctx); return rc; }
    *out = ctx;
    return SHG_OK;
}

void shg_destroy(shg_ctx* ctx) { free_ctx(ctx); }

int shg_set_option(shg_ctx* ctx, int option, int value) {
    if (!ctx) return SHG_EINVAL;
    switch (option) {
        case SHG_OPT_PERSISTENT: ctx->persistent = (value != 0); return SHG_OK;
        case SHG_OPT_ACQUIRE_FENCE:
            // 0 (no acquire at all) is outside the PTX memory model: not in the product build; -DSHG_ALLOW_UNFENCED
            // brings it back for a measurement
#ifdef SHG_ALLOW_UNFENCED
            if (value < 0 || value > 2) return SHG_EINVAL;
#else
            if (value < 1 || value > 2) return SHG_EINVAL;
#endif
            ctx->acquire_fence = value;
            return SHG_OK;
        case SHG_OPT_SPIN_LIMIT:
            if (value < 0) return SHG_EINVAL;
            ctx->spin_limit = (unsigned long long)value * 1000000ULL;
            return SHG_OK;
        case SHG_OPT_TABLES_SMEM: ctx->tables_smem = (value != 0); return SHG_OK;
        case SHG_OPT_CLUSTER:
            if (value != 0 && value != 1 && value != 8 && value != 16) return SHG_EINVAL;
            ctx->cluster_mode = value;
            return SHG_OK;
        case SHG_OPT_PIPELINE:
            if (value < 0 || value > 2) return SHG_EINVAL;
            ctx->pipeline = value;
            return SHG_OK;
        case SHG_OPT_SCHEME:
            if (value != 0 && value != 1) return SHG_EINVAL;
            ctx->scheme = value;
            return SHG_OK;
        case SHG_OPT_UNDEPLETED:
            if (ctx->undepleted != (value != 0)) { ctx->undepleted = (value != 0); ctx->tables_dirty = true; }
            return SHG_OK;
        case SHG_OPT_PRECISE:
            if (ctx->precise != (value != 0)) { ctx->precise = (value != 0); ctx->tables_dirty = true; }
            return SHG_OK;
        case SHG_OPT_TRACE: {
            if (value < 0 || value > 4096) return SHG_EINVAL;
            if (value != ctx->trace_steps) {
                CU(cudaStreamSynchronize(ctx->last_stream));
                cudaFree(ctx->d_trace);
                ctx->d_trace = nullptr;
                ctx->trace_steps = 0;
                if (value > 0) {
                    const size_t bytes = sizeof(long long) * (size_t)value * ctx->sm_count * 8;
                    CU(cudaMalloc((void**)&ctx->d_trace, bytes));
                    CU(cudaMemset(ctx->d_trace, 0, bytes));
                    ctx->trace_steps = value;
                }
            }
            return SHG_OK;
        }
        default: return SHG_EINVAL;
    }
}

int shg_set_temperature(shg_ctx* ctx, const float* T_device, double T_uniform, int per_member) {
    if (!ctx) return SHG_EINVAL;
    if (ctx->g.nzt > 0 && (!T_device || !aligned16(T_device))) return SHG_EINVAL;
    ctx->d_T = (ctx->g.nzt > 0) ? T_device : nullptr;
    ctx->T_per_member = per_member ? 1 : 0;
    if (ctx->T_uniform != T_uniform) { ctx->T_uniform = T_uniform; ctx->uniform_dirty = true; }
    ctx->T_set = true;
    if (T_device != ctx->d_T_owned) { ctx->up_chunks = 0; ctx->up_host = nullptr; }
    return SHG_OK;
}

int shg_set_temperature_host(shg_ctx* ctx, const float* T_host, double T_uniform, int per_member,
                             void* cuda_stream) {
    if (!ctx) return SHG_EINVAL;
    if (ctx->g.nzt == 0) return shg_set_temperature(ctx, nullptr, T_uniform, per_member);
    if (!T_host) return SHG_EINVAL;
    const size_t bytes = sizeof(float) * (size_t)(per_member ? ctx->g.batch : 1) * ctx->g.nzt * np_of(ctx);
    if (ctx->T_owned_bytes < bytes) {
        CU(cudaStreamSynchronize(ctx->last_stream));      // an earlier propagate may still read the old copy
        cudaFree(ctx->d_T_owned);
        ctx->d_T_owned = nullptr;
        ctx->T_owned_bytes = 0;
        CU(cudaMalloc((void**)&ctx->d_T_owned, bytes));
        ctx->T_owned_bytes = bytes;
    }
    // One array for all members, large enough to matter: upload it plane chunk by plane chunk on the copy stream
    // (after whatever the caller's stream and the last propagate still have in flight), one event per chunk.
    // shg_propagate makes its kernels wait for the chunks they need: the persistent kernel of a single simulation
    // runs the z-steps that the first chunk covers while the second is copied, and so on (a z-step reads the planes
    // around its two nodes only, G15), everything else waits for the last chunk.
    const int nzt = ctx->g.nzt;
    ctx->up_chunks = 0;
    ctx->up_host = nullptr;
    // Deferring means the array is read AFTER this call returns, which only page-locked memory makes worthwhile (an
    // asynchronous copy from pageable memory blocks the host until it is staged: no overlap) and which a caller of a
    // pageable buffer does not expect: such a buffer is copied during the call, as before.
    bool pinned = false;
    {
        cudaPointerAttributes at{};
        if (cudaPointerGetAttributes(&at, T_host) == cudaSuccess)
            pinned = (at.type == cudaMemoryTypeHost || at.type == cudaMemoryTypeManaged);
        else
            cudaGetLastError();
    }
    if (pinned && !(per_member && ctx->g.batch > 1) && nzt >= 8 && bytes >= ((size_t)32 << 20)) {
        // deferred: the next shg_propagate enqueues the chunked copy (enqueue_upload) behind its own field uploads
        const int rc = shg_set_temperature(ctx, ctx->d_T_owned, T_uniform, per_member);
        ctx->up_host = T_host;
        return rc;
    }
    CU(cudaMemcpyAsync(ctx->d_T_owned, T_host, bytes, cudaMemcpyHostToDevice, (cudaStream_t)cuda_stream));
    return shg_set_temperature(ctx, ctx->d_T_owned, T_uniform, per_member);
}

int shg_set_heat_output(shg_ctx* ctx, float* Q_device, int nq) {
    if (!ctx) return SHG_EINVAL;
    if (!Q_device) { ctx->d_Q = nullptr; ctx->nq = 0; return SHG_OK; }
    const int nz = ctx->g.nz;
    if (nq < 1 || nq > nz || !aligned16(Q_device)) return SHG_EINVAL;
    if (nq != ctx->nq || !ctx->d_qmap) {
        std::vector<int> map((size_t)nz, -1);
        for (int k = 0; k < nq; ++k) {
            long long nk = ((2LL * k + 1) * nz) / (2LL * nq);
            if (nk > nz - 1) nk = nz - 1;
            map[(size_t)nk] = k;
        }
        CU(cudaStreamSynchronize(ctx->last_stream));      // an earlier propagate may still read the old map
        if (!ctx->d_qmap) CU(cudaMalloc((void**)&ctx->d_qmap, sizeof(int) * (size_t)nz));
        CU(cudaMemcpy(ctx->d_qmap, map.data(), sizeof(int) * (size_t)nz, cudaMemcpyHostToDevice));
    }
    ctx->d_Q = Q_device;
    ctx->nq = nq;
    return SHG_OK;
}

// The chunked upload of a host temperature array that shg_set_temperature_host deferred: plane chunk by plane chunk
// on the library's copy stream, after everything the propagate's stream (its field uploads) and the last propagate
// have in flight, one event per chunk.
static int enqueue_upload(shg_ctx* ctx, cudaStream_t st) {
    const float* T_host = ctx->up_host;
    ctx->up_host = nullptr;
    const int nzt = ctx->g.nzt;
    const size_t plane_f = np_of(ctx);
    const size_t bytes = sizeof(float) * (size_t)nzt * plane_f;
    if (!ctx->copy_stream) CU(cudaStreamCreateWithFlags(&ctx->copy_stream, cudaStreamNonBlocking));
    if (!ctx->guard_ev) CU(cudaEventCreateWithFlags(&ctx->guard_ev, cudaEventDisableTiming));
    int chunks = (int)(bytes >> 26);                           // ~64 MB each ...
    chunks = chunks < 2 ? 2 : (chunks > 16 ? 16 : chunks);
    const int planes = (nzt + chunks - 1) / chunks;
    // ... after two small ones (1/8 and 1/4 of a chunk, at least two planes: a z-step needs two), so that the first
    // launch of the z-loop waits for a few megabytes only
    ctx->up_end.clear();
    for (int p = 0, c = 0; p < nzt; ++c) {
        int len = (c == 0) ? planes / 8 : (c == 1 ? planes / 4 : planes);
        len = len < 2 ? 2 : len;
        p = (p + len < nzt) ? p + len : nzt;
        ctx->up_end.push_back(p);
    }
    chunks = (int)ctx->up_end.size();
    while ((int)ctx->up_ev.size() < chunks) {
        cudaEvent_t e;
        CU(cudaEventCreateWithFlags(&e, cudaEventDisableTiming));
        ctx->up_ev.push_back(e);
    }
    CU(cudaEventRecord(ctx->guard_ev, st));
    CU(cudaStreamWaitEvent(ctx->copy_stream, ctx->guard_ev, 0));
    if (ctx->last_stream != st && ctx->last_batch != 0) {      // the last propagate (another stream) may still read T
        CU(cudaEventRecord(ctx->guard_ev, ctx->last_stream));
        CU(cudaStreamWaitEvent(ctx->copy_stream, ctx->guard_ev, 0));
    }
    for (int c = 0; c < chunks; ++c) {
        const int p0 = c ? ctx->up_end[(size_t)c - 1] : 0, p1 = ctx->up_end[(size_t)c];
        CU(cudaMemcpyAsync(ctx->d_T_owned + (size_t)p0 * plane_f, T_host + (size_t)p0 * plane_f,
                           sizeof(float) * (size_t)(p1 - p0) * plane_f, cudaMemcpyHostToDevice, ctx->copy_stream));
        CU(cudaEventRecord(ctx->up_ev[(size_t)c], ctx->copy_stream));
    }
    ctx->up_chunks = chunks;
    return SHG_OK;
}

int shg_propagate(shg_ctx* ctx, const void* A1_in, const void* A2_in, void* A1_out, void* A2_out, int batch,
                  void* cuda_stream) {
    if (!ctx || !A1_out || !A2_out) return SHG_EINVAL;
    if (batch < 1 || batch > ctx->g.batch) return SHG_EINVAL;
    if (!aligned16(A1_in) || !aligned16(A2_in) || !aligned16(A1_out) || !aligned16(A2_out)) return SHG_EINVAL;
    {   // A field may be propagated in place (out == in, exactly); any other overlap is an error: the first row
        // pass reads both inputs of a row while it writes both outputs of other rows.
        const size_t bytes = sizeof(float2) * (size_t)batch * np_of(ctx);
        auto overlap = [bytes](const void* a, const void* b) {
            if (!a || !b) return false;
            const uintptr_t x = reinterpret_cast<uintptr_t>(a), y = reinterpret_cast<uintptr_t>(b);
            return x < y + bytes && y < x + bytes;
        };
        if (overlap(A1_out, A2_out) || overlap(A1_in, A2_out) || overlap(A2_in, A1_out) || overlap(A1_in, A2_in))
            return SHG_EINVAL;
        if ((A1_in != A1_out && overlap(A1_in, A1_out)) || (A2_in != A2_out && overlap(A2_in, A2_out)))
            return SHG_EINVAL;
    }
    if (!ctx->T_set) return SHG_ESTATE;
    // the paper's ordering (SHG_OPT_SCHEME = 1) exists with hi+lo constants and without heat output only; refused
    // here, before anything is enqueued or any state of the last run is touched
    if (ctx->scheme == 1 && (!ctx->precise || ctx->d_Q)) return SHG_EINVAL;
    if (!A1_in)                      // Gaussian pump of Eq. 6 / Eq. 5 from the beams of shg_create
        for (int b = 0; b < batch; ++b)
            if (!(ctx->beams[b].w0 > 0) || !(ctx->beams[b].P >= 0)) return SHG_EINVAL;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    if (ctx->tables_dirty) {
        // tables are uploaded with synchronous copies; make sure no earlier propagate still reads them
        CU(cudaStreamSynchronize(ctx->last_stream));
        int rc = upload_tables(ctx);
        if (rc != SHG_OK) return rc;
    }
    if (ctx->uniform_dirty) {
        // Only T_uniform changed: two small kernels on this propagate's stream, no copy, no host wait (a sweep over
        // T_uniform enqueues and returns).  A propagate still running on ANOTHER stream reads the same scalars: this
        // stream waits for it on the device.
        if (ctx->last_batch != 0 && ctx->last_stream != st) {
            if (!ctx->guard_ev) CU(cudaEventCreateWithFlags(&ctx->guard_ev, cudaEventDisableTiming));
            CU(cudaEventRecord(ctx->guard_ev, ctx->last_stream));
            CU(cudaStreamWaitEvent(st, ctx->guard_ev, 0));
        }
        const double dk = ctx->c.dk0 + ctx->c.ddk_dT * (ctx->T_uniform - ctx->c.T_pm);
        k_set_dk_uniform<<<(ctx->g.batch + 127) / 128, 128, 0, st>>>(ctx->d_mem, ctx->g.batch, dk);
        CU(cudaGetLastError());
        if (ctx->d_ucoef) {
            k_uniform_coefs<<<(ctx->g.nz + 127) / 128, 128, 0, st>>>(ctx->d_mem, ctx->d_ucoef, ctx->g.nz);
            CU(cudaGetLastError());
        }
        ctx->uniform_dirty = false;
    }
    if (!A1_in) {
        int rc = shg_gaussian_input(ctx, A1_out, batch, cuda_stream);
        if (rc != SHG_OK) return rc;
        A1_in = A1_out;
    }
    const shg_grid& g = ctx->g;
    shg::Params P{};
    P.nx = g.nx; P.ny = g.ny; P.nz = g.nz; P.nzt = g.nzt; P.batch = batch;
    P.n_begin = 0; P.n_end = g.nz;
    P.ny_log2 = 0;
    while ((1 << P.ny_log2) < g.ny) ++P.ny_log2;
    P.A[0] = (float2*)A1_out; P.A[1] = (float2*)A2_out;
    P.Ain[0] = (const float2*)A1_in; P.Ain[1] = (const float2*)A2_in;
    P.T = ctx->d_T; P.T_per_member = ctx->T_per_member;
    P.phi = ctx->d_phi;
    P.twx = ctx->d_twx; P.twy = ctx->d_twy;
    for (int hs = 0; hs < 2; ++hs) { P.hx[hs] = ctx->d_hx[hs]; P.hy[hs] = ctx->d_hy[hs]; }
    P.mem = ctx->d_mem;
    P.ucoef = ctx->d_ucoef;
    P.hfix = ctx->d_hfix; P.pfix = ctx->d_pfix;
    P.rec_every = ctx->rec_every; P.nrec = ctx->nrec;
    P.spin_limit = ctx->spin_limit;
    P.Q = ctx->d_Q; P.qmap = ctx->d_qmap; P.nq = ctx->nq;
    P.barrier = ctx->d_barrier;
    P.status = reinterpret_cast<int*>(ctx->d_barrier + 1);
    P.trace = ctx->d_trace;
    P.acquire_fence = ctx->acquire_fence;
    P.scheme = ctx->scheme;
    P.trace_steps = ctx->trace_steps;

    const size_t np = np_of(ctx);
    int launches = 0;
    // A host temperature array may still be on its way (shg_set_temperature_host): kernels that read T wait for the
    // chunk events.  pending: this propagate reads the library's copy and an upload is outstanding.
    if (ctx->up_host != nullptr && P.T != nullptr && P.T == ctx->d_T_owned) {
        const int rc = enqueue_upload(ctx, st);
        if (rc != SHG_OK) return rc;
    }
    const bool pending = ctx->up_chunks > 0 && P.T != nullptr && P.T == ctx->d_T_owned;
    auto wait_all_chunks = [&]() -> cudaError_t {
        return pending ? cudaStreamWaitEvent(st, ctx->up_ev[(size_t)ctx->up_chunks - 1], 0) : cudaSuccess;
    };
    // highest temperature plane that z-step n reads: the planes around its two nodes n and n + 1 (G15, t_node)
    auto last_plane_of_step = [&](int n) {
        if (g.nzt <= 1) return 0;
        const long long num = (long long)(n + 1) * (g.nzt - 1);
        long long k = num / g.nz;
        long long rem = num - k * g.nz;
        if (k > g.nzt - 2) { k = g.nzt - 2; rem = g.nz; }
        return (int)(k + (rem != 0 ? 1 : 0));
    };
    ctx->hist_valid = false;             // from here on the device history belongs to this run
    CU(cudaMemsetAsync(ctx->d_hfix, 0, sizeof(long long) * (size_t)g.batch * (ctx->nrec + 1) * 2, st));
    // barrier counters start at zero; the status word [1] is NOT cleared here: a timeout of an earlier propagate that
    // nobody has synchronised on yet stays raised (this run's kernels then give up at their first barrier) until
    // shg_synchronize / shg_power* has reported it
    CU(cudaMemsetAsync(ctx->d_barrier, 0, sizeof(unsigned int), st));
    CU(cudaMemsetAsync(ctx->d_barrier + 2, 0, 6 * sizeof(unsigned int), st));
    if (g.nzt > 0) CU(cudaMemsetAsync(ctx->d_phi, 0, sizeof(float) * (size_t)batch * np, st));
    {   // P_j(0) and the fixed-point scale of every member, from the input (before anything overwrites it)
        int ch = (int)(np / 4096);
        ch = ch < 1 ? 1 : (ch > 64 ? 64 : ch);
        k_input_power<<<dim3(ch, batch), 256, 0, st>>>((const float2*)A1_in, (const float2*)A2_in, np, ctx->nrec,
                                                       ctx->d_inpart, ctx->d_ticket, ctx->d_pfix, ctx->d_hfix);
        CU(cudaGetLastError());
        ++launches;
    }

    // Small square grids: the whole run of a member in one thread-block cluster (shg_cluster.cuh), one launch.
    if (ctx->cluster_mode != 0 && ctx->persistent && g.nx == g.ny && g.nx <= 128 && ctx->scheme == 0 && ctx->precise &&
        !P.Q) {
        int csize = 0;
        const int cand[2] = {16, 8};
        for (int i = 0; i < 2 && csize == 0; ++i) {
            const int c = cand[i];
            if (ctx->cluster_mode >= 8 && ctx->cluster_mode != c) continue;
            int cap = 0;
            const cudaError_t e = ctx->Lx.cluster(P, c, false, &cap, st);
            if (e != cudaSuccess) { cudaGetLastError(); continue; }         // this size is not built / not possible
            // auto: only when every member's cluster is resident at once (a latency optimisation for one or a few
            // simulations; a sweep of many members fills the device better through the batched kernels).  256 x 256
            // has no cluster kernel: measured at 36 us per z-step in a 16-CTA cluster against 11 us in the
            // persistent kernel on 148 SMs (profiles/r02a_cluster.md) -- one simulation's arithmetic alone keeps
            // 16 SMs busier than the device-wide barriers cost.
            if (ctx->cluster_mode >= 8 ? cap >= 1 : batch <= cap) csize = c;
        }
        if (csize != 0) {
            P.trace_grid = batch * csize < ctx->sm_count ? batch * csize : ctx->sm_count;
            ctx->trace_grid = P.trace_grid;
            CU(wait_all_chunks());
            if (ctx->timing) CU(cudaEventRecord(ctx->ev[0], st));
            const cudaError_t e = ctx->Lx.cluster(P, csize, true, nullptr, st);
            if (e == cudaSuccess) {
                ++launches;
                if (ctx->timing) { CU(cudaEventRecord(ctx->ev[1], st)); ctx->ev_recorded = true; }
                ctx->last_stream = st;
                ctx->last_batch = batch;
                ctx->last_launches = launches;
                ctx->last_scheme = 0;
                ctx->last_cluster = csize;
                ctx->last_kernel = 4;
                if (pending) ctx->up_chunks = 0;
                ctx->hist_valid = false;
                return SHG_OK;
            }
            if (!coop_unavailable(e) && e != cudaErrorInvalidValue && e != cudaErrorInvalidConfiguration)
                return cuda_fail(e, "cluster kernel launch");
            cudaGetLastError();                                             // fall through to the batched kernels
        }
    }
    ctx->last_cluster = 0;

    const shg::LaunchInfo ix = ctx->Lx.info(), iy = ctx->Ly.info();
    const int UR = batch * g.ny / ix.rows_per_item;          // row-pass items
    const int UC = batch * 2 * (g.nx / iy.cols_per_item);    // column-pass strips
    const int max_grid = ctx->sm_count;
    const int grid_r = UR < max_grid ? UR : max_grid;
    const int grid_c = UC < max_grid ? UC : max_grid;
    const bool use_persist = ctx->persistent && g.nx == g.ny;
    // How many slots / teams of a CTA take items.  A CTA owns ipc = ceil(U / grid) items; they are dealt round
    // robin, so with `rounds` = ceil(ipc / slots) rounds it is better to use just enough slots for full
    // rounds (every busy warp then runs the same number of items back to back) than to leave a ragged last
    // round in which a few warps run alone.  Rounded up so that the busy warps spread evenly over the four
    // schedulers of the SM.
    auto active = [](int U, int grid, int slots, int warps_per_slot) {
        const int ipc = (U + grid - 1) / grid;
        const int rounds = (ipc + slots - 1) / slots;
        int act = (ipc + rounds - 1) / rounds;
        const int mult = warps_per_slot >= 4 ? 1 : 4 / warps_per_slot;
        act = (act + mult - 1) / mult * mult;
        return act < slots ? act : slots;
    };
    {
        const int gr = use_persist ? (grid_r > grid_c ? grid_r : grid_c) : grid_r;
        const int gc = use_persist ? gr : grid_c;
        P.row_slots = active(UR, gr, ix.row_slots, ix.warps / ix.row_slots);
        P.col_teams = active(UC, gc, iy.col_teams, iy.team_warps);
    }
    const bool prec = ctx->precise;
    P.tab_smem = (use_persist && ctx->tables_smem && batch == 1 && prec && ctx->scheme == 0 && !P.Q) ? 1 : 0;
    {   // Batched runs: the software-pipelined kernel pays once a warp has a few row items per phase (two groups of
        // members: half the items of a pass each); with less than two (cfg4: 0.9) a phase is one item per warp
        // and the split only adds phases.  SHG_OPT_PIPELINE: 0 never, 1 auto (default), 2 whenever batch >= 2.
        const int grid_p = grid_r > grid_c ? grid_r : grid_c;
        const long long slots = (long long)grid_p * ix.row_slots;
        const bool enough = ctx->pipeline == 2 || (long long)UR >= 4 * slots;
        P.pipeline = (use_persist && ctx->pipeline != 0 && enough && batch >= 2 && ctx->scheme == 0 && !P.Q &&
                      !P.trace) ? 1 : 0;
    }
    {   // Sparse launch: every CTA owns at most one row item per slot and at most half of its warps have one
        // (single small simulations).  The persistent kernel then spreads the nonlinear step over the whole CTA.
        const int grid_p = grid_r > grid_c ? grid_r : grid_c;
        const int ipc = (UR + grid_p - 1) / grid_p;
        const int warps_per_slot = ix.warps / ix.row_slots;
        P.flat_rows = (use_persist && !P.pipeline && ctx->scheme == 0 && !P.Q && ipc <= ix.row_slots &&
                       2 * ipc * warps_per_slot <= ix.warps) ? 1 : 0;
    }

    if (ctx->scheme == 1) {
        // The paper's ordering (Eq. 14-15): N(dz/2) - L(dz) - N(dz/2).  ROW_FIRST takes the first
        // half-step of step 0, the row pass n of the loop the second half of step n and the first half of step
        // n + 1, ROW_FINAL the second half of step nz - 1; every linear step is a full dz (tables 0).
        CU(wait_all_chunks());
        CU(ctx->Lx.row(P, shg::ROW_FIRST, 0, 0, prec, grid_r, st)); ++launches;
        CU(ctx->Ly.col(P, 0, prec, grid_c, st)); ++launches;
        if (ctx->timing) CU(cudaEventRecord(ctx->ev[0], st));
        bool looped = false;
        ctx->last_kernel = 0;
        if (use_persist && g.nz > 1) {
            const int grid_p = grid_r > grid_c ? grid_r : grid_c;
            ctx->trace_grid = grid_p;
            const cudaError_t e = ctx->Lx.persist(P, prec, grid_p, st);
            if (e == cudaSuccess) { ++launches; looped = true; ctx->last_kernel = 5; }
            else if (!coop_unavailable(e)) return cuda_fail(e, "persistent kernel launch");
        }
        if (!looped) {
            for (int n = 0; n < g.nz - 1; ++n) {
                CU(ctx->Lx.row(P, shg::ROW_MID, n, 0, prec, grid_r, st)); ++launches;
                CU(ctx->Ly.col(P, 0, prec, grid_c, st)); ++launches;
            }
        }
        if (ctx->timing) { CU(cudaEventRecord(ctx->ev[1], st)); ctx->ev_recorded = true; }
        CU(ctx->Lx.row(P, shg::ROW_FINAL, g.nz - 1, 0, prec, grid_r, st)); ++launches;
    } else {
    // opening half-step (x part) on the input, then its y part
    CU(ctx->Lx.row(P, shg::ROW_FIRST, 0, 1, prec, grid_r, st)); ++launches;
    CU(ctx->Ly.col(P, 1, prec, grid_c, st)); ++launches;
    if (ctx->timing) CU(cudaEventRecord(ctx->ev[0], st));
    bool looped = false;
    ctx->last_kernel = 0;
    if (use_persist) {
        const int grid_p = grid_r > grid_c ? grid_r : grid_c;
        ctx->trace_grid = grid_p;
        if (pending && !P.pipeline) {
            // Temperature array still uploading: one launch per chunk, over the z-steps whose planes that chunk
            // completes (k_persist / k_persist_flat take a step range; the device-wide barrier counts from zero in
            // every launch).  The copy of chunk c + 1 runs under the z-steps of chunk c.
            int n0 = 0;
            for (int c = 0; c < ctx->up_chunks && n0 < g.nz; ++c) {
                const int have = ctx->up_end[(size_t)c];                   // planes [0, have) have arrived
                int n1 = n0;
                while (n1 < g.nz && last_plane_of_step(n1) < have) ++n1;
                if (c == ctx->up_chunks - 1) n1 = g.nz;
                if (n1 == n0) continue;
                CU(cudaStreamWaitEvent(st, ctx->up_ev[(size_t)c], 0));
                if (n0 > 0) CU(cudaMemsetAsync(ctx->d_barrier, 0, sizeof(unsigned int), st));
                P.n_begin = n0; P.n_end = n1;
                const cudaError_t e = ctx->Lx.persist(P, prec, grid_p, st);
                if (e != cudaSuccess) {
                    if (n0 == 0 && coop_unavailable(e)) break;             // fall back to the per-pass launches below
                    return cuda_fail(e, "persistent kernel launch");
                }
                ++launches; looped = true;
                n0 = n1;
            }
            P.n_begin = 0; P.n_end = g.nz;
            if (looped) ctx->last_kernel = P.flat_rows ? 2 : 1;
        } else {
            CU(wait_all_chunks());
            const cudaError_t e = ctx->Lx.persist(P, prec, grid_p, st);
            if (e == cudaSuccess) { ++launches; looped = true; ctx->last_kernel = P.flat_rows ? 2 : (P.pipeline ? 3 : 1); }
            else if (!coop_unavailable(e)) return cuda_fail(e, "persistent kernel launch");
        }
    }
    if (!looped) {
        CU(wait_all_chunks());
        for (int n = 0; n < g.nz; ++n) {
            const int hsel = (n == g.nz - 1) ? 1 : 0;
            CU(ctx->Lx.row(P, shg::ROW_MID, n, hsel, prec, grid_r, st)); ++launches;
            CU(ctx->Ly.col(P, hsel, prec, grid_c, st)); ++launches;
        }
    }
    if (ctx->timing) { CU(cudaEventRecord(ctx->ev[1], st)); ctx->ev_recorded = true; }
    CU(ctx->Lx.row(P, shg::ROW_FINAL, 0, 0, prec, grid_r, st)); ++launches;
    }

    ctx->last_stream = st;
    ctx->last_batch = batch;
    ctx->last_launches = launches;
    ctx->last_scheme = ctx->scheme;
    ctx->hist_valid = false;
    if (pending) ctx->up_chunks = 0;         // this stream has waited for every chunk: the copy is complete for what follows
    return SHG_OK;
}

int shg_propagate_host(shg_ctx* ctx, const void* A1_in, const void* A2_in, void* A1_out, void* A2_out, int batch,
                       void* cuda_stream) {
    if (!ctx || !A1_out || !A2_out) return SHG_EINVAL;
    if (batch < 1 || batch > ctx->g.batch) return SHG_EINVAL;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const size_t cap = sizeof(float2) * (size_t)ctx->g.batch * np_of(ctx);
    const size_t bytes = sizeof(float2) * (size_t)batch * np_of(ctx);
    for (int i = 0; i < 2; ++i)
        if (!ctx->d_stage[i]) CU(cudaMalloc((void**)&ctx->d_stage[i], cap));
    if (A1_in) CU(cudaMemcpyAsync(ctx->d_stage[0], A1_in, bytes, cudaMemcpyHostToDevice, st));
    if (A2_in) CU(cudaMemcpyAsync(ctx->d_stage[1], A2_in, bytes, cudaMemcpyHostToDevice, st));
    int rc = shg_propagate(ctx, A1_in ? ctx->d_stage[0] : nullptr, A2_in ? ctx->d_stage[1] : nullptr,
                           ctx->d_stage[0], ctx->d_stage[1], batch, cuda_stream);
    if (rc != SHG_OK) return rc;
    // (a barrier timeout of the persistent kernel is reported by shg_synchronize / shg_power*, not here: this
    // call only enqueues)
    CU(cudaMemcpyAsync(A1_out, ctx->d_stage[0], bytes, cudaMemcpyDeviceToHost, st));
    CU(cudaMemcpyAsync(A2_out, ctx->d_stage[1], bytes, cudaMemcpyDeviceToHost, st));
    return SHG_OK;
}

int shg_synchronize(shg_ctx* ctx) {
    if (!ctx) return SHG_EINVAL;
    if (ctx->last_batch == 0) return SHG_OK;
    CU(cudaStreamSynchronize(ctx->last_stream));
    unsigned int bs[2] = {0, 0};
    CU(cudaMemcpy(bs, ctx->d_barrier, sizeof(bs), cudaMemcpyDeviceToHost));
    if (bs[1] != 0) {
        CU(cudaMemset(ctx->d_barrier + 1, 0, sizeof(unsigned int)));     // reported once, then cleared
        ctx->hist_valid = false;
        g_cuda_msg = "persistent kernel: a device-wide barrier timed out (not all CTAs co-resident, or the spin limit "
                     "of SHG_OPT_SPIN_LIMIT is too short for this run); the outputs of every propagate enqueued since "
                     "the last successful shg_synchronize / shg_power are invalid";
        return SHG_ECUDA;
    }
    return SHG_OK;
}

static int fetch_history(shg_ctx* ctx) {
    if (ctx->last_batch == 0) return SHG_ESTATE;
    if (ctx->hist_valid) return SHG_OK;
    int rc = shg_synchronize(ctx);
    if (rc != SHG_OK) return rc;
    CU(cudaMemcpy(ctx->hfix_host.data(), ctx->d_hfix, sizeof(long long) * ctx->hfix_host.size(), cudaMemcpyDeviceToHost));
    CU(cudaMemcpy(ctx->pfix_host.data(), ctx->d_pfix, sizeof(float) * ctx->pfix_host.size(), cudaMemcpyDeviceToHost));
    // fixed point -> W: sum |A_j|^2 = fix / 2^e (exact in double up to 2^53), P_j = (eps0 c n_j/2) dx dy sum.
    // Scheme 0 takes the sums of nodes >= 1 right after the nonlinear step: Parseval factor exp(-alpha_j dz/2).
    const size_t per = (size_t)(ctx->nrec + 1) * 2;
    for (int b = 0; b < ctx->last_batch; ++b) {
        const double inv = 1.0 / (double)ctx->pfix_host[(size_t)b];
        for (size_t i = 0; i < per; ++i) {
            const int f = (int)(i & 1);
            const bool node0 = (i < 2);
            const double sc = (node0 || ctx->last_scheme == 1) ? ctx->pscale_in[(size_t)b * 2 + f]
                                                              : ctx->pscale_step[(size_t)b * 2 + f];
            ctx->hist_host[(size_t)b * per + i] = (double)ctx->hfix_host[(size_t)b * per + i] * inv * sc;
        }
    }
    ctx->hist_valid = true;
    return SHG_OK;
}

int shg_history_length(const shg_ctx* ctx) { return ctx ? ctx->nrec + 1 : SHG_EINVAL; }

int shg_history_nodes(const shg_ctx* ctx, int32_t* nodes) {
    if (!ctx || !nodes) return SHG_EINVAL;
    for (int k = 0; k < ctx->nrec; ++k) nodes[k] = k * ctx->rec_every;
    nodes[ctx->nrec] = ctx->g.nz;
    return SHG_OK;
}

int shg_power_history(shg_ctx* ctx, int member, double* out) {
    if (!ctx || !out || member < 0 || member >= ctx->g.batch) return SHG_EINVAL;
    int rc = fetch_history(ctx);
    if (rc != SHG_OK) return rc;
    if (member >= ctx->last_batch) return SHG_ESTATE;
    const size_t n = (size_t)(ctx->nrec + 1) * 2;
    std::memcpy(out, ctx->hist_host.data() + (size_t)member * n, sizeof(double) * n);
    return SHG_OK;
}

int shg_power(shg_ctx* ctx, int member, double z, double* P1, double* P2) {
    if (!ctx || !P1 || !P2 || member < 0 || member >= ctx->g.batch) return SHG_EINVAL;
    int rc = fetch_history(ctx);
    if (rc != SHG_OK) return rc;
    if (member >= ctx->last_batch) return SHG_ESTATE;
    // nearest RECORDED node: nodes k rec_every (k < nrec) and nz
    const double dz = ctx->c.L / ctx->g.nz;
    const int re = ctx->rec_every, nz = ctx->g.nz;
    double zn = z / dz;
    zn = zn < 0 ? 0 : (zn > nz ? nz : zn);
    long k = std::lround(zn / re);
    if (k > ctx->nrec - 1) k = ctx->nrec - 1;
    const long slot = (std::fabs(zn - (double)nz) <= std::fabs(zn - (double)(k * re))) ? ctx->nrec : k;
    const double* h = ctx->hist_host.data() + (size_t)member * (ctx->nrec + 1) * 2;
    *P1 = h[2 * slot];
    *P2 = h[2 * slot + 1];
    return SHG_OK;
}

int shg_gaussian_input(shg_ctx* ctx, void* A1_device, int batch, void* cuda_stream) {
    if (!ctx || !A1_device || batch < 1 || batch > ctx->g.batch) return SHG_EINVAL;
    for (int b = 0; b < batch; ++b)
        if (!(ctx->beams[b].w0 > 0) || !(ctx->beams[b].P >= 0)) return SHG_EINVAL;
    if (ctx->tables_dirty) {
        CU(cudaStreamSynchronize(ctx->last_stream));
        int rc = upload_tables(ctx);
        if (rc != SHG_OK) return rc;
    }
    const size_t total = np_of(ctx) * batch;
    const int threads = 256;
    const unsigned blocks = (unsigned)((total + threads - 1) / threads);
    k_gaussian<<<blocks, threads, 0, (cudaStream_t)cuda_stream>>>((float2*)A1_device, ctx->d_gauss, ctx->g.nx,
                                                                 ctx->g.ny, batch);
    CU(cudaGetLastError());
    return SHG_OK;
}

int shg_enable_timing(shg_ctx* ctx, int on) {
    if (!ctx) return SHG_EINVAL;
    if (on && !ctx->ev[0]) {
        CU(cudaEventCreate(&ctx->ev[0]));
        CU(cudaEventCreate(&ctx->ev[1]));
    }
    ctx->timing = (on != 0);
    return SHG_OK;
}

int shg_last_main_loop_ms(shg_ctx* ctx, float* ms) {
    if (!ctx || !ms) return SHG_EINVAL;
    if (!ctx->ev_recorded) return SHG_ESTATE;
    CU(cudaEventSynchronize(ctx->ev[1]));
    CU(cudaEventElapsedTime(ms, ctx->ev[0], ctx->ev[1]));
    return SHG_OK;
}

int shg_read_trace(shg_ctx* ctx, long long* out, int* steps, int* grid) {
    if (!ctx || !steps || !grid) return SHG_EINVAL;
    *steps = ctx->trace_steps < ctx->g.nz ? ctx->trace_steps : ctx->g.nz;
    *grid = ctx->trace_grid;
    if (!out) return SHG_OK;
    if (!ctx->d_trace || ctx->trace_grid == 0) return SHG_ESTATE;
    CU(cudaStreamSynchronize(ctx->last_stream));
    CU(cudaMemcpy(out, ctx->d_trace, sizeof(long long) * (size_t)(*steps) * ctx->trace_grid * 8, cudaMemcpyDeviceToHost));
    return SHG_OK;
}

int shg_last_launch_count(const shg_ctx* ctx) { return ctx ? ctx->last_launches : SHG_EINVAL; }

int shg_last_cluster_size(const shg_ctx* ctx) { return ctx ? ctx->last_cluster : SHG_EINVAL; }
int shg_last_kernel(const shg_ctx* ctx) { return ctx ? ctx->last_kernel : SHG_EINVAL; }

}  // extern "C"
