/*
 * shg_oracle.c -- plain double-precision CPU oracle for the SSFM hot path of arxiv/paper_2410_04994.
 * TEST INFRASTRUCTURE ONLY (see shg_oracle.h).  Shares nothing with the CUDA path.
 *
 * Algorithm (per batch member), following the paper step by step in its own notation:
 *   P:72-73  (Eq. 2)   coupled-wave equations for A_F (=A1) and A_SH (=A2)
 *   P:80     (Eq. 3)   phi(x,y,z) = int_0^z dk dz'
 *   P:138-145 (Eq. 11) split into the linear operator L_j and the nonlinear operator N
 *   P:157-161 (Eq. 14-15) symmetric split step; north_star fixes the order L/2 - N(dz) - L/2
 *   P:136              N is advanced with one classical fourth-order Runge-Kutta step
 *   P:334-352 (App. A) the linear part is a diagonal multiply in the 2-D transverse Fourier domain
 *   P:120              I = eps0 c n |A|^2 / 2, so P_j = (eps0 c n_j / 2) dx dy sum |A_j|^2
 *
 * Readings of garbled / inconsistent passages (full list with evidence: DESIGN.md §3):
 *   G2  kappa2 = 2 pi d_eff / (n2 lambda1)   (the printed lambda_SH makes it 2x too large for Eq. 17
 *       and for energy conservation with the intensity definition of)
 *   G3  diffraction propagator exp(-i (kx^2+ky^2) h / (2 k_j)) with the input beam of Eq. 6 as printed
 *   G4  e^{-i phi} in the FH line, e^{+i phi} in the SH line, exactly the form of Eq. 2
 *   G5  TPA term -(1/2) beta_j I_j A_j with I_j the intensity of P:120
 *   G15 T planes at z_k = k L/(nzt-1), linear interpolation to the step nodes; dk linear inside a step
 */
#include "shg_oracle.h"

#include <complex.h>
#include <math.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef double complex cplx;

static const double ORC_PI   = 3.14159265358979323846264338327950288;
static const double ORC_EPS0 = 8.8541878128e-12;   /* F/m  */
static const double ORC_C    = 299792458.0;        /* m/s  */

struct orc_ctx {
    orc_grid    g;
    orc_crystal c;
    orc_options o;
    orc_beam*   beams;       /* [batch] */
    const float* T;          /* borrowed */
    double      T_uniform;
    int         T_per_member;
    int         T_set;
    double*     hist;        /* [batch][nz+1][2] */
    int         propagated;
    double*     Q;           /* borrowed heat-source output [batch][nq][ny][nx], or NULL */
    int         nq;
};

void orc_set_num_threads(int n) {
#ifdef _OPENMP
    if (n >= 1) omp_set_num_threads(n);
#else
    (void)n;
#endif
}

int orc_num_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

static int is_pow2(int n) { return n >= 2 && (n & (n - 1)) == 0; }

/* ------------------------------------------------------------------------------------------------
 * Transforms.  Definition (Eq. A.2 is the inverse, kernel e^{+i 2 pi q x}; G12):
 *   forward  X[k] = sum_n x[n] e^{-2 pi i k n / N}            (unnormalised)
 *   inverse  x[n] = (1/N) sum_k X[k] e^{+2 pi i k n / N}
 * ------------------------------------------------------------------------------------------------ */

/* The definition, O(N^2) per line. */
static void dft1_brute(const cplx* in, cplx* out, int n, int sign) {
    for (int k = 0; k < n; ++k) {
        cplx acc = 0.0;
        for (int j = 0; j < n; ++j) {
            /* reduce k*j mod n before forming the angle so the argument stays small and exact */
            long long kj = ((long long)k * j) % n;
            double ang = sign * 2.0 * ORC_PI * (double)kj / (double)n;
            acc += in[j] * (cos(ang) + I * sin(ang));
        }
        out[k] = acc;
    }
}

/* Twiddle table for a line of length n: w[k] = e^{sign 2 pi i k / n}, k = 0 .. n/2-1. */
static cplx* twiddle_table(int n, int sign) {
    cplx* w = (cplx*)malloc(sizeof(cplx) * (size_t)(n / 2 > 0 ? n / 2 : 1));
    for (int k = 0; k < n / 2; ++k) {
        double ang = sign * 2.0 * ORC_PI * (double)k / (double)n;
        w[k] = cos(ang) + I * sin(ang);
    }
    return w;
}

/* Textbook iterative radix-2 decimation-in-time FFT, in place on a contiguous line of length n.
 * The butterfly of span `len` uses e^{sign 2 pi i k / len} = w[k * (n / len)]. */
static void fft1_radix2(cplx* x, int n, const cplx* w) {
    /* bit-reversal permutation */
    for (int i = 1, j = 0; i < n; ++i) {
        int bit = n >> 1;
        for (; j & bit; bit >>= 1) j ^= bit;
        j ^= bit;
        if (i < j) { cplx t = x[i]; x[i] = x[j]; x[j] = t; }
    }
    for (int len = 2; len <= n; len <<= 1) {
        int half = len >> 1;
        int step = n / len;
        for (int s = 0; s < n; s += len) {
            for (int k = 0; k < half; ++k) {
                cplx u = x[s + k];
                cplx v = x[s + k + half] * w[k * step];
                x[s + k]        = u + v;
                x[s + k + half] = u - v;
            }
        }
    }
}

static void line_transform(cplx* x, int n, int sign, int brute, const cplx* w) {
    if (brute) {
        cplx* tmp = (cplx*)malloc(sizeof(cplx) * (size_t)n);
        dft1_brute(x, tmp, n, sign);
        memcpy(x, tmp, sizeof(cplx) * (size_t)n);
        free(tmp);
    } else {
        fft1_radix2(x, n, w);
    }
}

/* 2-D transform: every row (x direction), then every column (y direction).  Inverse divides by nx*ny. */
static void transform2(cplx* a, int ny, int nx, int sign, int brute, int parallel) {
    cplx* wx = twiddle_table(nx, sign);
    cplx* wy = twiddle_table(ny, sign);
#pragma omp parallel for schedule(static) if (parallel)
    for (int y = 0; y < ny; ++y) line_transform(a + (size_t)y * nx, nx, sign, brute, wx);
#pragma omp parallel if (parallel)
    {
        cplx* col = (cplx*)malloc(sizeof(cplx) * (size_t)ny);
#pragma omp for schedule(static)
        for (int x = 0; x < nx; ++x) {
            for (int y = 0; y < ny; ++y) col[y] = a[(size_t)y * nx + x];
            line_transform(col, ny, sign, brute, wy);
            for (int y = 0; y < ny; ++y) a[(size_t)y * nx + x] = col[y];
        }
        free(col);
    }
    if (sign > 0) {
        double s = 1.0 / ((double)nx * (double)ny);
#pragma omp parallel for schedule(static) if (parallel)
        for (long long i = 0; i < (long long)nx * ny; ++i) a[i] *= s;
    }
    free(wx);
    free(wy);
}

int orc_fft2(double* data, int ny, int nx, int sign) {
    if (!data || !is_pow2(nx) || !is_pow2(ny) || (sign != 1 && sign != -1)) return -1;
    transform2((cplx*)data, ny, nx, sign, 0, 1);
    return 0;
}

/* The 2-D definition written out directly, O((nx ny)^2): no row/column factorisation at all. */
int orc_dft2_brute(const double* in_, double* out_, int ny, int nx, int sign) {
    if (!in_ || !out_ || nx < 1 || ny < 1 || (sign != 1 && sign != -1)) return -1;
    const cplx* in = (const cplx*)in_;
    cplx* out = (cplx*)out_;
    for (int ky = 0; ky < ny; ++ky)
        for (int kx = 0; kx < nx; ++kx) {
            cplx acc = 0.0;
            for (int y = 0; y < ny; ++y)
                for (int x = 0; x < nx; ++x) {
                    double ang = sign * 2.0 * ORC_PI *
                                 ((double)(((long long)kx * x) % nx) / nx + (double)(((long long)ky * y) % ny) / ny);
                    acc += in[(size_t)y * nx + x] * (cos(ang) + I * sin(ang));
                }
            if (sign > 0) acc /= ((double)nx * (double)ny);
            out[(size_t)ky * nx + kx] = acc;
        }
    return 0;
}

/* ------------------------------------------------------------------------------------------------
 * Context
 * ------------------------------------------------------------------------------------------------ */

int orc_create(const orc_grid* g, const orc_crystal* c, const orc_beam* beams, const orc_options* opt,
               orc_ctx** out) {
    if (!g || !c || !beams || !out) return -1;
    if (!is_pow2(g->nx) || !is_pow2(g->ny) || g->nz < 1 || g->nzt < 0 || g->batch < 1) return -1;
    if (!(c->L > 0) || !(c->lambda1 > 0) || !(c->n1 > 0) || !(c->n2 > 0)) return -1;
    for (int b = 0; b < g->batch; ++b)
        if (!(beams[b].lx > 0) || !(beams[b].ly > 0)) return -1;
    orc_ctx* ctx = (orc_ctx*)calloc(1, sizeof(orc_ctx));
    if (!ctx) return -2;
    ctx->g = *g;
    ctx->c = *c;
    if (opt) ctx->o = *opt;
    ctx->beams = (orc_beam*)malloc(sizeof(orc_beam) * (size_t)g->batch);
    memcpy(ctx->beams, beams, sizeof(orc_beam) * (size_t)g->batch);
    ctx->hist = (double*)calloc((size_t)g->batch * (size_t)(g->nz + 1) * 2, sizeof(double));
    ctx->T_uniform = c->T_pm;
    ctx->T_set = (g->nzt == 0);   /* uniform T = T_pm until told otherwise */
    *out = ctx;
    return 0;
}

void orc_destroy(orc_ctx* ctx) {
    if (!ctx) return;
    free(ctx->beams);
    free(ctx->hist);
    free(ctx);
}

int orc_set_heat_output(orc_ctx* ctx, double* Q, int nq) {
    if (!ctx) return -1;
    if (Q && (nq < 1 || nq > ctx->g.nz)) return -1;
    ctx->Q = Q;
    ctx->nq = Q ? nq : 0;
    return 0;
}

int orc_set_temperature(orc_ctx* ctx, const float* T, double T_uniform, int per_member) {
    if (!ctx) return -1;
    if (ctx->g.nzt > 0 && !T) return -1;
    ctx->T = T;
    ctx->T_uniform = T_uniform;
    ctx->T_per_member = per_member ? 1 : 0;
    ctx->T_set = 1;
    return 0;
}

/* Temperature of every transverse point at step node n (z_n = n dz), G15:
 *   s = z_n (nzt-1)/L = n (nzt-1)/nz,  k = min(floor(s), nzt-2),  T = (1-(s-k)) T[k] + (s-k) T[k+1]. */
static void temperature_at_node(const orc_ctx* ctx, int member, int n, double* Tn /*[ny*nx]*/) {
    const orc_grid* g = &ctx->g;
    size_t np = (size_t)g->nx * g->ny;
    if (g->nzt == 0) {
        for (size_t i = 0; i < np; ++i) Tn[i] = ctx->T_uniform;
        return;
    }
    const float* base = ctx->T + (ctx->T_per_member ? (size_t)member * g->nzt * np : 0);
    if (g->nzt == 1) {
        for (size_t i = 0; i < np; ++i) Tn[i] = (double)base[i];
        return;
    }
    double s = (double)n * (double)(g->nzt - 1) / (double)g->nz;
    int k = (int)floor(s);
    if (k > g->nzt - 2) k = g->nzt - 2;
    double f = s - (double)k;
    const float* T0 = base + (size_t)k * np;
    const float* T1 = T0 + np;
    for (size_t i = 0; i < np; ++i) Tn[i] = (1.0 - f) * (double)T0[i] + f * (double)T1[i];
}

/* Right-hand side of the nonlinear part of Eq. 2 / the operator N of Eq. 11:
 *   dA1/dz = i kappa1 A2 conj(A1) e^{-i phi} - (beta1/2) I1 A1,   I_j = c_j |A_j|^2  (G5)
 *   dA2/dz = i kappa2 A1^2        e^{+i phi} - (beta2/2) I2 A2                                      */
typedef struct { double kappa1, kappa2, c1, c2, beta1, beta2; int undepleted; } nl_par;

static inline void nl_rhs(const nl_par* p, cplx A1, cplx A2, double phi, cplx* d1, cplx* d2) {
    cplx em = cos(phi) - I * sin(phi);
    cplx ep = cos(phi) + I * sin(phi);
    double I1 = p->c1 * (creal(A1) * creal(A1) + cimag(A1) * cimag(A1));
    double I2 = p->c2 * (creal(A2) * creal(A2) + cimag(A2) * cimag(A2));
    cplx coupling1 = p->undepleted ? 0.0 : I * p->kappa1 * A2 * conj(A1) * em;
    *d1 = coupling1 - 0.5 * p->beta1 * I1 * A1;
    *d2 = I * p->kappa2 * A1 * A1 * ep - 0.5 * p->beta2 * I2 * A2;
}

/* One classical RK4 step of length h for one point; the accumulated phase is sampled at the start,
 * the middle and the end of the step (G8). */
static inline void rk4_point(const nl_par* p, cplx* A1, cplx* A2, double h,
                             double phi_a, double phi_m, double phi_b) {
    cplx k1a, k1b, k2a, k2b, k3a, k3b, k4a, k4b;
    nl_rhs(p, *A1, *A2, phi_a, &k1a, &k1b);
    nl_rhs(p, *A1 + 0.5 * h * k1a, *A2 + 0.5 * h * k1b, phi_m, &k2a, &k2b);
    nl_rhs(p, *A1 + 0.5 * h * k2a, *A2 + 0.5 * h * k2b, phi_m, &k3a, &k3b);
    nl_rhs(p, *A1 + h * k3a, *A2 + h * k3b, phi_b, &k4a, &k4b);
    *A1 += (h / 6.0) * (k1a + 2.0 * k2a + 2.0 * k3a + k4a);
    *A2 += (h / 6.0) * (k1b + 2.0 * k2b + 2.0 * k3b + k4b);
}

/* q = sum_j alpha_j I_j + beta_j I_j^2,  I_j = eps0 c n_j |A_j|^2 / 2   (Eq. 8) */
static inline double heat_source(const nl_par* p, const orc_crystal* c, cplx A1, cplx A2) {
    double I1 = p->c1 * (creal(A1) * creal(A1) + cimag(A1) * cimag(A1));
    double I2 = p->c2 * (creal(A2) * creal(A2) + cimag(A2) * cimag(A2));
    return c->alpha1 * I1 + c->beta1 * I1 * I1 + c->alpha2 * I2 + c->beta2 * I2 * I2;
}

/* Factor of the linear step of length h for one field (P:143 L_j; P:346-352 Eq. A.4-A.5; sign G3):
 *   Hj[my][mx] = exp(-i (kx^2+ky^2) h / (2 k_j) - i kx tan(rho_j) h - alpha_j h / 2),  kx = 2 pi m'/lx,
 *   m' = m or m-nx (G11).
 * The walk-off term tan(rho) dA/dx of P:387 (G21): the field of a beam with walk-off angle rho moves by
 * +tan(rho) h along x.                                                                              */
static cplx* linear_factor(const orc_grid* g, const orc_beam* bm, double kj, double alpha, double rho, double h) {
    int nx = g->nx, ny = g->ny;
    cplx* H = (cplx*)malloc(sizeof(cplx) * (size_t)nx * ny);
    for (int my = 0; my < ny; ++my) {
        int sy = (my < ny / 2) ? my : my - ny;
        double ky = 2.0 * ORC_PI * (double)sy / bm->ly;
        for (int mx = 0; mx < nx; ++mx) {
            int sx = (mx < nx / 2) ? mx : mx - nx;
            double kx = 2.0 * ORC_PI * (double)sx / bm->lx;
            double ang = -(kx * kx + ky * ky) * h / (2.0 * kj) - kx * tan(rho) * h;
            H[(size_t)my * nx + mx] = exp(-0.5 * alpha * h) * (cos(ang) + I * sin(ang));
        }
    }
    return H;
}

/* A <- F^-1 { H . F{A} } */
static void linear_step(cplx* A, const orc_grid* g, const cplx* H, int brute, int parallel) {
    int nx = g->nx, ny = g->ny;
    transform2(A, ny, nx, -1, brute, parallel);
#pragma omp parallel for schedule(static) if (parallel)
    for (long long i = 0; i < (long long)nx * ny; ++i) A[i] *= H[i];
    transform2(A, ny, nx, +1, brute, parallel);
}

static double grid_power(const cplx* A, size_t np, double cj, double dxdy) {
    double s = 0.0;
    for (size_t i = 0; i < np; ++i) s += creal(A[i]) * creal(A[i]) + cimag(A[i]) * cimag(A[i]);
    return cj * dxdy * s;
}

/* phi(z_n + s) for dk linear in z inside the step (G15):
 *   phi_n + s dk_n + s^2 (dk_{n+1} - dk_n) / (2 dz).   s = dz/2 gives phi_n + dz (3 dk_n + dk_{n+1})/8,
 *   s = dz gives the trapezoid phi_n + dz (dk_n + dk_{n+1})/2.                                       */
static inline double phase_at(double phi_n, double dk_n, double dk_np1, double s, double dz) {
    return phi_n + s * dk_n + s * s * (dk_np1 - dk_n) / (2.0 * dz);
}

static void propagate_member(orc_ctx* ctx, int b, const cplx* A1_in, const cplx* A2_in, cplx* A1, cplx* A2,
                             int parallel) {
    const orc_grid* g = &ctx->g;
    const orc_crystal* c = &ctx->c;
    const orc_beam* bm = &ctx->beams[b];
    const int nx = g->nx, ny = g->ny, nz = g->nz;
    const size_t np = (size_t)nx * ny;
    const double dz = c->L / (double)nz;
    const double dxdy = (bm->lx / nx) * (bm->ly / ny);
    const double lambda2 = 0.5 * c->lambda1;
    const double k1 = 2.0 * ORC_PI * c->n1 / c->lambda1;
    const double k2 = 2.0 * ORC_PI * c->n2 / lambda2;
    nl_par p;
    p.kappa1 = 2.0 * ORC_PI * c->d_eff / (c->n1 * c->lambda1);
    p.kappa2 = 2.0 * ORC_PI * c->d_eff / (c->n2 * c->lambda1);     /* P:73 with G2 */
    p.c1 = 0.5 * ORC_EPS0 * ORC_C * c->n1;
    p.c2 = 0.5 * ORC_EPS0 * ORC_C * c->n2;
    p.beta1 = c->beta1;
    p.beta2 = c->beta2;
    p.undepleted = ctx->o.undepleted;
    const int brute = ctx->o.brute_dft;

    for (size_t i = 0; i < np; ++i) {
        A1[i] = A1_in[i];
        A2[i] = A2_in ? A2_in[i] : 0.0;
    }
    double* hist = ctx->hist + (size_t)b * (size_t)(nz + 1) * 2;
    hist[0] = grid_power(A1, np, p.c1, dxdy);
    hist[1] = grid_power(A2, np, p.c2, dxdy);

    /* linear factors: half step for scheme 0, full step for scheme 1 */
    const double hlin = (ctx->o.scheme == 0) ? 0.5 * dz : dz;
    cplx* H1 = linear_factor(g, bm, k1, c->alpha1, c->rho1, hlin);
    cplx* H2 = linear_factor(g, bm, k2, c->alpha2, c->rho2, hlin);
    /* test aid (orc_options.merged, scheme 0 only): the closing half-step of z-step n and the opening half-step
     * of z-step n+1 are two diagonal multiplies in the same Fourier basis, so they may be applied as ONE step of
     * length dz (the half-steps of Eq. 15 commute with each other).  The power at node n+1 is then taken
     * right after the nonlinear step: the closing half-step multiplies every Fourier mode by a phase times
     * exp(-alpha_j dz/4), so P_j(z_{n+1}) = exp(-alpha_j dz/2) c_j dx dy sum |A_j|^2 (Parseval).          */
    const int merged = (ctx->o.scheme == 0 && ctx->o.merged);
    cplx* F1 = merged ? linear_factor(g, bm, k1, c->alpha1, c->rho1, dz) : NULL;
    cplx* F2 = merged ? linear_factor(g, bm, k2, c->alpha2, c->rho2, dz) : NULL;

    double* phi  = (double*)calloc(np, sizeof(double));
    double* Tcur = (double*)malloc(sizeof(double) * np);
    double* Tnxt = (double*)malloc(sizeof(double) * np);
    temperature_at_node(ctx, b, 0, Tcur);

    for (int n = 0; n < nz; ++n) {
        temperature_at_node(ctx, b, n + 1, Tnxt);
        if (ctx->o.scheme == 0) {
            /* L/2 (merged: the opening half-step of step 0 only; later ones were applied with the previous step) */
            if (!merged || n == 0) {
                linear_step(A1, g, H1, brute, parallel);
                linear_step(A2, g, H2, brute, parallel);
            }
            /* heat source of Eq. 8, plane k <- z-step n_k = floor((2k+1) nz/(2 nq)): mean of the source
             * on the real-space fields before and after the nonlinear step (both sit at z_n + dz/2 as far as
             * the linear part goes; the mean is the trapezoid rule over the nonlinear step), G27 */
            double* qplane = NULL;
            if (ctx->Q) {
                for (int k = 0; k < ctx->nq; ++k) {
                    long long nk = ((2LL * k + 1) * nz) / (2LL * ctx->nq);
                    if (nk > nz - 1) nk = nz - 1;
                    if (nk == n) qplane = ctx->Q + ((size_t)b * ctx->nq + k) * np;
                }
            }
            if (qplane) {
                for (size_t i = 0; i < np; ++i) qplane[i] = heat_source(&p, c, A1[i], A2[i]);
            }
            /* N(dz), one RK4 step per point */
#pragma omp parallel for schedule(static) if (parallel)
            for (long long i = 0; i < (long long)np; ++i) {
                double dk_n  = c->dk0 + c->ddk_dT * (Tcur[i] - c->T_pm);
                double dk_n1 = c->dk0 + c->ddk_dT * (Tnxt[i] - c->T_pm);
                double ph_a = phi[i];
                double ph_m = phase_at(phi[i], dk_n, dk_n1, 0.5 * dz, dz);
                double ph_b = phase_at(phi[i], dk_n, dk_n1, dz, dz);
                rk4_point(&p, &A1[i], &A2[i], dz, ph_a, ph_m, ph_b);
                phi[i] = ph_b;
            }
            /* heat source of Eq. 8 on the planes whose sampled step is n: second half of the mean (G27) */
            if (qplane) {
                for (size_t i = 0; i < np; ++i) qplane[i] = 0.5 * (qplane[i] + heat_source(&p, c, A1[i], A2[i]));
            }
            if (merged) {
                hist[2 * (n + 1) + 0] = exp(-0.5 * c->alpha1 * dz) * grid_power(A1, np, p.c1, dxdy);
                hist[2 * (n + 1) + 1] = exp(-0.5 * c->alpha2 * dz) * grid_power(A2, np, p.c2, dxdy);
                /* closing half-step of step n and opening half-step of step n+1 as one step of length dz */
                linear_step(A1, g, (n == nz - 1) ? H1 : F1, brute, parallel);
                linear_step(A2, g, (n == nz - 1) ? H2 : F2, brute, parallel);
                double* tt = Tcur; Tcur = Tnxt; Tnxt = tt;
                continue;
            }
            /* L/2 */
            linear_step(A1, g, H1, brute, parallel);
            linear_step(A2, g, H2, brute, parallel);
        } else {
            /* paper's own order, Eq. 14-15: N(dz/2) - L(dz) - N(dz/2) */
#pragma omp parallel for schedule(static) if (parallel)
            for (long long i = 0; i < (long long)np; ++i) {
                double dk_n  = c->dk0 + c->ddk_dT * (Tcur[i] - c->T_pm);
                double dk_n1 = c->dk0 + c->ddk_dT * (Tnxt[i] - c->T_pm);
                rk4_point(&p, &A1[i], &A2[i], 0.5 * dz, phi[i],
                          phase_at(phi[i], dk_n, dk_n1, 0.25 * dz, dz),
                          phase_at(phi[i], dk_n, dk_n1, 0.5 * dz, dz));
            }
            linear_step(A1, g, H1, brute, parallel);
            linear_step(A2, g, H2, brute, parallel);
#pragma omp parallel for schedule(static) if (parallel)
            for (long long i = 0; i < (long long)np; ++i) {
                double dk_n  = c->dk0 + c->ddk_dT * (Tcur[i] - c->T_pm);
                double dk_n1 = c->dk0 + c->ddk_dT * (Tnxt[i] - c->T_pm);
                double ph_b = phase_at(phi[i], dk_n, dk_n1, dz, dz);
                rk4_point(&p, &A1[i], &A2[i], 0.5 * dz,
                          phase_at(phi[i], dk_n, dk_n1, 0.5 * dz, dz),
                          phase_at(phi[i], dk_n, dk_n1, 0.75 * dz, dz), ph_b);
                phi[i] = ph_b;
            }
        }
        hist[2 * (n + 1) + 0] = grid_power(A1, np, p.c1, dxdy);
        hist[2 * (n + 1) + 1] = grid_power(A2, np, p.c2, dxdy);
        double* t = Tcur; Tcur = Tnxt; Tnxt = t;
    }
    free(phi);
    free(Tcur);
    free(Tnxt);
    free(H1);
    free(H2);
    free(F1);
    free(F2);
}

int orc_propagate(orc_ctx* ctx, const double* A1_in, const double* A2_in, double* A1_out, double* A2_out,
                  int batch) {
    if (!ctx || !A1_in || !A1_out || !A2_out) return -1;
    if (batch < 1 || batch > ctx->g.batch) return -1;
    if (!ctx->T_set) return -3;
    const size_t np = (size_t)ctx->g.nx * ctx->g.ny;
    if (batch == 1) {
        propagate_member(ctx, 0, (const cplx*)A1_in, (const cplx*)A2_in, (cplx*)A1_out, (cplx*)A2_out, 1);
    } else {
        /* members are independent (no exchange step): one member per thread */
#pragma omp parallel for schedule(dynamic, 1)
        for (int b = 0; b < batch; ++b)
            propagate_member(ctx, b, (const cplx*)A1_in + b * np, A2_in ? (const cplx*)A2_in + b * np : NULL,
                             (cplx*)A1_out + b * np, (cplx*)A2_out + b * np, 0);
    }
    ctx->propagated = batch;
    return 0;
}

int orc_power_history(orc_ctx* ctx, int member, double* out) {
    if (!ctx || !out || member < 0 || member >= ctx->g.batch) return -1;
    if (member >= ctx->propagated) return -3;
    memcpy(out, ctx->hist + (size_t)member * (size_t)(ctx->g.nz + 1) * 2,
           sizeof(double) * (size_t)(ctx->g.nz + 1) * 2);
    return 0;
}

int orc_power(orc_ctx* ctx, int member, double z, double* P1, double* P2) {
    if (!ctx || !P1 || !P2 || member < 0 || member >= ctx->g.batch) return -1;
    if (member >= ctx->propagated) return -3;
    double dz = ctx->c.L / ctx->g.nz;
    long n = lround(z / dz);
    if (n < 0) n = 0;
    if (n > ctx->g.nz) n = ctx->g.nz;
    const double* h = ctx->hist + (size_t)member * (size_t)(ctx->g.nz + 1) * 2;
    *P1 = h[2 * n];
    *P2 = h[2 * n + 1];
    return 0;
}

/* Eq. 5 at z = 0 for a focus at focus_z: tau0 = (0 - focus_z)/zR, zR = w0^2 k1/2;
 * focus_z = L/2 gives Eq. 6 with xi = L/(2 zR).  Grid x_i = (i - nx/2) dx (G11).            */
int orc_gaussian_input(const orc_grid* g, const orc_crystal* c, const orc_beam* bm, double* out_) {
    if (!g || !c || !bm || !out_) return -1;
    cplx* out = (cplx*)out_;
    double k1 = 2.0 * ORC_PI * c->n1 / c->lambda1;
    double zR = 0.5 * bm->w0 * bm->w0 * k1;
    double tau0 = -bm->focus_z / zR;
    double A0 = sqrt(4.0 * bm->P / (ORC_EPS0 * ORC_C * c->n1 * ORC_PI * bm->w0 * bm->w0));   /* G17 */
    cplx q = 1.0 + I * tau0;
    double dx = bm->lx / g->nx, dy = bm->ly / g->ny;
    for (int iy = 0; iy < g->ny; ++iy) {
        double y = (iy - g->ny / 2) * dy;
        for (int ix = 0; ix < g->nx; ++ix) {
            double x = (ix - g->nx / 2) * dx;
            out[(size_t)iy * g->nx + ix] = (A0 / q) * cexp(-(x * x + y * y) / (bm->w0 * bm->w0 * q));
        }
    }
    return 0;
}
