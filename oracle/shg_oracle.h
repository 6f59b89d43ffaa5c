/*
 * shg_oracle.h -- CPU reference ("oracle") for the split-step Fourier propagation of the coupled
 * fundamental (FH, A1) and second-harmonic (SH, A2) envelopes of arxiv/paper_2410_04994 (cuSHG).
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke() and the
 * cpu_baseline / --impl reference legs of bench.py may build, link, import or call it.  It shares no
 * source, header, table or constant generator with the CUDA path under paper_2410_04994_b200/.
 *
 * Plain C99, double precision throughout, its own brute-force DFT and iterative radix-2 FFT, no
 * blocking / fusion / reordering beyond what the paper's algorithm states.  "P:n" below cites line n of
 * /root/reference/PAPER.md; "G<k>" cites the reading of an ambiguous passage listed in DESIGN.md §3.
 *
 * What is pinned (tests/test_oracle_pins.py, all `-m "not gpu"`):
 *   orc_fft2            vs orc_dft2_brute (the definition), Parseval, inverse(forward(x)) = x
 *   linear half-step    vs the analytic Gaussian beam of P:95 (Eq. 5): profile, w(z), Gouy phase
 *   absorption          vs exp(-alpha z)
 *   coupling + RK4      vs power conservation, tanh^2 depletion, sinc^2 mismatch, Boyd-Kleinman h(sigma, xi)
 *   TPA                 vs I0/(1+beta I0 z)
 *   temperature/phase   vs sinc^2 with dk = dk0 + g dT for every nzt encoding of the same field,
 *                       and the closed form for a linear-in-z mismatch
 *   walk-off            vs an exact translation by whole cells and the centroid law tan(rho) z
 *   heat source         vs alpha I0 e^{-alpha z}, beta I^2 of the TPA closed form, and P(0) - P(L) = integral of q
 *   the complete path   (diffraction + walk-off + coupling + depletion + temperature-dependent mismatch +
 *                       absorption + TPA at once) vs an independent solver of Eq. 2 written in the test (method
 *                       of lines in the interaction picture, numpy FFT, scipy DOP853 at 1e-11): second-order
 *                       convergence in dz, Richardson-extrapolated fields within 5e-8 (measured 3e-9, 6e-9).
 * No value printed in the paper exists for the five BASELINE configs themselves (the paper prints none).
 */
#ifndef SHG_ORACLE_H
#define SHG_ORACLE_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct orc_ctx orc_ctx;

/* Transverse grid, z discretisation, temperature-plane count, batch capacity.  P:78. */
typedef struct {
    int32_t nx, ny;   /* transverse points, powers of two >= 2 (FFT grid, x fastest in memory)       */
    int32_t nz;       /* z-steps >= 1, dz = L / nz                                          */
    int32_t nzt;      /* temperature planes: 0 = uniform scalar, 1 = one plane for every z,
                         >= 2 = planes at z_k = k L/(nzt-1), linear interpolation in z (G15)         */
    int32_t batch;    /* independent simulations                                                      */
} orc_grid;

/* Crystal constants, SI.  P:72-76 (Eq. 2), P:80-84 (Eq. 3-4, linearised per north_star).          */
typedef struct {
    double L, lambda1, n1, n2, d_eff;
    double dk0, ddk_dT, T_pm;      /* dk(T) = dk0 + ddk_dT (T - T_pm)   [rad/m, rad/(m K), K or C]   */
    double alpha1, alpha2;         /* linear intensity absorption, 1/m                               */
    double beta1, beta2;           /* two-photon absorption, m/W (G5)                                */
    double rho1, rho2;             /* spatial walk-off angles along x, rad (0 in the paper's runs) */
} orc_crystal;

/* Per-member beam / window.  P:95-104 (Eq. 5-6). P, w0, focus_z are used only by orc_gaussian_input. */
typedef struct {
    double P, w0, focus_z;         /* W, m (1/e field radius), m from the entrance face              */
    double lx, ly;                 /* transverse window of this member, m; dx = lx / nx              */
} orc_beam;

/* Scheme switches (test aids; all 0 = the north_star path). */
typedef struct {
    int32_t scheme;      /* 0: L/2 - N(dz) - L/2 (north_star);  1: N/2 - L - N/2 (Eq. 14-15) */
    int32_t undepleted;  /* 1: drop the coupling term of dA1/dz ("dPump = 0")                  */
    int32_t brute_dft;   /* 1: use the O(N^2)-per-line DFT definition instead of the radix-2 FFT      */
    int32_t merged;      /* 1 (scheme 0 only): apply the closing half-step of z-step n and the opening one of
                            z-step n+1 as one linear step of length dz, and take P_j(z_{n+1}) right after the
                            nonlinear step with the factor exp(-alpha_j dz/2) (Parseval) -- what a fused
                            implementation does; pinned equal to the unmerged path at 1e-12               */
} orc_options;

int  orc_create(const orc_grid*, const orc_crystal*, const orc_beam* beams /*[batch]*/,
                const orc_options* opt /*NULL = defaults*/, orc_ctx** out);
/* T: host fp32 [per_member ? batch : 1][nzt][ny][nx]; ignored (may be NULL) when nzt == 0, in which
 * case every point has temperature T_uniform.  The array is borrowed until orc_propagate returns.  */
int  orc_set_temperature(orc_ctx*, const float* T, double T_uniform, int per_member);
/* Fields: host complex128 (interleaved re, im), [batch][ny][nx].  A2_in may be NULL (zeros).        */
int  orc_propagate(orc_ctx*, const double* A1_in, const double* A2_in, double* A1_out, double* A2_out,
                   int batch);
/* Power (W) of both fields of one member at the recorded node nearest to z.  P:120 (I).      */
int  orc_power(orc_ctx*, int member, double z, double* P1, double* P2);
/* Internal heat source of P:118 (Eq. 8), q = sum_j alpha_j I_j + beta_j I_j^2 with I_j = eps0 c n_j |A_j|^2/2
 * (P:120), sampled on nq (1 <= nq <= nz) planes along z: plane k holds the mean of q evaluated on the
 * real-space fields right before and right after the nonlinear step of z-step n_k = floor((2k+1) nz / (2 nq)),
 * i.e. q at z = z_{n_k} + dz/2 to second order in dz (the middle of the cell [k L/nq, (k+1) L/nq) rounded to
 * a step; reading G27 in DESIGN.md: the paper does not say where along a step the source is taken).  Q: host double [batch][nq][ny][nx], borrowed, filled by the next
 * orc_propagate (scheme 0 only); NULL switches it off.                                                */
int  orc_set_heat_output(orc_ctx*, double* Q, int nq);
/* Whole history of one member: out[(nz+1)][2] = {P1(z_n), P2(z_n)}, n = 0..nz.                       */
int  orc_power_history(orc_ctx*, int member, double* out);
void orc_destroy(orc_ctx*);

/* Gaussian input of P:104 (Eq. 6) generalised to any focus by P:95-100 (Eq. 5, tau0 = -focus_z/zR)
 * with |A_F0|^2 = 4P/(eps0 c n1 pi w0^2) (G17).  out: complex128 [ny][nx] for member `member`.      */
int  orc_gaussian_input(const orc_grid*, const orc_crystal*, const orc_beam* beam, double* out);

/* Stand-alone transforms for the pins.  data: complex128 [ny][nx] interleaved.  sign = -1 forward
 * (kernel e^{-i...}, unnormalised), +1 inverse (kernel e^{+i...}, divided by nx*ny).  P:340 (Eq. A.2). */
int  orc_fft2(double* data, int ny, int nx, int sign);
int  orc_dft2_brute(const double* in, double* out, int ny, int nx, int sign);

int  orc_num_threads(void);
void orc_set_num_threads(int n);   /* OpenMP threads of the following calls (timing the oracle on one core) */

#ifdef __cplusplus
}
#endif
#endif
