/*
 * shg.h -- C ABI of libshg: B200-native (sm_100a) split-step Fourier propagation of the coupled
 * fundamental (FH, A1) and second-harmonic (SH, A2) slowly-varying envelopes through a chi(2) crystal,
 * the computation that dominates cuSHG (arxiv/paper_2410_04994).
 *
 * "P:n" cites line n of the paper text; "G<k>" a reading listed in DESIGN.md §3.
 *
 * What one call to shg_propagate computes, per batch member (members are independent):
 *   for n = 0 .. nz-1:                                  dz = L/nz
 *     A_j <- F^-1{ exp(-i(kx^2+ky^2)(dz/2)/(2k_j) - alpha_j dz/4) F{A_j} }, j = 1,2    (G3)
 *            (with walk-off angles: one more factor exp(-i kx tan(rho_j) dz/2), G21)
 *     one classical RK4 step of length dz, independently at every (x,y), of              (Eq. 2, G2, G5)
 *        dA1/dz = i kappa1 A2 conj(A1) e^{-i phi} - (beta1/2) I1 A1
 *        dA2/dz = i kappa2 A1^2        e^{+i phi} - (beta2/2) I2 A2,   I_j = eps0 c n_j |A_j|^2 / 2
 *        phi(x,y,z) = int_0^z dk dz',  dk = dk0 + ddk_dT (T(x,y,z) - T_pm)                (Eq. 3; north_star)
 *     the same linear half-step again                                                     (order L/2-N-L/2)
 *     P_j(z_{n+1}) = (eps0 c n_j / 2) dx dy sum |A_j|^2
 *   (the two half-steps of neighbouring z-steps are applied as one full step; this is exact.)
 *
 * Conventions
 *   - SI units.  Fields are complex fp32, interleaved (re, im), layout [batch][ny][nx], x fastest.
 *     Grid point (iy, ix) sits at x = (ix - nx/2) lx/nx, y = (iy - ny/2) ly/ny (periodic FFT grid, G11).
 *   - Every pointer argument says HOST or DEVICE.  Device pointers must be 16-byte aligned and belong to
 *     the current CUDA device; the caller owns them.  The library owns its tables, the phase accumulator
 *     phi, the power history and staging buffers, freed in shg_destroy.  They are allocated in shg_create,
 *     except: the device copy of a host temperature array (shg_set_temperature_host, on first use or growth),
 *     the two staging fields of shg_propagate_host (on its first call), the plane map of shg_set_heat_output
 *     and the trace buffer of SHG_OPT_TRACE.  shg_propagate (device pointers) allocates no memory; the first one
 *     that uploads a large host temperature array creates the library's copy stream and its chunk events.
 *   - shg_propagate enqueues work on the given stream and returns without waiting.  shg_synchronize,
 *     shg_power and shg_power_history synchronise that stream and report a failed run (SHG_ECUDA).
 *   - Every call returns SHG_OK (0) or a negative code; nothing aborts or throws across the ABI.
 *   - There is no CPU fallback: without a CUDA device every call that needs one returns SHG_ECUDA.
 */
#ifndef SHG_H
#define SHG_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define SHG_OK       0
#define SHG_EINVAL  (-1)   /* NULL / out-of-range argument, unsupported grid size                     */
#define SHG_ESTATE  (-2)   /* call made in the wrong state (temperature not set, power before run)   */
#define SHG_ECUDA   (-3)   /* a CUDA call failed; shg_strerror(SHG_ECUDA) carries the CUDA message    */
#define SHG_ENOMEM  (-4)   /* host or device allocation failed                                        */
#define SHG_ELIMIT  (-5)   /* size beyond the fixed capacity of a static-scratch entry point          */

typedef struct shg_ctx shg_ctx;   /* opaque, owned by the library */

/* Transverse grid, z discretisation, temperature planes, batch capacity. */
typedef struct {
    int32_t nx, ny;   /* powers of two in {64,128,256,512,1024}; nx != ny is allowed                 */
    int32_t nz;       /* z-steps >= 1                                                                */
    int32_t nzt;      /* temperature planes: 0 = uniform scalar; 1 = one plane used at every z;
                         >= 2 = planes at z_k = k L/(nzt-1), linearly interpolated to the step nodes
                         z_n = n dz: s = n (nzt-1)/nz, k = min(floor(s), nzt-2), T = (1-f)T[k] + f T[k+1] (G15) */
    int32_t batch;    /* capacity: number of independent simulations one propagate may carry         */
    int32_t record_every; /* power history stride in z-steps: nodes n = 0, r, 2r, .. (< nz) and n = nz are
                         recorded; 0 or 1 = every node.  shg_history_length / shg_history_nodes describe it. */
} shg_grid;

/* Crystal constants (Eq. 2; Eq. 3-4 in the linearised form the north_star fixes). */
typedef struct {
    double L, lambda1, n1, n2, d_eff;   /* m, m (FH vacuum wavelength; SH is lambda1/2), -, -, m/V    */
    double dk0, ddk_dT, T_pm;           /* rad/m, rad/(m K), same unit as T                           */
    double alpha1, alpha2;              /* linear intensity absorption, 1/m, >= 0                     */
    double beta1, beta2;                /* two-photon absorption, m/W, >= 0 (the power sums are kept in
                                           fixed point scaled to the input power: no gain media)      */
    double rho1, rho2;                  /* spatial walk-off angles along x, rad: term tan(rho) dA/dx of P:387
                                           (the paper's runs use 0; P:314 names it for birefringent crystals) */
} shg_crystal;

/* One batch member's beam and transverse window (Eq. 5-6). */
typedef struct {
    double P, w0, focus_z;   /* W; m, 1/e field radius at the waist; focus distance from the entrance face, m.
                                Used only by shg_gaussian_input.                                       */
    double lx, ly;           /* transverse window, m (dx = lx/nx).  Members may differ (parameter sweeps). */
} shg_beam;

/* Options for shg_set_option. */
#define SHG_OPT_PERSISTENT 1   /* 1 (default): one persistent cooperative kernel runs the whole z-loop with
                                  device-wide barriers between the row and column passes (square grids; if
                                  the device cannot make all its CTAs co-resident -- SMs held by another
                                  context, MPS / MIG -- the call falls back to the scheme of value 0);
                                  0: two ordinary kernel launches per z-step (any nx, ny).  Same device code,
                                  bit-identical fields.                                                  */
#define SHG_OPT_PRECISE    2   /* 1 (default): every reused constant (FFT twiddles, propagator tables) is an
                                  fp32 hi+lo pair whose lo part enters the FMA addend, so constant rounding
                                  does not accumulate linearly over thousands of z-steps; 0: plain fp32.  */

#define SHG_OPT_TRACE      3   /* value = number of leading z-steps whose phase timeline the persistent kernel
                                  records (0 = off, default; <= 4096): per step, CTA and device-wide barrier
                                  (0 = after the row pass, 1 = after the column pass) four int64: SM clock when
                                  the CTA finished its share of the pass, SM clock when the barrier released it,
                                  %globaltimer (ns) at release, SM id.  Read back with shg_read_trace.            */
#define SHG_OPT_ACQUIRE_FENCE 4 /* persistent kernel, acquire side of the device-wide barrier.  2 (default): the poll
                                  ends with an ld.acquire.gpu of the barrier counter (pairs with the arrivals'
                                  red.release.gpu; conforms to the PTX memory model); 1: a gpu-scope fence.acq_rel
                                  after a relaxed poll (same guarantee).  Bit-identical results in both modes.  (0, no
                                  acquire at all with the fields read by L2-only loads, is outside the memory model
                                  and is refused with SHG_EINVAL unless the library is built with
                                  -DSHG_ALLOW_UNFENCED for a measurement; DESIGN.md 5.5 has round 2's numbers.)       */
#define SHG_OPT_UNDEPLETED 5    /* 1: drop the coupling term of dA1/dz (the pump only diffracts and is absorbed), the
                                  "dPump = 0" check against Boyd-Kleinman of P:292; 0 (default): full Eq. 2.       */
#define SHG_OPT_SCHEME     6    /* 0 (default): L/2 - N(dz) - L/2 with neighbouring half-steps merged (north_star);
                                  1: the paper's own ordering N(dz/2) - L(dz) - N(dz/2), Eq. 14-15:
                                  two RK4 half-steps per z-step, powers summed at the true nodes.  Variant for
                                  comparison with the paper's scheme (differs from scheme 0 by O(dz^2)); needs
                                  SHG_OPT_PRECISE = 1 and no heat output (else shg_propagate returns SHG_EINVAL). */

#define SHG_OPT_SPIN_LIMIT 7    /* persistent kernel: a CTA that waits longer than `value` million SM clocks at a
                                  device-wide barrier raises the status word (reported by shg_synchronize /
                                  shg_power*) instead of hanging the GPU.  Default 4000 (~2 s); 0 = wait forever
                                  (use under profilers / sanitizers that serialise or replay the kernel).          */
#define SHG_OPT_TABLES_SMEM 8   /* 1 (default): a single simulation's persistent kernel keeps the propagator tables
                                  hx, hy in shared memory; 0: reads them through L1 like the batched runs do.       */
#define SHG_OPT_CLUSTER    9    /* small grids (nx = ny <= 128).  1 (default): when every member of the propagate fits
                                  one co-resident wave of thread-block clusters, the whole run (opening half-step,
                                  z-loop, closing half-step) is ONE launch of k_cluster: one cluster of 16 (else 8)
                                  CTAs per member, the fields resident in distributed shared memory, the 2-D
                                  transform's transposition as bulk asynchronous copies between the CTAs' shared
                                  memories signalled on mbarriers, no device-wide barrier; 0: never; 8 or 16: that
                                  cluster size whenever the grid size allows, even if the clusters run in several
                                  waves.  64-point lines use the other kernels' line transform: bit-identical fields
                                  and powers.  128-point lines are transformed over twice the lanes, in another
                                  summation order: fields and powers agree with the other kernels to fp32 rounding
                                  (rel. L2 ~1e-6 per propagate, tested < 2e-6), NOT bit for bit.  Since mode 1 picks
                                  the kernel from the batch size and from how many clusters the device can hold, the
                                  last bits of a 128 x 128 member may differ between a single run and the same member
                                  inside a large batch; set 0 where bit-reproducibility across batch sizes matters.  */

#define SHG_OPT_PIPELINE   10   /* batched runs (batch >= 2) in the persistent kernel.  The members are split into
                                  two groups whose row and column phases interleave, every device-wide barrier is
                                  split-phase (arrive when a phase is done, wait one phase later), and no CTA-wide
                                  barrier remains (k_persist_pipe): the barriers' latency and the skew between CTAs
                                  stop nothing.  1 (default): when a warp has at least two row items per phase;
                                  2: whenever batch >= 2; 0: never (one pair of device-wide barriers per z-step for
                                  the whole batch, k_persist).  Not used with a heat output, SHG_OPT_SCHEME = 1 or
                                  SHG_OPT_TRACE.  Same device code per row and strip: bit-identical results.      */

/* beams: HOST array [grid->batch].  *out receives the context. */
int shg_create(const shg_grid* grid, const shg_crystal* crystal, const shg_beam* beams, shg_ctx** out);

int shg_set_option(shg_ctx* ctx, int option, int value);

/* Temperature field.  nzt == 0: T is ignored (may be NULL) and every point has temperature T_uniform.
 * A new T_uniform alone costs two small kernels at the head of the next shg_propagate, on that call's stream: no host
 * copy and no host wait, so a sweep over T_uniform enqueues propagate after propagate without synchronising.
 * (shg_set_option(SHG_OPT_UNDEPLETED | SHG_OPT_PRECISE) rebuilds all tables: the next propagate then waits for the
 * context's last one and uploads them with blocking copies.)
 * nzt >= 1: T is a DEVICE fp32 array [per_member ? batch : 1][nzt][ny][nx]; it is BORROWED (not copied)
 * and must stay valid and unchanged until every propagate that uses it has completed. */
int shg_set_temperature(shg_ctx* ctx, const float* T_device, double T_uniform, int per_member);

/* Same, from a HOST array: copied (asynchronously when the memory is pinned) into a library-owned device buffer that is
 * allocated on first use and reused afterwards.  An array in pageable memory, and any small array, is copied on
 * `cuda_stream` during the call: the caller may free or reuse a pageable buffer as soon as the call returns.  One array
 * shared by all members of 32 MB or more in PAGE-LOCKED memory (cudaMallocHost / cudaHostRegister / managed) is
 * uploaded by the NEXT shg_propagate[_host] instead, in chunks of planes on
 * the library's own copy stream, behind that call's field uploads: the persistent kernel of a single simulation is
 * launched once per chunk, over the z-steps whose planes the chunk completes (a z-step reads only the planes around
 * its two nodes), so the transfer of chunk c + 1 runs under the z-steps of chunk c; every other kernel waits for the
 * last chunk.  A page-locked T_host must therefore stay valid and unchanged until that propagate has completed (as any
 * buffer handed to an asynchronous copy must). */
int shg_set_temperature_host(shg_ctx* ctx, const float* T_host, double T_uniform, int per_member,
                             void* cuda_stream);

/* Propagate `batch` (<= capacity) members from z = 0 to z = L.
 * A1_in, A2_in, A1_out, A2_out: DEVICE complex fp32 [batch][ny][nx].  A1_in may be NULL: the pump is then the
 * Gaussian of Eq. 6 / Eq. 5 of every member's beam (as shg_gaussian_input writes it; SHG_EINVAL if a
 * beam has w0 <= 0).  A2_in may be NULL (zeros: the configs' A_SH(0) = 0).  In-place (A1_out == A1_in and/or
 * A2_out == A2_in, the same pointer) is allowed; any other overlap between the four buffers is SHG_EINVAL.
 * The outputs are also the kernels' working storage.
 * cuda_stream: a cudaStream_t (NULL = the legacy default stream). */
int shg_propagate(shg_ctx* ctx, const void* A1_in, const void* A2_in, void* A1_out, void* A2_out,
                  int batch, void* cuda_stream);

/* Same with HOST buffers (pinned memory makes the copies asynchronous): copies the inputs to
 * library-owned device buffers, propagates, copies both outputs back, all on `cuda_stream`.  Returns
 * after enqueueing; synchronise the stream (or call shg_power) before reading the outputs. */
int shg_propagate_host(shg_ctx* ctx, const void* A1_in, const void* A2_in, void* A1_out, void* A2_out,
                       int batch, void* cuda_stream);

/* Internal heat source of P:118 (Eq. 8), q = sum_j alpha_j I_j + beta_j I_j^2 with I_j = eps0 c n_j |A_j|^2 / 2
 * (P:120), in W/m^3 -- the quantity the paper's thermal solver consumes (S§8(f) rank 1).  Q: DEVICE fp32
 * [batch capacity][nq][ny][nx], 1 <= nq <= nz, BORROWED: every later shg_propagate fills it on its stream.
 * Plane k holds the mean of q on the real-space fields right before and right after the nonlinear step of
 * z-step n_k = floor((2k+1) nz / (2 nq)), i.e. q at z = z_{n_k} + dz/2 to second order in dz: the middle of
 * the cell [k L/nq, (k+1) L/nq) rounded to a step (reading G27 of DESIGN.md).  Q == NULL switches it off.
 * It is written from the epilogue of the nonlinear step: 2 extra sweeps over a row on nq of the nz steps. */
int shg_set_heat_output(shg_ctx* ctx, float* Q_device, int nq);

/* Wait for the last propagate of this context and report how it ended: SHG_OK, or SHG_ECUDA when the stream
 * failed or a device-wide barrier of the persistent kernel timed out (the outputs are then invalid).  Call it
 * (or shg_power*) before trusting A1_out / A2_out of a run whose history you do not read.  The timeout flag is
 * sticky: it survives later propagates of the context (whose kernels then stop at their first barrier) and is cleared
 * only by the call that reports it, so the error covers every propagate enqueued since the last successful
 * shg_synchronize / shg_power*. */
int shg_synchronize(shg_ctx* ctx);

/* Power (W) of both fields of `member` at the RECORDED node nearest to z (step nodes z_n = n L/nz; recorded:
 * shg_grid.record_every).  The SH efficiency is derived by the caller: eta = P2(L) / (P1(0) + P2(0))  (P:288,
 * G16).  The sums behind these numbers are accumulated in fixed point (integers): they are bit-reproducible
 * from run to run, and identical between launch schemes whose fields are identical (all of them except the cluster
 * kernel on 128-point lines, see SHG_OPT_CLUSTER). */
int shg_power(shg_ctx* ctx, int member, double z, double* P1, double* P2);

/* Number of recorded nodes (ceil(nz / record_every) + 1), and their step indices n (HOST int32 array of that
 * length: 0, r, 2r, .., nz). */
int shg_history_length(const shg_ctx* ctx);
int shg_history_nodes(const shg_ctx* ctx, int32_t* nodes);

/* Whole history of `member`: out is a HOST array [shg_history_length()][2] = {P1(z_n), P2(z_n)}. */
int shg_power_history(shg_ctx* ctx, int member, double* out);

/* Fill A1 (DEVICE complex fp32 [batch][ny][nx]) with the Gaussian pump of Eq. 6 / Eq. 5 of every
 * member's beam: A = A0/(1+i tau0) exp(-(x^2+y^2)/(w0^2 (1+i tau0))), tau0 = -focus_z/zR, zR = k1 w0^2/2,
 * |A0|^2 = 4P/(eps0 c n1 pi w0^2) (G17). */
int shg_gaussian_input(shg_ctx* ctx, void* A1_device, int batch, void* cuda_stream);

/* Device timing of the z-loop: with timing enabled, shg_propagate records CUDA events on its stream right
 * before and after the main-loop kernel(s) (the persistent kernel, or the 2 nz per-pass launches); the
 * opening / closing half-step launches are outside.  shg_last_main_loop_ms synchronises the stream. */
int shg_enable_timing(shg_ctx* ctx, int on);
int shg_last_main_loop_ms(shg_ctx* ctx, float* ms);

/* Phase timeline of the last shg_propagate run with SHG_OPT_TRACE (persistent kernel only).
 * out: HOST int64 [*steps][*grid][2][4] (see SHG_OPT_TRACE); out == NULL only queries *steps and *grid.
 * Synchronises the stream of the last propagate. */
int shg_read_trace(shg_ctx* ctx, long long* out, int* steps, int* grid);

/* Number of kernels the last shg_propagate / shg_propagate_host launched. */
int shg_last_launch_count(const shg_ctx* ctx);

/* Cluster size (8 or 16) when the last propagate ran in the cluster kernel (SHG_OPT_CLUSTER), else 0. */
int shg_last_cluster_size(const shg_ctx* ctx);

/* Which kernel ran the z-loop of the last propagate: 0 = two launches per z-step (k_row + k_col), 1 = k_persist,
 * 2 = k_persist_flat (sparse launch), 3 = k_persist_pipe (SHG_OPT_PIPELINE), 4 = k_cluster, 5 = k_persist_paper
 * (SHG_OPT_SCHEME = 1).  Lets bench.py and the tests name what they measured. */
int shg_last_kernel(const shg_ctx* ctx);

/* The power integral for callers that must not allocate.
 *
 * Everything else in this header hangs off a context, and shg_create allocates device memory.  That rules the library
 * out for code that runs where cudaMalloc / cudaFree may not be called: a hook inside another allocator or memory pool
 * (an allocation there re-enters the pool or blocks on its lock), a plug-in whose host application owns all device
 * memory and hands out fixed buffers, a latency-critical loop that cannot afford the driver's allocation lock or the
 * device-wide wait inside cudaFree, a job sized to the last byte of HBM.  This one call needs no context and calls
 * no cudaMalloc, cudaFree, nor any other routine that allocates:
 *
 *     P[b][j] = scale_j * sum over (iy, ix) of |A_j[b][iy][ix]|^2,   j = 1, 2,  b = 0 .. batch-1
 *
 * i.e. the power of both fields in W when scale_j = (eps0 c n_j / 2) dx dy -- the quantity shg_power reports at
 * z = 0 for the inputs of a propagate, summed the same way (chunks of a member in double in a fixed order, then the
 * chunk sums in chunk order: the result does not depend on scheduling and is the same bits on every call).
 *
 *   A1_device, A2_device  DEVICE complex fp32 [batch][ny][nx], 8-byte aligned, read only; A2_device may be NULL
 *                         (then P[b][1] = 0).  nx, ny >= 1, any size (not only the powers of two of shg_grid).
 *   P_device              DEVICE double [batch][2], 8-byte aligned, written by the kernel on `cuda_stream`; the caller
 *                         owns it (and every other buffer) and reads it after synchronising the stream.
 *   batch                 1 .. SHG_STATIC_MAX_BATCH.  More members than that: SHG_ELIMIT, nothing is enqueued --
 *                         split the members over several calls.
 *
 * Where the scratch lives.  The chunk sums and the per-member tickets of the two-level sum sit in a fixed array of
 * SHG_STATIC_SCRATCH_BYTES (257 KiB) inside the library's device image.  Every GPU on which the library is used holds
 * that array from the moment the image is loaded there until the process exits, whether or not this call is used.
 *
 * First call on a device.  The first call made with a given device current looks up the array's address on that
 * device (cudaGetSymbolAddress; this may also be what makes the CUDA runtime load the library's device image) and
 * keeps it; later calls on that device only enqueue a 1 KiB memset of the tickets and one kernel.  Make that first
 * call during set-up, with the right device current, and before you begin any stream capture on it.
 *
 * Sharing.  All calls on one device use the same array, and it keeps what the last call left in it (the call clears
 * the part that must start at zero).  Two calls that can run on the GPU at the same time -- different streams without
 * an event between them, or two host threads each with their own stream -- race on it and both results are
 * undefined.  Calls on one stream, or ordered by events, are safe.
 *
 * Returns SHG_OK after enqueueing (it does not wait), SHG_EINVAL (NULL / misaligned pointer, size < 1), SHG_ELIMIT,
 * or SHG_ECUDA (shg_strerror has the CUDA message). */
#define SHG_STATIC_MAX_BATCH     256
#define SHG_STATIC_SCRATCH_BYTES 263168
int shg_field_power_static(const void* A1_device, const void* A2_device, int nx, int ny, int batch,
                           double scale1, double scale2, double* P_device, void* cuda_stream);

void shg_destroy(shg_ctx* ctx);

const char* shg_strerror(int code);

#ifdef __cplusplus
}
#endif
#endif
