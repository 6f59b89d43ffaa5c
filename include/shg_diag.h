/*
 * shg_diag.h -- C ABI of libshg_diag: measuring equipment of bench.py, kept OUT of libshg (the product library holds
 * the method's calls only, include/shg.h).  Built by paper_2410_04994_b200/build.py from csrc/shg_diag.cu.
 * Both calls allocate and free two small device buffers, run on the legacy default stream and wait for the result.
 * Returns: SHG_DIAG_OK, SHG_DIAG_EINVAL (NULL argument), SHG_DIAG_ECUDA (a CUDA call failed, e.g. no device).
 */
#ifndef SHG_DIAG_H
#define SHG_DIAG_H

#ifdef __cplusplus
extern "C" {
#endif

#define SHG_DIAG_OK       0
#define SHG_DIAG_EINVAL (-1)
#define SHG_DIAG_ECUDA  (-3)

/* Measured fp32 pipe peak of the current device: a register-only FFMA kernel (16 independent chains per
 * thread, 512 threads per SM) timed with CUDA events.  *tflops receives 2 flops per FFMA lane-op over the
 * elapsed time.  It is the denominator of bench.py's "alu" roofline (nominal: SMs x 128 lanes x 2 x clock). */
int shg_measure_fp32_peak(double* tflops);

/* The same measurement with three distinct register operands per FFMA (no operand reuse between neighbouring
 * instructions), which is what the butterflies and the RK4 stages of this library look like to the register file. */
int shg_measure_fp32_peak_distinct(double* tflops);

#ifdef __cplusplus
}
#endif
#endif
