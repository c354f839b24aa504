/* include/p3t_diag.h -- DIAGNOSTICS, not part of the product library: micro-benchmarks of the FP32 pipe of the
 * device, exported by the separate libp3t_diag.so (paper_2110_11658_b200/csrc/p3t_pipebench.cu).  bench.py uses them
 * to state the ALU roofline of the force kernel (MEASURED_PEAKS.json holds no FP32 figure) and
 * DESIGN.md section 6 to account for the kernel's instruction mix.  Nothing in libp3t.so depends on this.
 */
#ifndef P3T_DIAG_H
#define P3T_DIAG_H
#ifdef __cplusplus
extern "C" {
#endif

/* cycles_out: HOST double[n_out >= 8], SM-clock cycles per SM sub-partition of: [0] FFMA (best case: operands in
 * the reuse cache), [1] FFMA2 with two distinct register pairs, [2] FFMA2 with three, [3] FMUL2, [4] one FMUL2 + one
 * FFMA, [5] eight FMUL2 + two MUFU.RSQ, [6] MUFU.RSQ, [7] FFMA with three distinct registers.  sm_clock_mhz /
 * num_sms: HOST, may be NULL (the device's nominal maximum clock, which the cycle counts assume).
 * Returns 0, -1 (bad argument), -3 (allocation) or -4 (CUDA failure).  Synchronises the device; ~20 ms. */
int p3t_diag_pipe_bench(int device, double* cycles_out, int n_out, double* sm_clock_mhz, int* num_sms);

#ifdef __cplusplus
}
#endif
#endif
