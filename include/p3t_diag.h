/* include/p3t_diag.h -- DIAGNOSTICS, not part of the product library: micro-benchmarks of the FP32 pipe of the
 * device, and the measurement / fault-injection knobs of a context, exported by the separate libp3t_diag.so
 * (paper_2110_11658_b200/csrc/p3t_pipebench.cu, p3t_diagknobs.cu).  bench.py uses them
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
 * FFMA, [5] eight FMUL2 + two MUFU.RSQ, [6] MUFU.RSQ, [7] FFMA with three distinct registers, and, if n_out >= 9, [8] FFMA2 with three distinct register pairs one of
 * which is the same in consecutive instructions.  sm_clock_mhz /
 * num_sms: HOST, may be NULL (the device's nominal maximum clock, which the cycle counts assume).
 * Returns 0, -1 (bad argument), -3 (allocation) or -4 (CUDA failure).  Synchronises the device; ~20 ms. */
int p3t_diag_pipe_bench(int device, double* cycles_out, int n_out, double* sm_clock_mhz, int* num_sms);

/* Knobs of one context (a p3t_ctx* from p3t_create, passed as void*).  libp3t.so itself reads no environment variable
 * and exports no such setter: a host integrator cannot switch these on by accident.  libp3t_diag.so is built from the
 * same p3t_internal.cuh as libp3t.so and writes the fields directly; use the two libraries of ONE build together.
 * Both return 0 or -1 (null context, value out of range) and take effect at the next force call.
 *
 * p3t_diag_set_overlap: overlap 1 (default) = the list walk runs beside the force kernel, 0 = one after the other
 * (how bench.py times the force kernel with the SMs to itself); walk_ctas_per_sm = CTAs per SM left to the walk while
 * they overlap (default 2; <= 0 keeps the current value). */
int p3t_diag_set_overlap(void* ctx, int overlap, int walk_ctas_per_sm);
/* p3t_diag_set_fault: fault injection for the tests of the repair and error paths, bits: 1 = every force warp gives
 * up waiting for the walker at once (those groups are repaired), 2 = no spill space behind the walk stack (a wide-open
 * walk then reports stack_overflow), 4 = p3t_step_host meets a CUDA failure while its force call is in flight.  0 = off. */
int p3t_diag_set_fault(void* ctx, int bits);

#ifdef __cplusplus
}
#endif
#endif
