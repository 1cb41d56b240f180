/* grx_probe.h -- measurement probes of bench.py (libgrx_probe.so).  NOT part of the product ABI (include/grx.h): nothing a
 * user of the library links or calls; bench.py loads it to put the FP64 roofline denominator and the issue-cost table next
 * to the kernel's numbers (profiles/r3_issue_probe.md). */
#ifndef GRX_PROBE_H
#define GRX_PROBE_H
#ifdef __cplusplus
extern "C" {
#endif

/* Throughput of a dependent-chain-free DFMA loop on the whole device: launches the micro-benchmark kernel once (iters FMAs
 * per chain, 8 chains per thread, one resident wave) and writes a checksum to `sink` (DEVICE pointer to one double).
 * flops_out (HOST) receives the flop count of that launch; time it with CUDA events on `cuda_stream`.  Returns 0 or a
 * cudaError_t value. */
int grx_probe_dfma_peak(int iters, double* sink, double* flops_out, void* cuda_stream);

/* Issue probe: one launch of a dependency-free FP64 loop over the whole device (4 warps per scheduler, 16 independent
 * values r[0..15] per thread, every instruction reads values written 9 or more instructions earlier) in one of the
 * operand / neighbour patterns below.  fp64_instr_out (HOST): FP64 thread-instructions of the launch; divide by the event
 * time, the SM count and the clock to get FP64 lanes per clock per SM (64 = the nominal peak).
 *   0  r[i] = fma(r[i], m, c), m and c fixed registers      1  r[i] = fma(r[i+1], r[i+7], r[i+11])  (same index parity)
 *   2  r[i] = r[i+1] * r[i+7]                               3  pattern 2 + one independent IMAD per multiply
 *   4  pattern 2 + one STS.64 per multiply                  5  pattern 2 + one SHFL per multiply
 *   6  r[i] = fma(r[i+1], r[i+2], r[i+4])  (mixed parity)   7  r[i] = fma(r[i+1], r[i+2], r[i])  (accumulate in place)
 *   8  r[i] = fma(r[i+1], r[s], r[i+4]), s shared by two consecutive instructions (operand reuse)
 *   9  r[i] = fma(r[i+1], r[i+2], k), k a kernel parameter (constant-bank operand)
 * Returns 0, or a cudaError_t value (cudaErrorInvalidValue for an unknown mode). */
int grx_probe_fp64_issue(int mode, int iters, double* sink, double* fp64_instr_out, void* cuda_stream);
int grx_probe_fp64_issue_modes(void);

#ifdef __cplusplus
}
#endif
#endif
