/* include/lrdmc_probe.h -- C-ABI of liblrdmc_probe.so: FP64 peak micro-benchmarks, the roofline denominators of bench.py.
 *
 * NOT part of the product library (liblrdmc.so does not contain them): SURVEY.md 8(d) asks to "measure DFMA and DMMA peaks on the
 * box" because MEASURED_PEAKS.json carries no FP64 figure.  Host outputs, TFLOP/s; each call launches a few short kernels on the
 * current device's default stream and synchronises.  Return 0 on success, -4 on a CUDA error.
 */
#ifndef LRDMC_PROBE_H
#define LRDMC_PROBE_H
#ifdef __cplusplus
extern "C" {
#endif
/* independent FP64 FMA chains (8 per thread), mma.sync m8n8k4 f64 chains, and both issued together */
int lrdmc_measure_fp64_peaks(double *dfma_tflops, double *dmma_tflops, double *mixed_tflops);
/* the two instruction forms that set the real ceiling of the path (dispatch model):
 * dfma_3reg_tflops -- FMAs whose three source operands are three different registers (3 dispatch cycles instead of 2);
 * dfma_alu_tflops  -- two-register FMAs each followed by two independent integer ALU instructions of the same warp
 *                     (FP64 flop only).  The second pointer may be NULL. */
int lrdmc_measure_fp64_operand_peak(double *dfma_3reg_tflops, double *dfma_alu_tflops);
/* FMAs with ONE source register shared with the neighbouring FMAs (acc[i] += g[i] * b; operand-reuse cache): between the 2- and the 3-register forms */
int lrdmc_measure_fp64_shared_operand_peak(double *dfma_shared1_tflops);
#ifdef __cplusplus
}
#endif
#endif
