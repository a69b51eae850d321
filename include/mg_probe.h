/* mg_probe.h — C ABI of libmg_probe.so: on-box microbenchmarks that bench.py prints next to the nominal ALU peak.
 * Measurement tooling, deliberately NOT in the product library libmg_b200.so (include/mg.h).
 *
 * SURVEY.md §8(d) asks for the FP64/FP32 lane counts behind the "alu" roofline to be confirmed on the box with an
 * FMA-chain microbenchmark; DESIGN.md §6 uses the three modes to show how the way an FMA is fed decides its rate on
 * sm_100a. */
#ifndef MG_PROBE_H
#define MG_PROBE_H
#ifdef __cplusplus
extern "C" {
#endif
/* Measured FMA throughput of `device` in TFLOP/s (FMA = 2), register-only kernels, synchronous, ~0.1 s.
 *   precision 0 = FP64, 1 = FP32
 *   mode 0 = chains with one register operand and two loop constants per FMA
 *        1 = three distinct register operands per FMA (a product of two loaded operands accumulated into a third)
 *        2 = the FP64 tensor-core instruction mma.sync m8n8k4 (precision must be 0)
 * Returns 0, -1 (bad argument) or -3 (CUDA error / no such device). */
int mg_probe_alu(int precision, int device, int mode, double* h_tflops_out);
#ifdef __cplusplus
}
#endif
#endif
