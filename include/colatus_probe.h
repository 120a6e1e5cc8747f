/*
 * colatus_probe.h -- C ABI of libcolatus_probe: device microbenchmarks behind DESIGN.md 6.1-6.2.
 *
 * NOT part of the product library: libcolatus.so does not contain, link or need these kernels.  They exist so
 * that the denominator of the "alu" roofline (FP32 FMA peak, which MEASURED_PEAKS.json does not carry) and the
 * issue rules DESIGN.md quotes can be re-measured from committed code.  bench.py and tests/test_gpu_probe.py
 * are the only callers.  Self-contained: each call selects `device`, allocates a 256-byte sink, runs on the
 * default stream, synchronises and frees.  Returns 0, or a negative value on a CUDA error / bad argument.
 */
#ifndef COLATUS_PROBE_H
#define COLATUS_PROBE_H

#ifdef __cplusplus
extern "C" {
#endif

/* Plain FP32 FMA throughput of a register-only loop (packed = 0: scalar FFMA; 1: FFMA2 / fma.rn.f32x2):
 * *tflops = 2 flop x lane-FMAs / best of three timed launches (16 waves of 8 CTAs/SM, 8 independent chains
 * per thread); *ms_out (may be NULL) = that launch's duration. */
int colatus_probe_fp32_peak(int device, int packed, double *tflops, double *ms_out);

/* Issue-rule probes: register-only loops whose body is one group of 12 packed FP32 ops (the FP work of one
 * packed pair-interaction of eq. (1)) plus
 *   mode 0: nothing                     1: 2 MUFU.RSQ                2: 2 integer adds
 *   mode 3: (12 accumulates a = w*d + a in triples sharing w: the operand pattern of eq. (1)'s sums)
 *   mode 4: one broadcast LDS.128       5: 24 scalar FFMA + 2 MUFU.RSQ instead of the packed ops
 *   mode 6: as 3 but ordered so that w changes every instruction (no operand reuse possible)
 *   mode 7: 12 packed ops + 6 DFMA (FP64 pipe next to the FP32 pipe)
 * *cycles_per_group = SMSP cycles one group costs (launch time x max SM clock / groups per SMSP;
 * 24 = FMA pipe saturated). */
int colatus_probe_pipe(int device, int mode, double *cycles_per_group);

#ifdef __cplusplus
}
#endif
#endif /* COLATUS_PROBE_H */
