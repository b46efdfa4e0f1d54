/* mlcc_probe.h — measurement probes of libmlcc.so.  NOT part of the product interface: include/mlcc.h does not
 * include this file.  bench.py uses these calls for the denominators of its "alu" roofline
 * (MEASURED_PEAKS.json has no FP64 entry) and for the issue model in DESIGN.md "Measured issue model".
 * Conventions as in mlcc.h: `stream` is a cudaStream_t as void*, return value mlcc_status.            */
#ifndef MLCC_PROBE_H_
#define MLCC_PROBE_H_

#ifdef __cplusplus
extern "C" {
#endif

/* Runs a dependent-free DFMA loop on every SM for about `ms_target` milliseconds and returns the FP64 FMA
 * rate reached, in TFLOP/s (2 flop per FMA) through *out_tflops (host).  Synchronises `stream`.         */
int mlcc_fp64_peak(double ms_target, double *out_tflops, void *stream);

/* The same loop with other operand forms,
 * rate returned as 2 x FP64 instructions per second / 1e12 (so form 0 equals mlcc_fp64_peak).
 *   form 0: DFMA, two distinct register sources (the peak form)
 *   form 1: DFMA, three distinct register sources
 *   form 2: DADD, two distinct register sources
 *   form 3: form 0 interleaved 1:1 with packed FP32 FMAs (fma.f32x2, three 64-bit sources); the
 *           rate counts the FP64 instructions only
 *   form 4: packed FP32 FMAs alone (fma.rn.f32x2): the rate is FP32 flop/s / 1e12 (2 lanes x 2 flop per
 *           instruction and thread), the denominator for work that runs in packed FP32
 * Synchronises `stream`.  Errors: INVALID_ARG, CUDA.                                              */
int mlcc_fp64_issue_probe(int form, double ms_target, double *out_rate, void *stream);

#ifdef __cplusplus
}
#endif
#endif /* MLCC_PROBE_H_ */
