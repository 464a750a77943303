/* nep_b200_measure.h -- MEASUREMENT helpers of libnep_b200.so.  They are not part of the boundary of SURVEY.md 8(b)
 * (include/nep_b200.h): bench.py uses them for the roofline entry of its JSON line (per-phase CUDA-event timing on the
 * launching stream, kernel-launch count, the measured FP32 peak and the attainable ceilings of k_main's inner-loop
 * patterns).  Same conventions as nep_b200.h: plain C, device pointers, NEP_OK or a negative nep_error. */
#ifndef NEP_B200_MEASURE_H
#define NEP_B200_MEASURE_H

#include "nep_b200.h"

#ifdef __cplusplus
extern "C" {
#endif

/* Number of CUDA kernels this system has launched since nep_system_create (host counter). */
int64_t nep_launch_count(const nep_system*);

/* Per-phase device timing with CUDA events on the launching stream (for bench.py's roofline entry).
 * nep_profile(s, 1) resets and enables it (adds one event record per phase; at most 2048 events between
 * two nep_get_profile calls, further phases go untimed), nep_profile(s, 0) disables it.
 * nep_get_profile synchronises and returns accumulated milliseconds and launch-group counts for the
 * phases 0 kick+drift, 1 neighbour build (gated), 2 list filter, 3 descriptor+network+partial forces
 * (k_main), 4 assembly, 5 state load/store; entries 6-7 are reserved (0). */
int  nep_profile(nep_system*, int enable);
int  nep_get_profile(nep_system*, double ms[8], int64_t count[8]);

/* Register-resident FMA-chain microbenchmark (a few ms): achieved FP32 non-tensor TFLOP/s with scalar
 * FFMA and with packed fma.rn.f32x2 -- the measured denominator of the "alu" roofline. */
int  nep_measure_fp32_peak(double* tflops_ffma, double* tflops_ffma2, void* cuda_stream);

/* Three more register-resident patterns at k_main's residency (4 x 64 threads per SM), in TFLOP/s:
 * [0] FFMA whose three source registers all differ (the register-file read limit), [1] the packed
 * descriptor contraction s[n][lm] += g_n b_lm, [2] the packed force contraction S'/S += A[n][lm] g'_n / g_n.
 * They are the attainable ceilings of k_main's inner loops, reported beside the nominal peak. */
int  nep_measure_fp32_patterns(double tflops[3], void* cuda_stream);

#ifdef __cplusplus
}
#endif

#endif /* NEP_B200_MEASURE_H */
