/*
 * catapult_probe.h -- C-ABI of libcatapult_probe.so: measurement and test hooks that are NOT part of the
 * product library (include/catapult.h).  bench.py uses the two peak measurements as roofline
 * denominators (MEASURED_PEAKS.json carries neither an FP64 nor an L2 figure); tests/test_gpu_parity.py
 * uses the math probe.  Same conventions as catapult.h: d_* are device pointers, every call returns a
 * catapult_status, catapult_probe_last_error() gives the message of the last failing call.
 */
#ifndef CATAPULT_PROBE_H
#define CATAPULT_PROBE_H

#include "catapult.h"

#ifdef __cplusplus
extern "C" {
#endif

/* catapult_measure_fp64_peak: runs a register-only DFMA kernel on every SM and returns the sustained
 * double-precision rate in FLOP/s (2 per DFMA).
 * catapult_measure_l2_bandwidth: repeatedly reads a `bytes`-sized device buffer (choose it below the L2
 * size) with 16-byte loads and returns bytes/s.  Both synchronise. */
catapult_status catapult_measure_fp64_peak(double *flops_per_s);
catapult_status catapult_measure_l2_bandwidth(size_t bytes, double *bytes_per_s);

/* the device-side fp64 elementary functions the tracer's scalar path uses (csrc/gc_math.cuh; the probe
   library compiles the same header) evaluated elementwise on d_a[n] (and d_b[n] where a second argument
   exists):
     ATAN2: out0 = atan2(a, b);  SINCOS: out0 = sin(a), out1 = cos(a);  EXP: out0 = exp(a);
     SQRT_RSQRT: out0 = sqrt(a), out1 = 1/sqrt(a);  RCP: out0 = 1/a;
     POW_NEG_INV: out0 = a^(-1/5), out1 = a^(-1/3) (the step-size controller's powers);
     CONTROLLER: the tracer's step-size controller itself (S2) for an attempted step of
       length 1 with error ratio a and maximum step b: out0 = next step length, out1 = 1 if accepted else 0.
   d_b and d_out1 may be NULL where unused. */
#define CATAPULT_FN_ATAN2 0
#define CATAPULT_FN_SINCOS 1
#define CATAPULT_FN_EXP 2
#define CATAPULT_FN_SQRT_RSQRT 3
#define CATAPULT_FN_RCP 4
#define CATAPULT_FN_POW_NEG_INV 5
#define CATAPULT_FN_CONTROLLER 6
catapult_status catapult_math_probe(int32_t fn, int64_t n, const double *d_a, const double *d_b,
                                    double *d_out0, double *d_out1, void *stream);

const char *catapult_probe_last_error(void);

#ifdef __cplusplus
}
#endif
#endif /* CATAPULT_PROBE_H */
