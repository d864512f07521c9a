/*
 * helios_rt_selftest.h -- C ABI of libhelios_rt_selftest.so: TEST AND BENCHMARK hooks, not part of the product
 * library (libhelios_rt.so, include/helios_rt.h).  They expose the device primitives the RT kernels are built from
 * (csrc/helios_rt_math.cuh: the same source, compiled into this library too) so that tests/ can check them against
 * high-precision references, and the fp64 FMA microbenchmark bench.py quotes its ALU roofline against.
 */
#ifndef HELIOS_RT_SELFTEST_H
#define HELIOS_RT_SELFTEST_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

/* Device self-test of the fp64 primitives the kernels use instead of the CUDA math library
 * (reciprocal, reciprocal square root, exp / 1-exp).  x: n HOST values; outputs n HOST values each:
 * rcp = 1/x, rsq = 1/sqrt(|x|), ex = exp(-|x|), omx = 1 - exp(-|x|).  Returns 0 or a negative HELIOS_RT_E* code. */
int helios_rt_selftest_math(int32_t n, const double *x, double *rcp, double *rsq, double *ex, double *omx);

/* Device evaluation of the band Planck function used by S2: out[i] = B_b(T[i]) for the bin
 * [lam_lo[i], lam_hi[i]] (HOST arrays of length n). */
int helios_rt_selftest_planck(int32_t n, const double *T, const double *lam_lo, const double *lam_hi, double *out);

/* Device evaluation of G(x) = int_x^inf t^3/(e^t - 1) dt as S2 computes it (HOST arrays of length n). */
int helios_rt_selftest_planck_G(int32_t n, const double *x, double *G);

/* Sustained fp64 FMA rate of the device in DFMA/s (8 independent chains per thread, one resident wave on all SMs),
 * measured over `iters` dependent FMAs per chain; *sm_clock_mhz receives the SM clock during the run, from the
 * clock64() and globaltimer spans of the same thread (maximum over blocks of cycles / nanoseconds). */
int helios_rt_measure_dfma_peak(int32_t iters, double *dfma_per_s, double *sm_clock_mhz);

/* Dependent-issue latencies in SM cycles, measured by single-warp chains on the device: lat[0] DFMA -> DFMA,
 * lat[1] MUFU.RCP64H-seeded reciprocal (rcp_fast) link, lat[2] shared-memory load -> use, lat[3] DADD -> DADD.
 * DESIGN.md section 9 quotes these; bench.py --latencies prints them. */
int helios_rt_measure_latencies(double lat[4]);

#ifdef __cplusplus
}
#endif
#endif /* HELIOS_RT_SELFTEST_H */
