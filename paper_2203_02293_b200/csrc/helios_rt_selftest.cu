// helios_rt_selftest.cu -- test and benchmark hooks (include/helios_rt_selftest.h); built into libhelios_rt_selftest.so,
// never into the product library.  The device primitives under test come from helios_rt_math.cuh, the header the
// product kernels include.

#include "../../include/helios_rt.h"
#include "../../include/helios_rt_selftest.h"
#include "helios_rt_math.cuh"

#include <stdlib.h>

namespace {

using namespace hrt;

int check_device() {
  int n = 0;
  if (cudaGetDeviceCount(&n) != cudaSuccess || n == 0) { cudaGetLastError(); return HELIOS_RT_ENODEV; }
  int dev = 0, major = 0;
  if (cudaGetDevice(&dev) != cudaSuccess) return HELIOS_RT_ENODEV;
  cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev);
  return major == 10 ? HELIOS_RT_OK : HELIOS_RT_ENODEV;
}

__global__ void selftest_math_kernel(int n, const double *x, double *rcp, double *rsq, double *ex, double *omx) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  __shared__ double T32[32];
  if (threadIdx.x < 32) T32[threadIdx.x] = kExp2Tab[threadIdx.x];
  __syncthreads();
  if (i >= n) return;
  const double v = x[i];
  rcp[i] = rcp_fast(v);
  rsq[i] = rsqrt_fast(fabs(v));
  // e^-|x| through the three entry points the step kernel uses: e^-a, e^-2(a/2) (+ 1 - e^-a), e^(-a)
  const double a = fmin(fabs(v), 708.0);
  double om;
  const double e2 = exp_hot<2, true>(0.5 * a, T32, &om);
  const double e1 = exp_hot<1, false>(a, T32, nullptr);
  const double e0 = exp_hot<0, false>(-a, T32, nullptr);
  ex[i] = (i % 3 == 0) ? e0 : ((i % 3 == 1) ? e1 : e2);
  omx[i] = om;
}

__global__ void selftest_planck_kernel(int n, const double *gtab, const double *T, const double *lo, const double *hi,
                                       double *out) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  __shared__ double T32[32];
  if (threadIdx.x < 32) T32[threadIdx.x] = kExp2Tab[threadIdx.x];
  __syncthreads();
  if (i >= n) return;
  const double t = T[i];
  if (!(t > 0.0)) { out[i] = 0.0; return; }
  double l_hi, l_lo;
  const double g_hi = planck_G((kPlanckC2 / hi[i]) * (1.0 / t), gtab, T32, &l_hi),
               g_lo = planck_G((kPlanckC2 / lo[i]) * (1.0 / t), gtab, T32, &l_lo);   // x formed as S2 forms it
  const double t2 = t * t;
  out[i] = kPlanckC1 * t2 * t2 * planck_dG(g_lo, l_lo, g_hi, l_hi) / (hi[i] - lo[i]);
}

__global__ void selftest_G_kernel(int n, const double *gtab, const double *x, double *G) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  __shared__ double T32[32];
  if (threadIdx.x < 32) T32[threadIdx.x] = kExp2Tab[threadIdx.x];
  __syncthreads();
  if (i >= n) return;
  double low;
  G[i] = planck_G(x[i], gtab, T32, &low);
}

__device__ __forceinline__ unsigned long long globaltimer_ns() {
  unsigned long long t;
  asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t));
  return t;
}

// cyc_ns[2 b], [2 b + 1]: clock64 span and globaltimer span of thread 0 of block b around its own loop
__global__ void dfma_peak_kernel(int iters, double seed, double *sink, unsigned long long *cyc_ns) {
  double a0 = seed, a1 = seed + 1, a2 = seed + 2, a3 = seed + 3, a4 = seed + 4, a5 = seed + 5, a6 = seed + 6,
         a7 = seed + 7;
  const double m = 0.999999, k = 1e-9;
  const unsigned long long g0 = globaltimer_ns();
  const long long t0 = clock64();
#pragma unroll 4
  for (int i = 0; i < iters; ++i) {
    a0 = fma(a0, m, k); a1 = fma(a1, m, k); a2 = fma(a2, m, k); a3 = fma(a3, m, k);
    a4 = fma(a4, m, k); a5 = fma(a5, m, k); a6 = fma(a6, m, k); a7 = fma(a7, m, k);
  }
  const long long t1 = clock64();
  const unsigned long long g1 = globaltimer_ns();
  const double s = a0 + a1 + a2 + a3 + a4 + a5 + a6 + a7;
  if (s == 123.456) sink[0] = s;
  if (threadIdx.x == 0) { cyc_ns[2 * blockIdx.x] = (unsigned long long)(t1 - t0); cyc_ns[2 * blockIdx.x + 1] = g1 - g0; }
}

// single-warp dependent chains; out[k] = cycles per link
__global__ void latency_kernel(int iters, double seed, double *out, double *sink) {
  __shared__ double s_ring[64];
  const int lane = threadIdx.x;
  s_ring[lane] = (double)((lane + 1) & 31);
  s_ring[32 + lane] = 0.0;
  __syncthreads();
  double a = seed;
  long long t0 = clock64();
#pragma unroll 8
  for (int i = 0; i < iters; ++i) a = fma(a, 0.999999, 1e-9);
  long long t1 = clock64();
  if (lane == 0) out[0] = (double)(t1 - t0) / iters;
  double b = seed + 1.5;
  t0 = clock64();
#pragma unroll 4
  for (int i = 0; i < iters; ++i) b = rcp_fast(b) + 1.0;
  t1 = clock64();
  // one link = MUFU.RCP64H + 3 DFMA + 1 DADD
  if (lane == 0) out[1] = (double)(t1 - t0) / iters;
  int idx = lane;
  t0 = clock64();
#pragma unroll 8
  for (int i = 0; i < iters; ++i) idx = (int)s_ring[idx];
  t1 = clock64();
  // one link = LDS + F2I (double -> int)
  if (lane == 0) out[2] = (double)(t1 - t0) / iters;
  double c = seed;
  t0 = clock64();
#pragma unroll 8
  for (int i = 0; i < iters; ++i) c = c + 1e-9;
  t1 = clock64();
  if (lane == 0) out[3] = (double)(t1 - t0) / iters;
  if (a + b + c + idx == 123.456) sink[0] = a;
}

}  // namespace

extern "C" int helios_rt_selftest_math(int32_t n, const double *x, double *rcp, double *rsq, double *ex, double *omx) {
  if (n < 0 || (n > 0 && (!x || !rcp || !rsq || !ex || !omx))) return HELIOS_RT_EINVAL;
  int rc = check_device();
  if (rc) return rc;
  if (n == 0) return HELIOS_RT_OK;
  double *d = nullptr;
  if (cudaMalloc((void **)&d, sizeof(double) * 5 * (size_t)n) != cudaSuccess) { cudaGetLastError(); return HELIOS_RT_ENOMEM; }
  cudaError_t e = cudaMemcpy(d, x, sizeof(double) * n, cudaMemcpyHostToDevice);
  if (e == cudaSuccess) {
    selftest_math_kernel<<<(n + 127) / 128, 128>>>(n, d, d + n, d + 2 * (size_t)n, d + 3 * (size_t)n, d + 4 * (size_t)n);
    e = cudaGetLastError();
  }
  if (e == cudaSuccess) e = cudaMemcpy(rcp, d + n, sizeof(double) * n, cudaMemcpyDeviceToHost);
  if (e == cudaSuccess) e = cudaMemcpy(rsq, d + 2 * (size_t)n, sizeof(double) * n, cudaMemcpyDeviceToHost);
  if (e == cudaSuccess) e = cudaMemcpy(ex, d + 3 * (size_t)n, sizeof(double) * n, cudaMemcpyDeviceToHost);
  if (e == cudaSuccess) e = cudaMemcpy(omx, d + 4 * (size_t)n, sizeof(double) * n, cudaMemcpyDeviceToHost);
  cudaFree(d);
  return e == cudaSuccess ? HELIOS_RT_OK : HELIOS_RT_ECUDA;
}

static int upload_gtab(double **d_gtab) {
  double tab[kGIntervals * kGCoef];
  build_planck_table(tab);
  if (cudaMalloc((void **)d_gtab, sizeof(tab)) != cudaSuccess) { cudaGetLastError(); return HELIOS_RT_ENOMEM; }
  if (cudaMemcpy(*d_gtab, tab, sizeof(tab), cudaMemcpyHostToDevice) != cudaSuccess) { cudaFree(*d_gtab); return HELIOS_RT_ECUDA; }
  return HELIOS_RT_OK;
}

extern "C" int helios_rt_selftest_planck(int32_t n, const double *T, const double *lam_lo, const double *lam_hi,
                                         double *out) {
  if (n < 0 || (n > 0 && (!T || !lam_lo || !lam_hi || !out))) return HELIOS_RT_EINVAL;
  int rc = check_device();
  if (rc) return rc;
  if (n == 0) return HELIOS_RT_OK;
  double *d = nullptr, *g = nullptr;
  rc = upload_gtab(&g);
  if (rc) return rc;
  if (cudaMalloc((void **)&d, sizeof(double) * 4 * (size_t)n) != cudaSuccess) { cudaGetLastError(); cudaFree(g); return HELIOS_RT_ENOMEM; }
  cudaError_t e = cudaMemcpy(d, T, sizeof(double) * n, cudaMemcpyHostToDevice);
  if (e == cudaSuccess) e = cudaMemcpy(d + n, lam_lo, sizeof(double) * n, cudaMemcpyHostToDevice);
  if (e == cudaSuccess) e = cudaMemcpy(d + 2 * (size_t)n, lam_hi, sizeof(double) * n, cudaMemcpyHostToDevice);
  if (e == cudaSuccess) {
    selftest_planck_kernel<<<(n + 127) / 128, 128>>>(n, g, d, d + n, d + 2 * (size_t)n, d + 3 * (size_t)n);
    e = cudaGetLastError();
  }
  if (e == cudaSuccess) e = cudaMemcpy(out, d + 3 * (size_t)n, sizeof(double) * n, cudaMemcpyDeviceToHost);
  cudaFree(d);
  cudaFree(g);
  return e == cudaSuccess ? HELIOS_RT_OK : HELIOS_RT_ECUDA;
}

extern "C" int helios_rt_selftest_planck_G(int32_t n, const double *x, double *G) {
  if (n < 0 || (n > 0 && (!x || !G))) return HELIOS_RT_EINVAL;
  int rc = check_device();
  if (rc) return rc;
  if (n == 0) return HELIOS_RT_OK;
  double *d = nullptr, *g = nullptr;
  rc = upload_gtab(&g);
  if (rc) return rc;
  if (cudaMalloc((void **)&d, sizeof(double) * 2 * (size_t)n) != cudaSuccess) { cudaGetLastError(); cudaFree(g); return HELIOS_RT_ENOMEM; }
  cudaError_t e = cudaMemcpy(d, x, sizeof(double) * n, cudaMemcpyHostToDevice);
  if (e == cudaSuccess) {
    selftest_G_kernel<<<(n + 127) / 128, 128>>>(n, g, d, d + n);
    e = cudaGetLastError();
  }
  if (e == cudaSuccess) e = cudaMemcpy(G, d + n, sizeof(double) * n, cudaMemcpyDeviceToHost);
  cudaFree(d);
  cudaFree(g);
  return e == cudaSuccess ? HELIOS_RT_OK : HELIOS_RT_ECUDA;
}

extern "C" int helios_rt_measure_dfma_peak(int32_t iters, double *dfma_per_s, double *sm_clock_mhz) {
  if (iters < 1 || !dfma_per_s) return HELIOS_RT_EINVAL;
  int rc = check_device();
  if (rc) return rc;
  int dev = 0, sms = 0;
  cudaGetDevice(&dev);
  cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
  // one resident wave: 2 blocks of 1024 threads per SM (32 registers per thread), so the event time of the launch is
  // the time of every block's loop and no block waits for a slot
  const int blocks = sms * 2, threads = 1024;
  double *sink = nullptr;
  unsigned long long *cyc = nullptr;
  unsigned long long *hc = (unsigned long long *)malloc(sizeof(unsigned long long) * 2 * blocks);
  if (!hc) return HELIOS_RT_ENOMEM;
  if (cudaMalloc((void **)&sink, sizeof(double)) != cudaSuccess) { free(hc); return HELIOS_RT_ENOMEM; }
  if (cudaMalloc((void **)&cyc, sizeof(unsigned long long) * 2 * blocks) != cudaSuccess) { cudaFree(sink); free(hc); return HELIOS_RT_ENOMEM; }
  cudaEvent_t e0, e1;
  cudaEventCreate(&e0); cudaEventCreate(&e1);
  dfma_peak_kernel<<<blocks, threads>>>(iters / 8 + 1, 1.0, sink, cyc);   // warm-up
  float best = 1e30f;
  double mhz = 0.0;
  for (int rep = 0; rep < 3; ++rep) {
    cudaEventRecord(e0);
    dfma_peak_kernel<<<blocks, threads>>>(iters, 1.0, sink, cyc);
    cudaEventRecord(e1);
    if (cudaEventSynchronize(e1) != cudaSuccess) { rc = HELIOS_RT_ECUDA; break; }
    float ms = 0;
    cudaEventElapsedTime(&ms, e0, e1);
    if (ms < best) {
      best = ms;
      cudaMemcpy(hc, cyc, sizeof(unsigned long long) * 2 * blocks, cudaMemcpyDeviceToHost);
      mhz = 0.0;
      for (int b = 0; b < blocks; ++b)
        if (hc[2 * b + 1] > 0) { const double f = (double)hc[2 * b] / (double)hc[2 * b + 1] * 1e3; if (f > mhz) mhz = f; }
    }
  }
  cudaEventDestroy(e0); cudaEventDestroy(e1);
  cudaFree(sink); cudaFree(cyc); free(hc);
  if (rc) return rc;
  *dfma_per_s = 8.0 * (double)iters * (double)blocks * threads / (best * 1e-3);
  if (sm_clock_mhz) *sm_clock_mhz = mhz;
  return HELIOS_RT_OK;
}

extern "C" int helios_rt_measure_latencies(double lat[4]) {
  if (!lat) return HELIOS_RT_EINVAL;
  int rc = check_device();
  if (rc) return rc;
  double *d = nullptr;
  if (cudaMalloc((void **)&d, sizeof(double) * 5) != cudaSuccess) { cudaGetLastError(); return HELIOS_RT_ENOMEM; }
  latency_kernel<<<1, 32>>>(1 << 12, 1.0, d, d + 4);      // warm-up
  latency_kernel<<<1, 32>>>(1 << 14, 1.0, d, d + 4);
  cudaError_t e = cudaMemcpy(lat, d, sizeof(double) * 4, cudaMemcpyDeviceToHost);
  cudaFree(d);
  return e == cudaSuccess ? HELIOS_RT_OK : HELIOS_RT_ECUDA;
}
