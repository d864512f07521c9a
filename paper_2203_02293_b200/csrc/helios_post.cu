// helios_post.cu -- the steps either side of the RT step, sm_100a.
//
//   helios_rt_extend_top   PAPER.md L385: columns extended isothermally to <= p_min before the post-processing step
//   helios_rt_phase_curve  Eqs.(25)-(26) L546-552 (+ the wavelength integral of Eq.(23))
//   helios_rt_advance_1d   Sec. 3 "1-D mode": T <- T + dt dT/dt, hydrostatic re-balance Eq.(20)
//   helios_rt_phase_curve_noalloc   helios_rt_phase_curve with its scratch in a built-in device array, for callers
//                          that cannot allocate (described where it is defined, near the end of this file)
//
// C ABI: include/helios_rt.h.  All pointers are DEVICE pointers; every call is asynchronous on the given
// stream, allocates nothing and synchronises nothing, so the calls can be captured in a CUDA graph together
// with helios_rt_step.  Readings R21-R26: DESIGN.md.

#include "../../include/helios_rt.h"

#include <cuda_runtime.h>
#include <math.h>
#include <stdint.h>

#include <mutex>

namespace {

constexpr double kPi = 3.14159265358979323846;

int device_ok() {
  static int cached = 1;   // the device check is made once: later calls may sit inside a CUDA-graph capture
  if (cached <= 0) return cached;
  const auto done = [&](int rc) { if (rc == HELIOS_RT_OK) cached = 0; return rc; };
  int n = 0;
  if (cudaGetDeviceCount(&n) != cudaSuccess || n == 0) { cudaGetLastError(); return HELIOS_RT_ENODEV; }
  int dev = 0, major = 0;
  if (cudaGetDevice(&dev) != cudaSuccess) return HELIOS_RT_ENODEV;
  cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev);
  return done(major == 10 ? HELIOS_RT_OK : HELIOS_RT_ENODEV);
}

// ---------------------------------------------------------------------------------------------------------
// extend_top: one thread per OUTPUT element (column, extended layer), so that consecutive threads write consecutive
// addresses (one thread per column wrote with a stride of N + n_extra doubles).  n_extra layers above the top layer,
// equally spaced in ln p with the ratio q = min(p[N-1]/p[N-2], (p_min/p[N-1])^(1/n_extra)) (reading R21);
// T = T[N-1] (L385).  Every element is the same expression as before: p_top * q^k, bit for bit.
// ---------------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) extend_top_kernel(int ncol, int N, int n_extra, double p_min,
                                                         const double *__restrict__ p, const double *__restrict__ T,
                                                         double *__restrict__ p_ext, double *__restrict__ T_ext) {
  const int Ne = N + n_extra;
  const size_t e = (size_t)blockIdx.x * 256 + threadIdx.x;
  if (e >= (size_t)ncol * Ne) return;
  const int c = (int)(e / Ne), j = (int)(e - (size_t)c * Ne);
  const double *pc = p + (size_t)c * N, *Tc = T + (size_t)c * N;
  if (j < N) { p_ext[e] = pc[j]; T_ext[e] = Tc[j]; return; }
  const double p_top = pc[N - 1];
  const double q_own = (N > 1) ? p_top / pc[N - 2] : sqrt(0.1);
  const double q_need = pow(p_min / p_top, 1.0 / (double)n_extra);
  const double q = fmin(q_own, q_need);
  p_ext[e] = p_top * pow(q, (double)(j - (N - 1)));
  T_ext[e] = Tc[N - 1];
}

// ---------------------------------------------------------------------------------------------------------
// phase_curve: out[a][b] = sum_i F[i][b] * w_a[i],  w_a[i] = cos(lat_i) max(cos(lon_i - alpha_a), 0) A_i / (pi R_p^2)
// (Eqs. 25-26; visibility modulo 2 pi, reading R22).  Two launches, F read once per 32 phases:
//   phase_partial_kernel  grid = (bin tiles of 128 NB, column chunks of 128, phase tiles of NPH).  Each thread first
//       builds the NPH weights of one column of the chunk in shared memory (angle-addition form), then accumulates its NB
//       bins over the chunk's columns in index order: F rows read coalesced, weights broadcast from shared memory two at
//       a time, NB x NPH independent FMA chains in registers.  Writes part[chunk][phase][bin] to the caller's workspace.
//   phase_reduce_kernel   out[a][b] = sum over chunks in chunk order.
// Both sums run in a fixed order: deterministic run to run.
// ---------------------------------------------------------------------------------------------------------
constexpr int PC_BINS = 128, PC_COLS = 128;

// NB bins per thread (bins tid, tid + 128, ... of a tile of 128 NB bins) x NPH phases per block.  The weights reach the
// FMAs as broadcast 16-byte shared-memory loads, each of which fills 512 B of registers: at <1, 32> that is 8.25 B per FMA
// against the ~2 B per FMA an SM can deliver at its DFMA rate, and the kernel ran at a quarter of that rate.  <4, 16>
// uses every loaded weight for four bins (2.5 B per FMA; 64 accumulators per thread) and is what wide spectra take;
// <1, 32> stays for spectra of up to 256 bins, where a 512-bin tile would be mostly padding.  Every output is the same
// chain of FMAs in the same order in both shapes: bit-identical results.
template <int NB, int NPH>
__global__ void __launch_bounds__(PC_BINS) phase_partial_kernel(int ncol, int nb, int nph, const double *__restrict__ F,
                                                                 const double *__restrict__ lon,
                                                                 const double *__restrict__ lat,
                                                                 const double *__restrict__ area,
                                                                 const double *__restrict__ alpha,
                                                                 double *__restrict__ part) {
  __shared__ __align__(16) double s_w[PC_COLS][NPH];
  __shared__ __align__(16) double2 s_cs[NPH];   // (cos alpha, sin alpha) of the tile's phases
  const int tid = threadIdx.x;
  const int bin0 = blockIdx.x * (PC_BINS * NB) + tid;
  const int chunk = blockIdx.y, c0 = chunk * PC_COLS;
  const int ph0 = blockIdx.z * NPH;
  if (tid < NPH) {
    double sa = 0.0, ca = 0.0;
    if (ph0 + tid < nph) sincos(alpha[ph0 + tid], &sa, &ca);
    s_cs[tid] = make_double2(ca, sa);
  }
  __syncthreads();
  {
    // cos(lon - alpha) = cos lon cos alpha + sin lon sin alpha: one sincos per column and per phase instead of one cos per
    // (column, phase) -- the weights were as expensive as the sum they feed (32 fp64 cosines against 128 FMAs per thread
    // and phase).  The two forms differ by a few 1e-16 (absolute), also in which side of the terminator a column with
    // |cos| < 1e-16 falls on; its weight is below 1e-16 of the disc either way.
    const int i = c0 + tid;
    if (i < ncol) {
      double sl, clon;
      sincos(lon[i], &sl, &clon);
      const double cl = cos(lat[i]) * (area[i] / kPi);
      for (int k = 0; k < NPH; ++k) {
        const double2 cs = s_cs[k];
        const double c = fma(sl, cs.y, clon * cs.x);
        s_w[tid][k] = (c > 0.0) ? cl * c : 0.0;     // Eq.(26)
      }
    } else {
      for (int k = 0; k < NPH; ++k) s_w[tid][k] = 0.0;
    }
  }
  __syncthreads();
  if (bin0 >= nb) return;
  double acc[NB][NPH];
#pragma unroll
  for (int q = 0; q < NB; ++q)
#pragma unroll
    for (int k = 0; k < NPH; ++k) acc[q][k] = 0.0;
  const int nj = (ncol - c0 < PC_COLS) ? (ncol - c0) : PC_COLS;
  // bins past the end of the spectrum read the thread's first bin instead (no test in the loop); their sums are dropped
  const double *Fp[NB];
#pragma unroll
  for (int q = 0; q < NB; ++q) Fp[q] = F + (size_t)c0 * nb + ((bin0 + q * PC_BINS < nb) ? bin0 + q * PC_BINS : bin0);
  // F is read once, from HBM: the loads of the next UNR columns (16 per thread) are in flight while this batch is summed
  // (with one or two columns ahead the kernel sat on its global loads: long_scoreboard 3.8 warps per issue-active cycle,
  // fp64 pipes 35 % busy at 8 warps per SM).  Rows past the end of a ragged chunk re-read its last row and are not summed.
  constexpr int UNR = 16 / NB;
  double fa[UNR][NB];
#pragma unroll
  for (int u = 0; u < UNR; ++u) {
    const size_t row = (size_t)(u < nj ? u : nj - 1) * nb;
#pragma unroll
    for (int q = 0; q < NB; ++q) fa[u][q] = __ldg(Fp[q] + row);
  }
  for (int j0 = 0; j0 < nj; j0 += UNR) {
    double fb[UNR][NB];
#pragma unroll
    for (int u = 0; u < UNR; ++u) {
      const int jn = j0 + UNR + u;
      const size_t row = (size_t)(jn < nj ? jn : nj - 1) * nb;
#pragma unroll
      for (int q = 0; q < NB; ++q) fb[u][q] = __ldg(Fp[q] + row);
    }
#pragma unroll
    for (int u = 0; u < UNR; ++u) {
      if (j0 + u < nj) {
        const double2 *w2 = reinterpret_cast<const double2 *>(&s_w[j0 + u][0]);
#pragma unroll
        for (int k = 0; k < NPH / 2; ++k) {
          const double2 w = w2[k];
#pragma unroll
          for (int q = 0; q < NB; ++q) {
            acc[q][2 * k] = fma(w.x, fa[u][q], acc[q][2 * k]);         // Eq.(25)
            acc[q][2 * k + 1] = fma(w.y, fa[u][q], acc[q][2 * k + 1]);
          }
        }
      }
    }
#pragma unroll
    for (int u = 0; u < UNR; ++u)
#pragma unroll
      for (int q = 0; q < NB; ++q) fa[u][q] = fb[u][q];
  }
#pragma unroll
  for (int q = 0; q < NB; ++q) {
    const int bin = bin0 + q * PC_BINS;
    if (bin < nb) {
#pragma unroll
      for (int k = 0; k < NPH; ++k)
        if (ph0 + k < nph) part[((size_t)chunk * nph + ph0 + k) * nb + bin] = acc[q][k];
    }
  }
}

__global__ void __launch_bounds__(256) phase_reduce_kernel(int nchunk, size_t n_out, const double *__restrict__ part,
                                                           double *__restrict__ out) {
  const size_t i = (size_t)blockIdx.x * 256 + threadIdx.x;
  if (i >= n_out) return;
  double sum = 0.0;
  for (int c = 0; c < nchunk; ++c) sum += part[(size_t)c * n_out + i];
  out[i] = sum;
}

// band integral of Eq.(23): out[a] = sum_b overlap([edges[b], edges[b+1]], [lam1, lam2]) * F[a][b] (reading R24).
// One block per phase; fixed-order tree reduction.
__global__ void __launch_bounds__(256) phase_band_kernel(int nb, const double *__restrict__ edges, double lam1, double lam2,
                                                         const double *__restrict__ Fph, double *__restrict__ out) {
  __shared__ double s[256];
  const int a = blockIdx.x, tid = threadIdx.x;
  double sum = 0.0;
  for (int b = tid; b < nb; b += 256) {
    const double lo = fmax(edges[b], lam1), hi = fmin(edges[b + 1], lam2);
    const double w = (hi > lo) ? hi - lo : 0.0;
    sum = fma(w, Fph[(size_t)a * nb + b], sum);
  }
  s[tid] = sum;
  __syncthreads();
  for (int o = 128; o > 0; o >>= 1) {
    if (tid < o) s[tid] += s[tid + o];
    __syncthreads();
  }
  if (tid == 0) out[a] = s[0];
}

// ---------------------------------------------------------------------------------------------------------
// advance_1d: one thread per column (columns longer than 62 layers; shorter ones take advance_1d_tile_kernel below, which
// is this kernel with its loads and stores staged through shared memory).  T <- T + dt dT/dt (reading R26); p[0] = p_ref and Eq.(20) upward with the
// sign of reading R25; rho = p / (R_d T).
// ---------------------------------------------------------------------------------------------------------
__global__ void advance_1d_kernel(int ncol, int N, double dt, double gravity, double R_d, double p_ref,
                                  const double *__restrict__ z, const double *__restrict__ dTdt, double *__restrict__ T,
                                  double *__restrict__ p, double *__restrict__ rho) {
  const int c = blockIdx.x * blockDim.x + threadIdx.x;
  if (c >= ncol) return;
  double *Tc = T + (size_t)c * N, *pc = p + (size_t)c * N;
  const double *hc = dTdt ? dTdt + (size_t)c * N : nullptr;
  const double g2R = gravity / (2.0 * R_d);
  double T_prev = hc ? __dadd_rn(Tc[0], __dmul_rn(dt, hc[0])) : Tc[0];
  double p_prev = p_ref;
  Tc[0] = T_prev;
  pc[0] = p_prev;
  if (rho) rho[(size_t)c * N] = p_prev / (R_d * T_prev);
  for (int i = 1; i < N; ++i) {
    const double Ti = hc ? __dadd_rn(Tc[i], __dmul_rn(dt, hc[i])) : Tc[i];
    const double inv_dz = 1.0 / (z[i] - z[i - 1]);
    const double pi = p_prev * (inv_dz - g2R / T_prev) / (inv_dz + g2R / Ti);
    Tc[i] = Ti;
    pc[i] = pi;
    if (rho) rho[(size_t)c * N + i] = pi / (R_d * Ti);
    T_prev = Ti;
    p_prev = pi;
  }
}

// The same step with coalesced memory traffic: a block of 32 threads owns 32 consecutive columns, whose T, dT/dt and
// outputs are one contiguous range of 32 N doubles each.  The block copies T and dT/dt into shared memory with
// consecutive threads on consecutive addresses, each thread then walks ITS column in shared memory (row stride N + 1:
// odd or not, the 32 rows start in different banks for every N that is not a multiple of 16) with exactly the
// arithmetic of advance_1d_kernel -- same operations in the same order, so the results are bit-identical -- and the
// block writes T, p and rho back as linear copies.  Shared memory: 3 x 32 x (N + 1) doubles (N <= 62 fits 48 KB; longer
// columns take the kernel above).
constexpr int A1_COLS = 32;
__global__ void __launch_bounds__(A1_COLS) advance_1d_tile_kernel(int ncol, int N, double dt, double gravity, double R_d,
                                                                  double p_ref, const double *__restrict__ z,
                                                                  const double *__restrict__ dTdt, double *__restrict__ T,
                                                                  double *__restrict__ p, double *__restrict__ rho) {
  extern __shared__ double a1_smem[];
  const int ld = N + 1;
  double *sT = a1_smem, *sH = sT + A1_COLS * ld, *sP = sH + A1_COLS * ld;
  const int tid = threadIdx.x, c0 = blockIdx.x * A1_COLS;
  const int nc = (ncol - c0 < A1_COLS) ? ncol - c0 : A1_COLS;
  const size_t base = (size_t)c0 * N;
  const int n_el = nc * N;
  for (int e = tid; e < n_el; e += A1_COLS) {
    const int c = e / N, i = e - c * N;
    sT[c * ld + i] = T[base + e];
    if (dTdt) sH[c * ld + i] = dTdt[base + e];
  }
  __syncwarp();
  if (tid < nc) {
    double *Tc = sT + tid * ld, *pc = sP + tid * ld;
    const double *hc = dTdt ? sH + tid * ld : nullptr;
    const double g2R = gravity / (2.0 * R_d);
    double T_prev = hc ? __dadd_rn(Tc[0], __dmul_rn(dt, hc[0])) : Tc[0];
    double p_prev = p_ref;
    Tc[0] = T_prev;
    pc[0] = p_prev;
    for (int i = 1; i < N; ++i) {
      const double Ti = hc ? __dadd_rn(Tc[i], __dmul_rn(dt, hc[i])) : Tc[i];
      const double inv_dz = 1.0 / (z[i] - z[i - 1]);
      const double pi = p_prev * (inv_dz - g2R / T_prev) / (inv_dz + g2R / Ti);
      Tc[i] = Ti;
      pc[i] = pi;
      T_prev = Ti;
      p_prev = pi;
    }
  }
  __syncwarp();
  for (int e = tid; e < n_el; e += A1_COLS) {
    const int c = e / N, i = e - c * N;
    const double Ti = sT[c * ld + i], pi = sP[c * ld + i];
    T[base + e] = Ti;
    p[base + e] = pi;
    if (rho) rho[base + e] = pi / (R_d * Ti);
  }
}

}  // namespace

extern "C" int helios_rt_extend_top(int32_t n_columns, int32_t n_layers, int32_t n_extra, double p_min, const double *p,
                                    const double *T, double *p_ext, double *T_ext, void *cuda_stream) {
  if (n_columns < 0 || n_layers < 1 || n_extra < 0 || !(p_min > 0.0)) return HELIOS_RT_EINVAL;
  if (n_columns > 0 && (!p || !T || !p_ext || !T_ext)) return HELIOS_RT_EINVAL;
  const int rc = device_ok();
  if (rc) return rc;
  if (n_columns == 0) return HELIOS_RT_OK;
  const size_t n_el = (size_t)n_columns * (n_layers + n_extra);
  extend_top_kernel<<<(unsigned)((n_el + 255) / 256), 256, 0, (cudaStream_t)cuda_stream>>>(n_columns, n_layers, n_extra, p_min, p,
                                                                                          T, p_ext, T_ext);
  return cudaGetLastError() == cudaSuccess ? HELIOS_RT_OK : HELIOS_RT_ECUDA;
}

extern "C" int64_t helios_rt_phase_curve_workspace_bytes(int32_t n_columns, int32_t n_bins, int32_t n_phases) {
  if (n_columns < 0 || n_bins < 1 || n_phases < 0) return HELIOS_RT_EINVAL;
  const int64_t nchunk = (n_columns + PC_COLS - 1) / PC_COLS;
  return (int64_t)sizeof(double) * (nchunk > 0 ? nchunk : 1) * n_phases * n_bins;
}

extern "C" int helios_rt_phase_curve(int32_t n_columns, int32_t n_bins, int32_t n_phases, const double *F_toa_bin,
                                     const double *lon, const double *lat, const double *area, const double *alpha,
                                     const double *bin_edges, double lam1, double lam2, double *F_phase_bin,
                                     double *F_phase_band, double *workspace, void *cuda_stream) {
  if (n_columns < 0 || n_bins < 1 || n_phases < 0) return HELIOS_RT_EINVAL;
  if (n_phases > 0 && (!alpha || !F_phase_bin)) return HELIOS_RT_EINVAL;
  if (n_columns > 0 && n_phases > 0 && (!F_toa_bin || !lon || !lat || !area || !workspace)) return HELIOS_RT_EINVAL;
  if (F_phase_band && (!bin_edges || !(lam2 >= lam1))) return HELIOS_RT_EINVAL;
  const int rc = device_ok();
  if (rc) return rc;
  if (n_phases == 0) return HELIOS_RT_OK;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  const int nchunk = (n_columns + PC_COLS - 1) / PC_COLS;
  const size_t n_out = (size_t)n_phases * n_bins;
  if (nchunk > 0) {
    if (n_bins > 2 * PC_BINS) {
      dim3 grid((unsigned)((n_bins + 4 * PC_BINS - 1) / (4 * PC_BINS)), (unsigned)nchunk, (unsigned)((n_phases + 15) / 16));
      phase_partial_kernel<4, 16><<<grid, PC_BINS, 0, st>>>(n_columns, n_bins, n_phases, F_toa_bin, lon, lat, area, alpha, workspace);
    } else {
      dim3 grid((unsigned)((n_bins + PC_BINS - 1) / PC_BINS), (unsigned)nchunk, (unsigned)((n_phases + 31) / 32));
      phase_partial_kernel<1, 32><<<grid, PC_BINS, 0, st>>>(n_columns, n_bins, n_phases, F_toa_bin, lon, lat, area, alpha, workspace);
    }
    if (cudaGetLastError() != cudaSuccess) return HELIOS_RT_ECUDA;
  }
  phase_reduce_kernel<<<(unsigned)((n_out + 255) / 256), 256, 0, st>>>(nchunk, n_out, workspace, F_phase_bin);
  if (cudaGetLastError() != cudaSuccess) return HELIOS_RT_ECUDA;
  if (F_phase_band) {
    phase_band_kernel<<<(unsigned)n_phases, 256, 0, st>>>(n_bins, bin_edges, lam1, lam2, F_phase_bin, F_phase_band);
    if (cudaGetLastError() != cudaSuccess) return HELIOS_RT_ECUDA;
  }
  return HELIOS_RT_OK;
}

// ---------------------------------------------------------------------------------------------------------
// helios_rt_phase_curve_noalloc: the phase curve for callers that may not allocate device memory (a plug-in inside
// an application that owns the whole device, a real-time path that must stay out of the driver's allocator, a
// worker whose memory budget is spent; include/helios_rt.h has the full contract).  The partial sums of
// phase_partial_kernel go to g_phase_scratch, an array that is part of this library's device image, instead of a
// buffer the caller had to allocate.
//
// g_phase_scratch is a DEVICE symbol.  In host code its name is only a host-side stand-in -- it is not a device
// address, and a kernel handed `g_phase_scratch` from the host would fault (or, on a system where the GPU can reach
// host memory, quietly use the wrong memory).  Each device holds its own copy at its own address, so the address is
// asked for once per device, with that device current, and cached by device ordinal.
// ---------------------------------------------------------------------------------------------------------
static __device__ __align__(256) double g_phase_scratch[HELIOS_RT_PHASE_CURVE_NOALLOC_MAX_BYTES / sizeof(double)];

namespace {

constexpr int kMaxDevices = 64;
std::mutex g_scratch_mutex;
double *g_scratch_addr[kMaxDevices];   // [device ordinal] -> address of g_phase_scratch on that device; nullptr = not asked yet

// Device address of g_phase_scratch on the CURRENT device.  The first call per device asks the runtime (which may
// load this library's device code: do it before any stream capture); later calls read the cache.  No allocation.
int phase_scratch_address(double **out) {
  int dev = -1;
  if (cudaGetDevice(&dev) != cudaSuccess) { cudaGetLastError(); return HELIOS_RT_ENODEV; }
  if (dev < 0 || dev >= kMaxDevices) return HELIOS_RT_ENODEV;
  std::lock_guard<std::mutex> lock(g_scratch_mutex);
  if (!g_scratch_addr[dev]) {
    void *addr = nullptr;
    const cudaError_t e = cudaGetSymbolAddress(&addr, g_phase_scratch);
    if (e != cudaSuccess || !addr) { cudaGetLastError(); return HELIOS_RT_ECUDA; }
    g_scratch_addr[dev] = static_cast<double *>(addr);
  }
  *out = g_scratch_addr[dev];
  return HELIOS_RT_OK;
}

}  // namespace

extern "C" int helios_rt_phase_curve_noalloc(int32_t n_columns, int32_t n_bins, int32_t n_phases, const double *F_toa_bin,
                                             const double *lon, const double *lat, const double *area,
                                             const double *alpha, const double *bin_edges, double lam1, double lam2,
                                             double *F_phase_bin, double *F_phase_band, void *cuda_stream) {
  // Size first: a problem that does not fit the built-in array is refused before anything is queued.
  const int64_t need = helios_rt_phase_curve_workspace_bytes(n_columns, n_bins, n_phases);
  if (need < 0) return HELIOS_RT_EINVAL;
  if (need > (int64_t)HELIOS_RT_PHASE_CURVE_NOALLOC_MAX_BYTES) return HELIOS_RT_ETOOBIG;
  int rc = device_ok();
  if (rc) return rc;
  double *scratch = nullptr;
  rc = phase_scratch_address(&scratch);
  if (rc) return rc;
  // Same kernels, same order as the caller-workspace path; only where the partial sums live differs.  The array
  // keeps the previous call's partial sums; phase_partial_kernel overwrites every element phase_reduce_kernel reads
  // (chunk < nchunk, phase < n_phases, bin < n_bins), so nothing has to be cleared.  Calls that overlap on the GPU
  // would share these partial sums and race: callers keep them stream-ordered.
  return helios_rt_phase_curve(n_columns, n_bins, n_phases, F_toa_bin, lon, lat, area, alpha, bin_edges, lam1, lam2,
                               F_phase_bin, F_phase_band, scratch, cuda_stream);
}

extern "C" int helios_rt_advance_1d(int32_t n_columns, int32_t n_layers, double dt, double gravity, double R_d, double p_ref,
                                    const double *z, const double *dTdt, double *T, double *p, double *rho,
                                    void *cuda_stream) {
  if (n_columns < 0 || n_layers < 1 || !(gravity > 0.0) || !(R_d > 0.0) || !(p_ref > 0.0) || !(dt == dt))
    return HELIOS_RT_EINVAL;
  if (n_columns > 0 && (!z || !T || !p)) return HELIOS_RT_EINVAL;
  const int rc = device_ok();
  if (rc) return rc;
  if (n_columns == 0) return HELIOS_RT_OK;
  const size_t smem = sizeof(double) * 3 * A1_COLS * ((size_t)n_layers + 1);
  if (smem <= 48 * 1024)
    advance_1d_tile_kernel<<<(n_columns + A1_COLS - 1) / A1_COLS, A1_COLS, smem, (cudaStream_t)cuda_stream>>>(
        n_columns, n_layers, dt, gravity, R_d, p_ref, z, dTdt, T, p, rho);
  else
    advance_1d_kernel<<<(n_columns + 63) / 64, 64, 0, (cudaStream_t)cuda_stream>>>(n_columns, n_layers, dt, gravity, R_d, p_ref, z,
                                                                                   dTdt, T, p, rho);
  return cudaGetLastError() == cudaSuccess ? HELIOS_RT_OK : HELIOS_RT_ECUDA;
}
