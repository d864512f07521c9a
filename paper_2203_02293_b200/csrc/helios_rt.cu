// helios_rt.cu -- B200 (sm_100a) implementation of the THOR+HELIOS radiative-transfer step.
//
// C ABI: include/helios_rt.h.  Citations are PAPER.md lines (arXiv 2203.02293); R-numbers are DESIGN.md readings.
//
// ONE launch per step: rt_step_kernel, a persistent grid of (tiles per column) x (workers) thread blocks.  A block
// is bound to one tile of the (bin, Gauss point) axis for the whole launch -- so its per-bin optical constants,
// weights and table addresses are built once -- and pulls atmospheric columns from its tile's queue.  Per column:
//
//   S1  level geometry: interface p, T (R9), layer masses, k-table cell + bilinear corner weights per level
//   S2  band Planck B_b(T_level) for the tile's bins (piecewise-polynomial G, helios_rt_math.cuh), pi B_b(T_int)
//       -- both computed by the block itself into shared memory (no second kernel, no workspace round trip)
//   sweep 1 (TOA -> BOA), one thread = PPT adjacent spectral points of one bin, each a monochromatic two-stream
//       problem (the unit the paper solves independently, L449/L592): S3 bilinear ln(kappa) + exp (the four
//       k-table corner rows of a level reach shared memory by one-dimensional bulk async copies -- TMA -- into a
//       per-warp two-stage ring guarded by mbarriers, or by register-prefetched loads), S4 omega0/g0/dtau, tau
//       prefix and direct beam (Eq. B6), S5 layer coefficients (Eq. 19, B1, B2, B5, B8, Eq. 11 guard) and the
//       forward elimination of S6.  The block-tridiagonal system of Eq.(12) has one non-zero in each off-diagonal
//       2x2 block, so Eqs.(13)-(14) reduce to the scalar recurrences (R, U, c, d) below, carried in registers.
//       The back-substitution coefficients (c, W d, R) of every interface go to a per-block slab of a global
//       workspace sized to the resident grid (coalesced 16-byte stores), which the persistent block reuses column
//       after column.  Where the slabs of the whole grid fit the 126 MB L2 (config 3: 75 MB) they stay there; at the
//       default config-2 shape they do not (141 MiB: about 40 % of the row stores are written back to HBM and 0.2 GB
//       read again, 0.83 GB of DRAM traffic per launch; DESIGN.md section 9 has the measurements).  Lines are
//       discarded (discard.global.L2) once sweep 2 has read them, which saves the write-back of those still in L2.
//   sweep 2 (BOA -> TOA): back-substitution Eq.(15) fused with S7, the Gauss-/bin-weighted reduction (shared-memory
//       transposes + warp shuffles, then a fixed-order sum over warps and tiles).
//
//   rt_iter_kernel   the pair-wise iterative scheme the paper replaces (helios_rt_step_iterative; comparison only).
//
// The layer relations are used in transmission/reflection form.  With zeta+- and T of Eq.(B2),
//   t = psi/chi = s T / (a b),  r = -xi/chi = zeta+ zeta- (1 - T^2) / (a b),
//   a = zeta+ - zeta- T,  b = zeta+ + zeta- T,  s = zeta+ - zeta-,  1 - t - r = s (1 - T) / b,
// Eqs.(2),(3) read  F_up[j+1] = t F_up[j] + r F_dn[j+1] + S_up,  F_dn[j] = t F_dn[j+1] + r F_up[j] + S_dn.
// These forms avoid the cancellations of chi + xi - psi and 1 - T^2.



#include "helios_rt_kernels.cuh"

#include <mutex>

namespace {

using namespace hrt;
using namespace hrt_k;

// --------------------------------------------------------------------------------------------
// host side
// --------------------------------------------------------------------------------------------
__global__ void zero_kernel(double *p, size_t n) {
  for (size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x)
    p[i] = 0.0;
}

// all compiled instantiations of rt_step_kernel, class by class; filled exactly once (std::call_once), so host threads
// that create handles at the same time all see the complete table
Variant kVariants[64];
int kNumVariants = 0;
std::once_flag kVariantsOnce;
void collect_variants() {
  std::call_once(kVariantsOnce, [] {
    const Variant *tabs[4] = {kVariantsIsoFull, kVariantsIsoToa, kVariantsNoniso, kVariantsSampling};
    const int n[4] = {kNumIsoFull, kNumIsoToa, kNumNoniso, kNumSampling};
    int k = 0;
    for (int t = 0; t < 4; ++t)
      for (int i = 0; i < n[t] && k < 64; ++i) kVariants[k++] = tabs[t][i];
    kNumVariants = k;
  });
}

typedef void (*iter_fn)(const KParams, const int);

// spectral points per thread: columns whose number of Gauss points is a multiple of it, with enough points
// to fill the tiles.  2 with the back-substitution pass (isothermal and non-isothermal), 4 in isothermal TOA mode.
int default_ppt(int npt, int ng, bool noniso, bool toa) {
  const bool can2 = ng > 1 && (ng % 2) == 0, can4 = can2 && !noniso && toa && (ng % 4) == 0;
  if (npt < 256) return 1;
  return can4 ? 4 : (can2 ? 2 : 1);
}

// warps per block: tiles of 128 spectral points for long columns; small columns take the
// block with the fewest padded lanes, ties -> larger block (fewer tiles)
int default_warps(int npt, int ppt, bool noniso) {
  if (npt >= 256) return ppt == 4 ? 1 : (ppt == 2 ? 2 : 4);
  int best = 1;
  long best_waste = -1;
  for (int w = 1; w <= 4; ++w) {
    const long tp = 32L * w * ppt, tiles = (npt + tp - 1) / tp;
    const long waste = tiles * tp - npt;
    if (best_waste < 0 || waste < best_waste || (waste == best_waste && w > best)) { best = w; best_waste = waste; }
  }
  return best;
}

}  // namespace


struct helios_rt {
  helios_rt_config cfg;   // pointers nulled
  int npt, nlev;
  bool noniso, toa;
  // launch shape of rt_step_kernel
  int variant, warps, ppt, tiles, workers, occ;
  Lay lay;
  int iter_warps, iter_tiles;      // rt_iter_kernel keeps one point per thread
  unsigned row_stride;
  double inv_dlp, inv_dt;
  // device tables
  double *d_lnk, *d_tab_lp, *d_tab_t, *d_edges, *d_gw, *d_gtab, *d_c2lam;
  BinConst *d_bins;
  // workspace
  double *d_stack, *d_partial;
  unsigned char *d_ws_rec, *d_ws_B;
  size_t stack_block, stack_bytes, partial_bytes, ws_bytes;
  unsigned *d_counter, *d_queue, *d_flags;
  BinSlot *d_bslot, *d_bslot_iter;
  int *d_slot_ptr, *d_slots, *d_slot_ptr_iter, *d_slots_iter;   // bin -> Planck-block slots (step tiling / comparison tiling)
  Lay iter_lay;
  double *inv_dlam;          // host copy, [n_bins]
  // device + pinned host staging for step_host
  double *d_in, *d_out, *h_in, *h_out;
  cudaStream_t own_stream;   // step_host runs on it
  int regs, lmem, sm_count;
  int force_two_launches;   // helios_rt_debug_force_two_launches: always take the fallback path (tests)
  int force_stuck;          // helios_rt_debug_force_stuck: the next steps never see their columns published (tests)
  unsigned *h_err, *d_err;  // error word: page-locked mapped host memory and its device alias (KParams::err)
  int workers_cap;          // helios_rt_debug_set_workers: upper bound of workers per tile (0 = none; tuning runs)
  cudaError_t last_err;
};

#define CK(h, call)                                                   \
  do {                                                                \
    cudaError_t e_ = (call);                                          \
    if (e_ != cudaSuccess) { if (h) (h)->last_err = e_; return HELIOS_RT_ECUDA; } \
  } while (0)

extern "C" const char *helios_rt_strerror(int code) {
  switch (code) {
    case HELIOS_RT_OK: return "success";
    case HELIOS_RT_EINVAL: return "invalid argument";
    case HELIOS_RT_ENOMEM: return "out of memory";
    case HELIOS_RT_ECUDA: return "CUDA runtime error (see helios_rt_last_cuda_error)";
    case HELIOS_RT_ENODEV: return "no usable CUDA device (compute capability 10.x required)";
    case HELIOS_RT_ESTUCK: return "a step of this handle gave up waiting for a column's level data (its publication flag never "
                                  "arrived); the outputs of that step are invalid";
    case HELIOS_RT_ETOOBIG: return "problem too large for the built-in scratch array of helios_rt_phase_curve_noalloc "
                                   "(HELIOS_RT_PHASE_CURVE_NOALLOC_MAX_BYTES); use helios_rt_phase_curve with your own workspace";
    default: return "unknown error code";
  }
}

extern "C" const char *helios_rt_last_cuda_error(const helios_rt *h) {
  if (!h || h->last_err == cudaSuccess) return "";
  return cudaGetErrorString(h->last_err);
}

static int check_device() {
  int n = 0;
  if (cudaGetDeviceCount(&n) != cudaSuccess || n == 0) { cudaGetLastError(); return HELIOS_RT_ENODEV; }
  int dev = 0, major = 0;
  if (cudaGetDevice(&dev) != cudaSuccess) return HELIOS_RT_ENODEV;
  cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev);
  return major == 10 ? HELIOS_RT_OK : HELIOS_RT_ENODEV;
}

static bool strictly_ascending(const double *a, int n) {
  for (int i = 0; i < n; ++i) if (!(a[i] == a[i])) return false;
  for (int i = 1; i < n; ++i) if (!(a[i] > a[i - 1])) return false;
  return true;
}

static int validate_config(const helios_rt_config *c) {
  if (!c) return HELIOS_RT_EINVAL;
  if (c->n_layers < 1 || c->n_layers > MAXL || c->n_bins < 1 || c->n_gauss < 1 || c->n_ktab_p < 2 ||
      c->n_ktab_t < 2 || c->max_columns < 1)
    return HELIOS_RT_EINVAL;
  if ((long long)c->n_bins * c->n_gauss > (1 << 24)) return HELIOS_RT_EINVAL;
  if ((long long)c->n_ktab_p * c->n_ktab_t * ((long long)c->n_bins * c->n_gauss + 2) >= (1LL << 31)) return HELIOS_RT_EINVAL;   // 32-bit table offsets
  if (!c->ktab_p || !c->ktab_t || !c->ktab || !c->bin_edges || !c->gauss_w || !c->scat_gas || !c->cloud_ext ||
      !c->cloud_w0 || !c->cloud_g0)
    return HELIOS_RT_EINVAL;
  if (c->flags & ~(HELIOS_RT_IMPROVED | HELIOS_RT_NONISOTHERMAL | HELIOS_RT_TOA_SPECTRUM)) return HELIOS_RT_EINVAL;
  if (!strictly_ascending(c->ktab_p, c->n_ktab_p) || !(c->ktab_p[0] > 0)) return HELIOS_RT_EINVAL;
  if (!strictly_ascending(c->ktab_t, c->n_ktab_t)) return HELIOS_RT_EINVAL;
  if (!strictly_ascending(c->bin_edges, c->n_bins + 1) || !(c->bin_edges[0] > 0)) return HELIOS_RT_EINVAL;
  double sw = 0;
  for (int g = 0; g < c->n_gauss; ++g) { if (!(c->gauss_w[g] > 0)) return HELIOS_RT_EINVAL; sw += c->gauss_w[g]; }
  if (!(fabs(sw - 1.0) <= 1e-10)) return HELIOS_RT_EINVAL;
  for (int b = 0; b < c->n_bins; ++b) {
    if (!(c->scat_gas[b] >= 0) || !(c->cloud_ext[b] >= 0)) return HELIOS_RT_EINVAL;
    if (!(c->cloud_w0[b] >= 0 && c->cloud_w0[b] <= 1)) return HELIOS_RT_EINVAL;
    if (!(c->cloud_g0[b] >= 0 && c->cloud_g0[b] < 1)) return HELIOS_RT_EINVAL;
  }
  if (!(c->gravity > 0) || !(c->cp > 0) || !(c->eps2 > 0) || !(c->e_tau >= 0) || !(c->gcrit_tol >= 0) ||
      !(c->w0_transition >= 0) || !(c->f_toa >= 0))
    return HELIOS_RT_EINVAL;
  if (!(c->cloud_p_top == c->cloud_p_top) || !(c->cloud_p_bot == c->cloud_p_bot)) return HELIOS_RT_EINVAL;
  // kappa in [1e-300, 1e300]: |ln kappa| <= 691 stays inside the domain of the table exp (|x| <= 708)
  const size_t nk = (size_t)c->n_ktab_p * c->n_ktab_t * c->n_bins * c->n_gauss;
  for (size_t i = 0; i < nk; ++i) if (!(c->ktab[i] >= 1e-300) || !(c->ktab[i] <= 1e300)) return HELIOS_RT_EINVAL;
  return HELIOS_RT_OK;
}

template <class T>
static cudaError_t upload(T **dst, const T *src, size_t n) {
  cudaError_t e = cudaMalloc((void **)dst, sizeof(T) * n);
  if (e != cudaSuccess) return e;
  return cudaMemcpy(*dst, src, sizeof(T) * n, cudaMemcpyHostToDevice);
}

extern "C" int helios_rt_destroy(helios_rt *h) {
  if (!h) return HELIOS_RT_OK;
  cudaFree(h->d_lnk); cudaFree(h->d_tab_lp); cudaFree(h->d_tab_t); cudaFree(h->d_edges); cudaFree(h->d_gw);
  cudaFree(h->d_gtab); cudaFree(h->d_c2lam); cudaFree(h->d_bins); cudaFree(h->d_partial); cudaFree(h->d_counter); cudaFree(h->d_queue);
  cudaFree(h->d_stack); cudaFree(h->d_in); cudaFree(h->d_out);
  cudaFree(h->d_ws_rec); cudaFree(h->d_ws_B); cudaFree(h->d_flags);
  cudaFree(h->d_slot_ptr); cudaFree(h->d_slots); cudaFree(h->d_slot_ptr_iter); cudaFree(h->d_slots_iter);
  cudaFree(h->d_bslot); cudaFree(h->d_bslot_iter);
  free(h->inv_dlam);
  if (h->h_in) cudaFreeHost(h->h_in);
  if (h->h_out) cudaFreeHost(h->h_out);
  if (h->h_err) cudaFreeHost(h->h_err);
  if (h->own_stream) cudaStreamDestroy(h->own_stream);
  delete h;
  return HELIOS_RT_OK;
}

// bin -> slots of the per-(column, tile) Planck blocks: bin b is stored once in the block of every tile that owns
// points of it, at row offset (b - first bin of the tile)
static int build_slots(helios_rt *h, int tp, const Lay &lay, const double *inv_dlam, int **d_ptr, int **d_slots,
                       BinSlot **d_bslot) {
  const int nb = h->cfg.n_bins, ng = h->cfg.n_gauss;
  int *ptr = (int *)malloc(sizeof(int) * (nb + 1));
  int total = 0;
  if (!ptr) return HELIOS_RT_ENOMEM;
  for (int b = 0; b < nb; ++b) { ptr[b] = total; total += ((b + 1) * ng - 1) / tp - (b * ng) / tp + 1; }
  ptr[nb] = total;
  int *sl = (int *)malloc(sizeof(int) * (total > 0 ? total : 1));
  if (!sl) { free(ptr); return HELIOS_RT_ENOMEM; }
  for (int b = 0, k = 0; b < nb; ++b)
    for (int t = (b * ng) / tp; t <= ((b + 1) * ng - 1) / tp; ++t) sl[k++] = t * (int)(lay.b_bytes / 8) + (b - (t * tp) / ng);
  BinSlot *bs = (BinSlot *)malloc(sizeof(BinSlot) * nb);
  if (!bs) { free(ptr); free(sl); return HELIOS_RT_ENOMEM; }
  for (int b = 0; b < nb; ++b) {
    const int n = ptr[b + 1] - ptr[b];
    bs[b].s0 = sl[ptr[b]];
    bs[b].s1 = n == 1 ? -1 : (n == 2 ? sl[ptr[b] + 1] : -2);
    bs[b].inv_dlam = inv_dlam[b];
  }
  cudaError_t e = cudaMalloc((void **)d_ptr, sizeof(int) * (nb + 1));
  if (e == cudaSuccess) e = cudaMemcpy(*d_ptr, ptr, sizeof(int) * (nb + 1), cudaMemcpyHostToDevice);
  if (e == cudaSuccess) e = cudaMalloc((void **)d_bslot, sizeof(BinSlot) * nb);
  if (e == cudaSuccess) e = cudaMemcpy(*d_bslot, bs, sizeof(BinSlot) * nb, cudaMemcpyHostToDevice);
  free(bs);
  if (e == cudaSuccess) e = cudaMalloc((void **)d_slots, sizeof(int) * (total > 0 ? total : 1));
  if (e == cudaSuccess) e = cudaMemcpy(*d_slots, sl, sizeof(int) * (total > 0 ? total : 1), cudaMemcpyHostToDevice);
  free(ptr); free(sl);
  if (e != cudaSuccess) { h->last_err = e; return e == cudaErrorMemoryAllocation ? HELIOS_RT_ENOMEM : HELIOS_RT_ECUDA; }
  return HELIOS_RT_OK;
}

// launch shape + workspace for the chosen variant / warps per block.  Frees and re-allocates the workspace whose size
// depends on the shape; called by create and by helios_rt_debug_set_launch.
static int configure_launch(helios_rt *h) {
  const helios_rt_config &c = h->cfg;
  const Variant &v = kVariants[h->variant];
  const int N = c.n_layers;
  h->ppt = v.ppt;
  if (h->warps * 32 > v.maxt || (v.warps != 0 && v.warps != h->warps)) return HELIOS_RT_EINVAL;
  const int tp = h->warps * 32 * h->ppt;
  h->tiles = (h->npt + tp - 1) / tp;
  h->lay = make_lay(N, h->nlev, h->warps, h->ppt, c.n_gauss, c.n_bins, h->toa, h->noniso ? 2 : 1, v.rows, v.bdirect);
  h->iter_lay = make_lay(N, h->nlev, h->iter_warps, 1, c.n_gauss, c.n_bins, false, h->noniso ? 2 : 1, 0, false);
  if (h->lay.total > 227u * 1024u) return HELIOS_RT_EINVAL;
  CK(h, cudaFuncSetAttribute(v.fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)h->lay.total));
  cudaFuncAttributes fa;
  CK(h, cudaFuncGetAttributes(&fa, v.fn));
  h->regs = fa.numRegs;
  h->lmem = (int)fa.localSizeBytes;
  CK(h, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&h->occ, v.fn, h->warps * 32, h->lay.total));
  if (h->occ < 1) return HELIOS_RT_EINVAL;
  // persistent grid: as many blocks as are resident at once, split evenly over the tiles; never more workers per
  // tile than columns
  long workers = (long)h->sm_count * h->occ / h->tiles;
  if (workers < 1) workers = 1;
  if (workers > c.max_columns) workers = c.max_columns;
  if (h->workers_cap > 0 && workers > h->workers_cap) workers = h->workers_cap;
  h->workers = (int)workers;
  // workspace
  cudaFree(h->d_stack); h->d_stack = nullptr;
  cudaFree(h->d_partial); h->d_partial = nullptr;
  cudaFree(h->d_queue); h->d_queue = nullptr;
  cudaFree(h->d_ws_rec); h->d_ws_rec = nullptr;
  cudaFree(h->d_ws_B); h->d_ws_B = nullptr;
  {
    // S1/S2 blocks of every column: sized for the step kernel's tiling and for the comparison kernel's
    size_t bB = (size_t)h->tiles * h->lay.b_bytes;
    if (!h->toa && (size_t)h->iter_tiles * h->iter_lay.b_bytes > bB) bB = (size_t)h->iter_tiles * h->iter_lay.b_bytes;
    const size_t bR = h->lay.rec_bytes;   // the same for both (depends on N and nlev only)
    h->ws_bytes = (size_t)c.max_columns * (bB + bR);
    CK(h, cudaMalloc((void **)&h->d_ws_rec, (size_t)c.max_columns * bR));
    CK(h, cudaMalloc((void **)&h->d_ws_B, (size_t)c.max_columns * bB));
  }
  cudaFree(h->d_slot_ptr); h->d_slot_ptr = nullptr;
  cudaFree(h->d_slots); h->d_slots = nullptr;
  cudaFree(h->d_slot_ptr_iter); h->d_slot_ptr_iter = nullptr;
  cudaFree(h->d_slots_iter); h->d_slots_iter = nullptr;
  cudaFree(h->d_bslot); h->d_bslot = nullptr;
  cudaFree(h->d_bslot_iter); h->d_bslot_iter = nullptr;
  {
    int rc = build_slots(h, tp, h->lay, h->inv_dlam, &h->d_slot_ptr, &h->d_slots, &h->d_bslot);
    if (rc == HELIOS_RT_OK && !h->toa)
      rc = build_slots(h, h->iter_warps * 32, h->iter_lay, h->inv_dlam, &h->d_slot_ptr_iter, &h->d_slots_iter, &h->d_bslot_iter);
    if (rc) return rc;
  }
  // back-substitution workspace: per block [warp][N + 1 rows][96 ppt]
  h->stack_block = (size_t)(N + 1) * h->warps * 96 * h->ppt;
  h->stack_bytes = !h->toa ? sizeof(double) * h->stack_block * h->tiles * h->workers : 0;
  if (h->stack_bytes) CK(h, cudaMalloc((void **)&h->d_stack, h->stack_bytes));
  const int mt = h->tiles > h->iter_tiles ? h->tiles : h->iter_tiles;
  h->partial_bytes = sizeof(double) * (size_t)c.max_columns * mt * 4 * (N + 1);
  CK(h, cudaMalloc((void **)&h->d_partial, h->partial_bytes));
  CK(h, cudaMalloc((void **)&h->d_queue, sizeof(unsigned) * (h->tiles + 2)));
  CK(h, cudaMemset(h->d_queue, 0, sizeof(unsigned) * (h->tiles + 2)));
  return HELIOS_RT_OK;
}

// first instantiation of the class that matches; one compiled for exactly `warps` warps is preferred to a generic one
static int find_variant(bool noniso, bool toa, bool bdirect, int ppt, int rows, int maxt, int minb, int warps) {
  for (int pass = 0; pass < 2; ++pass)
  for (int i = 0; i < kNumVariants; ++i) {
    const Variant &v = kVariants[i];
    if (v.noniso != noniso || v.toa != toa || v.bdirect != bdirect || v.ppt != ppt) continue;
    if (pass == 0 ? v.warps != warps : v.warps != 0) continue;
    if (rows >= 0 && v.rows != rows) continue;
    if (maxt >= 0 && v.maxt != maxt) continue;
    if (minb >= 0 && v.minb != minb) continue;
    return i;
  }
  return -1;
}

extern "C" int helios_rt_create(const helios_rt_config *cfg, helios_rt **out) {
  if (!out) return HELIOS_RT_EINVAL;
  *out = nullptr;
  int rc = validate_config(cfg);
  if (rc) return rc;
  rc = check_device();
  if (rc) return rc;
  collect_variants();
  helios_rt *h = new (std::nothrow) helios_rt();
  if (!h) return HELIOS_RT_ENOMEM;
  memset(h, 0, sizeof(*h));
  h->cfg = *cfg;
  h->cfg.ktab_p = h->cfg.ktab_t = h->cfg.ktab = h->cfg.bin_edges = h->cfg.gauss_w = nullptr;
  h->cfg.scat_gas = h->cfg.cloud_ext = h->cfg.cloud_w0 = h->cfg.cloud_g0 = nullptr;
  const int N = cfg->n_layers, nb = cfg->n_bins, ng = cfg->n_gauss;
  h->npt = nb * ng;
  h->noniso = (cfg->flags & HELIOS_RT_NONISOTHERMAL) != 0;
  h->toa = (cfg->flags & HELIOS_RT_TOA_SPECTRUM) != 0;
  h->nlev = h->noniso ? 2 * N + 1 : N;
  h->iter_warps = default_warps(h->npt, 1, false);
  h->iter_tiles = (h->npt + h->iter_warps * 32 - 1) / (h->iter_warps * 32);
  int ppt = default_ppt(h->npt, ng, h->noniso, h->toa);
  h->warps = default_warps(h->npt, ppt, h->noniso);
  h->variant = find_variant(h->noniso, h->toa, ng == 1, ppt, -1, -1, -1, h->warps);
  if (h->variant < 0) {
    ppt = 1;
    h->warps = default_warps(h->npt, 1, h->noniso);
    h->variant = find_variant(h->noniso, h->toa, ng == 1, 1, -1, -1, -1, h->warps);
  }
  int dev = 0;
  cudaGetDevice(&dev);
  cudaDeviceGetAttribute(&h->sm_count, cudaDevAttrMultiProcessorCount, dev);
  if (h->variant < 0) { helios_rt_destroy(h); return HELIOS_RT_EINVAL; }

  // ln(kappa) table (rows padded to an even length, zero-filled, + a tail so that a warp's bulk copy of its 32 PPT
  // points never leaves the allocation), log10 pressure grid, per-bin constants, Planck polynomial pieces
  h->row_stride = (unsigned)((h->npt + 1) & ~1);
  const size_t nrows = (size_t)cfg->n_ktab_p * cfg->n_ktab_t;
  const size_t nk = nrows * h->row_stride + 256;
  double *lnk = (double *)calloc(nk, sizeof(double));
  double *lp = (double *)malloc(sizeof(double) * cfg->n_ktab_p);
  BinConst *bins = (BinConst *)malloc(sizeof(BinConst) * nb);
  double *gtab = (double *)malloc(sizeof(double) * kGIntervals * kGCoef);
  if (!lnk || !lp || !bins || !gtab) { free(lnk); free(lp); free(bins); free(gtab); helios_rt_destroy(h); return HELIOS_RT_ENOMEM; }
  for (size_t r = 0; r < nrows; ++r)
    for (int i = 0; i < h->npt; ++i) lnk[r * h->row_stride + i] = log(cfg->ktab[r * h->npt + i]);
  for (int i = 0; i < cfg->n_ktab_p; ++i) lp[i] = log10(cfg->ktab_p[i]);
  h->inv_dlp = (cfg->n_ktab_p - 1) / (lp[cfg->n_ktab_p - 1] - lp[0]);
  h->inv_dt = (cfg->n_ktab_t - 1) / (cfg->ktab_t[cfg->n_ktab_t - 1] - cfg->ktab_t[0]);
  for (int b = 0; b < nb; ++b) {
    // Eqs.(17)-(18) in per-mass units: sb = what is added to kappa_abs, ss = scattering part, gg = g0
    BinConst &bc = bins[b];
    bc.dlam = cfg->bin_edges[b + 1] - cfg->bin_edges[b];
    bc.inv_dlam = 1.0 / bc.dlam;
    const double sg = cfg->scat_gas[b], kc = cfg->cloud_ext[b], sc = cfg->cloud_w0[b] * kc;
    bc.sb[0] = sg;            bc.sb[1] = sg + kc;
    bc.ss[0] = sg;            bc.ss[1] = sg + sc;
    bc.gg[0] = 0.0;           bc.gg[1] = (sg + sc > 0.0) ? sc * cfg->cloud_g0[b] / (sg + sc) : 0.0;
    // omega0 = ss / (kappa_abs + sb) must stay below 1 after rounding (E - omega0 = 0 is the singular conservative limit,
    // SURVEY.md Q5): a purely scattering constituent is capped one ulp below its extinction
    for (int cl = 0; cl < 2; ++cl)
      if (bc.ss[cl] > bc.sb[cl] * (1.0 - 0x1p-52)) bc.ss[cl] = bc.sb[cl] * (1.0 - 0x1p-52);
  }
  build_planck_table(gtab);
  h->inv_dlam = (double *)malloc(sizeof(double) * nb);
  if (!h->inv_dlam) { free(lnk); free(lp); free(bins); free(gtab); helios_rt_destroy(h); return HELIOS_RT_ENOMEM; }
  for (int b = 0; b < nb; ++b) h->inv_dlam[b] = bins[b].inv_dlam;
  cudaError_t e = cudaSuccess;
  auto step = [&](cudaError_t r) { if (e == cudaSuccess) e = r; };
  step(upload(&h->d_lnk, lnk, nk));
  step(upload(&h->d_tab_lp, lp, (size_t)cfg->n_ktab_p));
  step(upload(&h->d_tab_t, cfg->ktab_t, (size_t)cfg->n_ktab_t));
  step(upload(&h->d_edges, cfg->bin_edges, (size_t)nb + 1));
  step(upload(&h->d_gw, cfg->gauss_w, (size_t)ng));
  step(upload(&h->d_bins, bins, (size_t)nb));
  step(upload(&h->d_gtab, gtab, (size_t)kGIntervals * kGCoef));
  {
    double *c2l = (double *)malloc(sizeof(double) * (nb + 1));
    if (!c2l) step(cudaErrorMemoryAllocation);
    else {
      for (int i = 0; i <= nb; ++i) c2l[i] = kPlanckC2 / cfg->bin_edges[i];
      step(upload(&h->d_c2lam, c2l, (size_t)nb + 1));
      free(c2l);
    }
  }
  free(lnk); free(lp); free(bins); free(gtab);
  const size_t ncol = (size_t)cfg->max_columns;
  step(cudaMalloc((void **)&h->d_counter, sizeof(unsigned) * ncol));
  if (e == cudaSuccess) step(cudaMemset(h->d_counter, 0, sizeof(unsigned) * ncol));
  step(cudaMalloc((void **)&h->d_flags, sizeof(unsigned) * ncol));
  if (e == cudaSuccess) step(cudaMemset(h->d_flags, 0, sizeof(unsigned) * ncol));
  // step_host staging: inputs packed as [p | T | mu | F*], outputs as [F_up | F_down | F_net | F_beam | dTdt | toa]
  const size_t n_in = ncol * (2 * (size_t)N + 1) + nb, n_out = ncol * (4 * ((size_t)N + 1) + N + nb);
  step(cudaMalloc((void **)&h->d_in, sizeof(double) * n_in));
  step(cudaMalloc((void **)&h->d_out, sizeof(double) * n_out));
  step(cudaStreamCreateWithFlags(&h->own_stream, cudaStreamNonBlocking));
  step(cudaHostAlloc((void **)&h->h_err, 64, cudaHostAllocMapped));
  if (e == cudaSuccess) {
    memset(h->h_err, 0, 64);
    step(cudaHostGetDevicePointer((void **)&h->d_err, h->h_err, 0));
  }
  if (e == cudaSuccess) {
    iter_fn it = h->noniso ? rt_iter_kernel<true> : rt_iter_kernel<false>;
    if (!h->toa)
      step(cudaFuncSetAttribute(it, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                (int)make_lay(N, h->nlev, h->iter_warps, 1, ng, nb, false, h->noniso ? 2 : 1, 0, false).total));
  }
  if (e != cudaSuccess) {
    const bool oom = (e == cudaErrorMemoryAllocation);
    helios_rt_destroy(h);
    cudaGetLastError();
    return oom ? HELIOS_RT_ENOMEM : HELIOS_RT_ECUDA;
  }
  rc = configure_launch(h);
  if (rc) {
    const bool oom = (h->last_err == cudaErrorMemoryAllocation);
    helios_rt_destroy(h);
    cudaGetLastError();
    return oom ? HELIOS_RT_ENOMEM : rc;
  }
  *out = h;
  return HELIOS_RT_OK;
}

static int validate_step(const helios_rt *h, const helios_rt_inputs *in, const helios_rt_outputs *out) {
  if (!h || !in || !out) return HELIOS_RT_EINVAL;
  if (in->n_columns < 0 || in->n_columns > h->cfg.max_columns) return HELIOS_RT_EINVAL;
  if (in->n_columns == 0) return in->f_internal >= 0 ? HELIOS_RT_OK : HELIOS_RT_EINVAL;   // nothing to do
  if (in->n_columns > 0 && (!in->p || !in->T || !in->mu_star || !in->stellar_flux)) return HELIOS_RT_EINVAL;
  if (!(in->f_internal >= 0)) return HELIOS_RT_EINVAL;
  const bool any_flux = out->F_up || out->F_down || out->F_net || out->dTdt || out->F_beam;
  if (h->toa) { if (!out->F_up_toa_bin || any_flux) return HELIOS_RT_EINVAL; }
  else if (!any_flux && !out->F_up_toa_bin) return HELIOS_RT_EINVAL;
  return HELIOS_RT_OK;
}

// Enqueues one step on `st`: rt_step_kernel (n_iter == 0) or the comparison scheme rt_prep_kernel + rt_iter_kernel
// (n_iter > 0).  Pointers in `in` / `out` are device pointers (or device aliases of mapped host memory).
static int launch_step(helios_rt *h, const helios_rt_inputs *in, const helios_rt_outputs *out, cudaStream_t st,
                       int n_iter = 0) {
  const helios_rt_config &c = h->cfg;
  if (in->n_columns == 0) return HELIOS_RT_OK;
  KParams P;
  P.lnk = h->d_lnk; P.tab_lp = h->d_tab_lp; P.tab_t = h->d_tab_t; P.edges = h->d_edges; P.gauss_w = h->d_gw;
  P.bins = h->d_bins; P.gtab = h->d_gtab; P.c2lam = h->d_c2lam;
  P.nP = c.n_ktab_p; P.nT = c.n_ktab_t; P.N = c.n_layers; P.nlev = h->nlev; P.nb = c.n_bins; P.ng = c.n_gauss; P.npt = h->npt;
  P.tiles = n_iter > 0 ? h->iter_tiles : h->tiles;
  P.ncol = in->n_columns;
  P.row_stride = h->row_stride; P.inv_dlp = h->inv_dlp; P.inv_dt = h->inv_dt;
  P.cloud_p_top = c.cloud_p_top; P.cloud_p_bot = c.cloud_p_bot; P.inv_g = 1.0 / c.gravity; P.inv_cp = 1.0 / c.cp;
  P.inv_eps2 = 1.0 / c.eps2; P.e_tau = c.e_tau; P.gcrit_tol = c.gcrit_tol; P.w0_transition = (c.flags & HELIOS_RT_IMPROVED) ? c.w0_transition : INFINITY;   // regular two-stream: E = 1
  P.f_toa = c.f_toa;
  P.p = in->p; P.T = in->T; P.mu = in->mu_star; P.fstar = in->stellar_flux;
  P.T_int = in->f_internal > 0 ? sqrt(sqrt(in->f_internal / kSigmaSB)) : 0.0;
  P.F_up = out->F_up; P.F_down = out->F_down; P.F_net = out->F_net; P.dTdt = out->dTdt; P.F_beam = out->F_beam;
  P.F_toa_bin = out->F_up_toa_bin;
  P.ws_rec = h->d_ws_rec; P.ws_B = h->d_ws_B; P.flags = h->d_flags;
  P.slot_ptr = h->d_slot_ptr; P.slots = h->d_slots; P.bslot = h->d_bslot;
  P.fused_prep = 0;
  P.stack = h->d_stack; P.stack_block = h->stack_block;
  P.partial = h->d_partial; P.counter = h->d_counter; P.queue = h->d_queue;
  P.err = h->d_err; P.poll_limit = h->force_stuck ? 64u : (1u << 26);
  if (n_iter > 0) {
    if (in->n_columns > 65535) return HELIOS_RT_EINVAL;   // the comparison kernel puts columns in gridDim.y
    iter_fn fn = h->noniso ? rt_iter_kernel<true> : rt_iter_kernel<false>;
    const Lay &lay = h->iter_lay;
    const long items = (long)in->n_columns * (h->nlev + 1);
    const int pblocks = (int)((items + 127) / 128 < 16L * h->sm_count ? (items + 127) / 128 : 16L * h->sm_count);
    P.slot_ptr = h->d_slot_ptr_iter; P.slots = h->d_slots_iter; P.bslot = h->d_bslot_iter;
    if (h->noniso) rt_prep_kernel<true><<<pblocks, 128, 0, st>>>(P, h->iter_warps * 32, 0, 0);
    else rt_prep_kernel<false><<<pblocks, 128, 0, st>>>(P, h->iter_warps * 32, 0, 0);
    CK(h, cudaGetLastError());
    dim3 grid((unsigned)h->iter_tiles, (unsigned)in->n_columns);
    fn<<<grid, h->iter_warps * 32, lay.total, st>>>(P, n_iter);
    CK(h, cudaGetLastError());
    return HELIOS_RT_OK;
  }
  // bins that straddle two tiles are accumulated with atomics: start from zero
  const int tp = h->warps * 32 * h->ppt;
  if (P.F_toa_bin && h->tiles > 1 && (tp % c.n_gauss) != 0) {
    const size_t n = (size_t)in->n_columns * c.n_bins;
    zero_kernel<<<(unsigned)((n + 255) / 256 < 1024 ? (n + 255) / 256 : 1024), 256, 0, st>>>(P.F_toa_bin, n);
  }
  int workers = h->workers;
  if (workers > in->n_columns) workers = in->n_columns;
  // One cooperative launch: phase A (S1 + S2 of all columns, spread over the grid) and phase B (the sweeps) in the same
  // kernel; blocks of phase B wait on per-column publication flags, which is safe because the cooperative launch
  // guarantees that the whole grid is resident.  If the device cannot host the grid at once (another context's kernels
  // hold SMs), phase A runs as a launch of its own instead.
  cudaLaunchConfig_t lc;
  memset(&lc, 0, sizeof(lc));
  lc.gridDim = dim3((unsigned)h->tiles, (unsigned)workers);
  lc.blockDim = dim3((unsigned)(h->warps * 32));
  lc.dynamicSmemBytes = h->lay.total;
  lc.stream = st;
  cudaLaunchAttribute attr;
  attr.id = cudaLaunchAttributeCooperative;
  attr.val.cooperative = 1;
  lc.attrs = &attr;
  lc.numAttrs = 1;
  P.fused_prep = 1;
  void *args[1] = {&P};
  if (h->force_stuck) {   // tests: no phase A at all, so no column is ever published and every block gives up
    P.fused_prep = 0;
    lc.numAttrs = 0;
    CK(h, cudaLaunchKernelExC(&lc, kVariants[h->variant].fn, args));
    return HELIOS_RT_OK;
  }
  cudaError_t e = h->force_two_launches ? cudaErrorCooperativeLaunchTooLarge : cudaLaunchKernelExC(&lc, kVariants[h->variant].fn, args);
  if (e == cudaErrorCooperativeLaunchTooLarge || e == cudaErrorNotSupported) {
    cudaGetLastError();
    P.fused_prep = 0;
    const long items = (long)in->n_columns * (h->nlev + 1);
    const int pblocks = (int)((items + 127) / 128 < 16L * h->sm_count ? (items + 127) / 128 : 16L * h->sm_count);
    const int tp2 = h->warps * 32 * h->ppt;
    const int bd = kVariants[h->variant].bdirect ? 1 : 0;
    if (h->noniso) rt_prep_kernel<true><<<pblocks, 128, 0, st>>>(P, tp2, 1, bd);
    else rt_prep_kernel<false><<<pblocks, 128, 0, st>>>(P, tp2, 1, bd);
    CK(h, cudaGetLastError());
    lc.numAttrs = 0;
    e = cudaLaunchKernelExC(&lc, kVariants[h->variant].fn, args);
  }
  CK(h, e);
  return HELIOS_RT_OK;
}

// Reads and clears the handle's error word (written by the kernel through its device alias).  No synchronisation: a
// step still in flight is seen by a later call.
static bool take_stuck(helios_rt *h) {
  volatile unsigned *w = h->h_err;
  if (!w || *w == 0u) return false;
  *w = 0u;
  return true;
}

extern "C" int helios_rt_step(helios_rt *h, const helios_rt_inputs *in, const helios_rt_outputs *out,
                              void *cuda_stream) {
  const int rc = validate_step(h, in, out);
  if (rc) return rc;
  if (take_stuck(h)) return HELIOS_RT_ESTUCK;   // an EARLIER step of the handle: nothing is launched by this call
  return launch_step(h, in, out, (cudaStream_t)cuda_stream);
}

extern "C" int helios_rt_step_iterative(helios_rt *h, const helios_rt_inputs *in, const helios_rt_outputs *out,
                                        int32_t n_iterations, void *cuda_stream) {
  const int rc = validate_step(h, in, out);
  if (rc) return rc;
  if (n_iterations < 1 || h->toa || out->F_up_toa_bin) return HELIOS_RT_EINVAL;
  if (take_stuck(h)) return HELIOS_RT_ESTUCK;
  return launch_step(h, in, out, (cudaStream_t)cuda_stream, n_iterations);
}

// device alias of a host pointer that the device can write directly (page-locked, mapped: cudaHostAlloc /
// cudaHostRegister memory under unified addressing); nullptr for pageable memory
static double *mapped_alias(double *host) {
  cudaPointerAttributes a;
  if (cudaPointerGetAttributes(&a, host) != cudaSuccess) { cudaGetLastError(); return nullptr; }
  return a.type == cudaMemoryTypeHost ? (double *)a.devicePointer : nullptr;
}

extern "C" int helios_rt_step_host(helios_rt *h, const helios_rt_inputs *in, const helios_rt_outputs *out) {
  int rc = validate_step(h, in, out);
  if (rc) return rc;
  if (take_stuck(h)) return HELIOS_RT_ESTUCK;   // an earlier asynchronous step of the handle
  if (in->n_columns == 0) return HELIOS_RT_OK;
  const size_t ncol = (size_t)in->n_columns, N = (size_t)h->cfg.n_layers, nb = (size_t)h->cfg.n_bins;
  cudaStream_t st = h->own_stream;
  double *d_p = h->d_in, *d_T = d_p + ncol * N, *d_mu = d_T + ncol * N, *d_fs = d_mu + ncol;
  CK(h, cudaMemcpyAsync(d_p, in->p, sizeof(double) * ncol * N, cudaMemcpyHostToDevice, st));
  CK(h, cudaMemcpyAsync(d_T, in->T, sizeof(double) * ncol * N, cudaMemcpyHostToDevice, st));
  CK(h, cudaMemcpyAsync(d_mu, in->mu_star, sizeof(double) * ncol, cudaMemcpyHostToDevice, st));
  CK(h, cudaMemcpyAsync(d_fs, in->stellar_flux, sizeof(double) * nb, cudaMemcpyHostToDevice, st));
  helios_rt_inputs din = *in;
  din.p = d_p; din.T = d_T; din.mu_star = d_mu; din.stellar_flux = d_fs;
  // Outputs.  Page-locked, mapped host buffers are written by the kernel itself (each column's results leave over
  // PCIe as soon as its last tile has summed them, under the sweeps of the other columns); pageable buffers, and a
  // per-bin spectrum whose bins straddle tiles (accumulated with atomics), go through device staging and a copy each.
  const int tp = h->warps * 32 * h->ppt;
  const bool toa_atomics = h->tiles > 1 && (tp % h->cfg.n_gauss) != 0;
  double *const host[6] = {out->F_up, out->F_down, out->F_net, out->F_beam, out->dTdt, out->F_up_toa_bin};
  const size_t ni = ncol * (N + 1);
  const size_t count[6] = {ni, ni, ni, ni, ncol * N, ncol * nb};
  double *dev[6], *stage = h->d_out;
  bool staged[6];
  for (int k = 0; k < 6; ++k) {
    dev[k] = nullptr;
    staged[k] = false;
    if (host[k]) {
      double *alias = (k == 5 && toa_atomics) ? nullptr : mapped_alias(host[k]);
      dev[k] = alias ? alias : stage;
      staged[k] = alias == nullptr;
    }
    stage += count[k];
  }
  helios_rt_outputs dout;
  dout.F_up = dev[0]; dout.F_down = dev[1]; dout.F_net = dev[2]; dout.F_beam = dev[3]; dout.dTdt = dev[4];
  dout.F_up_toa_bin = dev[5];
  rc = launch_step(h, &din, &dout, st);
  if (rc) return rc;
  for (int k = 0; k < 6; ++k)
    if (staged[k]) CK(h, cudaMemcpyAsync(host[k], dev[k], sizeof(double) * count[k], cudaMemcpyDeviceToHost, st));
  CK(h, cudaStreamSynchronize(st));
  return take_stuck(h) ? HELIOS_RT_ESTUCK : HELIOS_RT_OK;   // this very step
}

extern "C" int helios_rt_launch_info(const helios_rt *h, int32_t info[8]) {
  if (!h || !info) return HELIOS_RT_EINVAL;
  info[0] = h->warps * 32; info[1] = h->tiles; info[2] = (int32_t)h->lay.total; info[3] = h->regs; info[4] = h->occ;
  info[5] = h->lmem;
  // rt_step_kernel, + 1 zero-fill launch where F_up_toa_bin is accumulated with atomics (bins that straddle tiles)
  info[6] = (h->toa && h->tiles > 1 && ((h->warps * 32 * h->ppt) % h->cfg.n_gauss) != 0) ? 2 : 1;
  info[7] = h->sm_count;
  return HELIOS_RT_OK;
}

// ---- include/helios_rt_debug.h: not part of the product API ----
extern "C" int helios_rt_debug_set_launch(helios_rt *h, int32_t warps, int32_t ppt, int32_t rows, int32_t maxt,
                                          int32_t minb) {
  if (!h) return HELIOS_RT_EINVAL;
  const Variant &cur = kVariants[h->variant];
  const int want_ppt = ppt > 0 ? ppt : cur.ppt;
  if (want_ppt > 1 && (h->cfg.n_gauss % want_ppt) != 0) return HELIOS_RT_EINVAL;
  const int want_warps = warps > 0 ? warps : h->warps;
  const int v = find_variant(h->noniso, h->toa, cur.bdirect, want_ppt, rows, maxt, minb, want_warps);
  if (v < 0) return HELIOS_RT_EINVAL;
  const int old_v = h->variant, old_w = h->warps;
  h->variant = v;
  h->warps = want_warps;
  int rc = configure_launch(h);
  if (rc) { h->variant = old_v; h->warps = old_w; configure_launch(h); }
  return rc;
}

extern "C" int helios_rt_debug_set_workers(helios_rt *h, int32_t workers) {
  if (!h || workers < 0) return HELIOS_RT_EINVAL;
  const int old = h->workers_cap;
  h->workers_cap = workers;
  int rc = configure_launch(h);
  if (rc) { h->workers_cap = old; configure_launch(h); }
  return rc;
}

extern "C" int helios_rt_debug_force_stuck(helios_rt *h, int32_t on) {
  if (!h) return HELIOS_RT_EINVAL;
  h->force_stuck = on != 0;
  return HELIOS_RT_OK;
}

extern "C" int helios_rt_debug_force_two_launches(helios_rt *h, int32_t on) {
  if (!h) return HELIOS_RT_EINVAL;
  h->force_two_launches = on != 0;
  return HELIOS_RT_OK;
}

extern "C" int helios_rt_debug_get_launch(const helios_rt *h, int32_t info[16]) {
  if (!h || !info) return HELIOS_RT_EINVAL;
  const Variant &v = kVariants[h->variant];
  info[0] = h->warps; info[1] = v.ppt; info[2] = v.rows; info[3] = 0; info[4] = v.maxt; info[5] = v.minb;
  info[6] = h->tiles; info[7] = h->workers; info[8] = h->occ; info[9] = h->regs; info[10] = h->lmem;
  info[11] = (int32_t)h->lay.total; info[12] = (int32_t)(h->stack_bytes >> 20); info[13] = h->variant;
  info[14] = kNumVariants; info[15] = 0;
  return HELIOS_RT_OK;
}
