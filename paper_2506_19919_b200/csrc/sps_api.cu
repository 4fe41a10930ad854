// sps_api.cu -- C-ABI entry points (include/sps.h), error plumbing and scratch management.
#include <algorithm>
#include <atomic>
#include <cstdarg>
#include <cstdio>
#include <cstring>
#include "sps_internal.h"
#include "sps_ptx.cuh"

static thread_local char g_err[512] = "";
static std::atomic<int64_t> g_launches{0};

void sps_set_error(const char* fmt, ...) {
  va_list ap; va_start(ap, fmt);
  vsnprintf(g_err, sizeof(g_err), fmt, ap);
  va_end(ap);
}
void sps_count_launch(int n) { g_launches += n; }
extern "C" int64_t sps_launch_count(void) { return g_launches.load(); }
extern "C" const char* sps_last_error(void) { return g_err; }
extern "C" const char* sps_version(void) { return "sps-b200 0.1 (sm_100a)"; }

// ---- optional per-kernel event timing ---------------------------------------------------------
#include <vector>
struct ProfSlot { std::vector<cudaEvent_t> ev; int64_t launches = 0; bool open = false; };
static ProfSlot g_prof[SPS_K_COUNT];
static int g_prof_on = 0, g_prof_stride = 1;
void sps_prof_begin(int id, cudaStream_t s) {
  if (!g_prof_on) return;
  ProfSlot& P = g_prof[id];
  P.open = (P.launches++ % g_prof_stride) == 0 && P.ev.size() < 16384;
  if (!P.open) return;
  cudaEvent_t e; cudaEventCreate(&e); cudaEventRecord(e, s); P.ev.push_back(e);
}
void sps_prof_end(int id, cudaStream_t s) {
  if (!g_prof_on) return;
  ProfSlot& P = g_prof[id];
  if (!P.open) return;
  cudaEvent_t e; cudaEventCreate(&e); cudaEventRecord(e, s); P.ev.push_back(e); P.open = false;
}
bool sps_prof_enabled() { return g_prof_on != 0; }
extern "C" sps_status sps_profile(int enable, int stride) {
  g_prof_on = enable; g_prof_stride = stride > 0 ? stride : 1;
  for (auto& P : g_prof) { for (auto e : P.ev) cudaEventDestroy(e); P.ev.clear(); P.launches = 0; P.open = false; }
  return SPS_OK;
}
extern "C" sps_status sps_profile_read(int id, double* total_ms, int64_t* timed, int64_t* all) {
  if (id < 0 || id >= SPS_K_COUNT || !total_ms || !timed || !all) { sps_set_error("sps_profile_read: bad argument"); return SPS_EINVAL; }
  cudaDeviceSynchronize();
  ProfSlot& P = g_prof[id];
  double tot = 0; int64_t n = 0;
  for (size_t i = 0; i + 1 < P.ev.size(); i += 2) { float ms = 0; if (cudaEventElapsedTime(&ms, P.ev[i], P.ev[i + 1]) == cudaSuccess) { tot += ms; ++n; } }
  *total_ms = tot; *timed = n; *all = P.launches;
  for (auto e : P.ev) cudaEventDestroy(e);
  P.ev.clear(); P.launches = 0;
  return SPS_OK;
}

sps_status sps_check_cuda(cudaError_t e, const char* what) {
  if (e == cudaSuccess) return SPS_OK;
  sps_set_error("%s: %s", what, cudaGetErrorString(e));
  return e == cudaErrorMemoryAllocation ? SPS_ENOMEM : SPS_ECUDA;
}

sps_status sps_require_device() {
  int dev = 0, major = 0;
  if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev) != cudaSuccess) {
    cudaGetLastError();
    sps_set_error("no CUDA device: this library has no CPU fallback");
    return SPS_EUNSUPPORTED;
  }
  if (major != 10) { sps_set_error("device compute capability %d.x is not sm_100: unsupported", major); return SPS_EUNSUPPORTED; }
  return SPS_OK;
}

// ---- library options ---------------------------------------------------------------------------------
static std::atomic<int> g_options[SPS_OPT_COUNT];
int sps_option(int option) { return (option >= 0 && option < SPS_OPT_COUNT) ? g_options[option].load() : 0; }
extern "C" sps_status sps_set_option(int option, int value) {
  if (option < 0 || option >= SPS_OPT_COUNT) { sps_set_error("sps_set_option: unknown option %d", option); return SPS_EINVAL; }
  g_options[option].store(value);
  return SPS_OK;
}

SpsEncodeTiledFn sps_tensor_map_encoder() {
  static SpsEncodeTiledFn fn_cached = nullptr;
  if (fn_cached) return fn_cached;
  void* fn = nullptr;
  cudaDriverEntryPointQueryResult qr;
  if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qr) != cudaSuccess || !fn || qr != cudaDriverEntryPointSuccess) {
    cudaGetLastError();
    sps_set_error("cuTensorMapEncodeTiled is not available from this driver");
    return nullptr;
  }
  fn_cached = (SpsEncodeTiledFn)fn;
  return fn_cached;
}

// ---- pipe peaks measured in the same run as the kernels (bench.py's "alu" roofline denominators) ---------------------
// what = SPS_PEAK_MUFU: ex2.approx operations per second; SPS_PEAK_FFMA: fp32 fused multiply-adds per second.  Every SM
// runs 64 warps of eight independent dependency chains per thread; timed with CUDA events on `stream`; synchronises.
template <int WHAT> __global__ void __launch_bounds__(256) peak_kernel(float* out, int iters) {
  float x[8];
#pragma unroll
  for (int k = 0; k < 8; ++k) x[k] = 0.25f + 0.01f * (float)((threadIdx.x + k) & 31);
  for (int i = 0; i < iters; ++i) {
#pragma unroll
    for (int k = 0; k < 8; ++k) {
      if (WHAT == SPS_PEAK_MUFU) asm volatile("ex2.approx.ftz.f32 %0, %1;" : "=f"(x[k]) : "f"(-x[k]));     // stays in (0.5, 1]
      else asm volatile("fma.rn.f32 %0, %0, %1, %2;" : "+f"(x[k]) : "f"(0.999f), "f"(0.001f));
    }
  }
  float s = 0.f;
#pragma unroll
  for (int k = 0; k < 8; ++k) s += x[k];
  if (s == 123.456f) out[0] = s;                             // never true: keeps the chains alive
}
extern "C" sps_status sps_measure_peak(int what, double* per_second, void* stream) {
  if ((what != SPS_PEAK_MUFU && what != SPS_PEAK_FFMA) || !per_second) { sps_set_error("sps_measure_peak: bad argument"); return SPS_EINVAL; }
  sps_status st = sps_require_device(); if (st != SPS_OK) return st;
  cudaStream_t s = (cudaStream_t)stream;
  int dev = 0, sms = 0; cudaGetDevice(&dev); cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
  float* out = nullptr;
  st = sps_check_cuda(cudaMalloc(&out, sizeof(float)), "sps_measure_peak"); if (st != SPS_OK) return st;
  const int iters = what == SPS_PEAK_MUFU ? 4096 : 16384, blocks = sms * 8;
  cudaEvent_t e0, e1; cudaEventCreate(&e0); cudaEventCreate(&e1);
  double best = 0.0;
  for (int rep = 0; rep < 4; ++rep) {                        // first repetition warms the clocks up
    cudaEventRecord(e0, s);
    if (what == SPS_PEAK_MUFU) peak_kernel<SPS_PEAK_MUFU><<<blocks, 256, 0, s>>>(out, iters);
    else peak_kernel<SPS_PEAK_FFMA><<<blocks, 256, 0, s>>>(out, iters);
    cudaEventRecord(e1, s);
    sps_count_launch();
    st = sps_check_cuda(cudaEventSynchronize(e1), "sps_measure_peak"); if (st != SPS_OK) break;
    float ms = 0.f; cudaEventElapsedTime(&ms, e0, e1);
    if (rep > 0 && ms > 0.f) best = std::max(best, (double)blocks * 256.0 * 8.0 * iters / (ms * 1e-3));
  }
  cudaEventDestroy(e0); cudaEventDestroy(e1); cudaFree(out);
  *per_second = best;
  return st;
}

// ---- SPS_OPT_CHECK_FINITE -------------------------------------------------------------------------------
__global__ void check_finite_kernel(const float* __restrict__ a, int64_t na, const float* __restrict__ b, int64_t nb,
                                    const float* __restrict__ pos, int64_t np, int* __restrict__ bad) {
  const int64_t stride = (int64_t)gridDim.x * blockDim.x;
  int f = 0;
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < na; i += stride) f |= !isfinite(a[i]);
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < nb; i += stride) f |= !isfinite(b[i]);
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < np; i += stride) f |= !(isfinite(pos[i]) && pos[i] > 0.f);
  if (__any_sync(FULL_MASK, f) && (threadIdx.x & 31) == 0) atomicOr(bad, 1);
}
sps_status sps_check_finite(const float* a, int64_t na, const float* b, int64_t nb, const float* pos, int64_t np, cudaStream_t s) {
  if (!sps_option(SPS_OPT_CHECK_FINITE)) return SPS_OK;
  int* bad = nullptr;
  sps_status st = sps_check_cuda(cudaMalloc(&bad, sizeof(int)), "finite-check flag");
  if (st != SPS_OK) return st;
  cudaMemsetAsync(bad, 0, sizeof(int), s);
  const int64_t tot = std::max<int64_t>(std::max(a ? na : 0, b ? nb : 0), pos ? np : 0);
  check_finite_kernel<<<(unsigned)std::min<int64_t>(1024, (tot + 255) / 256 + 1), 256, 0, s>>>(a, a ? na : 0, b, b ? nb : 0, pos, pos ? np : 0, bad);
  sps_count_launch();
  int h = 0;
  st = sps_check_cuda(cudaMemcpyAsync(&h, bad, sizeof(int), cudaMemcpyDeviceToHost, s), "finite check");
  if (st == SPS_OK) st = sps_check_cuda(cudaStreamSynchronize(s), "finite check");
  cudaFree(bad);
  if (st == SPS_OK && h) { sps_set_error("non-finite parameter or observation, or sigma <= 0, in the inputs (SPS_OPT_CHECK_FINITE)"); return SPS_ENONFINITE; }
  return st;
}

// ---- scratch per (table, stream) ----------------------------------------------------------------------------
static void free_row_buffers(RowBuffers& B) {
  void* ptrs[] = {B.a, B.m, B.a_bar, B.m_bar, B.sc, B.flux, B.part, B.order, B.bins, B.cell_list};
  for (void* p : ptrs) if (p) cudaFree(p);
  B = RowBuffers();
}
// ---- cache of device blocks for the samplers' per-run state ---------------------------------------------------------
// sps_hmc_run / sps_leapfrog need a few buffers per call (chain state, row lists, NUTS trees).  cudaFree of such a block was
// measured at 150-700 ms every few calls on a busy device (a 2.7 s run: +15 %), so the blocks go back to a process-wide
// cache instead and are handed to the next run of the same size; sps_destroy_table releases the ones not in use.
namespace {
struct PoolBlock { void* p; size_t bytes; int dev; bool used; };
std::mutex g_pool_mu;
std::vector<PoolBlock> g_pool;
}  // namespace
cudaError_t sps_pool_alloc(void** p, size_t bytes) {
  int dev = 0;
  cudaGetDevice(&dev);
  bytes = std::max<size_t>(bytes, 256);
  {
    std::lock_guard<std::mutex> lock(g_pool_mu);
    PoolBlock* best = nullptr;
    for (auto& b : g_pool)
      if (!b.used && b.dev == dev && b.bytes >= bytes && b.bytes <= 2 * bytes + 4096 && (!best || b.bytes < best->bytes)) best = &b;
    if (best) { best->used = true; *p = best->p; return cudaSuccess; }
  }
  const cudaError_t e = cudaMalloc(p, bytes);
  if (e == cudaSuccess) { std::lock_guard<std::mutex> lock(g_pool_mu); g_pool.push_back(PoolBlock{*p, bytes, dev, true}); }
  return e;
}
void sps_pool_free(void* p) {
  if (!p) return;
  std::lock_guard<std::mutex> lock(g_pool_mu);
  for (auto& b : g_pool) if (b.p == p) { b.used = false; return; }
  cudaFree(p);                                               // (not one of ours)
}
void sps_pool_release_unused() {
  std::lock_guard<std::mutex> lock(g_pool_mu);
  size_t k = 0;
  for (size_t i = 0; i < g_pool.size(); ++i) {
    if (g_pool[i].used) g_pool[k++] = g_pool[i];
    else cudaFree(g_pool[i].p);
  }
  g_pool.resize(k);
}

void sps_free_workspace(Workspace* ws) {
  if (!ws) return;
  free_row_buffers(ws->rows);
  sps_exact_free_scratch(ws->x);
  delete ws;
}
Workspace* sps_workspace(const sps_table* t, cudaStream_t s) {
  std::lock_guard<std::mutex> lock(t->mu);
  Workspace*& w = t->ws[s];
  if (!w) w = new Workspace();
  t->last_ws = w;
  return w;
}

sps_status sps_ensure_row_buffers(const sps_table* t, Workspace& ws, int64_t n, cudaStream_t s) {
  RowBuffers& B = ws.rows;
  if (B.capacity >= n) return SPS_OK;
  cudaStreamSynchronize(s);                                  // earlier calls on this stream may still use the old scratch
  free_row_buffers(B);
  ws.bins_clean = false;
  const int64_t cap = n;
  cudaError_t e = cudaSuccess;
  auto al = [&](void** p, size_t bytes) { if (e == cudaSuccess) e = cudaMalloc(p, bytes); };
  al((void**)&B.a, cap * ROW_A_STRIDE * sizeof(float));
  al((void**)&B.a_bar, cap * ROW_A_STRIDE * sizeof(float));
  al((void**)&B.m, cap * ROW_M_STRIDE * sizeof(float));
  al((void**)&B.m_bar, cap * ROW_M_STRIDE * sizeof(float));
  al((void**)&B.sc, cap * sizeof(RowScalars));
  al((void**)&B.flux, cap * SPS_MAX_BAND * sizeof(float));
  al((void**)&B.part, cap * ROW_PARTS * ROW_A_STRIDE * sizeof(float));
  al((void**)&B.order, cap * sizeof(int));
  al((void**)&B.bins, 4 * (size_t)(t->dev.n_z + 1) * sizeof(int));
  // per-cell row lists for the approximate path (the prologue appends, the contraction walks them): [n_cells][cap] ints,
  // kept under 1 GiB (beyond that the rows are grouped by a scan / scatter pass instead)
  const size_t list_bytes = (size_t)std::max(t->dev.n_z - 1, 1) * cap * sizeof(int);
  if (t->dev.n_z >= 2 && list_bytes <= ((size_t)1 << 30) && t->approx_tc) { al((void**)&B.cell_list, list_bytes); B.cell_cap = cap; }
  if (e != cudaSuccess) { free_row_buffers(B); return sps_check_cuda(e, "row scratch allocation"); }
  B.capacity = cap;
  return SPS_OK;
}

// Bounds and prior of the table's model.  Slots that the model does not sample get the identity map and no prior.
sps_status sps_prior_to_dev(const sps_table* t, const sps_prior* p, PriorDev& out) {
  memset(&out, 0, sizeof(out));
  for (int i = 0; i < SPS_NDIM; ++i) { out.y_hi[i] = 1.f; out.k[i] = 1.f; out.omega[i] = 1.f; }
  if (!p) return SPS_OK;
  if (!p->y_lo || !p->y_hi || !p->k || !p->x0 || !p->xi || !p->omega || !p->skew) { sps_set_error("sps_prior: null array"); return SPS_EINVAL; }
  const int D = t->dev.n_dim;
  for (int i = 0; i < SPS_NDIM; ++i) {
    if (i < D && (!(p->y_hi[i] > p->y_lo[i]) || !(p->omega[i] > 0))) { sps_set_error("sps_prior: parameter %d needs y_hi > y_lo and omega > 0", i); return SPS_EINVAL; }
    out.y_lo[i] = (float)p->y_lo[i]; out.y_hi[i] = (float)p->y_hi[i]; out.k[i] = (float)p->k[i]; out.x0[i] = (float)p->x0[i];
    out.xi[i] = (float)p->xi[i]; out.omega[i] = (float)p->omega[i]; out.skew[i] = (float)p->skew[i];
  }
  if (t->dev.model == SPS_MODEL_DPL13 && !(p->y_lo[6] > p->y_hi[5])) {
    // Eq. (A7): sigma = (logT_max - logT_peak)/3 must stay positive over the whole box
    sps_set_error("sps_prior: the bounds must keep logT_max above logT_peak (y_lo[6] > y_hi[5])"); return SPS_EINVAL;
  }
  return SPS_OK;
}

sps_status sps_eval(const sps_table* t, Workspace& ws, const PriorDev& P, int path, const float* theta, int64_t n, bool unbounded,
                    bool with_prior, const int* rows, const int* gal_of_row, const float* obs_flux,
                    const float* obs_sigma, const float* flux_bar, bool want_grad, float* logp, float* grad,
                    cudaStream_t s, const LeapfrogFuse* lf, bool overlap) {
  const TableDev& T = t->dev;
  const LeapfrogFuse fuse = (lf && want_grad) ? *lf : LeapfrogFuse{nullptr, nullptr, nullptr, nullptr};
  if (T.model == SPS_MODEL_GAUSS_TEST) {
    launch_gauss_eval(T, theta, n, rows, logp, want_grad ? grad : nullptr, fuse, s);
    return sps_check_cuda(cudaGetLastError(), "sps_eval launch");
  }
  const bool tiny5 = T.model == SPS_MODEL_TINY5, nonsep = T.agez_gamma != 0.f;
  const bool bucket = path == SPS_PATH_APPROX && !nonsep;   // the separable approximate kernels want rows grouped by z cell
  // tensor-core contraction on the prologue's cell lists: it leaves the cell counts cleared (Workspace::bins_clean)
  const bool direct_tc = bucket && sps_approx_tc_active(t) && ws.rows.cell_list != nullptr;
  if (tiny5) launch_prologue_tiny5(T, P, theta, n, unbounded, rows, ws.rows, bucket, s);
  else launch_prologue(T, P, theta, n, unbounded, want_grad, rows, ws.rows, bucket, s, overlap, !(direct_tc && ws.bins_clean));
  if (bucket) ws.bins_clean = direct_tc;
  if (path == SPS_PATH_APPROX) {
    if (nonsep) launch_nonsep_approx(T, n, rows, gal_of_row, obs_flux, obs_sigma, flux_bar, want_grad, ws.rows, s);
    else if (sps_approx_tc_active(t)) {
      sps_status st = sps_approx_tc_contract(t, ws, n, rows, gal_of_row, obs_flux, obs_sigma, flux_bar, want_grad, s);
      if (st != SPS_OK) return st;
    } else launch_approx_contract(T, t->sm_count, n, rows, gal_of_row, obs_flux, obs_sigma, flux_bar, want_grad, ws.rows, s);
  } else {
    sps_status st = sps_exact_contract(t, ws, n, rows, gal_of_row, obs_flux, obs_sigma, flux_bar, want_grad, s);
    if (st != SPS_OK) return st;
  }
  if (want_grad || logp) {
    if (tiny5) launch_epilogue_tiny5(T, P, theta, n, unbounded, with_prior, rows, ws.rows, logp, want_grad ? grad : nullptr, fuse, s);
    else launch_epilogue(T, P, theta, n, unbounded, with_prior, rows, ws.rows, logp, want_grad ? grad : nullptr, fuse, s);
  }
  return sps_check_cuda(cudaGetLastError(), "sps_eval launch");
}

#define REQUIRE(cond, msg) do { if (!(cond)) { sps_set_error("%s: %s", __func__, msg); return SPS_EINVAL; } } while (0)

extern "C" int32_t sps_model_ndim(const sps_table* t) { return t ? t->dev.n_dim : -1; }

extern "C" sps_status sps_weights(const sps_table* t, const sps_prior* prior, const float* theta, int64_t n, int unbounded,
                                  float* w_age, float* w_met, float* mstar, void* stream) {
  REQUIRE(n >= 0, "negative n");
  if (n == 0) return SPS_OK;
  REQUIRE(t && theta, "null table or theta");
  REQUIRE(t->dev.model != SPS_MODEL_GAUSS_TEST, "the Gaussian test model has no SSP weights");
  REQUIRE(!unbounded || prior, "unbounded parameters need a prior (bounds)");
  sps_status st = sps_require_device(); if (st != SPS_OK) return st;
  cudaStream_t s = (cudaStream_t)stream;
  PriorDev P; st = sps_prior_to_dev(t, prior, P); if (st != SPS_OK) return st;
  st = sps_check_finite(theta, n * SPS_NDIM, nullptr, 0, nullptr, 0, s); if (st != SPS_OK) return st;
  Workspace& ws = *sps_workspace(t, s);
  st = sps_ensure_row_buffers(t, ws, n, s); if (st != SPS_OK) return st;
  if (t->dev.model == SPS_MODEL_TINY5) launch_prologue_tiny5(t->dev, P, theta, n, unbounded != 0, nullptr, ws.rows, false, s);
  else launch_prologue(t->dev, P, theta, n, unbounded != 0, false, nullptr, ws.rows, false, s);
  launch_copy_weights(t->dev, n, ws.rows, w_age, w_met, mstar, s);
  return sps_check_cuda(cudaGetLastError(), "sps_weights launch");
}

extern "C" sps_status sps_photometry(const sps_table* t, const sps_prior* prior, int path, const float* theta, int64_t n,
                                     int unbounded, float* flux, const float* flux_bar, float* theta_bar, void* stream) {
  REQUIRE(n >= 0, "negative n");
  if (n == 0) return SPS_OK;
  REQUIRE(t && theta && flux, "null table, theta or flux");
  REQUIRE(t->dev.model != SPS_MODEL_GAUSS_TEST, "the Gaussian test model has no photometry");
  REQUIRE(path == SPS_PATH_EXACT || path == SPS_PATH_APPROX, "bad path");
  REQUIRE(!unbounded || prior, "unbounded parameters need a prior (bounds)");
  REQUIRE((flux_bar == nullptr) == (theta_bar == nullptr), "flux_bar and theta_bar must be given together");
  sps_status st = sps_require_device(); if (st != SPS_OK) return st;
  cudaStream_t s = (cudaStream_t)stream;
  PriorDev P; st = sps_prior_to_dev(t, prior, P); if (st != SPS_OK) return st;
  st = sps_check_finite(theta, n * SPS_NDIM, flux_bar, n * t->dev.n_band, nullptr, 0, s); if (st != SPS_OK) return st;
  Workspace& ws = *sps_workspace(t, s);
  st = sps_ensure_row_buffers(t, ws, n, s); if (st != SPS_OK) return st;
  const bool vjp = flux_bar != nullptr;
  // with flux_bar == NULL the contraction needs no observations: it is told so by a dummy flux_bar = flux buffer
  st = sps_eval(t, ws, P, path, theta, n, unbounded != 0, false, nullptr, nullptr, nullptr, nullptr,
                vjp ? flux_bar : ws.rows.flux /* ignored: want_grad = false */, vjp, nullptr, theta_bar, s);
  if (st != SPS_OK) return st;
  launch_copy_flux(t->dev, n, ws.rows, flux, s);
  return sps_check_cuda(cudaGetLastError(), "sps_photometry launch");
}

extern "C" sps_status sps_loglike_grad(const sps_table* t, const sps_prior* prior, int path, const float* theta_unb, int64_t n,
                                       const int32_t* gal_of_row, const float* obs_flux, const float* obs_sigma, float* logp,
                                       float* grad, void* stream) {
  REQUIRE(n >= 0, "negative n");
  if (n == 0) return SPS_OK;
  REQUIRE(t && theta_unb, "null argument");
  const bool gauss = t->dev.model == SPS_MODEL_GAUSS_TEST;
  REQUIRE(gauss || (prior && obs_flux && obs_sigma), "null argument");
  REQUIRE(logp || grad, "nothing to compute");
  REQUIRE(path == SPS_PATH_EXACT || path == SPS_PATH_APPROX, "bad path");
  sps_status st = sps_require_device(); if (st != SPS_OK) return st;
  cudaStream_t s = (cudaStream_t)stream;
  PriorDev P; st = sps_prior_to_dev(t, prior, P); if (st != SPS_OK) return st;
  st = sps_check_finite(theta_unb, n * SPS_NDIM, nullptr, 0, nullptr, 0, s); if (st != SPS_OK) return st;
  Workspace& ws = *sps_workspace(t, s);
  if (!gauss) { st = sps_ensure_row_buffers(t, ws, n, s); if (st != SPS_OK) return st; }
  return sps_eval(t, ws, P, path, theta_unb, n, true, true, nullptr, gal_of_row, obs_flux, obs_sigma, nullptr, grad != nullptr,
                  logp, grad, s);
}
