// sps_api.cu -- C-ABI entry points (include/sps.h), error plumbing and scratch management.
#include <atomic>
#include <cstdarg>
#include <cstdio>
#include <cstring>
#include "sps_internal.h"

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

void sps_free_row_buffers(sps_table* t) {
  RowBuffers& B = t->rows;
  void* ptrs[] = {B.a, B.m, B.a_bar, B.m_bar, B.sc, B.flux, B.part, B.order, B.bins};
  for (void* p : ptrs) if (p) cudaFree(p);
  B = RowBuffers();
}

sps_status sps_ensure_row_buffers(sps_table* t, int64_t n) {
  RowBuffers& B = t->rows;
  if (B.capacity >= n) return SPS_OK;
  cudaDeviceSynchronize();
  sps_free_row_buffers(t);
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
  if (e != cudaSuccess) { sps_free_row_buffers(t); return sps_check_cuda(e, "row scratch allocation"); }
  B.capacity = cap;
  return SPS_OK;
}

sps_status sps_prior_to_dev(const sps_prior* p, PriorDev& out) {
  memset(&out, 0, sizeof(out));
  for (int i = 0; i < SPS_NDIM; ++i) { out.y_hi[i] = 1.f; out.k[i] = 1.f; out.omega[i] = 1.f; }
  if (!p) return SPS_OK;
  if (!p->y_lo || !p->y_hi || !p->k || !p->x0 || !p->xi || !p->omega || !p->skew) { sps_set_error("sps_prior: null array"); return SPS_EINVAL; }
  for (int i = 0; i < SPS_NDIM; ++i) {
    if (!(p->y_hi[i] > p->y_lo[i]) || !(p->omega[i] > 0)) { sps_set_error("sps_prior: parameter %d needs y_hi > y_lo and omega > 0", i); return SPS_EINVAL; }
    out.y_lo[i] = (float)p->y_lo[i]; out.y_hi[i] = (float)p->y_hi[i]; out.k[i] = (float)p->k[i]; out.x0[i] = (float)p->x0[i];
    out.xi[i] = (float)p->xi[i]; out.omega[i] = (float)p->omega[i]; out.skew[i] = (float)p->skew[i];
  }
  return SPS_OK;
}

sps_status sps_eval(sps_table* t, const PriorDev& P, int path, const float* theta, int64_t n, bool unbounded,
                    bool with_prior, const int* rows, const int* gal_of_row, const float* obs_flux,
                    const float* obs_sigma, const float* flux_bar, bool want_grad, float* logp, float* grad,
                    cudaStream_t s, const LeapfrogFuse* lf) {
  const TableDev& T = t->dev;
  launch_prologue(T, P, theta, n, unbounded, want_grad, rows, t->rows, path == SPS_PATH_APPROX, s);
  if (path == SPS_PATH_APPROX) {
    if (sps_approx_tc_active(t)) {
      sps_status st = sps_approx_tc_contract(t, n, rows, gal_of_row, obs_flux, obs_sigma, flux_bar, want_grad, s);
      if (st != SPS_OK) return st;
    } else launch_approx_contract(T, n, rows, gal_of_row, obs_flux, obs_sigma, flux_bar, want_grad, t->rows, s);
  } else {
    sps_status st = sps_exact_contract(t, n, rows, gal_of_row, obs_flux, obs_sigma, flux_bar, want_grad, s);
    if (st != SPS_OK) return st;
  }
  if (want_grad || logp) launch_epilogue(T, P, theta, n, unbounded, with_prior, rows, t->rows, logp, want_grad ? grad : nullptr,
                                           (lf && want_grad) ? *lf : LeapfrogFuse{nullptr, nullptr, nullptr, nullptr}, s);
  return sps_check_cuda(cudaGetLastError(), "sps_eval launch");
}

#define REQUIRE(cond, msg) do { if (!(cond)) { sps_set_error("%s: %s", __func__, msg); return SPS_EINVAL; } } while (0)

extern "C" sps_status sps_weights(const sps_table* tc, const sps_prior* prior, const float* theta, int64_t n, int unbounded,
                                  float* w_age, float* w_met, float* mstar, void* stream) {
  REQUIRE(n >= 0, "negative n");
  if (n == 0) return SPS_OK;
  REQUIRE(tc && theta, "null table or theta");
  REQUIRE(!unbounded || prior, "unbounded parameters need a prior (bounds)");
  sps_table* t = const_cast<sps_table*>(tc);
  PriorDev P; sps_status st = sps_prior_to_dev(prior, P); if (st != SPS_OK) return st;
  st = sps_ensure_row_buffers(t, n); if (st != SPS_OK) return st;
  cudaStream_t s = (cudaStream_t)stream;
  launch_prologue(t->dev, P, theta, n, unbounded != 0, false, nullptr, t->rows, false, s);
  launch_copy_weights(t->dev, n, t->rows, w_age, w_met, mstar, s);
  return sps_check_cuda(cudaGetLastError(), "sps_weights launch");
}

extern "C" sps_status sps_photometry(const sps_table* tc, const sps_prior* prior, int path, const float* theta, int64_t n,
                                     int unbounded, float* flux, const float* flux_bar, float* theta_bar, void* stream) {
  REQUIRE(n >= 0, "negative n");
  if (n == 0) return SPS_OK;
  REQUIRE(tc && theta && flux, "null table, theta or flux");
  REQUIRE(path == SPS_PATH_EXACT || path == SPS_PATH_APPROX, "bad path");
  REQUIRE(!unbounded || prior, "unbounded parameters need a prior (bounds)");
  REQUIRE((flux_bar == nullptr) == (theta_bar == nullptr), "flux_bar and theta_bar must be given together");
  if (n == 0) return SPS_OK;
  sps_table* t = const_cast<sps_table*>(tc);
  PriorDev P; sps_status st = sps_prior_to_dev(prior, P); if (st != SPS_OK) return st;
  st = sps_ensure_row_buffers(t, n); if (st != SPS_OK) return st;
  cudaStream_t s = (cudaStream_t)stream;
  const bool vjp = flux_bar != nullptr;
  // with flux_bar == NULL the contraction needs no observations: it is told so by a dummy flux_bar = flux buffer
  st = sps_eval(t, P, path, theta, n, unbounded != 0, false, nullptr, nullptr, nullptr, nullptr,
                vjp ? flux_bar : t->rows.flux /* ignored: want_grad = false */, vjp, nullptr, theta_bar, s);
  if (st != SPS_OK) return st;
  launch_copy_flux(t->dev, n, t->rows, flux, s);
  return sps_check_cuda(cudaGetLastError(), "sps_photometry launch");
}

extern "C" sps_status sps_loglike_grad(const sps_table* tc, const sps_prior* prior, int path, const float* theta_unb, int64_t n,
                                       const int32_t* gal_of_row, const float* obs_flux, const float* obs_sigma, float* logp,
                                       float* grad, void* stream) {
  REQUIRE(n >= 0, "negative n");
  if (n == 0) return SPS_OK;
  REQUIRE(tc && prior && theta_unb && obs_flux && obs_sigma, "null argument");
  REQUIRE(logp || grad, "nothing to compute");
  REQUIRE(path == SPS_PATH_EXACT || path == SPS_PATH_APPROX, "bad path");
  if (n == 0) return SPS_OK;
  sps_table* t = const_cast<sps_table*>(tc);
  PriorDev P; sps_status st = sps_prior_to_dev(prior, P); if (st != SPS_OK) return st;
  st = sps_ensure_row_buffers(t, n); if (st != SPS_OK) return st;
  return sps_eval(t, P, path, theta_unb, n, true, true, nullptr, gal_of_row, obs_flux, obs_sigma, nullptr, grad != nullptr,
                  logp, grad, (cudaStream_t)stream);
}
