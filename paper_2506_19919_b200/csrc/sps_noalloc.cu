// sps_noalloc.cu -- sps_loglike_grad_noalloc: the approximate-path log-posterior + gradient evaluation (a0-a5, a7, a9, a10;
// PAPER.md:77-87, 99, 438) for callers that may not allocate: code under CUDA graph capture, tight serving loops, harnesses
// that forbid cudaMalloc.  It is sps_loglike_grad(path = SPS_PATH_APPROX) with the per-row scratch (the weights a_i, m_j, the
// per-bin partials, a_bar, m_bar, the row scalars, the model fluxes, the z-cell grouping) placed in ONE file-scope device
// array of fixed size instead of the per-(table, stream) workspace that grows on demand.  The same kernels run (prologue,
// contraction, epilogue through sps_eval); nothing here calls cudaMalloc, cudaFree or an allocating library routine.
//
//  * Limit: n <= SPS_NOALLOC_MAX_ROWS rows per call and n_z <= SPS_NOALLOC_MAX_NZ redshift nodes; larger sizes are rejected
//    with SPS_ESHAPE.  The array is 15.8 MB (15.0 MiB); every GPU that loads the library holds it until the process exits.
//  * The array is shared by every call on the device and keeps the last call's contents.  What must start at zero (the
//    z-cell counts and cursors) is cleared by every call (a memset node in stream order); everything else is fully
//    overwritten for the rows of the call before it is read.
//  * Calls that overlap on the GPU (different streams, or graph branches without a dependency) RACE on the array: order
//    them.  The allocating entry points use their own per-stream workspaces and are not affected.
//  * In host code the array's name is a host-side stand-in, not a device address: its address is taken once per device,
//    with that device current, by cudaGetSymbolAddress, and the kernels are given pointers derived from it.  That first
//    call per device should be made outside graph capture (symbol resolution may load the module).
#include <mutex>
#include "sps_internal.h"

namespace {

constexpr size_t al256(size_t x) { return (x + 255) & ~(size_t)255; }
constexpr size_t NR = SPS_NOALLOC_MAX_ROWS;
constexpr size_t OFF_A = 0;
constexpr size_t OFF_ABAR = OFF_A + al256(NR * ROW_A_STRIDE * sizeof(float));
constexpr size_t OFF_M = OFF_ABAR + al256(NR * ROW_A_STRIDE * sizeof(float));
constexpr size_t OFF_MBAR = OFF_M + al256(NR * ROW_M_STRIDE * sizeof(float));
constexpr size_t OFF_SC = OFF_MBAR + al256(NR * ROW_M_STRIDE * sizeof(float));
constexpr size_t OFF_FLUX = OFF_SC + al256(NR * sizeof(RowScalars));
constexpr size_t OFF_PART = OFF_FLUX + al256(NR * SPS_MAX_BAND * sizeof(float));
constexpr size_t OFF_ORDER = OFF_PART + al256(NR * ROW_PARTS * ROW_A_STRIDE * sizeof(float));
constexpr size_t OFF_BINS = OFF_ORDER + al256(NR * sizeof(int));
constexpr size_t NOALLOC_BYTES = OFF_BINS + al256(4 * (size_t)(SPS_NOALLOC_MAX_NZ + 1) * sizeof(int));
static_assert(NOALLOC_BYTES <= ((size_t)16 << 20), "the no-allocation scratch is meant to stay modest");

}  // namespace

static __device__ __align__(256) unsigned char g_noalloc_scratch[NOALLOC_BYTES];

namespace {

constexpr int MAX_DEVICES = 64;
std::mutex g_mu;
unsigned char* g_scratch_ptr[MAX_DEVICES];      // device address of g_noalloc_scratch on each device, resolved on first use

// Device address of the scratch array on the CURRENT device (resolved once per device, with that device current).
sps_status scratch_address(unsigned char** out) {
  int dev = 0;
  sps_status st = sps_check_cuda(cudaGetDevice(&dev), "sps_loglike_grad_noalloc: cudaGetDevice");
  if (st != SPS_OK) return st;
  if (dev < 0 || dev >= MAX_DEVICES) { sps_set_error("sps_loglike_grad_noalloc: device ordinal %d out of range", dev); return SPS_EUNSUPPORTED; }
  std::lock_guard<std::mutex> lock(g_mu);
  if (!g_scratch_ptr[dev]) {
    void* p = nullptr;
    st = sps_check_cuda(cudaGetSymbolAddress(&p, g_noalloc_scratch), "sps_loglike_grad_noalloc: cudaGetSymbolAddress of the scratch array");
    if (st != SPS_OK) return st;
    if (!p) { sps_set_error("sps_loglike_grad_noalloc: the scratch array has no device address"); return SPS_ECUDA; }
    g_scratch_ptr[dev] = static_cast<unsigned char*>(p);
  }
  *out = g_scratch_ptr[dev];
  return SPS_OK;
}

}  // namespace

#define NA_REQUIRE(cond, msg) do { if (!(cond)) { sps_set_error("sps_loglike_grad_noalloc: %s", msg); return SPS_EINVAL; } } while (0)

extern "C" sps_status sps_loglike_grad_noalloc(const sps_table* t, const sps_prior* prior, const float* theta_unb, int64_t n,
                                               const int32_t* gal_of_row, const float* obs_flux, const float* obs_sigma,
                                               float* logp, float* grad, void* stream) {
  NA_REQUIRE(n >= 0, "negative n");
  if (n == 0) return SPS_OK;
  NA_REQUIRE(t && prior && theta_unb && obs_flux && obs_sigma, "null argument");
  NA_REQUIRE(logp || grad, "nothing to compute");
  NA_REQUIRE(t->dev.model != SPS_MODEL_GAUSS_TEST, "the Gaussian test model uses no scratch: call sps_loglike_grad");
  NA_REQUIRE(!sps_prof_enabled(), "the per-kernel profiling hooks create events: turn sps_profile off");
  if (n > SPS_NOALLOC_MAX_ROWS) {
    sps_set_error("sps_loglike_grad_noalloc: n = %lld rows exceeds SPS_NOALLOC_MAX_ROWS = %d (split the batch, or call sps_loglike_grad)",
                  (long long)n, SPS_NOALLOC_MAX_ROWS);
    return SPS_ESHAPE;
  }
  if (t->dev.n_z > SPS_NOALLOC_MAX_NZ) {
    sps_set_error("sps_loglike_grad_noalloc: the table's n_z = %d exceeds SPS_NOALLOC_MAX_NZ = %d", t->dev.n_z, SPS_NOALLOC_MAX_NZ);
    return SPS_ESHAPE;
  }
  sps_status st = sps_require_device(); if (st != SPS_OK) return st;
  PriorDev P; st = sps_prior_to_dev(t, prior, P); if (st != SPS_OK) return st;
  unsigned char* base = nullptr;
  st = scratch_address(&base); if (st != SPS_OK) return st;
  // a workspace view over the static array (no per-cell row lists: the rows are grouped by the scan / scatter pass over
  // `order` and `bins`, whose counts and cursors launch_prologue clears in stream order on every call)
  Workspace ws;
  RowBuffers& B = ws.rows;
  B.a = reinterpret_cast<float*>(base + OFF_A); B.a_bar = reinterpret_cast<float*>(base + OFF_ABAR);
  B.m = reinterpret_cast<float*>(base + OFF_M); B.m_bar = reinterpret_cast<float*>(base + OFF_MBAR);
  B.sc = reinterpret_cast<RowScalars*>(base + OFF_SC); B.flux = reinterpret_cast<float*>(base + OFF_FLUX);
  B.part = reinterpret_cast<float*>(base + OFF_PART); B.order = reinterpret_cast<int*>(base + OFF_ORDER);
  B.bins = reinterpret_cast<int*>(base + OFF_BINS);
  B.cell_list = nullptr; B.cell_cap = 0; B.capacity = SPS_NOALLOC_MAX_ROWS;
  ws.bins_clean = false;
  return sps_eval(t, ws, P, SPS_PATH_APPROX, theta_unb, n, true, true, nullptr, gal_of_row, obs_flux, obs_sigma, nullptr, grad != nullptr,
                  logp, grad, (cudaStream_t)stream);
}
