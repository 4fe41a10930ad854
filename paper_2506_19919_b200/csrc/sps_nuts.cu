// sps_nuts.cu -- NUTS engine (a13; reading R15).
//
// Multinomial NUTS with iterative doubling and O(depth) U-turn checkpoints, half a warp per chain (lane p < 13 of the half
// owns parameter p; a warp advances two chains).  The paper's finding is that lock-step batches of NUTS transitions run at the speed of the slowest
// chain.  Here the batch dimension is the LEAPFROG STEP, not the transition: every batch-wide step is
//   (1) one model evaluation (log-posterior + gradient) at each live chain's working point (sps_eval), then
//   (2) nuts_step_kernel: each chain advances its own state machine by one leaf -- finish the leapfrog, weigh the
//       leaf, update the subtree proposal and the U-turn checkpoints, and then either take the next leapfrog of the
//       subtree, merge the subtree and start the next doubling, or finish the transition (adaptation, sample record)
//       and start its next transition at once.
// A chain that finishes its tree never waits for the others; chains that have completed all their transitions are
// compacted out of the evaluation lists.  The counter-based RNG indexed by (chain, transition, purpose, index)
// makes the result independent of this scheduling.
//
// Leaf weights are kept as logarithms (log W, log-sum-exp): the decisions u W_sub < w and u < W_sub / W are taken as
// log u + log W_sub < -dH and log u < log W_sub - log W, which cannot overflow for dH << 0 early in warmup.
#include <vector>
#include "sps_sampler.cuh"

namespace {

enum { V_LQ = 0, V_LP, V_LG, V_RQ, V_RP, V_RG, V_RHO, V_PQ, V_PG, V_SRHO, V_SQ, V_SG, V_SPARE, V_PCK = 13, V_RCK = 13 + NUTS_MAX_DEPTH + 1 };
enum { F_FWD = 1, F_DIV = 2, F_HASSUB = 4 };

struct NutsScalars {
  float *logW, *logW_sub, *acc_sum, *prop_lp, *sub_lp;
  int *it, *depth, *leaf, *n_leaf, *flags, *done;
  int* n_done;                 // single counter
  int* depth_hist;             // [NUTS_MAX_DEPTH + 1] tree depths of the sampling phase
};

__device__ __forceinline__ float logaddexpf_(float a, float b) {
  const float hi = fmaxf(a, b), lo = fminf(a, b);
  if (hi == -INFINITY) return -INFINITY;
  return hi + log1pf(expf(lo - hi));
}

__device__ __forceinline__ float* vec(const ChainState& C, int64_t c, int v) { return C.nuts + (c * NUTS_VECTORS + v) * SPS_NDIM; }

// A chain occupies HALF a warp (16 lanes, 13 of them parameters), so a warp advances two chains: `hm` is the lane mask of the
// chain's half, and every collective of a chain names it (the two halves take different branches of the state machine).
__device__ __forceinline__ float sum16(float x, unsigned hm) {
#pragma unroll
  for (int o = 8; o > 0; o >>= 1) x += __shfl_xor_sync(hm, x, o);
  return x;
}

// generalised U-turn criterion: stop unless rho.(invM p_a) > 0 and rho.(invM p_b) > 0
__device__ __forceinline__ bool uturn(float rho, float pa, float pb, float v, bool act, unsigned hm) {
  const float da = sum16(act ? rho * v * pa : 0.f, hm), db = sum16(act ? rho * v * pb : 0.f, hm);
  return !(da > 0.f) || !(db > 0.f);
}

// start transition `it`: momentum draw, H0, single-node tree
__device__ __forceinline__ void begin_transition(ChainState& C, NutsScalars& S, int64_t c, int l, bool act, int64_t o, int it, uint2 key, unsigned hm) {
  float kin = 0.f;
  if (act) {
    const float v = C.inv_mass[o];
    const float p = l < C.D ? chain_normal(key, (uint32_t)C.rng_id[c], (uint32_t)it, RNG_MOMENTUM, l) * rsqrtf(v) : 0.f;
    kin = 0.5f * v * p * p;
    const float q = C.theta[o], g = C.grad[o];
    vec(C, c, V_LQ)[l] = q; vec(C, c, V_LP)[l] = p; vec(C, c, V_LG)[l] = g;
    vec(C, c, V_RQ)[l] = q; vec(C, c, V_RP)[l] = p; vec(C, c, V_RG)[l] = g;
    vec(C, c, V_RHO)[l] = p; vec(C, c, V_PQ)[l] = q; vec(C, c, V_PG)[l] = g;
  }
  kin = sum16(kin, hm);
  if (l == 0) {
    C.H0[c] = -C.logp[c] + kin;
    S.logW[c] = 0.f; S.acc_sum[c] = 0.f; S.prop_lp[c] = C.logp[c];
    S.n_leaf[c] = 0; S.depth[c] = 0; S.flags[c] = 0;
  }
}

// start the doubling at the current depth: pick the direction, take the first half kick and drift from that end
__device__ __forceinline__ void begin_doubling(ChainState& C, NutsScalars& S, int64_t c, int l, bool act, int64_t o, int it, int depth, int flags, uint2 key) {
  const float u = philox_u01(philox4x32_10(make_uint4((uint32_t)C.rng_id[c], (uint32_t)it, RNG_DIRECTION, (uint32_t)depth), key).x);
  const bool fwd = u < 0.5f;
  if (act) {
    const float eps = C.eps[c], step = fwd ? eps : -eps, v = C.inv_mass[o];
    const float q = vec(C, c, fwd ? V_RQ : V_LQ)[l], p = vec(C, c, fwd ? V_RP : V_LP)[l], g = vec(C, c, fwd ? V_RG : V_LG)[l];
    const float ph = p + 0.5f * step * g;
    C.p_w[o] = ph;
    C.theta_w[o] = q + step * v * ph;
    vec(C, c, V_SRHO)[l] = 0.f;
  }
  if (l == 0) {
    S.logW_sub[c] = -INFINITY; S.leaf[c] = 0;
    S.flags[c] = (flags & F_DIV) | (fwd ? F_FWD : 0);
  }
}

// two chains per warp: lanes 0-15 / 16-31
#define NUTS_HALF_PROLOGUE(SLOT_COUNT)                                                         \
  const int64_t slot = (((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5) * 2 + ((threadIdx.x >> 4) & 1); \
  const int l = threadIdx.x & 15;                                                              \
  const unsigned hm = 0xFFFFu << (threadIdx.x & 16);                                           \
  if (slot >= (SLOT_COUNT)) return;

__global__ void __launch_bounds__(256) nuts_begin_kernel(ChainState C, NutsScalars S, int first, uint2 key) {
  NUTS_HALF_PROLOGUE(C.n);
  const int64_t c = slot;
  const bool act = l < SPS_NDIM;
  const int64_t o = c * SPS_NDIM + (act ? l : 0);
  if (l == 0) { S.it[c] = 0; S.done[c] = 0; }
  begin_transition(C, S, c, l, act, o, first, key, hm);
  __syncwarp(hm);
  begin_doubling(C, S, c, l, act, o, first, 0, 0, key);
}

// One leaf per call for every live chain (see the header).  `live` lists the chains to advance (NULL: all).
__global__ void __launch_bounds__(256) nuts_step_kernel(ChainState C, NutsScalars S, WarmupSched W, int max_depth, uint2 key,
                                                        const int* __restrict__ live, int64_t n_live, float* __restrict__ samples) {
  NUTS_HALF_PROLOGUE(n_live);
  const int64_t c = live ? live[slot] : slot;
  if (S.done[c]) return;
  const bool act = l < SPS_NDIM;
  const int64_t o = c * SPS_NDIM + (act ? l : 0);
  const int it = S.it[c], depth = S.depth[c], leaf = S.leaf[c];
  const int tr = it + W.first;                               // transition index of the RNG streams (continued runs)
  int flags = S.flags[c];
  const bool fwd = flags & F_FWD;
  const float v = C.inv_mass[o], eps = C.eps[c], step = fwd ? eps : -eps;
  // ---- finish the leapfrog: second half kick with the gradient just evaluated at theta_w ----
  const float g = C.grad_w[o], q = C.theta_w[o], lp = C.logp_w[c];
  const float p = C.p_w[o] + 0.5f * step * g;
  const float kin = sum16(act ? 0.5f * v * p * p : 0.f, hm);
  float dH = -lp + kin - C.H0[c];
  const bool fin = __all_sync(hm, !act || (isfinite(g) && isfinite(q))) && isfinite(dH);
  if (!fin) dH = INFINITY;
  const float acc_sum = S.acc_sum[c] + expf(fminf(0.f, -dH));
  const int n_leaf = S.n_leaf[c] + 1;
  bool bad = false;
  float logW_sub = S.logW_sub[c];
  float rho_sub = 0.f;
  if (dH > 1000.f) { flags |= F_DIV; bad = true; }
  else {
    logW_sub = logaddexpf_(logW_sub, -dH);
    rho_sub = (act ? vec(C, c, V_SRHO)[l] : 0.f) + p;
    const float u = philox_u01(philox4x32_10(make_uint4((uint32_t)C.rng_id[c], (uint32_t)tr, RNG_LEAF, (uint32_t)(depth * 65536 + leaf)), key).x);
    if (logf(u) + logW_sub < -dH) {                       // multinomial sampling inside the subtree
      if (act) { vec(C, c, V_SQ)[l] = q; vec(C, c, V_SG)[l] = g; }
      if (l == 0) S.sub_lp[c] = lp;
      flags |= F_HASSUB;
    }
    // checkpoints of the power-of-two aligned sub-subtrees that end at this leaf
    const int i_max = __popc(leaf >> 1);
    const int trailing = __ffs(~leaf) - 1;
    const int i_min = i_max - trailing + 1;
    if ((leaf & 1) == 0) {
      if (act) { vec(C, c, V_PCK + i_max)[l] = p; vec(C, c, V_RCK + i_max)[l] = rho_sub; }
    } else {
      for (int i = i_max; i >= i_min && !bad; --i) {
        const float pc = act ? vec(C, c, V_PCK + i)[l] : 0.f, rc = act ? vec(C, c, V_RCK + i)[l] : 0.f;
        if (uturn(rho_sub - rc + pc, pc, p, v, act, hm)) bad = true;
      }
    }
  }
  bool finish = bad;
  if (!bad) {
    if (leaf + 1 < (1 << depth)) {
      // ---- next leapfrog of this subtree ----
      if (act) {
        const float ph = p + 0.5f * step * g;
        C.p_w[o] = ph; C.theta_w[o] = q + step * v * ph;
        vec(C, c, V_SRHO)[l] = rho_sub;
      }
      if (l == 0) { S.leaf[c] = leaf + 1; S.logW_sub[c] = logW_sub; S.acc_sum[c] = acc_sum; S.n_leaf[c] = n_leaf; S.flags[c] = flags; }
      return;
    }
    // ---- subtree complete: biased progressive sampling across doublings, merge ----
    const float logW = S.logW[c];
    const float u = philox_u01(philox4x32_10(make_uint4((uint32_t)C.rng_id[c], (uint32_t)tr, RNG_SUBTREE, (uint32_t)depth), key).x);
    if ((flags & F_HASSUB) && logf(u) < fminf(0.f, logW_sub - logW)) {
      if (act) { vec(C, c, V_PQ)[l] = vec(C, c, V_SQ)[l]; vec(C, c, V_PG)[l] = vec(C, c, V_SG)[l]; }
      if (l == 0) S.prop_lp[c] = S.sub_lp[c];
    }
    float rho = 0.f, pl = 0.f, pr = 0.f;
    if (act) {
      rho = vec(C, c, V_RHO)[l] + rho_sub;
      vec(C, c, V_RHO)[l] = rho;
      vec(C, c, fwd ? V_RQ : V_LQ)[l] = q; vec(C, c, fwd ? V_RP : V_LP)[l] = p; vec(C, c, fwd ? V_RG : V_LG)[l] = g;
      pl = fwd ? vec(C, c, V_LP)[l] : p; pr = fwd ? p : vec(C, c, V_RP)[l];
    }
    const int new_depth = depth + 1;
    if (l == 0) { S.logW[c] = logaddexpf_(logW, logW_sub); S.depth[c] = new_depth; S.acc_sum[c] = acc_sum; S.n_leaf[c] = n_leaf; }
    finish = uturn(rho, pl, pr, v, act, hm) || new_depth >= max_depth;
    if (!finish) {
      __syncwarp(hm);
      begin_doubling(C, S, c, l, act, o, tr, new_depth, flags, key);
      return;
    }
  }
  // ---- transition complete: the proposal becomes the state; adaptation and summaries; next transition ----
  __syncwarp(hm);
  float th = 0.f;
  if (act) { th = vec(C, c, V_PQ)[l]; C.theta[o] = th; C.grad[o] = vec(C, c, V_PG)[l]; }
  if (l == 0) C.logp[c] = S.prop_lp[c];
  const AdaptFlags A = adapt_flags_dev(it, W);
  if (!A.warmup && l == 0) atomicAdd(&S.depth_hist[min(S.depth[c] + (bad ? 1 : 0), NUTS_MAX_DEPTH)], 1);
  chain_adapt_and_record(C, c, l, act, o, th, acc_sum / (float)n_leaf, n_leaf, (flags & F_DIV) ? 1 : 0, A, samples, it - W.n_warmup, W.n_sample, W.bm_len, W.bm_n);
  __syncwarp(hm);
  const int it1 = it + 1;
  if (it1 >= W.n_warmup + W.n_sample) {
    if (l == 0) { S.it[c] = it1; S.done[c] = 1; atomicAdd(S.n_done, 1); }
    return;
  }
  if (l == 0) S.it[c] = it1;
  begin_transition(C, S, c, l, act, o, it1 + W.first, key, hm);
  __syncwarp(hm);
  begin_doubling(C, S, c, l, act, o, it1 + W.first, 0, 0, key);
}

// live-chain lists per photometry path after some chains have finished
__global__ void nuts_compact_kernel(int64_t n, const int* __restrict__ done, const unsigned char* __restrict__ path_of_chain,
                                    int* __restrict__ list0, int* __restrict__ list1, int* __restrict__ all, int* __restrict__ counts) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n || done[i]) return;
  all[atomicAdd(&counts[2], 1)] = (int)i;
  if (path_of_chain[i] == 0) list0[atomicAdd(&counts[0], 1)] = (int)i;
  else list1[atomicAdd(&counts[1], 1)] = (int)i;
}

}  // namespace


sps_status nuts_run(const sps_table* t, Workspace& ws, const PriorDev& P, const sps_hmc_config* cfg, HmcProblem& Q, ChainState& C, float* samples,
                    int32_t* depth_hist_out, cudaStream_t s) {
  const int64_t n = C.n;
  if (cfg->n_warmup + cfg->n_sample == 0) return SPS_OK;
  NutsScalars S; memset(&S, 0, sizeof(S));
  float* fbase = nullptr; int* ibase = nullptr; int* lists = nullptr;
  sps_status st = sps_check_cuda(sps_pool_alloc((void**)&fbase, 5 * n * sizeof(float)), "NUTS state");
  if (st == SPS_OK) st = sps_check_cuda(sps_pool_alloc((void**)&ibase, (6 * n + 4 + NUTS_MAX_DEPTH + 1 + 4) * sizeof(int)), "NUTS state");
  if (st == SPS_OK) st = sps_check_cuda(sps_pool_alloc((void**)&lists, 3 * n * sizeof(int)), "NUTS live lists");
  if (st != SPS_OK) { if (fbase) sps_pool_free(fbase); if (ibase) sps_pool_free(ibase); if (lists) sps_pool_free(lists); return st; }
  S.logW = fbase; S.logW_sub = fbase + n; S.acc_sum = fbase + 2 * n; S.prop_lp = fbase + 3 * n; S.sub_lp = fbase + 4 * n;
  S.it = ibase; S.depth = ibase + n; S.leaf = ibase + 2 * n; S.n_leaf = ibase + 3 * n; S.flags = ibase + 4 * n; S.done = ibase + 5 * n;
  S.n_done = ibase + 6 * n; S.depth_hist = ibase + 6 * n + 4;
  int* counts = ibase + 6 * n + 4 + NUTS_MAX_DEPTH + 1;
  cudaMemsetAsync(ibase, 0, (6 * n + 4 + NUTS_MAX_DEPTH + 1 + 4) * sizeof(int), s);
  const WarmupSched W = make_warmup_sched(cfg);
  const uint2 key = make_uint2((uint32_t)cfg->seed, (uint32_t)(cfg->seed >> 32));
  const unsigned cb = (unsigned)((n * 16 + 255) / 256);          // two chains per warp
  nuts_begin_kernel<<<cb, 256, 0, s>>>(C, S, (int)cfg->first_transition, key); sps_count_launch();
  // live lists: start from the problem's own per-path lists (NULL = all rows on one path)
  HmcProblem L = Q;
  const int* live = nullptr; int64_t n_live = n;
  const int64_t max_steps = (int64_t)(cfg->n_warmup + cfg->n_sample) * ((1ll << cfg->max_depth) - 1) + 8;
  int done_host = 0;
  for (int64_t step = 0; step < max_steps && st == SPS_OK; ++step) {
    for (int path = 0; path < 2 && st == SPS_OK; ++path) {
      if (L.n_rows_path[path] == 0) continue;
      st = sps_eval(t, ws, P, path, C.theta_w, L.n_rows_path[path], true, true, L.rows_path[path], Q.gal_of_chain, Q.obs_flux, Q.obs_sigma,
                    nullptr, true, C.logp_w, C.grad_w, s);
    }
    if (st != SPS_OK) break;
    nuts_step_kernel<<<(unsigned)((n_live * 16 + 255) / 256), 256, 0, s>>>(C, S, W, cfg->max_depth, key, live, n_live, samples); sps_count_launch();
    if ((step & 15) == 15) {
      st = sps_check_cuda(cudaMemcpyAsync(&done_host, S.n_done, sizeof(int), cudaMemcpyDeviceToHost, s), "NUTS poll");
      if (st == SPS_OK) st = sps_check_cuda(cudaStreamSynchronize(s), "NUTS poll");
      if (done_host >= n) break;
      if (n - done_host < (n_live * 7) / 8) {               // drop finished chains from the evaluation lists
        cudaMemsetAsync(counts, 0, 4 * sizeof(int), s);
        nuts_compact_kernel<<<(unsigned)((n + 255) / 256), 256, 0, s>>>(n, S.done, Q.path_of_chain, lists, lists + n, lists + 2 * n, counts);
        sps_count_launch();
        int ch[4];
        st = sps_check_cuda(cudaMemcpyAsync(ch, counts, 4 * sizeof(int), cudaMemcpyDeviceToHost, s), "NUTS compaction");
        if (st == SPS_OK) st = sps_check_cuda(cudaStreamSynchronize(s), "NUTS compaction");
        L.rows_path[0] = lists; L.n_rows_path[0] = ch[0];
        L.rows_path[1] = lists + n; L.n_rows_path[1] = ch[1];
        live = lists + 2 * n; n_live = ch[2];
      }
    }
  }
  if (st == SPS_OK && depth_hist_out)                       // kept transitions per final tree depth
    cudaMemcpyAsync(depth_hist_out, S.depth_hist, (NUTS_MAX_DEPTH + 1) * sizeof(int), cudaMemcpyDeviceToDevice, s);
  cudaStreamSynchronize(s);
  sps_pool_free(fbase); sps_pool_free(ibase); sps_pool_free(lists);
  return st;
}
