// sps_approx_tc.cu -- tensor-core formulation of the approximate-photometry contraction (a7 + a9 + a10).
//
// After the rows of a call are grouped by z cell, Eq. (6) and its reverse are two small GEMMs per cell:
//   pass 1   P[r, e]     = sum_i a[r, i] C[i, e]          e = s*128 + (j n_band + b),  s = 0: c_t, s = 1: D_t = c_{t+1} - c_t
//   pass 2   a_bar[r, i] = sum_e V[r, e] C[i, e]          V[r, e] = g_b F_b M m_j {1, f_r}
// One persistent CTA per SM works on 128-row tiles of one cell:
//   warps 0-3  thread = row: split the row's weights a (fp32) into FP16 hi + lo and write them into shared memory in the
//              128-byte-swizzled K-major operand layout; after pass 1 read P from TMEM (tcgen05.ld), do the band step (dust at
//              lambda_eff/(1+z), fluxes, likelihood, the direct bars, m_bar), generate V (split, swizzled) for pass 2, and at the
//              end store a_bar from TMEM
//   warp 4     one thread: TMA loads of the cell's table operands (FP16 hi + lo, both majornesses, built at table creation)
//              and the tcgen05.mma issue (three split products a_lo c_hi + a_hi c_lo + a_hi c_hi, fp32 accumulation in TMEM)
// P and a_bar never leave TMEM / registers; the table operands are L2 resident (51 MB for 199 cells).
// FP16 rather than BF16 split: two FP16 terms carry 22 significant bits (BF16: 16), which the reverse pass needs -- the epilogue
// contracts a_bar with partials that cancel to ~1e-3 of their size.  Operands are scaled by powers of two into the FP16 range:
// a_i <= 1 by 2^14, the table arrays by one scale each (largest |c_t|, |D_t| -> [2^13, 2^14)), V by a per-row scale.
#include <cuda.h>
#include <cuda_fp16.h>
#include <algorithm>
#include <cmath>
#include <cstring>
#include "sps_internal.h"
#include "sps_ptx.cuh"

struct ApproxTc {
  __half *C1_hi, *C1_lo;      // [n_cells * 256][128]  pass-1 B operand: row = (cell, entry), K = age contiguous
  __half *C2_hi, *C2_lo;      // [n_cells * 128][256]  pass-2 B operand: row = (cell, age),   K = entry contiguous
  CUtensorMap m1_hi, m1_lo, m2_hi, m2_lo;
  float* Cm;                         // [n_cells][128] power of two >= max_e |c_t[i][e]| of each (cell, age): a_i Cm_i and c_t / Cm_i are what is split
  float sD;                          // power of two: D_t sD / Cm_i <= 1 everywhere
};

namespace {

constexpr int TM = 128;                         // rows per tile
constexpr int KB = 64;                          // fp16 elements per 128-byte operand row (one k block)
constexpr int NE = 256;                         // table entries per cell as GEMM dimension: [0,128) c_t, [128,256) D_t
constexpr int NA = 128;                         // ages as GEMM dimension
constexpr int TILE_A = TM * 128;                // 16 KB: 128 rows x 128 B
constexpr int REG_AV = 4 * TILE_A;              // 64 KB: A (hi, lo) x 2 k blocks; later V (hi, lo) x 2 k blocks of a phase
constexpr int REG_B = 128 * 1024;               // pass 1: 2 k blocks x (hi 32 KB + lo 32 KB); pass 2: 4 k blocks x (hi 16 KB + lo 16 KB)
constexpr int OFF_EXTRA = REG_AV + REG_B + 256;     // cm_s[128], rs_s[128], red_s[6][128], mb_s[16][128] floats
constexpr int BINS_S = 2048;                     // ints of shared memory for the cell offsets (row_start, cta_start)
constexpr int SMEM_TC = OFF_EXTRA + (2 + 6 + 16) * 128 * 4 + BINS_S * 4 + 1024;
constexpr int THREADS_TC = 288;                 // 8 row warps + the TMA / MMA warp
constexpr float H_TOP = 16384.f;                // operands are scaled so that their largest magnitude sits just below 2^14 before the FP16 split

// band counts the kernel is instantiated for (other tables use the SIMT kernel of sps_kernels.cu)
#define SPS_APPROX_TC_BANDS(X) X(3) X(10) X(12)


// K-major operand tile, 128-byte rows, SWIZZLE_128B: 8-row atoms of 1024 B stacked along M/N
__device__ __forceinline__ uint64_t desc_sw128(uint32_t saddr) { return umma_desc_kmajor(saddr, 128); }
// byte offset of the 16-byte chunk `c` (0..7) of row r in a 128-byte-swizzled tile (what TMA writes and tcgen05 reads)
__device__ __forceinline__ uint32_t sw128_off(int r, int c) { return (uint32_t)((r >> 3) * 1024 + (r & 7) * 128 + ((c ^ (r & 7)) << 4)); }
#define TLD16(taddr, v) TMEM_LD16(taddr, v)
__device__ __forceinline__ void tld_wait() { tmem_ld_wait(); }

__device__ __forceinline__ void split8(const float* v, uint4& hi, uint4& lo) {
  __half h[8], l[8];
#pragma unroll
  for (int k = 0; k < 8; ++k) { h[k] = __float2half_rn(v[k]); l[k] = __float2half_rn(v[k] - __half2float(h[k])); }
  hi = *reinterpret_cast<const uint4*>(h); lo = *reinterpret_cast<const uint4*>(l);
}

// table operands (one-time, at table creation): entry e = s*128 + (j n_band + b)
// one warp per (cell, age): Cm = 2^ceil(log2 max_e |c_t[i][e]|); the largest |D_t| / Cm over the table goes to *dmax
__global__ void cssp_rowmax_kernel(TableDev T, float* __restrict__ Cm, int* __restrict__ dmax) {
  const int64_t wid = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
  const int lane = threadIdx.x & 31;
  if (wid >= (int64_t)(T.n_z - 1) * NA) return;
  const int i = (int)(wid % NA), cell = (int)(wid / NA);
  float cm = 1.f;
  if (i < T.n_age) {
    const float* c0 = T.cssp + (((int64_t)cell * 2) * T.n_age + i) * T.cs_stride;
    const float* c1 = c0 + (int64_t)T.n_age * T.cs_stride;
    const int E = T.n_Z * T.n_band;
    float mx = 0.f, dx = 0.f;
    for (int e = lane; e < E; e += 32) { mx = fmaxf(mx, fabsf(c0[e])); dx = fmaxf(dx, fabsf(c1[e])); }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) { mx = fmaxf(mx, __shfl_xor_sync(FULL_MASK, mx, o)); dx = fmaxf(dx, __shfl_xor_sync(FULL_MASK, dx, o)); }
    if (mx > 1.0e-30f && mx < 1.0e30f) cm = __uint_as_float(((__float_as_uint(mx) >> 23) + 1u) << 23);       // 2^(ex+1) > mx
    if (lane == 0 && dx > 0.f) atomicMax(dmax, __float_as_int(dx / cm));
  }
  if (lane == 0) Cm[wid] = cm;
}
__global__ void build_c_operands_kernel(TableDev T, const float* __restrict__ Cm, float sD, __half* __restrict__ c1h, __half* __restrict__ c1l,
                                        __half* __restrict__ c2h, __half* __restrict__ c2l) {
  const int64_t idx = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  const int n_cells = T.n_z - 1;
  if (idx >= (int64_t)n_cells * NE * NA) return;
  const int i = (int)(idx % NA), e = (int)((idx / NA) % NE), cell = (int)(idx / ((int64_t)NA * NE));
  const int s = e >> 7, ee = e & 127;
  float v = 0.f;
  if (i < T.n_age && ee < T.n_Z * T.n_band) v = T.cssp[(((int64_t)cell * 2 + s) * T.n_age + i) * T.cs_stride + ee] * (H_TOP / Cm[cell * NA + i]) * (s ? sD : 1.f);
  const __half h = __float2half_rn(v), l = __float2half_rn(v - __half2float(h));
  c1h[((int64_t)cell * NE + e) * NA + i] = h; c1l[((int64_t)cell * NE + e) * NA + i] = l;
  c2h[((int64_t)cell * NA + i) * NE + e] = h; c2l[((int64_t)cell * NA + i) * NE + e] = l;
}

// shared memory: [0, 64 KB) A / V operand tiles, [64 KB, 192 KB) table operand tiles, then the barriers
constexpr uint32_t OFF_B = REG_AV, OFF_BAR = REG_AV + REG_B;
enum { BAR_B1 = 0, BAR_A, BAR_P, BAR_B2, BAR_V0, BAR_M1, N_BARS };


struct ApproxArgs {
  int64_t n;
  const int* order; int* bins;   // (direct mode: the last CTA to read the counts clears them for the next prologue)
  int64_t cap;             // > 0: `order` is the prologue's per-cell row lists [cell][cap] and bins[0..nb) their lengths (no scan / scatter pass)
  const int* gal_of_row; const float* obs_flux; const float* obs_sigma; const float* flux_bar;
  int want_grad;
  const float* Cm;         // [n_cells][128]
  float inv_sD;
};

// NB = n_band (compile time: entry e -> (j, b) = (e / NB, e % NB) resolves to register names in the unrolled band step)
template <int NB>
#ifndef ATC_MINB
#define ATC_MINB 1
#endif
__global__ void __launch_bounds__(THREADS_TC, ATC_MINB)
approx_tc_kernel(TableDev T, ApproxArgs G, RowBuffers B, const __grid_constant__ CUtensorMap m1h, const __grid_constant__ CUtensorMap m1l,
                 const __grid_constant__ CUtensorMap m2h, const __grid_constant__ CUtensorMap m2l) {
  extern __shared__ unsigned char smem_dyn[];
  __shared__ int s_last;
  const int nb = T.n_z - 1, stride = nb + 2;
  const bool direct = G.cap > 0;
  const int* row_start_g = G.bins + stride; const int* cta_start_g = G.bins + 2 * stride;
  const uint32_t base = (smem_u32(smem_dyn) + 1023u) & ~1023u;
  unsigned char* gbase = smem_dyn + (base - smem_u32(smem_dyn));
  const uint32_t bars = base + OFF_BAR;
  volatile uint32_t* tmem_ptr = reinterpret_cast<volatile uint32_t*>(gbase + OFF_BAR + 128);
  float* cm_s = reinterpret_cast<float*>(gbase + OFF_EXTRA);         // [128] Cm_i / 2^14 of the current tile's cell
  float* rs_s = cm_s + 128;                                          // [128] power-of-two scale of each tile row's a_i Cm_i
  float* red_s = rs_s + 128;                                         // [6][128] band-loop partial sums of the h = 1 threads
  float* mb_s = red_s + 6 * 128;                                     // [16][128] partial m_bar of the h = 1 threads
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
#define BAR(i) (bars + 8u * (i))
  // cell offsets of the call in shared memory when they fit (they are walked once per tile by every thread)
  int* bins_s = reinterpret_cast<int*>(gbase + OFF_EXTRA + (2 + 6 + 16) * 128 * 4);
  pdl_wait();                                               // the prologue's counts, lists and row buffers
  if (!direct) {
    for (int i = threadIdx.x; i <= nb; i += blockDim.x) { bins_s[i] = row_start_g[i]; bins_s[nb + 1 + i] = cta_start_g[i]; }
  } else {
    // the prologue left a row list and a count per z cell: every CTA turns the counts into tile offsets itself
    for (int i = threadIdx.x; i <= nb; i += blockDim.x) { const int c = i < nb ? G.bins[i] : 0; bins_s[i] = c; bins_s[nb + 1 + i] = (c + TM - 1) / TM; }
    __syncthreads();
    // arrival count (bins[3 stride]): the last CTA to have read the counts clears them, so the next prologue of this
    // workspace can append to its cells without a memset in between
    if (threadIdx.x == 0) { __threadfence(); s_last = atomicAdd(G.bins + 3 * stride, 1) == (int)gridDim.x - 1; }
    if (warp == 0) {
      int carry = 0;
      for (int b0 = 0; b0 <= nb; b0 += 32) {
        const int idx = b0 + lane, v = idx <= nb ? bins_s[nb + 1 + idx] : 0;
        int inc = v;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) { const int u = __shfl_up_sync(FULL_MASK, inc, o); if (lane >= o) inc += u; }
        if (idx <= nb) bins_s[nb + 1 + idx] = carry + inc - v;
        carry += __shfl_sync(FULL_MASK, inc, 31);
      }
    }
  }
  __syncthreads();
  if (direct && s_last) {
    for (int i = threadIdx.x; i < nb; i += blockDim.x) G.bins[i] = 0;
    if (threadIdx.x == 0) G.bins[3 * stride] = 0;
  }
  const int* row_start = bins_s;                            // legacy: first position of each cell in `order`; direct: the cell's row count
  const int* cta_start = bins_s + nb + 1;
  auto cell_begin = [&](int c) { return direct ? (int64_t)c * G.cap : (int64_t)row_start[c]; };
  auto cell_end = [&](int c) { return direct ? (int64_t)c * G.cap + row_start[c] : (int64_t)row_start[c + 1]; };
  const int total = cta_start[nb];
  const int per = total / (int)gridDim.x, rem = total % (int)gridDim.x;
  const int w_begin = (int)blockIdx.x * per + min((int)blockIdx.x, rem);
  const int w_end = w_begin + per + ((int)blockIdx.x < rem ? 1 : 0);
  if (w_begin >= w_end) return;
  if (threadIdx.x == 0) {
    mbar_init(BAR(BAR_B1), 1); mbar_init(BAR(BAR_A), 2 * TM); mbar_init(BAR(BAR_P), 1); mbar_init(BAR(BAR_B2), 1);
    mbar_init(BAR(BAR_V0), 2 * TM); mbar_init(BAR(BAR_M1), 1);
    mbar_fence_init();
  }
  if (warp == 8) {
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(bars + 128u), "n"(512) : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
  }
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem_base = *tmem_ptr;
  int lo = 0, hi = nb;
  while (hi - lo > 1) { const int mid = (lo + hi) >> 1; if (cta_start[mid] <= w_begin) lo = mid; else hi = mid; }
  int cell = lo;

  if (warp == 8) {
    // ===== TMA loads + MMA issue =================================================================
    if (lane == 0) {
      // instruction descriptor: D = F32, A and B = F16 (format 0), both K-major
      const uint32_t idesc1 = (1u << 4) | ((uint32_t)(NE >> 3) << 17) | ((uint32_t)(TM >> 4) << 24);
      const uint32_t idesc2 = (1u << 4) | ((uint32_t)(NA >> 3) << 17) | ((uint32_t)(TM >> 4) << 24);
      uint32_t ph = 0;
      for (int w = w_begin; w < w_end; ++w, ph ^= 1u) {
        while (cta_start[cell + 1] <= w) ++cell;
        // pass-1 operands: C1 tiles [256 entries][64 ages], hi k-block 0, 1 then lo k-block 0, 1
        mbar_expect_tx(BAR(BAR_B1), (uint32_t)REG_B);
        tma_load_2d(base + OFF_B, &m1h, BAR(BAR_B1), 0, cell * NE);
        tma_load_2d(base + OFF_B + 32768u, &m1h, BAR(BAR_B1), KB, cell * NE);
        tma_load_2d(base + OFF_B + 65536u, &m1l, BAR(BAR_B1), 0, cell * NE);
        tma_load_2d(base + OFF_B + 98304u, &m1l, BAR(BAR_B1), KB, cell * NE);
        mbar_wait(BAR(BAR_B1), ph);
        mbar_wait(BAR(BAR_A), ph);
        tc_fence_after();
        // Split products in ONE accumulator, the cross terms a_lo c_hi + a_hi c_lo (2^-11 of the main one) first: tensor-core
        // accumulation truncates every update to fp32, an error relative to the accumulator's size at that
        // moment, so the 16 cross updates cost nothing and the sum sees the 8 full-size updates of the main products only.
#pragma unroll
        for (int kb = 0; kb < 2; ++kb)
#pragma unroll
          for (int kk = 0; kk < 4; ++kk) {
            const uint64_t a_hi = desc_sw128(base + kb * TILE_A + kk * 32), a_lo = desc_sw128(base + (2 + kb) * TILE_A + kk * 32);
            const uint64_t b_hi = desc_sw128(base + OFF_B + kb * 32768u + kk * 32), b_lo = desc_sw128(base + OFF_B + 65536u + kb * 32768u + kk * 32);
            tc_mma_f16(tmem_base, a_lo, b_hi, idesc1, (kb | kk) ? 1u : 0u);
            tc_mma_f16(tmem_base, a_hi, b_lo, idesc1, 1u);
          }
#pragma unroll
        for (int kb = 0; kb < 2; ++kb)
#pragma unroll
          for (int kk = 0; kk < 4; ++kk)
            tc_mma_f16(tmem_base, desc_sw128(base + kb * TILE_A + kk * 32), desc_sw128(base + OFF_B + kb * 32768u + kk * 32), idesc1, 1u);
        tc_commit(BAR(BAR_P));
        mbar_wait(BAR(BAR_P), ph);                          // pass 1 retired: the table region may be overwritten
        if (!G.want_grad) continue;
        // pass-2 operands: C2 tiles [128 ages][64 entries], hi entry block 0..3 then lo entry block 0..3
        mbar_expect_tx(BAR(BAR_B2), (uint32_t)REG_B);
#pragma unroll
        for (int eb = 0; eb < 4; ++eb) {
          tma_load_2d(base + OFF_B + eb * 16384u, &m2h, BAR(BAR_B2), eb * KB, cell * NA);
          tma_load_2d(base + OFF_B + 65536u + eb * 16384u, &m2l, BAR(BAR_B2), eb * KB, cell * NA);
        }
        mbar_wait(BAR(BAR_B2), ph);
        mbar_wait(BAR(BAR_V0), ph);
        tc_fence_after();
        // Both table arrays are contracted with the same operand V (the row's factor f on the D_t part is applied when the
        // accumulators are read): acc^(s) = sum_e V[e] C^(s)[i][e], cross terms first (see pass 1).  The accumulators reuse the
        // columns of P (dead once V is being written): s = 0 at columns 0, s = 1 at NA.
#pragma unroll
        for (int s = 0; s < 2; ++s) {
#pragma unroll
          for (int kb = 0; kb < 2; ++kb)
#pragma unroll
            for (int kk = 0; kk < 4; ++kk) {
              const int eb = 2 * s + kb;
              const uint64_t a_hi = desc_sw128(base + kb * TILE_A + kk * 32), a_lo = desc_sw128(base + (2 + kb) * TILE_A + kk * 32);
              const uint64_t b_hi = desc_sw128(base + OFF_B + eb * 16384u + kk * 32), b_lo = desc_sw128(base + OFF_B + 65536u + eb * 16384u + kk * 32);
              tc_mma_f16(tmem_base + s * NA, a_lo, b_hi, idesc2, (kb | kk) ? 1u : 0u);
              tc_mma_f16(tmem_base + s * NA, a_hi, b_lo, idesc2, 1u);
            }
#pragma unroll
          for (int kb = 0; kb < 2; ++kb)
#pragma unroll
            for (int kk = 0; kk < 4; ++kk)
              tc_mma_f16(tmem_base + s * NA, desc_sw128(base + kb * TILE_A + kk * 32), desc_sw128(base + OFF_B + (2 * s + kb) * 16384u + kk * 32), idesc2, 1u);
        }
        tc_commit(BAR(BAR_M1));
        mbar_wait(BAR(BAR_M1), ph);                         // pass 2 retired: both regions are free for the next tile
      }
    }
  } else {
    // ===== row warps: two threads per tile row.  Warps w and w + 4 share TMEM lane quarter w & 3; h = w >> 2 picks the
    //       thread's share of every phase (P chunks, bands, V k-block, a_bar columns) ===================================
    const int h = warp >> 2;
    const int r = (warp & 3) * 32 + lane;                   // tile row = TMEM lane
    const uint32_t tlane = tmem_base + ((uint32_t)((warp & 3) * 32) << 16);
    uint32_t ph = 0;
    // The row index and galaxy of a tile row are fetched one tile ahead (dependent loads order -> gal_of_row off the critical path).
    int rw_next, gal_next = 0;
    {
      while (cta_start[cell + 1] <= w_begin) ++cell;
      const int64_t rb = cell_begin(cell) + (int64_t)(w_begin - cta_start[cell]) * TM;
      rw_next = (rb + r < min(cell_end(cell), rb + TM)) ? __ldg(G.order + rb + r) : -1;
      if (rw_next >= 0 && !G.flux_bar) gal_next = G.gal_of_row ? __ldg(G.gal_of_row + rw_next) : rw_next;
    }
    RowScalars sc_n;
    float m_n[16], ob0_n[(NB + 1) / 2], ob1_n[(NB + 1) / 2];
    auto load_row = [&](int rw, int64_t gal) {
      float4* scq = reinterpret_cast<float4*>(&sc_n);
      float4* mq = reinterpret_cast<float4*>(m_n);
#pragma unroll
      for (int q = 0; q < 4; ++q) {
        scq[q] = rw >= 0 ? reinterpret_cast<const float4*>(B.sc + rw)[q] : make_float4(0.f, 0.f, 0.f, 0.f);
        mq[q] = rw >= 0 ? __ldg(reinterpret_cast<const float4*>(B.m + (int64_t)rw * ROW_M_STRIDE) + q) : make_float4(0.f, 0.f, 0.f, 0.f);
      }
#pragma unroll
      for (int j = 0; j < 16; ++j) if (j >= T.n_Z) m_n[j] = 0.f;
#pragma unroll
      for (int k = 0; k < (NB + 1) / 2; ++k) {
        const int b = min(h + 2 * k, NB - 1);
        ob0_n[k] = 0.f; ob1_n[k] = 1.f;
        if (rw >= 0) {
          if (G.flux_bar) ob0_n[k] = __ldg(G.flux_bar + (int64_t)rw * NB + b);
          else { ob0_n[k] = __ldg(G.obs_flux + gal * NB + b); ob1_n[k] = __ldg(G.obs_sigma + gal * NB + b); }
        }
      }
    };
    load_row(rw_next, gal_next);
    for (int w = w_begin; w < w_end; ++w, ph ^= 1u) {
      while (cta_start[cell + 1] <= w) ++cell;
      const int64_t r_begin = cell_begin(cell) + (int64_t)(w - cta_start[cell]) * TM;
      const int64_t r_end = min(cell_end(cell), r_begin + TM);
      const int rw = rw_next;
      const int64_t gal = gal_next;
      const int n_rows = (int)(r_end - r_begin);
      // the next tile's rows
      rw_next = -1;
      if (w + 1 < w_end) {
        int cn = cell;
        while (cta_start[cn + 1] <= w + 1) ++cn;
        const int64_t rbn = cell_begin(cn) + (int64_t)(w + 1 - cta_start[cn]) * TM;
        if (rbn + r < min(cell_end(cn), rbn + TM)) rw_next = __ldg(G.order + rbn + r);
      }
      gal_next = 0;
      // ---- the row's scalars, metallicity weights and this thread's bands of the observations: requested during the
      //      previous tile (before its wait for pass 2) ----
      const RowScalars sc = sc_n;
      float m[16], ob0[(NB + 1) / 2], ob1[(NB + 1) / 2];
#pragma unroll
      for (int j = 0; j < 16; ++j) m[j] = m_n[j];
#pragma unroll
      for (int k = 0; k < (NB + 1) / 2; ++k) { ob0[k] = ob0_n[k]; ob1[k] = ob1_n[k]; }
      // ---- stage a (split, swizzled): warp-cooperative, lane = 4 consecutive ages of one row; warp (q, h) stages rows
      //      32 q + 16 h .. + 15 ----
      {
        const int kb = lane >> 4, c = (lane & 15) >> 1, half = lane & 1;
        const float4 cm4 = __ldg(reinterpret_cast<const float4*>(G.Cm + (int64_t)cell * NA) + lane);
        asm volatile("bar.sync 1, %0;" ::"n"(2 * TM) : "memory");        // every row thread is done with the previous tile's shared arrays
        if (h == 0) cm_s[r] = __ldg(G.Cm + (int64_t)cell * NA + r) * (1.f / H_TOP);
        float4 av[16];
#pragma unroll
        for (int u = 0; u < 16; ++u) {
          const int row_u = __shfl_sync(FULL_MASK, rw, 16 * h + u);                // rows past the tile's end: any valid row, zeroed below
          av[u] = __ldg(reinterpret_cast<const float4*>(B.a + (int64_t)max(row_u, 0) * ROW_A_STRIDE) + lane);
        }
#pragma unroll
        for (int u = 0; u < 16; ++u) {
          const int tr = (warp & 3) * 32 + 16 * h + u;       // tile row being staged
          float v[4] = {av[u].x * cm4.x, av[u].y * cm4.y, av[u].z * cm4.z, av[u].w * cm4.w};
          float mx = 0.f;
#pragma unroll
          for (int k = 0; k < 4; ++k) { if (4 * lane + k >= T.n_age || tr >= n_rows) v[k] = 0.f; mx = fmaxf(mx, fabsf(v[k])); }
          mx = __uint_as_float(__reduce_max_sync(FULL_MASK, __float_as_uint(mx)));
          float rs = 1.f;                                   // rs mx in [2^13, 2^14)
          if (mx > 1.0e-30f && mx < 1.0e30f) rs = __uint_as_float((uint32_t)(127 + 13 + 127 - (int)((__float_as_uint(mx) >> 23) & 0xffu)) << 23);
          if (lane == u) rs_s[tr] = rs;
          __half hh[4], ll[4];
#pragma unroll
          for (int k = 0; k < 4; ++k) {
            v[k] *= rs;
            hh[k] = __float2half_rn(v[k]); ll[k] = __float2half_rn(v[k] - __half2float(hh[k]));
          }
          const uint32_t off = kb * TILE_A + sw128_off(tr, c) + half * 8;
          *reinterpret_cast<uint2*>(gbase + off) = *reinterpret_cast<const uint2*>(hh);
          *reinterpret_cast<uint2*>(gbase + 2 * TILE_A + off) = *reinterpret_cast<const uint2*>(ll);
        }
      }
      if (rw_next >= 0) {                                   // the next tile's weights start their way into L2
        if (h == 0) {
          const char* np_ = reinterpret_cast<const char*>(B.a + (int64_t)rw_next * ROW_A_STRIDE);
#pragma unroll
          for (int q = 0; q < 4; ++q) asm volatile("prefetch.global.L2 [%0];" ::"l"(np_ + 128 * q));
        }
        if (!G.flux_bar) gal_next = G.gal_of_row ? __ldg(G.gal_of_row + rw_next) : rw_next;
      }
      tc_fence_before();                                    // the previous tile's TMEM reads are complete
      fence_proxy_async_smem();
      mbar_arrive(BAR(BAR_A));
      asm volatile("bar.sync 1, %0;" ::"n"(2 * TM) : "memory");            // cm_s and rs_s of this tile are complete
      const float u0 = 1.f / (H_TOP * rs_s[r]), u1 = u0 * G.inv_sD;       // P^(s) back to table units
      const float f = sc.zfrac, Mn = sc.Mn, zp = 1.f + sc.z;
      const int E = T.n_Z * NB;
      // ---- sweep 1 over P (this thread's chunks): S^(s)_b = sum_j m_j P^(s)[j NB + b] ----
      float S0[NB], S1[NB];
#pragma unroll
      for (int b = 0; b < NB; ++b) S0[b] = S1[b] = 0.f;
      mbar_wait(BAR(BAR_P), ph);
      tc_fence_after();
#pragma unroll
      for (int c = 0; c < 8; ++c) {
        if ((c & 1) == h && 16 * c < E) {
          uint32_t v0[16], v1[16];
          TLD16(tlane + 16 * c, v0); TLD16(tlane + 128 + 16 * c, v1);
          tld_wait();
#pragma unroll
          for (int k = 0; k < 16; ++k) {
            const int e = 16 * c + k, j = e / NB, b = e % NB;
            if (j < 16) {
              S0[b] = fmaf(m[j], __uint_as_float(v0[k]), S0[b]);
              S1[b] = fmaf(m[j], __uint_as_float(v1[k]), S1[b]);
            }
          }
        }
      }
      // ---- band step (Eq. 6, dust at lambda_eff / (1+z) R14; Gaussian likelihood).  A rolled loop over this
      //      thread's bands keeps the kernel inside the instruction cache; per-band inputs and sbar_b sit in a scratch column
      //      of the A / V region (pass 1 has retired, V is written later).
      //      scr[slot * TM]: slots 0-15 / 16-31 partial S^(0) of h = 0 / 1, 32-47 / 48-63 partial S^(1), 64-79 / 80-95
      //      observations, 96-111 sbar ----
      float* scr = reinterpret_cast<float*>(gbase) + r;
#pragma unroll
      for (int b = 0; b < NB; ++b) { scr[(16 * h + b) * TM] = S0[b] * u0; scr[(32 + 16 * h + b) * TM] = S1[b] * u1; }
#pragma unroll
      for (int k = 0; k < (NB + 1) / 2; ++k)
        if (h + 2 * k < NB) { scr[(64 + h + 2 * k) * TM] = ob0[k]; scr[(80 + h + 2 * k) * TM] = ob1[k]; }
      asm volatile("bar.sync 1, %0;" ::"n"(2 * TM) : "memory");
      float chi2 = 0.f, v_mn = 0.f, v_z = 0.f, v_av = 0.f, v_de = 0.f, v_fl = 0.f;
      const float izp = __fdividef(1.f, zp);
      float* fo = B.flux + (int64_t)max(rw, 0) * SPS_MAX_BAND;
#pragma unroll 1
      for (int b = h; b < NB; b += 2) {
        float F, F_av, F_del, F_fl, F_lam;
        const float lam_r = T.lam_eff[b] * izp;
        dust_at(lam_r, sc.AV, sc.delta, sc.Ffloor, F, F_av, F_del, F_fl, F_lam, T.model == SPS_MODEL_TINY5);
        const float s1 = scr[(32 + b) * TM] + scr[(48 + b) * TM];
        const float Sint = (scr[b * TM] + scr[(16 + b) * TM]) + f * s1;
        const float flux = F * Mn * Sint;
        if (rw >= 0) fo[b] = flux;
        float g = scr[(64 + b) * TM];
        if (!G.flux_bar) {
          const float isg = __fdividef(1.f, scr[(80 + b) * TM]);
          const float rr = (flux - g) * isg;
          chi2 = fmaf(rr, rr, chi2);
          g = -rr * isg;
        }
        v_mn += g * F * Sint;
        v_z += g * (F * Mn * s1 * T.inv_dz + Mn * Sint * F_lam * (-lam_r * izp));
        v_av += g * Mn * Sint * F_av; v_de += g * Mn * Sint * F_del; v_fl += g * Mn * Sint * F_fl;
        scr[(96 + b) * TM] = g * F * Mn;
      }
      if (h == 1) { red_s[r] = chi2; red_s[TM + r] = v_mn; red_s[2 * TM + r] = v_z; red_s[3 * TM + r] = v_av; red_s[4 * TM + r] = v_de; red_s[5 * TM + r] = v_fl; }
      asm volatile("bar.sync 1, %0;" ::"n"(2 * TM) : "memory");
      if (h == 0 && rw >= 0) {
        RowScalars* out = B.sc + rw;
        out->logp_like = -0.5f * (chi2 + red_s[r]);
        if (G.want_grad) {
          out->Mn_bar = v_mn + red_s[TM + r]; out->z_bar = v_z + red_s[2 * TM + r]; out->AV_bar = v_av + red_s[3 * TM + r];
          out->delta_bar = v_de + red_s[4 * TM + r]; out->Ffloor_bar = v_fl + red_s[5 * TM + r];
        }
      }
      if (!G.want_grad) { if (w + 1 < w_end) load_row(rw_next, gal_next); continue; }
      // ---- sweep 2 over P (this thread's chunks): m_bar_j = sum_b sbar_b (P^(0) + f P^(1))[j NB + b] ----
      float sbar[NB];
#pragma unroll
      for (int b = 0; b < NB; ++b) sbar[b] = scr[(96 + b) * TM];
      float mb[16];
      {
        const float fu1 = f * u1;
#pragma unroll
        for (int j = 0; j < 16; ++j) mb[j] = 0.f;
#pragma unroll
        for (int c = 0; c < 8; ++c) {
          if ((c & 1) == h && 16 * c < E) {
            uint32_t v0[16], v1[16];
            TLD16(tlane + 16 * c, v0); TLD16(tlane + 128 + 16 * c, v1);
            tld_wait();
#pragma unroll
            for (int k = 0; k < 16; ++k) {
              const int e = 16 * c + k, j = e / NB, b = e % NB;
              if (j < 16) mb[j] = fmaf(sbar[b], fmaf(fu1, __uint_as_float(v1[k]), u0 * __uint_as_float(v0[k])), mb[j]);
            }
          }
        }
        if (h == 1) {
#pragma unroll
          for (int j = 0; j < 16; ++j) mb_s[j * TM + r] = mb[j];
        }
      }
      tc_fence_before();
      asm volatile("bar.sync 1, %0;" ::"n"(2 * TM) : "memory");            // partial m_bar parked; every thread has read its scratch: V may overwrite it
      if (h == 0 && rw >= 0) {
        float4* mo = reinterpret_cast<float4*>(B.m_bar + (int64_t)rw * ROW_M_STRIDE);
#pragma unroll
        for (int q = 0; q < 4; ++q)
          mo[q] = make_float4(mb[4 * q] + mb_s[(4 * q) * TM + r], mb[4 * q + 1] + mb_s[(4 * q + 1) * TM + r], mb[4 * q + 2] + mb_s[(4 * q + 2) * TM + r], mb[4 * q + 3] + mb_s[(4 * q + 3) * TM + r]);
      }
      // ---- V[e] = sbar_b m_j: the A operand of pass 2 (both table arrays), this thread's k block (64 entries); the row is
      //      scaled by a power of two sv that puts its largest entry near 2^14 ----
      float sv = 1.f;
      {
        float smax = 0.f, mmax = 0.f;
#pragma unroll
        for (int b = 0; b < NB; ++b) smax = fmaxf(smax, fabsf(sbar[b]));
#pragma unroll
        for (int j = 0; j < 16; ++j) mmax = fmaxf(mmax, fabsf(m[j]));
        const float vmax = smax * mmax;
        if (vmax > 1.0e-30f && vmax < 1.0e30f) {
          const int ex = (int)((__float_as_uint(vmax) >> 23) & 0xffu) - 127;      // vmax in [2^ex, 2^(ex+1))
          sv = __uint_as_float((uint32_t)(127 + 13 - ex) << 23);                 // sv vmax in [2^13, 2^14)
        }
      }
      {
        const float scale = (rw >= 0) ? sv : 0.f;
        if (h == 0) {
#pragma unroll
          for (int c = 0; c < 8; ++c) {
            float v[8];
#pragma unroll
            for (int k = 0; k < 8; ++k) {
              const int e = 8 * c + k, j = e / NB, b = e % NB;
              v[k] = (j < 16) ? scale * sbar[b] * m[j] : 0.f;
            }
            uint4 vh, vl;
            split8(v, vh, vl);
            const uint32_t off = sw128_off(r, c);
            *reinterpret_cast<uint4*>(gbase + off) = vh;
            *reinterpret_cast<uint4*>(gbase + 2 * TILE_A + off) = vl;
          }
        } else {
#pragma unroll
          for (int c = 0; c < 8; ++c) {
            float v[8];
#pragma unroll
            for (int k = 0; k < 8; ++k) {
              const int e = 64 + 8 * c + k, j = e / NB, b = e % NB;
              v[k] = (j < 16) ? scale * sbar[b] * m[j] : 0.f;
            }
            uint4 vh, vl;
            split8(v, vh, vl);
            const uint32_t off = TILE_A + sw128_off(r, c);
            *reinterpret_cast<uint4*>(gbase + off) = vh;
            *reinterpret_cast<uint4*>(gbase + 2 * TILE_A + off) = vl;
          }
        }
        fence_proxy_async_smem();
        mbar_arrive(BAR(BAR_V0));
      }
      // ---- a_bar from TMEM (main + cross-term accumulators), this thread's 64 columns ----
      if (w + 1 < w_end) load_row(rw_next, gal_next);       // the next tile's row inputs travel while pass 2 runs
      mbar_wait(BAR(BAR_M1), ph);
      tc_fence_after();
      // thread = (row, half of the ages) reads its TMEM lane and parks the scaled values in the (free) A / V region, 16-byte
      // chunks XOR-swizzled by the row; then each warp writes 16 rows to global memory 512 contiguous bytes at a time
      const float ua = 1.f / sv, fa = f * G.inv_sD;      // a_bar_i = (acc^(0)_i + f / sD acc^(1)_i) Cm_i / (2^14 sv)
      float4* stage = reinterpret_cast<float4*>(gbase);                   // [TM][32] float4
#pragma unroll 1
      for (int c = 4 * h; c < 4 * h + 4; ++c) {
        uint32_t v[16], v1[16];
        TLD16(tlane + 16 * c, v); TLD16(tlane + NA + 16 * c, v1);
        tld_wait();
#pragma unroll
        for (int k = 0; k < 16; ++k) v[k] = __float_as_uint(fmaf(fa, __uint_as_float(v1[k]), __uint_as_float(v[k])));
#pragma unroll
        for (int q = 0; q < 4; ++q) {
          float4 o;
          o.x = __uint_as_float(v[4 * q]) * (ua * cm_s[16 * c + 4 * q]);
          o.y = __uint_as_float(v[4 * q + 1]) * (ua * cm_s[16 * c + 4 * q + 1]);
          o.z = __uint_as_float(v[4 * q + 2]) * (ua * cm_s[16 * c + 4 * q + 2]);
          o.w = __uint_as_float(v[4 * q + 3]) * (ua * cm_s[16 * c + 4 * q + 3]);
          stage[r * 32 + ((4 * c + q) ^ (r & 7))] = o;
        }
      }
      tc_fence_before();
      asm volatile("bar.sync 1, %0;" ::"n"(2 * TM) : "memory");
#pragma unroll 4
      for (int t = 0; t < 16; ++t) {
        const int row_t = __shfl_sync(FULL_MASK, rw, 16 * h + t);
        const int rr = (warp & 3) * 32 + 16 * h + t;
        if (row_t >= 0) reinterpret_cast<float4*>(B.a_bar + (int64_t)row_t * ROW_A_STRIDE)[lane] = stage[rr * 32 + (lane ^ (rr & 7))];
      }
    }
  }
  tc_fence_before();
  __syncthreads();
  if (warp == 8) {
    tc_fence_after();
    asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem_base), "n"(512) : "memory");
  }
#undef BAR
}


typedef SpsEncodeTiledFn EncodeTiledFn;

// [rows][cols] fp16 row-major -> boxes of box_rows x 64 elements (128 bytes), 128-byte swizzle
sps_status make_map_f16(EncodeTiledFn enc, CUtensorMap* m, const void* ptr, uint64_t rows, uint64_t cols, uint32_t box_rows) {
  const cuuint64_t dims[2] = {cols, rows};
  const cuuint64_t strides[1] = {cols * 2};
  const cuuint32_t box[2] = {(cuuint32_t)KB, box_rows};
  const cuuint32_t es[2] = {1, 1};
  const CUresult r = enc(m, CU_TENSOR_MAP_DATA_TYPE_FLOAT16, 2, const_cast<void*>(ptr), dims, strides, box, es, CU_TENSOR_MAP_INTERLEAVE_NONE,
                         CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  if (r != CUDA_SUCCESS) { sps_set_error("cuTensorMapEncodeTiled (approximate path) failed with CUresult %d", (int)r); return SPS_ECUDA; }
  return SPS_OK;
}

template <int NB>
sps_status launch_nb(const ApproxTc* S, int sm_count, const TableDev& T, const ApproxArgs& G, const RowBuffers& B, cudaStream_t s, bool configure_only) {
  if (configure_only)
    return sps_check_cuda(cudaFuncSetAttribute(approx_tc_kernel<NB>, cudaFuncAttributeMaxDynamicSharedMemorySize, SMEM_TC), "approximate tensor-core kernel shared memory opt-in");
  return sps_check_cuda(sps_launch(approx_tc_kernel<NB>, dim3(sm_count), dim3(THREADS_TC), SMEM_TC, s, T, G, B, S->m1_hi, S->m1_lo, S->m2_hi, S->m2_lo), "approximate contraction (tcgen05) launch");
}
sps_status dispatch(const ApproxTc* S, int sm_count, const TableDev& T, const ApproxArgs& G, const RowBuffers& B, cudaStream_t s, bool configure_only) {
  switch (T.n_band) {
#define CASE(NB) case NB: return launch_nb<NB>(S, sm_count, T, G, B, s, configure_only);
    SPS_APPROX_TC_BANDS(CASE)
#undef CASE
    default: return SPS_EUNSUPPORTED;
  }
}

}  // namespace

bool sps_approx_tc_active(const sps_table* t) { return t->approx_tc != nullptr && !sps_option(SPS_OPT_APPROX_SIMT); }

// Table operands of the tensor-core contraction; leaves t->approx_tc null (SIMT kernel) for shapes outside its range.
sps_status sps_approx_tc_setup(sps_table* t) {
  const TableDev& T = t->dev;
  t->approx_tc = nullptr;
  bool band_ok = false;
#define CASE(NB) band_ok = band_ok || T.n_band == NB;
  SPS_APPROX_TC_BANDS(CASE)
#undef CASE
  if (!band_ok || T.n_Z * T.n_band > 128 || T.n_age > NA || T.n_Z > 16 || 2 * T.n_z > BINS_S) return SPS_OK;
  if (sps_option(SPS_OPT_NO_TC_SETUP)) return SPS_OK;
  EncodeTiledFn enc = sps_tensor_map_encoder();
  if (!enc) return SPS_EUNSUPPORTED;
  ApproxTc* S = new ApproxTc();
  memset(S, 0, sizeof(*S));
  const int n_cells = T.n_z - 1;
  const size_t elems = (size_t)n_cells * NE * NA;
  sps_status st = SPS_OK;
  __half** arrs[4] = {&S->C1_hi, &S->C1_lo, &S->C2_hi, &S->C2_lo};
  for (auto a : arrs)
    if (st == SPS_OK && cudaMalloc(a, elems * sizeof(__half)) != cudaSuccess) { cudaGetLastError(); sps_set_error("cudaMalloc of the approximate-path tensor-core operands failed"); st = SPS_ENOMEM; }
  int* d_max = nullptr;
  if (st == SPS_OK && (cudaMalloc(&d_max, sizeof(int)) != cudaSuccess || cudaMalloc(&S->Cm, (size_t)n_cells * NA * sizeof(float)) != cudaSuccess)) {
    cudaGetLastError(); sps_set_error("cudaMalloc of the approximate-path scales failed"); st = SPS_ENOMEM;
  }
  if (st == SPS_OK) {
    cudaMemset(d_max, 0, sizeof(int));
    cssp_rowmax_kernel<<<(unsigned)(((int64_t)n_cells * NA * 32 + 255) / 256), 256>>>(T, S->Cm, d_max);
    float rho = 0.f;
    st = sps_check_cuda(cudaMemcpy(&rho, d_max, sizeof(float), cudaMemcpyDeviceToHost), "c_SSP range");
    int ex = 0;
    S->sD = 1.f;
    if (rho > 0.f) { std::frexp(rho, &ex); S->sD = std::ldexp(1.f, std::max(-60, std::min(60, -ex))); }         // rho sD in [1/2, 1)
  }
  if (d_max) cudaFree(d_max);
  if (st == SPS_OK) {
    build_c_operands_kernel<<<(unsigned)((elems + 255) / 256), 256>>>(T, S->Cm, S->sD, S->C1_hi, S->C1_lo, S->C2_hi, S->C2_lo);
    sps_count_launch(2);
    st = sps_check_cuda(cudaDeviceSynchronize(), "approximate-path operand build");
  }
  if (st == SPS_OK) st = make_map_f16(enc, &S->m1_hi, S->C1_hi, (uint64_t)n_cells * NE, NA, NE);
  if (st == SPS_OK) st = make_map_f16(enc, &S->m1_lo, S->C1_lo, (uint64_t)n_cells * NE, NA, NE);
  if (st == SPS_OK) st = make_map_f16(enc, &S->m2_hi, S->C2_hi, (uint64_t)n_cells * NA, NE, NA);
  if (st == SPS_OK) st = make_map_f16(enc, &S->m2_lo, S->C2_lo, (uint64_t)n_cells * NA, NE, NA);
  if (st == SPS_OK) st = dispatch(S, t->sm_count, T, ApproxArgs(), RowBuffers(), 0, true);
  t->approx_tc = S;
  if (st != SPS_OK) sps_approx_tc_teardown(t);
  return st;
}

void sps_approx_tc_teardown(sps_table* t) {
  ApproxTc* S = t->approx_tc;
  if (!S) return;
  void* ptrs[] = {S->C1_hi, S->C1_lo, S->C2_hi, S->C2_lo, S->Cm};
  for (void* p : ptrs) if (p) cudaFree(p);
  delete S;
  t->approx_tc = nullptr;
}

sps_status sps_approx_tc_contract(const sps_table* t, Workspace& ws, int64_t n, const int* rows, const int* gal_of_row, const float* obs_flux,
                                  const float* obs_sigma, const float* flux_bar, bool want_grad, cudaStream_t s) {
  if (n <= 0) return SPS_OK;
  const ApproxTc* S = t->approx_tc;
  const TableDev& T = t->dev;
  ApproxArgs G;
  if (ws.rows.cell_list) { G.order = ws.rows.cell_list; G.cap = ws.rows.cell_cap; }      // the prologue filled the per-cell lists
  else { approx_group_rows(T, n, rows, ws.rows, TM, s); G.order = ws.rows.order; G.cap = 0; }
  G.n = n; G.bins = ws.rows.bins; G.gal_of_row = gal_of_row; G.obs_flux = obs_flux; G.obs_sigma = obs_sigma;
  G.flux_bar = flux_bar; G.want_grad = want_grad ? 1 : 0;
  G.Cm = S->Cm; G.inv_sD = 1.f / S->sD;
  sps_prof_begin(SPS_K_APPROX, s);
  sps_status st = dispatch(S, t->sm_count, T, G, ws.rows, s, false);
  sps_prof_end(SPS_K_APPROX, s);
  sps_count_launch();
  if (st != SPS_OK) return st;
  return sps_check_cuda(cudaGetLastError(), "approximate contraction (tcgen05) launch");
}
