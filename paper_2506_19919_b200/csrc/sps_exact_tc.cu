// sps_exact_tc.cu -- tcgen05 / TMA / TMEM kernels of the exact photometry path (a6, a10).
//
// Both contractions of the exact path are dense GEMMs with fp32 operands:
//   forward   S[r,k]    = sum_c W[r,c]      L[c,k]      M = rows, N = wavelengths, K = n_age*n_Z
//   reverse   Wbar[r,c] = sum_k SEDbar[r,k] L[c,k]      M = rows, N = n_age*n_Z,  K = wavelengths
// They run on the 5th-generation tensor cores as three split products with fp32 accumulation in TMEM,
//   x = x_hi + x_lo,   a b ~= a_lo b_hi + a_hi b_lo + a_hi b_hi,
// in one of two operand formats chosen at table creation (sps_table_desc.exact_precision):
//   SPS_EXACT_BF16X3 (default)  hi, lo as BF16 ( 8-bit significands): ~2^-17 per product, 16 K-elements per MMA;
//   SPS_EXACT_TF32X3            hi, lo as TF32 (11-bit significands): ~2^-21 per product, twice the operand bytes, half
//                               the MMA rate and twice the accumulator updates.
// tcgen05 adds each MMA's partial dot product into the fp32 TMEM accumulator with truncation; measured here as a
// relative bias of about -2.4e-8 per update (-7e-6 on S after the 252 updates of the BF16X3 forward pass, -1.2e-5 after
// the 504 of TF32X3), so on this problem BF16X3 is the faster AND the more accurate of the two.
// The SSP table is split once at table creation, in both majornesses; the row-side operands (W, SEDbar) are split by
// the kernels that generate them.
//
// Work restriction (what makes the path fast): the rows of a call are ordered by redshift (counting sort, sps_exact.cu),
// so the 128 rows of a row tile share a narrow z range and only the wavelength tiles under some filter's (5 sigma)
// support at those redshifts are touched: forward items = (row tile, wavelength tile in range), reverse k loop =
// wavelength blocks in range.  Everything outside contributes exactly zero to Eq. (4) and is never computed.
//
// One persistent CTA per SM, 576 threads, warp-specialised:
//   warp 0      TMA producer: 64B-swizzled K-major tiles (A_hi, A_lo: 128 rows; B_hi, B_lo: BN rows; 64 B of K per
//               row) into a 4-stage, 48 KB/stage shared-memory ring, mbarrier complete_tx
//   warp 1      allocates 512 TMEM columns (two 256-column fp32 accumulators) and issues tcgen05.mma
//               (cta_group::1, M = 128, N = BN, 32 B of K per instruction): 6 MMAs per k block
//   warps 2-17  epilogue: tcgen05.ld of their 32 TMEM lanes (thread = row; four warps share a lane quarter and split
//               the columns) while the MMA warp fills the other accumulator.
//               forward: dust attenuation (Eq. A8-A9), redshifted Gaussian filters, trapezoid weight and the
//               reduction over wavelength (Eq. 3-4) fused on the accumulators -- S never reaches HBM; flux and
//               its four direct partials (A_V, delta, F_floor, z) per band stay in registers across the wavelength
//               tiles of a row tile.   reverse: plain store of Wbar.
#include <cuda.h>
#include <cuda_bf16.h>
#include <algorithm>
#include <cstring>
#include <vector>
#include "sps_exact.cuh"
#include "sps_ptx.cuh"

namespace {

#ifndef TC_ROW_BYTES
#define TC_ROW_BYTES 64
#endif
constexpr int BM = 128, BN_MAX = 256;
constexpr int ROW_BYTES = TC_ROW_BYTES;                               // bytes of K per operand row per stage (= swizzle span)
constexpr int STAGES = 256 / ROW_BYTES;                               // 192 KB of operand tiles in flight either way
constexpr int A_TILE_BYTES = BM * ROW_BYTES;
constexpr int B_TILE_BYTES = BN_MAX * ROW_BYTES;
constexpr int STAGE_BYTES = 2 * A_TILE_BYTES + 2 * B_TILE_BYTES;      // 48 KB (64-byte rows) or 96 KB (128-byte rows)
constexpr int CW_BYTES = 5 * BN_MAX * 4;                              // per-wavelength constants of the current tile (forward epilogue)
constexpr int SMEM_BYTES = STAGES * STAGE_BYTES + 1024 + 256 + CW_BYTES;
#ifndef TC_EPI_WARPS
#define TC_EPI_WARPS 16
#endif
constexpr int EPI_WARPS = TC_EPI_WARPS;                              // 4 TMEM lane quarters x EPI_PARTS column parts
constexpr int EPI_PARTS = EPI_WARPS / 4;
constexpr int NUM_THREADS = 64 + 32 * EPI_WARPS;
constexpr int TMEM_COLS = 512;

// operand formats
template <int PREC> struct Op;
template <> struct Op<SPS_EXACT_TF32X3> {
  typedef float T;
  static constexpr int BK = ROW_BYTES / 4;                           // elements per operand row of a k block
  static constexpr uint32_t FMT = 2;                                 // instruction-descriptor format code (TF32)
  static __device__ __forceinline__ float rna(float v) { uint32_t u; asm("cvt.rna.tf32.f32 %0, %1;" : "=r"(u) : "f"(v)); return __uint_as_float(u); }
  static __device__ __forceinline__ void split(float v, T& hi, T& lo) { hi = rna(v); lo = rna(v - hi); }
};
template <> struct Op<SPS_EXACT_BF16X3> {
  typedef __nv_bfloat16 T;
  static constexpr int BK = ROW_BYTES / 2;
  static constexpr uint32_t FMT = 1;                                 // BF16
  static __device__ __forceinline__ void split(float v, T& hi, T& lo) { hi = __float2bfloat16_rn(v); lo = __float2bfloat16_rn(v - __bfloat162float(hi)); }
};

struct FilterConsts {                 // x = lam (1+z) isg + nmu ; T_b = exp2(-x^2) for |x| <= 5 FILT_SCALE
  float isg[SPS_MAX_BAND], nmu[SPS_MAX_BAND], dz[SPS_MAX_BAND], lo[SPS_MAX_BAND], hi[SPS_MAX_BAND];
};

struct TcState {                    // table constants of the tensor-core exact path
  int prec, es, BK;                 // operand format, element size, elements per k block
  void *LT_hi, *LT_lo;              // [n_wave_pad][Wld]    forward B operand (wavelength-major, K = ij contiguous)
  void *Lc_hi, *Lc_lo;              // [nb*BNb][n_wave_pad] reverse B operand (ij-major, K = wavelength contiguous)
  float4* wconst;                   // [n_wave_pad][2]      {lam, dlam, k0, drude}, {log2(lam/5500), -, -, -}
  CUtensorMap mLT_hi, mLT_lo, mLc_hi, mLc_lo;
  FilterConsts fc;
  int Kpad, Wld, nb, BNb;
};

struct GemmArgs {
  int64_t n;
  int m_tiles, n_tiles, k_blocks, BN, BK;
  const int* rows;
  const int* plan; int plan_cap;
  long long* part;        // forward: [n][5][SPS_MAX_BAND] fixed-point band sums (integer atomicAdd: order-independent)
  float* Wbar; int ldw;   // reverse
};

template <int PREC>
__device__ __forceinline__ void tc_mma(uint32_t d_tmem, uint64_t a_desc, uint64_t b_desc, uint32_t idesc, uint32_t accumulate) {
  if (PREC == SPS_EXACT_BF16X3) tc_mma_f16(d_tmem, a_desc, b_desc, idesc, accumulate);
  else tc_mma_tf32(d_tmem, a_desc, b_desc, idesc, accumulate);
}
__device__ __forceinline__ uint64_t umma_desc(uint32_t saddr) { return umma_desc_kmajor(saddr, ROW_BYTES); }

// 2^x for the moderate arguments of the epilogues (|x| < 64): the bare SFU instruction, without exp2f's denormal-range fix-up
__device__ __forceinline__ float ex2_fast(float x) { float y; asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }

// exp(-x^2/2) = exp2(-(x * FILT_SCALE)^2)
#define FILT_SCALE 0.84932180028801907f
#define FILT_CUT (5.f * FILT_SCALE)

// Work items.  forward: item w -> (row tile m, wavelength tile nt) through the per-row-tile prefix plan[0][m] and
// first tile plan[1][m]; reverse: w -> (m, w % n_tiles), k blocks plan[2][m] .. plan[3][m].
struct ItemCursor {
  const int* plan; int plan_cap, n_tiles, m;
  template <int MODE> __device__ __forceinline__ void seek(int w, int& m_out, int& nt, int& kb_lo, int& kb_hi, int k_blocks) {
    if (MODE == 0) {
      while (w >= __ldg(plan + m + 1)) ++m;
      m_out = m; nt = __ldg(plan + plan_cap + m) + (w - __ldg(plan + m)); kb_lo = 0; kb_hi = k_blocks;
    } else {
      m_out = w / n_tiles; nt = w - m_out * n_tiles;
      kb_lo = __ldg(plan + 2 * plan_cap + m_out); kb_hi = __ldg(plan + 3 * plan_cap + m_out);
    }
  }
};

// ---------------------------------------------------------------------------------------------------------------
template <int MODE, int PREC, int NB, int FILT>   // MODE 0: forward with the fused photometry epilogue (NB = compiled band slots; FILT 0 Gaussian / 1 tabulated filters), 1: reverse, store epilogue
__global__ void __launch_bounds__(NUM_THREADS, 1)
exact_gemm_kernel(const __grid_constant__ CUtensorMap tmAh, const __grid_constant__ CUtensorMap tmAl,
                  const __grid_constant__ CUtensorMap tmBh, const __grid_constant__ CUtensorMap tmBl,
                  TableDev T, RowBuffers B, GemmArgs G, FilterConsts FC, const float4* __restrict__ wconst) {
  extern __shared__ uint8_t smem_raw[];
  uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~(uintptr_t)1023);
  const uint32_t smem_base = smem_u32(smem);
  const uint32_t bar_base = smem_base + STAGES * STAGE_BYTES;
  // barriers: full[s] +0, empty[s] +32, tfull[b] +64, tempty[b] +80 ; tmem pointer +96
  auto bar_full = [&](int s) { return bar_base + 8u * s; };
  auto bar_empty = [&](int s) { return bar_base + 32u + 8u * s; };
  auto bar_tfull = [&](int b) { return bar_base + 64u + 8u * b; };
  auto bar_tempty = [&](int b) { return bar_base + 80u + 8u * b; };
  volatile uint32_t* tmem_ptr = reinterpret_cast<volatile uint32_t*>(smem + STAGES * STAGE_BYTES + 96);
  float* cw = reinterpret_cast<float*>(smem + STAGES * STAGE_BYTES + 256);   // [5][BN_MAX] lam, dlam, k0, drude, log2(lam/5500)

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int total = (MODE == 0) ? __ldg(G.plan + G.m_tiles) : G.m_tiles * G.n_tiles;
  const int per = total / (int)gridDim.x, rem = total % (int)gridDim.x;
  const int w_begin = (int)blockIdx.x * per + min((int)blockIdx.x, rem);
  const int w_end = w_begin + per + ((int)blockIdx.x < rem ? 1 : 0);
  ItemCursor cur; cur.plan = G.plan; cur.plan_cap = G.plan_cap; cur.n_tiles = G.n_tiles; cur.m = 0;

  if (threadIdx.x == 0) {
    for (int s = 0; s < STAGES; ++s) { mbar_init(bar_full(s), 1); mbar_init(bar_empty(s), 1); }
    for (int b = 0; b < 2; ++b) { mbar_init(bar_tfull(b), 1); mbar_init(bar_tempty(b), EPI_WARPS); }
    mbar_fence_init();
  }
  if (warp == 1) {
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(bar_base + 96u), "r"(TMEM_COLS) : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
  }
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem_base = *tmem_ptr;

  if (warp == 0) {
    // ===== TMA producer ==========================================================================
    if (lane == 0) {
      const uint32_t tx = 2u * A_TILE_BYTES + 2u * (uint32_t)G.BN * ROW_BYTES;
      int stage = 0; uint32_t phase = 0;
      for (int w = w_begin; w < w_end; ++w) {
        int m, nt, kb_lo, kb_hi;
        cur.seek<MODE>(w, m, nt, kb_lo, kb_hi, G.k_blocks);
        for (int kb = kb_lo; kb < kb_hi; ++kb) {
          mbar_wait(bar_empty(stage), phase ^ 1u);
          const uint32_t sb = smem_base + stage * STAGE_BYTES;
          mbar_expect_tx(bar_full(stage), tx);
          tma_load_2d(sb, &tmAh, bar_full(stage), kb * G.BK, m * BM);
          tma_load_2d(sb + A_TILE_BYTES, &tmAl, bar_full(stage), kb * G.BK, m * BM);
          tma_load_2d(sb + 2 * A_TILE_BYTES, &tmBh, bar_full(stage), kb * G.BK, nt * G.BN);
          tma_load_2d(sb + 2 * A_TILE_BYTES + B_TILE_BYTES, &tmBl, bar_full(stage), kb * G.BK, nt * G.BN);
          if (++stage == STAGES) { stage = 0; phase ^= 1u; }
        }
      }
    }
  } else if (warp == 1) {
    // ===== MMA issuer ============================================================================
    if (lane == 0) {
      // instruction descriptor: D = F32, A and B in the operand format, both K-major, N = BN, M = 128
      const uint32_t idesc = (1u << 4) | (Op<PREC>::FMT << 7) | (Op<PREC>::FMT << 10) | ((uint32_t)(G.BN >> 3) << 17) | ((uint32_t)(BM >> 4) << 24);
      int stage = 0; uint32_t phase = 0; int buf = 0; uint32_t bphase = 0;
      for (int w = w_begin; w < w_end; ++w) {
        int m, nt, kb_lo, kb_hi;
        cur.seek<MODE>(w, m, nt, kb_lo, kb_hi, G.k_blocks);
        mbar_wait(bar_tempty(buf), bphase ^ 1u);
        tc_fence_after();
        const uint32_t d_tmem = tmem_base + (uint32_t)buf * BN_MAX;
        for (int kb = kb_lo; kb < kb_hi; ++kb) {
          mbar_wait(bar_full(stage), phase);
          tc_fence_after();
          const uint32_t sb = smem_base + stage * STAGE_BYTES;
#pragma unroll
          for (int kk = 0; kk < ROW_BYTES / 32; ++kk) {
            const uint64_t a_hi = umma_desc(sb + kk * 32), a_lo = umma_desc(sb + A_TILE_BYTES + kk * 32);
            const uint64_t b_hi = umma_desc(sb + 2 * A_TILE_BYTES + kk * 32);
            const uint64_t b_lo = umma_desc(sb + 2 * A_TILE_BYTES + B_TILE_BYTES + kk * 32);
            tc_mma<PREC>(d_tmem, a_lo, b_hi, idesc, (kb > kb_lo || kk > 0) ? 1u : 0u);    // small terms first
            tc_mma<PREC>(d_tmem, a_hi, b_lo, idesc, 1u);
            tc_mma<PREC>(d_tmem, a_hi, b_hi, idesc, 1u);
          }
          tc_commit(bar_empty(stage));                      // frees the smem stage when these MMAs retire
          if (kb == kb_hi - 1) tc_commit(bar_tfull(buf));
          if (++stage == STAGES) { stage = 0; phase ^= 1u; }
        }
        buf ^= 1; if (buf == 0) bphase ^= 1u;
      }
    }
  } else {
    // ===== epilogue warps ==========================================================================
    const int q = warp & 3;                                  // TMEM lane quarter this warp may read
    const int half = (warp - 2) >> 2;                        // which part of the tile's columns
    const int row_in_tile = q * 32 + lane;
    int buf = 0; uint32_t bphase = 0;
    if (MODE == 0) {
      constexpr int COLS = BN_MAX / EPI_PARTS;
      int cur_m = -1; int64_t r = 0; bool valid = false;
      float zp = 1.f, AVs = 0.f, delta = 0.f, Ffl = 1.f, Eb = 0.85f, zp_min = 1.f, zp_max = 1.f;
      float sc0 = 0.f, sc1 = 0.f, sc2 = 0.f, sc3 = 0.f, sc4 = 0.f;          // fixed-point scales of the row's five band sums
      for (int w = w_begin; w < w_end; ++w) {
        int m, nt, kb_lo, kb_hi;
        cur.seek<MODE>(w, m, nt, kb_lo, kb_hi, G.k_blocks);
        if (m != cur_m) {
          cur_m = m;
          r = (int64_t)m * BM + row_in_tile;
          valid = r < G.n;
          zp = 1.f; AVs = 0.f; delta = 0.f; Ffl = 1.f;
          float Mn = 1.f;
          if (valid) {
            const RowScalars sc = B.sc[G.rows ? G.rows[r] : r];
            zp = 1.f + sc.z; AVs = sc.AV * (1.f / 4.05f); delta = sc.delta; Ffl = sc.Ffloor; Mn = sc.Mn;
          }
          sc0 = part_scale(Mn, T.part_bound, PART_SHIFT_FLUX); sc1 = part_scale(Mn, T.part_bound, PART_SHIFT_AV);
          sc2 = part_scale(Mn, T.part_bound, PART_SHIFT_DELTA); sc3 = part_scale(Mn, T.part_bound, PART_SHIFT_FFLOOR);
          sc4 = part_scale(Mn, T.part_bound, T.part_shift_z);
          Eb = 0.85f - 1.9f * delta;
          float lo = valid ? zp : 1e30f, hi = valid ? zp : 0.f;
#pragma unroll
          for (int o = 16; o > 0; o >>= 1) { lo = fminf(lo, __shfl_xor_sync(FULL_MASK, lo, o)); hi = fmaxf(hi, __shfl_xor_sync(FULL_MASK, hi, o)); }
          zp_min = lo; zp_max = hi;
        }
        // the tile's per-wavelength constants go to shared memory once (coalesced), then are read as broadcasts
        {
          const int et = (int)threadIdx.x - 64;               // 0..255 over the epilogue warps = column of the tile
          asm volatile("bar.sync 1, %0;" ::"n"(32 * EPI_WARPS) : "memory");   // every epilogue warp is done with the previous tile's constants
          if (et < BN_MAX) {
            const float4 c0 = __ldg(&wconst[2 * (nt * BN_MAX + et)]);
            const float l2 = __ldg(&wconst[2 * (nt * BN_MAX + et) + 1].x);
            cw[et] = c0.x; cw[BN_MAX + et] = c0.y; cw[2 * BN_MAX + et] = c0.z; cw[3 * BN_MAX + et] = c0.w; cw[4 * BN_MAX + et] = l2;
          }
          asm volatile("bar.sync 1, %0;" ::"n"(32 * EPI_WARPS) : "memory");
        }
        // bands whose (truncated) support can meet this warp's columns for some of its rows
        unsigned mask = 0;
        {
          const float lam_lo = cw[half * COLS] * zp_min * 0.99999f, lam_hi = cw[half * COLS + COLS - 1] * zp_max * 1.00001f;
#pragma unroll
          for (int b = 0; b < NB; ++b)
            if (b < T.n_band && lam_hi >= FC.lo[b] && lam_lo <= FC.hi[b]) mask |= 1u << b;
        }
        mbar_wait(bar_tfull(buf), bphase);
        tc_fence_after();
        if (mask != 0) {
          // Partial band sums of this warp's columns of this tile, from zero: what a (row, tile, column part) contributes is a
          // fixed sequence of operations on that row's data alone, and the contributions are combined by integer atomics
          // below, so a row's fluxes do not depend on the rows it shares a tile with nor on how tiles are spread over CTAs.
          float s0[NB], s1[NB], s2[NB], s3[NB], s4[NB];
#pragma unroll
          for (int b = 0; b < NB; ++b) s0[b] = s1[b] = s2[b] = s3[b] = s4[b] = 0.f;
          const uint32_t taddr = tmem_base + ((uint32_t)(q * 32) << 16) + (uint32_t)(buf * BN_MAX + half * COLS);
          constexpr int CH = EPI_WARPS > 8 ? 4 : 8;          // columns per step: fewer live registers with more warps
          for (int c = 0; c < COLS / CH; ++c) {
            uint32_t v[CH];
            if (CH == 8) { TMEM_LD8(taddr + c * CH, v); } else { TMEM_LD4(taddr + c * CH, v); }
            const int cb = half * COLS + c * CH;
            float lam8[CH], dl8[CH], k08[CH], dr8[CH], l28[CH];
#pragma unroll
            for (int h = 0; h < CH / 4; ++h) {
              const float4 a0 = *reinterpret_cast<const float4*>(cw + cb + 4 * h), a1 = *reinterpret_cast<const float4*>(cw + BN_MAX + cb + 4 * h);
              const float4 a2 = *reinterpret_cast<const float4*>(cw + 2 * BN_MAX + cb + 4 * h), a3 = *reinterpret_cast<const float4*>(cw + 3 * BN_MAX + cb + 4 * h);
              const float4 a4 = *reinterpret_cast<const float4*>(cw + 4 * BN_MAX + cb + 4 * h);
              lam8[4 * h] = a0.x; lam8[4 * h + 1] = a0.y; lam8[4 * h + 2] = a0.z; lam8[4 * h + 3] = a0.w;
              dl8[4 * h] = a1.x; dl8[4 * h + 1] = a1.y; dl8[4 * h + 2] = a1.z; dl8[4 * h + 3] = a1.w;
              k08[4 * h] = a2.x; k08[4 * h + 1] = a2.y; k08[4 * h + 2] = a2.z; k08[4 * h + 3] = a2.w;
              dr8[4 * h] = a3.x; dr8[4 * h + 1] = a3.y; dr8[4 * h + 2] = a3.z; dr8[4 * h + 3] = a3.w;
              l28[4 * h] = a4.x; l28[4 * h + 1] = a4.y; l28[4 * h + 2] = a4.z; l28[4 * h + 3] = a4.w;
            }
            tmem_ld_wait();
            float G0[CH], G1[CH], G2[CH], G3[CH], G4[CH], lamz[CH];
#pragma unroll
            for (int j = 0; j < CH; ++j) {
              const float lam = lam8[j], dl = dl8[j], k0 = k08[j], dr = dr8[j], l2r = l28[j];
              // dust, Eq. (A8)-(A9) with the tabulated k0, Drude profile and log2(lam/lam_V) (R10)
              const float pw = ex2_fast(delta * l2r);
              const float br = fmaf(k0, pw, Eb * dr);
              float A = AVs * br, A_av = br * (1.f / 4.05f), A_del = AVs * (k0 * pw * l2r * LN2F - 1.9f * dr);
              if (!(A > 0.f)) { A = 0.f; A_av = 0.f; A_del = 0.f; }
              const float Tt = ex2_fast(-0.4f * 3.321928094887362f * A);
              const float dF = -(1.f - Ffl) * 0.4f * LN10F * Tt;
              const float Sd = __uint_as_float(v[j]) * dl;
              G0[j] = Sd * fmaf(1.f - Ffl, Tt, Ffl); G1[j] = Sd * dF * A_av; G2[j] = Sd * dF * A_del; G3[j] = Sd * (1.f - Tt);
              G4[j] = G0[j] * lam; lamz[j] = lam * zp;
            }
#pragma unroll
            for (int b = 0; b < NB; ++b) {
              if (mask & (1u << b)) {
                if (FILT == 0) {
                  const float isg = FC.isg[b], nmu = FC.nmu[b];
#pragma unroll
                  for (int j = 0; j < CH; ++j) {
                    const float x = fmaf(lamz[j], isg, nmu);
                    const float Tb = (fabsf(x) <= FILT_CUT) ? ex2_fast(-x * x) : 0.f;
                    s0[b] = fmaf(Tb, G0[j], s0[b]); s1[b] = fmaf(Tb, G1[j], s1[b]); s2[b] = fmaf(Tb, G2[j], s2[b]); s3[b] = fmaf(Tb, G3[j], s3[b]);
                    s4[b] = fmaf(Tb * x, G4[j], s4[b]);   // d/dz of T_b(lam (1+z)) = -T x' lam / sigma: the band's factor FC.dz is applied at the flush
                  }
                } else {
#pragma unroll
                  for (int j = 0; j < CH; ++j) {
                    float Tb, dTb;
                    filter_tab_eval(T.ft, b, lamz[j], Tb, dTb);
                    s0[b] = fmaf(Tb, G0[j], s0[b]); s1[b] = fmaf(Tb, G1[j], s1[b]); s2[b] = fmaf(Tb, G2[j], s2[b]); s3[b] = fmaf(Tb, G3[j], s3[b]);
                    s4[b] = fmaf(dTb, G4[j], s4[b]);      // d/dz of T_b(lam (1+z)) = T_b' lam
                  }
                }
              }
            }
          }
          if (valid) {
            long long* p = G.part + r * 5 * SPS_MAX_BAND;
#pragma unroll
            for (int b = 0; b < NB; ++b) {
              if (mask & (1u << b)) {
                part_add(p + b, s0[b], sc0); part_add(p + SPS_MAX_BAND + b, s1[b], sc1); part_add(p + 2 * SPS_MAX_BAND + b, s2[b], sc2);
                part_add(p + 3 * SPS_MAX_BAND + b, s3[b], sc3); part_add(p + 4 * SPS_MAX_BAND + b, s4[b] * (FILT == 0 ? FC.dz[b] : 1.f), sc4);
              }
            }
          }
        }
        tc_fence_before();
        __syncwarp();
        if (lane == 0) mbar_arrive(bar_tempty(buf));
        buf ^= 1; if (buf == 0) bphase ^= 1u;
      }
    } else {
      for (int w = w_begin; w < w_end; ++w) {
        int m, nt, kb_lo, kb_hi;
        cur.seek<MODE>(w, m, nt, kb_lo, kb_hi, G.k_blocks);
        const int64_t r = (int64_t)m * BM + row_in_tile;
        mbar_wait(bar_tfull(buf), bphase);
        tc_fence_after();
        const uint32_t taddr = tmem_base + ((uint32_t)(q * 32) << 16) + (uint32_t)buf * BN_MAX;
        float* dst = G.Wbar + r * G.ldw + nt * G.BN;
        for (int c = half; c < G.BN / 16; c += EPI_PARTS) {
          uint32_t v[16];
          TMEM_LD16(taddr + c * 16, v);
          tmem_ld_wait();
          if (r < G.n) {
#pragma unroll
            for (int j = 0; j < 4; ++j)
              reinterpret_cast<float4*>(dst + c * 16)[j] = make_float4(__uint_as_float(v[4 * j]), __uint_as_float(v[4 * j + 1]),
                                                                      __uint_as_float(v[4 * j + 2]), __uint_as_float(v[4 * j + 3]));
          }
        }
        tc_fence_before();
        __syncwarp();
        if (lane == 0) mbar_arrive(bar_tempty(buf));
        buf ^= 1; if (buf == 0) bphase ^= 1u;
      }
    }
  }
  tc_fence_before();
  __syncthreads();
  if (warp == 1) {
    tc_fence_after();
    asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem_base), "r"(TMEM_COLS) : "memory");
  }
}

// ---- plan: per row tile, the wavelength range under some filter's support for the tile's redshifts -------------------
// plan[0][m] = prefix of forward items, plan[1][m] = first wavelength tile, plan[2][m], plan[3][m] = k-block range (reverse)
// One CTA per row tile (thread = row): redshift range of the tile -> wavelength ranges; also counts the tile's
// (row, wavelength) pairs under some filter's support (the algorithmic work reported by sps_exact_last_work).
__global__ void __launch_bounds__(BM) exact_plan_kernel(TableDev T, int64_t n, const int* __restrict__ rows, RowBuffers B, FilterConsts FC,
                                                        int BKe, int* __restrict__ plan, int plan_cap, unsigned long long* __restrict__ work) {
  __shared__ float s_min[BM / 32], s_max[BM / 32];
  __shared__ unsigned s_pairs[BM / 32];
  const int m = blockIdx.x;
  const int64_t r = (int64_t)m * BM + threadIdx.x;
  float obs_lo = 1e30f, obs_hi = 0.f;
  for (int b = 0; b < T.n_band; ++b) { obs_lo = fminf(obs_lo, FC.lo[b]); obs_hi = fmaxf(obs_hi, FC.hi[b]); }
  float zmin = 1e30f, zmax = -1e30f; unsigned pairs = 0;
  if (r < n) {
    const float z = B.sc[rows ? rows[r] : r].z; zmin = zmax = z;
    const float rlo = obs_lo / (1.f + z), rhi = obs_hi / (1.f + z);
    int a = 0, c = T.n_wave;
    while (a < c) { const int mid = (a + c) >> 1; if (T.wave[mid] < rlo) a = mid + 1; else c = mid; }
    const int first = a; c = T.n_wave;
    while (a < c) { const int mid = (a + c) >> 1; if (T.wave[mid] <= rhi) a = mid + 1; else c = mid; }
    pairs = (unsigned)(a - first);
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    zmin = fminf(zmin, __shfl_xor_sync(FULL_MASK, zmin, o)); zmax = fmaxf(zmax, __shfl_xor_sync(FULL_MASK, zmax, o));
    pairs += __shfl_xor_sync(FULL_MASK, pairs, o);
  }
  if ((threadIdx.x & 31) == 0) { s_min[threadIdx.x >> 5] = zmin; s_max[threadIdx.x >> 5] = zmax; s_pairs[threadIdx.x >> 5] = pairs; }
  __syncthreads();
  if (threadIdx.x == 0) {
    unsigned long long tot = 0;
    for (int w = 0; w < BM / 32; ++w) { zmin = fminf(zmin, s_min[w]); zmax = fmaxf(zmax, s_max[w]); tot += s_pairs[w]; }
    atomicAdd(work, tot);                                   // this call
    atomicAdd(work + 1, tot);                               // running total (sps_exact_work_since)
    const float lo = obs_lo / (1.f + zmax) * 0.99999f, hi = obs_hi / (1.f + zmin) * 1.00001f;
    int a = 0, c = T.n_wave;
    while (a < c) { const int mid = (a + c) >> 1; if (T.wave[mid] < lo) a = mid + 1; else c = mid; }
    const int k_lo = max(a - 1, 0);
    a = k_lo; c = T.n_wave;
    while (a < c) { const int mid = (a + c) >> 1; if (T.wave[mid] <= hi) a = mid + 1; else c = mid; }
    int k_hi = min(a, T.n_wave - 1);                         // inclusive
    if (k_hi < k_lo) k_hi = k_lo;
    plan[plan_cap + m] = k_lo / BN_MAX;
    plan[2 * plan_cap + m] = k_lo / BKe;
    plan[3 * plan_cap + m] = k_hi / BKe + 1;
    plan[m] = k_hi / BN_MAX + 1 - k_lo / BN_MAX;             // number of wavelength tiles; exact_scan_kernel turns it into a prefix
  }
}
__global__ void exact_scan_kernel(int m_tiles, int* __restrict__ plan) {
  if (threadIdx.x != 0 || blockIdx.x != 0) return;
  int acc = 0;
  for (int m = 0; m < m_tiles; ++m) { const int c = plan[m]; plan[m] = acc; acc += c; }
  plan[m_tiles] = acc;
}

// ---- operand generation -----------------------------------------------------------------------------------------
// forward B operand: LT[k][c] = L[c][k]  (one-time, at table creation)
template <int PREC>
__global__ void build_LT_kernel(TableDev T, int Wld, typename Op<PREC>::T* __restrict__ hi, typename Op<PREC>::T* __restrict__ lo) {
  __shared__ float tile[32][33];
  const int k0 = blockIdx.x * 32, c0 = blockIdx.y * 32;
  for (int i = threadIdx.y; i < 32; i += blockDim.y) {
    const int c = c0 + i, k = k0 + threadIdx.x;
    tile[i][threadIdx.x] = (c < T.K && k < T.n_wave) ? T.ssp[(int64_t)c * T.n_wave_pad + k] : 0.f;
  }
  __syncthreads();
  for (int i = threadIdx.y; i < 32; i += blockDim.y) {
    const int k = k0 + i, c = c0 + threadIdx.x;
    if (k < T.n_wave_pad && c < Wld) Op<PREC>::split(tile[threadIdx.x][i], hi[(int64_t)k * Wld + c], lo[(int64_t)k * Wld + c]);
  }
}
// reverse B operand: Lc[c][k] = L[c][k], zero rows for c >= K
template <int PREC>
__global__ void build_Lc_kernel(TableDev T, int rows, typename Op<PREC>::T* __restrict__ hi, typename Op<PREC>::T* __restrict__ lo) {
  const int64_t idx = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= (int64_t)rows * T.n_wave_pad) return;
  const int c = (int)(idx / T.n_wave_pad), k = (int)(idx % T.n_wave_pad);
  const float v = (c < T.K && k < T.n_wave) ? T.ssp[(int64_t)c * T.n_wave_pad + k] : 0.f;
  Op<PREC>::split(v, hi[idx], lo[idx]);
}
__global__ void build_wconst_kernel(TableDev T, float4* __restrict__ wc) {
  const int k = blockIdx.x * blockDim.x + threadIdx.x;
  if (k >= T.n_wave_pad) return;
  wc[2 * k] = make_float4(T.wave[k], T.dlam[k], T.k0[k], T.drude[k]);
  wc[2 * k + 1] = make_float4(T.l2r[k], 0.f, 0.f, 0.f);
}

// forward A operand: W[r][ij] = Mn a_i m_j (a5: Eq. 2 and M_star), split.  One block per row, two consecutive entries per
// thread (packed stores); a_i and m_j of the row are staged in shared memory, ij -> (i, j) without an integer division.
template <int PREC>
__global__ void __launch_bounds__(128) tc_weights_kernel(TableDev T, int64_t n, const int* __restrict__ rows, RowBuffers B, int Wld,
                                                         typename Op<PREC>::T* __restrict__ hi, typename Op<PREC>::T* __restrict__ lo) {
  typedef typename Op<PREC>::T E;
  const int64_t r = blockIdx.x;
  const int64_t row = rows ? rows[r] : r;
  __shared__ float a_s[ROW_A_STRIDE], m_s[ROW_M_STRIDE];
  __shared__ float mt_s[SPS_MAX_AGE * SPS_MAX_Z];            // non-separable weights (R26): the MDF of every age bin
  const bool nonsep = T.agez_gamma != 0.f;
  a_s[threadIdx.x] = B.a[row * ROW_A_STRIDE + threadIdx.x] * B.sc[row].Mn;
  if (threadIdx.x < ROW_M_STRIDE) m_s[threadIdx.x] = B.m[row * ROW_M_STRIDE + threadIdx.x];
  if (nonsep && threadIdx.x < T.n_age) {
    float d1[SPS_MAX_Z], d2[SPS_MAX_Z];
    mdf_row(T, B.sc[row].pad1 + T.agez_gamma * T.la9[threadIdx.x], B.sc[row].pad2, mt_s + threadIdx.x * SPS_MAX_Z, d1, d2);
  }
  __syncthreads();
  const float inv_nZ = 1.f / (float)T.n_Z;
  for (int e = 2 * threadIdx.x; e < Wld; e += 2 * blockDim.x) {          // Wld is a multiple of the k block, hence even
    E h2[2], l2[2];
    int i = (int)(((float)e + 0.5f) * inv_nZ), j = e - i * T.n_Z;         // exact for e < 2^16 (n_age n_Z <= 2048)
#pragma unroll
    for (int u = 0; u < 2; ++u) {
      const float v = (e + u < T.K) ? a_s[min(i, ROW_A_STRIDE - 1)] * (nonsep ? mt_s[min(i, ROW_A_STRIDE - 1) * SPS_MAX_Z + j] : m_s[j]) : 0.f;
      Op<PREC>::split(v, h2[u], l2[u]);
      if (++j == T.n_Z) { j = 0; ++i; }
    }
    const int64_t o = r * Wld + e;
    if (sizeof(E) == 2) {
      *reinterpret_cast<uint32_t*>(hi + o) = *reinterpret_cast<const uint32_t*>(h2);
      *reinterpret_cast<uint32_t*>(lo + o) = *reinterpret_cast<const uint32_t*>(l2);
    } else {
      *reinterpret_cast<uint2*>(hi + o) = *reinterpret_cast<const uint2*>(h2);
      *reinterpret_cast<uint2*>(lo + o) = *reinterpret_cast<const uint2*>(l2);
    }
  }
}

// reverse A operand: SEDbar[r][k] = F_att(lam_k) dlam_k sum_b g_b T_b(lam_k (1+z))  (reverse of Eq. 3-4), split.
// Only the k blocks of the row tile's plan range are written (the reverse GEMM reads nothing else).
// One block per row; per pass a warp owns 256 consecutive wavelengths (a thread: four pairs 64 apart, so loads and stores
// stay coalesced): the bands whose 5-sigma support meets the warp's span at the row's redshift are found once per pass,
// warp-uniformly (the filters overlap little, so two to four of them), and only those are evaluated.  The kernel is
// instruction-issue bound (a per-element loop over all bands cost 148 instructions per element).
constexpr int SB_G = 4, SB_THREADS = 128, SB_SPAN = 64 * SB_G;
template <int PREC, int FILT>
__global__ void __launch_bounds__(SB_THREADS) tc_sedbar_kernel(TableDev T, int64_t n, const int* __restrict__ rows, RowBuffers B, FilterConsts FC,
                                                               const float* __restrict__ gbuf, const float4* __restrict__ wconst,
                                                               const int* __restrict__ plan, int plan_cap,
                                                               typename Op<PREC>::T* __restrict__ hi, typename Op<PREC>::T* __restrict__ lo) {
  typedef typename Op<PREC>::T E;
  const int64_t r = blockIdx.x;
  const int m = (int)(r / BM);
  const int k_begin = plan[2 * plan_cap + m] * Op<PREC>::BK, k_end = plan[3 * plan_cap + m] * Op<PREC>::BK;
  __shared__ float g_s[SPS_MAX_BAND];
  __shared__ float sc_s[4];
  if (threadIdx.x < SPS_MAX_BAND) g_s[threadIdx.x] = gbuf[r * SPS_MAX_BAND + threadIdx.x];
  if (threadIdx.x == 32) {
    const RowScalars sc = B.sc[rows ? rows[r] : r];
    sc_s[0] = 1.f + sc.z; sc_s[1] = sc.AV * (1.f / 4.05f); sc_s[2] = sc.delta; sc_s[3] = sc.Ffloor;
  }
  __syncthreads();
  const float zp = sc_s[0], AVs = sc_s[1], delta = sc_s[2], Ffl = sc_s[3], Eb = 0.85f - 1.9f * delta;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  for (int kb = k_begin + SB_SPAN * warp; kb < k_end; kb += SB_SPAN * (SB_THREADS / 32)) {
    float4 c0[2 * SB_G];
    float tsum[2 * SB_G], lamz[2 * SB_G];
    float mx = 0.f;
#pragma unroll
    for (int e = 0; e < 2 * SB_G; ++e) {
      const int k = kb + 64 * (e >> 1) + 2 * lane + (e & 1);
      c0[e] = (k < k_end) ? __ldg(&wconst[2 * k]) : make_float4(0.f, 0.f, 0.f, 0.f);
      lamz[e] = c0[e].x * zp; tsum[e] = 0.f;
      mx = fmaxf(mx, lamz[e]);                              // padded columns carry no wavelength: take the largest
    }
    const float lam_lo = __shfl_sync(FULL_MASK, lamz[0], 0) * 0.99999f;
    const float lam_hi = __uint_as_float(__reduce_max_sync(FULL_MASK, __float_as_uint(mx))) * 1.00001f;
    for (int b = 0; b < T.n_band; ++b) {
      if (lam_hi >= FC.lo[b] && lam_lo <= FC.hi[b]) {
        const float isg = FC.isg[b], nmu = FC.nmu[b], g = g_s[b];
#pragma unroll
        for (int e = 0; e < 2 * SB_G; ++e) {
          if (FILT == 0) {
            const float x = fmaf(lamz[e], isg, nmu);
            if (fabsf(x) <= FILT_CUT) tsum[e] = fmaf(g, ex2_fast(-x * x), tsum[e]);
          } else {
            float Tb, dTb;
            filter_tab_eval(T.ft, b, lamz[e], Tb, dTb);
            tsum[e] = fmaf(g, Tb, tsum[e]);
          }
        }
      }
    }
#pragma unroll
    for (int q = 0; q < SB_G; ++q) {
      const int k = kb + 64 * q + 2 * lane;
      E h2[2], l2[2];
#pragma unroll
      for (int u = 0; u < 2; ++u) {
        const int e = 2 * q + u;
        float v = 0.f;
        if (c0[e].y > 0.f && tsum[e] != 0.f) {
          const float l2r = __ldg(&wconst[2 * (k + u) + 1].x);
          const float pw = ex2_fast(delta * l2r);
          float A = AVs * fmaf(c0[e].z, pw, Eb * c0[e].w);
          if (!(A > 0.f)) A = 0.f;
          const float Tt = ex2_fast(-0.4f * 3.321928094887362f * A);
          v = fmaf(1.f - Ffl, Tt, Ffl) * c0[e].y * tsum[e];
        }
        Op<PREC>::split(v, h2[u], l2[u]);
      }
      if (k < k_end) {
        const int64_t o = r * T.n_wave_pad + k;
        if (sizeof(E) == 2) {
          *reinterpret_cast<uint32_t*>(hi + o) = *reinterpret_cast<const uint32_t*>(h2);
          *reinterpret_cast<uint32_t*>(lo + o) = *reinterpret_cast<const uint32_t*>(l2);
        } else {
          *reinterpret_cast<uint2*>(hi + o) = *reinterpret_cast<const uint2*>(h2);
          *reinterpret_cast<uint2*>(lo + o) = *reinterpret_cast<const uint2*>(l2);
        }
      }
    }
  }
}

// ---- host side --------------------------------------------------------------------------------------------------
// [rows][cols] row-major with pitch `ld` elements -> tiles of box_rows x ROW_BYTES, swizzled
sps_status make_map(const TcState* S, CUtensorMap* m, const void* base, uint64_t rows, uint64_t cols, uint64_t ld, uint32_t box_rows) {
  SpsEncodeTiledFn enc = sps_tensor_map_encoder();
  if (!enc) return SPS_EUNSUPPORTED;
  const cuuint64_t dims[2] = {cols, rows};
  const cuuint64_t strides[1] = {ld * (uint64_t)S->es};
  const cuuint32_t box[2] = {(cuuint32_t)S->BK, box_rows};
  const cuuint32_t es[2] = {1, 1};
  const CUresult r = enc(m, S->prec == SPS_EXACT_BF16X3 ? CU_TENSOR_MAP_DATA_TYPE_BFLOAT16 : CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 2,
                         const_cast<void*>(base), dims, strides, box, es, CU_TENSOR_MAP_INTERLEAVE_NONE, ROW_BYTES == 128 ? CU_TENSOR_MAP_SWIZZLE_128B : CU_TENSOR_MAP_SWIZZLE_64B,
                         CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  if (r != CUDA_SUCCESS) { sps_set_error("cuTensorMapEncodeTiled failed with CUresult %d", (int)r); return SPS_ECUDA; }
  return SPS_OK;
}

template <int PREC, int NB, int FILT>
sps_status optin_fwd() { return sps_check_cuda(cudaFuncSetAttribute(exact_gemm_kernel<0, PREC, NB, FILT>, cudaFuncAttributeMaxDynamicSharedMemorySize, SMEM_BYTES), "smem opt-in"); }

template <int PREC>
sps_status build_tables(const TableDev& T, TcState* S, size_t lc_rows) {
  typedef typename Op<PREC>::T E;
  const size_t lc_n = lc_rows * T.n_wave_pad;
  build_LT_kernel<PREC><<<dim3((T.n_wave_pad + 31) / 32, (S->Wld + 31) / 32), dim3(32, 8)>>>(T, S->Wld, (E*)S->LT_hi, (E*)S->LT_lo);
  build_Lc_kernel<PREC><<<(unsigned)((lc_n + 255) / 256), 256>>>(T, (int)lc_rows, (E*)S->Lc_hi, (E*)S->Lc_lo);
  build_wconst_kernel<<<(T.n_wave_pad + 255) / 256, 256>>>(T, S->wconst);
  sps_count_launch(3);
  sps_status st = sps_check_cuda(cudaDeviceSynchronize(), "tensor-core operand build");
  if (st == SPS_OK) st = optin_fwd<PREC, 4, 0>();
  if (st == SPS_OK) st = optin_fwd<PREC, 10, 0>();
  if (st == SPS_OK) st = optin_fwd<PREC, 16, 0>();
  if (st == SPS_OK) st = optin_fwd<PREC, 16, 1>();
  if (st == SPS_OK) st = sps_check_cuda(cudaFuncSetAttribute(exact_gemm_kernel<1, PREC, 1, 0>, cudaFuncAttributeMaxDynamicSharedMemorySize, SMEM_BYTES), "smem opt-in");
  return st;
}

template <int PREC>
sps_status launch_forward(const sps_table* t, const TcState* S, Workspace& ws, int64_t n, const int* rows, cudaStream_t s) {
  typedef typename Op<PREC>::T E;
  ExactScratch& X = ws.x; const TableDev& T = t->dev;
  tc_weights_kernel<PREC><<<(unsigned)n, 128, 0, s>>>(T, n, rows, ws.rows, S->Wld, (E*)X.W_hi, (E*)X.W_lo);
  GemmArgs G; memset(&G, 0, sizeof(G));
  G.n = n; G.m_tiles = (int)((n + BM - 1) / BM); G.n_tiles = T.n_wave_pad / BN_MAX; G.k_blocks = S->Kpad / S->BK; G.BN = BN_MAX; G.BK = S->BK;
  G.rows = rows; G.part = X.part; G.plan = X.plan; G.plan_cap = X.plan_cap;
  cudaMemsetAsync(X.work, 0, sizeof(unsigned long long), s);
  exact_plan_kernel<<<G.m_tiles, BM, 0, s>>>(T, n, rows, ws.rows, S->fc, S->BK, X.plan, X.plan_cap, X.work);
  ++X.work_calls;
  exact_scan_kernel<<<1, 32, 0, s>>>(G.m_tiles, X.plan);
  const int grid = std::min(t->sm_count, G.m_tiles * G.n_tiles);
  sps_prof_begin(SPS_K_EXACT_FWD, s);
#define FWD(NBV, FV) exact_gemm_kernel<0, PREC, NBV, FV><<<grid, NUM_THREADS, SMEM_BYTES, s>>>(X.mW_hi, X.mW_lo, S->mLT_hi, S->mLT_lo, T, ws.rows, G, S->fc, S->wconst)
  if (T.filt_tab) FWD(16, 1);
  else if (T.n_band <= 4) FWD(4, 0);
  else if (T.n_band <= 10) FWD(10, 0);
  else FWD(16, 0);
#undef FWD
  sps_prof_end(SPS_K_EXACT_FWD, s);
  sps_count_launch(4);
  return sps_check_cuda(cudaGetLastError(), "exact forward (tcgen05) launch");
}

template <int PREC>
sps_status launch_backward(const sps_table* t, const TcState* S, Workspace& ws, int64_t n, const int* rows, cudaStream_t s) {
  typedef typename Op<PREC>::T E;
  ExactScratch& X = ws.x; const TableDev& T = t->dev;
  if (T.filt_tab) tc_sedbar_kernel<PREC, 1><<<(unsigned)n, SB_THREADS, 0, s>>>(T, n, rows, ws.rows, S->fc, X.gbuf, S->wconst, X.plan, X.plan_cap, (E*)X.SB_hi, (E*)X.SB_lo);
  else tc_sedbar_kernel<PREC, 0><<<(unsigned)n, SB_THREADS, 0, s>>>(T, n, rows, ws.rows, S->fc, X.gbuf, S->wconst, X.plan, X.plan_cap, (E*)X.SB_hi, (E*)X.SB_lo);
  GemmArgs G; memset(&G, 0, sizeof(G));
  G.n = n; G.m_tiles = (int)((n + BM - 1) / BM); G.n_tiles = S->nb; G.k_blocks = T.n_wave_pad / S->BK; G.BN = S->BNb; G.BK = S->BK;
  G.rows = rows; G.Wbar = X.Wbar; G.ldw = t->exact->ldw; G.plan = X.plan; G.plan_cap = X.plan_cap;
  const int grid = std::min(t->sm_count, G.m_tiles * G.n_tiles);
  sps_prof_begin(SPS_K_EXACT_BWD, s);
  exact_gemm_kernel<1, PREC, 1, 0><<<grid, NUM_THREADS, SMEM_BYTES, s>>>(X.mSB_hi, X.mSB_lo, S->mLc_hi, S->mLc_lo, T, ws.rows, G, S->fc, S->wconst);
  sps_prof_end(SPS_K_EXACT_BWD, s);
  sps_count_launch(2);
  return sps_check_cuda(cudaGetLastError(), "exact reverse (tcgen05) launch");
}

}  // namespace

sps_status sps_exact_tc_setup(sps_table* t, int precision) {
  ExactState* X = t->exact;
  X->use_tc = false; X->tc = nullptr;
  if (sps_option(SPS_OPT_NO_TC_SETUP)) return SPS_OK;
  if (precision != SPS_EXACT_TF32X3 && precision != SPS_EXACT_BF16X3) { sps_set_error("exact_precision must be SPS_EXACT_TF32X3 or SPS_EXACT_BF16X3"); return SPS_EINVAL; }
  if (!sps_tensor_map_encoder()) return SPS_EUNSUPPORTED;
  const TableDev& T = t->dev;
  TcState* S = new TcState();
  memset(S, 0, sizeof(*S));
  S->prec = precision; S->es = precision == SPS_EXACT_BF16X3 ? 2 : 4; S->BK = ROW_BYTES / S->es;
  S->Kpad = (T.K + 63) / 64 * 64;
  S->nb = (S->Kpad + BN_MAX - 1) / BN_MAX;
  S->BNb = ((S->Kpad + S->nb - 1) / S->nb + 15) / 16 * 16;
  S->Wld = (std::max(S->Kpad, S->nb * S->BNb) + 63) / 64 * 64;
  for (int b = 0; b < SPS_MAX_BAND; ++b) {
    const float mu = b < T.n_band ? T.filt_mu[b] : 1.f, sg = b < T.n_band ? T.filt_sigma[b] : 1.f;
    S->fc.isg[b] = FILT_SCALE / sg; S->fc.nmu[b] = -mu * (FILT_SCALE / sg);
    S->fc.dz[b] = -1.f / (sg * FILT_SCALE);
    S->fc.lo[b] = mu - 5.f * sg; S->fc.hi[b] = mu + 5.f * sg;
    if (T.filt_tab && b < T.n_band) { S->fc.lo[b] = T.ft.lo[b]; S->fc.hi[b] = T.ft.hi[b]; }     // the support of a tabulated curve
  }
  const size_t lt_n = (size_t)T.n_wave_pad * S->Wld, lc_rows = (size_t)S->nb * S->BNb, lc_n = lc_rows * T.n_wave_pad;
  cudaError_t e = cudaMalloc(&S->LT_hi, lt_n * S->es);
  if (e == cudaSuccess) e = cudaMalloc(&S->LT_lo, lt_n * S->es);
  if (e == cudaSuccess) e = cudaMalloc(&S->Lc_hi, lc_n * S->es);
  if (e == cudaSuccess) e = cudaMalloc(&S->Lc_lo, lc_n * S->es);
  if (e == cudaSuccess) e = cudaMalloc(&S->wconst, (size_t)T.n_wave_pad * 2 * sizeof(float4));
  X->tc = S;
  if (e != cudaSuccess) { sps_exact_tc_teardown(t); return sps_check_cuda(e, "tensor-core operand allocation"); }
  sps_status st = precision == SPS_EXACT_BF16X3 ? build_tables<SPS_EXACT_BF16X3>(T, S, lc_rows) : build_tables<SPS_EXACT_TF32X3>(T, S, lc_rows);
  if (st == SPS_OK) st = make_map(S, &S->mLT_hi, S->LT_hi, T.n_wave_pad, S->Wld, S->Wld, BN_MAX);
  if (st == SPS_OK) st = make_map(S, &S->mLT_lo, S->LT_lo, T.n_wave_pad, S->Wld, S->Wld, BN_MAX);
  if (st == SPS_OK) st = make_map(S, &S->mLc_hi, S->Lc_hi, lc_rows, T.n_wave_pad, T.n_wave_pad, S->BNb);
  if (st == SPS_OK) st = make_map(S, &S->mLc_lo, S->Lc_lo, lc_rows, T.n_wave_pad, T.n_wave_pad, S->BNb);
  if (st != SPS_OK) { sps_exact_tc_teardown(t); return st; }
  X->ldw = S->Wld;
  X->use_tc = true;
  return SPS_OK;
}

void sps_exact_tc_teardown(sps_table* t) {
  ExactState* X = t->exact;
  if (!X || !X->tc) return;
  TcState* S = (TcState*)X->tc;
  void* ptrs[] = {S->LT_hi, S->LT_lo, S->Lc_hi, S->Lc_lo, S->wconst};
  for (void* p : ptrs) if (p) cudaFree(p);
  delete S;
  X->tc = nullptr; X->use_tc = false;
}

void sps_exact_tc_free_scratch(ExactScratch& X) {
  void* ptrs[] = {X.W_hi, X.W_lo, X.SB_hi, X.SB_lo, X.plan, X.work};
  for (void* p : ptrs) if (p) cudaFree(p);
  X.W_hi = X.W_lo = X.SB_hi = X.SB_lo = nullptr; X.plan = nullptr; X.work = nullptr; X.tc_cap = 0; X.plan_cap = 0;
}

// row-side operand buffers for `cap` rows (cap is a multiple of 128); called when the exact scratch grows
sps_status sps_exact_tc_ensure(const sps_table* t, ExactScratch& X, int64_t cap) {
  if (!t->exact->use_tc) return SPS_OK;
  const TcState* S = (const TcState*)t->exact->tc;
  if (X.tc_cap >= cap) return SPS_OK;
  sps_exact_tc_free_scratch(X);
  const TableDev& T = t->dev;
  const size_t wn = (size_t)cap * S->Wld, sn = (size_t)cap * T.n_wave_pad;
  X.plan_cap = (int)(cap / BM) + 2;
  cudaError_t e = cudaMalloc(&X.W_hi, wn * S->es);
  if (e == cudaSuccess) e = cudaMalloc(&X.W_lo, wn * S->es);
  if (e == cudaSuccess) e = cudaMalloc(&X.SB_hi, sn * S->es);
  if (e == cudaSuccess) e = cudaMalloc(&X.SB_lo, sn * S->es);
  if (e == cudaSuccess) e = cudaMalloc(&X.plan, (size_t)4 * X.plan_cap * sizeof(int));
  if (e == cudaSuccess) e = cudaMalloc(&X.work, 2 * sizeof(unsigned long long));
  if (e != cudaSuccess) { sps_exact_tc_free_scratch(X); return sps_check_cuda(e, "tensor-core row operand allocation"); }
  cudaMemset(X.W_hi, 0, wn * S->es); cudaMemset(X.W_lo, 0, wn * S->es);
  cudaMemset(X.SB_hi, 0, sn * S->es); cudaMemset(X.SB_lo, 0, sn * S->es);
  cudaMemset(X.work, 0, 2 * sizeof(unsigned long long));
  X.work_calls = 0;
  X.tc_cap = cap;
  sps_status st = make_map(S, &X.mW_hi, X.W_hi, cap, S->Wld, S->Wld, BM);
  if (st == SPS_OK) st = make_map(S, &X.mW_lo, X.W_lo, cap, S->Wld, S->Wld, BM);
  if (st == SPS_OK) st = make_map(S, &X.mSB_hi, X.SB_hi, cap, T.n_wave_pad, T.n_wave_pad, BM);
  if (st == SPS_OK) st = make_map(S, &X.mSB_lo, X.SB_lo, cap, T.n_wave_pad, T.n_wave_pad, BM);
  return st;
}

sps_status sps_exact_tc_forward(const sps_table* t, Workspace& ws, int64_t n, const int* rows, cudaStream_t s) {
  const TcState* S = (const TcState*)t->exact->tc;
  return S->prec == SPS_EXACT_BF16X3 ? launch_forward<SPS_EXACT_BF16X3>(t, S, ws, n, rows, s) : launch_forward<SPS_EXACT_TF32X3>(t, S, ws, n, rows, s);
}

sps_status sps_exact_tc_backward(const sps_table* t, Workspace& ws, int64_t n, const int* rows, cudaStream_t s) {
  const TcState* S = (const TcState*)t->exact->tc;
  return S->prec == SPS_EXACT_BF16X3 ? launch_backward<SPS_EXACT_BF16X3>(t, S, ws, n, rows, s) : launch_backward<SPS_EXACT_TF32X3>(t, S, ws, n, rows, s);
}

extern "C" sps_status sps_exact_last_work(const sps_table* t, int64_t* row_wavelength_pairs) {
  if (!t || !row_wavelength_pairs) { sps_set_error("sps_exact_last_work: null argument"); return SPS_EINVAL; }
  *row_wavelength_pairs = 0;
  Workspace* ws = t->last_ws;
  if (!t->exact || !t->exact->use_tc || !ws || !ws->x.work) return SPS_OK;
  cudaDeviceSynchronize();
  unsigned long long v = 0;
  sps_status st = sps_check_cuda(cudaMemcpy(&v, ws->x.work, sizeof(v), cudaMemcpyDeviceToHost), "sps_exact_last_work");
  *row_wavelength_pairs = (int64_t)v;
  return st;
}

extern "C" sps_status sps_exact_work_since(const sps_table* t, int64_t* row_wavelength_pairs, int64_t* calls) {
  if (!t || !row_wavelength_pairs || !calls) { sps_set_error("sps_exact_work_since: null argument"); return SPS_EINVAL; }
  *row_wavelength_pairs = 0; *calls = 0;
  Workspace* ws = t->last_ws;
  if (!t->exact || !t->exact->use_tc || !ws || !ws->x.work) return SPS_OK;
  cudaDeviceSynchronize();
  unsigned long long v = 0;
  sps_status st = sps_check_cuda(cudaMemcpy(&v, ws->x.work + 1, sizeof(v), cudaMemcpyDeviceToHost), "sps_exact_work_since");
  if (st == SPS_OK) st = sps_check_cuda(cudaMemset(ws->x.work + 1, 0, sizeof(v)), "sps_exact_work_since");
  *row_wavelength_pairs = (int64_t)v; *calls = ws->x.work_calls;
  ws->x.work_calls = 0;
  return st;
}
