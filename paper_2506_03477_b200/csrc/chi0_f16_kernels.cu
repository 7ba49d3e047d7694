// Stage (b), mixed mode (default): acc_j[I,J] += sum_p conj(z[p,I]) w_j(p) z[p,J] for one 128x128 tile and
// one frequency per CTA (Eq. 14; Alg. 1 lines 16-21) on the 5th-generation
// tensor cores with FP32-grade products built from FP16 pieces: tcgen05.mma kind::f16, FP32 accumulators in
// TMEM, FP64 accumulation across batches and k.
//
//   An FP32 value v (scaled by a power of two into the FP16 range) is carried as v = h + l with
//   h = fp16(v), l = fp16(v - h): 22 significant bits.  With A = w_j * (x_I, y_I) and B = (x_J, y_J):
//     a b ~= a_h b_h + a_l b_h + a_h b_l          (three exact FP16 products, the dropped a_l b_l is 2^-22)
//     Re += A_x B_x + A_y B_y,     Im += A_x B_y - A_y B_x      ("4M"; the minus is the a_negate bit)
//   = 12 MMAs of 128x128x16 per 16 band pairs, on the tensor pipe that runs at twice the TF32 rate (and
//   about half the energy per product): 2x the throughput of the 3xTF32 split at the same accuracy.
//
//   z tiles ("hl16" planes, kernels.h) are K-major FP16: one 128-byte swizzled row = h[32 pairs] | l[32
//   pairs], written to shared memory by TMA and read by the MMA as the B operand; the frequency-scaled
//   operand A is formed in registers and stored to TENSOR MEMORY (tcgen05.st).  The scaling itself runs in
//   packed FP16 arithmetic with an exact-residual FMA (no conversions): with w = w_h + w_l,
//     a_h = w_h (x) z_h,   a_l = fma(w_h, z_h, -a_h) + w_h z_l + w_l z_h        (a_h + a_l = w z to 2^-22).
//
//   The tensor core accumulates FP32 with truncation (bias ~ -4e-8 x MMA steps into one accumulator on
//   same-sign sums), so D is drained every WIN stages into FP32 register accumulators with round-to-nearest
//   adds; those go to the FP64 accumulators in HBM once per launch, rescaled by 1 / sigma_j (the 2^(-2S) of each
//   staged band batch is folded into that batch's weights).
//
//   FP8 = true (selected per flush on the device from the weights of the staged pairs, kernels.h MixedCtl): the two
//   correction products
//   a_l b_h + a_h b_l are 2^-11 of the main one and need ~3 significant bits, so each runs as ONE kind::f8f6f4
//   MMA of K = 32 on E5M2 operands (FP16's exponent range: no rescaling) into the same TMEM accumulators:
//   8 + 8 instead of 24 MMAs per 32 pairs.  B rows then come from the "hb8" workspace
//   (h[32] halves | e5m2(v)[32] | e5m2(v - h)[32]: the same 128 bytes, K offsets +64 B and +96 B).
//
// Roles (384 threads): warp 0 = TMA producer, warp 1 = MMA issuer (one thread) + TMEM allocator,
// warps 4-11 = scale + drain ("SA") warps: thread <-> tile row I; warps 4-7 own Re, 8-11 own Im.
#include <cuda_fp16.h>

#include "kernels.h"
#include "ptx.cuh"

namespace qsgw {

namespace {

constexpr int kThreadsH = 384;
constexpr int kPlaneTileH = 128 * 128;   // bytes of one 128-row x (32 h | 32 l) operand tile
constexpr int kBoxBytes = 64 * 128;      // one TMA box: 64 rows x 128 B

// Two shared-memory rings with their own producer threads: the B tiles (read by the MMAs, released by the MMA
// commit) and the A-source tiles + weight rows (read by the scaling warps, released as soon as they are in
// registers), so that the scaling warps' data runs ahead of the MMAs instead of waiting for a slot the tensor pipe
// still reads (ncu, round 2: 25 % of the scaling warps' time was the wait for the common ring).
struct HCfg {
  static constexpr int STAGES = 4;                               // B ring
  static constexpr int ASTAGES = 2;                              // A-source ring
  static constexpr int B_BYTES = 2 * kPlaneTileH;
  static constexpr int A_BYTES = 2 * kPlaneTileH;
  static constexpr int W_BYTES = kPairStage * 4;                 // w_h[32] | w_l[32] halves
  static constexpr int ASTAGE_BYTES = A_BYTES + 1024;            // w slot padded: tiles stay 1024-B aligned
  static constexpr int A_RING_OFF = STAGES * B_BYTES;
  static constexpr int BAR_OFF = A_RING_OFF + ASTAGES * ASTAGE_BYTES;
  static constexpr int TSLOT_COLS = 64;                          // h_x, h_y, l_x, l_y: 16 columns each
  static constexpr int TSLOTS = 4;
  static constexpr int SMEM_BYTES = BAR_OFF + 256 + 1024 /*align slack*/;
};

// global stage index of the i-th stage a launch runs (the list of live stages, or all of them)
__device__ __forceinline__ int stage_of(const Chi0F16Args& a, bool mapped, int i) { return mapped ? a.d_live[i] : i; }

// One 32-pair stage of the frequency-scaled operand: thread <-> tile row `row`, pair half h (16 pairs); reads the hl16 row of
// both planes and the weight row from the A-source stage at shared address sb, writes the TMEM slot (address incl. lane base).
template <bool FP8, int A_BYTES>
__device__ __forceinline__ void scale_stage_to_tmem(uint32_t sb, int row, int h, uint32_t slot) {
  const uint32_t sw = (uint32_t)(row & 7);
  const uint32_t src = sb + (uint32_t)row * 128u;
  const uint32_t swp = sb + A_BYTES + 32u * (uint32_t)h;                // this thread's 16 pairs
  const uint32_t tdst = slot + 8 * h;
  uint32_t wh[8], wl[8];
#pragma unroll
  for (int cc = 0; cc < 2; ++cc) {
    const uint4 t = ld_shared_u4(swp + 16 * cc), u4 = ld_shared_u4(swp + 64 + 16 * cc);
    wh[4 * cc] = t.x; wh[4 * cc + 1] = t.y; wh[4 * cc + 2] = t.z; wh[4 * cc + 3] = t.w;
    wl[4 * cc] = u4.x; wl[4 * cc + 1] = u4.y; wl[4 * cc + 2] = u4.z; wl[4 * cc + 3] = u4.w;
  }
#pragma unroll
  for (int xy = 0; xy < 2; ++xy) {
    uint32_t hv[8], lv[8], ah[8], al[8];
#pragma unroll
    for (int cc = 0; cc < 2; ++cc) {
      const uint4 th = ld_shared_u4(src + xy * kPlaneTileH + ((((uint32_t)(2 * h + cc)) ^ sw) << 4));
      const uint4 tl = ld_shared_u4(src + xy * kPlaneTileH + ((((uint32_t)(4 + 2 * h + cc)) ^ sw) << 4));
      hv[4 * cc] = th.x; hv[4 * cc + 1] = th.y; hv[4 * cc + 2] = th.z; hv[4 * cc + 3] = th.w;
      lv[4 * cc] = tl.x; lv[4 * cc + 1] = tl.y; lv[4 * cc + 2] = tl.z; lv[4 * cc + 3] = tl.w;
    }
#pragma unroll
    for (int e = 0; e < 8; ++e) {                  // pairs 2e, 2e+1 of this thread's 16
      const __half2 zh = *reinterpret_cast<const __half2*>(&hv[e]), zl = *reinterpret_cast<const __half2*>(&lv[e]);
      const __half2 w_h = *reinterpret_cast<const __half2*>(&wh[e]), w_l = *reinterpret_cast<const __half2*>(&wl[e]);
      const __half2 p = __hmul2(w_h, zh);
      __half2 r = __hfma2(w_h, zh, __hneg2(p));    // exact: the rounding error of p
      r = __hfma2(w_h, zl, r);
      r = __hfma2(w_l, zh, r);
      ah[e] = *reinterpret_cast<const uint32_t*>(&p);
      al[e] = *reinterpret_cast<const uint32_t*>(&r);
    }
    tmem_st8(tdst + 16 * xy, ah);
    if (FP8) {
      uint32_t a8[4], l8[4];
#pragma unroll
      for (int c = 0; c < 4; ++c) {
        a8[c] = cvt_e5m2x2_f16x2(ah[2 * c]) | (cvt_e5m2x2_f16x2(ah[2 * c + 1]) << 16);
        l8[c] = cvt_e5m2x2_f16x2(al[2 * c]) | (cvt_e5m2x2_f16x2(al[2 * c + 1]) << 16);
      }
      const uint32_t t8 = slot + 32 + 4 * h;
      tmem_st4(t8 + 8 * xy, a8);
      tmem_st4(t8 + 16 + 8 * xy, l8);
    } else {
      tmem_st8(tdst + 32 + 16 * xy, al);
    }
  }
}

// FP32 window sums of one tile row (in units 2^(2S) sigma_j) -> FP64 accumulators
__device__ __forceinline__ void writeback_row(const Chi0F16Args& a, const float (&racc)[128], int j, int2 tt, int row, int h) {
  const double sc = a.wscale[j];     // the batches' 2^(-2S) are folded into the weights (pair_weights_kernel)
  const long long plane = (long long)a.n_m_pad * a.n_m_pad;
  double* dst = (h ? a.acc_im : a.acc_re) + (long long)j * plane + (long long)(tt.x * kTileMx + row) * a.n_m_pad +
                tt.y * kTileMx;
  if (a.split > 1) {
#pragma unroll
    for (int c = 0; c < 128; ++c) atomicAdd(dst + c, sc * (double)racc[c]);
  } else {                           // exclusive owner of (tile, j)
#pragma unroll
    for (int c = 0; c < 64; ++c) {
      double2 v = *reinterpret_cast<double2*>(dst + 2 * c);
      v.x += sc * (double)racc[2 * c];
      v.y += sc * (double)racc[2 * c + 1];
      *reinterpret_cast<double2*>(dst + 2 * c) = v;
    }
  }
}

// FP8 = true: the two correction products run on kind::f8f6f4 (E5M2) -- 8 f16 + 8 fp8 MMAs per 32 pairs
// instead of 24 f16 MMAs; B rows come from the "hb8" workspace, the A source stays the full-precision hl16 rows.
template <bool FP8>
__global__ void __launch_bounds__(kThreadsH, 1) chi0_f16_kernel(const __grid_constant__ Chi0F16Args a) {
  using C = HCfg;
  extern __shared__ unsigned char smem_dyn[];
  const uint32_t raw = smem_u32(smem_dyn);
  const uint32_t base = (raw + 1023u) & ~1023u;
  unsigned char* sm = smem_dyn + (base - raw);
  uint64_t* bars = reinterpret_cast<uint64_t*>(sm + C::BAR_OFF);
  uint64_t* full = bars;                     // B ring
  uint64_t* empty = full + C::STAGES;
  uint64_t* s_full = empty + C::STAGES;      // A-source ring
  uint64_t* s_empty = s_full + C::ASTAGES;
  uint64_t* a_full = s_empty + C::ASTAGES;   // scaled operand in TMEM
  uint64_t* a_empty = a_full + C::TSLOTS;
  uint64_t* d_full = a_empty + C::TSLOTS;
  uint64_t* d_empty = d_full + 1;
  uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(d_empty + 1);

  if ((a.ctl->use_fp8 != 0) != FP8) return;     // the other variant of this flush runs (uniform over the grid)
  const int tid = threadIdx.x, warp = uniform_warp_idx(), lane = tid & 31;
  // blockIdx.x = ((tile * n_freq) + j) * split + chunk: the `split` CTAs of a (tile, j) share the staged pairs
  // (few-tile problems: fills the SMs; their partial sums meet in the FP64 accumulator by atomic adds)
  const int chunk = blockIdx.x % a.split, bid = blockIdx.x / a.split;
  const int j = a.j0 + bid % a.n_freq;
  const int4 tq = a.d_tiles[bid / a.n_freq];
  const int2 tt = make_int2(tq.x, tq.y);
  const int n_all = a.d_live ? *a.d_n_live : a.n_stages;                // stages to run (dead stages are skipped)
  const bool mapped = a.d_live && n_all != a.n_stages;                  // every stage live: no look-up
  int s_base = (int)((long long)n_all * chunk / a.split);               // first stage of this CTA
  int n_stages = (int)((long long)n_all * (chunk + 1) / a.split) - s_base;
  if (n_stages <= 0 && !a.d_ranges) return;
  const int win = a.win;
  if (a.d_ranges) {           // binned real-axis path: only the stages that cover the rows carrying weight in this bin
    const int2 r = a.d_ranges[j];
    s_base = r.x / kPairStage;
    n_stages = r.y > r.x ? (r.y + kPairStage - 1) / kPairStage - s_base : 0;
    if (n_stages <= 0) return;
  }

  if (tid == 0) {
    tma_prefetch_desc(&a.tmap);
    for (int s = 0; s < C::STAGES; ++s) {
      mbar_init(&full[s], 1);
      mbar_init(&empty[s], 1);         // the MMA commit
    }
    for (int s = 0; s < C::ASTAGES; ++s) {
      mbar_init(&s_full[s], 1);
      mbar_init(&s_empty[s], 8);       // 8 SA warps
    }
    for (int s = 0; s < C::TSLOTS; ++s) {
      mbar_init(&a_full[s], 8);
      mbar_init(&a_empty[s], 1);
    }
    mbar_init(d_full, 1);
    mbar_init(d_empty, 8);
    mbar_fence_init();
  }
  if (warp == 1) tmem_alloc(tmem_slot, 512);
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tbase = *tmem_slot;
  const uint32_t d_re = tbase, d_im = tbase + 128, a_ring = tbase + 256;

  if (warp < 4) {
    setmaxnreg_dec<56>();
    if (warp == 0) {
      // ------------------------------------------------------------------ TMA producer, B tiles
      int st = 0, u = 0;
      for (int s = 0; s < n_stages; ++s) {
        if (u > 0) mbar_wait(&empty[st], (u - 1) & 1);
        unsigned char* sb = sm + st * C::B_BYTES;
        if (elect_one()) {
          mbar_arrive_expect_tx(&full[st], C::B_BYTES);
#pragma unroll
          for (int i = 0; i < 4; ++i) {                  // box i: plane (x | y), row half
            const int plane = i >> 1, rh = i & 1;
            const CUtensorMap* tm = FP8 ? &a.tmap_b : &a.tmap;                 // hb8 rows are addressed in bytes
            tma_load_3d(sb + plane * kPlaneTileH + rh * kBoxBytes, tm, &full[st], stage_of(a, mapped, s_base + s) * (FP8 ? 128 : 64),
                        tt.y * kTileMx + rh * 64, plane);
          }
        }
        __syncwarp();
        if (++st == C::STAGES) { st = 0; ++u; }
      }
    } else if (warp == 2) {
      // ------------------------------------------------------------------ TMA producer, A-source tiles + weights
      const __half* wrow = a.wtab16 + (long long)j * a.kpad * 2;
      int st = 0, u = 0;
      for (int s = 0; s < n_stages; ++s) {
        if (u > 0) mbar_wait(&s_empty[st], (u - 1) & 1);
        unsigned char* sa = sm + C::A_RING_OFF + st * C::ASTAGE_BYTES;
        if (elect_one()) {
          mbar_arrive_expect_tx(&s_full[st], C::A_BYTES + C::W_BYTES);
#pragma unroll
          for (int i = 0; i < 4; ++i) {
            const int plane = i >> 1, rh = i & 1;
            tma_load_3d(sa + plane * kPlaneTileH + rh * kBoxBytes, &a.tmap, &s_full[st], stage_of(a, mapped, s_base + s) * 64,
                        tt.x * kTileMx + rh * 64, plane);
          }
          bulk_load_1d(sa + C::A_BYTES, wrow + (long long)stage_of(a, mapped, s_base + s) * 64, C::W_BYTES, &s_full[st]);
        }
        __syncwarp();
        if (++st == C::ASTAGES) { st = 0; ++u; }
      }
    } else if (warp == 1) {
      // ------------------------------------------------------------------ MMA issuer: the whole warp runs the loop
      // (uniform control flow and operands), one elected lane issues
      const uint32_t idesc = umma_idesc_f16(128, 128, 0), idesc_neg = umma_idesc_f16(128, 128, 1);
      const uint32_t idesc8 = umma_idesc_e5m2(128, 128, 0), idesc8_neg = umma_idesc_e5m2(128, 128, 1);
      int st = 0, u = 0, ts = 0, tu = 0, wpos = 0, widx = 0;     // ring positions / window position without divisions
      for (int s = 0; s < n_stages; ++s) {
        const bool win_first = wpos == 0;
        if (win_first && s > 0) mbar_wait(d_empty, (widx - 1) & 1);
        mbar_wait(&full[st], u & 1);
        mbar_wait(&a_full[ts], tu & 1);
        tc_fence_after();
        const uint32_t sb = base + st * C::B_BYTES;
        const uint64_t bx = umma_desc_k_sw128(sb), by = umma_desc_k_sw128(sb + kPlaneTileH);
        const uint32_t ab = a_ring + ts * C::TSLOT_COLS;
        const bool last_of_win = (wpos + 1 == win) || s == n_stages - 1;
        if (elect_one()) {
        if (FP8) {
#pragma unroll
          for (int g = 0; g < 2; ++g) {                     // main products: a_h b_h
            const uint32_t acc0 = (win_first && g == 0) ? 0u : 1u;
            const uint64_t kh = (uint64_t)(2 * g);
            const uint32_t ahx = ab + 8 * g, ahy = ab + 16 + 8 * g;
            umma_f16_ts(d_re, ahx, bx + kh, idesc, acc0);
            umma_f16_ts(d_im, ahx, by + kh, idesc, acc0);
            umma_f16_ts(d_re, ahy, by + kh, idesc, 1u);
            umma_f16_ts(d_im, ahy, bx + kh, idesc_neg, 1u);
          }
          // corrections a_l8 b_8 + a_8 b_l8: one K = 32 step; b_8 at byte 64, b_l8 at byte 96 of the row
          const uint32_t a8x = ab + 32, a8y = ab + 40, l8x = ab + 48, l8y = ab + 56;
          umma_f8_ts(d_re, l8x, bx + 4, idesc8, 1u);
          umma_f8_ts(d_im, l8x, by + 4, idesc8, 1u);
          umma_f8_ts(d_re, l8y, by + 4, idesc8, 1u);
          umma_f8_ts(d_im, l8y, bx + 4, idesc8_neg, 1u);
          umma_f8_ts(d_re, a8x, bx + 6, idesc8, 1u);
          umma_f8_ts(d_im, a8x, by + 6, idesc8, 1u);
          umma_f8_ts(d_re, a8y, by + 6, idesc8, 1u);
          umma_f8_ts(d_im, a8y, bx + 6, idesc8_neg, 1u);
        }
#pragma unroll
        for (int g = 0; g < (FP8 ? 0 : 2); ++g) {           // 16 pairs = one K step of kind::f16
          const uint32_t acc0 = (win_first && g == 0) ? 0u : 1u;
          const uint64_t kh = (uint64_t)(2 * g);            // 16 halves = 32 B along K inside the swizzle row
          const uint64_t kl = (uint64_t)(4 + 2 * g);        // the l half of the row starts at byte 64
          const uint32_t ahx = ab + 8 * g, ahy = ab + 16 + 8 * g, alx = ab + 32 + 8 * g, aly = ab + 48 + 8 * g;
          umma_f16_ts(d_re, ahx, bx + kh, idesc, acc0);
          umma_f16_ts(d_im, ahx, by + kh, idesc, acc0);
          umma_f16_ts(d_re, ahy, by + kh, idesc, 1u);
          umma_f16_ts(d_im, ahy, bx + kh, idesc_neg, 1u);
          umma_f16_ts(d_re, alx, bx + kh, idesc, 1u);
          umma_f16_ts(d_im, alx, by + kh, idesc, 1u);
          umma_f16_ts(d_re, aly, by + kh, idesc, 1u);
          umma_f16_ts(d_im, aly, bx + kh, idesc_neg, 1u);
          umma_f16_ts(d_re, ahx, bx + kl, idesc, 1u);
          umma_f16_ts(d_im, ahx, by + kl, idesc, 1u);
          umma_f16_ts(d_re, ahy, by + kl, idesc, 1u);
          umma_f16_ts(d_im, ahy, bx + kl, idesc_neg, 1u);
        }
        umma_commit(&empty[st]);
        umma_commit(&a_empty[ts]);
        if (last_of_win) umma_commit(d_full);
        }
        __syncwarp();
        if (++wpos == win) { wpos = 0; ++widx; }
        if (++st == C::STAGES) { st = 0; ++u; }
        if (++ts == C::TSLOTS) { ts = 0; ++tu; }
      }
    }
  } else {
    // -------------------------------------------------------------------- scale + drain warps
    setmaxnreg_inc<224>();
    const int q = warp & 3, h = (warp - 4) >> 2;       // TMEM lane quarter; pair half / Re-Im owner
    const int row = 32 * q + lane;
    const uint32_t lane_base = (uint32_t)(32 * q) << 16;
    float racc[128];
#pragma unroll
    for (int i = 0; i < 128; ++i) racc[i] = 0.f;

    auto drain = [&](int widx) {
      mbar_wait(d_full, widx & 1);
      tc_fence_after();
      const uint32_t dcol = (h ? d_im : d_re) + lane_base;
#pragma unroll
      for (int c = 0; c < 4; ++c) {
        uint32_t v[32];
        tmem_ld32(dcol + 32 * c, v);
        tmem_wait_ld();
#pragma unroll
        for (int i = 0; i < 32; ++i) racc[32 * c + i] += __uint_as_float(v[i]);
      }
      tc_fence_before();
      __syncwarp();
      if (lane == 0) mbar_arrive(d_empty);
    };

    int st = 0, u = 0, ts = 0, tu = 0, wpos = 0, widx = 0;
    for (int s = 0; s < n_stages; ++s) {
      mbar_wait(&s_full[st], u & 1);
      if (tu > 0) mbar_wait(&a_empty[ts], (tu - 1) & 1);
      tc_fence_after();
      scale_stage_to_tmem<FP8, C::A_BYTES>(base + C::A_RING_OFF + st * C::ASTAGE_BYTES, row, h,
                                           a_ring + ts * C::TSLOT_COLS + lane_base);
      tmem_wait_st();
      tc_fence_before();
      __syncwarp();
      if (lane == 0) {
        mbar_arrive(&a_full[ts]);
        mbar_arrive(&s_empty[st]);
      }
      if (s >= 1 && wpos == 0) drain(widx - 1);            // stage s-1 closed a window
      if (++wpos == win) { wpos = 0; ++widx; }
      if (++st == C::ASTAGES) { st = 0; ++u; }
      if (++ts == C::TSLOTS) { ts = 0; ++tu; }
    }
    drain(wpos == 0 ? widx - 1 : widx);

    writeback_row(a, racc, j, tt, row, h);
  }
  tc_fence_before();
  __syncthreads();
  if (warp == 1) tmem_dealloc(tbase, 512);
}

// ---- CTA-pair variant (cluster of 2, tcgen05 cta_group::2) ------------------------------------------------------------
// The two CTAs of a pair work on the SAME 128x128 tile at two consecutive frequencies.  z_J (the B operand) does not
// depend on the frequency, so the pair shares it: each CTA fetches only its 64 of the 128 J rows (16 KB instead of
// 32 KB per 32-pair stage) and one thread of the rank-0 CTA issues MMAs of M = 256: rows 0..127 = the rank-0 CTA's
// scaled operand (its frequency) from ITS tensor memory into ITS accumulators, rows 128..255 the same for rank 1,
// B = the two 64-row halves in the two shared memories.  Per SM and stage this takes 16 KB out of the L2 -> SM
// traffic and 32 KB out of the MMAs' shared-memory reads (64 rows per MMA instead of 128).  Everything else is as
// in chi0_f16_kernel; cross-CTA signalling: the B "full" barrier (both halves' TMA bytes), the "A slot written" and
// "window drained" barriers live in the rank-0 CTA (remote arrives from rank 1), every MMA-completion signal is a
// multicast commit to the same barrier in both CTAs.  An odd frequency count leaves rank 1 of the last pair as a
// passenger: it works on the last frequency again and skips the write-back.
struct PCfg {
  static constexpr int STAGES = 6;                               // B ring (this CTA's half of the J rows)
  static constexpr int ASTAGES = 3;                              // A-source ring
  static constexpr int B_BYTES = kPlaneTileH;                    // 2 planes x 64 rows x 128 B
  static constexpr int A_BYTES = 2 * kPlaneTileH;
  static constexpr int W_BYTES = kPairStage * 4;
  static constexpr int ASTAGE_BYTES = A_BYTES + 1024;
  static constexpr int A_RING_OFF = STAGES * B_BYTES;
  static constexpr int BAR_OFF = A_RING_OFF + ASTAGES * ASTAGE_BYTES;
  static constexpr int TSLOT_COLS = 64;
  static constexpr int TSLOTS = 4;
  static constexpr int SMEM_BYTES = BAR_OFF + 256 + 1024 /*align slack*/;
};

template <bool FP8>
__global__ void __cluster_dims__(2, 1, 1) __launch_bounds__(kThreadsH, 1)
    chi0_f16_pair_kernel(const __grid_constant__ Chi0F16Args a) {
  using C = PCfg;
  extern __shared__ unsigned char smem_dyn[];
  const uint32_t raw = smem_u32(smem_dyn);
  const uint32_t base = (raw + 1023u) & ~1023u;
  unsigned char* sm = smem_dyn + (base - raw);
  uint64_t* bars = reinterpret_cast<uint64_t*>(sm + C::BAR_OFF);
  uint64_t* full = bars;                     // B ring: both halves have landed            (used in rank 0)
  uint64_t* empty = full + C::STAGES;        //         the MMAs have read the slot        (multicast commit)
  uint64_t* s_full = empty + C::STAGES;      // A-source ring (per CTA)
  uint64_t* s_empty = s_full + C::ASTAGES;
  uint64_t* a_full = s_empty + C::ASTAGES;   // scaled operand in TMEM, both CTAs          (used in rank 0, 16 arrivals)
  uint64_t* a_empty = a_full + C::TSLOTS;    //                                            (multicast commit)
  uint64_t* d_full = a_empty + C::TSLOTS;    // window complete                            (multicast commit)
  uint64_t* d_empty = d_full + 1;            // window drained by both CTAs                (used in rank 0, 16 arrivals)
  uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(d_empty + 1);

  if ((a.ctl->use_fp8 != 0) != FP8) return;     // the other variant of this flush runs (uniform over the grid)
  const int tid = threadIdx.x, warp = uniform_warp_idx(), lane = tid & 31;
  const uint32_t rank = cluster_ctarank();
  // cluster = ((tile * ceil(n_freq / 2)) + m) * split + chunk; this CTA's frequency = 2 m + rank
  const int nf2 = (a.n_freq + 1) >> 1;
  const int cid = blockIdx.x >> 1;
  const int chunk = cid % a.split, bid = cid / a.split;
  int jl = 2 * (bid % nf2) + (int)rank;
  const bool passenger = jl >= a.n_freq;
  if (passenger) jl = a.n_freq - 1;
  const int j = a.j0 + jl;
  const int4 tq = a.d_tiles[bid / nf2];
  const int2 tt = make_int2(tq.x, tq.y);
  const int n_all = a.d_live ? *a.d_n_live : a.n_stages;                      // stages to run (dead stages are skipped)
  const bool mapped = a.d_live && n_all != a.n_stages;                        // every stage live: no look-up
  const int s_base = (int)((long long)n_all * chunk / a.split);               // first stage of this pair
  const int n_stages = (int)((long long)n_all * (chunk + 1) / a.split) - s_base;
  if (n_stages <= 0) return;                                                  // both CTAs of the pair
  const int win = a.win;

  if (tid == 0) {
    tma_prefetch_desc(&a.tmap);
    for (int s = 0; s < C::STAGES; ++s) {
      mbar_init(&full[s], 1);
      mbar_init(&empty[s], 1);
    }
    for (int s = 0; s < C::ASTAGES; ++s) {
      mbar_init(&s_full[s], 1);
      mbar_init(&s_empty[s], 8);
    }
    for (int s = 0; s < C::TSLOTS; ++s) {
      mbar_init(&a_full[s], 16);       // 8 SA warps of each CTA
      mbar_init(&a_empty[s], 1);
    }
    mbar_init(d_full, 1);
    mbar_init(d_empty, 16);
    mbar_fence_init();
  }
  if (warp == 1) tmem_alloc_pair(tmem_slot, 512);
  tc_fence_before();
  cluster_sync_all();
  tc_fence_after();
  const uint32_t tbase = *tmem_slot;
  const uint32_t d_re = tbase, d_im = tbase + 128, a_ring = tbase + 256;

  if (warp < 4) {
    setmaxnreg_dec<56>();
    if (warp == 0) {
      // ------------------------------------------------------------------ TMA producer, this CTA's half of the B tiles
      const CUtensorMap* tm = FP8 ? &a.tmap_b : &a.tmap;                     // hb8 rows are addressed in bytes
      int st = 0, u = 0;
      for (int s = 0; s < n_stages; ++s) {
        if (u > 0) mbar_wait(&empty[st], (u - 1) & 1);
        unsigned char* sb = sm + st * C::B_BYTES;
        const uint32_t bar = mapa_shared(smem_u32(&full[st]), 0);
        if (elect_one()) {
          if (rank == 0) mbar_arrive_expect_tx(&full[st], 2 * C::B_BYTES);   // both halves
#pragma unroll
          for (int plane = 0; plane < 2; ++plane)
            tma_load_3d_pair(sb + plane * kBoxBytes, tm, bar, stage_of(a, mapped, s_base + s) * (FP8 ? 128 : 64),
                             tt.y * kTileMx + (int)rank * 64, plane);
        }
        __syncwarp();
        if (++st == C::STAGES) { st = 0; ++u; }
      }
    } else if (warp == 2) {
      // ------------------------------------------------------------------ TMA producer, A-source tiles + weights
      const __half* wrow = a.wtab16 + (long long)j * a.kpad * 2;
      int st = 0, u = 0;
      for (int s = 0; s < n_stages; ++s) {
        if (u > 0) mbar_wait(&s_empty[st], (u - 1) & 1);
        unsigned char* sa = sm + C::A_RING_OFF + st * C::ASTAGE_BYTES;
        if (elect_one()) {
          mbar_arrive_expect_tx(&s_full[st], C::A_BYTES + C::W_BYTES);
#pragma unroll
          for (int i = 0; i < 4; ++i) {
            const int plane = i >> 1, rh = i & 1;
            tma_load_3d(sa + plane * kPlaneTileH + rh * kBoxBytes, &a.tmap, &s_full[st], stage_of(a, mapped, s_base + s) * 64,
                        tt.x * kTileMx + rh * 64, plane);
          }
          bulk_load_1d(sa + C::A_BYTES, wrow + (long long)stage_of(a, mapped, s_base + s) * 64, C::W_BYTES, &s_full[st]);
        }
        __syncwarp();
        if (++st == C::ASTAGES) { st = 0; ++u; }
      }
    } else if (warp == 1 && rank == 0) {
      // ------------------------------------------------------------------ MMA issuer of the pair: the whole warp
      // runs the loop (uniform control flow and operands), one elected lane issues
      const uint32_t idesc = umma_idesc_f16(256, 128, 0), idesc_neg = umma_idesc_f16(256, 128, 1);
      const uint32_t idesc8 = umma_idesc_e5m2(256, 128, 0), idesc8_neg = umma_idesc_e5m2(256, 128, 1);
      int st = 0, u = 0, ts = 0, tu = 0, wpos = 0, widx = 0;
      for (int s = 0; s < n_stages; ++s) {
        const bool win_first = wpos == 0;
        if (win_first && s > 0) mbar_wait_cluster(d_empty, (widx - 1) & 1);
        mbar_wait_cluster(&full[st], u & 1);
        mbar_wait_cluster(&a_full[ts], tu & 1);
        tc_fence_after();
        const uint32_t sb = base + st * C::B_BYTES;
        const uint64_t bx = umma_desc_k_sw128(sb), by = umma_desc_k_sw128(sb + kBoxBytes);
        const uint32_t ab = a_ring + ts * C::TSLOT_COLS;
        const bool last_of_win = (wpos + 1 == win) || s == n_stages - 1;
        if (elect_one()) {
        if (FP8) {
#pragma unroll
          for (int g = 0; g < 2; ++g) {                     // main products: a_h b_h
            const uint32_t acc0 = (win_first && g == 0) ? 0u : 1u;
            const uint64_t kh = (uint64_t)(2 * g);
            const uint32_t ahx = ab + 8 * g, ahy = ab + 16 + 8 * g;
            umma_f16_ts_pair(d_re, ahx, bx + kh, idesc, acc0);
            umma_f16_ts_pair(d_im, ahx, by + kh, idesc, acc0);
            umma_f16_ts_pair(d_re, ahy, by + kh, idesc, 1u);
            umma_f16_ts_pair(d_im, ahy, bx + kh, idesc_neg, 1u);
          }
          const uint32_t a8x = ab + 32, a8y = ab + 40, l8x = ab + 48, l8y = ab + 56;
          umma_f8_ts_pair(d_re, l8x, bx + 4, idesc8, 1u);
          umma_f8_ts_pair(d_im, l8x, by + 4, idesc8, 1u);
          umma_f8_ts_pair(d_re, l8y, by + 4, idesc8, 1u);
          umma_f8_ts_pair(d_im, l8y, bx + 4, idesc8_neg, 1u);
          umma_f8_ts_pair(d_re, a8x, bx + 6, idesc8, 1u);
          umma_f8_ts_pair(d_im, a8x, by + 6, idesc8, 1u);
          umma_f8_ts_pair(d_re, a8y, by + 6, idesc8, 1u);
          umma_f8_ts_pair(d_im, a8y, bx + 6, idesc8_neg, 1u);
        }
#pragma unroll
        for (int g = 0; g < (FP8 ? 0 : 2); ++g) {
          const uint32_t acc0 = (win_first && g == 0) ? 0u : 1u;
          const uint64_t kh = (uint64_t)(2 * g);
          const uint64_t kl = (uint64_t)(4 + 2 * g);
          const uint32_t ahx = ab + 8 * g, ahy = ab + 16 + 8 * g, alx = ab + 32 + 8 * g, aly = ab + 48 + 8 * g;
          umma_f16_ts_pair(d_re, ahx, bx + kh, idesc, acc0);
          umma_f16_ts_pair(d_im, ahx, by + kh, idesc, acc0);
          umma_f16_ts_pair(d_re, ahy, by + kh, idesc, 1u);
          umma_f16_ts_pair(d_im, ahy, bx + kh, idesc_neg, 1u);
          umma_f16_ts_pair(d_re, alx, bx + kh, idesc, 1u);
          umma_f16_ts_pair(d_im, alx, by + kh, idesc, 1u);
          umma_f16_ts_pair(d_re, aly, by + kh, idesc, 1u);
          umma_f16_ts_pair(d_im, aly, bx + kh, idesc_neg, 1u);
          umma_f16_ts_pair(d_re, ahx, bx + kl, idesc, 1u);
          umma_f16_ts_pair(d_im, ahx, by + kl, idesc, 1u);
          umma_f16_ts_pair(d_re, ahy, by + kl, idesc, 1u);
          umma_f16_ts_pair(d_im, ahy, bx + kl, idesc_neg, 1u);
        }
        umma_commit_pair(&empty[st]);
        umma_commit_pair(&a_empty[ts]);
        if (last_of_win) umma_commit_pair(d_full);
        }
        __syncwarp();
        if (++wpos == win) { wpos = 0; ++widx; }
        if (++st == C::STAGES) { st = 0; ++u; }
        if (++ts == C::TSLOTS) { ts = 0; ++tu; }
      }
    }
  } else {
    // -------------------------------------------------------------------- scale + drain warps (both CTAs)
    setmaxnreg_inc<224>();
    const int q = warp & 3, h = (warp - 4) >> 2;
    const int row = 32 * q + lane;
    const uint32_t lane_base = (uint32_t)(32 * q) << 16;
    const uint32_t a_full0 = mapa_shared(smem_u32(a_full), 0), d_empty0 = mapa_shared(smem_u32(d_empty), 0);
    float racc[128];
#pragma unroll
    for (int i = 0; i < 128; ++i) racc[i] = 0.f;

    auto drain = [&](int widx) {
      mbar_wait(d_full, widx & 1);
      tc_fence_after();
      const uint32_t dcol = (h ? d_im : d_re) + lane_base;
#pragma unroll
      for (int c = 0; c < 4; ++c) {
        uint32_t v[32];
        tmem_ld32(dcol + 32 * c, v);
        tmem_wait_ld();
#pragma unroll
        for (int i = 0; i < 32; ++i) racc[32 * c + i] += __uint_as_float(v[i]);
      }
      tc_fence_before();
      __syncwarp();
      if (lane == 0) mbar_arrive_cluster(d_empty0);
    };

    int st = 0, u = 0, ts = 0, tu = 0, wpos = 0, widx = 0;
    for (int s = 0; s < n_stages; ++s) {
      mbar_wait(&s_full[st], u & 1);
      if (tu > 0) mbar_wait(&a_empty[ts], (tu - 1) & 1);
      tc_fence_after();
      scale_stage_to_tmem<FP8, C::A_BYTES>(base + C::A_RING_OFF + st * C::ASTAGE_BYTES, row, h,
                                           a_ring + ts * C::TSLOT_COLS + lane_base);
      tmem_wait_st();
      tc_fence_before();
      __syncwarp();
      if (lane == 0) {
        mbar_arrive_cluster(a_full0 + 8u * (uint32_t)ts);
        mbar_arrive(&s_empty[st]);
      }
      if (s >= 1 && wpos == 0) drain(widx - 1);
      if (++wpos == win) { wpos = 0; ++widx; }
      if (++st == C::ASTAGES) { st = 0; ++u; }
      if (++ts == C::TSLOTS) { ts = 0; ++tu; }
    }
    drain(wpos == 0 ? widx - 1 : widx);

    if (!passenger) writeback_row(a, racc, j, tt, row, h);
  }
  tc_fence_before();
  cluster_sync_all();        // no CTA leaves while its partner's MMAs, commits or arrives may still touch it
  if (warp == 1) tmem_dealloc_pair(tbase, 512);
}

}  // namespace

cudaError_t chi0_f16_configure() {
  cudaError_t e = cudaFuncSetAttribute(chi0_f16_pair_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, PCfg::SMEM_BYTES);
  if (e != cudaSuccess) return e;
  e = cudaFuncSetAttribute(chi0_f16_pair_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, PCfg::SMEM_BYTES);
  if (e != cudaSuccess) return e;
  e = cudaFuncSetAttribute(chi0_f16_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, HCfg::SMEM_BYTES);
  if (e != cudaSuccess) return e;
  return cudaFuncSetAttribute(chi0_f16_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, HCfg::SMEM_BYTES);
}

cudaError_t launch_chi0_f16(const Chi0F16Args& a_in, cudaStream_t s) {
  if (a_in.n_stages <= 0 || a_in.n_tiles <= 0) return cudaSuccess;
  Chi0F16Args a = a_in;
  // Few (tile, frequency) work items: split the staged pairs over 2..4 CTAs each, choosing the split that
  // minimises rounds(CTAs / SMs) / split; every CTA keeps >= 32 stages.
  a.split = 1;
  if (!a.d_ranges) {
    const int n_sm = a.n_sm;
    const long long items = (long long)a.n_tiles * a.n_freq;
    double best = (double)((items + n_sm - 1) / n_sm);
    for (int sp = 2; sp <= 4; ++sp) {
      if (a.n_stages < 32 * sp || items * sp > 8LL * n_sm) break;
      const double cost = (double)((items * sp + n_sm - 1) / n_sm) / sp;
      if (cost < 0.95 * best) { best = cost; a.split = sp; }
    }
  }
  if (a.pair && !a.d_ranges) {       // CTA pairs: two consecutive frequencies of a tile share the B tiles
    const unsigned grid2 = (unsigned)(a.n_tiles * ((a.n_freq + 1) / 2) * a.split) * 2u;
    chi0_f16_pair_kernel<true><<<dim3(grid2), kThreadsH, PCfg::SMEM_BYTES, s>>>(a);
    cudaError_t e2 = cudaGetLastError();
    if (e2 != cudaSuccess) return e2;
    chi0_f16_pair_kernel<false><<<dim3(grid2), kThreadsH, PCfg::SMEM_BYTES, s>>>(a);
    return cudaGetLastError();
  }
  const unsigned grid = (unsigned)(a.n_tiles * a.n_freq * a.split);
  chi0_f16_kernel<true><<<dim3(grid), kThreadsH, HCfg::SMEM_BYTES, s>>>(a);
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return e;
  chi0_f16_kernel<false><<<dim3(grid), kThreadsH, HCfg::SMEM_BYTES, s>>>(a);
  return cudaGetLastError();
}

}  // namespace qsgw
