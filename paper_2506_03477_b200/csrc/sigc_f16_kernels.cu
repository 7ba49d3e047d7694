// Imaginary-axis correlation self-energy, mixed mode (Eq. 22; Alg. 2 lines 15-25,
// PAPER.md:443-462): the frequency loop  ZW^c[p, nu] = sum_i w_i(p) sum_mu z[p, mu] W^c_i[mu, nu]  on the 5th-generation
// tensor cores with FP32-grade products built from FP16 pieces (the paper runs this GEMM in TF32: "GEMM-dominated kernel
// (imaginary-axis I^c) ~ 4x MP over DP").
//
//   Both operands are carried as v = h + l (h = fp16(v 2^S), l = fp16(v 2^S - h): 22 significant bits) in "hl16" rows
//   (kernels.h): per matrix row and 32 contraction indices mu one 128-byte row h[32] | l[32], K-major, so that TMA boxes
//   with the 128-byte swizzle are UMMA operand tiles.  a b ~= a_h b_h + a_l b_h + a_h b_l: 3 x 4 real MMAs
//   (kind::f16, 128x128x16) per 16 mu for the complex product  Re = x u - y v,  Im = x v + y u  (a_negate bit).
//   A = z rows (pairs p), copied from shared memory to TENSOR MEMORY by the staging warps (tcgen05.st; the MMA reads A
//   from TMEM and only B from shared memory: half the shared-memory operand traffic of an SS MMA);
//   B = (W^c_i)^T rows (nu), K = mu.
//   The quadrature weight of Alg. 2 line 18 depends on the ROW p and the frequency i only, so it is not applied to the
//   operand at all: D = z W_i accumulates in TMEM over windows of 16 stages inside one frequency (the tensor core's FP32
//   accumulation truncates: short windows keep its error below the operand split's), and the drain warps add
//   w_i(p) 2^(-S_z - S_W,i) D into FP32 registers (thread <-> row p) with round-to-nearest FMAs.
//   One CTA = one 128 x 128 tile of ZW^c, all frequencies; output complex128 (the closing contraction with z stays FP64).
//
// Roles (384 threads) as in chi0_f16_kernel: warp 0 = TMA producer of the B tiles, warp 2 = TMA producer of the A-source
// tiles, warp 1 = MMA issuer + TMEM allocator, warps 4-11 = staging + drain warps (warps 4-7 own Re, 8-11 own Im).
#include <cuda_fp16.h>
#include <cuda_fp8.h>

#include "kernels.h"
#include "ptx.cuh"

namespace qsgw {

namespace {

constexpr int kThreadsS = 384;
constexpr int kTileS = 128 * 128;        // bytes of one 128-row x (32 h | 32 l) operand tile
constexpr int kBoxS = 64 * 128;
constexpr int kSigcWin = 16;             // stages per TMEM drain window (the tensor core's FP32 accumulation truncates)

struct SCfg {
  static constexpr int STAGES = 4;       // B ring
  static constexpr int ASTAGES = 2;      // A-source ring
  static constexpr int B_BYTES = 2 * kTileS;
  static constexpr int A_BYTES = 2 * kTileS;
  static constexpr int A_RING_OFF = STAGES * B_BYTES;
  static constexpr int BAR_OFF = A_RING_OFF + ASTAGES * A_BYTES;
  static constexpr int TSLOT_COLS = 64;  // x_h, y_h, x_l, y_l: 16 columns each
  static constexpr int TSLOTS = 4;
  static constexpr int SMEM_BYTES = BAR_OFF + 256 + 1024;
};

struct SigcF16Args {
  CUtensorMap tmap_z;    // 3-D FLOAT16 {64 * kst, pairs_pad, 2}: z hl16 rows, box {64, 64, 1}
  CUtensorMap tmap_w;    // 3-D FLOAT16 {64 * kst, n_m_pad * n_freq, 2}: (W^c_i)^T hl16 rows, frequency-major
  CUtensorMap tmap_w8;   // FP8 variant: 3-D UINT8 {128 * kst, n_m_pad * n_freq, 2}: (W^c_i)^T hb8 rows h[32] | e5m2(v)[32] | e5m2(v - h)[32]
  const double* w;       // quadrature weights [n_freq][ld_w]
  long long ld_w;
  const float* zmax;     // max |Re z|, |Im z|
  const float* wmax;     // [n_freq] max |Re W_i|, |Im W_i|
  double2* zw;           // out: complex128 [pairs][n_m]
  int pairs, n_m, n_m_pad, n_freq, kst;   // kst = stages of 32 mu per frequency
  int n_tiles_n;
};

// FP8 = true: the two correction products z_l W_h + z_h W_l run as one kind::f8f6f4 (E5M2) MMA of K = 32 each (as in
// chi0_f16_kernel<fp8>): 8 + 8 instead of 24 MMAs per 32 mu; B rows from the hb8 copy of (W^c_i)^T.
template <bool FP8>
__global__ void __launch_bounds__(kThreadsS, 1) sigc_f16_kernel(const __grid_constant__ SigcF16Args a) {
  using C = SCfg;
  extern __shared__ unsigned char smem_dyn[];
  const uint32_t raw = smem_u32(smem_dyn);
  const uint32_t base = (raw + 1023u) & ~1023u;
  unsigned char* sm = smem_dyn + (base - raw);
  uint64_t* bars = reinterpret_cast<uint64_t*>(sm + C::BAR_OFF);
  uint64_t* full = bars;
  uint64_t* empty = full + C::STAGES;
  uint64_t* s_full = empty + C::STAGES;
  uint64_t* s_empty = s_full + C::ASTAGES;
  uint64_t* a_full = s_empty + C::ASTAGES;
  uint64_t* a_empty = a_full + C::TSLOTS;
  uint64_t* d_full = a_empty + C::TSLOTS;
  uint64_t* d_empty = d_full + 1;
  uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(d_empty + 1);

  const int tid = threadIdx.x, warp = uniform_warp_idx(), lane = tid & 31;
  const int tn = blockIdx.x % a.n_tiles_n, tp = blockIdx.x / a.n_tiles_n;     // tile column (nu), tile row (pairs)
  const int kst = a.kst, n_stages = a.n_freq * kst;

  if (tid == 0) {
    tma_prefetch_desc(&a.tmap_z);
    tma_prefetch_desc(&a.tmap_w);
    for (int s = 0; s < C::STAGES; ++s) { mbar_init(&full[s], 1); mbar_init(&empty[s], 1); }
    for (int s = 0; s < C::ASTAGES; ++s) { mbar_init(&s_full[s], 1); mbar_init(&s_empty[s], 8); }
    for (int s = 0; s < C::TSLOTS; ++s) { mbar_init(&a_full[s], 8); mbar_init(&a_empty[s], 1); }
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
    // warps 0-2: the whole warp runs its loop (uniform control flow and operands), one elected lane issues
    if (warp == 0) {
      // ------------------------------------------------------------------ B tiles: (W_i)^T rows of this tile column
      int st = 0, u = 0;
      for (int s = 0; s < n_stages; ++s) {
        const int i = s / kst, ks = s - i * kst;
        if (u > 0) mbar_wait(&empty[st], (u - 1) & 1);
        unsigned char* sb = sm + st * C::B_BYTES;
        if (elect_one()) {
          mbar_arrive_expect_tx(&full[st], C::B_BYTES);
#pragma unroll
          for (int b = 0; b < 4; ++b) {
            const int plane = b >> 1, rh = b & 1;
            tma_load_3d(sb + plane * kTileS + rh * kBoxS, FP8 ? &a.tmap_w8 : &a.tmap_w, &full[st], ks * (FP8 ? 128 : 64),
                        i * a.n_m_pad + tn * 128 + rh * 64, plane);
          }
        }
        __syncwarp();
        if (++st == C::STAGES) { st = 0; ++u; }
      }
    } else if (warp == 2) {
      // ------------------------------------------------------------------ A-source tiles: z rows of this tile row
      int st = 0, u = 0;
      for (int s = 0; s < n_stages; ++s) {
        const int ks = s % kst;
        if (u > 0) mbar_wait(&s_empty[st], (u - 1) & 1);
        unsigned char* sa = sm + C::A_RING_OFF + st * C::A_BYTES;
        if (elect_one()) {
          mbar_arrive_expect_tx(&s_full[st], C::A_BYTES);
#pragma unroll
          for (int b = 0; b < 4; ++b) {
            const int plane = b >> 1, rh = b & 1;
            tma_load_3d(sa + plane * kTileS + rh * kBoxS, &a.tmap_z, &s_full[st], ks * 64, tp * 128 + rh * 64, plane);
          }
        }
        __syncwarp();
        if (++st == C::ASTAGES) { st = 0; ++u; }
      }
    } else if (warp == 1) {
      // ------------------------------------------------------------------ MMA issuer
      const uint32_t idesc = umma_idesc_f16(128, 128, 0), idesc_neg = umma_idesc_f16(128, 128, 1);
      int st = 0, u = 0, ts = 0, tu = 0, kpos = 0, wpos = 0, widx = 0;
      for (int s = 0; s < n_stages; ++s) {
        const bool first = wpos == 0;                       // first stage of a drain window: D restarts
        if (first && s > 0) mbar_wait(d_empty, (widx - 1) & 1);
        mbar_wait(&full[st], u & 1);
        mbar_wait(&a_full[ts], tu & 1);
        tc_fence_after();
        const uint32_t sb = base + st * C::B_BYTES;
        const uint64_t bu = umma_desc_k_sw128(sb), bv = umma_desc_k_sw128(sb + kTileS);
        const uint32_t ab = a_ring + ts * C::TSLOT_COLS;
        ++wpos;
        if (++kpos == kst) kpos = 0;
        const bool win_last = wpos == kSigcWin || kpos == 0;    // a window ends with its frequency
        if (elect_one()) {
        if (FP8) {
          const uint32_t idesc8 = umma_idesc_e5m2(128, 128, 0), idesc8_neg = umma_idesc_e5m2(128, 128, 1);
#pragma unroll
          for (int g = 0; g < 2; ++g) {                     // main products (h h)
            const uint32_t acc0 = (first && g == 0) ? 0u : 1u;
            const uint64_t kh = (uint64_t)(2 * g);
            const uint32_t xh = ab + 8 * g, yh = ab + 16 + 8 * g;
            umma_f16_ts(d_re, xh, bu + kh, idesc, acc0);
            umma_f16_ts(d_im, xh, bv + kh, idesc, acc0);
            umma_f16_ts(d_re, yh, bv + kh, idesc_neg, 1u);
            umma_f16_ts(d_im, yh, bu + kh, idesc, 1u);
          }
          // corrections z_l8 W_8 + z_8 W_l8: one K = 32 step each; W_8 at byte 64, W_l8 at byte 96 of the row
          const uint32_t x8 = ab + 32, y8 = ab + 40, xl8 = ab + 48, yl8 = ab + 56;
          umma_f8_ts(d_re, xl8, bu + 4, idesc8, 1u);
          umma_f8_ts(d_im, xl8, bv + 4, idesc8, 1u);
          umma_f8_ts(d_re, yl8, bv + 4, idesc8_neg, 1u);
          umma_f8_ts(d_im, yl8, bu + 4, idesc8, 1u);
          umma_f8_ts(d_re, x8, bu + 6, idesc8, 1u);
          umma_f8_ts(d_im, x8, bv + 6, idesc8, 1u);
          umma_f8_ts(d_re, y8, bv + 6, idesc8_neg, 1u);
          umma_f8_ts(d_im, y8, bu + 6, idesc8, 1u);
        }
#pragma unroll
        for (int g = 0; g < (FP8 ? 0 : 2); ++g) {           // 16 mu = one K step
          const uint32_t acc0 = (first && g == 0) ? 0u : 1u;
          const uint64_t kh = (uint64_t)(2 * g), kl = (uint64_t)(4 + 2 * g);
          const uint32_t xh = ab + 8 * g, yh = ab + 16 + 8 * g, xl = ab + 32 + 8 * g, yl = ab + 48 + 8 * g;
          umma_f16_ts(d_re, xh, bu + kh, idesc, acc0);      // Re += x u - y v,  Im += x v + y u   (h h)
          umma_f16_ts(d_im, xh, bv + kh, idesc, acc0);
          umma_f16_ts(d_re, yh, bv + kh, idesc_neg, 1u);
          umma_f16_ts(d_im, yh, bu + kh, idesc, 1u);
          umma_f16_ts(d_re, xl, bu + kh, idesc, 1u);        // (l h)
          umma_f16_ts(d_im, xl, bv + kh, idesc, 1u);
          umma_f16_ts(d_re, yl, bv + kh, idesc_neg, 1u);
          umma_f16_ts(d_im, yl, bu + kh, idesc, 1u);
          umma_f16_ts(d_re, xh, bu + kl, idesc, 1u);        // (h l)
          umma_f16_ts(d_im, xh, bv + kl, idesc, 1u);
          umma_f16_ts(d_re, yh, bv + kl, idesc_neg, 1u);
          umma_f16_ts(d_im, yh, bu + kl, idesc, 1u);
        }
        umma_commit(&empty[st]);
        umma_commit(&a_empty[ts]);
        if (win_last) umma_commit(d_full);
        }
        __syncwarp();
        if (win_last) { wpos = 0; ++widx; }
        if (++st == C::STAGES) { st = 0; ++u; }
        if (++ts == C::TSLOTS) { ts = 0; ++tu; }
      }
    }
  } else {
    // -------------------------------------------------------------------- staging + drain warps
    setmaxnreg_inc<224>();
    const int q = warp & 3, h = (warp - 4) >> 2;       // TMEM lane quarter; mu half of the stage / Re-Im owner
    const int row = 32 * q + lane;
    const uint32_t lane_base = (uint32_t)(32 * q) << 16;
    const uint32_t sw = (uint32_t)(row & 7);
    const int p = tp * 128 + row;                      // this thread's pair
    float racc[128];
#pragma unroll
    for (int c = 0; c < 128; ++c) racc[c] = 0.f;
    const double sz = exp2(-(double)f16_scale_exp(*a.zmax));

    auto drain = [&](int widx, int i) {                // racc += w_i(p) 2^(-S_z - S_W,i) D(window widx of frequency i)
      const float wi = p < a.pairs ? (float)(a.w[(long long)i * a.ld_w + p] * sz * exp2(-(double)f16_scale_exp(a.wmax[i]))) : 0.f;
      mbar_wait(d_full, widx & 1);
      tc_fence_after();
      const uint32_t dcol = (h ? d_im : d_re) + lane_base;
#pragma unroll
      for (int c = 0; c < 4; ++c) {
        uint32_t v[32];
        tmem_ld32(dcol + 32 * c, v);
        tmem_wait_ld();
#pragma unroll
        for (int e = 0; e < 32; ++e) racc[32 * c + e] = fmaf(wi, __uint_as_float(v[e]), racc[32 * c + e]);
      }
      tc_fence_before();
      __syncwarp();
      if (lane == 0) mbar_arrive(d_empty);
    };

    int st = 0, u = 0, ts = 0, tu = 0, kpos = 0, fidx = 0, wpos = 0, widx = 0, f_prev = 0;
    for (int s = 0; s < n_stages; ++s) {
      mbar_wait(&s_full[st], u & 1);
      if (tu > 0) mbar_wait(&a_empty[ts], (tu - 1) & 1);
      tc_fence_after();
      const uint32_t src = base + C::A_RING_OFF + st * C::A_BYTES + (uint32_t)row * 128u;
      const uint32_t tdst = a_ring + ts * C::TSLOT_COLS + 8 * h + lane_base;
#pragma unroll
      for (int xy = 0; xy < 2; ++xy) {
        uint32_t hv[8], lv[8];
#pragma unroll
        for (int cc = 0; cc < 2; ++cc) {
          const uint4 th = ld_shared_u4(src + xy * kTileS + ((((uint32_t)(2 * h + cc)) ^ sw) << 4));
          const uint4 tl = ld_shared_u4(src + xy * kTileS + ((((uint32_t)(4 + 2 * h + cc)) ^ sw) << 4));
          hv[4 * cc] = th.x; hv[4 * cc + 1] = th.y; hv[4 * cc + 2] = th.z; hv[4 * cc + 3] = th.w;
          lv[4 * cc] = tl.x; lv[4 * cc + 1] = tl.y; lv[4 * cc + 2] = tl.z; lv[4 * cc + 3] = tl.w;
        }
        tmem_st8(tdst + 16 * xy, hv);
        if (FP8) {
          uint32_t a8[4], l8[4];
#pragma unroll
          for (int c = 0; c < 4; ++c) {
            a8[c] = cvt_e5m2x2_f16x2(hv[2 * c]) | (cvt_e5m2x2_f16x2(hv[2 * c + 1]) << 16);
            l8[c] = cvt_e5m2x2_f16x2(lv[2 * c]) | (cvt_e5m2x2_f16x2(lv[2 * c + 1]) << 16);
          }
          const uint32_t t8 = a_ring + ts * C::TSLOT_COLS + 32 + 4 * h + lane_base;
          tmem_st4(t8 + 8 * xy, a8);
          tmem_st4(t8 + 16 + 8 * xy, l8);
        } else {
          tmem_st8(tdst + 32 + 16 * xy, lv);
        }
      }
      tmem_wait_st();
      tc_fence_before();
      __syncwarp();
      if (lane == 0) {
        mbar_arrive(&a_full[ts]);
        mbar_arrive(&s_empty[st]);
      }
      if (s >= 1 && wpos == 0) drain(widx - 1, f_prev);   // stage s-1 closed a window (of frequency f_prev)
      f_prev = fidx;
      ++wpos;
      if (++kpos == kst) { kpos = 0; ++fidx; }
      if (wpos == kSigcWin || kpos == 0) { wpos = 0; ++widx; }
      if (++st == C::ASTAGES) { st = 0; ++u; }
      if (++ts == C::TSLOTS) { ts = 0; ++tu; }
    }
    drain(widx - 1, a.n_freq - 1);

    if (p < a.pairs) {
      double* dst = reinterpret_cast<double*>(a.zw + (long long)p * a.n_m + tn * 128) + h;     // .x (Re) or .y (Im)
      const int ncol = min(128, a.n_m - tn * 128);
#pragma unroll
      for (int c = 0; c < 128; ++c)
        if (c < ncol) dst[2 * c] = (double)racc[c];
    }
  }
  tc_fence_before();
  __syncthreads();
  if (warp == 1) tmem_dealloc(tbase, 512);
}

// max |Re|, |Im| per batch entry (atomicMax on the float bits; *amax zeroed by the caller)
__global__ void cplx_absmax_kernel(const double2* __restrict__ x, long long n, long long batch_stride,
                                   float* __restrict__ amax) {
  const double2* xb = x + (long long)blockIdx.y * batch_stride;
  float m = 0.f;
  for (long long e = blockIdx.x * (long long)blockDim.x + threadIdx.x; e < n; e += (long long)gridDim.x * blockDim.x)
    m = fmaxf(m, fmaxf(fabsf((float)xb[e].x), fabsf((float)xb[e].y)));
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) m = fmaxf(m, __shfl_xor_sync(0xffffffffu, m, o));
  if ((threadIdx.x & 31) == 0 && m > 0.f) atomicMax(reinterpret_cast<unsigned int*>(amax + blockIdx.y), __float_as_uint(m * 1.0000002f));
}

// complex128 matrix X[rows][cols] (leading dimension ld; batch entries at x_bs) -> hl16 rows: out[plane][batch * rows_pad + r]
// [kst][64] = h[32] | l[32] of X[r][32 s + k] * 2^S (TRANSPOSE: of X[32 s + k][r]), S from amax[batch]; padding = zeros.
// One block = 32 output rows x one 32-wide stage.
template <bool TRANSPOSE>
__global__ void __launch_bounds__(256) cplx_to_hl16_rows_kernel(const double2* __restrict__ x, long long ld, int rows, int kcols,
                                                                long long x_bs, __half* __restrict__ out, int rows_pad,
                                                                int kst, long long plane_halves, const float* __restrict__ amax,
                                                                unsigned char* __restrict__ out8 = nullptr) {
  __shared__ float tx[32][33], ty[32][33];
  const int b = blockIdx.z, sg = blockIdx.x, r0 = blockIdx.y * 32;
  const double scale = exp2((double)f16_scale_exp(amax[b]));
  const double2* xb = x + (long long)b * x_bs;
  const int tl = threadIdx.x & 31, th = threadIdx.x >> 5;
  if (TRANSPOSE) {
    // read X[32 sg + kk][r0 + rr] coalesced along rr, transpose through shared memory
    for (int kk = th; kk < 32; kk += 8) {
      const int k = 32 * sg + kk, r = r0 + tl;
      double2 v = make_double2(0.0, 0.0);
      if (k < kcols && r < rows) v = xb[(long long)k * ld + r];
      tx[kk][tl] = (float)(v.x * scale);
      ty[kk][tl] = (float)(v.y * scale);
    }
    __syncthreads();
  }
  for (int rr = th; rr < 32; rr += 8) {
    const int r = r0 + rr, k = 32 * sg + tl;
    if (r >= rows_pad) continue;
    float fx = 0.f, fy = 0.f;
    if (TRANSPOSE) {
      fx = tx[tl][rr];
      fy = ty[tl][rr];
    } else if (r < rows && k < kcols) {
      const double2 v = xb[(long long)r * ld + k];
      fx = (float)(v.x * scale);
      fy = (float)(v.y * scale);
    }
    const __half hx = __float2half_rn(fx), hy = __float2half_rn(fy);
    const long long o = ((long long)b * rows_pad + r) * kst * 64 + (long long)sg * 64 + tl;
    out[o] = hx;
    out[o + 32] = __float2half_rn(fx - __half2float(hx));
    out[plane_halves + o] = hy;
    out[plane_halves + o + 32] = __float2half_rn(fy - __half2float(hy));
    if (out8) {   // hb8 rows: h[32] halves | e5m2(v)[32] | e5m2(v - h)[32]
      reinterpret_cast<__half*>(out8)[o] = hx;
      reinterpret_cast<__half*>(out8)[plane_halves + o] = hy;
      unsigned char* bx = out8 + 2 * (o - tl) + tl;
      unsigned char* by = bx + 2 * plane_halves;
      bx[64] = (unsigned char)__nv_cvt_float_to_fp8(fx, __NV_SATFINITE, __NV_E5M2);
      bx[96] = (unsigned char)__nv_cvt_float_to_fp8(fx - __half2float(hx), __NV_SATFINITE, __NV_E5M2);
      by[64] = (unsigned char)__nv_cvt_float_to_fp8(fy, __NV_SATFINITE, __NV_E5M2);
      by[96] = (unsigned char)__nv_cvt_float_to_fp8(fy - __half2float(hy), __NV_SATFINITE, __NV_E5M2);
    }
  }
}

}  // namespace

cudaError_t sigc_f16_configure() {
  cudaError_t e = cudaFuncSetAttribute(sigc_f16_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, SCfg::SMEM_BYTES);
  if (e != cudaSuccess) return e;
  return cudaFuncSetAttribute(sigc_f16_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, SCfg::SMEM_BYTES);
}

size_t sigc_f16_z_halves(long long pairs_cap, int n_m) {
  return (size_t)2 * ((pairs_cap + 127) / 128 * 128) * ((n_m + 31) / 32) * 64;
}
size_t sigc_f16_w_halves(int n_m, int n_freq) {
  return (size_t)2 * n_freq * ((n_m + 127) / 128 * 128) * ((n_m + 31) / 32) * 64;
}

cudaError_t launch_sigc_zw_f16(const double2* z, const double2* wc, const double* w, long long ld_w, int pairs, int n_m,
                               int n_freq, __half* zk16, __half* w16, unsigned char* w8 /*hb8 copy of W: E5M2 corrections; or null*/,
                               float* amax /*[1 + n_freq]*/, double2* zw, cudaStream_t s) {
  const int kst = (n_m + 31) / 32, n_m_pad = (n_m + 127) / 128 * 128;
  const long long pairs_pad = ((long long)pairs + 127) / 128 * 128;
  cudaError_t e = cudaMemsetAsync(amax, 0, sizeof(float) * (1 + n_freq), s);
  if (e != cudaSuccess) return e;
  cplx_absmax_kernel<<<dim3(592, 1), 256, 0, s>>>(z, (long long)pairs * n_m, 0, amax);
  cplx_absmax_kernel<<<dim3(148, n_freq), 256, 0, s>>>(wc, (long long)n_m * n_m, (long long)n_m * n_m, amax + 1);
  const long long zplane = pairs_pad * kst * 64, wplane = (long long)n_freq * n_m_pad * kst * 64;
  cplx_to_hl16_rows_kernel<false><<<dim3(kst, (unsigned)(pairs_pad / 32), 1), 256, 0, s>>>(z, n_m, pairs, n_m, 0, zk16, (int)pairs_pad,
                                                                                         kst, zplane, amax);
  cplx_to_hl16_rows_kernel<true><<<dim3(kst, n_m_pad / 32, n_freq), 256, 0, s>>>(wc, n_m, n_m, n_m, (long long)n_m * n_m, w16,
                                                                                n_m_pad, kst, wplane, amax + 1, w8);
  if ((e = cudaGetLastError()) != cudaSuccess) return e;
  SigcF16Args a;
  e = make_hl16_map(&a.tmap_z, zk16, (long long)kst * 64, pairs_pad, zplane);
  if (e == cudaSuccess) e = make_hl16_map(&a.tmap_w, w16, (long long)kst * 64, (long long)n_freq * n_m_pad, wplane);
  if (e == cudaSuccess && w8) e = make_hb8_map(&a.tmap_w8, w8, (long long)kst * 64, (long long)n_freq * n_m_pad, wplane);
  if (e != cudaSuccess) return e;
  a.w = w;
  a.ld_w = ld_w;
  a.zmax = amax;
  a.wmax = amax + 1;
  a.zw = zw;
  a.pairs = pairs;
  a.n_m = n_m;
  a.n_m_pad = n_m_pad;
  a.n_freq = n_freq;
  a.kst = kst;
  a.n_tiles_n = n_m_pad / 128;
  const dim3 grid((unsigned)(a.n_tiles_n * (pairs_pad / 128)));
  if (w8) sigc_f16_kernel<true><<<grid, kThreadsS, SCfg::SMEM_BYTES, s>>>(a);
  else sigc_f16_kernel<false><<<grid, kThreadsS, SCfg::SMEM_BYTES, s>>>(a);
  return cudaGetLastError();
}

}  // namespace qsgw
