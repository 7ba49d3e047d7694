// Stage (b), mixed mode: acc_j[I,J] += sum_p conj(z[p,I]) w_j(p) z[p,J] for one 128x128 tile and one
// frequency per CTA (Eq. 14; Alg. 1 lines 16-21) on the 5th-generation
// tensor cores: tcgen05.mma kind::tf32, FP32 accumulators in TMEM, FP64 accumulation across batches.
//
//   z = x + i y (FP32 planes, K-major: pair index contiguous).  With A = w_j * (x_I, y_I) and B = (x_J, y_J):
//     Re += A_x B_x + A_y B_y,     Im += A_x B_y - A_y B_x          ("4M"; the minus is the a_negate bit)
//   B tiles are TMA-written shared memory shared by all uses (unscaled z); the frequency-scaled operand A
//   is formed in registers (w * z, rounded to TF32) and stored to TENSOR MEMORY (tcgen05.st), from where
//   the MMA reads it.  NPASS = 3 ("3xTF32", FP32-grade products): A = A_hi + A_lo, B = B_hi + B_lo and
//   D += A_hi B_hi + A_lo B_hi + A_hi B_lo; NPASS = 1: single TF32 product.
//
//   The tensor core accumulates FP32 with truncation: measured bias ~ -6e-8 x (MMA steps into one
//   accumulator) on same-sign sums.  So D is drained every WIN stages (<= 64 steps per accumulator)
//   into FP32 register accumulators with round-to-nearest adds, and those go to the FP64 accumulators
//   in HBM once per launch.
//
// Roles (384 threads): warp 0 = TMA producer, warp 1 = MMA issuer (one thread) + TMEM allocator,
// warps 4-11 = scale + drain ("SA") warps: thread <-> tile row I; warps 4-7 own Re, 8-11 own Im.
#include "kernels.h"
#include "ptx.cuh"

namespace qsgw {

namespace {

constexpr int kThreadsMx = 384;
constexpr int kPlaneTile = 128 * 128;   // bytes of one 128-row x 32-float operand tile

template <int NPASS>
struct MxCfg {
  static constexpr int NPB = NPASS == 3 ? 4 : 2;          // B planes per stage
  static constexpr int STAGES = NPASS == 3 ? 2 : 3;
  static constexpr int B_BYTES = NPB * kPlaneTile;
  static constexpr int A_BYTES = 2 * kPlaneTile;
  static constexpr int W_BYTES = kPairStage * 4;
  static constexpr int STAGE_BYTES = B_BYTES + A_BYTES + 1024;   // w slot padded: tiles stay 1024-B aligned
  static constexpr int TSLOT_COLS = NPASS == 3 ? 128 : 64;       // TMEM columns of A per stage
  static constexpr int TSLOTS = 256 / TSLOT_COLS;
  static constexpr int WIN = NPASS == 3 ? 2 : 8;                 // stages per drain window
  static constexpr int SMEM_BYTES = STAGES * STAGE_BYTES + 256 + 1024 /*align slack*/;
};

template <int NPASS>
__global__ void __launch_bounds__(kThreadsMx, 1) chi0_tf32_kernel(const __grid_constant__ Chi0Tf32Args a) {
  using C = MxCfg<NPASS>;
  extern __shared__ unsigned char smem_dyn[];
  const uint32_t raw = smem_u32(smem_dyn);
  const uint32_t base = (raw + 1023u) & ~1023u;
  unsigned char* sm = smem_dyn + (base - raw);
  uint64_t* bars = reinterpret_cast<uint64_t*>(sm + C::STAGES * C::STAGE_BYTES);
  uint64_t* full = bars;
  uint64_t* empty = full + C::STAGES;
  uint64_t* a_full = empty + C::STAGES;
  uint64_t* a_empty = a_full + C::TSLOTS;
  uint64_t* d_full = a_empty + C::TSLOTS;
  uint64_t* d_empty = d_full + 1;
  uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(d_empty + 1);

  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int j = blockIdx.x % a.n_freq;
  const int2 tt = a.d_tiles[blockIdx.x / a.n_freq];
  const bool diag = (tt.x == tt.y);
  const bool need_a = !(NPASS == 3 && diag);     // 3xTF32 diagonal tile: A source = B planes 0/1
  const int n_stages = a.n_stages;

  if (tid == 0) {
    tma_prefetch_desc(&a.tmap2);
    tma_prefetch_desc(&a.tmap4);
    for (int s = 0; s < C::STAGES; ++s) {
      mbar_init(&full[s], 1);
      mbar_init(&empty[s], 9);       // 8 SA warps + the MMA commit
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
    if (warp == 0 && lane == 0) {
      // ------------------------------------------------------------------ TMA producer
      const float* wrow = a.wtab32 + (long long)j * a.kpad;
      const uint32_t bytes = C::B_BYTES + C::W_BYTES + (need_a ? C::A_BYTES : 0);
      for (int s = 0; s < n_stages; ++s) {
        const int st = s % C::STAGES, u = s / C::STAGES;
        if (u > 0) mbar_wait(&empty[st], (u - 1) & 1);
        unsigned char* sb = sm + st * C::STAGE_BYTES;
        mbar_arrive_expect_tx(&full[st], bytes);
        if (NPASS == 3) tma_load_3d(sb, &a.tmap4, &full[st], s * kPairStage, tt.y * kTileMx, 0);
        else tma_load_3d(sb, &a.tmap2, &full[st], s * kPairStage, tt.y * kTileMx, 2);
        if (need_a) tma_load_3d(sb + C::B_BYTES, &a.tmap2, &full[st], s * kPairStage, tt.x * kTileMx, 0);
        bulk_load_1d(sb + C::B_BYTES + C::A_BYTES, wrow + (long long)s * kPairStage, C::W_BYTES, &full[st]);
      }
    } else if (warp == 1 && lane == 0) {
      // ------------------------------------------------------------------ MMA issuer
      const uint32_t idesc = umma_idesc_tf32(128, 128, 0), idesc_neg = umma_idesc_tf32(128, 128, 1);
      for (int s = 0; s < n_stages; ++s) {
        const int st = s % C::STAGES, u = s / C::STAGES, ts = s % C::TSLOTS, tu = s / C::TSLOTS;
        const bool win_first = (s % C::WIN) == 0;
        if (win_first && s > 0) mbar_wait(d_empty, ((s / C::WIN) - 1) & 1);
        mbar_wait(&full[st], u & 1);
        mbar_wait(&a_full[ts], tu & 1);
        tc_fence_after();
        const uint32_t sb = base + st * C::STAGE_BYTES;
        const uint64_t bx = umma_desc_k_sw128(sb), by = umma_desc_k_sw128(sb + kPlaneTile);
        const uint64_t bxl = umma_desc_k_sw128(sb + 2 * kPlaneTile), byl = umma_desc_k_sw128(sb + 3 * kPlaneTile);
        const uint32_t ab = a_ring + ts * C::TSLOT_COLS;
#pragma unroll
        for (int g = 0; g < kPairStage / 8; ++g) {
          const uint32_t acc0 = (win_first && g == 0) ? 0u : 1u;
          const uint64_t ko = (uint64_t)(2 * g);            // 8 floats = 32 B along K inside the swizzle row
          const uint32_t ax = ab + 8 * g, ay = ab + 32 + 8 * g;
          umma_tf32_ts(d_re, ax, bx + ko, idesc, acc0);
          umma_tf32_ts(d_re, ay, by + ko, idesc, 1u);
          umma_tf32_ts(d_im, ax, by + ko, idesc, acc0);
          umma_tf32_ts(d_im, ay, bx + ko, idesc_neg, 1u);
          if (NPASS == 3) {
            const uint32_t axl = ab + 64 + 8 * g, ayl = ab + 96 + 8 * g;
            umma_tf32_ts(d_re, axl, bx + ko, idesc, 1u);
            umma_tf32_ts(d_re, ayl, by + ko, idesc, 1u);
            umma_tf32_ts(d_im, axl, by + ko, idesc, 1u);
            umma_tf32_ts(d_im, ayl, bx + ko, idesc_neg, 1u);
            umma_tf32_ts(d_re, ax, bxl + ko, idesc, 1u);
            umma_tf32_ts(d_re, ay, byl + ko, idesc, 1u);
            umma_tf32_ts(d_im, ax, byl + ko, idesc, 1u);
            umma_tf32_ts(d_im, ay, bxl + ko, idesc_neg, 1u);
          }
        }
        umma_commit(&empty[st]);
        umma_commit(&a_empty[ts]);
        if (((s + 1) % C::WIN) == 0 || s == n_stages - 1) umma_commit(d_full);
      }
    }
  } else {
    // -------------------------------------------------------------------- scale + drain warps
    setmaxnreg_inc<224>();
    const int q = warp & 3, h = (warp - 4) >> 2;       // TMEM lane quarter; pair half / Re-Im owner
    const int row = 32 * q + lane;
    const uint32_t lane_base = (uint32_t)(32 * q) << 16;
    const uint32_t sw = (uint32_t)(row & 7);
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

    for (int s = 0; s < n_stages; ++s) {
      const int st = s % C::STAGES, u = s / C::STAGES, ts = s % C::TSLOTS, tu = s / C::TSLOTS;
      mbar_wait(&full[st], u & 1);
      if (tu > 0) mbar_wait(&a_empty[ts], (tu - 1) & 1);
      tc_fence_after();
      const uint32_t sb = base + st * C::STAGE_BYTES;
      const uint32_t src = (need_a ? sb + C::B_BYTES : sb) + (uint32_t)row * 128u;
      const uint32_t swp = sb + C::B_BYTES + C::A_BYTES;
      const uint32_t tdst = a_ring + ts * C::TSLOT_COLS + 16 * h + lane_base;
      float4 w4[4];
#pragma unroll
      for (int cc = 0; cc < 4; ++cc) w4[cc] = ld_shared_f4(swp + 16 * (4 * h + cc));
#pragma unroll
      for (int xy = 0; xy < 2; ++xy) {
        uint32_t hi[16], lo[16];
#pragma unroll
        for (int cc = 0; cc < 4; ++cc) {
          const uint32_t c = (uint32_t)(4 * h + cc);
          const float4 v = ld_shared_f4(src + xy * kPlaneTile + ((c ^ sw) << 4));
          const float av[4] = {w4[cc].x * v.x, w4[cc].y * v.y, w4[cc].z * v.z, w4[cc].w * v.w};
#pragma unroll
          for (int e = 0; e < 4; ++e) {
            hi[4 * cc + e] = cvt_tf32_rna(av[e]);
            lo[4 * cc + e] = __float_as_uint(av[e] - __uint_as_float(hi[4 * cc + e]));
          }
        }
        tmem_st16(tdst + 32 * xy, hi);
        if (NPASS == 3) tmem_st16(tdst + 64 + 32 * xy, lo);
      }
      tmem_wait_st();
      tc_fence_before();
      __syncwarp();
      if (lane == 0) {
        mbar_arrive(&a_full[ts]);
        mbar_arrive(&empty[st]);
      }
      if (s >= 1 && (s % C::WIN) == 0) drain(s / C::WIN - 1);   // stage s-1 closed a window
    }
    drain((n_stages - 1) / C::WIN);

    // FP32 window sums -> FP64 accumulators (exclusive owner of (tile, j))
    const long long plane = (long long)a.n_m_pad * a.n_m_pad;
    double* dst = (h ? a.acc_im : a.acc_re) + (long long)j * plane +
                  (long long)(tt.x * kTileMx + row) * a.n_m_pad + tt.y * kTileMx;
#pragma unroll
    for (int c = 0; c < 64; ++c) {
      double2 v = *reinterpret_cast<double2*>(dst + 2 * c);
      v.x += (double)racc[2 * c];
      v.y += (double)racc[2 * c + 1];
      *reinterpret_cast<double2*>(dst + 2 * c) = v;
    }
  }
  tc_fence_before();
  __syncthreads();
  if (warp == 1) tmem_dealloc(tbase, 512);
}

// Issue-rate probe of the TF32 tensor pipe: every SM issues back-to-back 128x128x8 MMAs (A in TMEM,
// B in shared memory, no global traffic).  The operand contents are whatever the memories hold.
__global__ void __launch_bounds__(128, 1) tf32_peak_kernel(int iters) {
  extern __shared__ unsigned char smem_dyn[];
  const uint32_t raw = smem_u32(smem_dyn);
  const uint32_t base = (raw + 1023u) & ~1023u;
  unsigned char* sm = smem_dyn + (base - raw);
  uint64_t* bar = reinterpret_cast<uint64_t*>(sm + kPlaneTile);
  uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(bar + 1);
  const int tid = threadIdx.x, warp = tid >> 5;
  for (int i = tid; i < kPlaneTile / 4; i += 128) reinterpret_cast<float*>(sm)[i] = 1.0f + 0.001f * (i & 255);
  if (tid == 0) {
    mbar_init(bar, 1);
    mbar_fence_init();
  }
  if (warp == 0) tmem_alloc(tmem_slot, 512);
  asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tbase = *tmem_slot;
  uint32_t v[16];
#pragma unroll
  for (int i = 0; i < 16; ++i) v[i] = cvt_tf32_rna(0.5f + 0.01f * i);
  tmem_st16(tbase + 256 + ((uint32_t)(32 * warp) << 16), v);
  tmem_st16(tbase + 272 + ((uint32_t)(32 * warp) << 16), v);
  tmem_wait_st();
  tc_fence_before();
  __syncthreads();
  if (tid == 0) {
    tc_fence_after();
    const uint32_t idesc = umma_idesc_tf32(128, 128, 0);
    const uint64_t bd = umma_desc_k_sw128(base);
    for (int it = 0; it < iters; ++it) {
#pragma unroll
      for (int g = 0; g < 4; ++g) {
        umma_tf32_ts(tbase, tbase + 256 + 8 * g, bd + (uint64_t)(2 * g), idesc, (it | g) ? 1u : 0u);
        umma_tf32_ts(tbase + 128, tbase + 256 + 8 * g, bd + (uint64_t)(2 * g), idesc, (it | g) ? 1u : 0u);
      }
    }
    umma_commit(bar);
    mbar_wait(bar, 0);
  }
  tc_fence_before();
  __syncthreads();
  if (warp == 0) tmem_dealloc(tbase, 512);
}

}  // namespace

cudaError_t chi0_tf32_configure() {
  cudaError_t e = cudaFuncSetAttribute(chi0_tf32_kernel<1>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                       MxCfg<1>::SMEM_BYTES);
  if (e != cudaSuccess) return e;
  e = cudaFuncSetAttribute(chi0_tf32_kernel<3>, cudaFuncAttributeMaxDynamicSharedMemorySize, MxCfg<3>::SMEM_BYTES);
  if (e != cudaSuccess) return e;
  return cudaFuncSetAttribute(tf32_peak_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, 20480);
}

cudaError_t launch_chi0_tf32(const Chi0Tf32Args& a, int n_pass, cudaStream_t s) {
  if (a.n_stages <= 0 || a.n_tiles <= 0) return cudaSuccess;
  dim3 grid((unsigned)(a.n_tiles * a.n_freq));
  if (n_pass == 3) chi0_tf32_kernel<3><<<grid, kThreadsMx, MxCfg<3>::SMEM_BYTES, s>>>(a);
  else chi0_tf32_kernel<1><<<grid, kThreadsMx, MxCfg<1>::SMEM_BYTES, s>>>(a);
  return cudaGetLastError();
}

cudaError_t probe_tf32_mma(cudaStream_t s, double* out_tflops, double* out_ms) {
  int dev = 0, n_sm = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return e;
  e = cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev);
  if (e != cudaSuccess) return e;
  e = chi0_tf32_configure();
  if (e != cudaSuccess) return e;
  cudaEvent_t e0 = nullptr, e1 = nullptr;
  cudaEventCreate(&e0);
  cudaEventCreate(&e1);
  const int iters = 40000;   // x 8 MMAs x 64 clk = 20.5 Mclk ~ 11-17 ms
  tf32_peak_kernel<<<n_sm, 128, 20480, s>>>(iters / 4);
  float best = 1e30f;
  for (int rep = 0; rep < 4; ++rep) {
    cudaEventRecord(e0, s);
    tf32_peak_kernel<<<n_sm, 128, 20480, s>>>(iters);
    cudaEventRecord(e1, s);
    e = cudaEventSynchronize(e1);
    if (e != cudaSuccess) break;
    float ms = 0.f;
    cudaEventElapsedTime(&ms, e0, e1);
    if (ms < best) best = ms;
  }
  cudaEventDestroy(e0);
  cudaEventDestroy(e1);
  if (e != cudaSuccess) return e;
  e = cudaGetLastError();
  if (e != cudaSuccess) return e;
  const double flop = 2.0 * 128.0 * 128.0 * 8.0 * 8.0 * (double)iters * n_sm;
  if (out_tflops) *out_tflops = flop / (best * 1e-3) / 1e12;
  if (out_ms) *out_ms = best;
  return cudaSuccess;
}

}  // namespace qsgw
