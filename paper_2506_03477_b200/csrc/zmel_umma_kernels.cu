// Stage (a), mixed mode, on the 5th-generation tensor cores: muffin-tin product-basis matrix elements, Eq. (8) with the
// eigenfunction expansion of Eq. (4), two-step contraction of Alg. 1 line 12, written
// straight into the FP16-split operand rows of stage (b) ("hl16" / "hb8", kernels.h): no FP64 z array, no conversion pass.
//
//   step 1 (CUDA cores, FP64):  T[alpha][I][n] = sum_beta P[I,alpha,beta] C_k[beta,n]          per site, 7 % of the flops
//   step 2 (tcgen05.mma kind::f16, FP32-grade products from FP16 pieces, as stage (b)):
//       z[n, n', I] = sum_alpha conj(C_kq[alpha, n']) T[alpha][I][n]
//       D[n' (128 rows), (I, n) (16 x 8 = 128 columns)] += A[n', alpha] B[(I, n), alpha]^T,   K = the <= 32 orbitals of the site
//       A = C_kq rows of the site as h[32] | l[32] halves (one 128-byte swizzle row per band, written once per k-point by
//       ckq_to_hl16_kernel, loaded by TMA), B = 2^St T written by the CTA's threads into the same swizzled layout;
//       a b ~= a_h b_h + a_l b_h + a_h b_l;  Re = cr tr + ci ti,  Im = cr ti - ci tr  (a_negate bit): 12 MMAs per 16 alpha.
//   epilogue: D (TMEM) -> registers (thread <-> band n', so that the 32 lanes of a warp hold 32 consecutive pair rows of one
//       band n = one 64-byte run of an operand row) -> h = fp16(x), l = fp16(x - h), e5m2 pieces -> global.
//   Two CTAs per SM (256 TMEM columns and ~100 KB of shared memory each): step 1 and the MMAs of one run under the epilogue
//   of the other.
//
// The FP16 scale 2^S of the batch has to be known before the first row is written: where the FP64 path puts max |z| itself,
// zmax[b] receives the bound  max_s max_I ||P_I||_F max_n ||c_n,s|| max_n' ||c'_n',s||  (Cauchy-Schwarz per site).  Every
// consumer only derives S from it; a bound a few powers of two above the maximum costs FP16 exponent range at the small end
// (absolute error 2^-25 of the largest |z| 2^S), not mantissa bits.
#include <cuda_fp8.h>

#include "kernels.h"
#include "ptx.cuh"

namespace qsgw {

namespace {

constexpr int kZuThreads = 256;
constexpr int kZuNB = 8;              // bands n per CTA: 16 product functions x 8 bands = 128 accumulator columns
constexpr int kZuK = 32;              // orbitals per site the kernel holds (one swizzle row: h[32] | l[32])
constexpr int kZuTile = 128 * 128;    // bytes of one 128-row operand tile (one plane)
constexpr int kZuMaxSeg = 16;         // a 16-column group touches at most 16 sites

// pmax[s] = max_{I in s} ||P_I||_F  (once per product tensor)
__global__ void zu_pnorm_kernel(SiteTables st, const double2* __restrict__ P, float* __restrict__ pmax) {
  const int s = blockIdx.x;
  const int m0 = st.d_pb_off[s], m1 = st.d_pb_off[s + 1];
  const int b = st.d_orb_off[s + 1] - st.d_orb_off[s];
  const double2* Ps = P + st.d_p_off[s];
  __shared__ float red[32];
  float best = 0.f;
  for (int I = m0 + (threadIdx.x >> 5); I < m1; I += blockDim.x >> 5) {     // one warp per product function
    const double2* pi = Ps + (long long)(I - m0) * b * b;
    double acc = 0.0;
    for (int e = threadIdx.x & 31; e < b * b; e += 32) acc += pi[e].x * pi[e].x + pi[e].y * pi[e].y;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
    best = fmaxf(best, (float)sqrt(acc) * 1.0001f);
  }
  if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = best;
  __syncthreads();
  if (threadIdx.x == 0) {
    for (int w = 1; w < (int)(blockDim.x >> 5); ++w) best = fmaxf(best, red[w]);
    pmax[s] = best;
  }
}

// cnorm[b][s][0 | 1] = max over the bands n (n') of batch b of ||C_k[s-orbitals, n]|| (||C_kq[s-orbitals, n']||): one warp
// per band, atomicMax on the float bits (cnorm zeroed before the launch)
__global__ void zu_cnorm_kernel(SiteTables st, const double2* __restrict__ Ck, long long ld_k, long long Ck_bs, int n_begin,
                                int n_o, const double2* __restrict__ Ckq, long long ld_kq, long long Ckq_bs, int np_begin,
                                int n_u, float* __restrict__ cnorm) {
  const int lane = threadIdx.x & 31;
  const int r = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
  if (r >= n_o + n_u) return;
  const bool occ = r < n_o;
  const double2* c = occ ? Ck + (long long)blockIdx.y * Ck_bs + (long long)(n_begin + r) * ld_k
                         : Ckq + (long long)blockIdx.y * Ckq_bs + (long long)(np_begin + r - n_o) * ld_kq;
  float* dst = cnorm + (long long)blockIdx.y * st.n_sites * 2 + (occ ? 0 : 1);
  for (int s = 0; s < st.n_sites; ++s) {
    const int o0 = st.d_orb_off[s], b = st.d_orb_off[s + 1] - o0;
    double acc = 0.0;
    for (int e = lane; e < b; e += 32) acc += c[o0 + e].x * c[o0 + e].x + c[o0 + e].y * c[o0 + e].y;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
    if (lane == 0) atomicMax(reinterpret_cast<unsigned int*>(dst + 2 * s), __float_as_uint((float)sqrt(acc) * 1.0001f));
  }
}

// scales of batch b from the norms: bound of max |z|, S = f16_scale_exp(bound), Sa = f16_scale_exp(max_s max_n' ||c'_n',s||)
__device__ __forceinline__ void zu_scales(const SiteTables& st, const float* __restrict__ pmax, const float* __restrict__ cn,
                                          float& bound, int& Sa) {
  float bd = 0.f, cq = 0.f;
  for (int s = 0; s < st.n_sites; ++s) {
    bd = fmaxf(bd, pmax[s] * cn[2 * s] * cn[2 * s + 1]);
    cq = fmaxf(cq, cn[2 * s + 1]);
  }
  bound = bd * 1.001f;
  Sa = f16_scale_exp(cq);
}

// scales[b] = (2^St, 2^Sa) and zmax[b] = the bound, once per batch (one warp)
__global__ void zu_scale_kernel(SiteTables st, const float* __restrict__ pmax, const float* __restrict__ cnorm,
                                float2* __restrict__ scales, float* __restrict__ zmax) {
  const int b = blockIdx.x;
  if (threadIdx.x != 0) return;
  float bound;
  int Sa;
  zu_scales(st, pmax, cnorm + (long long)b * st.n_sites * 2, bound, Sa);
  scales[b] = make_float2(exp2f((float)(f16_scale_exp(bound) - Sa)), exp2f((float)Sa));     // D = (2^Sa c)(2^St t) = 2^S z
  zmax[b] = bound;
}

// A operand of step 2: aop[plane (Re, Im)][(b n_sites + s) n_u_pad + n'][64] = h[32] | l[32] of 2^Sa C_kq[alpha, n'] over the
// orbitals alpha of site s (zeros for alpha >= b_s and for n' >= n_u).  One thread per (row, alpha).
__global__ void ckq_to_hl16_kernel(SiteTables st, const float2* __restrict__ scales,
                                   const double2* __restrict__ Ckq, long long ld_kq, long long Ckq_bs, int np_begin, int n_u,
                                   int n_u_pad, int n_batch, __half* __restrict__ aop) {
  const long long rows = (long long)n_batch * st.n_sites * n_u_pad;
  const long long plane = rows * 64;
  for (long long e = blockIdx.x * (long long)blockDim.x + threadIdx.x; e < rows * kZuK; e += (long long)gridDim.x * blockDim.x) {
    const int alpha = (int)(e & (kZuK - 1));
    const long long row = e >> 5;
    const int np = (int)(row % n_u_pad);
    const long long bs = row / n_u_pad;
    const int s = (int)(bs % st.n_sites), b = (int)(bs / st.n_sites);
    const int o0 = st.d_orb_off[s], nb = st.d_orb_off[s + 1] - o0;
    float x = 0.f, y = 0.f;
    if (alpha < nb && np < n_u) {
      const double2 c = Ckq[(long long)b * Ckq_bs + (long long)(np_begin + np) * ld_kq + o0 + alpha];
      const double sc = (double)scales[b].y;
      x = (float)(c.x * sc);
      y = (float)(c.y * sc);
    }
    const __half hx = __float2half_rn(x), hy = __float2half_rn(y);
    __half* o = aop + row * 64 + alpha;
    o[0] = hx;
    o[32] = __float2half_rn(x - __half2float(hx));
    o[plane] = hy;
    o[plane + 32] = __float2half_rn(y - __half2float(hy));
  }
}

struct HlOut {
  __half* hl;            // hl16 rows of this batch
  unsigned char* hb8;    // hb8 rows (may be null)
  long long kpad;
  long long oplane;      // halves per plane
};

// one value pair (x, y) = 2^S z of pair row p, product function I -> the operand rows
__device__ __forceinline__ void store_hl(const HlOut& o, int I, long long p, float x, float y) {
  const __half hx = __float2half_rn(x), hy = __float2half_rn(y);
  const float rx = x - __half2float(hx), ry = y - __half2float(hy);
  const long long r = (long long)I * o.kpad * 2 + (p >> 5) * 64 + (p & 31);
  o.hl[r] = hx;
  o.hl[r + 32] = __float2half_rn(rx);
  o.hl[o.oplane + r] = hy;
  o.hl[o.oplane + r + 32] = __float2half_rn(ry);
  if (o.hb8) {
    reinterpret_cast<__half*>(o.hb8)[r] = hx;
    reinterpret_cast<__half*>(o.hb8)[o.oplane + r] = hy;
    unsigned char* bx = o.hb8 + 2 * ((long long)I * o.kpad * 2 + (p >> 5) * 64) + (p & 31);
    unsigned char* by = bx + 2 * o.oplane;
    bx[64] = (unsigned char)__nv_cvt_float_to_fp8(x, __NV_SATFINITE, __NV_E5M2);
    bx[96] = (unsigned char)__nv_cvt_float_to_fp8(rx, __NV_SATFINITE, __NV_E5M2);
    by[64] = (unsigned char)__nv_cvt_float_to_fp8(y, __NV_SATFINITE, __NV_E5M2);
    by[96] = (unsigned char)__nv_cvt_float_to_fp8(ry, __NV_SATFINITE, __NV_E5M2);
  }
}

struct ZuCfg {
  static constexpr int A_SLOTS = 2;
  static constexpr int A_BYTES = 2 * kZuTile;                 // planes cr | ci of one 128-band tile
  static constexpr int B_OFF = A_SLOTS * A_BYTES;
  static constexpr int B_BYTES = 2 * kZuTile;                 // planes tr | ti, rows = (I_loc, n_loc)
  static constexpr int CS_OFF = B_OFF + B_BYTES;              // double2 cs[kZuNB][kZuK]
  static constexpr int BAR_OFF = CS_OFF + kZuNB * kZuK * 16;
  static constexpr int SMEM_BYTES = BAR_OFF + 128 + 1024 /*align slack*/;
};

__global__ void __launch_bounds__(kZuThreads, 2)
    zmel_umma_kernel(const __grid_constant__ CUtensorMap tmap_a, ZmelArgs a, const float2* __restrict__ scales, __half* zhl, unsigned char* zhb8, int n_m_pad, long long n_rows,
                     int n_u_pad) {
  using C = ZuCfg;
  extern __shared__ unsigned char smem_dyn[];
  const uint32_t raw = smem_u32(smem_dyn);
  const uint32_t base = (raw + 1023u) & ~1023u;
  unsigned char* sm = smem_dyn + (base - raw);
  double2* cs = reinterpret_cast<double2*>(sm + C::CS_OFF);
  uint64_t* bars = reinterpret_cast<uint64_t*>(sm + C::BAR_OFF);
  uint64_t* a_full = bars;            // [2]
  uint64_t* a_empty = bars + 2;       // [2]
  uint64_t* d_full = bars + 4;        // [2]
  uint64_t* d_empty = bars + 6;       // [2]
  uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(bars + 8);
  __shared__ int seg_o0[kZuMaxSeg], seg_b[kZuMaxSeg], seg_c0[kZuMaxSeg], seg_c1[kZuMaxSeg], seg_site[kZuMaxSeg];
  __shared__ int n_seg_s;
  __shared__ float scale_s[2];

  const int tid = threadIdx.x, warp = uniform_warp_idx(), lane = tid & 31;
  const int kb = blockIdx.z;                              // k-point of this CTA
  a.Ck += (long long)kb * a.Ck_bs;
  HlOut out;
  out.kpad = a.kpad;
  out.oplane = (long long)n_m_pad * a.kpad * 2;
  out.hl = zhl + (long long)kb * (a.z_bs / kPairStage) * 64;
  out.hb8 = zhb8 ? zhb8 + (long long)kb * (a.z_bs / kPairStage) * 128 : nullptr;
  const int cg = blockIdx.x;
  const int n0 = blockIdx.y * kZuNB;
  const int nb = min(kZuNB, a.n_o - n0);
  const int I0 = cg * kCG;
  const int I1 = min(I0 + kCG, a.st.n_m);
  const long long n_pairs = (long long)a.n_o * a.n_u;
  const int n_mt = (a.n_u + 127) >> 7;

  if (tid == 0) {
    tma_prefetch_desc(&tmap_a);
    for (int i = 0; i < 2; ++i) {
      mbar_init(&a_full[i], 1);
      mbar_init(&a_empty[i], 1);
      mbar_init(&d_full[i], 1);
      mbar_init(&d_empty[i], 8);
    }
    mbar_fence_init();
  }
  // segments of this column group (sites it touches): thread i looks at product function I0 + i
  if (tid < kCG) {
    const int I = I0 + tid;
    const int s = I < I1 ? a.st.d_pb_site[I] : -1;
    const int sp = (tid > 0 && I - 1 < I1) ? a.st.d_pb_site[I - 1] : -2;
    const unsigned first = __ballot_sync(0xffffu, s >= 0 && s != sp);       // bit i: a segment starts at column i
    if (s >= 0 && s != sp) {
      const int idx = __popc(first & ((1u << tid) - 1u));
      const int e = min(I1, a.st.d_pb_off[s + 1]);
      seg_site[idx] = s;
      seg_o0[idx] = a.st.d_orb_off[s];
      seg_b[idx] = a.st.d_orb_off[s + 1] - a.st.d_orb_off[s];
      seg_c0[idx] = tid;
      seg_c1[idx] = e - I0;
    }
    if (tid == 0) {
      n_seg_s = __popc(first);
      scale_s[0] = scales[kb].x;
    }
  }
  if (warp == 1) tmem_alloc(tmem_slot, 256);
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tbase = *tmem_slot;
  const double st_scale = (double)scale_s[0];

  // rows of pairs beyond the batch are zeros (once per column group)
  if (blockIdx.y == 0) {
    const int tail = (int)(n_rows - n_pairs);
    for (int idx = tid; idx < tail * (I1 - I0); idx += kZuThreads)
      store_hl(out, I0 + idx / tail, n_pairs + idx % tail, 0.f, 0.f);
  }

  int a_use = 0, d_use = 0;           // tiles loaded / accumulator buffers used so far (same count in every role)
  for (int sg = 0; sg < n_seg_s; ++sg) {
    const int o0 = seg_o0[sg], b = seg_b[sg], c0 = seg_c0[sg], c1 = seg_c1[sg], site = seg_site[sg];
    // ---- step 1: B operand = 2^St T of this segment (all threads) ----
    {
      uint4* bz = reinterpret_cast<uint4*>(sm + C::B_OFF);
      for (int i = tid; i < C::B_BYTES / 16; i += kZuThreads) bz[i] = make_uint4(0u, 0u, 0u, 0u);
      for (int idx = tid; idx < kZuNB * kZuK; idx += kZuThreads) {
        const int n = idx / kZuK, beta = idx - n * kZuK;
        double2 v = make_double2(0.0, 0.0);
        if (n < nb && beta < b) v = a.Ck[(long long)(a.n_begin + n0 + n) * a.ld_k + o0 + beta];
        cs[n * kZuK + beta] = v;
      }
      __syncthreads();
      const int m0 = a.st.d_pb_off[site];
      const double2* Ps = a.P + a.st.d_p_off[site];
      unsigned char* btr = sm + C::B_OFF;
      unsigned char* bti = btr + kZuTile;
      for (int item = tid; item < (c1 - c0) * b; item += kZuThreads) {
        const int il = c0 + item / b, alpha = item % b;
        const double2* prow = Ps + ((long long)(I0 + il - m0) * b + alpha) * b;
        double ar[kZuNB], ai[kZuNB];
#pragma unroll
        for (int n = 0; n < kZuNB; ++n) ar[n] = ai[n] = 0.0;
        for (int beta0 = 0; beta0 < b; beta0 += 8) {       // eight independent loads of P in flight per thread
          double2 pd[8];
#pragma unroll
          for (int j = 0; j < 8; ++j) pd[j] = beta0 + j < b ? prow[beta0 + j] : make_double2(0.0, 0.0);
#pragma unroll
          for (int j = 0; j < 8; ++j) {
#pragma unroll
            for (int n = 0; n < kZuNB; ++n) {
              const double2 c = cs[n * kZuK + beta0 + j];
              ar[n] += pd[j].x * c.x - pd[j].y * c.y;
              ai[n] += pd[j].x * c.y + pd[j].y * c.x;
            }
          }
        }
        const uint32_t ch = (uint32_t)(alpha >> 3), within = (uint32_t)(alpha & 7) * 2u;
#pragma unroll
        for (int n = 0; n < kZuNB; ++n) {
          const uint32_t r = (uint32_t)(il * kZuNB + n);
          const uint32_t oh = r * 128u + ((ch ^ (r & 7u)) << 4) + within, ol = r * 128u + (((4u + ch) ^ (r & 7u)) << 4) + within;
          const float x = (float)(ar[n] * st_scale), y = (float)(ai[n] * st_scale);
          const __half hx = __float2half_rn(x), hy = __float2half_rn(y);
          *reinterpret_cast<__half*>(btr + oh) = hx;
          *reinterpret_cast<__half*>(btr + ol) = __float2half_rn(x - __half2float(hx));
          *reinterpret_cast<__half*>(bti + oh) = hy;
          *reinterpret_cast<__half*>(bti + ol) = __float2half_rn(y - __half2float(hy));
        }
      }
      fence_proxy_async_smem();
      __syncthreads();
    }
    // ---- step 2: warp 0 feeds the A tiles (ring of two), warp 1 issues the MMAs, all eight warps run the epilogue ----
    {
      const int q = warp & 3, hsel = warp >> 2;       // TMEM lane quarter; first / second half of the segment's columns
      const uint32_t lane_base = (uint32_t)(32 * q) << 16;
      const int row_base = (kb * a.st.n_sites + site) * n_u_pad;
      const int half = (c1 - c0 + 1) >> 1;
      const int il0 = hsel == 0 ? c0 : c0 + half, il1 = hsel == 0 ? c0 + half : c1;
      auto load_tile = [&](int mt) {
        const int use = a_use + mt, slot = use & 1;
        if (use >= 2) mbar_wait(&a_empty[slot], ((use >> 1) - 1) & 1);
        if (elect_one()) {
          unsigned char* sa = sm + slot * C::A_BYTES;
          mbar_arrive_expect_tx(&a_full[slot], C::A_BYTES);
#pragma unroll
          for (int i = 0; i < 4; ++i) {
            const int plane = i >> 1, rh = i & 1;
            tma_load_3d(sa + plane * kZuTile + rh * (64 * 128), &tmap_a, &a_full[slot], 0, row_base + mt * 128 + rh * 64, plane);
          }
        }
        __syncwarp();
      };
      if (warp == 0) {
        load_tile(0);
        if (n_mt > 1) load_tile(1);
      }
      const uint32_t idesc = umma_idesc_f16(128, 128, 0), idesc_neg = umma_idesc_f16(128, 128, 1);
      const uint32_t sb = base + C::B_OFF;
      const uint64_t btr = umma_desc_k_sw128(sb), bti = umma_desc_k_sw128(sb + kZuTile);
      const int ksteps = b > 16 ? 2 : 1;
      for (int mt = 0; mt < n_mt; ++mt) {
        const int du = d_use + mt;
        if (warp == 1) {
          const int au = a_use + mt, slot = au & 1;
          mbar_wait(&a_full[slot], (au >> 1) & 1);
          if (du >= 1) mbar_wait(d_empty, (du - 1) & 1);
          tc_fence_after();
          if (elect_one()) {
            const uint32_t sa = base + slot * C::A_BYTES;
            const uint64_t acr = umma_desc_k_sw128(sa), aci = umma_desc_k_sw128(sa + kZuTile);
            const uint32_t d_re = tbase, d_im = tbase + 128;
            // the small correction products first, the main products h h last: the tensor core's FP32 accumulation
            // truncates, and only the last few additions then act on the full magnitude of the sum
            for (int g = 0; g < ksteps; ++g) {
              const uint64_t kh = (uint64_t)(2 * g), kl = (uint64_t)(4 + 2 * g);
              const uint32_t acc0 = g == 0 ? 0u : 1u;
              umma_f16_ss(d_re, acr + kl, btr + kh, idesc, acc0);            // Re = cr tr + ci ti
              umma_f16_ss(d_re, acr + kh, btr + kl, idesc, 1u);
              umma_f16_ss(d_re, aci + kl, bti + kh, idesc, 1u);
              umma_f16_ss(d_re, aci + kh, bti + kl, idesc, 1u);
              umma_f16_ss(d_im, acr + kl, bti + kh, idesc, acc0);            // Im = cr ti - ci tr
              umma_f16_ss(d_im, acr + kh, bti + kl, idesc, 1u);
              umma_f16_ss(d_im, aci + kl, btr + kh, idesc_neg, 1u);
              umma_f16_ss(d_im, aci + kh, btr + kl, idesc_neg, 1u);
            }
            for (int g = 0; g < ksteps; ++g) {
              const uint64_t kh = (uint64_t)(2 * g);
              umma_f16_ss(d_re, acr + kh, btr + kh, idesc, 1u);
              umma_f16_ss(d_re, aci + kh, bti + kh, idesc, 1u);
              umma_f16_ss(d_im, acr + kh, bti + kh, idesc, 1u);
              umma_f16_ss(d_im, aci + kh, btr + kh, idesc_neg, 1u);
            }
            umma_commit(&a_empty[slot]);
            umma_commit(d_full);
          }
          __syncwarp();
        } else if (warp == 0 && mt + 2 < n_mt) {
          load_tile(mt + 2);
        }
        // epilogue of tile mt: thread <-> band n'
        mbar_wait(d_full, du & 1);
        tc_fence_after();
        const int np = mt * 128 + 32 * q + lane;
        const bool np_ok = np < a.n_u;
        const uint32_t d_re = tbase + lane_base, d_im = d_re + 128;
        // positions of this thread's eight pair rows inside an operand row (the same for every product function):
        // off = halves from the start of the row, lo = pair index inside its 32-pair stage
        uint32_t off[kZuNB], lo[kZuNB];
#pragma unroll
        for (int n = 0; n < kZuNB; ++n) {
          long long pair = (long long)(n0 + n) * a.n_u + np;
          if (a.row_map && np_ok && n < nb) pair = a.row_map[pair];
          lo[n] = (uint32_t)(pair & 31);
          off[n] = (uint32_t)(pair >> 5) * 64u + lo[n];
        }
        uint32_t nr[8], ni[8];                     // the next product function's columns are in flight while this one is stored
        if (il0 < il1) {
          tmem_ld8(d_re + il0 * kZuNB, nr);
          tmem_ld8(d_im + il0 * kZuNB, ni);
        }
        for (int il = il0; il < il1; ++il) {
          uint32_t vr[8], vi[8];
          tmem_wait_ld();
#pragma unroll
          for (int n = 0; n < kZuNB; ++n) { vr[n] = nr[n]; vi[n] = ni[n]; }
          if (il + 1 < il1) {
            tmem_ld8(d_re + (il + 1) * kZuNB, nr);
            tmem_ld8(d_im + (il + 1) * kZuNB, ni);
          }
          if (np_ok) {
            const long long rowh = (long long)(I0 + il) * out.kpad * 2;              // halves
            __half* h0 = out.hl + rowh;
            __half* h1 = h0 + out.oplane;
            __half* g0 = reinterpret_cast<__half*>(out.hb8) + rowh;
            __half* g1 = g0 + out.oplane;
            unsigned char* b0 = out.hb8 + 2 * rowh;
            unsigned char* b1 = b0 + 2 * out.oplane;
#pragma unroll
            for (int n = 0; n < kZuNB; ++n) {
              if (n < nb) {
                const float x = __uint_as_float(vr[n]), y = __uint_as_float(vi[n]);
                const __half hx = __float2half_rn(x), hy = __float2half_rn(y);
                const float rx = x - __half2float(hx), ry = y - __half2float(hy);
                const uint32_t o = off[n];
                h0[o] = hx;
                h0[o + 32] = __float2half_rn(rx);
                h1[o] = hy;
                h1[o + 32] = __float2half_rn(ry);
                if (out.hb8) {
                  g0[o] = hx;
                  g1[o] = hy;
                  const uint32_t ob = 2u * o - lo[n];                                // bytes: 2 (stage start) + lo
                  b0[ob + 64] = (unsigned char)__nv_cvt_float_to_fp8(x, __NV_SATFINITE, __NV_E5M2);
                  b0[ob + 96] = (unsigned char)__nv_cvt_float_to_fp8(rx, __NV_SATFINITE, __NV_E5M2);
                  b1[ob + 64] = (unsigned char)__nv_cvt_float_to_fp8(y, __NV_SATFINITE, __NV_E5M2);
                  b1[ob + 96] = (unsigned char)__nv_cvt_float_to_fp8(ry, __NV_SATFINITE, __NV_E5M2);
                }
              }
            }
          }
        }
        tc_fence_before();
        __syncwarp();
        if (lane == 0) mbar_arrive(d_empty);
      }
    }
    a_use += n_mt;
    d_use += n_mt;
    __syncthreads();          // every MMA of this segment has completed (the epilogue warps waited for the last tile): B may be rewritten
  }
  tc_fence_before();
  __syncthreads();
  if (warp == 1) tmem_dealloc(tbase, 256);
}

}  // namespace

cudaError_t launch_zmel_pnorm(const SiteTables& st, const double2* P, float* pmax, cudaStream_t s) {
  zu_pnorm_kernel<<<st.n_sites, 256, 0, s>>>(st, P, pmax);
  return cudaGetLastError();
}

bool zmel_umma_supported(int b_max) { return b_max <= kZuK; }

size_t zmel_umma_aop_halves(int n_sites, int n_u, int n_batch) {
  return (size_t)2 * n_batch * n_sites * (size_t)((n_u + 127) / 128 * 128) * 64;
}

cudaError_t zmel_umma_configure() {
  return cudaFuncSetAttribute(zmel_umma_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, ZuCfg::SMEM_BYTES);
}

cudaError_t launch_zmel_umma(const ZmelArgs& a, const float* pmax, float* cnorm, __half* aop, void* zhl, void* zhb8, int n_m_pad,
                             long long n_rows, cudaStream_t s) {
  const int n_u_pad = (a.n_u + 127) / 128 * 128;
  cudaError_t e = cudaMemsetAsync(cnorm, 0, sizeof(float) * 2 * a.st.n_sites * a.n_batch, s);
  if (e != cudaSuccess) return e;
  zu_cnorm_kernel<<<dim3((a.n_o + a.n_u + 7) / 8, a.n_batch), 256, 0, s>>>(a.st, a.Ck, a.ld_k, a.Ck_bs, a.n_begin, a.n_o, a.Ckq,
                                                                           a.ld_kq, a.Ckq_bs, a.np_begin, a.n_u, cnorm);
  const long long rows = (long long)a.n_batch * a.st.n_sites * n_u_pad;
  long long blocks = (rows * kZuK + 255) / 256;
  if (blocks > 148 * 16) blocks = 148 * 16;
  float2* scales = reinterpret_cast<float2*>(cnorm + (size_t)2 * a.st.n_sites * a.n_batch);
  zu_scale_kernel<<<a.n_batch, 32, 0, s>>>(a.st, pmax, cnorm, scales, a.zmax);
  ckq_to_hl16_kernel<<<(unsigned)blocks, 256, 0, s>>>(a.st, scales, a.Ckq, a.ld_kq, a.Ckq_bs, a.np_begin, a.n_u, n_u_pad,
                                                      a.n_batch, aop);
  if ((e = cudaGetLastError()) != cudaSuccess) return e;
  CUtensorMap tmap;
  if ((e = make_hl16_map(&tmap, aop, 64, rows, rows * 64)) != cudaSuccess) return e;
  dim3 grid(a.ncg, (a.n_o + kZuNB - 1) / kZuNB, a.n_batch);
  zmel_umma_kernel<<<grid, kZuThreads, ZuCfg::SMEM_BYTES, s>>>(tmap, a, scales, static_cast<__half*>(zhl),
                                                              static_cast<unsigned char*>(zhb8), n_m_pad, n_rows, n_u_pad);
  return cudaGetLastError();
}

}  // namespace qsgw
