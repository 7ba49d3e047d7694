// Stage (a): muffin-tin product-basis matrix elements (Eq. 8 with Eq. 4), plus
// the export/import of the z batch in the boundary layout and the pair-weight table (Eq. 14).
#include <cuda_fp16.h>
#include <cuda_fp8.h>

#include "kernels.h"
#include "ptx.cuh"

namespace qsgw {

namespace {

constexpr int kZmelThreads = 256;
constexpr int kZmelNB = 8;  // occupied-side bands per CTA (register accumulators per thread)

// One CTA = one column group (16 product functions) x kZmelNB bands n.
//   step 1 (Alg. 1 line 12, first contraction):  T[n][alpha][I] = sum_beta P[I,alpha,beta] C_k[beta,n]
//   step 2:  z[n,n',I] = sum_alpha conj(C_kq[alpha,n']) T[n][alpha][I]
// A column group may straddle a site boundary; the segments are processed one after the other.
template <typename T>
__global__ void __launch_bounds__(kZmelThreads) zmel_kernel(ZmelArgs a) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  a.Ck += (long long)blockIdx.z * a.Ck_bs;               // k-point of this CTA
  a.Ckq += (long long)blockIdx.z * a.Ckq_bs;
  a.zws += (long long)blockIdx.z * a.z_bs * kCG;
  if (a.zmax) a.zmax += blockIdx.z;
  const int bmax = a.st.b_max;
  T* cs_re = reinterpret_cast<T*>(smem_raw);              // [NB][bmax]
  T* cs_im = cs_re + kZmelNB * bmax;
  T* ts_re = cs_im + kZmelNB * bmax;                      // [NB][bmax][16]
  T* ts_im = ts_re + kZmelNB * bmax * kCG;

  const int tid = threadIdx.x;
  const int cg = blockIdx.x;
  const int n0 = blockIdx.y * kZmelNB;
  const int nb = min(kZmelNB, a.n_o - n0);
  const int I0 = cg * kCG;
  const int I1 = min(I0 + kCG, a.st.n_m);

  T* zx = reinterpret_cast<T*>(a.zws);
  const long long plane = (long long)a.ncg * a.kpad * kCG;
  T* zy = zx + plane;
  float zmx = 0.f;     // max |Re z|, |Im z| of this thread (FP16-split mixed mode: batch scale)

  int I = I0;
  while (I < I1) {
    const int s = a.st.d_pb_site[I];
    const int seg_end = min(I1, a.st.d_pb_off[s + 1]);
    const int o0 = a.st.d_orb_off[s];
    const int b = a.st.d_orb_off[s + 1] - o0;
    const int m0 = a.st.d_pb_off[s];
    const double2* Ps = a.P + a.st.d_p_off[s];

    for (int idx = tid; idx < kZmelNB * b; idx += kZmelThreads) {
      const int n = idx / b, beta = idx - n * b;
      double2 v = make_double2(0.0, 0.0);
      if (n < nb) v = a.Ck[(long long)(a.n_begin + n0 + n) * a.ld_k + o0 + beta];
      cs_re[n * bmax + beta] = (T)v.x;
      cs_im[n * bmax + beta] = (T)v.y;
    }
    __syncthreads();

    const int nI = seg_end - I;
    for (int item = tid; item < nI * b; item += kZmelThreads) {
      const int il = item / b, alpha = item - il * b;
      const double2* prow = Ps + ((long long)(I + il - m0) * b + alpha) * b;
      T ar[kZmelNB], ai[kZmelNB];
#pragma unroll
      for (int n = 0; n < kZmelNB; ++n) ar[n] = ai[n] = (T)0;
      for (int beta = 0; beta < b; ++beta) {
        const double2 pd = prow[beta];
        const T pr = (T)pd.x, pi = (T)pd.y;
#pragma unroll
        for (int n = 0; n < kZmelNB; ++n) {
          const T cr = cs_re[n * bmax + beta], ci = cs_im[n * bmax + beta];
          ar[n] += pr * cr - pi * ci;
          ai[n] += pr * ci + pi * cr;
        }
      }
      const int col = I + il - I0;
#pragma unroll
      for (int n = 0; n < kZmelNB; ++n) {
        ts_re[(n * bmax + alpha) * kCG + col] = ar[n];
        ts_im[(n * bmax + alpha) * kCG + col] = ai[n];
      }
    }
    __syncthreads();

    const int col = tid & (kCG - 1);
    if (col >= I - I0 && col < seg_end - I0) {
      for (int np = tid >> 4; np < a.n_u; np += kZmelThreads / kCG) {
        const double2* cq = a.Ckq + (long long)(a.np_begin + np) * a.ld_kq + o0;
        T ar[kZmelNB], ai[kZmelNB];
#pragma unroll
        for (int n = 0; n < kZmelNB; ++n) ar[n] = ai[n] = (T)0;
        for (int alpha = 0; alpha < b; ++alpha) {
          const double2 cd = cq[alpha];
          const T cr = (T)cd.x, ci = (T)cd.y;
#pragma unroll
          for (int n = 0; n < kZmelNB; ++n) {
            const T tr = ts_re[(n * bmax + alpha) * kCG + col];
            const T ti = ts_im[(n * bmax + alpha) * kCG + col];
            ar[n] += cr * tr + ci * ti;   // conj(c) * t
            ai[n] += cr * ti - ci * tr;
          }
        }
#pragma unroll
        for (int n = 0; n < kZmelNB; ++n) {
          if (n < nb) {
            long long pair = (long long)(n0 + n) * a.n_u + np;
            if (a.row_map) pair = a.row_map[pair];
            const long long off = ((long long)cg * a.kpad + pair) * kCG + col;
            zx[off] = ar[n];
            zy[off] = ai[n];
            zmx = fmaxf(zmx, fmaxf(fabsf((float)ar[n]), fabsf((float)ai[n])));
          }
        }
      }
    }
    __syncthreads();
    I = seg_end;
  }
  if (a.zmax) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) zmx = fmaxf(zmx, __shfl_xor_sync(0xffffffffu, zmx, o));
    if ((tid & 31) == 0 && zmx > 0.f) atomicMax(reinterpret_cast<unsigned int*>(a.zmax), __float_as_uint(zmx));
  }
}

__global__ void z_export_kernel(const double* __restrict__ zws, long long kpad, int ncg, int n_m,
                                long long n_pairs, double2* __restrict__ out) {
  const long long total = n_pairs * n_m;
  const long long plane = (long long)ncg * kpad * kCG;
  for (long long e = blockIdx.x * (long long)blockDim.x + threadIdx.x; e < total;
       e += (long long)gridDim.x * blockDim.x) {
    const long long p = e / n_m;
    const int I = (int)(e - p * n_m);
    const long long off = ((long long)(I / kCG) * kpad + p) * kCG + (I % kCG);
    out[e] = make_double2(zws[off], zws[plane + off]);
  }
}

__global__ void z_import_kernel(double* __restrict__ zws, long long kpad, int ncg, int n_m, long long n_pairs,
                                const double2* __restrict__ in, float* __restrict__ zmax) {
  const long long total = n_pairs * n_m;
  const long long plane = (long long)ncg * kpad * kCG;
  float zmx = 0.f;
  for (long long e = blockIdx.x * (long long)blockDim.x + threadIdx.x; e < total;
       e += (long long)gridDim.x * blockDim.x) {
    const long long p = e / n_m;
    const int I = (int)(e - p * n_m);
    const long long off = ((long long)(I / kCG) * kpad + p) * kCG + (I % kCG);
    const double2 v = in[e];
    zws[off] = v.x;
    zws[plane + off] = v.y;
    zmx = fmaxf(zmx, fmaxf(fabsf((float)v.x), fabsf((float)v.y)));
  }
  if (zmax) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) zmx = fmaxf(zmx, __shfl_xor_sync(0xffffffffu, zmx, o));
    if ((threadIdx.x & 31) == 0 && zmx > 0.f) atomicMax(reinterpret_cast<unsigned int*>(zmax), __float_as_uint(zmx));
  }
}

// w_j(n,n') = -2 f_n (1-f_n') D / (D^2 + omega_j^2), D = eps_kq[n'] - eps_k[n]  (Eq. 14)
// kept iff f_n (1-f_n') > occ_tol; 0/0 -> 0; rows [n_pairs, n_pairs_padded) are zeroed.
__global__ void pair_weights_kernel(const double* __restrict__ eps_k, const double* __restrict__ f_k,
                                    const double* __restrict__ eps_kq, const double* __restrict__ f_kq,
                                    int n_o, int n_u, const double* __restrict__ omega, int n_freq,
                                    double occ_tol, double* __restrict__ wtab, long long kpad,
                                    long long n_pairs_padded, const float* __restrict__ zmax) {
  const long long n_pairs = (long long)n_o * n_u;
  const int kb = blockIdx.y;                                // k-point of this block
  eps_k += (long long)kb * n_o;
  f_k += (long long)kb * n_o;
  eps_kq += (long long)kb * n_u;
  f_kq += (long long)kb * n_u;
  wtab += (long long)kb * n_pairs_padded;
  // FP16-split mixed mode: this batch's z is staged as z * 2^S, so its weights carry 2^(-2S) (exact)
  const double zfac = zmax ? exp2(-2.0 * (double)f16_scale_exp(zmax[kb])) : 1.0;
  for (long long p = blockIdx.x * (long long)blockDim.x + threadIdx.x; p < n_pairs_padded;
       p += (long long)gridDim.x * blockDim.x) {
    double num = 0.0, d2 = 0.0;
    bool keep = false;
    if (p < n_pairs) {
      const int n = (int)(p / n_u), np = (int)(p - (long long)n * n_u);
      const double D = eps_kq[np] - eps_k[n];
      const double occ = f_k[n] * (1.0 - f_kq[np]);
      keep = occ > occ_tol;
      num = -2.0 * occ * D * zfac;
      d2 = D * D;
    }
    for (int j = 0; j < n_freq; ++j) {
      const double om = omega[j];
      const double den = d2 + om * om;
      wtab[(long long)j * kpad + p] = (keep && den != 0.0) ? num / den : 0.0;
    }
  }
}

// Mixed mode, FP16 split: FP64 z batch (column-group layout) -> "hl16" planes (kernels.h): per product
// function I and 32-pair stage one 128-byte row  h[32] | l[32]  with v = fp32(z * 2^S), h = fp16(v),
// l = fp16(v - h);  S = f16_scale_exp(max |z| of the batch) keeps every h below 2^14.  One block = one column
// group (16 product functions) x 128 pairs, transposed through shared memory so that both the reads ([p][16]
// doubles) and the writes (consecutive pairs of one I) are coalesced; rows of pairs beyond the batch are zeros.
__global__ void __launch_bounds__(256) z_to_hl16_kernel(const double* __restrict__ zws, long long kpad, int ncg,
                                                        int n_m, long long n_pairs, __half* __restrict__ out,
                                                        unsigned char* __restrict__ out8, int n_m_pad,
                                                        const float* __restrict__ zmax, long long n_rows,
                                                        long long z_bs) {
  __shared__ float tx[kCG][129], ty[kCG][129];
  const int cg = blockIdx.y;
  zws += (long long)blockIdx.z * z_bs * kCG;                // batch of this block: workspace slot at pair offset b*z_bs
  out += (long long)blockIdx.z * (z_bs / kPairStage) * 64;
  if (out8) out8 += (long long)blockIdx.z * (z_bs / kPairStage) * 128;
  zmax += blockIdx.z;
  const long long p0 = (long long)blockIdx.x * 128;
  const long long plane = (long long)ncg * kpad * kCG;
  const double scale = exp2((double)f16_scale_exp(*zmax));
  const double* src = zws + ((long long)cg * kpad + p0) * kCG;
  for (int idx = threadIdx.x; idx < 128 * kCG; idx += 256) {
    const int pl = idx / kCG, col = idx % kCG;
    float x = 0.f, y = 0.f;
    if (p0 + pl < n_pairs) {
      x = (float)(src[idx] * scale);
      y = (float)(src[plane + idx] * scale);
    }
    tx[col][pl] = x;
    ty[col][pl] = y;
  }
  __syncthreads();
  const long long oplane = (long long)n_m_pad * kpad * 2;     // halves per plane
  for (int idx = threadIdx.x; idx < 128 * kCG; idx += 256) {
    const int col = idx / 128, pl = idx % 128;
    const int I = cg * kCG + col;
    if (I >= n_m || p0 + pl >= n_rows) continue;
    const float x = tx[col][pl], y = ty[col][pl];
    const __half hx = __float2half_rn(x), hy = __float2half_rn(y);
    const __half lx = __float2half_rn(x - __half2float(hx)), ly = __float2half_rn(y - __half2float(hy));
    const long long p = p0 + pl;
    const long long o = (long long)I * kpad * 2 + (p >> 5) * 64 + (p & 31);
    out[o] = hx;
    out[o + 32] = lx;
    out[oplane + o] = hy;
    out[oplane + o + 32] = ly;
    if (out8) {   // FP8-variant B rows: h[32] halves | e5m2(v)[32] | e5m2(v - h)[32]   (128 B per 32 pairs)
      const long long ob = 2 * ((long long)I * kpad * 2 + (p >> 5) * 64) + (p & 31);      // byte offset in plane
      unsigned char* bx = out8 + ob;
      unsigned char* by = out8 + 2 * oplane + ob;
      reinterpret_cast<__half*>(out8)[o] = hx;
      reinterpret_cast<__half*>(out8)[oplane + o] = hy;
      bx[64] = (unsigned char)__nv_cvt_float_to_fp8(x, __NV_SATFINITE, __NV_E5M2);
      bx[96] = (unsigned char)__nv_cvt_float_to_fp8(x - __half2float(hx), __NV_SATFINITE, __NV_E5M2);
      by[64] = (unsigned char)__nv_cvt_float_to_fp8(y, __NV_SATFINITE, __NV_E5M2);
      by[96] = (unsigned char)__nv_cvt_float_to_fp8(y - __half2float(hy), __NV_SATFINITE, __NV_E5M2);
    }
  }
}

__global__ void z_export_hl16_kernel(const __half* __restrict__ zhl, long long kpad, int n_m_pad, int n_m,
                                     long long n_pairs, const float* __restrict__ zmax, double2* __restrict__ out) {
  const long long total = n_pairs * n_m;
  const long long oplane = (long long)n_m_pad * kpad * 2;
  const double inv = exp2(-(double)f16_scale_exp(*zmax));
  for (long long e = blockIdx.x * (long long)blockDim.x + threadIdx.x; e < total;
       e += (long long)gridDim.x * blockDim.x) {
    const long long p = e / n_m;
    const int I = (int)(e - p * n_m);
    const long long o = (long long)I * kpad * 2 + (p >> 5) * 64 + (p & 31);
    const float x = __half2float(zhl[o]) + __half2float(zhl[o + 32]);
    const float y = __half2float(zhl[oplane + o]) + __half2float(zhl[oplane + o + 32]);
    out[e] = make_double2((double)x * inv, (double)y * inv);
  }
}

// Weights scaled per frequency into (1/2, 1] and split into fp16 pieces:  v = fp32(w_j(p) * sigma_j),
// sigma_j = 2^-e with max_p |w_j(p)| = m 2^e, m in [1/2, 1);  w_h = fp16(v), w_l = fp16(v - w_h), stored per
// 32-pair stage as  w_h[32] | w_l[32];  wscale[j] = 1 / sigma_j.  One block per frequency.
// The same pass decides which product variant the flush runs (kernels.h, MixedCtl): P_eff_j = (sum_p w_j)^2 /
// sum_p w_j^2 is the effective number of pairs summed per output element at frequency j; the last block to
// finish takes the minimum over j and sets ctl->use_fp8.
__global__ void __launch_bounds__(1024) weights_scale_hl16_kernel(const double* __restrict__ wtab,
                                                                  __half* __restrict__ w16, double* __restrict__ wscale,
                                                                  long long kpad, long long n_pad, MixedCtl* ctl,
                                                                  const float* __restrict__ zfold) {
  __shared__ double red[3][32];
  const int j = blockIdx.x;
  const double* wr = wtab + (long long)j * kpad;
  const double fold = zfold ? exp2(-2.0 * (double)f16_scale_exp(*zfold)) : 1.0;
  double m = 0.0, s1 = 0.0, s2 = 0.0;
  for (long long p = threadIdx.x; p < n_pad; p += blockDim.x) {
    const double w = wr[p] * fold;
    m = fmax(m, fabs(w));
    s1 += w;
    s2 += w * w;
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    m = fmax(m, __shfl_xor_sync(0xffffffffu, m, o));
    s1 += __shfl_xor_sync(0xffffffffu, s1, o);
    s2 += __shfl_xor_sync(0xffffffffu, s2, o);
  }
  if ((threadIdx.x & 31) == 0) {
    red[0][threadIdx.x >> 5] = m;
    red[1][threadIdx.x >> 5] = s1;
    red[2][threadIdx.x >> 5] = s2;
  }
  __syncthreads();
  m = red[0][0];
  s1 = red[1][0];
  s2 = red[2][0];
  for (int i = 1; i < (int)(blockDim.x >> 5); ++i) {
    m = fmax(m, red[0][i]);
    s1 += red[1][i];
    s2 += red[2][i];
  }
  int e = 0;
  if (m > 0.0 && m < 1e300) (void)frexp(m, &e);
  const double sigma = exp2((double)-e);
  if (threadIdx.x == 0) wscale[j] = exp2((double)e);
  __half* o = w16 + (long long)j * kpad * 2;
  for (long long p = threadIdx.x; p < n_pad; p += blockDim.x) {
    const float v = (float)(wr[p] * fold * sigma);
    const __half h = __float2half_rn(v);
    o[(p >> 5) * 64 + (p & 31)] = h;
    o[(p >> 5) * 64 + 32 + (p & 31)] = __float2half_rn(v - __half2float(h));
  }
  if (threadIdx.x == 0) {
    // all-zero rows (every pair dropped) do not constrain the choice
    if (s2 > 0.0) atomicMin(reinterpret_cast<unsigned int*>(&ctl->peff_min), __float_as_uint((float)(s1 * s1 / s2)));
    __threadfence();
    if (atomicAdd(&ctl->ticket, 1u) == gridDim.x - 1) {     // last block: every frequency has contributed
      __threadfence();
      const float pe = *reinterpret_cast<volatile float*>(&ctl->peff_min);
      const int use = ctl->mode == 1 || (ctl->mode == 2 && pe >= ctl->thr_pairs);
      ctl->use_fp8 = use;
      ctl->n_flush += 1;
      ctl->n_flush_fp8 += use ? 1 : 0;
      ctl->peff_min_seen = fminf(ctl->peff_min_seen, pe);
      ctl->peff_min = 3.0e38f;                               // re-armed for the next flush
      ctl->ticket = 0;
    }
  }
}

// one warp per 32-pair stage: does any pair of the stage carry a nonzero weight at any frequency?
__global__ void stage_flags_kernel(const double* __restrict__ wtab, long long kpad, int n_stages, int n_freq,
                                   unsigned char* __restrict__ flags) {
  const int st = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5), lane = threadIdx.x & 31;
  if (st >= n_stages) return;
  bool live = false;
  for (int j = 0; j < n_freq; ++j) live = live || wtab[(long long)j * kpad + (long long)st * 32 + lane] != 0.0;
  const unsigned any = __ballot_sync(0xffffffffu, live);
  if (lane == 0) flags[st] = any ? 1 : 0;
}

// one block: ascending list of the live stages and their number
__global__ void __launch_bounds__(1024) stage_compact_kernel(const unsigned char* __restrict__ flags, int n_stages,
                                                             int* __restrict__ live, int* __restrict__ n_live) {
  __shared__ int wsum[32];
  __shared__ int base_s;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  if (tid == 0) base_s = 0;
  __syncthreads();
  for (int s0 = 0; s0 < n_stages; s0 += 1024) {
    const int st = s0 + tid;
    const int f = st < n_stages ? flags[st] : 0;
    const unsigned m = __ballot_sync(0xffffffffu, f != 0);
    if (lane == 0) wsum[warp] = __popc(m);
    __syncthreads();
    int before = base_s;
    for (int w = 0; w < warp; ++w) before += wsum[w];
    if (f) live[before + __popc(m & ((1u << lane) - 1u))] = st;
    __syncthreads();
    if (tid == 0) {
      int tot = 0;
      for (int w = 0; w < 32; ++w) tot += wsum[w];
      base_s += tot;
    }
    __syncthreads();
  }
  if (tid == 0) *n_live = base_s;
}

}  // namespace

cudaError_t launch_zmel_f64(const ZmelArgs& a, cudaStream_t s) {
  const size_t smem = sizeof(double) * (2 * kZmelNB * a.st.b_max + 2 * kZmelNB * a.st.b_max * kCG);
  static size_t configured[kMaxDevices] = {};      // the attribute is per device
  int dev = 0;
  cudaGetDevice(&dev);
  dev = dev < 0 || dev >= kMaxDevices ? 0 : dev;
  if (smem > 48 * 1024 && smem > configured[dev]) {
    cudaError_t e = cudaFuncSetAttribute(zmel_kernel<double>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                         (int)smem);
    if (e != cudaSuccess) return e;
    configured[dev] = smem;
  }
  dim3 grid(a.ncg, (a.n_o + kZmelNB - 1) / kZmelNB, a.n_batch);
  zmel_kernel<double><<<grid, kZmelThreads, smem, s>>>(a);
  return cudaGetLastError();
}

static int grid_for(long long total, int threads) {
  long long b = (total + threads - 1) / threads;
  if (b < 1) b = 1;
  if (b > 148LL * 16) b = 148LL * 16;
  return (int)b;
}

cudaError_t launch_z_export(const double* zws, long long kpad, int ncg, int n_m, long long n_pairs,
                            double2* out, cudaStream_t s) {
  z_export_kernel<<<grid_for(n_pairs * n_m, 256), 256, 0, s>>>(zws, kpad, ncg, n_m, n_pairs, out);
  return cudaGetLastError();
}

cudaError_t launch_z_import(double* zws, long long kpad, int ncg, int n_m, long long n_pairs,
                            const double2* in, float* zmax, cudaStream_t s) {
  z_import_kernel<<<grid_for(n_pairs * n_m, 256), 256, 0, s>>>(zws, kpad, ncg, n_m, n_pairs, in, zmax);
  return cudaGetLastError();
}

cudaError_t launch_pair_weights(const double* eps_k, const double* f_k, const double* eps_kq,
                                const double* f_kq, int n_o, int n_u, const double* d_omega, int n_freq,
                                double occ_tol, double* wtab, long long kpad, long long n_pairs_padded,
                                const float* zmax, int n_batch, cudaStream_t s) {
  pair_weights_kernel<<<dim3(grid_for(n_pairs_padded, 128), n_batch), 128, 0, s>>>(eps_k, f_k, eps_kq, f_kq, n_o, n_u, d_omega,
                                                                   n_freq, occ_tol, wtab, kpad, n_pairs_padded, zmax);
  return cudaGetLastError();
}

cudaError_t launch_stage_compaction(const double* wtab, long long kpad, long long n_pad, int n_freq, unsigned char* flags,
                                    int* live, int* n_live, cudaStream_t s) {
  const int n_stages = (int)(n_pad / kPairStage);
  stage_flags_kernel<<<(n_stages + 7) / 8, 256, 0, s>>>(wtab, kpad, n_stages, n_freq, flags);
  stage_compact_kernel<<<1, 1024, 0, s>>>(flags, n_stages, live, n_live);
  return cudaGetLastError();
}

cudaError_t launch_z_to_hl16(const double* zws, long long kpad, int ncg, int n_m, long long n_pairs, void* zhl,
                             void* zhb8, int n_m_pad, const float* zmax, int n_batch, long long z_bs,
                             cudaStream_t s) {
  const long long n_rows = (n_pairs + kPairStage - 1) / kPairStage * kPairStage;   // this batch's padded rows
  dim3 grid((unsigned)((n_rows + 127) / 128), ncg, n_batch);
  z_to_hl16_kernel<<<grid, 256, 0, s>>>(zws, kpad, ncg, n_m, n_pairs, static_cast<__half*>(zhl),
                                        static_cast<unsigned char*>(zhb8), n_m_pad, zmax, n_rows, z_bs);
  return cudaGetLastError();
}

cudaError_t launch_z_export_hl16(const void* zhl, long long kpad, int n_m_pad, int n_m, long long n_pairs,
                                 const float* zmax, double2* out, cudaStream_t s) {
  z_export_hl16_kernel<<<grid_for(n_pairs * n_m, 256), 256, 0, s>>>(static_cast<const __half*>(zhl), kpad, n_m_pad,
                                                                   n_m, n_pairs, zmax, out);
  return cudaGetLastError();
}

cudaError_t launch_weights_scale_hl16(const double* wtab, void* wtab16, double* wscale, long long kpad, long long n_pad,
                                      int n_freq, MixedCtl* ctl, const float* zfold, cudaStream_t s) {
  weights_scale_hl16_kernel<<<n_freq, 1024, 0, s>>>(wtab, static_cast<__half*>(wtab16), wscale, kpad, n_pad, ctl, zfold);
  return cudaGetLastError();
}

}  // namespace qsgw
