// Stage (a) on the FP64 tensor pipe (DMMA.8x8x4): muffin-tin product-basis matrix elements, Eq. (8) with the
// eigenfunction expansion of Eq. (4), two-step contraction of Alg. 1 line 12.
//
// One CTA = one column group (16 product functions I) x NB bands n.
//   step 1 (CUDA cores, 7 % of the flops):  T[n][alpha][I] = sum_beta P[I,alpha,beta] C_k[beta,n]   -> shared memory
//   step 2 (DMMA):  z[n,n',I] = sum_alpha conj(C_kq[alpha,n']) T[n][alpha][I]
//       per warp a tile of 8 bands n' x 16 I x NB n:  D[n'][I] += A[n'][alpha] B[alpha][I]  with
//       A = conj(C_kq) read from global/L2 (reused for NB x 2 x 4 DMMAs), B = T from shared memory.
// A column group may straddle site boundaries: the segments are concatenated along the contraction index
// (segment s owns rows [koff_s, koff_s + pad4(b_s)) of T and is zero outside its own columns).
#include "kernels.h"
#include "ptx.cuh"

namespace qsgw {

namespace {

constexpr int kZdThreads = 256;
constexpr int kZdNBMax = 6;       // bands n per CTA: template parameter NB in 4..6, chosen per launch (fewest rounds)
constexpr int kZdRow = 20;        // doubles per T row (16 columns + 4 padding: conflict-free fragment loads)
constexpr int kZdMaxSeg = 16;     // a 16-column group touches at most 16 sites

template <int kZdNB>
__global__ void __launch_bounds__(kZdThreads, 2) zmel_dmma_kernel(ZmelArgs a) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  a.Ck += (long long)blockIdx.z * a.Ck_bs;               // k-point of this CTA
  a.Ckq += (long long)blockIdx.z * a.Ckq_bs;
  a.zws += (long long)blockIdx.z * a.z_bs * kCG;
  if (a.zmax) a.zmax += blockIdx.z;
  const int bmax = a.st.b_max, kt = a.kt;
  double* cs_re = reinterpret_cast<double*>(smem_raw);    // [NB][bmax]
  double* cs_im = cs_re + kZdNB * bmax;
  double* ts_re = cs_im + kZdNB * bmax;                   // [NB][kt][kZdRow]
  double* ts_im = ts_re + kZdNB * kt * kZdRow;
  __shared__ int seg_o0[kZdMaxSeg], seg_b[kZdMaxSeg], seg_koff[kZdMaxSeg];
  __shared__ int n_seg_s;

  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int g = lane >> 2, t = lane & 3;
  const int cg = blockIdx.x;
  const int n0 = blockIdx.y * kZdNB;
  const int nb = min(kZdNB, a.n_o - n0);
  const int I0 = cg * kCG;
  const int I1 = min(I0 + kCG, a.st.n_m);

  for (int i = tid; i < 2 * kZdNB * kt * kZdRow; i += kZdThreads) ts_re[i] = 0.0;   // ts_re and ts_im are adjacent

  // ---- step 1, segment by segment ----
  int I = I0, koff = 0, n_seg = 0;
  while (I < I1) {
    const int s = a.st.d_pb_site[I];
    const int seg_end = min(I1, a.st.d_pb_off[s + 1]);
    const int o0 = a.st.d_orb_off[s];
    const int b = a.st.d_orb_off[s + 1] - o0;
    const int m0 = a.st.d_pb_off[s];
    const double2* Ps = a.P + a.st.d_p_off[s];
    __syncthreads();                                       // zero fill / previous segment's readers of cs done
    for (int idx = tid; idx < kZdNB * b; idx += kZdThreads) {
      const int n = idx / b, beta = idx - n * b;
      double2 v = make_double2(0.0, 0.0);
      if (n < nb) v = a.Ck[(long long)(a.n_begin + n0 + n) * a.ld_k + o0 + beta];
      cs_re[n * bmax + beta] = v.x;
      cs_im[n * bmax + beta] = v.y;
    }
    if (tid == 0) {
      seg_o0[n_seg] = o0;
      seg_b[n_seg] = b;
      seg_koff[n_seg] = koff;
    }
    __syncthreads();
    const int nI = seg_end - I;
    for (int item = tid; item < nI * b; item += kZdThreads) {
      const int il = item / b, alpha = item - il * b;
      const double2* prow = Ps + ((long long)(I + il - m0) * b + alpha) * b;
      double ar[kZdNB], ai[kZdNB];
#pragma unroll
      for (int n = 0; n < kZdNB; ++n) ar[n] = ai[n] = 0.0;
      for (int beta = 0; beta < b; ++beta) {
        const double2 pd = prow[beta];
#pragma unroll
        for (int n = 0; n < kZdNB; ++n) {
          const double cr = cs_re[n * bmax + beta], ci = cs_im[n * bmax + beta];
          ar[n] += pd.x * cr - pd.y * ci;
          ai[n] += pd.x * ci + pd.y * cr;
        }
      }
      const int col = I + il - I0;
#pragma unroll
      for (int n = 0; n < kZdNB; ++n) {
        ts_re[(n * kt + koff + alpha) * kZdRow + col] = ar[n];
        ts_im[(n * kt + koff + alpha) * kZdRow + col] = ai[n];
      }
    }
    koff += (b + 3) & ~3;
    ++n_seg;
    I = seg_end;
  }
  if (tid == 0) n_seg_s = n_seg;
  __syncthreads();

  // ---- step 2: DMMA over tiles of 8 bands n' ----
  double* zx = a.zws;
  double* zy = zx + (long long)a.ncg * a.kpad * kCG;
  float zmx = 0.f;
  const int n_tiles = (a.n_u + 7) >> 3;
  for (int tile = warp; tile < n_tiles; tile += kZdThreads / 32) {
    const int np = tile * 8 + g;                           // this lane's A row
    const bool np_ok = np < a.n_u;
    const double2* cq = a.Ckq + (long long)(a.np_begin + (np_ok ? np : 0)) * a.ld_kq;
    double zr[kZdNB][2][2], zi[kZdNB][2][2];
#pragma unroll
    for (int n = 0; n < kZdNB; ++n)
#pragma unroll
      for (int nt = 0; nt < 2; ++nt) zr[n][nt][0] = zr[n][nt][1] = zi[n][nt][0] = zi[n][nt][1] = 0.0;
    for (int sg = 0; sg < n_seg_s; ++sg) {
      const int o0 = seg_o0[sg], b = seg_b[sg], ko = seg_koff[sg];
      const int nkk = (b + 3) >> 2;
      double2 c = make_double2(0.0, 0.0);
      if (np_ok && t < b) c = cq[o0 + t];
      for (int kk = 0; kk < nkk; ++kk) {
        const double cr = c.x, ci = c.y;
        const int an = 4 * (kk + 1) + t;                   // prefetch the next A fragment
        c = make_double2(0.0, 0.0);
        if (np_ok && kk + 1 < nkk && an < b) c = cq[o0 + an];
        const double* tr_p = ts_re + (ko + 4 * kk + t) * kZdRow + g;
        const double* ti_p = ts_im + (ko + 4 * kk + t) * kZdRow + g;
        const double nci = -ci;
#pragma unroll
        for (int n = 0; n < kZdNB; ++n)
#pragma unroll
          for (int nt = 0; nt < 2; ++nt) {
            const double tr = tr_p[n * kt * kZdRow + 8 * nt], ti = ti_p[n * kt * kZdRow + 8 * nt];
            dmma884(zr[n][nt][0], zr[n][nt][1], cr, tr);   // conj(c) t = (cr tr + ci ti) + i (cr ti - ci tr)
            dmma884(zr[n][nt][0], zr[n][nt][1], ci, ti);
            dmma884(zi[n][nt][0], zi[n][nt][1], cr, ti);
            dmma884(zi[n][nt][0], zi[n][nt][1], nci, tr);
          }
      }
    }
    if (np_ok) {
#pragma unroll
      for (int n = 0; n < kZdNB; ++n) {
        if (n < nb) {
          long long pair = (long long)(n0 + n) * a.n_u + np;
          if (a.row_map) pair = a.row_map[pair];
#pragma unroll
          for (int nt = 0; nt < 2; ++nt) {
            const long long off = ((long long)cg * a.kpad + pair) * kCG + 8 * nt + 2 * t;
            *reinterpret_cast<double2*>(zx + off) = make_double2(zr[n][nt][0], zr[n][nt][1]);
            *reinterpret_cast<double2*>(zy + off) = make_double2(zi[n][nt][0], zi[n][nt][1]);
            zmx = fmaxf(zmx, fmaxf(fmaxf(fabsf((float)zr[n][nt][0]), fabsf((float)zr[n][nt][1])),
                                   fmaxf(fabsf((float)zi[n][nt][0]), fabsf((float)zi[n][nt][1]))));
          }
        }
      }
    }
  }
  if (a.zmax) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) zmx = fmaxf(zmx, __shfl_xor_sync(0xffffffffu, zmx, o));
    if (lane == 0 && zmx > 0.f) atomicMax(reinterpret_cast<unsigned int*>(a.zmax), __float_as_uint(zmx));
  }
}

}  // namespace

// Shared memory the DMMA kernel needs for a contraction length kt (padded, summed over a column group's
// segments) at the largest band block; the caller falls back to the CUDA-core kernel when this exceeds the limit.
static size_t smem_for(int nb, int b_max, int kt) {
  return sizeof(double) * ((size_t)2 * nb * b_max + (size_t)2 * nb * kt * kZdRow);
}
size_t zmel_dmma_smem_bytes(int b_max, int kt) { return smem_for(kZdNBMax, b_max, kt); }

template <int NB>
static cudaError_t launch_nb(const ZmelArgs& a, cudaStream_t s) {
  const size_t smem = smem_for(NB, a.st.b_max, a.kt);
  static size_t configured[kMaxDevices] = {};      // the attribute is per device
  int dev = 0;
  cudaGetDevice(&dev);
  dev = dev < 0 || dev >= kMaxDevices ? 0 : dev;
  if (smem > 48 * 1024 && smem > configured[dev]) {
    cudaError_t e = cudaFuncSetAttribute(zmel_dmma_kernel<NB>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    configured[dev] = smem;
  }
  dim3 grid(a.ncg, (a.n_o + NB - 1) / NB, a.n_batch);
  zmel_dmma_kernel<NB><<<grid, kZdThreads, smem, s>>>(a);
  return cudaGetLastError();
}

cudaError_t launch_zmel_dmma(const ZmelArgs& a, cudaStream_t s) {
  // bands per CTA: the choice with the fewest rounds x bands (2 CTAs per SM when the shared memory allows)
  const int n_sm = a.n_sm;
  int best_nb = 4;
  long long best = -1;
  for (int nb = 4; nb <= kZdNBMax; ++nb) {
    const int per_sm = smem_for(nb, a.st.b_max, a.kt) <= 110 * 1024 ? 2 : 1;
    const long long ctas = (long long)a.ncg * ((a.n_o + nb - 1) / nb) * a.n_batch;
    const long long cost = ((ctas + (long long)n_sm * per_sm - 1) / ((long long)n_sm * per_sm)) * nb;
    if (best < 0 || cost < best) { best = cost; best_nb = nb; }
  }
  if (best_nb == 6) return launch_nb<6>(a, s);
  if (best_nb == 5) return launch_nb<5>(a, s);
  return launch_nb<4>(a, s);
}

}  // namespace qsgw
