// Stage (a): muffin-tin product-basis matrix elements (Eq. 8 with Eq. 4), plus
// the export/import of the z batch in the boundary layout and the pair-weight table (Eq. 14).
#include "kernels.h"

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
            const long long pair = (long long)(n0 + n) * a.n_u + np;
            const long long off = ((long long)cg * a.kpad + pair) * kCG + col;
            zx[off] = ar[n];
            zy[off] = ai[n];
          }
        }
      }
    }
    __syncthreads();
    I = seg_end;
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
                                const double2* __restrict__ in) {
  const long long total = n_pairs * n_m;
  const long long plane = (long long)ncg * kpad * kCG;
  for (long long e = blockIdx.x * (long long)blockDim.x + threadIdx.x; e < total;
       e += (long long)gridDim.x * blockDim.x) {
    const long long p = e / n_m;
    const int I = (int)(e - p * n_m);
    const long long off = ((long long)(I / kCG) * kpad + p) * kCG + (I % kCG);
    const double2 v = in[e];
    zws[off] = v.x;
    zws[plane + off] = v.y;
  }
}

// w_j(n,n') = -2 f_n (1-f_n') D / (D^2 + omega_j^2), D = eps_kq[n'] - eps_k[n]  (Eq. 14)
// kept iff f_n (1-f_n') > occ_tol; 0/0 -> 0; rows [n_pairs, n_pairs_padded) are zeroed.
__global__ void pair_weights_kernel(const double* __restrict__ eps_k, const double* __restrict__ f_k,
                                    const double* __restrict__ eps_kq, const double* __restrict__ f_kq,
                                    int n_o, int n_u, const double* __restrict__ omega, int n_freq,
                                    double occ_tol, double* __restrict__ wtab, long long kpad,
                                    long long n_pairs_padded) {
  const long long n_pairs = (long long)n_o * n_u;
  for (long long p = blockIdx.x * (long long)blockDim.x + threadIdx.x; p < n_pairs_padded;
       p += (long long)gridDim.x * blockDim.x) {
    double num = 0.0, d2 = 0.0;
    bool keep = false;
    if (p < n_pairs) {
      const int n = (int)(p / n_u), np = (int)(p - (long long)n * n_u);
      const double D = eps_kq[np] - eps_k[n];
      const double occ = f_k[n] * (1.0 - f_kq[np]);
      keep = occ > occ_tol;
      num = -2.0 * occ * D;
      d2 = D * D;
    }
    for (int j = 0; j < n_freq; ++j) {
      const double om = omega[j];
      const double den = d2 + om * om;
      wtab[(long long)j * kpad + p] = (keep && den != 0.0) ? num / den : 0.0;
    }
  }
}

}  // namespace

cudaError_t launch_zmel_f64(const ZmelArgs& a, cudaStream_t s) {
  const size_t smem = sizeof(double) * (2 * kZmelNB * a.st.b_max + 2 * kZmelNB * a.st.b_max * kCG);
  static size_t configured = 0;
  if (smem > 48 * 1024 && smem > configured) {
    cudaError_t e = cudaFuncSetAttribute(zmel_kernel<double>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                         (int)smem);
    if (e != cudaSuccess) return e;
    configured = smem;
  }
  dim3 grid(a.ncg, (a.n_o + kZmelNB - 1) / kZmelNB);
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
                            const double2* in, cudaStream_t s) {
  z_import_kernel<<<grid_for(n_pairs * n_m, 256), 256, 0, s>>>(zws, kpad, ncg, n_m, n_pairs, in);
  return cudaGetLastError();
}

cudaError_t launch_pair_weights(const double* eps_k, const double* f_k, const double* eps_kq,
                                const double* f_kq, int n_o, int n_u, const double* d_omega, int n_freq,
                                double occ_tol, double* wtab, long long kpad, long long n_pairs_padded,
                                cudaStream_t s) {
  pair_weights_kernel<<<grid_for(n_pairs_padded, 128), 128, 0, s>>>(eps_k, f_k, eps_kq, f_kq, n_o, n_u, d_omega,
                                                                   n_freq, occ_tol, wtab, kpad, n_pairs_padded);
  return cudaGetLastError();
}

}  // namespace qsgw
