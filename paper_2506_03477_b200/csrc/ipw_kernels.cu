// Interstitial-plane-wave (IPW) block of the matrix elements (Eqs. 4, 5, 8; DESIGN.md
// reading R21):
//   z[n, n', I] = sum_{alpha, beta} conj(Bkq[n', alpha]) theta(g_k[beta] - g_kq[alpha] - g_ipw[I]) Bk[n, beta]
// (per unit cell volume; theta = Fourier coefficients of the interstitial indicator, an input table on an integer box).
// The structured "product tensor" is gathered once per chunk of alpha into a dense complex128 matrix and the two
// contractions run on the FP64 tensor pipe (zgemm_tma_kernel), in the conjugated form the GEMM's operand modes allow:
//   A1[(alpha, I), beta] = conj(theta(g_k[beta] - g_kq[alpha] - g_ipw[I]))                       (gather)
//   C1[(alpha, I), n]    = sum_beta A1[(alpha, I), beta] conj(Bk[n, beta])       = conj(T)       (GEMM, A k-contig., B conj)
//   O[n', (I, n)]       += sum_alpha Bkq[n', alpha] C1[alpha, (I, n)]            = conj(z)       (GEMM, accumulates over chunks)
//   z_out[(n n_u + n') ld_z + I] = conj(O[n', (I, n)])                                           (finish)
#include "kernels.h"

namespace qsgw {

namespace {

__global__ void ipw_theta_gather_kernel(const double2* __restrict__ theta, int L0, int L1, int L2,
                                        const int* __restrict__ g_kq, const int* __restrict__ g_k,
                                        const int* __restrict__ g_ipw, int a0, int a_cnt, int n_ipw, int n_k,
                                        double2* __restrict__ out) {
  const long long total = (long long)a_cnt * n_ipw * n_k;
  const int e1 = 2 * L1 + 1, e2 = 2 * L2 + 1;
  for (long long e = blockIdx.x * (long long)blockDim.x + threadIdx.x; e < total; e += (long long)gridDim.x * blockDim.x) {
    const int b = (int)(e % n_k);
    const long long row = e / n_k;
    const int i = (int)(row % n_ipw), a = a0 + (int)(row / n_ipw);
    const int d0 = g_k[3 * b] - g_kq[3 * a] - g_ipw[3 * i] + L0;
    const int d1 = g_k[3 * b + 1] - g_kq[3 * a + 1] - g_ipw[3 * i + 1] + L1;
    const int d2 = g_k[3 * b + 2] - g_kq[3 * a + 2] - g_ipw[3 * i + 2] + L2;
    double2 v = make_double2(0.0, 0.0);
    if (d0 >= 0 && d0 <= 2 * L0 && d1 >= 0 && d1 <= 2 * L1 && d2 >= 0 && d2 <= 2 * L2) {
      v = theta[((long long)d0 * e1 + d1) * e2 + d2];
      v.y = -v.y;
    }
    out[e] = v;
  }
}

__global__ void ipw_finish_kernel(const double2* __restrict__ O, int n_o, int n_u, int n_ipw, double2* __restrict__ z,
                                  long long ld_z) {
  const long long total = (long long)n_o * n_u * n_ipw;
  for (long long e = blockIdx.x * (long long)blockDim.x + threadIdx.x; e < total; e += (long long)gridDim.x * blockDim.x) {
    const int i = (int)(e % n_ipw);
    const long long pr = e / n_ipw;
    const int np = (int)(pr % n_u), n = (int)(pr / n_u);
    double2 v = O[(long long)np * n_ipw * n_o + (long long)i * n_o + n];
    v.y = -v.y;
    z[pr * ld_z + i] = v;
  }
}

unsigned grid_of(long long total) {
  const long long b = (total + 255) / 256;
  return (unsigned)(b > 148 * 32 ? 148 * 32 : (b < 1 ? 1 : b));
}

}  // namespace

// alpha chunk: A1 + C1 of one chunk stay below `cap_bytes`
int ipw_alpha_chunk(int n_pw_kq, int n_pw_k, int n_ipw, int n_o, size_t cap_bytes) {
  const size_t per_alpha = sizeof(double2) * (size_t)n_ipw * ((size_t)n_pw_k + (size_t)n_o);
  long long c = (long long)(cap_bytes / (per_alpha ? per_alpha : 1));
  if (c < 1) c = 1;
  if (c > n_pw_kq) c = n_pw_kq;
  return (int)c;
}
size_t ipw_work_elems(int a_chunk, int n_pw_k, int n_ipw, int n_o, int n_u) {
  return (size_t)a_chunk * n_ipw * ((size_t)n_pw_k + n_o) + (size_t)n_u * n_ipw * n_o;
}

cudaError_t launch_zmel_ipw(const int L[3], const double2* theta, int n_pw_kq, const int* g_kq, int n_pw_k, const int* g_k,
                            int n_ipw, const int* g_ipw, const double2* Bk, long long ld_k, int n_o, const double2* Bkq,
                            long long ld_kq, int n_u, double2* z_out, long long ld_z, int a_chunk, double2* work,
                            cudaStream_t s) {
  double2* A1 = work;
  double2* C1 = A1 + (size_t)a_chunk * n_ipw * n_pw_k;
  double2* O = C1 + (size_t)a_chunk * n_ipw * n_o;
  for (int a0 = 0; a0 < n_pw_kq; a0 += a_chunk) {
    const int cnt = a_chunk < n_pw_kq - a0 ? a_chunk : n_pw_kq - a0;
    ipw_theta_gather_kernel<<<grid_of((long long)cnt * n_ipw * n_pw_k), 256, 0, s>>>(theta, L[0], L[1], L[2], g_kq, g_k, g_ipw,
                                                                                    a0, cnt, n_ipw, n_pw_k, A1);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return e;
    ZgemmArgs g1;
    g1.A = A1; g1.lda = n_pw_k; g1.sA = 0;
    g1.B = Bk; g1.ldb = ld_k; g1.sB = 0;
    g1.C = C1; g1.ldc = n_o; g1.sC = 0;
    g1.m = cnt * n_ipw; g1.n = n_o; g1.k = n_pw_k;
    e = launch_zgemm(true, true, g1, s);
    if (e != cudaSuccess) return e;
    ZgemmArgs g2;
    g2.A = Bkq + a0; g2.lda = ld_kq; g2.sA = 0;
    g2.B = C1; g2.ldb = (long long)n_ipw * n_o; g2.sB = 0;
    g2.C = O; g2.ldc = (long long)n_ipw * n_o; g2.sC = 0;
    g2.m = n_u; g2.n = n_ipw * n_o; g2.k = cnt;
    g2.beta_one = a0 > 0 ? 1 : 0;
    e = launch_zgemm(true, false, g2, s);
    if (e != cudaSuccess) return e;
  }
  ipw_finish_kernel<<<grid_of((long long)n_o * n_u * n_ipw), 256, 0, s>>>(O, n_o, n_u, n_ipw, z_out, ld_z);
  return cudaGetLastError();
}

}  // namespace qsgw
