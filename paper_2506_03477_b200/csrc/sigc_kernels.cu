// Imaginary-axis part of the correlation self-energy: I^c of Eq. (22) in the order of
// Alg. 2 lines 12-25 and 44.  This file holds the quadrature weights of Eq. (23) and the launch
// sequence; both GEMMs (ZW^c += Z_w^dagger x W^c over the frequencies, and the closing contraction with Z) run in
// zgemm_tma_kernel with the weights applied to the A fragments in registers (Alg. 2 line 18 without a Z_w array).
#include "kernels.h"

namespace qsgw {

namespace {

// w[i][p] = w^I(dE_p, i omega_i), p = n' * n_qp + n, dE = eps_q[n] - eps_qk[n']   (Eq. 23, reading R17):
//   int_{-inf}^{inf} d omega / 2 pi X(i omega) / (dE - i omega) = int_0^inf K(dE, omega) X(i omega) d omega for even X,
//   K = dE / (pi (dE^2 + omega^2)), integrated exactly against the piecewise-linear interpolant of X on the mesh
//   (X = 0 beyond the last point).  Per interval [a, b]:  I0 = (atan(b/dE) - atan(a/dE)) / pi,
//   I1 = dE / (2 pi) log((dE^2 + b^2) / (dE^2 + a^2));  left node += (b I0 - I1) / h,  right node += (I1 - a I0) / h.
// dE = 0 -> 0 (principal value of an odd integrand).  Rows [n_pairs, ld) are zeroed.
__global__ void sigc_weights_kernel(const double* __restrict__ eps_q, const double* __restrict__ eps_qk, int n_all,
                                    int n_qp, const double* __restrict__ omega, int n_freq, double* __restrict__ w,
                                    long long ld) {
  const long long n_pairs = (long long)n_all * n_qp;
  const double inv_pi = 0.31830988618379067154;
  for (long long p = blockIdx.x * (long long)blockDim.x + threadIdx.x; p < ld; p += (long long)gridDim.x * blockDim.x) {
    double d = 0.0;
    if (p < n_pairs) {
      const int np = (int)(p / n_qp), n = (int)(p - (long long)np * n_qp);
      d = eps_q[n] - eps_qk[np];
    }
    if (d == 0.0) {
      for (int i = 0; i < n_freq; ++i) w[(long long)i * ld + p] = 0.0;
      continue;
    }
    double carry = 0.0;                 // contribution of the interval to the left of node i
    double a = omega[0], at_a = atan(a / d);
    for (int i = 0; i + 1 < n_freq; ++i) {
      const double b = omega[i + 1], at_b = atan(b / d);
      const double h = b - a;
      const double I0 = (at_b - at_a) * inv_pi;
      const double I1 = d * (0.5 * inv_pi) * log((d * d + b * b) / (d * d + a * a));
      w[(long long)i * ld + p] = carry + (b * I0 - I1) / h;
      carry = (I1 - a * I0) / h;
      a = b;
      at_a = at_b;
    }
    w[(long long)(n_freq - 1) * ld + p] = carry;
  }
}

}  // namespace

cudaError_t launch_sigc_weights(const double* eps_q, const double* eps_qk, int n_all, int n_qp, const double* d_omega,
                                int n_freq, double* w, long long ld, cudaStream_t s) {
  const long long blocks = (ld + 127) / 128;
  sigc_weights_kernel<<<(unsigned)(blocks > 4096 ? 4096 : blocks), 128, 0, s>>>(eps_q, eps_qk, n_all, n_qp, d_omega, n_freq, w, ld);
  return cudaGetLastError();
}

// ZW^c[(n', n), nu] = sum_i w_i(n', n) sum_mu z[(n', n), mu] W^c_i[mu, nu]            (Alg. 2 lines 15-25)
// sigc[n, m] += -(1/N_k) sum_{n', nu} ZW^c[(n', n), nu] conj(z[(n', m), nu])          (Alg. 2 line 44, Eq. 22)
cudaError_t launch_sigc_imag(const double2* z, const double* w, long long ld_w, const double2* wc, int n_all, int n_qp,
                             int n_m, int n_freq, double inv_nk, double2* zw, double2* sigc, int n_sm, cudaStream_t s) {
  const long long pairs = (long long)n_all * n_qp;
  ZgemmArgs g;
  g.A = z; g.lda = n_m; g.sA = 0;
  g.B = wc; g.ldb = n_m; g.sB = 0; g.rB = (long long)n_m * n_m;
  g.C = zw; g.ldc = n_m; g.sC = 0;
  g.m = (int)pairs; g.n = n_m; g.k = n_m; g.reps = n_freq;
  g.row_scale = w; g.ld_scale = ld_w;
  cudaError_t e = launch_zgemm(true, false, g, s);
  if (e != cudaSuccess) return e;
  return launch_sigc_close(z, zw, n_all, n_qp, n_m, inv_nk, sigc, n_sm, s);
}

cudaError_t launch_sigc_close(const double2* z, const double2* zw, int n_all, int n_qp, int n_m, double inv_nk, double2* sigc,
                              int n_sm, cudaStream_t s) {
  ZgemmArgs c;
  c.A = zw; c.lda = n_m; c.rA = (long long)n_qp * n_m;
  c.B = z; c.ldb = n_m; c.rB = (long long)n_qp * n_m;
  c.sA = c.sB = c.sC = 0;
  c.C = sigc; c.ldc = n_qp;
  c.m = n_qp; c.n = n_qp; c.k = n_m; c.reps = n_all;
  c.alpha = -inv_nk; c.beta_one = 1;
  const int tiles = ((n_qp + 63) / 64) * ((n_qp + 63) / 64);
  int split = (2 * n_sm + tiles - 1) / tiles;
  if (split > n_all) split = n_all;
  c.split = split < 1 ? 1 : split;
  return launch_zgemm(true, true, c, s);
}

}  // namespace qsgw
