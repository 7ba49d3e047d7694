// Orthonormal mixed product basis that diagonalises the Coulomb matrix (Eq. 7):
//   sum_J (v_IJ - v_mu O_IJ) z_{mu J} = 0,  z^H O z = 1,  v_mu descending;  U[I, mu] = z_{mu I}.
// Hermitian-definite pencil -> standard problem -> Jacobi:
//   O = L L^H, X = L^-1 (launch_chol_inverse: blocked Cholesky + triangular inverse on the FP64 tensor pipe),
//   C = X v X^H (two zgemm_tma_kernel GEMMs),
//   C = Q diag(lambda) Q^H by the two-sided Jacobi method with the round-robin parallel ordering: in each of the N - 1
//   rounds of a sweep the N / 2 disjoint index pairs (p, q) each get the rotation that annihilates C[p, q], computed from
//   the matrix at the start of the round (jacobi_params_kernel), and every 2 x 2 block (rows of pair i) x (columns of pair j)
//   is updated by one thread as J_i^H B J_j, in place (each block has exactly one reader and writer); the eigenvector
//   accumulator Q (rows in pairs, identity row rotation) goes through the same kernel (jacobi_apply_kernel).
//   U = X^H Q with the columns ordered by descending eigenvalue (one more GEMM).
// A round streams C and Q once (2 x 16 N^2 bytes read + written): the method is HBM/L2-bound, ~10 sweeps; the blocked
// variant (2b x 2b subproblems in shared memory + GEMM updates) is the next step for this row.
#include "kernels.h"

namespace qsgw {

namespace {

// pair i of round r (N even, m = N - 1 rotating indices, index N - 1 fixed)
__device__ __forceinline__ void rr_pair(int i, int r, int N, int& p, int& q) {
  const int m = N - 1;
  if (i == 0) { p = r; q = N - 1; return; }
  p = r + i; if (p >= m) p -= m;
  q = r - i; if (q < 0) q += m;
}

// params[i] = (c, sigma.x, sigma.y, 0): J = [[c, sigma], [-conj(sigma), c]] diagonalises [[a, b], [conj(b), d]]
__global__ void jacobi_params_kernel(const double2* __restrict__ A, int N, int r, double4* __restrict__ params) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= N / 2) return;
  int p, q;
  rr_pair(i, r, N, p, q);
  const double a = A[(long long)p * N + p].x, d = A[(long long)q * N + q].x;
  const double2 b = A[(long long)p * N + q];
  const double ab = hypot(b.x, b.y);
  double c = 1.0, sx = 0.0, sy = 0.0;
  if (ab > 0.0) {
    const double tau = (d - a) / (2.0 * ab);
    const double t = (tau >= 0.0 ? 1.0 : -1.0) / (fabs(tau) + sqrt(1.0 + tau * tau));
    if (isfinite(t)) {
      c = 1.0 / sqrt(1.0 + t * t);
      const double s = t * c;
      sx = s * b.x / ab;
      sy = s * b.y / ab;
    }
  }
  params[i] = make_double4(c, sx, sy, 0.0);
}

__device__ __forceinline__ double2 cmul(double2 a, double2 b) { return make_double2(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x); }
__device__ __forceinline__ double2 cmulc(double2 a, double2 b) {   // a * conj(b)
  return make_double2(a.x * b.x + a.y * b.y, a.y * b.x - a.x * b.y);
}

__device__ __forceinline__ double2 ldcs2(const double2* p) {
  double2 v;
  asm volatile("ld.global.cs.v2.f64 {%0, %1}, [%2];" : "=d"(v.x), "=d"(v.y) : "l"(p));
  return v;
}
__device__ __forceinline__ void stcs2(double2* p, double2 v) {
  asm volatile("st.global.cs.v2.f64 [%0], {%1, %2};" ::"l"(p), "d"(v.x), "d"(v.y) : "memory");
}

// grid.y in [0, N/2): rows (p_i, q_i) of A with the row rotation J_i^H; grid.y in [N/2, N): rows (2k, 2k+1) of V, no row
// rotation.  Thread <-> column pair j: B <- J_i^H B J_j on the 2 x 2 block.
__global__ void __launch_bounds__(256) jacobi_apply_kernel(double2* __restrict__ A, double2* __restrict__ V, int N, int r,
                                                           const double4* __restrict__ params) {
  const int j = blockIdx.x * blockDim.x + threadIdx.x;
  const int half = N / 2;
  if (j >= half) return;
  int pj, qj;
  rr_pair(j, r, N, pj, qj);
  const double4 fj = params[j];
  const double cj = fj.x;
  const double2 sj = make_double2(fj.y, fj.z);
  double2* M;
  int p, q;
  double ci = 1.0;
  double2 si = make_double2(0.0, 0.0);
  if ((int)blockIdx.y < half) {
    M = A;
    rr_pair(blockIdx.y, r, N, p, q);
    const double4 fi = params[blockIdx.y];
    ci = fi.x;
    si = make_double2(fi.y, fi.z);
  } else {
    M = V;
    p = 2 * ((int)blockIdx.y - half);
    q = p + 1;
  }
  double2* rp = M + (long long)p * N;
  double2* rq = M + (long long)q * N;
  // Q is streamed (evict-first) so that C, which every round reads twice (parameters + update), stays in the 126 MB L2
  const bool stream = M == V;
  double2 bpp, bpq, bqp, bqq;
  if (stream) {
    bpp = ldcs2(rp + pj); bpq = ldcs2(rp + qj); bqp = ldcs2(rq + pj); bqq = ldcs2(rq + qj);
  } else {
    bpp = rp[pj]; bpq = rp[qj]; bqp = rq[pj]; bqq = rq[qj];
  }
  // rows: x_p = c b_p - sigma b_q,  x_q = conj(sigma) b_p + c b_q
  double2 t;
  t = cmul(si, bqp);  const double2 xpp = make_double2(ci * bpp.x - t.x, ci * bpp.y - t.y);
  t = cmul(si, bqq);  const double2 xpq = make_double2(ci * bpq.x - t.x, ci * bpq.y - t.y);
  t = cmulc(bpp, si); const double2 xqp = make_double2(t.x + ci * bqp.x, t.y + ci * bqp.y);      // conj(sigma) b_pp = b_pp conj(sigma)
  t = cmulc(bpq, si); const double2 xqq = make_double2(t.x + ci * bqq.x, t.y + ci * bqq.y);
  // columns: y_p = c x_p - conj(sigma_j) x_q,  y_q = sigma_j x_p + c x_q
  t = cmulc(xpq, sj); const double2 ypp = make_double2(cj * xpp.x - t.x, cj * xpp.y - t.y);
  t = cmul(xpp, sj);  const double2 ypq = make_double2(t.x + cj * xpq.x, t.y + cj * xpq.y);
  t = cmulc(xqq, sj); const double2 yqp = make_double2(cj * xqp.x - t.x, cj * xqp.y - t.y);
  t = cmul(xqp, sj);  const double2 yqq = make_double2(t.x + cj * xqq.x, t.y + cj * xqq.y);
  if (stream) {
    stcs2(rp + pj, ypp); stcs2(rp + qj, ypq); stcs2(rq + pj, yqp); stcs2(rq + qj, yqq);
  } else {
    rp[pj] = ypp; rp[qj] = ypq; rq[pj] = yqp; rq[qj] = yqq;
  }
}

// out[0] += sum of |off-diagonal|^2, out[1] += sum of |diagonal|^2
__global__ void jacobi_offnorm_kernel(const double2* __restrict__ A, int N, double* __restrict__ out) {
  double off = 0.0, dg = 0.0;
  const long long total = (long long)N * N;
  for (long long e = blockIdx.x * (long long)blockDim.x + threadIdx.x; e < total; e += (long long)gridDim.x * blockDim.x) {
    const double2 v = A[e];
    const double m2 = v.x * v.x + v.y * v.y;
    if (e / N == e % N) dg += m2; else off += m2;
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    off += __shfl_xor_sync(0xffffffffu, off, o);
    dg += __shfl_xor_sync(0xffffffffu, dg, o);
  }
  if ((threadIdx.x & 31) == 0) {
    atomicAdd(out, off);
    atomicAdd(out + 1, dg);
  }
}

// [n][n] -> [N][N], zero padded (`unit_pad`: ones on the padded diagonal); herm: element (i, j), i > j, taken as conj of (j, i)
__global__ void eig_pad_kernel(const double2* __restrict__ src, int n, int N, int unit_pad, double2* __restrict__ dst) {
  const long long total = (long long)N * N;
  for (long long e = blockIdx.x * (long long)blockDim.x + threadIdx.x; e < total; e += (long long)gridDim.x * blockDim.x) {
    const int i = (int)(e / N), j = (int)(e % N);
    double2 x = make_double2((unit_pad && i == j) ? 1.0 : 0.0, 0.0);
    if (i < n && j < n) {
      if (i == j) x = make_double2(src[(long long)i * n + i].x, 0.0);
      else if (i < j) x = src[(long long)i * n + j];
      else { x = src[(long long)j * n + i]; x.y = -x.y; }
    }
    dst[e] = x;
  }
}

__global__ void eig_identity_kernel(double2* __restrict__ V, int N) {
  const long long total = (long long)N * N;
  for (long long e = blockIdx.x * (long long)blockDim.x + threadIdx.x; e < total; e += (long long)gridDim.x * blockDim.x)
    V[e] = make_double2(e / N == e % N ? 1.0 : 0.0, 0.0);
}

__global__ void eig_diag_kernel(const double2* __restrict__ A, int N, int n, double* __restrict__ d) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) d[i] = A[(long long)i * N + i].x;
}

// Qs[:, mu] = V[:, perm[mu]] for mu < n, zero beyond
__global__ void eig_gather_kernel(const double2* __restrict__ V, const int* __restrict__ perm, int N, int n,
                                  double2* __restrict__ Qs) {
  const long long total = (long long)N * N;
  for (long long e = blockIdx.x * (long long)blockDim.x + threadIdx.x; e < total; e += (long long)gridDim.x * blockDim.x) {
    const int i = (int)(e / N), mu = (int)(e % N);
    Qs[e] = mu < n ? V[(long long)i * N + perm[mu]] : make_double2(0.0, 0.0);
  }
}

__global__ void eig_unpad_kernel(const double2* __restrict__ src, int n, int N, double2* __restrict__ dst) {
  const long long total = (long long)n * n;
  for (long long e = blockIdx.x * (long long)blockDim.x + threadIdx.x; e < total; e += (long long)gridDim.x * blockDim.x)
    dst[e] = src[(e / n) * N + (e % n)];
}

}  // namespace

size_t eig_work_elems(int n_m) {
  const size_t N = (size_t)(n_m + 63) / 64 * 64, nb = N / 64;
  return 4 * N * N + 64 * N + nb * 4096 + N;      // A/C, X, V/T, Q, Tbuf, Linv, params (double4 = 2 elements each, N/2 of them)
}

// Stage 1 (stream-ordered): C = X v X^H in work[0 .. N^2), X in work[N^2 ..), Q = identity in work[2 N^2 ..).
cudaError_t launch_eig_reduce(int n_m, const double2* v, const double2* O, double2* work, int* d_info, cudaStream_t s) {
  const int N = (n_m + 63) / 64 * 64;
  const long long sM = (long long)N * N;
  double2* Abuf = work;
  double2* Xbuf = Abuf + sM;
  double2* Vbuf = Xbuf + sM;
  double2* Qbuf = Vbuf + sM;
  double2* Tbuf = Qbuf + sM;
  double2* Linv = Tbuf + 64LL * N;
  eig_pad_kernel<<<592, 256, 0, s>>>(O, n_m, N, 1, Abuf);
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return e;
  if ((e = launch_chol_inverse(N, 1, Abuf, Xbuf, Tbuf, Linv, d_info, s)) != cudaSuccess) return e;
  eig_pad_kernel<<<592, 256, 0, s>>>(v, n_m, N, 0, Vbuf);
  if ((e = cudaGetLastError()) != cudaSuccess) return e;
  ZgemmArgs g;                                            // T = X v
  g.A = Xbuf; g.B = Vbuf; g.C = Qbuf; g.lda = g.ldb = g.ldc = N; g.sA = g.sB = g.sC = 0; g.m = g.n = g.k = N;
  if ((e = launch_zgemm(true, false, g, s)) != cudaSuccess) return e;
  ZgemmArgs h = g;                                        // C = T X^H
  h.A = Qbuf; h.B = Xbuf; h.C = Abuf;
  if ((e = launch_zgemm(true, true, h, s)) != cudaSuccess) return e;
  eig_pad_kernel<<<592, 256, 0, s>>>(Abuf, N, N, 0, Vbuf);   // exact Hermitian copy of C (upper triangle mirrored)
  if ((e = cudaGetLastError()) != cudaSuccess) return e;
  e = cudaMemcpyAsync(Abuf, Vbuf, sizeof(double2) * sM, cudaMemcpyDeviceToDevice, s);
  if (e != cudaSuccess) return e;
  eig_identity_kernel<<<592, 256, 0, s>>>(Vbuf, N);
  return cudaGetLastError();
}

// One Jacobi sweep over C (work[0..)) and Q (work[2 N^2 ..)); then norms[0] = |off|^2, norms[1] = |diag|^2.
cudaError_t launch_eig_sweep(int n_m, double2* work, double* d_norms, cudaStream_t s) {
  const int N = (n_m + 63) / 64 * 64;
  const long long sM = (long long)N * N;
  double2* Abuf = work;
  double2* Vbuf = work + 2 * sM;
  double4* params = reinterpret_cast<double4*>(work + 4 * sM + 64LL * N + (long long)(N / 64) * 4096);
  const int half = N / 2;
  const dim3 grid((half + 255) / 256, N);
  for (int r = 0; r < N - 1; ++r) {
    jacobi_params_kernel<<<(half + 127) / 128, 128, 0, s>>>(Abuf, N, r, params);
    jacobi_apply_kernel<<<grid, 256, 0, s>>>(Abuf, Vbuf, N, r, params);
  }
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return e;
  if ((e = cudaMemsetAsync(d_norms, 0, 2 * sizeof(double), s)) != cudaSuccess) return e;
  jacobi_offnorm_kernel<<<592, 256, 0, s>>>(Abuf, N, d_norms);
  return cudaGetLastError();
}

cudaError_t launch_eig_diag(int n_m, const double2* work, double* d_diag, cudaStream_t s) {
  const int N = (n_m + 63) / 64 * 64;
  eig_diag_kernel<<<(n_m + 127) / 128, 128, 0, s>>>(work, N, n_m, d_diag);
  return cudaGetLastError();
}

// U = X^H Q[:, perm] -> U_out [n][n]
cudaError_t launch_eig_finish(int n_m, double2* work, const int* d_perm, double2* U_out, cudaStream_t s) {
  const int N = (n_m + 63) / 64 * 64;
  const long long sM = (long long)N * N;
  double2* Abuf = work;
  double2* Xbuf = Abuf + sM;
  double2* Vbuf = Xbuf + sM;
  double2* Qbuf = Vbuf + sM;
  eig_gather_kernel<<<592, 256, 0, s>>>(Vbuf, d_perm, N, n_m, Qbuf);
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return e;
  ZgemmArgs g;                                            // U = X^H Qs
  g.A = Xbuf; g.B = Qbuf; g.C = Abuf; g.lda = g.ldb = g.ldc = N; g.sA = g.sB = g.sC = 0; g.m = g.n = g.k = N;
  if ((e = launch_zgemm(false, false, g, s)) != cudaSuccess) return e;
  eig_unpad_kernel<<<592, 256, 0, s>>>(Abuf, n_m, N, U_out);
  return cudaGetLastError();
}

}  // namespace qsgw
