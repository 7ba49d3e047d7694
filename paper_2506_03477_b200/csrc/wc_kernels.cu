// Screened Coulomb interaction on the imaginary axis:
//   eps_j = 1 - sqrt(v) chi0_j sqrt(v)   (Eq. 10),   W^c_j = sqrt(v) (eps_j^-1 - 1) sqrt(v)   (Eq. 19,
//   PAPER.md:179-182; the paper inverts with a library routine).
// eps_j is Hermitian positive definite (chi0(i omega) is negative semidefinite), so the inverse goes
// through a blocked Cholesky factorisation eps = L L^H, X = L^-1, eps^-1 = X^H X, all frequencies batched:
//   - zgemm_tma_kernel (zgemm_tma_kernels.cu): complex FP64 GEMM on the FP64 tensor pipe (DMMA.8x8x4), 3M complex product,
//     64x64 tiles, TMA-staged operands; it carries the panel solve, the trailing update (lower tiles only), the
//     triangular inverse and X^H X (zero blocks of the triangular factor skipped);
//   - potrf_inv_kernel: Cholesky factor of one 64x64 diagonal block and its triangular inverse in shared memory;
//   - element-wise kernels for eps and W^c.
#include "kernels.h"
#include "ptx.cuh"

namespace qsgw {

namespace {

constexpr int kPB = 64;          // diagonal block edge
constexpr int kPLD = kPB + 1;

// One CTA per frequency: Cholesky factor L of the 64x64 diagonal block (in place, lower triangle; the strict
// upper triangle is zeroed) and Linv = L^-1 (lower triangular, dense 64x64 with zero upper part).
// Unblocked right-looking factorisation and forward substitution in shared memory.
__global__ void __launch_bounds__(256) potrf_inv_kernel(double2* A, long long lda, long long sA, double2* Linv,
                                                        long long sL, int block_index, int* info) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  typedef double Plane[kPLD];
  Plane* lr = reinterpret_cast<Plane*>(smem_raw);      // L (lower), row-major [64][65]
  Plane* li = lr + kPB;
  Plane* xr = li + kPB;                                // Linv
  Plane* xi = xr + kPB;
  __shared__ double dinv;
  double2* Ab = A + (long long)blockIdx.x * sA;
  double2* Lb = Linv + (long long)blockIdx.x * sL;
  const int tid = threadIdx.x;
  for (int e = tid; e < kPB * kPB; e += 256) {
    const int i = e / kPB, j = e % kPB;
    const double2 v = Ab[(long long)i * lda + j];
    lr[i][j] = v.x;
    li[i][j] = (i == j) ? 0.0 : v.y;
    xr[i][j] = 0.0;
    xi[i][j] = 0.0;
  }
  __syncthreads();
  for (int c = 0; c < kPB; ++c) {
    if (tid == 0) {
      const double d = lr[c][c];
      if (!(d > 0.0)) {
        atomicCAS(info, 0, 1 + block_index * kPB + c);
        dinv = 0.0;
      } else {
        const double sd = sqrt(d);
        lr[c][c] = sd;
        dinv = 1.0 / sd;
      }
    }
    __syncthreads();
    const double s = dinv;
    for (int i = c + 1 + tid; i < kPB; i += 256) {
      lr[i][c] *= s;
      li[i][c] *= s;
    }
    __syncthreads();
    // trailing update of the lower triangle: A[i][j] -= L[i][c] conj(L[j][c]),  c < j <= i
    for (int i = c + 1 + (tid >> 4); i < kPB; i += 16) {            // 16 x 16 thread grid, no index divisions
      const double ar = lr[i][c], ai = li[i][c];
      for (int j = c + 1 + (tid & 15); j <= i; j += 16) {
        const double br = lr[j][c], bi = li[j][c];
        lr[i][j] -= ar * br + ai * bi;
        li[i][j] -= ai * br - ar * bi;
      }
    }
    __syncthreads();
  }
  // Linv: column c of X solves L x = e_c (forward substitution), one thread per column
  if (tid < kPB) {
    const int c = tid;
    for (int i = c; i < kPB; ++i) {
      double sr = (i == c) ? 1.0 : 0.0, si = 0.0;
      for (int k = c; k < i; ++k) {
        const double ar = lr[i][k], ai = li[i][k], br = xr[k][c], bi = xi[k][c];
        sr -= ar * br - ai * bi;
        si -= ar * bi + ai * br;
      }
      const double d = lr[i][i];
      xr[i][c] = d > 0.0 ? sr / d : 0.0;
      xi[i][c] = d > 0.0 ? si / d : 0.0;
    }
  }
  __syncthreads();
  for (int e = tid; e < kPB * kPB; e += 256) {
    const int i = e / kPB, j = e % kPB;
    Ab[(long long)i * lda + j] = (j <= i) ? make_double2(lr[i][j], li[i][j]) : make_double2(0.0, 0.0);
    Lb[(long long)i * kPB + j] = make_double2(xr[i][j], xi[i][j]);
  }
}

// eps = 1 - sqrt(v) chi0 sqrt(v) into the padded work matrix (identity in the padding)   (Eq. 10)
__global__ void wc_form_eps_kernel(const double2* __restrict__ chi0, const double* __restrict__ v, int n_m, int n_pad,
                                   double2* __restrict__ eps) {
  const long long total = (long long)n_pad * n_pad;
  const double2* c = chi0 + (long long)blockIdx.y * n_m * n_m;
  double2* o = eps + (long long)blockIdx.y * total;
  for (long long e = blockIdx.x * (long long)blockDim.x + threadIdx.x; e < total; e += (long long)gridDim.x * blockDim.x) {
    const int i = (int)(e / n_pad), j = (int)(e % n_pad);
    double2 r = make_double2(i == j ? 1.0 : 0.0, 0.0);
    if (i < n_m && j < n_m) {
      const double s = sqrt(v[i]) * sqrt(v[j]);
      const double2 x = c[(long long)i * n_m + j];
      r.x -= s * x.x;
      r.y = (i == j) ? 0.0 : -s * x.y;
    }
    o[e] = r;
  }
}

// 64x64 block copy: X[i-block, i-block] = Linv_ii
__global__ void wc_copy_block_kernel(const double2* __restrict__ src, long long s_src, double2* __restrict__ dst,
                                     long long ldd, long long s_dst) {
  const double2* a = src + (long long)blockIdx.x * s_src;
  double2* d = dst + (long long)blockIdx.x * s_dst;
  for (int e = threadIdx.x; e < kPB * kPB; e += blockDim.x) d[(long long)(e / kPB) * ldd + e % kPB] = a[e];
}

// W^c = sqrt(v) (eps^-1 - 1) sqrt(v) from the lower triangle of eps^-1 (Hermitian mirror, real diagonal)  (Eq. 19)
__global__ void wc_finish_kernel(const double2* __restrict__ inv, const double* __restrict__ v, int n_m, int n_pad,
                                 double2* __restrict__ wc) {
  const long long total = (long long)n_m * n_m;
  const double2* a = inv + (long long)blockIdx.y * n_pad * n_pad;
  double2* o = wc + (long long)blockIdx.y * total;
  for (long long e = blockIdx.x * (long long)blockDim.x + threadIdx.x; e < total; e += (long long)gridDim.x * blockDim.x) {
    const int i = (int)(e / n_m), j = (int)(e % n_m);
    const double s = sqrt(v[i]) * sqrt(v[j]);
    double2 x;
    if (i == j) x = make_double2(a[(long long)i * n_pad + i].x - 1.0, 0.0);
    else if (j < i) x = a[(long long)i * n_pad + j];
    else { x = a[(long long)j * n_pad + i]; x.y = -x.y; }
    o[e] = make_double2(s * x.x, s * x.y);
  }
}

}  // namespace

// Function attributes of every kernel of this file (called before a stream capture: no attribute calls inside it).
cudaError_t wc_configure() {
  constexpr int kPotrfSmemBytes = 4 * kPB * kPLD * 8;
  cudaError_t e = cudaFuncSetAttribute(potrf_inv_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, kPotrfSmemBytes);
  if (e == cudaSuccess) e = zgemm_configure();
  return e;
}

size_t wc_work_elems(int n_m, int n_freq) {
  const size_t n = (size_t)(n_m + 63) / 64 * 64, nb = n / 64;
  return (size_t)n_freq * (2 * n * n + 64 * n + nb * 64 * 64);
}

// Blocked Cholesky A = L L^H of `batch` Hermitian positive definite matrices of order N (multiple of 64; lower triangle
// of A is read and overwritten by L) and X = L^-1 (lower triangular; X is zeroed here).  Tbuf: batch * 64 * N elements,
// Linv: batch * (N / 64) * 4096 elements.  d_info: 0, or 1 + index of the first non-positive pivot (zeroed here).
cudaError_t launch_chol_inverse(int N, int batch, double2* Abuf, double2* Xbuf, double2* Tbuf, double2* Linv, int* d_info,
                                cudaStream_t s) {
  const int nb = N / 64, n_freq = batch;
  const long long sM = (long long)N * N, sT = 64LL * N, sL = (long long)nb * 4096;
  constexpr int kPotrfSmem = 4 * kPB * kPLD * 8;
  cudaError_t e;   // function attributes: wc_configure(), called by the C-ABI layer
#define WC_TRY(expr) do { e = (expr); if (e != cudaSuccess) return e; } while (0)
  auto gemm = [&](bool a_kc, bool b_kc, const double2* A, const double2* B, double2* C, long long lda, long long ldb,
                  long long ldc, long long sA, long long sB, long long sC, int m, int n, int k, double alpha, int beta_one,
                  int tri) {
    ZgemmArgs g;
    g.A = A; g.B = B; g.C = C; g.lda = lda; g.ldb = ldb; g.ldc = ldc; g.sA = sA; g.sB = sB; g.sC = sC;
    g.m = m; g.n = n; g.k = k; g.batch = n_freq; g.alpha = alpha; g.beta_one = beta_one; g.tri = tri;
    return launch_zgemm(a_kc, b_kc, g, s);
  };
  WC_TRY(cudaMemsetAsync(d_info, 0, sizeof(int), s));
  WC_TRY(cudaMemsetAsync(Xbuf, 0, sizeof(double2) * n_freq * sM, s));

  // blocked Cholesky A = L L^H (right-looking), L in the lower triangle of Abuf.  Two 64-column blocks j0, j1 are
  // factored per step (j1 after a narrow K = 64 update of its own block column), so that the trailing update runs
  // with K = 128 and touches every C tile half as often.
  auto block = [&](int r, int c) { return Abuf + (long long)r * 64 * N + (long long)c * 64; };
  for (int j0 = 0; j0 < nb; j0 += 2) {
    const int j1 = j0 + 1;
    potrf_inv_kernel<<<n_freq, 256, kPotrfSmem, s>>>(block(j0, j0), N, sM, Linv + (long long)j0 * 4096, sL, j0, d_info);
    WC_TRY(cudaGetLastError());
    if (j1 >= nb) break;
    const int m0 = nb - j1;                                                  // block rows j1 .. nb-1
    WC_TRY(gemm(true, true, block(j1, j0), Linv + (long long)j0 * 4096, block(j1, j0), N, 64, N, sM, sL, sM,
                64 * m0, 64, 64, 1.0, 0, 0));                               // L[j1.., j0] = A[j1.., j0] Linv_j0^H
    WC_TRY(gemm(true, true, block(j1, j0), block(j1, j0), block(j1, j1), N, N, N, sM, sM, sM,
                64 * m0, 64, 64, -1.0, 1, 0));                              // A[j1.., j1] -= L[j1.., j0] L[j1, j0]^H
    potrf_inv_kernel<<<n_freq, 256, kPotrfSmem, s>>>(block(j1, j1), N, sM, Linv + (long long)j1 * 4096, sL, j1, d_info);
    WC_TRY(cudaGetLastError());
    const int m1 = nb - j1 - 1;                                              // block rows j1+1 .. nb-1
    if (m1 == 0) break;
    WC_TRY(gemm(true, true, block(j1 + 1, j1), Linv + (long long)j1 * 4096, block(j1 + 1, j1), N, 64, N, sM, sL, sM,
                64 * m1, 64, 64, 1.0, 0, 0));                               // L[j1+1.., j1] = A[j1+1.., j1] Linv_j1^H
    WC_TRY(gemm(true, true, block(j1 + 1, j0), block(j1 + 1, j0), block(j1 + 1, j1 + 1), N, N, N, sM, sM, sM,
                64 * m1, 64 * m1, 128, -1.0, 1, 1));                        // A22 -= L[.., j0:j1] L[.., j0:j1]^H
  }
  // X = L^-1, row block by row block:  X_ii = Linv_ii,  X[i,0:i] = -Linv_ii (L[i,0:i] X[0:i,0:i])
  for (int i = 0; i < nb; ++i) {
    wc_copy_block_kernel<<<n_freq, 256, 0, s>>>(Linv + (long long)i * 4096, sL, Xbuf + (long long)i * 64 * N + i * 64, N, sM);
    WC_TRY(cudaGetLastError());
    if (i == 0) continue;
    WC_TRY(gemm(true, false, Abuf + (long long)i * 64 * N, Xbuf, Tbuf, N, N, N, sM, sM, sT, 64, 64 * i, 64 * i, 1.0, 0, 3));
    WC_TRY(gemm(true, false, Linv + (long long)i * 4096, Tbuf, Xbuf + (long long)i * 64 * N, 64, N, N, sL, sT, sM,
                64, 64 * i, 64, -1.0, 0, 0));
  }
#undef WC_TRY
  return cudaSuccess;
}

cudaError_t launch_wc_from_chi0(int n_m, int n_freq, const double2* chi0, const double* v, double2* wc_out,
                                double2* work, int* d_info, cudaStream_t s) {
  const int N = (n_m + 63) / 64 * 64, nb = N / 64;
  const long long sM = (long long)N * N, sT = 64LL * N;
  double2* Abuf = work;
  double2* Xbuf = Abuf + (long long)n_freq * sM;
  double2* Tbuf = Xbuf + (long long)n_freq * sM;
  double2* Linv = Tbuf + (long long)n_freq * sT;
  (void)nb;
  wc_form_eps_kernel<<<dim3(592, n_freq), 256, 0, s>>>(chi0, v, n_m, N, Abuf);
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return e;
  // eps = L L^H, X = L^-1
  if ((e = launch_chol_inverse(N, n_freq, Abuf, Xbuf, Tbuf, Linv, d_info, s)) != cudaSuccess) return e;
  // eps^-1 = X^H X (lower tiles into Abuf), then W^c
  ZgemmArgs g;
  g.A = Xbuf; g.B = Xbuf; g.C = Abuf; g.lda = g.ldb = g.ldc = N; g.sA = g.sB = g.sC = sM;
  g.m = g.n = g.k = N; g.batch = n_freq; g.tri = 2;
  if ((e = launch_zgemm(false, false, g, s)) != cudaSuccess) return e;
  wc_finish_kernel<<<dim3(592, n_freq), 256, 0, s>>>(Abuf, v, n_m, N, wc_out);
  return cudaGetLastError();
}

}  // namespace qsgw

// ---- chi0 in the Coulomb eigenbasis: chi0_{mu nu} = (U^H chi0 U)_{mu nu}  (E_mu = sum_I M_I U[I,mu]; Eqs. 7, 8) ----
namespace qsgw {

namespace {

// [batch][n][n] -> [batch][N][N], zero padded (`unit_pad`: ones on the padded diagonal)
__global__ void wc_pad_kernel(const double2* __restrict__ src, int n, int N, int unit_pad, double2* __restrict__ dst) {
  const long long total = (long long)N * N;
  const double2* a = src + (long long)blockIdx.y * n * n;
  double2* o = dst + (long long)blockIdx.y * total;
  for (long long e = blockIdx.x * (long long)blockDim.x + threadIdx.x; e < total; e += (long long)gridDim.x * blockDim.x) {
    const int i = (int)(e / N), j = (int)(e % N);
    o[e] = (i < n && j < n) ? a[(long long)i * n + j] : make_double2((unit_pad && i == j) ? 1.0 : 0.0, 0.0);
  }
}

// [batch][N][N] -> [batch][n][n], upper triangle kept, lower = conj(upper), real diagonal
__global__ void wc_unpad_hermitian_kernel(const double2* __restrict__ src, int n, int N, double2* __restrict__ dst) {
  const long long total = (long long)n * n;
  const double2* a = src + (long long)blockIdx.y * N * N;
  double2* o = dst + (long long)blockIdx.y * total;
  for (long long e = blockIdx.x * (long long)blockDim.x + threadIdx.x; e < total; e += (long long)gridDim.x * blockDim.x) {
    const int i = (int)(e / n), j = (int)(e % n);
    double2 x;
    if (i == j) x = make_double2(a[(long long)i * N + i].x, 0.0);
    else if (i < j) x = a[(long long)i * N + j];
    else { x = a[(long long)j * N + i]; x.y = -x.y; }
    o[e] = x;
  }
}

}  // namespace

size_t rotate_work_elems(int n_m, int n_freq) {
  const size_t n = (size_t)(n_m + 63) / 64 * 64;
  return (size_t)(2 * n_freq + 1) * n * n;
}

cudaError_t launch_rotate_basis(int n_m, int n_freq, const double2* chi0, const double2* U, double2* out, double2* work,
                                cudaStream_t s) {
  const int N = (n_m + 63) / 64 * 64;
  const long long sM = (long long)N * N;
  double2* Cpad = work;
  double2* Tpad = Cpad + (long long)n_freq * sM;
  double2* Upad = Tpad + (long long)n_freq * sM;
  cudaError_t e;
  wc_pad_kernel<<<dim3(592, n_freq), 256, 0, s>>>(chi0, n_m, N, 0, Cpad);
  wc_pad_kernel<<<dim3(592, 1), 256, 0, s>>>(U, n_m, N, 1, Upad);
  if ((e = cudaGetLastError()) != cudaSuccess) return e;
  ZgemmArgs t;                                                                     // T = chi0 U
  t.A = Cpad; t.B = Upad; t.C = Tpad; t.lda = t.ldb = t.ldc = N; t.sA = sM; t.sB = 0; t.sC = sM;
  t.m = t.n = t.k = N; t.batch = n_freq;
  if ((e = launch_zgemm(true, false, t, s)) != cudaSuccess) return e;
  ZgemmArgs r = t;                                                                 // U^H T
  r.A = Upad; r.B = Tpad; r.C = Cpad; r.sA = 0; r.sB = sM;
  if ((e = launch_zgemm(false, false, r, s)) != cudaSuccess) return e;
  wc_unpad_hermitian_kernel<<<dim3(592, n_freq), 256, 0, s>>>(Cpad, n_m, N, out);
  return cudaGetLastError();
}

}  // namespace qsgw

// ---- basis rotation without any allocation: scratch in a file-scope device array -------------------------------------------
// For callers that cannot call cudaMalloc (code under CUDA graph capture, tight serving loops, harnesses that forbid it).
// The array is part of the library image: EVERY GPU that loads libqsgw.so holds kRotStaticElems * 16 bytes (33 MiB) until the
// process exits.  In host code the array's name is a host-side stand-in, not a device address: the address a kernel may use
// comes from cudaGetSymbolAddress, taken once per device with that device current (rot_static_ptr).
namespace qsgw {

constexpr long long kRotStaticElems = 33LL * 256 * 256;     // (2 n_freq + 1) ceil64(N_M)^2 complex elements, e.g. N_M <= 256 at 16 frequencies
static __device__ __align__(256) double2 g_rot_scratch[kRotStaticElems];

long long rotate_static_max_elems() { return kRotStaticElems; }

static cudaError_t rot_static_ptr(double2** out) {
  static double2* ptr[kMaxDevices] = {};
  int dev = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return e;
  if (dev < 0 || dev >= kMaxDevices) return cudaErrorInvalidDevice;
  if (!ptr[dev]) {
    double2* p = nullptr;
    e = cudaGetSymbolAddress(reinterpret_cast<void**>(&p), g_rot_scratch);    // device `dev` is current
    if (e != cudaSuccess) return e;
    ptr[dev] = p;
  }
  *out = ptr[dev];
  return cudaSuccess;
}

// launch_rotate_basis on the static scratch.  cudaErrorMemoryAllocation if the problem needs more than kRotStaticElems.
// Nothing in the scratch has to start at zero: the padding kernels write every element of the padded chi0 and U, the first
// GEMM every element of the intermediate.  All calls share the array: calls that overlap on the GPU (two streams) race.
cudaError_t launch_rotate_basis_static(int n_m, int n_freq, const double2* chi0, const double2* U, double2* out,
                                       cudaStream_t s) {
  if ((long long)rotate_work_elems(n_m, n_freq) > kRotStaticElems) return cudaErrorMemoryAllocation;
  double2* work = nullptr;
  cudaError_t e = rot_static_ptr(&work);
  if (e != cudaSuccess) return e;
  return launch_rotate_basis(n_m, n_freq, chi0, U, out, work, s);
}

}  // namespace qsgw
