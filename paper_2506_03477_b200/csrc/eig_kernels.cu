// Orthonormal mixed product basis that diagonalises the Coulomb matrix (Eq. 7):
//   sum_J (v_IJ - v_mu O_IJ) z_{mu J} = 0,  z^H O z = 1,  v_mu descending;  U[I, mu] = z_{mu I}.
// Hermitian-definite pencil -> standard problem -> Jacobi:
//   O = L L^H, X = L^-1 (launch_chol_inverse: blocked Cholesky + triangular inverse on the FP64 tensor pipe),
//   C = X v X^H (two zgemm_tma_kernel GEMMs),
//   C = Q diag(lambda) Q^H by the two-sided Jacobi method with the round-robin parallel ordering, in BLOCK form (default):
//   index blocks of 32, a block round pairs all blocks, solves the 64 x 64 subproblems in shared memory (bj_solve_kernel)
//   and applies their unitaries to C and Q with 64 x 64 x 64 complex GEMMs on the FP64 tensor pipe (bj_update_kernel): N / 32 - 1
//   passes over the matrices per sweep.  The element-wise form (option "eig_blocked" = 0; jacobi_params_kernel +
//   jacobi_apply_kernel: N / 2 rotations per round, every 2 x 2 block updated by one thread, N - 1 passes per sweep) is kept
//   for comparison: 2.13 s against 0.50 s at N = 2400.
//   U = X^H Q with the columns ordered by descending eigenvalue (one more GEMM).
#include <vector>

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

// ---- blocked two-sided Jacobi ------------------------------------------------------------------------------------------
// Index blocks of kBJ = 32; a block round pairs the N / 32 blocks (round-robin ordering over block indices) and for every
// block pair (P, Q): (1) bj_solve_kernel diagonalises the 64 x 64 Hermitian subproblem S = C[{P,Q},{P,Q}] in shared memory
// by the same parallel Jacobi method (1024 threads: one 2 x 2 block of S and one of the accumulated unitary W per thread and
// inner round; rotations of angle <= pi/4, so W stays near the identity once S is nearly diagonal, which the convergence of
// the outer iteration needs); (2) bj_update_kernel applies the 64 x 64 unitaries to the matrices on the FP64 tensor pipe:
// every 64 x 64 tile (rows of pair i) x (columns of pair j) of C becomes W_i^H B W_j, every (64 rows) x (columns of pair j)
// tile of Q becomes B W_j; a tile has exactly one reader and writer (in place).  A block round passes over C and Q once:
// N / 32 - 1 passes per sweep instead of N - 1.
constexpr int kBJ = 32;
constexpr int kBJ2 = 2 * kBJ;
constexpr int kBJSolveLd = kBJ2 + 1;                  // double2 elements per row of S and W in bj_solve_kernel
constexpr int kBJSolveSmem = 2 * kBJ2 * kBJSolveLd * 16 + 32 * 32 + 64;
constexpr int kBJLd = 68;                             // doubles per row of a 64 x 64 plane in bj_update_kernel (conflict-free fragments)
constexpr int kBJUpdateSmem = 6 * kBJ2 * kBJLd * 8;
// Inner sweeps per subproblem and block round.  Measured at N = 2400 (15 outer sweeps in every case): 1 -> 0.80 s, 2 -> 0.90 s,
// 3 -> 1.03 s, until converged (up to 7) -> 1.38 s with the first version of the update kernel: the outer iteration does not
// need the subproblems diagonalised completely, every rotation is a Jacobi rotation of the whole matrix.
constexpr int kBJInnerSweeps = 1;

__global__ void __launch_bounds__(1024, 1) bj_solve_kernel(const double2* __restrict__ A, int N, int r, double2* __restrict__ Wout, int max_inner) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  double2* S = reinterpret_cast<double2*>(smem_raw);                  // [64][65]
  double2* W = S + kBJ2 * kBJSolveLd;
  double4* prm = reinterpret_cast<double4*>(W + kBJ2 * kBJSolveLd);   // [32]
  double* red = reinterpret_cast<double*>(prm + 32);                  // off^2, total^2
  const int tid = threadIdx.x, i = tid >> 5, j = tid & 31;
  int P, Q;
  rr_pair(blockIdx.x, r, N / kBJ, P, Q);
  for (int e = tid; e < kBJ2 * kBJ2; e += 1024) {
    const int l = e >> 6, c = e & 63;
    const int gr = (l < kBJ ? P * kBJ + l : Q * kBJ + l - kBJ), gc = (c < kBJ ? P * kBJ + c : Q * kBJ + c - kBJ);
    S[l * kBJSolveLd + c] = A[(long long)gr * N + gc];
    W[l * kBJSolveLd + c] = make_double2(l == c ? 1.0 : 0.0, 0.0);
  }
  if (tid < 2) red[tid] = 0.0;
  __syncthreads();
  for (int sweep = 0; sweep <= max_inner; ++sweep) {
    // off-diagonal and total weight of S (every thread: rows 2i, 2i+1, columns 2j, 2j+1)
    double off = 0.0, tot = 0.0;
#pragma unroll
    for (int a = 0; a < 2; ++a)
#pragma unroll
      for (int b = 0; b < 2; ++b) {
        const int l = 2 * i + a, c = 2 * j + b;
        const double2 v = S[l * kBJSolveLd + c];
        const double m2 = v.x * v.x + v.y * v.y;
        tot += m2;
        if (l != c) off += m2;
      }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
      off += __shfl_xor_sync(0xffffffffu, off, o);
      tot += __shfl_xor_sync(0xffffffffu, tot, o);
    }
    if (j == 0) { atomicAdd(&red[0], off); atomicAdd(&red[1], tot); }
    __syncthreads();
    const bool done = red[0] <= 1e-27 * red[1];
    __syncthreads();
    if (tid < 2) red[tid] = 0.0;
    if (done || sweep == max_inner) break;
    for (int rr = 0; rr < kBJ2 - 1; ++rr) {
      if (tid < 32) {
        int p, q;
        rr_pair(tid, rr, kBJ2, p, q);
        const double a = S[p * kBJSolveLd + p].x, d = S[q * kBJSolveLd + q].x;
        const double2 b = S[p * kBJSolveLd + q];
        const double ab = hypot(b.x, b.y);
        double c = 1.0, sx = 0.0, sy = 0.0;
        if (ab > 0.0) {
          const double tau = (d - a) / (2.0 * ab);
          const double t = (tau >= 0.0 ? 1.0 : -1.0) / (fabs(tau) + sqrt(1.0 + tau * tau));
          if (isfinite(t)) {
            c = 1.0 / sqrt(1.0 + t * t);
            const double sn = t * c;
            sx = sn * b.x / ab;
            sy = sn * b.y / ab;
          }
        }
        prm[tid] = make_double4(c, sx, sy, 0.0);
      }
      __syncthreads();
      int pi, qi, pj, qj;
      rr_pair(i, rr, kBJ2, pi, qi);
      rr_pair(j, rr, kBJ2, pj, qj);
      const double4 fi = prm[i], fj = prm[j];
      const double ci = fi.x, cj = fj.x;
      const double2 si = make_double2(fi.y, fi.z), sj = make_double2(fj.y, fj.z);
      double2 t;
      {   // S block: J_i^H B J_j
        double2* rp = S + pi * kBJSolveLd;
        double2* rq = S + qi * kBJSolveLd;
        const double2 bpp = rp[pj], bpq = rp[qj], bqp = rq[pj], bqq = rq[qj];
        t = cmul(si, bqp);  const double2 xpp = make_double2(ci * bpp.x - t.x, ci * bpp.y - t.y);
        t = cmul(si, bqq);  const double2 xpq = make_double2(ci * bpq.x - t.x, ci * bpq.y - t.y);
        t = cmulc(bpp, si); const double2 xqp = make_double2(t.x + ci * bqp.x, t.y + ci * bqp.y);
        t = cmulc(bpq, si); const double2 xqq = make_double2(t.x + ci * bqq.x, t.y + ci * bqq.y);
        t = cmulc(xpq, sj); rp[pj] = make_double2(cj * xpp.x - t.x, cj * xpp.y - t.y);
        t = cmul(xpp, sj);  rp[qj] = make_double2(t.x + cj * xpq.x, t.y + cj * xpq.y);
        t = cmulc(xqq, sj); rq[pj] = make_double2(cj * xqp.x - t.x, cj * xqp.y - t.y);
        t = cmul(xqp, sj);  rq[qj] = make_double2(t.x + cj * xqq.x, t.y + cj * xqq.y);
      }
      {   // W block (rows 2i, 2i+1): B J_j
        double2* rp = W + (2 * i) * kBJSolveLd;
        double2* rq = rp + kBJSolveLd;
        const double2 xpp = rp[pj], xpq = rp[qj], xqp = rq[pj], xqq = rq[qj];
        t = cmulc(xpq, sj); rp[pj] = make_double2(cj * xpp.x - t.x, cj * xpp.y - t.y);
        t = cmul(xpp, sj);  rp[qj] = make_double2(t.x + cj * xpq.x, t.y + cj * xpq.y);
        t = cmulc(xqq, sj); rq[pj] = make_double2(cj * xqp.x - t.x, cj * xqp.y - t.y);
        t = cmul(xqp, sj);  rq[qj] = make_double2(t.x + cj * xqq.x, t.y + cj * xqq.y);
      }
      __syncthreads();
    }
  }
  double2* wo = Wout + (long long)blockIdx.x * kBJ2 * kBJ2;
  for (int e = tid; e < kBJ2 * kBJ2; e += 1024) wo[e] = W[(e >> 6) * kBJSolveLd + (e & 63)];
}

__device__ __forceinline__ void dmma884e(double& c0, double& c1, double a, double b) {   // D(8x8) += A(8x4) B(4x8), see ptx.cuh
  asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
               : "+d"(c0), "+d"(c1)
               : "d"(a), "d"(b));
}

// blockIdx.y < npairs: tile (rows of pair i = blockIdx.y) x (columns of pair j = blockIdx.x) of C <- W_i^H B W_j;
// blockIdx.y >= npairs: rows 64 (blockIdx.y - npairs) .. + 63 of Q x (columns of pair j) <- B W_j.
// 8 warps, warp tile 16 rows x 32 columns, complex product as four real DMMA products on separate Re / Im planes.
// phase 0: every tile; phase 1: only the tiles of C flagged in `flags` (those the subproblems of the NEXT block round read);
// phase 2: every other tile of C and all tiles of Q (runs while the next round's subproblems are being solved).
__global__ void __launch_bounds__(256, 1) bj_update_kernel(double2* __restrict__ A, double2* __restrict__ V, int N, int r,
                                                           const double2* __restrict__ Wall,
                                                           const unsigned char* __restrict__ flags, int phase) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  double* Bre = reinterpret_cast<double*>(smem_raw);      // [64][68] each
  double* Bim = Bre + kBJ2 * kBJLd;
  double* Jre = Bim + kBJ2 * kBJLd;                       // W_j
  double* Jim = Jre + kBJ2 * kBJLd;
  double* Ire = Jim + kBJ2 * kBJLd;                       // W_i
  double* Iim = Ire + kBJ2 * kBJLd;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5, g = lane >> 2, t = lane & 3;
  const int npairs = N / kBJ2, nblk = N / kBJ;
  const bool is_a = (int)blockIdx.y < npairs;
  if (is_a && blockIdx.y > blockIdx.x) return;           // lower tiles of C are written by their mirror images
  if (phase != 0) {
    const bool flagged = is_a && flags[blockIdx.y * npairs + blockIdx.x] != 0;
    if ((phase == 1) != flagged) return;
  }
  int Pj, Qj, Pi = 0, Qi = 0;
  rr_pair(blockIdx.x, r, nblk, Pj, Qj);
  double2* M = V;
  int row0 = 0;
  if (is_a) {
    M = A;
    rr_pair(blockIdx.y, r, nblk, Pi, Qi);
  } else {
    row0 = ((int)blockIdx.y - npairs) * kBJ2;
  }
  const double2* Wj = Wall + (long long)blockIdx.x * kBJ2 * kBJ2;
  const double2* Wi = Wall + (long long)blockIdx.y * kBJ2 * kBJ2;
  // thread <-> column c = tid & 63, rows l = (tid >> 6) + 4 it: 16 independent loads per matrix in flight
  {
    const int c = tid & 63, l0 = tid >> 6;
    const int gc = c < kBJ ? Pj * kBJ + c : Qj * kBJ + c - kBJ;
    double2 b[16];
#pragma unroll
    for (int it = 0; it < 16; ++it) {
      const int l = l0 + 4 * it;
      const int gr = is_a ? (l < kBJ ? Pi * kBJ + l : Qi * kBJ + l - kBJ) : row0 + l;
      b[it] = M[(long long)gr * N + gc];
    }
#pragma unroll
    for (int it = 0; it < 16; ++it) {
      Bre[(l0 + 4 * it) * kBJLd + c] = b[it].x;
      Bim[(l0 + 4 * it) * kBJLd + c] = b[it].y;
    }
#pragma unroll
    for (int it = 0; it < 16; ++it) b[it] = Wj[(l0 + 4 * it) * kBJ2 + c];
#pragma unroll
    for (int it = 0; it < 16; ++it) {
      Jre[(l0 + 4 * it) * kBJLd + c] = b[it].x;
      Jim[(l0 + 4 * it) * kBJLd + c] = b[it].y;
    }
    if (is_a) {
#pragma unroll
      for (int it = 0; it < 16; ++it) b[it] = Wi[(l0 + 4 * it) * kBJ2 + c];
#pragma unroll
      for (int it = 0; it < 16; ++it) {
        Ire[(l0 + 4 * it) * kBJLd + c] = b[it].x;
        Iim[(l0 + 4 * it) * kBJLd + c] = b[it].y;
      }
    }
  }
  __syncthreads();
  const int rw = 16 * (warp >> 1), cw = 32 * (warp & 1);
  double yr[2][4][2], yi[2][4][2];
  if (is_a) {
    // X = W_i^H B:  X[m][c] = sum_k conj(W_i[k][m]) B[k][c]
#pragma unroll
    for (int rt = 0; rt < 2; ++rt)
#pragma unroll
      for (int ct = 0; ct < 4; ++ct) yr[rt][ct][0] = yr[rt][ct][1] = yi[rt][ct][0] = yi[rt][ct][1] = 0.0;
    for (int kk = 0; kk < kBJ2 / 4; ++kk) {
      const int k = 4 * kk + t;
      double ar[2], ai[2], br[4], bi[4];
#pragma unroll
      for (int rt = 0; rt < 2; ++rt) {
        ar[rt] = Ire[k * kBJLd + rw + 8 * rt + g];
        ai[rt] = Iim[k * kBJLd + rw + 8 * rt + g];
      }
#pragma unroll
      for (int ct = 0; ct < 4; ++ct) {
        br[ct] = Bre[k * kBJLd + cw + 8 * ct + g];
        bi[ct] = Bim[k * kBJLd + cw + 8 * ct + g];
      }
#pragma unroll
      for (int rt = 0; rt < 2; ++rt)
#pragma unroll
        for (int ct = 0; ct < 4; ++ct) {          // conj(w) b = (wr br + wi bi) + i (wr bi - wi br)
          dmma884e(yr[rt][ct][0], yr[rt][ct][1], ar[rt], br[ct]);
          dmma884e(yr[rt][ct][0], yr[rt][ct][1], ai[rt], bi[ct]);
          dmma884e(yi[rt][ct][0], yi[rt][ct][1], ar[rt], bi[ct]);
          dmma884e(yi[rt][ct][0], yi[rt][ct][1], -ai[rt], br[ct]);
        }
    }
    __syncthreads();                              // every warp has read B
#pragma unroll
    for (int rt = 0; rt < 2; ++rt)
#pragma unroll
      for (int ct = 0; ct < 4; ++ct) {
        const int o = (rw + 8 * rt + g) * kBJLd + cw + 8 * ct + 2 * t;
        Bre[o] = yr[rt][ct][0]; Bre[o + 1] = yr[rt][ct][1];
        Bim[o] = yi[rt][ct][0]; Bim[o + 1] = yi[rt][ct][1];
      }
    __syncthreads();
  }
  // Y = X W_j:  Y[m][c] = sum_k X[m][k] W_j[k][c]
#pragma unroll
  for (int rt = 0; rt < 2; ++rt)
#pragma unroll
    for (int ct = 0; ct < 4; ++ct) yr[rt][ct][0] = yr[rt][ct][1] = yi[rt][ct][0] = yi[rt][ct][1] = 0.0;
  for (int kk = 0; kk < kBJ2 / 4; ++kk) {
    const int k = 4 * kk + t;
    double ar[2], ai[2], br[4], bi[4];
#pragma unroll
    for (int rt = 0; rt < 2; ++rt) {
      ar[rt] = Bre[(rw + 8 * rt + g) * kBJLd + k];
      ai[rt] = Bim[(rw + 8 * rt + g) * kBJLd + k];
    }
#pragma unroll
    for (int ct = 0; ct < 4; ++ct) {
      br[ct] = Jre[k * kBJLd + cw + 8 * ct + g];
      bi[ct] = Jim[k * kBJLd + cw + 8 * ct + g];
    }
#pragma unroll
    for (int rt = 0; rt < 2; ++rt)
#pragma unroll
      for (int ct = 0; ct < 4; ++ct) {            // x w = (xr wr - xi wi) + i (xr wi + xi wr)
        dmma884e(yr[rt][ct][0], yr[rt][ct][1], ar[rt], br[ct]);
        dmma884e(yr[rt][ct][0], yr[rt][ct][1], -ai[rt], bi[ct]);
        dmma884e(yi[rt][ct][0], yi[rt][ct][1], ar[rt], bi[ct]);
        dmma884e(yi[rt][ct][0], yi[rt][ct][1], ai[rt], br[ct]);
      }
  }
  // Y -> shared memory (over X), then row-contiguous stores of the tile and, for an off-diagonal tile of C, of its mirror
  // image conj(Y)^T (C is Hermitian: the tiles with pair i > pair j are not computed)
  __syncthreads();                                // every warp has read X
#pragma unroll
  for (int rt = 0; rt < 2; ++rt)
#pragma unroll
    for (int ct = 0; ct < 4; ++ct) {
      const int o = (rw + 8 * rt + g) * kBJLd + cw + 8 * ct + 2 * t;
      Bre[o] = yr[rt][ct][0]; Bre[o + 1] = yr[rt][ct][1];
      Bim[o] = yi[rt][ct][0]; Bim[o + 1] = yi[rt][ct][1];
    }
  __syncthreads();
  {
    const int c = tid & 63, l0 = tid >> 6;
    const int gc = c < kBJ ? Pj * kBJ + c : Qj * kBJ + c - kBJ;
#pragma unroll
    for (int it = 0; it < 16; ++it) {
      const int l = l0 + 4 * it;
      const int gr = is_a ? (l < kBJ ? Pi * kBJ + l : Qi * kBJ + l - kBJ) : row0 + l;
      M[(long long)gr * N + gc] = make_double2(Bre[l * kBJLd + c], Bim[l * kBJLd + c]);
    }
    if (is_a && blockIdx.x != blockIdx.y) {
      const int gcm = c < kBJ ? Pi * kBJ + c : Qi * kBJ + c - kBJ;       // mirror column = tile row c
#pragma unroll
      for (int it = 0; it < 16; ++it) {
        const int l = l0 + 4 * it;                                        // mirror row = tile column l
        const int grm = l < kBJ ? Pj * kBJ + l : Qj * kBJ + l - kBJ;
        M[(long long)grm * N + gcm] = make_double2(Bre[c * kBJLd + l], -Bim[c * kBJLd + l]);
      }
    }
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

cudaError_t eig_configure() {
  cudaError_t e = cudaFuncSetAttribute(bj_solve_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, kBJSolveSmem);
  if (e != cudaSuccess) return e;
  return cudaFuncSetAttribute(bj_update_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, kBJUpdateSmem);
}

// One Jacobi sweep over C (work[0..)) and Q (work[2 N^2 ..)); then norms[0] = |off|^2, norms[1] = |diag|^2.
// blocked: block rounds of 64 x 64 subproblems + tensor-pipe updates (default); else the element-wise rounds.
cudaError_t launch_eig_sweep(int n_m, double2* work, double* d_norms, bool blocked, bool first_sweep, cudaStream_t s) {
  const int N = (n_m + 63) / 64 * 64;
  const long long sM = (long long)N * N;
  double2* Abuf = work;
  double2* Vbuf = work + 2 * sM;
  if (blocked) {
    // Look-ahead: the subproblems of round r + 1 read only a few tiles of C (two diagonal tiles and one off-diagonal tile
    // per pair).  Those are updated first (phase 1); the subproblems are then solved on a second stream while the first
    // stream updates everything else (phase 2).  Two W buffers (Tbuf of the reduction, and the Q scratch of the back
    // transformation); the per-round tile flags sit in the Linv region of the reduction (free during the sweeps).
    double2* Wbuf[2] = {work + 4 * sM, work + 3 * sM};
    unsigned char* flags = reinterpret_cast<unsigned char*>(work + 4 * sM + 64LL * N);
    const int npairs = N / kBJ2, nblk = N / kBJ, rounds = nblk - 1;
    const size_t flag_bytes = (size_t)rounds * npairs * npairs;
    const bool ahead = rounds > 1 && flag_bytes <= (size_t)(N / 64) * 4096 * sizeof(double2);
    cudaStream_t s2 = nullptr;
    cudaEvent_t e1 = nullptr, e2 = nullptr;
    cudaError_t e = cudaSuccess;
    if (ahead && first_sweep) {       // the flag table is the same for every sweep: uploaded once per call
      std::vector<unsigned char> h(flag_bytes, 0);
      std::vector<int> pair_of((size_t)nblk);
      auto host_pair = [&](int i, int r, int& p, int& q) {
        const int m = nblk - 1;
        if (i == 0) { p = r; q = nblk - 1; return; }
        p = (r + i) % m;
        q = ((r - i) % m + m) % m;
      };
      for (int r = 0; r + 1 < rounds; ++r) {
        for (int i = 0; i < npairs; ++i) {
          int p, q;
          host_pair(i, r, p, q);
          pair_of[(size_t)p] = i;
          pair_of[(size_t)q] = i;
        }
        unsigned char* f = h.data() + (size_t)r * npairs * npairs;
        for (int i = 0; i < npairs; ++i) {
          int p, q;
          host_pair(i, r + 1, p, q);
          const int a = pair_of[(size_t)p], b = pair_of[(size_t)q];
          f[a * npairs + a] = 1;
          f[b * npairs + b] = 1;
          f[(a < b ? a : b) * npairs + (a < b ? b : a)] = 1;
        }
      }
      e = cudaMemcpyAsync(flags, h.data(), flag_bytes, cudaMemcpyHostToDevice, s);
      if (e == cudaSuccess) e = cudaStreamSynchronize(s);               // h is a host temporary
    }
    if (ahead) {
      if (e == cudaSuccess) {       // highest priority: the 38 subproblem CTAs must get their SMs before the update's 2000+ CTAs
        int lo = 0, hi = 0;
        e = cudaDeviceGetStreamPriorityRange(&lo, &hi);
        if (e == cudaSuccess) e = cudaStreamCreateWithPriority(&s2, cudaStreamNonBlocking, hi);
      }
      if (e == cudaSuccess) e = cudaEventCreateWithFlags(&e1, cudaEventDisableTiming);
      if (e == cudaSuccess) e = cudaEventCreateWithFlags(&e2, cudaEventDisableTiming);
    }
    if (e == cudaSuccess) {
      bj_solve_kernel<<<npairs, 1024, kBJSolveSmem, s>>>(Abuf, N, 0, Wbuf[0], kBJInnerSweeps);
      for (int r = 0; r < rounds && e == cudaSuccess; ++r) {
        const double2* W = Wbuf[r & 1];
        const bool la = ahead && r + 1 < rounds;
        if (!la) {
          bj_update_kernel<<<dim3(npairs, 2 * npairs), 256, kBJUpdateSmem, s>>>(Abuf, Vbuf, N, r, W, nullptr, 0);
          if (r + 1 < rounds) bj_solve_kernel<<<npairs, 1024, kBJSolveSmem, s>>>(Abuf, N, r + 1, Wbuf[(r + 1) & 1], kBJInnerSweeps);
          continue;
        }
        const unsigned char* f = flags + (size_t)r * npairs * npairs;
        bj_update_kernel<<<dim3(npairs, npairs), 256, kBJUpdateSmem, s>>>(Abuf, Vbuf, N, r, W, f, 1);
        e = cudaEventRecord(e1, s);
        if (e == cudaSuccess) e = cudaStreamWaitEvent(s2, e1, 0);
        if (e != cudaSuccess) break;
        bj_solve_kernel<<<npairs, 1024, kBJSolveSmem, s2>>>(Abuf, N, r + 1, Wbuf[(r + 1) & 1], kBJInnerSweeps);
        e = cudaEventRecord(e2, s2);
        bj_update_kernel<<<dim3(npairs, 2 * npairs), 256, kBJUpdateSmem, s>>>(Abuf, Vbuf, N, r, W, f, 2);
        if (e == cudaSuccess) e = cudaStreamWaitEvent(s, e2, 0);
      }
    }
    if (e == cudaSuccess) e = cudaGetLastError();
    if (e1) cudaEventDestroy(e1);
    if (e2) cudaEventDestroy(e2);
    if (s2) cudaStreamDestroy(s2);
    if (e != cudaSuccess) return e;
  } else {
    double4* params = reinterpret_cast<double4*>(work + 4 * sM + 64LL * N + (long long)(N / 64) * 4096);
    const int half = N / 2;
    const dim3 grid((half + 255) / 256, N);
    for (int r = 0; r < N - 1; ++r) {
      jacobi_params_kernel<<<(half + 127) / 128, 128, 0, s>>>(Abuf, N, r, params);
      jacobi_apply_kernel<<<grid, 256, 0, s>>>(Abuf, Vbuf, N, r, params);
    }
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
