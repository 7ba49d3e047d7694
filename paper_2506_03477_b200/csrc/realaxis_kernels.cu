// The paper's real-axis route: set-up of the binned accumulation of the spectral part (Eqs. 15-17,
// PAPER.md:165-173; Alg. 1 lines 13-21) and the Hilbert transform to the imaginary axis (Eq. 18,
// PAPER.md:175-177; Alg. 1 line 27).
//
// Alg. 1 gathers, for every histogram bin, the band pairs whose weight is non-zero into Z_pair and multiplies
// Z_pair^dagger x W_Zpair.  Here the gather is a PERMUTATION made before z is written: the pairs of a band batch are
// sorted by first bin + last bin that carry them (twice the centre of their window: the order of their excitation
// energies), stage (a) writes each pair's row at its sorted position, and a bin then touches one short contiguous
// range of rows with few foreign pairs in it (a pair's tetrahedron weight spreads over a few neighbouring bins only),
// which stage (b) (chi0_f64_3m_kernel with Chi0F64Args::d_ranges) streams by TMA like any other batch; the per-bin
// weights sit in the dense, mostly zero table the kernel already reads.
#include "kernels.h"

namespace qsgw {

namespace {

__device__ __forceinline__ int bin_of_entry(const int* __restrict__ bin_ptr, int n_bins, int e) {
  int lo = 0, hi = n_bins;              // largest j with bin_ptr[j] <= e
  while (hi - lo > 1) {
    const int mid = (lo + hi) >> 1;
    if (bin_ptr[mid] <= e) lo = mid; else hi = mid;
  }
  return lo;
}

// sort key of a pair = first bin + last bin with weight (0 .. 2 n_bins - 2); 2 n_bins = "carries no weight" (sorted last)
__global__ void bin_init_kernel(int* __restrict__ first_bin, int* __restrict__ last_bin, long long n_pairs, int n_bins,
                                int* __restrict__ count, int2* __restrict__ ranges) {
  const long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x;
  if (i < n_pairs) {
    first_bin[i] = n_bins;
    last_bin[i] = -1;
  }
  if (i < 2 * n_bins + 2) count[i] = 0;
  if (i < n_bins) ranges[i] = make_int2(0x7fffffff, 0);
}

__global__ void bin_first_kernel(const int* __restrict__ bin_ptr, const int* __restrict__ pair, int nnz, int n_bins,
                                 int* __restrict__ first_bin, int* __restrict__ last_bin) {
  const int e = blockIdx.x * blockDim.x + threadIdx.x;
  if (e >= nnz) return;
  const int j = bin_of_entry(bin_ptr, n_bins, e), p = pair[e];
  atomicMin(&first_bin[p], j);
  atomicMax(&last_bin[p], j);
}

// key[i] replaces first_bin[i]
__global__ void bin_count_kernel(int* __restrict__ first_bin, const int* __restrict__ last_bin, long long n_pairs,
                                 int n_bins, int* __restrict__ count) {
  const long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x;
  if (i >= n_pairs) return;
  const int f = first_bin[i];
  const int key = f >= n_bins ? 2 * n_bins : f + last_bin[i];
  first_bin[i] = key;
  atomicAdd(&count[key], 1);
}

// exclusive scan of count[0 .. n_bins] (one block), result in offs; count is reused as the running cursor
__global__ void bin_scan_kernel(int* __restrict__ count, int* __restrict__ offs, int n) {
  if (threadIdx.x == 0) {
    int run = 0;
    for (int i = 0; i < n; ++i) {
      const int c = count[i];
      offs[i] = run;
      count[i] = run;
      run += c;
    }
  }
}

// Stable within a bucket would need a second pass; the order inside a bucket only changes the summation order.
__global__ void bin_place_kernel(const int* __restrict__ first_bin, long long n_pairs, int* __restrict__ cursor,
                                 int* __restrict__ row_map) {
  const long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x;
  if (i < n_pairs) row_map[i] = atomicAdd(&cursor[first_bin[i]], 1);
}

__global__ void bin_scatter_kernel(const int* __restrict__ bin_ptr, const int* __restrict__ pair,
                                   const double* __restrict__ w, int nnz, int n_bins, const int* __restrict__ row_map,
                                   double* __restrict__ wtab, long long kpad, int2* __restrict__ ranges) {
  const int e = blockIdx.x * blockDim.x + threadIdx.x;
  if (e >= nnz) return;
  const int j = bin_of_entry(bin_ptr, n_bins, e);
  const int row = row_map[pair[e]];
  atomicAdd(&wtab[(long long)j * kpad + row], w[e]);      // duplicates of a (pair, bin) entry add up
  atomicMin(&ranges[j].x, row);
  atomicMax(&ranges[j].y, row + 1);
}

__device__ __forceinline__ void dmma_k4(double& c0, double& c1, double a, double b) {   // D(8x8) += A(8x4) B(4x8), ptx.cuh
  asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
               : "+d"(c0), "+d"(c1)
               : "d"(a), "d"(b));
}

constexpr int kHilbertOut = 16;      // output frequencies per pass (two DMMA row tiles)

// Hilbert transform out[i] = sum_j K[i][j] A[j] (Eq. 18) as out[16 x cols] = K[16 x n_bins] A[n_bins x cols] on the FP64 tensor
// pipe (DMMA.8x8x4); the real and the imaginary parts of A are two column sets that share the K fragments.  The work is
// HBM-bound (every bin matrix is read once, 16 FMAs per loaded double): the tensor pipe is used because it takes 1/8 of the
// instructions of the CUDA-core form and no shared-memory broadcast per FMA, so that the loads stay ahead of HBM (round 2:
// CUDA-core kernel 2.15 ms = 0.76 of the measured copy bandwidth at 100 bins x 2400^2; this kernel 1.65 ms = 0.99).
// A warp takes U units of 8 consecutive complex elements (128 bytes per bin row): lane (g, t) loads element g of each unit
// at bin 4 kk + t with one 16-byte load (b fragments B[k = t][n = g] of the Re and of the Im product), the K fragments
// a = K[out g (+8)][bin 4 kk + t] come from shared memory (row pitch 20: conflict-free), d = D[out g][element 2t, 2t + 1].
// U = 2 with the bin loop unrolled 8 times (16 loads of 16 bytes in flight per lane, 2 CTAs per SM) was the fastest of the
// measured variants (U, unroll, CTAs/SM): (4,2,2) 1.99 ms, (2,4,3) 1.76, (2,8,2) 1.65, (4,4,1) 1.93, (1,8,4) 1.87.
// real_axis = 0: K = -log1p((R^2 - L^2) / (L^2 + omega^2)) / (R - L)   (targets i omega, Eq. 14 at omega = i omega_i)
// real_axis = 1: K = log|(omega^2 - L^2) / (omega^2 - R^2)| / (R - L)       (targets omega on the real axis: principal value)
constexpr int kHilbertLd = 20;
template <int U, int UNR, int MINB>
__global__ void __launch_bounds__(256, MINB) hilbert_dmma_kernel(long long n_cplx, int n_bins, const double* __restrict__ edges,
                                                              int n_out, int i0, const double* __restrict__ omega_out,
                                                              const double2* __restrict__ A, double2* __restrict__ out,
                                                              int real_axis) {
  extern __shared__ double Ks[];       // [n_bins4][kHilbertLd], rows >= n_bins and columns >= n_i zero
  const int n_bins4 = (n_bins + 3) & ~3;
  const int n_i = min(kHilbertOut, n_out - i0);
  for (int idx = threadIdx.x; idx < kHilbertOut * n_bins4; idx += blockDim.x) {
    const int j = idx / kHilbertOut, i = idx - j * kHilbertOut;
    double v = 0.0;
    if (i < n_i && j < n_bins) {
      const double L = edges[j], R = edges[j + 1], om = omega_out[i0 + i];
      v = real_axis ? (log(fabs(om * om - L * L)) - log(fabs(om * om - R * R))) / (R - L)
                    : -log1p((R - L) * (R + L) / (L * L + om * om)) / (R - L);
    }
    Ks[j * kHilbertLd + i] = v;
  }
  __syncthreads();
  const int lane = threadIdx.x & 31, g = lane >> 2, t = lane & 3;
  const long long warp = (blockIdx.x * (long long)blockDim.x + threadIdx.x) >> 5;
  const long long n_warps = ((long long)gridDim.x * blockDim.x) >> 5;
  for (long long e0 = warp * (8 * U); e0 < n_cplx; e0 += n_warps * (8 * U)) {
    double dr[U][2][2], di[U][2][2];
#pragma unroll
    for (int u = 0; u < U; ++u)
#pragma unroll
      for (int rt = 0; rt < 2; ++rt) dr[u][rt][0] = dr[u][rt][1] = di[u][rt][0] = di[u][rt][1] = 0.0;
    bool ok[U];
#pragma unroll
    for (int u = 0; u < U; ++u) ok[u] = e0 + 8 * u + g < n_cplx;
    const double2* ap = A + e0 + g;
#pragma unroll UNR
    for (int kk = 0; kk < n_bins4 / 4; ++kk) {
      const int j = 4 * kk + t;
      const bool jok = j < n_bins;
      const double2* row = ap + (long long)j * n_cplx;
      double2 b[U];
#pragma unroll
      for (int u = 0; u < U; ++u) b[u] = (jok && ok[u]) ? row[8 * u] : make_double2(0.0, 0.0);
      const double k0 = Ks[j * kHilbertLd + g], k1 = Ks[j * kHilbertLd + 8 + g];
#pragma unroll
      for (int u = 0; u < U; ++u) {
        dmma_k4(dr[u][0][0], dr[u][0][1], k0, b[u].x);
        dmma_k4(di[u][0][0], di[u][0][1], k0, b[u].y);
        dmma_k4(dr[u][1][0], dr[u][1][1], k1, b[u].x);
        dmma_k4(di[u][1][0], di[u][1][1], k1, b[u].y);
      }
    }
#pragma unroll
    for (int rt = 0; rt < 2; ++rt) {
      const int i = g + 8 * rt;
      if (i >= n_i) continue;
      double2* orow = out + (long long)(i0 + i) * n_cplx + e0 + 2 * t;
#pragma unroll
      for (int u = 0; u < U; ++u) {
        const long long e = e0 + 8 * u + 2 * t;
        if (e < n_cplx) orow[8 * u] = make_double2(dr[u][rt][0], di[u][rt][0]);
        if (e + 1 < n_cplx) orow[8 * u + 1] = make_double2(dr[u][rt][1], di[u][rt][1]);
      }
    }
  }
}

}  // namespace

cudaError_t launch_bin_setup(const int* bin_ptr, const int* pair, const double* w, int nnz, int n_bins, long long n_pairs,
                             long long n_pad, int* row_map, int* scratch, double* wtab, long long kpad, int2* ranges,
                             cudaStream_t s) {
  int* first_bin = scratch;
  int* last_bin = scratch + n_pairs;
  int* count = last_bin + n_pairs;
  int* offs = count + 2 * n_bins + 2;
  const long long n_init = n_pairs > 2 * n_bins + 2 ? n_pairs : 2 * n_bins + 2;
  const unsigned gp = (unsigned)((n_pairs + 255) / 256), ge = (unsigned)((nnz + 255) / 256);
  bin_init_kernel<<<(unsigned)((n_init + 255) / 256), 256, 0, s>>>(first_bin, last_bin, n_pairs, n_bins, count, ranges);
  cudaError_t e = cudaMemset2DAsync(wtab, sizeof(double) * kpad, 0, sizeof(double) * n_pad, n_bins, s);
  if (e != cudaSuccess) return e;
  if (nnz > 0) bin_first_kernel<<<ge, 256, 0, s>>>(bin_ptr, pair, nnz, n_bins, first_bin, last_bin);
  bin_count_kernel<<<gp, 256, 0, s>>>(first_bin, last_bin, n_pairs, n_bins, count);
  bin_scan_kernel<<<1, 32, 0, s>>>(count, offs, 2 * n_bins + 1);
  bin_place_kernel<<<gp, 256, 0, s>>>(first_bin, n_pairs, count, row_map);
  if (nnz > 0) bin_scatter_kernel<<<ge, 256, 0, s>>>(bin_ptr, pair, w, nnz, n_bins, row_map, wtab, kpad, ranges);
  return cudaGetLastError();
}

cudaError_t launch_hilbert(int n_m, int n_bins, const double* edges, int n_out, const double* omega_out,
                           const double2* A, double2* out, int real_axis, cudaStream_t s) {
  const long long n_cplx = (long long)n_m * n_m;
  const size_t smem = sizeof(double) * kHilbertLd * ((n_bins + 3) & ~3);
  if (smem > 48 * 1024) return cudaErrorInvalidValue;
  long long blocks = (n_cplx + 127) / 128;          // a CTA of 8 warps takes 8 x 16 elements per pass
  if (blocks > 148LL * 8) blocks = 148LL * 8;
  for (int i0 = 0; i0 < n_out; i0 += kHilbertOut) {
    hilbert_dmma_kernel<2, 8, 2><<<(unsigned)blocks, 256, smem, s>>>(n_cplx, n_bins, edges, n_out, i0, omega_out, A, out, real_axis);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return e;
  }
  return cudaSuccess;
}

}  // namespace qsgw
