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

constexpr int kHilbertOut = 16;      // output frequencies per pass (register accumulators)

// One thread = one complex element of every bin matrix, 16 output frequencies in registers; the transform
// coefficients are broadcast reads from shared memory.  Two CTAs per SM and eight loads in flight per thread keep
// enough bytes in flight for HBM.
// real_axis = 0: K = -log1p((R^2 - L^2) / (L^2 + omega^2)) / (R - L)   (targets i omega, Eq. 14 at omega = i omega_i)
// real_axis = 1: K = log|(omega^2 - L^2) / (omega^2 - R^2)| / (R - L)       (targets omega on the real axis: principal value)
__global__ void __launch_bounds__(256, 2) hilbert_kernel(long long n_cplx, int n_bins, const double* __restrict__ edges,
                                                         int n_out, int i0, const double* __restrict__ omega_out,
                                                         const double2* __restrict__ A, double2* __restrict__ out,
                                                         int real_axis) {
  extern __shared__ double Ks[];       // [n_bins][kHilbertOut]
  const int n_i = min(kHilbertOut, n_out - i0);
  for (int idx = threadIdx.x; idx < kHilbertOut * n_bins; idx += blockDim.x) {
    const int j = idx / kHilbertOut, i = idx - j * kHilbertOut;
    double v = 0.0;
    if (i < n_i) {
      const double L = edges[j], R = edges[j + 1], om = omega_out[i0 + i];
      v = real_axis ? (log(fabs(om * om - L * L)) - log(fabs(om * om - R * R))) / (R - L)
                    : -log1p((R - L) * (R + L) / (L * L + om * om)) / (R - L);
    }
    Ks[idx] = v;
  }
  __syncthreads();
  for (long long e = blockIdx.x * (long long)blockDim.x + threadIdx.x; e < n_cplx; e += (long long)gridDim.x * blockDim.x) {
    double ar[kHilbertOut], ai[kHilbertOut];
#pragma unroll
    for (int i = 0; i < kHilbertOut; ++i) ar[i] = ai[i] = 0.0;
    const double2* ap = A + e;
#pragma unroll 8
    for (int j = 0; j < n_bins; ++j) {
      const double2 a = ap[(long long)j * n_cplx];
      const double* kj = Ks + j * kHilbertOut;
#pragma unroll
      for (int i = 0; i < kHilbertOut; ++i) {
        const double k = kj[i];
        ar[i] += k * a.x;
        ai[i] += k * a.y;
      }
    }
#pragma unroll
    for (int i = 0; i < kHilbertOut; ++i)
      if (i < n_i) out[(long long)(i0 + i) * n_cplx + e] = make_double2(ar[i], ai[i]);
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
  const size_t smem = sizeof(double) * kHilbertOut * n_bins;
  if (smem > 48 * 1024) return cudaErrorInvalidValue;
  long long blocks = (n_cplx + 255) / 256;
  if (blocks > 148LL * 8) blocks = 148LL * 8;
  for (int i0 = 0; i0 < n_out; i0 += kHilbertOut) {
    hilbert_kernel<<<(unsigned)blocks, 256, smem, s>>>(n_cplx, n_bins, edges, n_out, i0, omega_out, A, out, real_axis);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return e;
  }
  return cudaSuccess;
}

}  // namespace qsgw
