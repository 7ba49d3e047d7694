// Internal (C++) launch interface between the C-ABI layer (qsgw_api.cu) and the sm_100a kernels.
// Internal data layouts (free to change; the boundary layouts are those of include/qsgw.h):
//
//   z workspace, FP64 mode:  double zws[2 planes (Re,Im)][ncg][kpad][16]
//       column group cg = I / 16 ("CG"), pair row p = n_local * n_u + n'_local, 16 doubles = 128 B.
//       One 4-D TMA box {16, KP, 4, 2} then brings a 64-column x KP-pair tile of both planes into
//       shared memory as [plane][cg][row][128 B] with the 128-byte swizzle.
//   weight table:            double wtab[n_freq][kpad]        (zero beyond the batch's pairs)
//   accumulators:            double acc_re/acc_im[n_freq][n_m_pad][n_m_pad], n_m_pad = ceil64(N_M);
//       only tiles with tile_i <= tile_j are touched.
#pragma once
#include <cstdint>
#include <cuda.h>
#include <cuda_runtime.h>

namespace qsgw {

constexpr int kCG = 16;         // columns per column group (128 B of doubles)
constexpr int kTile = 64;       // stage (b) CTA tile edge (complex outputs)
constexpr int kPairAlign = 32;  // kpad and the padded pair count are multiples of this

struct SiteTables {
  int n_sites;
  int n_b, n_m, b_max;
  const int* d_pb_site;    // [n_m]   site of product function I
  const int* d_pb_off;     // [S+1]   first I of site s
  const int* d_orb_off;    // [S+1]   first orbital of site s
  const long long* d_p_off;  // [S]   offset (complex elements) of site s in packed P
};

struct ZmelArgs {
  SiteTables st;
  const double2* P;      // packed complex128
  const double2* Ck;     // band-major: (beta, n) at Ck[n*ld_k + beta]
  long long ld_k;
  const double2* Ckq;
  long long ld_kq;
  int n_begin, n_o, np_begin, n_u;
  double* zws;           // FP64 workspace (see above)
  long long kpad;
  int ncg;
};

cudaError_t launch_zmel_f64(const ZmelArgs& a, cudaStream_t s);
cudaError_t launch_z_export(const double* zws, long long kpad, int ncg, int n_m, long long n_pairs,
                            double2* out, cudaStream_t s);
cudaError_t launch_z_import(double* zws, long long kpad, int ncg, int n_m, long long n_pairs,
                            const double2* in, cudaStream_t s);
cudaError_t launch_pair_weights(const double* eps_k, const double* f_k, const double* eps_kq,
                                const double* f_kq, int n_o, int n_u, const double* d_omega, int n_freq,
                                double occ_tol, double* wtab, long long kpad, long long n_pairs_padded,
                                cudaStream_t s);

struct Chi0F64Args {
  CUtensorMap tmap_z;    // 4-D FLOAT64 {16, kpad, ncg, 2}, box {16, KP, 4, 2}, SWIZZLE_128B
  const double* wtab;
  long long kpad;
  double* acc_re;
  double* acc_im;
  int n_m_pad;
  int n_freq;
  long long n_pairs_padded;   // multiple of kPairAlign
  const int2* d_tiles;        // (tile_i, tile_j), tile_i <= tile_j
  int n_tiles;
};
constexpr int kChi0F64KP = 16;  // pairs per pipeline stage (box rows of the tensor map)
cudaError_t launch_chi0_f64(const Chi0F64Args& a, cudaStream_t s);
cudaError_t chi0_f64_configure();   // sets the dynamic shared-memory attribute once

// issue-rate probes (probe_kernels.cu): measured MMA-pipe peaks for the roofline denominators
cudaError_t probe_fp64_mma(cudaStream_t s, double* out_tflops, double* out_ms);

cudaError_t launch_finalize(const double* acc_re, const double* acc_im, int n_m, int n_m_pad, int n_freq,
                            double inv_nk, double2* out, cudaStream_t s);

}  // namespace qsgw
