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
#include <cuda_fp16.h>
#include <cuda_runtime.h>

namespace qsgw {

constexpr int kMaxDevices = 64; // per-device bookkeeping of kernel attributes
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
  float* zmax = nullptr; // optional: atomicMax of |Re z|, |Im z| over the batch (FP16-split mixed mode); [n_batch]
  // several k-points per launch (blockIdx.z): k-point b reads Ck + b*Ck_bs, Ckq + b*Ckq_bs (complex elements) and
  // writes the workspace slot at pair offset b*z_bs
  int n_batch = 1;
  long long Ck_bs = 0, Ckq_bs = 0, z_bs = 0;
  const int* row_map = nullptr;  // optional [n_o*n_u]: workspace row of pair n*n_u + n' (binned real-axis path)
  int kt = 0;            // DMMA kernel: padded contraction length, max over column groups of sum_seg pad4(b_seg)
  int n_sm = 148;        // SMs of the context's device
};

cudaError_t launch_zmel_f64(const ZmelArgs& a, cudaStream_t s);    // CUDA-core fallback
cudaError_t launch_zmel_dmma(const ZmelArgs& a, cudaStream_t s);   // step 2 on the FP64 tensor pipe (default)
size_t zmel_dmma_smem_bytes(int b_max, int kt);
// Mixed mode: stage (a) on tcgen05 that writes the hl16 / hb8 operand rows of stage (b) itself (zmel_umma_kernels.cu).
// a.zmax[b] receives an upper BOUND of max |z| of batch b (the FP16 scale has to be known before the rows are written);
// pmax[s] = max_{I in s} ||P_I||_F (launch_zmel_pnorm, once per product tensor); cnorm: scratch of (2 n_sites + 2) n_batch floats;
// aop: scratch of zmel_umma_aop_halves halves; zhl / zhb8 = the slot of batch 0; n_rows = padded pair rows of a batch.
bool zmel_umma_supported(int b_max);
size_t zmel_umma_aop_halves(int n_sites, int n_u, int n_batch);
cudaError_t zmel_umma_configure();
cudaError_t launch_zmel_pnorm(const SiteTables& st, const double2* P, float* pmax, cudaStream_t s);
cudaError_t launch_zmel_umma(const ZmelArgs& a, const float* pmax, float* cnorm, __half* aop, void* zhl, void* zhb8, int n_m_pad,
                             long long n_rows, cudaStream_t s);
cudaError_t launch_z_export(const double* zws, long long kpad, int ncg, int n_m, long long n_pairs,
                            double2* out, cudaStream_t s);
cudaError_t launch_z_import(double* zws, long long kpad, int ncg, int n_m, long long n_pairs,
                            const double2* in, float* zmax /*optional*/, cudaStream_t s);
// n_batch k-points per launch: k-point b reads eps_k + b*n_o, ..., eps_kq + b*n_u, ..., zmax[b] and writes the table
// columns [b*n_pairs_padded, (b+1)*n_pairs_padded)
cudaError_t launch_pair_weights(const double* eps_k, const double* f_k, const double* eps_kq,
                                const double* f_kq, int n_o, int n_u, const double* d_omega, int n_freq,
                                double occ_tol, double* wtab, long long kpad, long long n_pairs_padded,
                                const float* zmax /*optional: fold 2^(-2S) of the batch's FP16 scale*/, int n_batch,
                                cudaStream_t s);

struct Chi0F64Args {
  CUtensorMap tmap_z;    // 4-D FLOAT64 {16, kpad, ncg, 2}, box {16, KP, 4, 2}, SWIZZLE_128B
  const double* wtab;
  long long kpad;
  double* acc_re;
  double* acc_im;
  int n_m_pad;
  int n_freq;                 // frequencies of this launch: j0 .. j0 + n_freq - 1
  int j0 = 0;
  int split = 1;              // CTAs sharing the staged pairs of one (tile, frequency); set by launch_chi0_f64
  int n_sm = 148;             // SMs of the context's device
  long long n_pairs_padded;   // multiple of kPairAlign
  // CTA work list (tile_i, tile_j, first 16-column group, 0), tile_i <= tile_j: n_tiles full 64 x 64 tiles, then
  // n_tiles_half 64 x 32 pieces (last tile column when N_M mod 64 is in 1..32; right half of a diagonal tile), then
  // n_tiles_quarter 32 x 32 pieces (upper-left block of a diagonal tile)
  const int4* d_tiles;
  int n_tiles;
  int n_tiles_half = 0;
  int n_tiles_quarter = 0;
  const int2* d_ranges = nullptr;   // optional [n_freq]: pair rows [x, y) that carry weight at that frequency (bin);
                                    // the CTA runs only the 32-pair stages that cover them (no split)
  // optional: only the 32-pair stages listed in d_live[0 .. *d_n_live) are run (the others carry no weight at any frequency)
  const int* d_live = nullptr;
  const int* d_n_live = nullptr;
};
constexpr int kChi0F64KP3M = 32;  // pairs per pipeline stage (box rows of the tensor map)
cudaError_t launch_chi0_f64(const Chi0F64Args& a, cudaStream_t s);
cudaError_t chi0_f64_configure();   // sets the dynamic shared-memory attribute (per device: call at context creation)

constexpr int kTileMx = 128;       // stage (b) CTA tile edge in mixed mode (UMMA M = N = 128)
constexpr int kPairStage = 32;     // pairs per pipeline stage (one 128-byte swizzle row)

// ---- mixed mode, FP16 split (chi0_f16_kernels.cu) ---------------------------------------------------
//   z workspace "hl16": __half zhl[2 planes (Re,Im)][n_m_pad][kpad/32][64]: per product function I and
//   32-pair stage one 128-byte row  h[32] | l[32],  v = fp32(z * 2^S) = h + l (h = fp16(v), l = fp16(v-h)),
//   S = f16_scale_exp(*zmax) from the batch maximum.  3-D TMA boxes {64 halves, 64 rows, 1 plane} with the
//   128-byte swizzle give K-major UMMA operand tiles.  Weights: __half wtab16[n_freq][kpad/32][64], per 32-pair
//   stage  w_h[32] | w_l[32]  with w_h + w_l = fp32(w_j(p) / wscale[j]), wscale[j] a power of two such that
//   max_p |w_j(p)| / wscale[j] is in (1/2, 1].
//   FP8-corrected variant: a second workspace "hb8" with rows  h[32] halves | e5m2(v)[32] | e5m2(v - h)[32]
//   feeds the B operand (same 128 bytes per 32 pairs): a b ~= a_h b_h (kind::f16) + a_l8 b_8 + a_8 b_l8
//   (kind::f8f6f4, E5M2): the two correction products need only ~3 significant bits.
// Device-side control block of the mixed mode (one per context).
//   E5M2 correction products add a relative Frobenius error ~ c * sqrt(N_M / P_eff) with P_eff the effective number
//   of band pairs summed per output element, P_eff = (sum_p w)^2 / sum_p w^2 (participation ratio of the weights of
//   the staged pairs, minimum over the frequencies).  use_fp8 = mode 1, or mode 2 and P_eff >= thr_pairs.
struct MixedCtl {
  float peff_min;            // min over frequencies of P_eff of the flush being prepared (atomicMin on the bits)
  int use_fp8;               // decision for the current flush
  int mode;                  // 0 never | 1 always | 2 automatic
  float thr_pairs;           // automatic: threshold on P_eff (pairs), = T * N_M
  unsigned int ticket;       // last-block-done counter of weights_scale_hl16_kernel
  unsigned long long n_flush, n_flush_fp8;   // statistics (qsgw_mixed_stats)
  float peff_min_seen;       // smallest P_eff of any flush since the last reset
};

struct Chi0F16Args {
  CUtensorMap tmap;      // 3-D FLOAT16 {2*kpad, n_m_pad, 2}, box {64, 64, 1}, SWIZZLE_128B
  CUtensorMap tmap_b;    // FP8 variant: 3-D UINT8 {4*kpad, n_m_pad, 2}, box {128, 64, 1}, SWIZZLE_128B
  const __half* wtab16;  // [n_freq][kpad/32][64]
  const double* wscale;  // [n_freq]
  long long kpad;
  double* acc_re;
  double* acc_im;
  int n_m_pad;           // multiple of 128
  int n_freq;
  int n_stages;          // ceil(n_pairs / 32)
  int win;               // stages per drain window (12 MMA steps into each accumulator per stage)
  int j0 = 0;            // first frequency of this launch (n_freq = count)
  int split = 1;         // CTAs sharing the staged pairs of one (tile, frequency); set by launch_chi0_f16
  int n_sm = 148;        // SMs of the context's device
  int pair = 1;          // CTA pairs (cta_group::2) sharing the B tiles of two frequencies; 0 = one CTA per (tile, frequency)
  const MixedCtl* ctl;   // device: use_fp8 selects the variant that runs (the other one exits at once)
  const int2* d_ranges = nullptr;   // optional [n_freq]: pair rows [x, y) that carry weight at that frequency (bin); no split
  const int* d_live = nullptr;      // optional: only the stages d_live[0 .. *d_n_live) are run (the others carry no weight)
  const int* d_n_live = nullptr;
  const int4* d_tiles;   // 128x128 tiles (tile_i, tile_j, 0, 0), tile_i <= tile_j
  int n_tiles;
};
cudaError_t chi0_f16_configure();
// Launches BOTH product variants (three FP16 products | FP16 main + two E5M2 correction products); each CTA reads
// ctl->use_fp8 first and the variant that was not selected returns immediately (the selection is made on the
// device from the weights of the staged pairs, see weights_scale_hl16_kernel: no host synchronisation).
cudaError_t launch_chi0_f16(const Chi0F16Args& a, cudaStream_t s);
// n_batch batches of n_pairs pairs at pair offsets b*z_bs (a multiple of 32), scales zmax[b]
// live[0 .. *n_live) = the 32-pair stages of the first n_pad staged rows that carry a nonzero weight at some frequency, in
// ascending order (metals: whole bands fail the occupation filter); flags: scratch of n_pad / 32 bytes
cudaError_t launch_stage_compaction(const double* wtab, long long kpad, long long n_pad, int n_freq, unsigned char* flags,
                                    int* live, int* n_live, cudaStream_t s);
cudaError_t launch_z_to_hl16(const double* zws, long long kpad, int ncg, int n_m, long long n_pairs, void* zhl,
                             void* zhb8 /*optional FP8-variant B rows*/, int n_m_pad, const float* zmax, int n_batch,
                             long long z_bs, cudaStream_t s);
cudaError_t launch_z_export_hl16(const void* zhl, long long kpad, int n_m_pad, int n_m, long long n_pairs,
                                 const float* zmax, double2* out, cudaStream_t s);
// zfold (optional): the weights are multiplied by 2^(-2S), S = f16_scale_exp(*zfold) (binned path: one batch per flush, its
// weights come from the caller and do not carry the batch's FP16 scale yet)
cudaError_t launch_weights_scale_hl16(const double* wtab, void* wtab16, double* wscale, long long kpad, long long n_pad,
                                      int n_freq, MixedCtl* ctl, const float* zfold, cudaStream_t s);

// ---- batched complex FP64 GEMM on the FP64 tensor pipe, operands staged by TMA (zgemm_tma_kernels.cu) ----------
// C (+)= alpha * sum_{r < reps} diag(row_scale[r]) opA(A_r) opB(B_r)   on 64x64 tiles, complex128 interleaved, row-major.
//   a_kc:  A_r(i,k) = A[r*rA + i*lda + k]              else  A_r(i,k) = conj(A[r*rA + k*lda + i])   (conjugate transpose)
//   b_kc:  B_r(k,j) = conj(B[r*rB + j*ldb + k])        else  B_r(k,j) = B[r*rB + k*ldb + j]
// Extents are arbitrary (ragged tiles are zero-filled by TMA, stores are guarded); batch b reads A + b*sA, B + b*sB and
// writes C + b*sC (stride 0 = operand shared by all batches).  The repetitions are an outer contraction loop: the
// frequencies of the I^c product (A fixed, B = W^c(i omega_r), row_scale = the quadrature weights) or the
// intermediate states of its closing contraction.  split > 1: the repetitions are divided over `split` CTAs per tile,
// which add their partial sums to C atomically (C must hold the value to add to: beta_one semantics).
struct ZgemmArgs {
  const double2* A; const double2* B; double2* C;
  long long lda, ldb, ldc;      // leading dimensions in complex elements
  long long sA, sB, sC;         // batch strides in complex elements
  int m, n, k;                  // C is m x n; contraction length k per repetition
  int batch = 1;
  double alpha = 1.0;           // real scale
  int beta_one = 0;             // 1: C += ..., 0: C = ...
  int tri = 0;                  // 0 all tiles | 1 lower tiles only | 2 lower tiles and k starts at 64*max(ti,tj)
                                // | 3 all tiles and k starts at 64*tj (B lower triangular)
  int reps = 1; long long rA = 0, rB = 0;
  const double* row_scale = nullptr; long long ld_scale = 0;    // [reps][ld_scale], row i of C / opA
  int split = 1;
};
cudaError_t launch_zgemm(bool a_kc, bool b_kc, const ZgemmArgs& a, cudaStream_t s);
cudaError_t zgemm_configure();       // kernel attributes (per device)
// 4-D FP64 tensor map over interleaved complex128 data: dims {2*inner, outer, d2, d3} (strides in complex elements),
// box {16 doubles, box_rows, 1, 1}, 128-byte swizzle, zero fill out of bounds.  Defined in qsgw_api.cu.
cudaError_t make_zmap(CUtensorMap* out, const double2* base, long long inner, long long outer, long long ld,
                      long long d2, long long s2, long long d3, long long s3, int box_rows);

// ---- interstitial-plane-wave block of the matrix elements (ipw_kernels.cu) ---------------------------------
// z_out[(n n_u + n') ld_z + I] = sum_{alpha, beta} conj(Bkq[n', alpha]) theta(g_k[beta] - g_kq[alpha] - g_ipw[I]) Bk[n, beta];
// L = HOST array of the theta box half extents; work: ipw_work_elems complex elements; a_chunk from ipw_alpha_chunk.
int ipw_alpha_chunk(int n_pw_kq, int n_pw_k, int n_ipw, int n_o, size_t cap_bytes);
size_t ipw_work_elems(int a_chunk, int n_pw_k, int n_ipw, int n_o, int n_u);
cudaError_t launch_zmel_ipw(const int L[3], const double2* theta, int n_pw_kq, const int* g_kq, int n_pw_k, const int* g_k,
                            int n_ipw, const int* g_ipw, const double2* Bk, long long ld_k, int n_o, const double2* Bkq,
                            long long ld_kq, int n_u, double2* z_out, long long ld_z, int a_chunk, double2* work,
                            cudaStream_t s);

// ---- generalized eigenproblem of the Coulomb matrix in the mixed product basis (eig_kernels.cu) ---------------
// (v - v_mu O) z = 0, z^H O z = 1: Cholesky reduction to a standard Hermitian problem + two-sided parallel Jacobi.
// work: eig_work_elems complex elements.  Call order: launch_eig_reduce, launch_eig_sweep until converged
// (d_norms[0] = |off-diagonal|^2, d_norms[1] = |diagonal|^2 after each sweep), launch_eig_diag (eigenvalues, unsorted),
// launch_eig_finish with the column permutation (descending eigenvalues).
size_t eig_work_elems(int n_m);
cudaError_t launch_eig_reduce(int n_m, const double2* v, const double2* O, double2* work, int* d_info, cudaStream_t s);
cudaError_t eig_configure();        // kernel attributes (per device)
cudaError_t launch_eig_sweep(int n_m, double2* work, double* d_norms, bool blocked, bool first_sweep, cudaStream_t s);
cudaError_t launch_eig_diag(int n_m, const double2* work, double* d_diag, cudaStream_t s);
cudaError_t launch_eig_finish(int n_m, double2* work, const int* d_perm, double2* U_out, cudaStream_t s);

// ---- screened Coulomb interaction W^c (wc_kernels.cu) ---------------------------------------------------
// W^c[j] = sqrt(v) ((1 - sqrt(v) chi0[j] sqrt(v))^-1 - 1) sqrt(v) for all frequencies, stream-ordered.
// work: n_freq * (2 * n_pad^2 + 64 * n_pad + nb * 64 * 64) complex elements, n_pad = ceil64(n_m), nb = n_pad / 64.
// d_info: 0, or 1 + index of the first non-positive Cholesky pivot (eps not positive definite).
size_t wc_work_elems(int n_m, int n_freq);
// Blocked Cholesky A = L L^H of `batch` HPD matrices of order N (multiple of 64; lower triangle overwritten by L) and X = L^-1;
// Tbuf: batch * 64 * N, Linv: batch * (N / 64) * 4096 complex elements; d_info as below.
cudaError_t launch_chol_inverse(int N, int batch, double2* Abuf, double2* Xbuf, double2* Tbuf, double2* Linv, int* d_info,
                                cudaStream_t s);
cudaError_t wc_configure();          // kernel attributes (per device)
// chi0 -> U^H chi0 U for all frequencies (work: rotate_work_elems complex elements)
size_t rotate_work_elems(int n_m, int n_freq);
cudaError_t launch_rotate_basis(int n_m, int n_freq, const double2* chi0, const double2* U, double2* out, double2* work,
                                cudaStream_t s);
// The same on a file-scope device array of rotate_static_max_elems() complex elements (no allocation of any kind;
// cudaErrorMemoryAllocation when rotate_work_elems(n_m, n_freq) exceeds it).  Calls that overlap on the GPU race.
long long rotate_static_max_elems();
cudaError_t launch_rotate_basis_static(int n_m, int n_freq, const double2* chi0, const double2* U, double2* out,
                                       cudaStream_t s);
cudaError_t launch_wc_from_chi0(int n_m, int n_freq, const double2* chi0, const double* v, double2* wc_out,
                                double2* work, int* d_info, cudaStream_t s);

// ---- imaginary-axis correlation self-energy I^c (sigc_kernels.cu; Eq. 22, Alg. 2) -------------------------------
// w[i][p] (ld doubles per frequency) for the pairs p = n' * n_qp + n of one batch of intermediate states
cudaError_t launch_sigc_weights(const double* eps_q, const double* eps_qk, int n_all, int n_qp, const double* d_omega,
                                int n_freq, double* w, long long ld, cudaStream_t s);
// z: complex128 [n_all][n_qp][n_m]; wc: [n_freq][n_m][n_m]; zw: workspace of the size of z; sigc [n_qp][n_qp] += ...
cudaError_t launch_sigc_imag(const double2* z, const double* w, long long ld_w, const double2* wc, int n_all, int n_qp,
                             int n_m, int n_freq, double inv_nk, double2* zw, double2* sigc, int n_sm, cudaStream_t s);

// ---- real-axis route (realaxis_kernels.cu; Eqs. 15-18, Alg. 1 lines 13-27) ---------------------------------------
// From the CSR-by-bin weights (bin_ptr[n_bins+1], pair[nnz], w[nnz]) of one band batch: row_map[n_pairs] = workspace row
// of every pair after a counting sort by first + last bin that carry it (pairs without weight last), the dense table
// wtab[n_bins][kpad] (zero except the entries) and ranges[n_bins] = rows touched by each bin.
// scratch: 2*n_pairs + 4*(n_bins + 1) ints.
cudaError_t launch_bin_setup(const int* bin_ptr, const int* pair, const double* w, int nnz, int n_bins, long long n_pairs,
                             long long n_pad, int* row_map, int* scratch, double* wtab, long long kpad, int2* ranges,
                             cudaStream_t s);
// out[i][e] = sum_j K[i][j] A[j][e], K[i][j] = -log1p((R^2 - L^2) / (L^2 + omega_i^2)) / (R - L) over bin j = [L, R)
// (Eq. 18 on the imaginary axis), or for real_axis = 1 K[i][j] = log|(omega_i^2 - L^2) / (omega_i^2 - R^2)| / (R - L) (targets on
// the real axis, principal value); A, out complex128 [.][n_m][n_m]
cudaError_t launch_hilbert(int n_m, int n_bins, const double* edges, int n_out, const double* omega_out,
                           const double2* A, double2* out, int real_axis, cudaStream_t s);

// mixed mode (sigc_f16_kernels.cu): ZW^c on tcgen05 with FP16-split operands.  zk16 / w16: workspaces of sigc_f16_z_halves /
// sigc_f16_w_halves halves; amax: 1 + n_freq floats.  z: complex128 [pairs][n_m], wc: [n_freq][n_m][n_m], zw: out [pairs][n_m].
size_t sigc_f16_z_halves(long long pairs_cap, int n_m);
size_t sigc_f16_w_halves(int n_m, int n_freq);
cudaError_t sigc_f16_configure();
cudaError_t launch_sigc_zw_f16(const double2* z, const double2* wc, const double* w, long long ld_w, int pairs, int n_m,
                               int n_freq, __half* zk16, __half* w16, unsigned char* w8 /*optional: E5M2 corrections*/, float* amax,
                               double2* zw, cudaStream_t s);
// 3-D FLOAT16 tensor map over hl16 rows: dims {row_halves, rows, 2 planes}, box {64, 64, 1}, 128-byte swizzle (qsgw_api.cu)
cudaError_t make_hl16_map(CUtensorMap* out, const void* base, long long row_halves, long long rows, long long plane_halves);
// the same rows addressed in bytes (hb8 rows: h[32] halves | e5m2(v)[32] | e5m2(v - h)[32]): UINT8 {2 * row_halves, rows, 2}, box {128, 64, 1}
cudaError_t make_hb8_map(CUtensorMap* out, const void* base, long long row_halves, long long rows, long long plane_halves);
// closing contraction of I^c alone (sigc_kernels.cu): sigc[n, m] += -(1/N_k) sum_{n', nu} zw[(n', n), nu] conj(z[(n', m), nu])
cudaError_t launch_sigc_close(const double2* z, const double2* zw, int n_all, int n_qp, int n_m, double inv_nk, double2* sigc,
                              int n_sm, cudaStream_t s);

// issue-rate probes (probe_kernels.cu): measured MMA-pipe peaks for the roofline denominators
cudaError_t probe_fp64_mma(cudaStream_t s, double* out_tflops, double* out_ms);
cudaError_t probe_tf32_mma(cudaStream_t s, double* out_tflops, double* out_ms);
cudaError_t probe_f16_mma(cudaStream_t s, double* out_tflops, double* out_ms);

cudaError_t launch_finalize(const double* acc_re, const double* acc_im, int n_m, int n_m_pad, int n_freq,
                            double inv_nk, double2* out, cudaStream_t s);

}  // namespace qsgw
