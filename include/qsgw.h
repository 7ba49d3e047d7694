/*
 * qsgw.h -- C ABI of the B200-native polarization build chi0(q, i*omega) for QSGW.
 *
 * Method: arxiv 2506.03477.  One context = one (q, spin) problem:
 *
 *   stage (a)  z[n,n',I] = sum_{alpha,beta in site(I)} conj(C_{k+q}[alpha,n']) P_s[I,alpha,beta] C_k[beta,n]
 *              muffin-tin part of the matrix elements of Eq. (8) with the
 *              eigenfunction expansion of Eq. (4); "prepared on the fly"
 *               per band batch (Alg. 1 lines 10-12).
 *   stage (b)  acc_j[I,J] += sum_{pairs kept} w_j(n,n') conj(z[n,n',I]) z[n,n',J],  I <= J
 *              w_j = -2 f_n (1-f_n') D / (D^2 + omega_j^2),  D = eps_{k+q,n'} - eps_{k,n}
 *              Eq. (14) on the imaginary axis = Alg. 1 lines 16-21
 *               with a dense Lorentzian weight per frequency.
 *   finalize   chi0_j = acc_j / N_k, lower triangle = conj(upper), Im(diag) = 0
 *              (the matrix part is Hermitian).
 *
 * Conventions
 *   - Pointers named d_* are DEVICE pointers owned by the caller; h_* are HOST pointers that
 *     are read (or written, for outputs) during the call and never retained.
 *   - complex128 = interleaved (re, im) pairs of IEEE doubles.  Boundary data are always
 *     complex128 / float64; QSGW_PREC_MIXED converts internally.
 *   - Every call returns an int32 status (QSGW_OK = 0); nothing throws or aborts.  Calls are
 *     stream-ordered on the stream given to qsgw_create and never synchronise the device,
 *     except qsgw_sync, qsgw_destroy and the *_host entry point.  Asynchronous CUDA faults
 *     surface as QSGW_ERR_CUDA on a later call.
 *   - The library owns only its context (accumulators, z workspace, weight table, TMA
 *     descriptors).  There is no CPU fallback: without a CUDA device every compute call fails.
 *   - Orbitals are grouped by site: site s owns the contiguous orbital range
 *     [sum_{t<s} b_t, +b_s); product functions likewise with m_s.  N_b = sum b_s, N_M = sum m_s.
 *   - State machine: create -> set_product_tensor -> { zmel_build -> chi0_accumulate }* ->
 *     chi0_finalize -> ( reset -> ... ).  Out-of-order calls return QSGW_ERR_STATE.
 */
#ifndef QSGW_H_
#define QSGW_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct qsgw_ctx qsgw_ctx;

enum {
  QSGW_OK = 0,
  QSGW_ERR_INVALID_ARG = 1, /* null pointer, bad enum, bad leading dimension            */
  QSGW_ERR_SHAPE = 2,       /* non-positive extent, batch larger than declared, bad omega */
  QSGW_ERR_STATE = 3,       /* call out of order                                        */
  QSGW_ERR_ALLOC = 4,       /* device allocation failed or workspace cap too small      */
  QSGW_ERR_CUDA = 5,        /* CUDA runtime / driver error (see qsgw_last_error)        */
  QSGW_ERR_UNSUPPORTED = 6  /* no sm_100 device, or feature not built                   */
};

/* QSGW_PREC_MIXED: z held as FP32 complex and multiplied with FP32-grade products on the 5th-generation
 *   tensor cores: every FP32 operand v (scaled by a power of two) is carried as fp16 pieces v = h + l
 *   (22 significant bits) and a*b is formed as a_h*b_h + a_l*b_h + a_h*b_l by three exact FP16 MMAs
 *   (tcgen05 kind::f16, twice the TF32 rate); FP32 window sums, FP64 accumulation across batches and k.
 *   The two correction products a_l*b_h + a_h*b_l need only ~3 significant bits and run in E5M2
 *   (kind::f8f6f4) for every stage (b) launch whose staged pairs are numerous enough: the choice is made ON THE
 *   DEVICE, per launch, from the weights of the pairs that are actually accumulated (effective pair count
 *   P_eff = (sum w)^2 / sum w^2, minimum over the frequencies, against a multiple of N_M), never from the
 *   descriptor; launches below the threshold use the three-FP16-product form.  Contract of the mode in either
 *   case: relative Frobenius error <= 2e-5 per frequency against the FP64 result. */
enum { QSGW_PREC_FP64 = 0, QSGW_PREC_MIXED = 1 };

/* Problem descriptor (host memory; copied by qsgw_create). */
typedef struct {
  int32_t n_sites;               /* S >= 1                                                     */
  const int32_t* h_orb_per_site; /* b_s > 0, S entries                                         */
  const int32_t* h_pb_per_site;  /* m_s > 0, S entries                                         */
  int32_t n_freq;                /* N_omega >= 1                                               */
  const double* h_omega;         /* imaginary frequencies omega_j >= 0, strictly increasing    */
  int32_t n_k;                   /* N_k >= 1: the 1/N_k normalisation applied by finalize      */
  int32_t max_n_o, max_n_u;      /* largest band batch (n_o, n_u) any zmel_build call passes   */
  int32_t precision;             /* QSGW_PREC_FP64 | QSGW_PREC_MIXED                           */
  double occ_tol;                /* pair kept iff f_n*(1-f_n') > occ_tol; <0 selects 1e-12     */
  size_t workspace_bytes;        /* cap on the z workspace; 0 = library default (room for the  */
                                 /* larger of one band batch and ~32 Ki staged pairs).  If one */
                                 /* max_n_o*max_n_u batch does not fit under a non-zero cap,   */
                                 /* create fails with QSGW_ERR_ALLOC                           */
} qsgw_desc;

/* Create a context on the current CUDA device.  `cuda_stream` is a cudaStream_t (NULL =
 * legacy default stream) on which every later call is ordered.  Allocates the FP64
 * accumulator (N_omega * N_M * ld * 16 B), the z workspace and the weight table, and zeroes
 * the accumulator. */
int32_t qsgw_create(const qsgw_desc* desc, void* cuda_stream, qsgw_ctx** out);

/* Set P_s[I, alpha, beta] = <phi_alpha | M_I phi_beta> (Eq. 8 restricted to one muffin tin,
 * PAPER.md:130).  d_P: complex128, packed, site-major: for each site s a block
 * [m_s][b_s][b_s] (I slowest, beta fastest).  Copied/converted into the context. */
int32_t qsgw_set_product_tensor(qsgw_ctx* ctx, const void* d_P);

/* Stage (a) for one k-point and one band batch (Alg. 1 line 12).
 *   d_Ck  : complex128, column-major N_b x (>= n_begin+n_o), column = band n of C_k; element
 *           (beta, n) at d_Ck[n*ld_k + beta]; ld_k >= N_b.  Same memory as a row-major
 *           [band][orbital] array.
 *   d_Ckq : likewise for C_{k+q}, bands n'.
 *   Band batch: n in [n_begin, n_begin+n_o), n' in [np_begin, np_begin+n_u);
 *           n_o <= max_n_o, n_u <= max_n_u.
 *   d_z_out: optional complex128 [n_o][n_u][N_M] (I fastest) copy of the batch for tests;
 *           NULL keeps z internal only.  In mixed mode the exported values are the FP32 z
 *           widened to FP64.
 * The batch stays in the context until the next zmel_build. */
int32_t qsgw_zmel_build(qsgw_ctx* ctx, const void* d_Ck, int64_t ld_k, const void* d_Ckq,
                        int64_t ld_kq, int32_t n_begin, int32_t n_o, int32_t np_begin,
                        int32_t n_u, void* d_z_out);

/* Stage (b) for one band batch (Eq. 14; Alg. 1 lines 16-21).
 *   d_z   : NULL = use the batch built by the last zmel_build (the normal path; z never leaves
 *           the context).  Non-NULL = complex128 [n_o][n_u][N_M] (I fastest, the d_z_out layout),
 *           imported into the context first; lets stage (b) be driven with a caller-made z.
 *   d_eps_k, d_f_k   : float64[n_o]  energies (Ha) and occupations of the batch's bands n
 *   d_eps_kq, d_f_kq : float64[n_u]  same for n'
 *   With d_z == NULL, n_o and n_u must equal the last zmel_build's.
 * Adds into the accumulator (upper-triangle tiles only).  The library may stage the batch (its z and its
 * weights are computed now, stream-ordered; the caller's arrays are not read later) and run the accumulation
 * kernel once several band batches fill the z workspace (32 Ki pairs; for small N_M up to 256 Ki pairs within 1.5 GB); qsgw_chi0_finalize and qsgw_sync
 * accumulate whatever is staged, qsgw_reset drops it. */
int32_t qsgw_chi0_accumulate(qsgw_ctx* ctx, const void* d_z, const double* d_eps_k,
                             const double* d_f_k, const double* d_eps_kq, const double* d_f_kq,
                             int32_t n_o, int32_t n_u);

/* Convenience driver of the band-batch loop (Alg. 1 lines 9-23) for one k-point: splits
 * n in [0,n_o_total) x n' in [0,n_u_total) into batches of at most (max_n_o, max_n_u) and
 * calls zmel_build + chi0_accumulate for each.  Energies/occupations cover all bands. */
int32_t qsgw_chi0_add_kpoint(qsgw_ctx* ctx, const void* d_Ck, int64_t ld_k, const void* d_Ckq,
                             int64_t ld_kq, const double* d_eps_k, const double* d_f_k,
                             const double* d_eps_kq, const double* d_f_kq, int32_t n_o_total,
                             int32_t n_u_total);

/* The same for n_kpoints k-points at once (equivalent to n_kpoints calls of qsgw_chi0_add_kpoint): k-point k reads
 * d_Ck + k*stride_k and d_Ckq + k*stride_kq (strides in complex elements; a contiguous [k][band][orbital] array has
 * stride n_bands*ld) and rows k of d_eps_k, d_f_k (float64 [n_kpoints][n_o_total]) and d_eps_kq, d_f_kq
 * ([n_kpoints][n_u_total]).  When one k-point fits a band batch (n_o_total <= max_n_o, n_u_total <= max_n_u) the
 * k-points that fit the z workspace together are built by ONE stage (a) launch and ONE weight launch: small cells with
 * many k-points stop being bound by launch latency. */
int32_t qsgw_chi0_add_kpoints(qsgw_ctx* ctx, const void* d_Ck, int64_t ld_k, int64_t stride_k, const void* d_Ckq,
                              int64_t ld_kq, int64_t stride_kq, const double* d_eps_k, const double* d_f_k,
                              const double* d_eps_kq, const double* d_f_kq, int32_t n_o_total, int32_t n_u_total,
                              int32_t n_kpoints);

/* chi0[j][I][J] = acc/N_k as a full Hermitian matrix: d_chi0_out complex128
 * [n_freq][N_M][N_M], row-major.  May be called again after more accumulation. */
int32_t qsgw_chi0_finalize(qsgw_ctx* ctx, void* d_chi0_out);

/* Zero the accumulator and return to the state after set_product_tensor. */
int32_t qsgw_reset(qsgw_ctx* ctx);
/* Block until the context's stream is idle; reports deferred CUDA errors. */
int32_t qsgw_sync(qsgw_ctx* ctx);
void qsgw_destroy(qsgw_ctx* ctx);

/* Whole job from HOST buffers on an existing context: qsgw_reset, H2D of P and of every k-point's
 * arrays, the band-batch loop of all n_k_points k-points, finalize, D2H of the result.  Host arrays: h_P as
 * set_product_tensor; h_Ck complex128 [n_k_points][n_o][N_b] (row = band), h_Ckq [n_k_points][n_u][N_b];
 * h_eps_k,h_f_k float64 [n_k_points][n_o]; h_eps_kq,h_f_kq [n_k_points][n_u]; h_chi0_out complex128
 * [n_freq][N_M][N_M].  Pinned host memory makes the copies asynchronous; the library pins nothing itself.
 * The device staging buffers belong to the context (allocated by the first call, reused afterwards), the
 * copies and kernels run on the context's stream (results leave on a second stream while the last launches
 * run).  Synchronous: returns when h_chi0_out is complete.  *out_kernel_launches = kernels launched by
 * this call. */
int32_t qsgw_chi0_run_host(qsgw_ctx* ctx, const void* h_P, const void* h_Ck, const void* h_Ckq,
                           const double* h_eps_k, const double* h_f_k, const double* h_eps_kq,
                           const double* h_f_kq, int32_t n_k_points, int32_t n_o, int32_t n_u,
                           void* h_chi0_out, int64_t* out_kernel_launches);

/* Screened Coulomb interaction on the imaginary axis from the polarization (the step after the chi0 build):
 *   eps_j = 1 - sqrt(v) chi0_j sqrt(v)                    Eq. (10)
 *   W^c_j = sqrt(v) (eps_j^-1 - 1) sqrt(v)                Eq. (19)
 * for every frequency j, FP64.  eps_j must be Hermitian positive definite (it is for chi0(i omega) <= 0,
 * PAPER.md:161); the inverse is formed by a blocked Cholesky factorisation on the FP64 tensor pipe.
 *   d_chi0   : complex128 [n_freq][N_M][N_M], row-major, full Hermitian (what qsgw_chi0_finalize writes)
 *   d_v      : float64 [N_M], Coulomb eigenvalues v_mu > 0
 *   d_wc_out : complex128 [n_freq][N_M][N_M], full Hermitian; may not alias d_chi0
 *   d_info   : int32 on the device: 0, or 1 + the index of the first non-positive pivot (result then undefined)
 * Stream-ordered on `cuda_stream` (workspace from the stream-ordered allocator); does not synchronise.
 * On failure the text is in qsgw_last_create_error(). */
int32_t qsgw_wc_from_chi0(int32_t n_m, int32_t n_freq, const void* d_chi0, const double* d_v, void* d_wc_out,
                          int32_t* d_info, void* cuda_stream);

/* chi0 in the orthonormal basis E_mu = sum_I M_I U[I, mu] that diagonalises the Coulomb matrix (Eq. 7,
 * PAPER.md:118; Eq. 8 is written in terms of E_mu): z_mu = sum_I U[I, mu] z_I, hence
 *   chi0_out[j] = U^H chi0[j] U        for every frequency j (two batched FP64 tensor-pipe GEMMs),
 * the representation Eqs. (10)/(19) and qsgw_wc_from_chi0 (with the eigenvalues v_mu) are stated in.
 *   d_chi0 : complex128 [n_freq][N_M][N_M] row-major;  d_U : complex128 [N_M][N_M] row-major, U[I][mu], unitary
 *   d_out  : complex128 [n_freq][N_M][N_M], Hermitian (upper triangle mirrored); may not alias d_chi0
 * Stream-ordered, no synchronisation; error text in qsgw_last_create_error(). */
int32_t qsgw_chi0_to_coulomb_basis(int32_t n_m, int32_t n_freq, const void* d_chi0, const void* d_U, void* d_out,
                                   void* cuda_stream);

/* The paper's own real-axis route (Eqs. 15-18; Alg. 1 lines 9-27).
 * A context whose n_freq "frequencies" are the histogram bins [edges[j], edges[j+1]) of the real axis (h_omega = any
 * increasing labels, e.g. the lower edges; they are not used by this path) accumulates the bin-integrated spectral
 * weight
 *   A[j][I, J] = (1/N_k) sum_k sum_{pairs with w != 0} w(pair, j, k) conj(z[pair, I]) z[pair, J]        (Eq. 15 without pi/i)
 * qsgw_imchi_add_batch = Alg. 1 lines 12-21 for one k-point and band batch: stage (a) (as qsgw_zmel_build) and
 * the per-bin  Z_pair^dagger x W_Zpair  products.  The weights are inputs (the paper computes its tetrahedron weights,
 * Eqs. 16-17, on the CPU before the loop, Alg. 1 line 8) in CSR-by-bin form:
 *   d_bin_ptr : int32 [n_freq + 1], d_bin_ptr[0] = 0, non-decreasing, d_bin_ptr[n_freq] = nnz
 *   d_pair    : int32 [nnz]  pair index n_local * n_u + n'_local of the batch (n_local < n_o, n'_local < n_u)
 *   d_w       : float64 [nnz] weight of that pair in that bin (entries of one (pair, bin) add up)
 * The gather of Alg. 1 line 17 is a permutation applied when z is written (pairs sorted by the first bin that carries
 * them), so each bin multiplies one short contiguous row range; pairs without an entry cost nothing in stage (b).
 * Accumulates into the context's accumulator (qsgw_reset zeroes it, qsgw_chi0_finalize returns A with the Hermitian
 * mirror and 1/N_k); batches staged by qsgw_chi0_accumulate are flushed first.  QSGW_PREC_MIXED runs the per-bin products on
 * tcgen05 with FP16-split operands (three FP16 products unless "mixed_fp8" forces E5M2; <= 2e-5 per bin).
 * The summation order inside a bin is not fixed (atomic placement): results agree to rounding between runs. */
int32_t qsgw_imchi_add_batch(qsgw_ctx* ctx, const void* d_Ck, int64_t ld_k, const void* d_Ckq, int64_t ld_kq,
                             int32_t n_begin, int32_t n_o, int32_t np_begin, int32_t n_u, const int32_t* d_bin_ptr,
                             const int32_t* d_pair, const double* d_w, int32_t nnz);

/* Hilbert transform of the spectral part to the imaginary axis (Eq. 18; Alg. 1 line 27):
 *   out[i] = sum_j K[i][j] A[j],   K[i][j] = -log((R_j^2 + omega_i^2) / (L_j^2 + omega_i^2)) / (R_j - L_j),
 * the bracket of Eq. (14) at omega = i omega_i averaged over bin j = [L_j, R_j) = [d_edges[j], d_edges[j+1])
 * ("taking into account the size of histogram bins"; reading R20).
 *   d_edges : float64 [n_bins + 1], increasing, d_edges[0] > 0 when omega_out contains 0;  d_omega_out : float64 [n_out]
 *   d_A : complex128 [n_bins][N_M][N_M];  d_out : complex128 [n_out][N_M][N_M]; may not alias.  n_bins <= 384.
 * One streaming pass over A per 16 output frequencies (HBM-bound).  Stream-ordered; error text in
 * qsgw_last_create_error(). */
int32_t qsgw_hilbert_to_imag_axis(int32_t n_m, int32_t n_bins, const double* d_edges, int32_t n_out,
                                  const double* d_omega_out, const void* d_A, void* d_out, void* cuda_stream);

/* The same transform for targets omega_i ON THE REAL AXIS (Eq. 18 as printed: the Hermitian part of Pi from its spectral
 * part): K[i][j] = log|(omega_i^2 - L_j^2) / (omega_i^2 - R_j^2)| / (R_j - L_j), the principal value of
 * 1/(omega - w') - 1/(omega + w') averaged over bin j.  Logarithmically singular where omega_i sits on a bin edge: take the
 * targets inside bins (e.g. their centres).  Pi(omega_i) = out[i] - i pi A(omega_i) (the anti-Hermitian part is the
 * spectral part itself, reading R19).  Arguments as qsgw_hilbert_to_imag_axis. */
int32_t qsgw_hilbert_to_real_axis(int32_t n_m, int32_t n_bins, const double* d_edges, int32_t n_out,
                                  const double* d_omega_out, const void* d_A, void* d_out, void* cuda_stream);

/* Imaginary-axis part of the correlation self-energy for one k-point and one batch of intermediate states
 * (the step after W^c; Eq. (22); Alg. 2 lines 11-25 and 44):
 *   ZW^c[n', n, nu] = sum_i w^I_i(eps_qn - eps_{q-k,n'}) sum_mu z[n', n, mu] W^c[i][mu, nu]
 *   sigc[n, m]     += -(1/N_k) sum_{n', nu} ZW^c[n', n, nu] conj(z[n', m, nu])
 * with z[n', n, mu] = conj(Z_mu^{q-k n', q n}): the batch qsgw_zmel_build makes for d_Ck = C_{q-k} (bands n', the
 * n_all intermediate states) and d_Ckq = C_q (bands n, the n_qp states of the self-energy matrix).
 * Weights (Eq. 23; the paper defers to Aryasetiawan-Gunnarsson and prints no formula -- DESIGN.md reading R17):
 *   int d omega / 2 pi X(i omega) / (dE - i omega) = int_0^inf K(dE, omega) X(i omega) d omega for even X,
 *   K = dE / (pi (dE^2 + omega^2)), integrated exactly against the piecewise-linear interpolant of X on the context's
 *   mesh omega_0 = 0 < omega_1 < ... (X = 0 beyond the last point); dE = 0 gives weight 0.
 *   d_z      : NULL = the batch of the last qsgw_zmel_build (n_all = its n_o, n_qp = its n_u; in QSGW_PREC_MIXED
 *              that batch carries FP32-grade values), else complex128 [n_all][n_qp][N_M] (the d_z_out layout)
 *   d_eps_q  : float64 [n_qp]   eps_qn;      d_eps_qk : float64 [n_all]  eps_{q-k, n'} of the batch
 *   d_wc     : complex128 [n_freq][N_M][N_M] row-major, W^c(k, i omega_i) on the context's mesh (what
 *              qsgw_wc_from_chi0 writes); any matrix is accepted, Hermiticity is not assumed
 *   d_sigc   : complex128 [n_qp][n_qp] row-major, ACCUMULATED (the caller zeroes it before the first call);
 *              1/N_k is the context's n_k.  Not Hermitian: the weight carries eps_qn of the row index (Eq. 3
 *              symmetrises later).
 * QSGW_PREC_FP64: FP64 arithmetic on the FP64 tensor pipe (parity <= 1e-10).  QSGW_PREC_MIXED: the frequency loop ZW^c
 * runs on the tcgen05 tensor cores with z and W^c carried as FP16 pieces (FP32-grade products, three FP16 MMAs per
 * term; the paper runs this GEMM in TF32), FP32 sums over mu and the frequencies, the closing
 * contraction in FP64: relative Frobenius error of I^c <= 1e-5; option "sigc_f64" = 1 keeps the FP64 GEMM on the
 * context's FP32-grade z.  n_all <= max_n_o, n_qp <= max_n_u.  The context allocates its I^c workspace (two z-sized
 * buffers, the weight table and, in mixed mode, the FP16-split copies of z and W^c) at the first call.
 * Stream-ordered, does not synchronise; does not touch the chi0 accumulator or the staged batches. */
int32_t qsgw_sigc_imag_accumulate(qsgw_ctx* ctx, const void* d_z, const double* d_eps_q, const double* d_eps_qk,
                                  const void* d_wc, int32_t n_all, int32_t n_qp, void* d_sigc);

/* Per-stage device timing, for roofline measurement.  While enabled, every kernel launch of
 * the path is bracketed by CUDA events on the context's stream (Eq. 8 / Eq. 14 stages:
 * QSGW_STAGE_ZMEL, _WEIGHTS, _CHI0, _FINALIZE).  qsgw_stage_time_ms synchronises the stream,
 * returns the summed event time (ms) and launch count of `stage` since the last
 * qsgw_set_stage_timing call, and keeps accumulating.  Off by default (no events recorded). */
enum { QSGW_STAGE_ZMEL = 0, QSGW_STAGE_WEIGHTS = 1, QSGW_STAGE_CHI0 = 2, QSGW_STAGE_FINALIZE = 3,
       QSGW_N_STAGES = 4 };
int32_t qsgw_set_stage_timing(qsgw_ctx* ctx, int32_t enable);
int32_t qsgw_stage_time_ms(qsgw_ctx* ctx, int32_t stage, double* out_ms, int64_t* out_launches);

/* Roofline denominators measured on this device (MEASURED_PEAKS.json has no FP64 / TF32 tensor
 * figure): an issue-rate loop of register-resident MMAs with no memory traffic, timed with CUDA
 * events on a private stream (synchronous; a few tens of ms).  kind = QSGW_PEAK_FP64_MMA: FP64
 * tensor pipe (DMMA.8x8x4); QSGW_PEAK_TF32_MMA / QSGW_PEAK_F16_MMA: tcgen05.mma kind::tf32 128x128x8 /
 * kind::f16 128x128x16, A in TMEM, B in shared memory.  *out_tflops = real TFLOP/s (2 flop per FMA).
 * Does no work of the method. */
enum { QSGW_PEAK_FP64_MMA = 0, QSGW_PEAK_TF32_MMA = 1, QSGW_PEAK_F16_MMA = 2 };
int32_t qsgw_probe_peak(int32_t kind, double* out_tflops, double* out_ms);

/* Introspection (host side, no device work). */
const char* qsgw_last_error(const qsgw_ctx* ctx);       /* "" if none; valid until next call   */
const char* qsgw_last_create_error(void);               /* error text of a failed qsgw_create  */
int64_t qsgw_kernel_launches(const qsgw_ctx* ctx);      /* kernels launched by this context    */
int64_t qsgw_pairs_accumulated(const qsgw_ctx* ctx);    /* band pairs passed to stage (b)      */
size_t qsgw_device_bytes(const qsgw_ctx* ctx);          /* device memory owned by the context  */
int32_t qsgw_n_m(const qsgw_ctx* ctx);                  /* N_M                                 */
int32_t qsgw_n_b(const qsgw_ctx* ctx);                  /* N_b                                 */
const char* qsgw_version(void);

/* qsgw_chi0_to_coulomb_basis WITHOUT ANY ALLOCATION, for callers that cannot call cudaMalloc (code under CUDA graph
 * capture, tight serving loops, harnesses that forbid it).  Same arguments, layouts and result.  The scratch (padded chi0,
 * intermediate, padded U) lives in a file-scope device array of 33 * 256 * 256 complex128 elements (33 MiB) that every GPU
 * which loads the library holds until the process exits; the entry point calls no cudaMalloc, cudaFree, stream-ordered
 * allocator or allocating library routine (it sets kernel attributes on its first call per device).
 *   Limit: (2 n_freq + 1) * ceil64(n_m)^2 <= 33 * 256 * 256, e.g. n_m <= 256 at 16 frequencies, n_m <= 512 at 3;
 *   larger problems are rejected with QSGW_ERR_ALLOC and a text in qsgw_last_create_error().
 * All calls share the one array per GPU (it keeps the last call's contents; nothing in it has to start at zero, every
 * element that is read is written first by the same call): calls that OVERLAP on the GPU (different streams, no ordering
 * between them) race on it.  Stream-ordered on `cuda_stream`, no synchronisation. */
int32_t qsgw_chi0_to_coulomb_basis_static(int32_t n_m, int32_t n_freq, const void* d_chi0, const void* d_U, void* d_out,
                                          void* cuda_stream);

/* Orthonormal mixed product basis that diagonalises the Coulomb matrix (row f4; Eq. 7):
 *   |E_mu> = sum_I z_{mu I} |M_I>,   sum_J (v_IJ - v_mu O_IJ) z_{mu J} = 0,   z^H O z = 1,
 * O_IJ = <M_I|M_J> the overlap matrix (Hermitian positive definite), v_IJ = <M_I|v|M_J> the Coulomb matrix (Hermitian) of
 * the non-orthogonal basis {M_I}.  Eigenvalues in DESCENDING order ("mu = 1 corresponds to the largest eigenvalue",
 * PAPER.md:128).
 *   d_v, d_O   : device complex128 [N_M][N_M] row-major; the upper triangle (and the real part of the diagonal) is read
 *   d_vmu_out  : device double [N_M]
 *   d_U_out    : device complex128 [N_M][N_M] row-major, U[I][mu] = z_{mu I} (the layout qsgw_chi0_to_coulomb_basis takes;
 *                a column is fixed up to a phase, and up to a unitary mixing inside a degenerate eigenvalue)
 *   h_info     : HOST int32 (optional): 0 | 1 + index of the first non-positive Cholesky pivot of O (not positive
 *                definite; QSGW_ERR_INVALID_ARG) | -1 the Jacobi iteration did not converge (QSGW_ERR_CUDA)
 *   h_sweeps   : HOST int32 (optional): Jacobi sweeps taken
 * Method: blocked Cholesky O = L L^H and X = L^-1 on the FP64 tensor pipe, C = X v X^H, two-sided block Jacobi with the
 * round-robin parallel ordering (64 x 64 subproblems in shared memory, their unitaries applied to C and Q by 64^3 complex
 * GEMMs on the FP64 tensor pipe; process-wide option "eig_blocked" = 0: element-wise rounds), U = X^H Q.
 * SYNCHRONISES `cuda_stream` once per sweep (convergence is decided on the host).  Error text in qsgw_last_create_error(). */
int32_t qsgw_coulomb_eigenbasis(int32_t n_m, const void* d_v, const void* d_O, double* d_vmu_out, void* d_U_out,
                                int32_t* h_info, int32_t* h_sweeps, void* cuda_stream);

/* Interstitial-plane-wave (IPW) block of the matrix elements (row f4; Eqs. 4, 5 and 8; DESIGN.md
 * reading R21).  For the product functions of the mixed product basis that are IPWs, M_I = P_{G_I} of Eq. (5), the matrix
 * element is an integral over the interstitial region of three plane-wave expansions:
 *   z[n, n', I] = sum_{alpha, beta} conj(Bkq[n', alpha]) theta(g_k[beta] - g_kq[alpha] - g_ipw[I]) Bk[n, beta]
 * per unit cell volume, the same bilinear form and band-index convention as the muffin-tin block of qsgw_zmel_build
 * (bands n' = the conjugated eigenfunction that the IPW multiplies; crystal momenta k_kq + k_ipw = k_k, any umklapp is
 * the caller's shift of an integer list).  theta(g) = (1/Omega) int_cell Theta_I(r) exp(i G.r) d^3r are the Fourier
 * coefficients of the interstitial indicator function, an INPUT table on the integer box |g_i| <= L_i.
 *   h_L      : HOST int32[3], box half extents;  d_theta : device complex128 [2 L0 + 1][2 L1 + 1][2 L2 + 1], theta[g + L];
 *              a difference outside the box counts as theta = 0
 *   d_g_kq   : device int32 [n_pw_kq][3], d_g_k : [n_pw_k][3], d_g_ipw : [n_ipw][3]   integer reciprocal vectors
 *   d_Bk     : device complex128, beta^n_G at d_Bk[n * ld_k + beta] (n_o bands);  d_Bkq : d_Bkq[n' * ld_kq + alpha] (n_u bands)
 *   d_z_out  : device complex128, z[n, n', I] at d_z_out[(n * n_u + n') * ld_z + I]: with ld_z = N_MT + n_ipw and the pointer
 *              advanced by N_MT the block lands beside the muffin-tin columns of a z array for qsgw_chi0_accumulate(d_z).
 * Stream-ordered on `cuda_stream` (gather of the structured product tensor + two FP64 tensor-pipe GEMMs, workspace from
 * the stream-ordered allocator, at most 1 GiB + the output-sized buffer); no synchronisation.  Error text in
 * qsgw_last_create_error(). */
int32_t qsgw_zmel_ipw_build(const int32_t* h_L, const void* d_theta, int32_t n_pw_kq, const int32_t* d_g_kq, int32_t n_pw_k,
                            const int32_t* d_g_k, int32_t n_ipw, const int32_t* d_g_ipw, const void* d_Bk, int64_t ld_k,
                            int32_t n_o, const void* d_Bkq, int64_t ld_kq, int32_t n_u, void* d_z_out, int64_t ld_z,
                            void* cuda_stream);

/* Mixed mode: what the device-side selection did since the last qsgw_reset (synchronises the stream):
 * stage (b) launches in all, those that ran the E5M2 correction products, and the smallest effective pair
 * count P_eff any launch saw (qsgw.h, QSGW_PREC_MIXED).  QSGW_ERR_STATE in FP64 mode. */
int32_t qsgw_mixed_stats(qsgw_ctx* ctx, int64_t* out_launches, int64_t* out_launches_fp8,
                         double* out_min_effective_pairs);

/* Tuning and test knobs (never read from the environment).  ctx != NULL, allowed while nothing is staged:
 *   "stage_batches"   n >= 1   band batches staged per stage (b) launch (capped by the workspace)
 *   "skip_dead_stages" 0 | 1 | 2  stage (b) runs every staged 32-pair stage | skips the stages without weight at any frequency
 *                              (metals: whole bands fail the occupation filter) for flushes of >= 4 M staged matrix elements
 *                              (default; two small extra launches per flush) | always
 *   "zmel_dmma"       0 | 1    stage (a) step 2 on CUDA cores | on the FP64 tensor pipe (default 1)
 *   "zmel_direct"     0 | 1 | 2  mixed context, stage (a): FP64 tensor-pipe kernel + conversion to the FP16-split rows | the tcgen05
 *                              kernel that writes those rows itself for launches of >= 8 M matrix elements outside the binned
 *                              real-axis path (default; sites of at most 32 orbitals) | always.  The tcgen05 kernel forms z with FP32-grade products and FP32 sums
 *                              (error <= 8e-7 of max |z| instead of 2.5e-7) and scales by a bound of max |z|
 *   "mixed_fp8"       0 | 1 | 2  E5M2 correction products never | always | chosen on the device (default 2)
 *   "mixed_fp8_threshold_x100"  T*100: automatic choice takes E5M2 when P_eff >= T * N_M (default T = 4)
 *   "mixed_window"    1..64    pipeline stages per TMEM drain window (default 8)
 *   "mixed_pair"      0 | 1    mixed stage (b): one CTA per (tile, frequency) | CTA pairs (tcgen05 cta_group::2) that share
 *                              the B tiles of two consecutive frequencies (default 1; the binned real-axis path always uses 0)
 *   "sigc_f64"        0 | 1    mixed context: qsgw_sigc_imag_accumulate on tcgen05 (default) | with the FP64 GEMM
 *   "sigc_fp8"        0 | 1    mixed context, tcgen05 path of qsgw_sigc_imag_accumulate: three FP16 products per term | FP16 main
 *                              product + two E5M2 correction products (default 1)
 *   "e2e_groups"      1..4     frequency groups of the last launch of qsgw_chi0_run_host (default 4)
 * ctx == NULL, process-wide:
 *   "wc_graph"        0 | 1 | 2  qsgw_wc_from_chi0: plain launches | CUDA graph with fallback (default) | graph or fail
 *   "eig_blocked"     0 | 1    qsgw_coulomb_eigenbasis: element-wise Jacobi rounds | block rounds on the tensor pipe (default 1)
 *   "trim_workspace"  bytes    qsgw_wc_from_chi0 / qsgw_chi0_to_coulomb_basis keep their stream-ordered workspace in a
 *                              private memory pool between calls; this returns all but `bytes` of it to the driver
 * Unknown key or value out of range: QSGW_ERR_INVALID_ARG. */
int32_t qsgw_set_option(qsgw_ctx* ctx, const char* key, int64_t value);

#ifdef __cplusplus
}
#endif
#endif /* QSGW_H_ */
