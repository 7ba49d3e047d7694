// Stage (b), FP64 mode: acc_j[I,J] += sum_p conj(z[p,I]) w_j(p) z[p,J] for one 64x64 tile and one
// frequency per CTA (Eq. 14; Alg. 1 lines 16-21), on the FP64 tensor
// pipe (DMMA.8x8x4), and the finalize kernel (1/N_k, Hermitian mirror).
//
// The 64-column x 32-pair tiles of both planes (z = x + i y) arrive by one 4-D TMA box per operand with the
// 128-byte swizzle; w_j(p) for the stage arrives by a 1-D bulk copy; the frequency-scaled operand
// w*z is formed in registers.
#include "kernels.h"
#include "ptx.cuh"

namespace qsgw {

namespace {

constexpr int STAGES = 3;

// 3M form (three real products per complex one, 25 % fewer DMMAs than the four-product form):
//   T1 += x_I (w x_J),  T2 += y_I (w y_J),  T3 += (x_I + y_I) (w (y_J - x_J));   Re = T1 + T2,  Im = T3 + T1 - T2.
// 8 warps (2 along I x 4 along J), each a 32x16 complex sub-tile = 3 x 16 FP64 accumulator pairs; per 4 pairs a
// warp loads 12 operand doubles and issues 24 DMMAs.  Normwise error ~1e-15 (the parity bar is 1e-11).
constexpr int kThreads3M = 256;
constexpr int KP3 = kChi0F64KP3M;     // pairs per stage (1 CTA/SM)
constexpr int OPER_BYTES3 = 2 * 4 * KP3 * 128;
constexpr int PLANE_BYTES3 = 4 * KP3 * 128;
constexpr int CGRP_BYTES3 = KP3 * 128;
constexpr int W_BYTES3 = KP3 * 8;
constexpr int SMEM_OPERANDS3 = STAGES * 2 * OPER_BYTES3;
constexpr int SMEM_BYTES3 = SMEM_OPERANDS3 + STAGES * W_BYTES3 + 2 * STAGES * 8 + 1024 /*align slack*/;

// Three CTA shapes over the same 64-column TMA boxes (KIND):
//   0 full     64 x 64: 8 warps 2 (I) x 4 (J), 32 x 16 sub-tiles                      -- off-diagonal tiles
//   1 half     64 x 32 at column offset 0 or 32: warps 4 x 2, 16 x 16 sub-tiles       -- last tile column when its last 32
//              columns are padding (N_M mod 64 in 1..32); right half of a diagonal tile
//   2 quarter  32 x 32 (rows and columns 0..31): warps 2 x 4, 16 x 8 sub-tiles        -- upper-left block of a diagonal tile
// A diagonal tile is computed as half (columns 32..63) + quarter: 3/4 of the DMMAs of a full tile (its lower-left
// 32 x 32 block is never needed: finalize mirrors the upper triangle).
template <int KIND>
__device__ __forceinline__ void chi0_f64_3m_body(const Chi0F64Args& a, const unsigned block) {
  constexpr int MI = KIND == 0 ? 4 : 2;
  constexpr int NI = KIND == 2 ? 1 : 2;
  extern __shared__ unsigned char smem_dyn[];
  const uint32_t raw = smem_u32(smem_dyn);
  const uint32_t base = (raw + 1023u) & ~1023u;
  unsigned char* sm = smem_dyn + (base - raw);
  double* wsm = reinterpret_cast<double*>(sm + SMEM_OPERANDS3);
  uint64_t* full = reinterpret_cast<uint64_t*>(sm + SMEM_OPERANDS3 + STAGES * W_BYTES3);
  uint64_t* empty = full + STAGES;

  const int tid = threadIdx.x;
  const int lane = tid & 31, warp = tid >> 5;
  const int g = lane >> 2, t = lane & 3;
  const int wm = KIND == 1 ? warp >> 1 : warp >> 2, wn = KIND == 1 ? warp & 1 : warp & 3;

  // blockIdx.x = ((tile * n_freq) + j) * split + chunk: `split` CTAs share the staged pairs of a (tile, j) when
  // the grid would not fill the SMs; their partial sums meet in the accumulator by atomic adds
  const int chunk = block % a.split, bid = block / a.split;
  const int j = a.j0 + bid % a.n_freq;
  const int tile = bid / a.n_freq;
  const int4 tq = a.d_tiles[(KIND == 0 ? 0 : KIND == 1 ? a.n_tiles : a.n_tiles + a.n_tiles_half) + tile];
  const int2 tt = make_int2(tq.x, tq.y);
  const int col_cg = tq.z;                 // first 16-column group of the CTA's columns inside the tile (half: 0 or 2)
  const bool diag = (tt.x == tt.y);
  const int n_all = a.d_live ? *a.d_n_live : (int)(a.n_pairs_padded / KP3);     // stages to run (dead stages are skipped)
  const bool mapped = a.d_live && n_all != (int)(a.n_pairs_padded / KP3);          // every stage live: no look-up
  int it_base = (int)((long long)n_all * chunk / a.split);
  int n_iter = (int)((long long)n_all * (chunk + 1) / a.split) - it_base;
  if (a.d_ranges) {           // binned path: only the stages that cover the rows carrying weight in this bin
    const int2 r = a.d_ranges[j];
    it_base = r.x / KP3;
    n_iter = r.y > r.x ? (r.y + KP3 - 1) / KP3 - it_base : 0;
    if (n_iter <= 0) return;
  }
  const double* wrow = a.wtab + (long long)j * a.kpad;

  if (tid == 0) {
    tma_prefetch_desc(&a.tmap_z);
    for (int s = 0; s < STAGES; ++s) {
      mbar_init(&full[s], 1);
      mbar_init(&empty[s], kThreads3M / 32);
    }
    mbar_fence_init();
  }
  __syncthreads();

  const uint32_t stage_bytes = (diag ? OPER_BYTES3 : 2 * OPER_BYTES3) + W_BYTES3;
  auto issue = [&](int slot, int it) {
    unsigned char* dstA = sm + slot * (2 * OPER_BYTES3);
    mbar_arrive_expect_tx(&full[slot], stage_bytes);
    const int gi = mapped ? a.d_live[it_base + it] : it_base + it;
    tma_load_4d(dstA, &a.tmap_z, &full[slot], 0, gi * KP3, tt.x * 4, 0);
    if (!diag) tma_load_4d(dstA + OPER_BYTES3, &a.tmap_z, &full[slot], 0, gi * KP3, tt.y * 4, 0);
    bulk_load_1d(wsm + slot * KP3, wrow + (long long)gi * KP3, W_BYTES3, &full[slot]);
  };

  if (tid == 0) {
    for (int it = 0; it < STAGES - 1 && it < n_iter; ++it) issue(it, it);
  }

  // per-thread swizzled offsets: row r = 8*(q>>1) + 2t + (q&1); 16-byte chunk ^= r&7
  uint32_t thr_off[2][2];
#pragma unroll
  for (int s = 0; s < 2; ++s)
#pragma unroll
    for (int par = 0; par < 2; ++par)
      thr_off[s][par] = (uint32_t)((2 * t + s) * 128 + ((((4 * par + (g >> 1)) ^ (2 * t + s)) << 4) | ((g & 1) << 3)));

  double t1[MI][NI][2], t2[MI][NI][2], t3[MI][NI][2];
#pragma unroll
  for (int mi = 0; mi < MI; ++mi)
#pragma unroll
    for (int ni = 0; ni < NI; ++ni)
#pragma unroll
      for (int e = 0; e < 2; ++e) t1[mi][ni][e] = t2[mi][ni][e] = t3[mi][ni][e] = 0.0;

  for (int it = 0; it < n_iter; ++it) {
    const int slot = it % STAGES;
    if (tid == 0) {
      const int nxt = it + STAGES - 1;
      if (nxt < n_iter) {
        const int s2 = nxt % STAGES;
        if (nxt >= STAGES) mbar_wait(&empty[s2], ((nxt / STAGES) - 1) & 1);
        issue(s2, nxt);
      }
    }
    __syncwarp();
    mbar_wait(&full[slot], (it / STAGES) & 1);

    const uint32_t aBase = base + slot * (2 * OPER_BYTES3) + (KIND == 0 ? 2 * wm : wm) * CGRP_BYTES3;
    const uint32_t bBase = base + slot * (2 * OPER_BYTES3) + (diag ? 0 : OPER_BYTES3) +
                           (col_cg + (KIND == 2 ? wn >> 1 : wn)) * CGRP_BYTES3;
    const uint32_t wBase = base + SMEM_OPERANDS3 + slot * W_BYTES3;

#pragma unroll
    for (int q = 0; q < KP3 / 4; ++q) {
      const uint32_t rq = (uint32_t)((q >> 1) * 1024);
      const double w = ld_shared_f64(wBase + (uint32_t)((8 * (q >> 1) + 2 * t + (q & 1)) * 8));
      double ax[MI], ay[MI], as[MI], bx[NI], by[NI], bd[NI];
#pragma unroll
      for (int mi = 0; mi < MI; ++mi) {
        const uint32_t ad = aBase + (mi >> 1) * CGRP_BYTES3 + rq + thr_off[q & 1][mi & 1];
        ax[mi] = ld_shared_f64(ad);
        ay[mi] = ld_shared_f64(ad + PLANE_BYTES3);
        as[mi] = ax[mi] + ay[mi];
      }
#pragma unroll
      for (int ni = 0; ni < NI; ++ni) {
        const uint32_t ad = bBase + rq + thr_off[q & 1][KIND == 2 ? (wn & 1) : ni];
        bx[ni] = w * ld_shared_f64(ad);
        by[ni] = w * ld_shared_f64(ad + PLANE_BYTES3);
        bd[ni] = by[ni] - bx[ni];
      }
#pragma unroll
      for (int mi = 0; mi < MI; ++mi)
#pragma unroll
        for (int ni = 0; ni < NI; ++ni) {
          dmma884(t1[mi][ni][0], t1[mi][ni][1], ax[mi], bx[ni]);
          dmma884(t2[mi][ni][0], t2[mi][ni][1], ay[mi], by[ni]);
          dmma884(t3[mi][ni][0], t3[mi][ni][1], as[mi], bd[ni]);
        }
    }
    __syncwarp();
    if (lane == 0) mbar_arrive(&empty[slot]);
  }

  // epilogue: exclusive owner of (tile, j) -> plain read-modify-write
  const long long plane = (long long)a.n_m_pad * a.n_m_pad;
  double* are = a.acc_re + (long long)j * plane;
  double* aim = a.acc_im + (long long)j * plane;
#pragma unroll
  for (int mi = 0; mi < MI; ++mi) {
    const int row = tt.x * kTile + (MI * wm + mi) * 8 + g;
#pragma unroll
    for (int ni = 0; ni < NI; ++ni) {
      const int col = tt.y * kTile + 16 * col_cg + (KIND == 2 ? wn : 2 * wn + ni) * 8 + 2 * t;
      const long long off = (long long)row * a.n_m_pad + col;
      const double r0 = t1[mi][ni][0] + t2[mi][ni][0], r1 = t1[mi][ni][1] + t2[mi][ni][1];
      const double m0 = t3[mi][ni][0] + (t1[mi][ni][0] - t2[mi][ni][0]);
      const double m1 = t3[mi][ni][1] + (t1[mi][ni][1] - t2[mi][ni][1]);
      if (a.split > 1) {
        atomicAdd(are + off, r0);
        atomicAdd(are + off + 1, r1);
        atomicAdd(aim + off, m0);
        atomicAdd(aim + off + 1, m1);
      } else {
        double2 r = *reinterpret_cast<double2*>(are + off);
        r.x += r0;
        r.y += r1;
        *reinterpret_cast<double2*>(are + off) = r;
        double2 m = *reinterpret_cast<double2*>(aim + off);
        m.x += m0;
        m.y += m1;
        *reinterpret_cast<double2*>(aim + off) = m;
      }
    }
  }
}

// One grid for the three CTA shapes: the full tiles first, then the half and quarter tiles (short CTAs at the tail).
__global__ void __launch_bounds__(kThreads3M, 1) chi0_f64_3m_kernel(const __grid_constant__ Chi0F64Args a) {
  const unsigned per = (unsigned)(a.n_freq * a.split);
  const unsigned n_full = (unsigned)a.n_tiles * per, n_half = (unsigned)a.n_tiles_half * per;
  if (blockIdx.x < n_full) chi0_f64_3m_body<0>(a, blockIdx.x);
  else if (blockIdx.x < n_full + n_half) chi0_f64_3m_body<1>(a, blockIdx.x - n_full);
  else chi0_f64_3m_body<2>(a, blockIdx.x - n_full - n_half);
}

// chi0[j][I][J] = acc/N_k, lower = conj(upper), Im(diag) = 0  (Hermiticity)
__global__ void __launch_bounds__(256) finalize_kernel(const double* __restrict__ acc_re,
                                                       const double* __restrict__ acc_im, int n_m, int n_m_pad,
                                                       double inv_nk, double2* __restrict__ out) {
  __shared__ double tre[32][33], tim[32][33];
  const int bi = blockIdx.y, bj = blockIdx.x;
  if (bi > bj) return;
  const int j = blockIdx.z;
  const long long plane = (long long)n_m_pad * n_m_pad;
  const double* are = acc_re + (long long)j * plane;
  const double* aim = acc_im + (long long)j * plane;
  double2* o = out + (long long)j * n_m * n_m;
  const int tx = threadIdx.x & 31, ty = threadIdx.x >> 5;
  for (int r = ty; r < 32; r += 8) {
    const int I = bi * 32 + r, J = bj * 32 + tx;
    const long long off = (long long)I * n_m_pad + J;
    const double vr = are[off] * inv_nk, vi = aim[off] * inv_nk;
    tre[r][tx] = vr;
    tim[r][tx] = vi;
    if (bi != bj && I < n_m && J < n_m) o[(long long)I * n_m + J] = make_double2(vr, vi);
  }
  __syncthreads();
  if (bi != bj) {
    for (int r = ty; r < 32; r += 8) {
      const int I = bj * 32 + r, J = bi * 32 + tx;   // mirrored block: out[I][J] = conj(acc[J][I])
      if (I < n_m && J < n_m) o[(long long)I * n_m + J] = make_double2(tre[tx][r], -tim[tx][r]);
    }
  } else {
    for (int r = ty; r < 32; r += 8) {
      const int I = bi * 32 + r, J = bj * 32 + tx;
      if (I < n_m && J < n_m) {
        double2 v;
        if (r < tx) v = make_double2(tre[r][tx], tim[r][tx]);
        else if (r == tx) v = make_double2(tre[r][tx], 0.0);
        else v = make_double2(tre[tx][r], -tim[tx][r]);
        o[(long long)I * n_m + J] = v;
      }
    }
  }
}

}  // namespace

cudaError_t chi0_f64_configure() {
  return cudaFuncSetAttribute(chi0_f64_3m_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, SMEM_BYTES3);
}

cudaError_t launch_chi0_f64(const Chi0F64Args& a_in, cudaStream_t s) {
  if (a_in.n_pairs_padded <= 0 || a_in.n_tiles + a_in.n_tiles_half + a_in.n_tiles_quarter <= 0) return cudaSuccess;
  Chi0F64Args a = a_in;
  a.split = 1;
  if (!a.d_ranges) {
    // Few work items (1 CTA/SM): split the staged pairs over 2..4 CTAs per item when that shortens the schedule.
    // Estimate in units of one full tile (half tiles 0.5, quarter tiles 0.3), CTAs dispatched longest first:
    //   length(sp) = max(units / SMs, largest item / sp) + (half the smallest item) / sp + 0.01 (sp - 1)
    // (the last term: the atomic epilogues of split items).
    const int n_sm = a.n_sm;
    const long long items = (long long)(a.n_tiles + a.n_tiles_half + a.n_tiles_quarter) * a.n_freq, n_it = a.n_pairs_padded / KP3;
    const double units = ((double)a.n_tiles + 0.5 * a.n_tiles_half + 0.3 * a.n_tiles_quarter) * a.n_freq;
    const double largest = a.n_tiles ? 1.0 : (a.n_tiles_half ? 0.5 : 0.3);
    const double tail = 0.5 * (a.n_tiles_quarter ? 0.3 : (a.n_tiles_half ? 0.5 : 1.0));
    double best = 1e300;
    for (int sp = 1; sp <= 4; ++sp) {
      if (sp > 1 && (n_it < 16 * sp || items * sp > 16LL * n_sm)) break;
      const double len = fmax(units / n_sm, largest / sp) + tail / sp + 0.01 * (sp - 1);
      if (len < best) { best = len; a.split = sp; }
    }
  }
  chi0_f64_3m_kernel<<<dim3((unsigned)((a.n_tiles + a.n_tiles_half + a.n_tiles_quarter) * a.n_freq * a.split)), kThreads3M,
                       SMEM_BYTES3, s>>>(a);
  return cudaGetLastError();
}

cudaError_t launch_finalize(const double* acc_re, const double* acc_im, int n_m, int n_m_pad, int n_freq,
                            double inv_nk, double2* out, cudaStream_t s) {
  const int nb = (n_m + 31) / 32;
  dim3 grid(nb, nb, n_freq);
  finalize_kernel<<<grid, 256, 0, s>>>(acc_re, acc_im, n_m, n_m_pad, inv_nk, out);
  return cudaGetLastError();
}

}  // namespace qsgw
