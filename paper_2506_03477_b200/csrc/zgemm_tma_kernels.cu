// Batched complex FP64 GEMM on the FP64 tensor pipe (DMMA.8x8x4) with TMA-staged operands (kernels.h ZgemmArgs).
// It carries the blocked Cholesky inverse of W^c (Eqs. 10, 19), the basis rotation U^H chi0 U (Eqs. 7, 8) and both
// GEMMs of the imaginary-axis correlation self-energy I^c (Eq. 22; Alg. 2 lines 23 and 44).
//
//   One CTA = one 64x64 tile of C: 8 compute warps (2 along M x 4 along N, each a 32x16 complex sub-tile) + one
//   producer warp.  Operands stay complex128 interleaved: every 16-deep contraction step arrives as TMA boxes of
//   128-byte rows with the 128-byte swizzle (zero-filled out of bounds, so extents are arbitrary):
//     k-contiguous operand   [tile row][k]:  2 boxes {8 complex k, 64 rows}      -> smem [k half][row][128 B]
//     mn-contiguous operand  [k][tile col]:  8 boxes {8 complex cols, 16 k rows} -> smem [col group][k][128 B]
//   A DMMA fragment is then one conflict-free 16-byte shared load per thread in all four operand layouts (four
//   128-byte wavefronts per warp load = the minimum for 512 bytes).
//   Complex product in 3M form: T1 += x u, T2 += y v, T3 += (x + y)(u + v); Re = T1 - T2, Im = T3 - T1 - T2
//   (24 DMMAs per 4-deep step and warp instead of 32); a conjugated operand flips the sign of its imaginary part
//   on load; the optional row scale (the quadrature weight of Alg. 2 line 18) multiplies the A fragment in registers.
#include "kernels.h"
#include "ptx.cuh"

namespace qsgw {

namespace {

constexpr int kZT = 64;                   // tile edge
constexpr int kZK = 16;                   // contraction depth per pipeline stage
constexpr int kZStages = 4;
constexpr int kZOper = kZT * kZK * 16;    // bytes of one operand stage (16 KB)
constexpr int kZThreads = 288;            // 8 compute warps + 1 producer warp
constexpr int kZSmem = kZStages * 2 * kZOper + 2 * kZStages * 8 + 1024 /*align slack*/;

struct ZKernelArgs {
  CUtensorMap tmA, tmB;         // dims {2*inner, outer, rep, batch}
  double2* C;
  long long ldc, sC;
  int m, n, k, reps, split, tri, beta_one;
  int a_rep, a_batch, b_rep, b_batch;    // 1: the map has that dimension, 0: operand shared (coordinate 0)
  double alpha;
  const double* row_scale;
  long long ld_scale;
};

__device__ __forceinline__ double2 ld_shared_f64x2(uint32_t addr) {
  double2 v;
  asm volatile("ld.shared.v2.f64 {%0, %1}, [%2];" : "=d"(v.x), "=d"(v.y) : "r"(addr));
  return v;
}

template <bool A_KC, bool B_KC>
__global__ void __launch_bounds__(kZThreads, 1) zgemm_tma_kernel(const __grid_constant__ ZKernelArgs a) {
  // tile order: groups of 8 tile columns, tile rows fastest inside a group, so that the CTAs resident at one time share
  // a narrow slab of B (and a few row panels of A) in L2 instead of streaming all of B per wave
  int tj, ti;
  {
    const int nN = gridDim.x, nM = gridDim.y, pid = blockIdx.y * nN + blockIdx.x;
    const int grp = pid / (8 * nM), first = grp * 8, width = min(8, nN - first), r = pid - grp * 8 * nM;
    ti = r / width;
    tj = first + r - ti * width;
  }
  if ((a.tri == 1 || a.tri == 2) && tj > ti) return;
  extern __shared__ unsigned char smem_dyn[];
  const uint32_t raw = smem_u32(smem_dyn);
  const uint32_t base = (raw + 1023u) & ~1023u;
  unsigned char* sm = smem_dyn + (base - raw);
  uint64_t* full = reinterpret_cast<uint64_t*>(sm + kZStages * 2 * kZOper);
  uint64_t* empty = full + kZStages;

  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int batch = blockIdx.z / a.split, chunk = blockIdx.z % a.split;
  const int r0 = (int)((long long)a.reps * chunk / a.split), r1 = (int)((long long)a.reps * (chunk + 1) / a.split);
  const int k0 = (a.tri == 2) ? kZT * max(ti, tj) : (a.tri == 3 ? kZT * tj : 0);
  const int kt0 = k0 / kZK, n_kt = (a.k + kZK - 1) / kZK - kt0;       // stages per repetition
  const int n_it = (r1 - r0) * n_kt;

  if (tid == 0) {
    tma_prefetch_desc(&a.tmA);
    tma_prefetch_desc(&a.tmB);
    for (int s = 0; s < kZStages; ++s) {
      mbar_init(&full[s], 1);
      mbar_init(&empty[s], 8);
    }
    mbar_fence_init();
  }
  __syncthreads();

  if (warp == 8) {
    // ------------------------------------------------------------------ producer
    if (lane == 0) {
      for (int it = 0; it < n_it; ++it) {
        const int slot = it % kZStages;
        if (it >= kZStages) mbar_wait(&empty[slot], ((it / kZStages) - 1) & 1);
        const int rep = r0 + it / n_kt, kk = (kt0 + it % n_kt) * kZK;
        unsigned char* dA = sm + slot * 2 * kZOper;
        unsigned char* dB = dA + kZOper;
        mbar_arrive_expect_tx(&full[slot], 2 * kZOper);
        const int za2 = a.a_rep ? rep : 0, za3 = a.a_batch ? batch : 0;
        const int zb2 = a.b_rep ? rep : 0, zb3 = a.b_batch ? batch : 0;
        if (A_KC) {
#pragma unroll
          for (int h = 0; h < 2; ++h) tma_load_4d(dA + h * 8192, &a.tmA, &full[slot], 2 * (kk + 8 * h), ti * kZT, za2, za3);
        } else {
#pragma unroll
          for (int cg = 0; cg < 8; ++cg) tma_load_4d(dA + cg * 2048, &a.tmA, &full[slot], 2 * (ti * kZT + 8 * cg), kk, za2, za3);
        }
        if (B_KC) {
#pragma unroll
          for (int h = 0; h < 2; ++h) tma_load_4d(dB + h * 8192, &a.tmB, &full[slot], 2 * (kk + 8 * h), tj * kZT, zb2, zb3);
        } else {
#pragma unroll
          for (int cg = 0; cg < 8; ++cg) tma_load_4d(dB + cg * 2048, &a.tmB, &full[slot], 2 * (tj * kZT + 8 * cg), kk, zb2, zb3);
        }
      }
    }
    return;
  }

  // -------------------------------------------------------------------- compute warps
  const int g = lane >> 2, t = lane & 3;
  const int wm = warp >> 2, wn = warp & 3;
  // per-thread fragment offsets inside an operand stage, for the four 4-deep steps q of a stage.  Step q contracts the
  // k rows 8 (q >> 1) + 2 t + (q & 1) (t = lane & 3; the order of the contraction is free): a 16-byte shared load is
  // served per quarter-warp (lanes 8i..8i+7 = two values of g, all t), and with this mapping its 8 lanes hit the 8
  // distinct 16-byte chunks of a 128-byte row set (k = 4 (q & 1) + t would make the two g collide: 2x the wavefronts).
  uint32_t offA[4][4], offB[4][2];
#pragma unroll
  for (int q = 0; q < 4; ++q) {
    const int kl = 2 * t + (q & 1);            // k inside the 8-deep half
    const int kq = 8 * (q >> 1) + kl;          // k inside the stage
#pragma unroll
    for (int mi = 0; mi < 4; ++mi)
      offA[q][mi] = A_KC ? (uint32_t)((q >> 1) * 8192 + (32 * wm + 8 * mi + g) * 128 + ((kl ^ g) << 4))
                         : (uint32_t)((4 * wm + mi) * 2048 + kq * 128 + ((g ^ (kq & 7)) << 4));
#pragma unroll
    for (int ni = 0; ni < 2; ++ni)
      offB[q][ni] = B_KC ? (uint32_t)((q >> 1) * 8192 + (16 * wn + 8 * ni + g) * 128 + ((kl ^ g) << 4))
                         : (uint32_t)((2 * wn + ni) * 2048 + kq * 128 + ((g ^ (kq & 7)) << 4));
  }

  double t1[4][2][2], t2[4][2][2], t3[4][2][2];
#pragma unroll
  for (int mi = 0; mi < 4; ++mi)
#pragma unroll
    for (int ni = 0; ni < 2; ++ni)
#pragma unroll
      for (int e = 0; e < 2; ++e) t1[mi][ni][e] = t2[mi][ni][e] = t3[mi][ni][e] = 0.0;

  double sc[4] = {1.0, 1.0, 1.0, 1.0};
  int it = 0;
  for (int rep = r0; rep < r1; ++rep) {
    if (a.row_scale) {
#pragma unroll
      for (int mi = 0; mi < 4; ++mi) {
        const int row = ti * kZT + 32 * wm + 8 * mi + g;
        sc[mi] = row < a.m ? a.row_scale[(long long)rep * a.ld_scale + row] : 0.0;
      }
    }
    for (int kt = 0; kt < n_kt; ++kt, ++it) {
      const int slot = it % kZStages;
      mbar_wait(&full[slot], (it / kZStages) & 1);
      const uint32_t aB = base + slot * 2 * kZOper, bB = aB + kZOper;
#pragma unroll
      for (int q = 0; q < 4; ++q) {
        double fx[4], fy[4], fs[4], hx[2], hy[2], hs[2];
#pragma unroll
        for (int mi = 0; mi < 4; ++mi) {
          const double2 v = ld_shared_f64x2(aB + offA[q][mi]);
          fx[mi] = v.x * sc[mi];
          fy[mi] = (A_KC ? v.y : -v.y) * sc[mi];
          fs[mi] = fx[mi] + fy[mi];
        }
#pragma unroll
        for (int ni = 0; ni < 2; ++ni) {
          const double2 v = ld_shared_f64x2(bB + offB[q][ni]);
          hx[ni] = v.x;
          hy[ni] = B_KC ? -v.y : v.y;
          hs[ni] = hx[ni] + hy[ni];
        }
#pragma unroll
        for (int mi = 0; mi < 4; ++mi)
#pragma unroll
          for (int ni = 0; ni < 2; ++ni) {
            dmma884(t1[mi][ni][0], t1[mi][ni][1], fx[mi], hx[ni]);
            dmma884(t2[mi][ni][0], t2[mi][ni][1], fy[mi], hy[ni]);
            dmma884(t3[mi][ni][0], t3[mi][ni][1], fs[mi], hs[ni]);
          }
      }
      __syncwarp();
      if (lane == 0) mbar_arrive(&empty[slot]);
    }
  }

  // (x + i y)(u + i v): Re = xu - yv = T1 - T2,  Im = (x + y)(u + v) - xu - yv = T3 - T1 - T2
  double2* Cp = a.C + (long long)batch * a.sC;
#pragma unroll
  for (int mi = 0; mi < 4; ++mi) {
    const int row = ti * kZT + 32 * wm + 8 * mi + g;
    if (row >= a.m) continue;
#pragma unroll
    for (int ni = 0; ni < 2; ++ni) {
      const int col = tj * kZT + 16 * wn + 8 * ni + 2 * t;
      double2* c = Cp + (long long)row * a.ldc + col;
#pragma unroll
      for (int e = 0; e < 2; ++e) {
        if (col + e >= a.n) continue;
        double2 v = make_double2(a.alpha * (t1[mi][ni][e] - t2[mi][ni][e]),
                                 a.alpha * (t3[mi][ni][e] - t1[mi][ni][e] - t2[mi][ni][e]));
        if (a.split > 1) {
          atomicAdd(&c[e].x, v.x);
          atomicAdd(&c[e].y, v.y);
        } else {
          if (a.beta_one) {
            const double2 o = c[e];
            v.x += o.x;
            v.y += o.y;
          }
          c[e] = v;
        }
      }
    }
  }
}

template <bool A_KC, bool B_KC>
cudaError_t launch_t(const ZKernelArgs& k, dim3 grid, cudaStream_t s) {
  zgemm_tma_kernel<A_KC, B_KC><<<grid, kZThreads, kZSmem, s>>>(k);
  return cudaGetLastError();
}

}  // namespace

cudaError_t zgemm_configure() {
  cudaError_t e = cudaFuncSetAttribute(zgemm_tma_kernel<true, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, kZSmem);
  if (e == cudaSuccess) e = cudaFuncSetAttribute(zgemm_tma_kernel<true, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, kZSmem);
  if (e == cudaSuccess) e = cudaFuncSetAttribute(zgemm_tma_kernel<false, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, kZSmem);
  if (e == cudaSuccess) e = cudaFuncSetAttribute(zgemm_tma_kernel<false, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, kZSmem);
  return e;
}

cudaError_t launch_zgemm(bool a_kc, bool b_kc, const ZgemmArgs& a, cudaStream_t s) {
  if (a.m <= 0 || a.n <= 0 || a.k <= 0 || a.batch <= 0 || a.reps <= 0) return cudaSuccess;
  if (a.split > 1 && !a.beta_one) return cudaErrorInvalidValue;
  ZKernelArgs k;
  k.C = a.C;
  k.ldc = a.ldc;
  k.sC = a.sC;
  k.m = a.m;
  k.n = a.n;
  k.k = a.k;
  k.reps = a.reps;
  k.split = a.split < 1 ? 1 : (a.split > a.reps ? a.reps : a.split);
  k.tri = a.tri;
  k.beta_one = a.beta_one;
  k.alpha = a.alpha;
  k.row_scale = a.row_scale;
  k.ld_scale = a.ld_scale;
  k.a_rep = (a.reps > 1 && a.rA != 0) ? 1 : 0;
  k.b_rep = (a.reps > 1 && a.rB != 0) ? 1 : 0;
  k.a_batch = (a.batch > 1 && a.sA != 0) ? 1 : 0;
  k.b_batch = (a.batch > 1 && a.sB != 0) ? 1 : 0;
  // stored extents: k-contiguous [rows][k], mn-contiguous [k][cols]
  cudaError_t e = make_zmap(&k.tmA, a.A, a_kc ? a.k : a.m, a_kc ? a.m : a.k, a.lda, k.a_rep ? a.reps : 1, a.rA,
                            k.a_batch ? a.batch : 1, a.sA, a_kc ? kZT : kZK);
  if (e != cudaSuccess) return e;
  e = make_zmap(&k.tmB, a.B, b_kc ? a.k : a.n, b_kc ? a.n : a.k, a.ldb, k.b_rep ? a.reps : 1, a.rB,
                k.b_batch ? a.batch : 1, a.sB, b_kc ? kZT : kZK);
  if (e != cudaSuccess) return e;
  const dim3 grid((unsigned)((a.n + kZT - 1) / kZT), (unsigned)((a.m + kZT - 1) / kZT), (unsigned)(a.batch * k.split));
  if (a_kc) return b_kc ? launch_t<true, true>(k, grid, s) : launch_t<true, false>(k, grid, s);
  return b_kc ? launch_t<false, true>(k, grid, s) : launch_t<false, false>(k, grid, s);
}

}  // namespace qsgw
