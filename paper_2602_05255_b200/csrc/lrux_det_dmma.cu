// Immediate Woodbury update on the FP64 tensor pipe, real data.
//
//   Ti[j][:] -= sum_a g[j][a] C[a][:],   g[j][:] = R^-1 (N Ti[j][:] - [j == P])      (Eq. 5)
//
// The scalar kernels (det_update_kernel, det_update_tma_kernel) spend one shared-memory
// or register operand per DFMA and 5 shuffles per dot product; from k = 4 on they are
// bound by that, not by HBM (k = 8: 0.40-0.59 of the copy bandwidth in round 1).  Here an
// 8-ROW STRIP of Ti is the M side of mma.sync.m8n8k4.f64 (SASS DMMA.8x8x4):
//
//   dots   D[8 x 8]   = X[8 x n] N^T[n x 8]        2 DMMAs per 8 x 8 block of X
//   core   G[8 x 8]   = (D - [j == P]) R^-T          2 DMMAs per strip
//   apply  X[8 x 8]  -= G[8 x 8] C[8 x 8 block]     2 DMMAs per 8 x 8 block of X
//
// so every N / C fragment read from shared memory serves 8 rows, there is no warp
// reduction, and the strip never leaves the registers between its load and its store:
// HBM traffic = read n^2 e + write n^2 e, the compulsory minimum.
//
// Fragment layouts of m8n8k4 (lane l, r = l / 4, q = l % 4): A[r][q], B[q][r], C/D[r][2q, 2q+1].
// The contraction index of the dots is a COLUMN of X, and its order is free as long as X and
// N agree: lane (r, q) loads the 16-byte pair X[j0+r][c0+2q, c0+2q+1] -- exactly the
// accumulator layout the apply step needs -- and uses its two halves as the A fragments of
// two DMMAs whose B fragments are the same pair of N[a = r][.].  The apply contracts over
// a = 2q (first DMMA) and a = 2q + 1 (second), with C stored pair-interleaved
// (C[2q][c], C[2q+1][c] adjacent) so that one 16-byte load feeds both.
//
// The columns of a strip are split over the NW warps of a CTA and, for large n, over the
// CL CTAs of a thread-block cluster (each CTA keeps only ITS columns of N and C in shared
// memory: k n 16 / CL bytes).  The 8 x 8 partial D of every warp meets in shared memory,
// those of the CTAs in every peer's shared memory (DSMEM), always summed in the same
// order, one barrier per strip.  The next strip's loads are issued before the current
// strip's arithmetic.  KT = 8 covers every k <= 8 (unused rows of N, C, R^-1 are zero).
#include <cooperative_groups.h>

#include "lrux_common.cuh"
#include "lrux_internal.h"

// most columns of a strip one CTA takes (more: the columns are split over a cluster)
#ifndef LRUX_DMMA_MAXCOLS
#define LRUX_DMMA_MAXCOLS 1024
#endif

// 1: warp-owned strips for n <= 128; 2: also for n <= 256 (32 blocks per warp, one CTA per SM: n=256 k=4 / 8
// 0.88 / 0.87 of HBM against 0.81 / 0.80 with the strip split over the 8 warps)
#ifndef LRUX_DMMA_WARP_STRIPS
#define LRUX_DMMA_WARP_STRIPS 2
#endif

namespace lrux {

namespace cg = cooperative_groups;

__device__ __forceinline__ void dmma884u(double& d0, double& d1, double a, double b) {
  asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
               : "+d"(d0), "+d"(d1)
               : "d"(a), "d"(b));
}

// NB = 8-column blocks per warp and strip, NW = warps per CTA, CLUSTER: columns also split
// over the CTAs of a cluster (cluster size taken at run time).
template <int NB, int NW, bool CLUSTER>
__global__ void __launch_bounds__(NW * 32, NW <= 8 ? 2 : 1) det_update_dmma_kernel(State st, int k, int ncl) {
  constexpr int KT = 8;
  extern __shared__ __align__(128) unsigned char smem_raw[];
  const int n = st.n, kmax = st.kmax;
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int r8 = lane >> 2, q = lane & 3;
  int CL = 1, cr = 0;
  if constexpr (CLUSTER) {
    cg::cluster_group cluster = cg::this_cluster();
    CL = (int)cluster.num_blocks();
    cr = (int)cluster.block_rank();
  }
  const int ngrp = (int)gridDim.x / CL, grp = (int)blockIdx.x / CL;   // groups of CTAs that share strips
  const int ldn = ncl + 8;                                 // row stride of Ns: odd multiple of 64 B
  const int ldc = ncl + 2;                                 // row stride of Cs2 in pairs: 32 B mod 128 B
  double* Ns = (double*)smem_raw;                          // [KT][ldn]        N, this CTA's columns
  double* Cs2 = Ns + (size_t)KT * ldn;                     // [KT/2][ldc][2]   C, rows paired
  double* part = Cs2 + (size_t)KT * ldc;                   // [2][NW][64]      partial D per warp
  double* cpart = part + 2 * NW * 64;                      // [2][CL][64]      partial D per CTA (cluster)
  __shared__ double Ris[KT * KT];
  __shared__ int sidx[KT];

  const int count = st.counters[0];
  const int spw = (n + 7) >> 3;                            // strips per walker
  const int64_t S = (int64_t)count * spw;
  const int64_t first = S * grp / ngrp, last = S * (grp + 1) / ngrp;
  const int my = (int)(last - first);
  const int wi0 = (int)(first / spw), s00 = (int)(first % spw);   // 32-bit strip arithmetic from here on
  const int col_base = cr * ncl;
  const int col_end = min(n, col_base + ncl);
  const double* Ti = (const double*)st.Ti;

  auto load_strip = [&](int li, double2 (&x)[NB]) {
    const int sx = s00 + li;
    const int w = st.list[wi0 + sx / spw];
    const int j = min((sx % spw) * 8 + r8, n - 1);        // rows past the end: clamped, never stored
    const double* row = Ti + ((size_t)w * n + j) * n;
#pragma unroll
    for (int t = 0; t < NB; ++t) {
      const int c = col_base + 8 * (t * NW + warp) + 2 * q;
      x[t] = c < col_end ? *(const double2*)(row + c) : make_double2(0.0, 0.0);
    }
  };

  double2 xc[NB], xn[NB];
  if (my > 0) load_strip(0, xc);
  int cur_w = -1;
  double ri0 = 0.0, ri1 = 0.0;   // B fragments of R^-T: Ri[b = r8][2q], Ri[r8][2q+1]
  for (int li = 0; li < my; ++li) {
    const int sx = s00 + li;
    const int w = st.list[wi0 + sx / spw];
    const int j0 = (sx % spw) * 8;
    const int slot = li & 1;
    if (w != cur_w) {
      __syncthreads();   // every warp is done with the previous walker's N, C
      const double* gN = (const double*)st.pend_N + (size_t)w * kmax * n;
      const double* gC = (const double*)st.pend_C + (size_t)w * kmax * n;
      const int nc = col_end - col_base;
      for (int idx = tid; idx < KT * (ncl >> 1); idx += NW * 32) {
        const int a = idx / (ncl >> 1), c = 2 * (idx % (ncl >> 1));
        double2 nv = make_double2(0.0, 0.0), cv = nv;
        if (a < k && c < nc) {
          nv = *(const double2*)(gN + (size_t)a * n + col_base + c);
          cv = *(const double2*)(gC + (size_t)a * n + col_base + c);
        }
        *(double2*)(Ns + (size_t)a * ldn + c) = nv;
        Cs2[((size_t)(a >> 1) * ldc + c) * 2 + (a & 1)] = cv.x;
        Cs2[((size_t)(a >> 1) * ldc + c + 1) * 2 + (a & 1)] = cv.y;
      }
      if (tid < KT * KT) {
        const int a = tid / KT, b = tid % KT;
        Ris[tid] = (a < k && b < k) ? ((const double*)st.pend_Rinv)[(size_t)w * st.kc * st.kc + a * st.kc + b] : 0.0;
      }
      if (tid < KT) sidx[tid] = tid < k ? st.pend_idx[(size_t)w * kmax + tid] : -1;
      cur_w = w;
      __syncthreads();
      ri0 = Ris[r8 * KT + 2 * q];
      ri1 = Ris[r8 * KT + 2 * q + 1];
    }
    if (li + 1 < my) load_strip(li + 1, xn);   // in flight during this strip's arithmetic

    // ---- dots: partial D[r][a] over this warp's columns (two independent accumulator chains)
    double d0 = 0.0, d1 = 0.0, e0 = 0.0, e1 = 0.0;
#pragma unroll
    for (int t = 0; t < NB; ++t) {
      const int cl = 8 * (t * NW + warp) + 2 * q;           // column within this CTA's range
      if (8 * (t * NW + warp) < ncl) {
        const double2 nv = *(const double2*)(Ns + (size_t)r8 * ldn + cl);
        dmma884u(d0, d1, xc[t].x, nv.x);
        dmma884u(e0, e1, xc[t].y, nv.y);
      }
    }
    d0 += e0;
    d1 += e1;
    *(double2*)(part + ((size_t)(slot * NW + warp) * 32 + lane) * 2) = make_double2(d0, d1);
    __syncthreads();
    if constexpr (CLUSTER) {
      cg::cluster_group cluster = cg::this_cluster();
      if (warp == 0) {
        double2 sum = *(const double2*)(part + ((size_t)(slot * NW) * 32 + lane) * 2);
#pragma unroll 4
        for (int v = 1; v < NW; ++v) {
          const double2 p = *(const double2*)(part + ((size_t)(slot * NW + v) * 32 + lane) * 2);
          sum.x += p.x;
          sum.y += p.y;
        }
        for (int peer = 0; peer < CL; ++peer)
          *(double2*)(cluster.map_shared_rank(cpart, peer) + ((size_t)(slot * CL + cr) * 32 + lane) * 2) = sum;
      }
      cluster.sync();
      d0 = 0.0;
      d1 = 0.0;
      for (int c = 0; c < CL; ++c) {
        const double2 p = *(const double2*)(cpart + ((size_t)(slot * CL + c) * 32 + lane) * 2);
        d0 += p.x;
        d1 += p.y;
      }
    } else {
      d0 = 0.0;
      d1 = 0.0;
#pragma unroll 4
      for (int v = 0; v < NW; ++v) {
        const double2 p = *(const double2*)(part + ((size_t)(slot * NW + v) * 32 + lane) * 2);
        d0 += p.x;
        d1 += p.y;
      }
    }
    // ---- core: G = (D - [j == P]) R^-T, negated for the apply
    if (j0 + r8 == sidx[2 * q]) d0 -= 1.0;
    if (j0 + r8 == sidx[2 * q + 1]) d1 -= 1.0;
    double g0 = 0.0, g1 = 0.0;
    dmma884u(g0, g1, d0, ri0);
    dmma884u(g0, g1, d1, ri1);
    g0 = -g0;
    g1 = -g1;
    // ---- apply and store
    const int j = j0 + r8;
    double* orow = (double*)st.Ti + ((size_t)w * n + min(j, n - 1)) * n;
#pragma unroll
    for (int t = 0; t < NB; ++t) {
      const int cb = 8 * (t * NW + warp);
      if (cb < ncl) {
        const double2 cv = *(const double2*)(Cs2 + ((size_t)q * ldc + cb + r8) * 2);
        double2 v = xc[t];
        dmma884u(v.x, v.y, g0, cv.x);
        dmma884u(v.x, v.y, g1, cv.y);
        const int c = col_base + cb + 2 * q;
        if (j < n && c < col_end) *(double2*)(orow + c) = v;
      }
    }
#pragma unroll
    for (int t = 0; t < NB; ++t) xc[t] = xn[t];
  }
  if constexpr (CLUSTER) cg::this_cluster().sync();   // no CTA exits while a peer may still write its cpart
}

// Narrow matrices (n <= 256): ONE WARP owns a whole 8-row strip (NB <= 32 blocks of 8 columns), so
// the dots need no exchange and there is no barrier per strip -- only one per walker, when N and C
// are restaged.  With the strip split over 8 warps a strip of n = 128 is 8 KB of work per CTA
// barrier (0.31 / 0.56 of HBM at n = 64 / 128, k = 4).  Strips of a walker go round-robin to the
// 8 warps of the CTA that holds the walker's N, C; CTAs take contiguous balanced strip ranges.
template <int NB>
__global__ void __launch_bounds__(256, NB <= 16 ? 2 : 1) det_update_dmma_warp_kernel(State st, int k, int ncl) {
  constexpr int KT = 8, NW = 8;
  extern __shared__ __align__(128) unsigned char smem_raw[];
  const int n = st.n, kmax = st.kmax;
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int r8 = lane >> 2, q = lane & 3;
  const int ldn = ncl + 8, ldc = ncl + 2;
  double* Ns = (double*)smem_raw;                          // [KT][ldn]
  double* Cs2 = Ns + (size_t)KT * ldn;                     // [KT/2][ldc][2]
  __shared__ double Ris[KT * KT];
  __shared__ int sidx[KT];
  const int count = st.counters[0];
  const int spw = (n + 7) >> 3;
  const int64_t S = (int64_t)count * spw;
  const int64_t first = S * blockIdx.x / gridDim.x, last = S * (blockIdx.x + 1) / gridDim.x;
  const double* Ti = (const double*)st.Ti;
  for (int64_t u = first; u < last;) {
    const int wi = (int)(u / spw);
    const int w = st.list[wi];
    const int s_beg = (int)(u - (int64_t)wi * spw);
    const int s_end = (int)(min(last, (int64_t)(wi + 1) * spw) - (int64_t)wi * spw);
    __syncthreads();   // every warp is done with the previous walker's N, C
    {
      const double* gN = (const double*)st.pend_N + (size_t)w * kmax * n;
      const double* gC = (const double*)st.pend_C + (size_t)w * kmax * n;
      for (int idx = tid; idx < KT * (ncl >> 1); idx += NW * 32) {
        const int a = idx / (ncl >> 1), c = 2 * (idx % (ncl >> 1));
        double2 nv = make_double2(0.0, 0.0), cv = nv;
        if (a < k && c < n) {
          nv = *(const double2*)(gN + (size_t)a * n + c);
          cv = *(const double2*)(gC + (size_t)a * n + c);
        }
        *(double2*)(Ns + (size_t)a * ldn + c) = nv;
        Cs2[((size_t)(a >> 1) * ldc + c) * 2 + (a & 1)] = cv.x;
        Cs2[((size_t)(a >> 1) * ldc + c + 1) * 2 + (a & 1)] = cv.y;
      }
      if (tid < KT * KT) {
        const int a = tid / KT, b = tid % KT;
        Ris[tid] = (a < k && b < k) ? ((const double*)st.pend_Rinv)[(size_t)w * st.kc * st.kc + a * st.kc + b] : 0.0;
      }
      if (tid < KT) sidx[tid] = tid < k ? st.pend_idx[(size_t)w * kmax + tid] : -1;
    }
    __syncthreads();
    const double ri0 = Ris[r8 * KT + 2 * q], ri1 = Ris[r8 * KT + 2 * q + 1];
    double* Tw = (double*)st.Ti + (size_t)w * n * n;
    auto load_strip = [&](int sx, double2 (&x)[NB]) {
      const int j = min(sx * 8 + r8, n - 1);               // rows past the end: clamped, never stored
      const double* row = Ti + ((size_t)w * n + j) * n;
#pragma unroll
      for (int t = 0; t < NB; ++t) {
        const int c = 8 * t + 2 * q;
        x[t] = c < n ? *(const double2*)(row + c) : make_double2(0.0, 0.0);
      }
    };
    constexpr bool PF = NB <= 8;       // a second strip in registers only where it fits (n <= 64)
    double2 xc[NB], xn[PF ? NB : 1];
    if (PF && s_beg + warp < s_end) load_strip(s_beg + warp, xc);
    for (int sx = s_beg + warp; sx < s_end; sx += NW) {
      if constexpr (PF) {
        if (sx + NW < s_end) load_strip(sx + NW, (double2(&)[NB])xn);   // in flight during this strip's arithmetic
      } else {
        load_strip(sx, xc);
      }
      const int j0 = sx * 8;
      double d0 = 0.0, d1 = 0.0, e0 = 0.0, e1 = 0.0;
#pragma unroll
      for (int t = 0; t < NB; ++t) {
        if (8 * t < ncl) {
          const double2 nv = *(const double2*)(Ns + (size_t)r8 * ldn + 8 * t + 2 * q);
          dmma884u(d0, d1, xc[t].x, nv.x);
          dmma884u(e0, e1, xc[t].y, nv.y);
        }
      }
      d0 += e0;
      d1 += e1;
      if (j0 + r8 == sidx[2 * q]) d0 -= 1.0;
      if (j0 + r8 == sidx[2 * q + 1]) d1 -= 1.0;
      double g0 = 0.0, g1 = 0.0;
      dmma884u(g0, g1, d0, ri0);
      dmma884u(g0, g1, d1, ri1);
      g0 = -g0;
      g1 = -g1;
      const int j = j0 + r8;
      double* orow = Tw + (size_t)min(j, n - 1) * n;
#pragma unroll
      for (int t = 0; t < NB; ++t) {
        const int cb = 8 * t;
        if (cb < ncl) {
          const double2 cv = *(const double2*)(Cs2 + ((size_t)q * ldc + cb + r8) * 2);
          double2 v = xc[t];
          dmma884u(v.x, v.y, g0, cv.x);
          dmma884u(v.x, v.y, g1, cv.y);
          const int c = cb + 2 * q;
          if (j < n && c < n) *(double2*)(orow + c) = v;
        }
      }
      if constexpr (PF) {
#pragma unroll
        for (int t = 0; t < NB; ++t) xc[t] = xn[t];
      }
    }
    u = (int64_t)wi * spw + s_end;
  }
}

template <int NB>
static int launch_dmma_warp(const State& st, int k, int ncl, Ctx& cx, cudaStream_t s, bool probe) {
  const size_t smem = ((size_t)8 * (ncl + 8) + (size_t)8 * (ncl + 2)) * sizeof(double);
  if (probe) return 1;
  auto kern = det_update_dmma_warp_kernel<NB>;
  const int occ = cx.configure((const void*)kern, 256, smem);
  if (occ < 0) return -1;
  const int64_t strips = (int64_t)st.W * ((st.n + 7) / 8);
  kern<<<persistent_grid(cx.num_sms, occ, (strips + 7) / 8), 256, smem, s>>>(st, k, ncl);
  cx.name(LRUX_PROF_UPDATE, "det_update_dmma_warp_kernel");
  return 1;
}

// ---------------------------------------------------------------- launcher
// 1 = launched, 0 = shape not eligible (complex data, odd n, no instance), -1 = CUDA error.
template <int NB, int NW>
static int launch_dmma_inst(const State& st, int k, int CL, int ncl, Ctx& cx, cudaStream_t s, bool probe) {
  const size_t smem = ((size_t)8 * (ncl + 8) + (size_t)8 * (ncl + 2) + 2 * NW * 64 + 2 * (size_t)CL * 64) * sizeof(double);
  if (smem > 200 * 1024) return 0;
  if (probe) return 1;
  State stc = st;
  int kk = k, nc = ncl;
  void* args[3] = {&stc, &kk, &nc};
  if (CL == 1) {
    auto kern = det_update_dmma_kernel<NB, NW, false>;
    const int occ = cx.configure((const void*)kern, NW * 32, smem);
    if (occ < 0) return -1;
    const int64_t strips = (int64_t)st.W * ((st.n + 7) / 8);
    kern<<<persistent_grid(cx.num_sms, occ, strips), NW * 32, smem, s>>>(st, k, ncl);
  } else {
    const void* kern = (const void*)det_update_dmma_kernel<NB, NW, true>;
    const int ncl_max = cx.configure_cluster(kern, NW * 32, smem, CL);   // co-resident clusters
    if (ncl_max < 1) return 0;
    cudaLaunchConfig_t cfg = {};
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeClusterDimension;
    attr[0].val.clusterDim.x = CL;
    attr[0].val.clusterDim.y = 1;
    attr[0].val.clusterDim.z = 1;
    cfg.blockDim = dim3(NW * 32);
    cfg.dynamicSmemBytes = smem;
    cfg.stream = s;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    cfg.gridDim = dim3((unsigned)(CL * ncl_max));
    if (cudaLaunchKernelExC(&cfg, kern, args) != cudaSuccess) return -1;
  }
  cx.name(LRUX_PROF_UPDATE, "det_update_dmma_kernel");
  return 1;
}

int launch_det_update_dmma(const State& st, int k, Ctx& cx, cudaStream_t s, bool probe) {
  const int n = st.n;
  if (st.dt != LRUX_F64 || (n & 1) || k > 8) return 0;
  // columns per CTA: at most 8 blocks of 8 columns per warp, 16 warps -> 1024; N and C of
  // those columns (k <= 8 padded to 8 rows: 128 B per column) stay in shared memory
  int CL = 1;
  while ((n + CL - 1) / CL > LRUX_DMMA_MAXCOLS) CL *= 2;
  if (CL > 8) return 0;
  const int ncl = (((n + CL - 1) / CL) + 7) & ~7;
  const int blocks = ncl / 8;
#if LRUX_DMMA_WARP_STRIPS
  if (blocks <= 8) return launch_dmma_warp<8>(st, k, ncl, cx, s, probe);     // n <= 64
  if (blocks <= 16) return launch_dmma_warp<16>(st, k, ncl, cx, s, probe);   // n <= 128
#if LRUX_DMMA_WARP_STRIPS >= 2
  if (blocks <= 32) return launch_dmma_warp<32>(st, k, ncl, cx, s, probe);   // n <= 256: one CTA per SM
#endif
#endif
#define LRUX_DMMA_CASE(NB_, NW_) \
  if (blocks <= NB_ * NW_) return launch_dmma_inst<NB_, NW_>(st, k, CL, ncl, cx, s, probe);
  LRUX_DMMA_CASE(1, 8)
  LRUX_DMMA_CASE(2, 8)
  LRUX_DMMA_CASE(4, 8)
  LRUX_DMMA_CASE(8, 8)
  LRUX_DMMA_CASE(6, 16)
  LRUX_DMMA_CASE(8, 16)
#undef LRUX_DMMA_CASE
  return 0;
}

}  // namespace lrux
