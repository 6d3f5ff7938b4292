// Immediate Pfaffian update on the FP64 tensor pipe, real data.
//
//   A^-1 += Y' R'^-1 Y'^T   (Eq. 21; k = 1: Eq. 22),   Y' = (A^-1 N + E_P, C)   (n x 2k)
//   <=>  Ti[i][j] += sum_beta g[beta][i] y[beta][j],   y = Y'^T,  g[beta][i] = sum_alpha y[alpha][i] R'^-1[alpha][beta]
//
// a rank-2k outer-product accumulation into every element: the "apply" half of
// det_update_dmma_kernel without its dot products, so there is no reduction and no barrier
// between strips.  An 8-ROW STRIP of Ti is the M side of mma.sync.m8n8k4.f64: lane (r, q) loads
// the 16-byte pair Ti[j0+r][cb+2q, cb+2q+1] -- the accumulator layout -- and each 8 x 8 block
// takes 2k/4 DMMAs whose A fragment (g of the strip's rows) lives in registers for the whole
// strip and whose B fragment (y of the block's columns) comes from shared memory, against 2k
// shared-memory operands and 2k DFMAs PER ELEMENT in pf_update_stream_kernel.
//
// Exact skewness (reading 7): as in the scalar kernels every element is produced by
// its own thread, and an element below the diagonal is the exact negative of its mirror image
// because it is computed from the same operands in the same order: block (rows J, columns I)
// below the diagonal starts from -Ti[j][i] (= Ti[i][j] bit for bit), contracts A = y[.][j] with
// B = g[.][i] -- the products g[beta][i] y[beta][j] of the mirrored element, same beta order
// inside and across the DMMAs -- and stores the negative.  Diagonal blocks evaluate both forms
// and select per element; the diagonal itself is written as zero.
//
// Work = 8-row strips of the concatenated accepted list, a contiguous balanced range per CTA;
// y and g of the current walker (2k x n each, zero-padded to MH rows) staged in shared memory
// once per walker and CTA; the next strip's loads are in flight during the current strip's DMMAs.
#include "lrux_common.cuh"
#include "lrux_internal.h"

// 1: warp-owned strips for n <= 128; 2: also for n <= 256 (32 blocks per warp, one CTA per SM) -- measured at
// n = 256: k=2 0.80 (same), k=4 0.72 against 0.73-0.77, k=8 0.53 against 0.58: not shipped
#ifndef LRUX_PF_DMMA_PAD
#define LRUX_PF_DMMA_PAD 4
#endif
#ifndef LRUX_PF_DMMA_WARP_STRIPS
#define LRUX_PF_DMMA_WARP_STRIPS 1
#endif

namespace lrux {

__device__ __forceinline__ void dmma884p(double& d0, double& d1, double a, double b) {
  asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
               : "+d"(d0), "+d"(d1)
               : "d"(a), "d"(b));
}

// NB = 8-column blocks per warp and strip, NW = warps per CTA, MQ = DMMAs per block (4 MQ >= 2k).
// The columns are cut into ncr ranges of ncl (8 NB NW >= ncl; ncr = 1 up to n = 1024): CTA b
// works on range b mod ncr for all of its strips and keeps only that range of y and g in
// shared memory (row stride ld >= ncl, 4 mod 16 doubles: the 8-byte fragment loads of a half-warp --
// rows q = 0..3, columns r = 0..3 -- then fall into 16 different bank pairs; with 8 mod 16 the ncu capture at
// 2k = 16 showed 1.8 bank conflicts per shared load).  With ncr > 1
// the A fragments (y, g of the strip's own ROWS, which may lie in another range) come from a
// second, small pair of panels that holds y and g of `rmax` consecutive rows and is restaged
// whenever the strips leave it -- the same staging arithmetic, so that mirrored elements
// produced by different CTAs still see identical operands.
template <int NB, int NW, int MQ, bool RANGES>
__global__ void __launch_bounds__(NW * 32, NW <= 8 ? 2 : 1)
pf_update_dmma_kernel(State st, int k, int ld, int ncr_, int ncl, int rmax) {
  const int ncr = RANGES ? ncr_ : 1;
  constexpr int MH = 4 * MQ;
  constexpr int kMaxC = 2 * kMaxK;
  extern __shared__ __align__(128) unsigned char smem_raw[];
  const int n = st.n, kmax = st.kmax, m = 2 * k;
  double* yv = (double*)smem_raw;           // [MH][ld]
  double* gv = yv + (size_t)MH * ld;        // [MH][ld]
  const int ldr = rmax + LRUX_PF_DMMA_PAD;
  double* yr = gv + (size_t)MH * ld;        // [MH][ldr]  (ncr > 1) y of rows [row_lo, row_lo + rmax)
  double* gr = yr + (size_t)MH * ldr;       // [MH][ldr]
  __shared__ double Ri[kMaxC * kMaxC];
  __shared__ int P[kMaxK];
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int r8 = lane >> 2, q = lane & 3;

  const int count = st.counters[0];
  const int spw = (n + 7) >> 3;
  const int64_t S = (int64_t)count * spw;
  const int ngrp = (int)gridDim.x / ncr, grp = (int)blockIdx.x / ncr;   // CTAs that share a column range
  const int col_base = ((int)blockIdx.x % ncr) * ncl, col_end = min(n, col_base + ncl);
  const int64_t first = S * grp / ngrp, last = S * (grp + 1) / ngrp;
  const int my = (int)(last - first);
  const int wi0 = (int)(first / spw), s00 = (int)(first % spw);
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

  // y[a][i] = Y'[a][i], g[b][i] = sum_a y[a][i] R'^-1[a][b] for i in [i0, i0 + cnt) -> panels of stride lds
  auto stage = [&](int w, int i0, int cnt, double* ys, double* gs, int lds) {
    const double* pC = (const double*)st.pend_C + (size_t)w * kmax * n;
    const double* pY = (const double*)st.pend_Y + (size_t)w * kmax * n;
    for (int il = tid; il < cnt; il += NW * 32) {
      const int i = i0 + il;
      double yp[MH];
#pragma unroll
      for (int a = 0; a < MH; ++a) {
        double v = 0.0;
        if (a < m && i < n) {
          v = a < k ? pY[(size_t)a * n + i] : pC[(size_t)(a - k) * n + i];
          if (a < k && i == P[a]) v += 1.0;
        }
        yp[a] = v;
        ys[(size_t)a * lds + il] = v;
      }
#pragma unroll 1
      for (int b = 0; b < MH; ++b) {
        double g = 0.0;
        if (b < m) {
#pragma unroll
          for (int a = 0; a < MH; ++a)
            if (a < m) g = fma(yp[a], Ri[a * kMaxC + b], g);
        }
        gs[(size_t)b * lds + il] = g;
      }
    }
  };

  double2 xc[NB], xn[NB];
  if (my > 0) load_strip(0, xc);
  int cur_w = -1, row_lo = 0;
  for (int li = 0; li < my; ++li) {
    const int sx = s00 + li;
    const int w = st.list[wi0 + sx / spw];
    const int j0 = (sx % spw) * 8;
    if (w != cur_w) {
      __syncthreads();   // every warp is done with the previous walker's y, g
      for (int idx = tid; idx < m * m; idx += NW * 32)
        Ri[(idx / m) * kMaxC + (idx % m)] =
            ((const double*)st.pend_Rinv)[(size_t)w * st.kc * st.kc + (idx / m) * st.kc + (idx % m)];
      if (tid < k) P[tid] = st.pend_idx[(size_t)w * kmax + tid];
      __syncthreads();
      stage(w, col_base, ld, yv, gv, ld);
      if constexpr (RANGES) { row_lo = j0; stage(w, row_lo, ldr, yr, gr, ldr); }
      cur_w = w;
      __syncthreads();
    } else if (RANGES && j0 >= row_lo + rmax) {
      __syncthreads();   // every warp is done with the previous rows' panels
      row_lo = j0;
      stage(w, row_lo, ldr, yr, gr, ldr);
      __syncthreads();
    }
    if (li + 1 < my) load_strip(li + 1, xn);   // in flight during this strip's arithmetic

    double ag[MQ], ay[MQ];                      // A fragments: g / y of the strip's rows
    if constexpr (!RANGES) {
#pragma unroll
      for (int s = 0; s < MQ; ++s) {
        ag[s] = gv[(size_t)(4 * s + q) * ld + j0 + r8];
        ay[s] = yv[(size_t)(4 * s + q) * ld + j0 + r8];
      }
    } else {
#pragma unroll
      for (int s = 0; s < MQ; ++s) {
        ag[s] = gr[(size_t)(4 * s + q) * ldr + (j0 - row_lo) + r8];
        ay[s] = yr[(size_t)(4 * s + q) * ldr + (j0 - row_lo) + r8];
      }
    }
    const int j = j0 + r8;
    double* orow = (double*)st.Ti + ((size_t)w * n + min(j, n - 1)) * n;
#pragma unroll
    for (int t = 0; t < NB; ++t) {
      const int cl = 8 * (t * NW + warp);   // block's first column within the range, and overall
      const int cb = col_base + cl;
      if (cb < col_end) {
        double2 v = xc[t];
        if (cb > j0) {                          // above the diagonal: v(r, c)
#pragma unroll
          for (int s = 0; s < MQ; ++s) dmma884p(v.x, v.y, ag[s], yv[(size_t)(4 * s + q) * ld + cl + r8]);
        } else if (cb < j0) {                   // below: -v(c, r)
          v.x = -v.x;
          v.y = -v.y;
#pragma unroll
          for (int s = 0; s < MQ; ++s) dmma884p(v.x, v.y, ay[s], gv[(size_t)(4 * s + q) * ld + cl + r8]);
          v.x = -v.x;
          v.y = -v.y;
        } else {                                // the diagonal block: both forms, selected per element
          double2 lo = make_double2(-v.x, -v.y);
#pragma unroll
          for (int s = 0; s < MQ; ++s) {
            dmma884p(v.x, v.y, ag[s], yv[(size_t)(4 * s + q) * ld + cl + r8]);
            dmma884p(lo.x, lo.y, ay[s], gv[(size_t)(4 * s + q) * ld + cl + r8]);
          }
          const int c0 = cb + 2 * q;
          v.x = c0 > j ? v.x : c0 < j ? -lo.x : 0.0;
          v.y = c0 + 1 > j ? v.y : c0 + 1 < j ? -lo.y : 0.0;
        }
        const int c = cb + 2 * q;
        if (j < n && c < col_end) *(double2*)(orow + c) = v;
      }
    }
#pragma unroll
    for (int t = 0; t < NB; ++t) xc[t] = xn[t];
  }
}

// Narrow matrices (n <= 128): ONE WARP owns a whole 8-row strip (NB <= 16 blocks) and the strips of a
// walker go round-robin to the 8 warps of the CTA that holds the walker's y, g -- with the strip
// split over 8 warps each warp had 1-2 blocks (0.5-1 KB) of work per loop iteration.  CTAs take
// contiguous balanced strip ranges; the only barriers are those around the staging of y, g.
template <int NB, int MQ>
__global__ void __launch_bounds__(256, NB <= 16 ? 2 : 1) pf_update_dmma_warp_kernel(State st, int k, int ld) {
  constexpr int MH = 4 * MQ, NW = 8;
  constexpr int kMaxC = 2 * kMaxK;
  constexpr bool PF = NB <= 8;                  // a second strip in registers only where it fits
  extern __shared__ __align__(128) unsigned char smem_raw[];
  const int n = st.n, kmax = st.kmax, m = 2 * k;
  double* yv = (double*)smem_raw;           // [MH][ld]
  double* gv = yv + (size_t)MH * ld;        // [MH][ld]
  __shared__ double Ri[kMaxC * kMaxC];
  __shared__ int P[kMaxK];
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int r8 = lane >> 2, q = lane & 3;
  const int count = st.counters[0];
  const int spw = (n + 7) >> 3;
  const int64_t S = (int64_t)count * spw;
  const int64_t first = S * blockIdx.x / gridDim.x, last = S * (blockIdx.x + 1) / gridDim.x;
  for (int64_t u = first; u < last;) {
    const int wi = (int)(u / spw);
    const int w = st.list[wi];
    const int s_beg = (int)(u - (int64_t)wi * spw);
    const int s_end = (int)(min(last, (int64_t)(wi + 1) * spw) - (int64_t)wi * spw);
    __syncthreads();   // every warp is done with the previous walker's y, g
    for (int idx = tid; idx < m * m; idx += NW * 32)
      Ri[(idx / m) * kMaxC + (idx % m)] =
          ((const double*)st.pend_Rinv)[(size_t)w * st.kc * st.kc + (idx / m) * st.kc + (idx % m)];
    if (tid < k) P[tid] = st.pend_idx[(size_t)w * kmax + tid];
    __syncthreads();
    {
      const double* pC = (const double*)st.pend_C + (size_t)w * kmax * n;
      const double* pY = (const double*)st.pend_Y + (size_t)w * kmax * n;
      for (int i = tid; i < ld; i += NW * 32) {
        double yp[MH];
#pragma unroll
        for (int a = 0; a < MH; ++a) {
          double v = 0.0;
          if (a < m && i < n) {
            v = a < k ? pY[(size_t)a * n + i] : pC[(size_t)(a - k) * n + i];
            if (a < k && i == P[a]) v += 1.0;
          }
          yp[a] = v;
          yv[(size_t)a * ld + i] = v;
        }
#pragma unroll 1
        for (int b = 0; b < MH; ++b) {
          double g = 0.0;
          if (b < m) {
#pragma unroll
            for (int a = 0; a < MH; ++a)
              if (a < m) g = fma(yp[a], Ri[a * kMaxC + b], g);
          }
          gv[(size_t)b * ld + i] = g;
        }
      }
    }
    __syncthreads();
    double* Tw = (double*)st.Ti + (size_t)w * n * n;
    auto load_strip = [&](int sx, double2 (&x)[NB]) {
      const int j = min(sx * 8 + r8, n - 1);               // rows past the end: clamped, never stored
      const double* row = Tw + (size_t)j * n;
#pragma unroll
      for (int t = 0; t < NB; ++t) {
        const int c = 8 * t + 2 * q;
        x[t] = c < n ? *(const double2*)(row + c) : make_double2(0.0, 0.0);
      }
    };
    double2 xc[NB], xn[PF ? NB : 1];
    if (PF && s_beg + warp < s_end) load_strip(s_beg + warp, xc);
    for (int sx = s_beg + warp; sx < s_end; sx += NW) {
      if constexpr (PF) {
        if (sx + NW < s_end) load_strip(sx + NW, (double2(&)[NB])xn);
      } else {
        load_strip(sx, xc);
      }
      const int j0 = sx * 8, j = j0 + r8;
      double ag[MQ], ay[MQ];
#pragma unroll
      for (int s2 = 0; s2 < MQ; ++s2) {
        ag[s2] = gv[(size_t)(4 * s2 + q) * ld + j0 + r8];
        ay[s2] = yv[(size_t)(4 * s2 + q) * ld + j0 + r8];
      }
      double* orow = Tw + (size_t)min(j, n - 1) * n;
#pragma unroll
      for (int t = 0; t < NB; ++t) {
        const int cb = 8 * t;
        if (cb < n) {
          double2 v = xc[t];
          if (cb > j0) {                          // above the diagonal: v(r, c)
#pragma unroll
            for (int s2 = 0; s2 < MQ; ++s2) dmma884p(v.x, v.y, ag[s2], yv[(size_t)(4 * s2 + q) * ld + cb + r8]);
          } else if (cb < j0) {                   // below: -v(c, r)
            v.x = -v.x;
            v.y = -v.y;
#pragma unroll
            for (int s2 = 0; s2 < MQ; ++s2) dmma884p(v.x, v.y, ay[s2], gv[(size_t)(4 * s2 + q) * ld + cb + r8]);
            v.x = -v.x;
            v.y = -v.y;
          } else {                                // the diagonal block: both forms, selected per element
            double2 lo = make_double2(-v.x, -v.y);
#pragma unroll
            for (int s2 = 0; s2 < MQ; ++s2) {
              dmma884p(v.x, v.y, ag[s2], yv[(size_t)(4 * s2 + q) * ld + cb + r8]);
              dmma884p(lo.x, lo.y, ay[s2], gv[(size_t)(4 * s2 + q) * ld + cb + r8]);
            }
            const int c0 = cb + 2 * q;
            v.x = c0 > j ? v.x : c0 < j ? -lo.x : 0.0;
            v.y = c0 + 1 > j ? v.y : c0 + 1 < j ? -lo.y : 0.0;
          }
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

template <int NB, int MQ>
static int launch_pf_dmma_warp(const State& st, int k, int ld, Ctx& cx, cudaStream_t s, bool probe) {
  const size_t smem = (size_t)2 * 4 * MQ * ld * sizeof(double);
  if (probe) return 1;
  auto kern = pf_update_dmma_warp_kernel<NB, MQ>;
  const int occ = cx.configure((const void*)kern, 256, smem);
  if (occ < 0) return -1;
  const int64_t strips = (int64_t)st.W * ((st.n + 7) / 8);
  kern<<<persistent_grid(cx.num_sms, occ, (strips + 7) / 8), 256, smem, s>>>(st, k, ld);
  cx.name(LRUX_PROF_UPDATE, "pf_update_dmma_warp_kernel");
  return 1;
}

template <int NB, int NW, int MQ, bool RANGES>
static int launch_pf_dmma_inst(const State& st, int k, int ld, int ncr, int ncl, int rmax, Ctx& cx, cudaStream_t s, bool probe) {
  const size_t smem = (size_t)2 * 4 * MQ * (ld + (ncr > 1 ? rmax + 8 : 0)) * sizeof(double);
  if (smem > 200 * 1024) return 0;
  if (probe) return 1;
  auto kern = pf_update_dmma_kernel<NB, NW, MQ, RANGES>;
  const int occ = cx.configure((const void*)kern, NW * 32, smem);
  if (occ < 0) return -1;
  const int64_t strips = (int64_t)st.W * ((st.n + 7) / 8);
  int grid = persistent_grid(cx.num_sms, occ, strips * ncr);
  grid = grid / ncr * ncr;                     // whole groups of ncr CTAs (one per column range)
  if (grid < ncr) grid = ncr;
  kern<<<grid, NW * 32, smem, s>>>(st, k, ld, ncr, ncl, rmax);
  cx.name(LRUX_PROF_UPDATE, "pf_update_dmma_kernel");
  return 1;
}

// 1 = launched, 0 = shape not eligible (complex data, odd n, more than 16 column ranges),
// -1 = CUDA error.  Expects Y in pend_Y (launch_y) and the accepted list (select).
int launch_pf_update_dmma(const State& st, int k, Ctx& cx, cudaStream_t s, bool probe) {
  const int n = st.n;
  if (st.dt != LRUX_F64 || (n & 1) || k > 8) return 0;
  const int mq = k <= 2 ? 1 : k <= 4 ? 2 : 4;
  // column ranges: at most 1024 columns per CTA, and y, g of a range (2 x 4 mq x ld doubles) within 200 KB
  // (+ with more than one range, y and g of rmax rows for the A fragments)
  const int rmax = mq == 4 ? 128 : 256;
  int ncr = 1, ncl = 0, ld = 0;
  for (;; ncr *= 2) {
    if (ncr > 16) return 0;
    ncl = (((n + ncr - 1) / ncr) + 7) & ~7;
    ld = ((ncl + 15) & ~15) + LRUX_PF_DMMA_PAD;
    // (2k = 16 with ranges narrow enough for two CTAs per SM was measured too: no gain, 0.53-0.67 either way)
    if (ncl <= 1024 && (size_t)2 * 4 * mq * (ld + (ncr > 1 ? rmax + 8 : 0)) * sizeof(double) <= 200 * 1024) break;
  }
  const int blocks = ncl / 8;
#define LRUX_PFD_MQ(NB_, NW_, RG_)                                                                   \
  return mq == 1 ? launch_pf_dmma_inst<NB_, NW_, 1, RG_>(st, k, ld, ncr, ncl, rmax, cx, s, probe)    \
       : mq == 2 ? launch_pf_dmma_inst<NB_, NW_, 2, RG_>(st, k, ld, ncr, ncl, rmax, cx, s, probe)    \
                 : launch_pf_dmma_inst<NB_, NW_, 4, RG_>(st, k, ld, ncr, ncl, rmax, cx, s, probe);
  if (ncr > 1) {                       // column ranges: 16 warps (the panels leave one CTA per SM)
    if (blocks <= 64) { LRUX_PFD_MQ(4, 16, true) }
    LRUX_PFD_MQ(8, 16, true)
  }
#if LRUX_PF_DMMA_WARP_STRIPS
  if (blocks <= 8)
    return mq == 1 ? launch_pf_dmma_warp<8, 1>(st, k, ld, cx, s, probe)
         : mq == 2 ? launch_pf_dmma_warp<8, 2>(st, k, ld, cx, s, probe) : launch_pf_dmma_warp<8, 4>(st, k, ld, cx, s, probe);
  if (blocks <= 16)
    return mq == 1 ? launch_pf_dmma_warp<16, 1>(st, k, ld, cx, s, probe)
         : mq == 2 ? launch_pf_dmma_warp<16, 2>(st, k, ld, cx, s, probe) : launch_pf_dmma_warp<16, 4>(st, k, ld, cx, s, probe);
#if LRUX_PF_DMMA_WARP_STRIPS >= 2
  if (blocks <= 32)     // n <= 256: 32 blocks per warp, one CTA per SM
    return mq == 1 ? launch_pf_dmma_warp<32, 1>(st, k, ld, cx, s, probe)
         : mq == 2 ? launch_pf_dmma_warp<32, 2>(st, k, ld, cx, s, probe) : launch_pf_dmma_warp<32, 4>(st, k, ld, cx, s, probe);
#endif
#endif
  if (blocks <= 16) { LRUX_PFD_MQ(2, 8, false) }
  if (blocks <= 32) { LRUX_PFD_MQ(4, 8, false) }
  // panels beyond half the shared memory leave one CTA per SM: 16 warps instead of 8
  // (n = 512, k = 8: 0.61 of HBM against 0.38)
  if (blocks <= 64 && (size_t)2 * 4 * mq * ld * sizeof(double) > 100 * 1024)
    return launch_pf_dmma_inst<4, 16, 4, false>(st, k, ld, ncr, ncl, rmax, cx, s, probe);
  if (blocks <= 64) { LRUX_PFD_MQ(8, 8, false) }
  if (blocks <= 128) { LRUX_PFD_MQ(8, 16, false) }
#undef LRUX_PFD_MQ
  return 0;
}

}  // namespace lrux
