// Flush of the delay buffers on the FP64 tensor-core path.
//
//   det:  Ti[j][i] -= sum_s Bbuf[s][j] Abuf[s][i]          (Eq. 12; Ti = A^-T)
//   pf :  Ti[i][j] += sum_s Bbuf[s][i] Abuf[s][j], j > i,  (Eq. 26)
//         Ti[j][i] = -Ti[i][j] exactly
// i.e. out[r][c] (-/+)= sum_s Bbuf[s][r] Abuf[s][c]: an (n x fill)(fill x n) contraction
// per flushed walker.  sm_100a has no tcgen05 kind for f64; the FP64 tensor path is the
// warp-level DMMA (mma.sync.m8n8k4.f64 -> SASS DMMA.8x8x4), fed from shared memory.
//
// Work item = (walker on the flush list, output tile); persistent grid, two CTAs per SM.
// float64: 128 x 64 tiles, 8 warps, warp tile 32 x 32 (4 x 4 MMA tiles, 8 fragment loads per
// 16 DMMAs); complex128: 64 x 64 tiles, 8 warps, warp tile 16 x 32, one complex MMA = 4 real
// DMMAs on (re, im) pairs read with ONE 16-byte fragment load each -- the buffers stay
// interleaved, nothing is de-interleaved while staging.
//
// Both buffer panels move global -> shared with 16-byte cp.async (LDGSTS) through a ring of
// NS stages of KC buffer rows; the ring runs ACROSS work items (the first chunks of a
// CTA's next tile are in flight while it finishes the current one), which is what the
// HBM-bound regime (K k <= 32: one or two chunks per tile) needs.  Rows past `fill` and
// columns past n are zero-filled by the copy itself.  Row strides of the staged panels
// are chosen so that the four buffer rows a fragment load touches fall into disjoint bank
// groups (stride = 4 mod 16 doubles, 2 mod 8 complex elements): no bank conflicts.
//
// The accumulators START as the output tile (loaded while the first chunk lands) and
// the MMAs run with the negated (det) B-side fragment, so the epilogue is a plain store
// and needs no second set of registers.  Pf: tiles that hold an element above the
// diagonal only; each result is also written, negated, at its mirror position.
#include "lrux_common.cuh"
#include "lrux_internal.h"

namespace lrux {

__device__ __forceinline__ void dmma884(double& d0, double& d1, double a, double b) {
  asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
               : "+d"(d0), "+d"(d1)
               : "d"(a), "d"(b));
}
// 16-byte (or 8-byte) asynchronous copy global -> shared; src_bytes = 0 zero-fills
__device__ __forceinline__ void cp_async_16(void* smem_dst, const void* gsrc, int src_bytes) {
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;" ::"r"((uint32_t)__cvta_generic_to_shared(smem_dst)),
               "l"(gsrc), "r"(src_bytes)
               : "memory");
}
__device__ __forceinline__ void cp_async_8(void* smem_dst, const void* gsrc, int src_bytes) {
  asm volatile("cp.async.ca.shared.global [%0], [%1], 8, %2;" ::"r"((uint32_t)__cvta_generic_to_shared(smem_dst)),
               "l"(gsrc), "r"(src_bytes)
               : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N>
__device__ __forceinline__ void cp_async_wait() {
  asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory");
}

// Tile configurations (warps per CTA as WR x WC over the output tile).  A tile's own traffic
// (the output tile read into the accumulators and stored back: 128 KB of a 64 x 64 complex
// tile's 390 KB at K k = 128) is NOT covered by the cp.async ring, and the contraction is only
// ~2x above the machine balance (10.7 flop/B against 36.6 TF/s / 6.5 TB/s = 5.6), so one CTA
// per SM leaves the DMMA pipe idle for a third of the time (66 % busy in the ncu capture of the
// 16-warp configuration).  Two co-resident CTAs of 8 warps overlap one tile's load / store with
// the other's MMAs.  Measured on B200 (profiles/r02_flush_variants.md), fraction of cuBLAS DGEMM:
//   complex128 64 x 64: 2 CTAs x 8 warps (warp tile 16 x 32, 3 stages) 0.655 / 0.681 (configs[3]
//     Metropolis / forced) against 0.621 / 0.619 for 1 CTA x 16 warps and 0.615 / 0.629 for 1 x 8;
//   float64: 128 x 64, 2 CTAs x 8 warps (warp tile 32 x 32, 3 stages) 0.700 (n = 1024, K k = 256,
//     Metropolis), 0.617 (n = 2048, K k = 128), 0.455 of HBM (configs[1], K k = 32) against
//     0.644 / 0.563 / 0.397 for 128 x 128 with one CTA per SM; all walkers at once: 0.67-0.74 both.
// (An L2 prefetch of the next item's output tile was measured too: no difference.)
template <typename T>
struct FlushCfg;
#ifndef LRUX_FLUSH_R_BN
#define LRUX_FLUSH_R_BN 64
#define LRUX_FLUSH_R_NS 3
#define LRUX_FLUSH_R_MINB 2
#endif
template <>
struct FlushCfg<double> {   // 128 x 64, warps 4 x 2, warp tile 32 x 32, two CTAs per SM
  static constexpr int WR = 4, WC = 2, MINB = LRUX_FLUSH_R_MINB;
  static constexpr int BM = 128, BN = LRUX_FLUSH_R_BN, MT = 4, NT = LRUX_FLUSH_R_BN / 16, KC = 16, NS = LRUX_FLUSH_R_NS,
                       LDB = 132, LDA = LRUX_FLUSH_R_BN + 4;
};
#ifndef LRUX_FLUSH_CX_WC
#define LRUX_FLUSH_CX_WC 2
#define LRUX_FLUSH_CX_NS 3
#define LRUX_FLUSH_CX_MINB 2
#endif
template <>
struct FlushCfg<cplx> {     // 64 x 64, warps 4 x 2, warp tile 16 x 32, two CTAs per SM
  static constexpr int WR = 4, WC = LRUX_FLUSH_CX_WC, MINB = LRUX_FLUSH_CX_MINB;
  static constexpr int BM = 64, BN = 64, MT = 2, NT = 8 / LRUX_FLUSH_CX_WC, KC = 16, NS = LRUX_FLUSH_CX_NS, LDB = 66, LDA = 66;
};

struct FlushItem {
  int w, r0, c0, fill, nch;
};

// V16: rows of the buffers are 16-byte aligned (always for complex; real: n even)
template <typename T, bool SKEW, bool V16>
__global__ void __launch_bounds__(FlushCfg<T>::WR * FlushCfg<T>::WC * 32, FlushCfg<T>::MINB)
flush_dmma_kernel(State st, int tr, int tc, int tiles) {
  using S = Sc<T>;
  using Cfg = FlushCfg<T>;
  constexpr int NTHR = Cfg::WR * Cfg::WC * 32;
  constexpr int BM = Cfg::BM, BN = Cfg::BN, MT = Cfg::MT, NT = Cfg::NT, KC = Cfg::KC, NS = Cfg::NS;
  constexpr int LDB = Cfg::LDB, LDA = Cfg::LDA;
  constexpr bool CX = sizeof(T) == 16;
  constexpr int STAGE = KC * (LDB + LDA);          // elements of T per stage
  extern __shared__ __align__(128) unsigned char smem_raw[];
  T* ring = (T*)smem_raw;                          // [NS][ Bs[KC][LDB] | As[KC][LDA] ]
  const int n = st.n, cap = st.cap;
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int wr = warp / Cfg::WC, wc = warp % Cfg::WC;   // warp position in the WR x WC grid
  const int lm = lane >> 2, lk = lane & 3;         // fragment row / k index
  const int count = st.counters[1];
  const int64_t total = (int64_t)count * tiles;
  const int G = (int)gridDim.x;
  const int my_items = (int)((total - blockIdx.x + G - 1) / G);   // items blockIdx.x, +G, ...
  if (total <= (int64_t)blockIdx.x) return;

  auto decode = [&](int i) {
    FlushItem it;
    const int64_t item = (int64_t)blockIdx.x + (int64_t)i * G;
    it.w = st.flist[item / tiles];
    int t = (int)(item % tiles), R, Cc;
    if (SKEW) {
      // row tile R needs the column tiles Cc >= (R * BM) / BN (an element with col > row)
      R = 0;
      while (true) {
        const int first_c = (R * BM) / BN;
        if (t < tc - first_c) { Cc = first_c + t; break; }
        t -= tc - first_c;
        ++R;
      }
    } else {
      R = t / tc;
      Cc = t % tc;
    }
    it.r0 = R * BM;
    it.c0 = Cc * BN;
    it.fill = st.fill[it.w];
    it.nch = max(1, (it.fill + KC - 1) / KC);
    return it;
  };

  // ---- producer: one chunk = KC rows of both panels into one stage
  auto issue = [&](const FlushItem& it, int ch, int stage) {
    const T* Ab = (const T*)st.Abuf + (size_t)it.w * cap * n;
    const T* Bb = (const T*)st.Bbuf + (size_t)it.w * cap * n;
    T* Bs = ring + (size_t)stage * STAGE;
    T* As = Bs + KC * LDB;
    const int s0 = ch * KC;
    constexpr int EPV = V16 ? (CX ? 1 : 2) : 1;            // elements per copy
    constexpr int VB = BM / EPV, VA = BN / EPV;            // copies per row
#pragma unroll
    for (int u = 0; u < (KC * VB + NTHR - 1) / NTHR; ++u) {
      const int qd = tid + NTHR * u;
      if (qd < KC * VB) {
        const int kk = qd / VB, c = (qd % VB) * EPV;
        const bool ok = s0 + kk < it.fill && it.r0 + c < n;
        const T* src = Bb + (size_t)(ok ? s0 + kk : 0) * n + (ok ? it.r0 + c : 0);
        if (V16) cp_async_16(Bs + kk * LDB + c, src, ok ? 16 : 0);
        else cp_async_8(Bs + kk * LDB + c, src, ok ? 8 : 0);
      }
    }
#pragma unroll
    for (int u = 0; u < (KC * VA + NTHR - 1) / NTHR; ++u) {
      const int qd = tid + NTHR * u;
      if (qd < KC * VA) {
        const int kk = qd / VA, c = (qd % VA) * EPV;
        const bool ok = s0 + kk < it.fill && it.c0 + c < n;
        const T* src = Ab + (size_t)(ok ? s0 + kk : 0) * n + (ok ? it.c0 + c : 0);
        if (V16) cp_async_16(As + kk * LDA + c, src, ok ? 16 : 0);
        else cp_async_8(As + kk * LDA + c, src, ok ? 8 : 0);
      }
    }
  };

  int p_item = 0, p_ch = 0;                       // producer cursor
  FlushItem pit = decode(0);
  int issued = 0;
  auto produce = [&]() {                          // issue the next chunk (if any) and commit a group
    if (p_item < my_items) {
      issue(pit, p_ch, issued % NS);
      if (++p_ch == pit.nch) {
        p_ch = 0;
        if (++p_item < my_items) pit = decode(p_item);
      }
    }
    ++issued;
    cp_async_commit();
  };
#pragma unroll 1
  for (int s = 0; s < NS - 1; ++s) produce();

  int consumed = 0;
#pragma unroll 1
  for (int i = 0; i < my_items; ++i) {
    const FlushItem it = decode(i);
    T* Tw = (T*)st.Ti + (size_t)it.w * n * n;
    // accumulators = the output tile (zero where nothing will be stored)
    double acc[CX ? 2 : 1][MT][NT][2];
#pragma unroll
    for (int mt = 0; mt < MT; ++mt) {
      const int row = it.r0 + wr * (MT * 8) + mt * 8 + lm;
#pragma unroll
      for (int nt = 0; nt < NT; ++nt) {
        const int col = it.c0 + wc * (NT * 8) + nt * 8 + 2 * lk;
        if constexpr (V16 && !CX) {   // both elements wanted: one 16-byte load
          if (row < n && col + 1 < n && (!SKEW || col > row)) {
            const double2 v = *(const double2*)((const double*)Tw + (size_t)row * n + col);
            acc[0][mt][nt][0] = v.x;
            acc[0][mt][nt][1] = v.y;
            continue;
          }
        }
#pragma unroll
        for (int e = 0; e < 2; ++e) {
          const bool need = row < n && col + e < n && (!SKEW || col + e > row);
          // component-wise 8-byte accesses on purpose: the DMMA accumulators keep the re and im
          // planes in separate register pairs, a 16-byte access would need a staging quad
          // (spills at the 128-register cap of two CTAs per SM)
          const double* src = (const double*)(Tw + (size_t)row * n + col + e);
          acc[0][mt][nt][e] = need ? src[0] : 0.0;
          if (CX) acc[CX ? 1 : 0][mt][nt][e] = need ? src[1] : 0.0;
        }
      }
    }
#pragma unroll 1
    for (int ch = 0; ch < it.nch; ++ch) {
      cp_async_wait<NS - 2>();
      __syncthreads();            // chunk `consumed` has landed for everyone; stage (consumed-1)%NS is free
      produce();
      const T* Bs = ring + (size_t)(consumed % NS) * STAGE;
      const T* As = Bs + KC * LDB;
      ++consumed;
      const int kend = min(KC, (it.fill - ch * KC + 3) & ~3);
      for (int k4 = 0; k4 < kend; k4 += 4) {
        if constexpr (!CX) {
          double bf[MT], af[NT];
#pragma unroll
          for (int mt = 0; mt < MT; ++mt) {
            const double b = ((const double*)Bs)[(k4 + lk) * LDB + wr * (MT * 8) + mt * 8 + lm];
            bf[mt] = SKEW ? b : -b;
          }
#pragma unroll
          for (int nt = 0; nt < NT; ++nt) af[nt] = ((const double*)As)[(k4 + lk) * LDA + wc * (NT * 8) + nt * 8 + lm];
#pragma unroll
          for (int mt = 0; mt < MT; ++mt)
#pragma unroll
            for (int nt = 0; nt < NT; ++nt) dmma884(acc[0][mt][nt][0], acc[0][mt][nt][1], bf[mt], af[nt]);
        } else {
          double2 bf[MT], af[NT];
#pragma unroll
          for (int mt = 0; mt < MT; ++mt) {
            double2 b = ((const double2*)Bs)[(k4 + lk) * LDB + wr * (MT * 8) + mt * 8 + lm];
            if (!SKEW) { b.x = -b.x; b.y = -b.y; }
            bf[mt] = b;
          }
#pragma unroll
          for (int nt = 0; nt < NT; ++nt) af[nt] = ((const double2*)As)[(k4 + lk) * LDA + wc * (NT * 8) + nt * 8 + lm];
          // (br + i bi)(ar + i ai) = (br ar - bi ai) + i (br ai + bi ar): four passes over the
          // MT x NT tiles, so that the two DMMAs into one accumulator are 2 MT NT instructions apart
          double nby[MT];
#pragma unroll
          for (int mt = 0; mt < MT; ++mt) nby[mt] = -bf[mt].y;
#pragma unroll
          for (int mt = 0; mt < MT; ++mt)
#pragma unroll
            for (int nt = 0; nt < NT; ++nt) {
              dmma884(acc[0][mt][nt][0], acc[0][mt][nt][1], bf[mt].x, af[nt].x);
              dmma884(acc[CX ? 1 : 0][mt][nt][0], acc[CX ? 1 : 0][mt][nt][1], bf[mt].x, af[nt].y);
            }
#pragma unroll
          for (int mt = 0; mt < MT; ++mt)
#pragma unroll
            for (int nt = 0; nt < NT; ++nt) {
              dmma884(acc[0][mt][nt][0], acc[0][mt][nt][1], nby[mt], af[nt].y);
              dmma884(acc[CX ? 1 : 0][mt][nt][0], acc[CX ? 1 : 0][mt][nt][1], bf[mt].y, af[nt].x);
            }
        }
      }
    }
    // ---- epilogue: accumulator (row lm, cols 2*lk, 2*lk+1) of each 8x8 tile
#pragma unroll
    for (int mt = 0; mt < MT; ++mt) {
      const int row = it.r0 + wr * (MT * 8) + mt * 8 + lm;
      if (row >= n) continue;
#pragma unroll
      for (int nt = 0; nt < NT; ++nt) {
        const int col = it.c0 + wc * (NT * 8) + nt * 8 + 2 * lk;
        if constexpr (V16 && !CX && !SKEW) {
          if (col + 1 < n) {
            *(double2*)((double*)Tw + (size_t)row * n + col) = make_double2(acc[0][mt][nt][0], acc[0][mt][nt][1]);
            continue;
          }
        }
#pragma unroll
        for (int e = 0; e < 2; ++e) {
          if (col + e >= n) continue;
          double* dst = (double*)(Tw + (size_t)row * n + col + e);
          if (SKEW) {
            if (col + e > row) {
              double* mir = (double*)(Tw + (size_t)(col + e) * n + row);
              dst[0] = acc[0][mt][nt][e];
              mir[0] = -acc[0][mt][nt][e];
              if (CX) { dst[1] = acc[CX ? 1 : 0][mt][nt][e]; mir[1] = -acc[CX ? 1 : 0][mt][nt][e]; }
            }
          } else {
            dst[0] = acc[0][mt][nt][e];
            if (CX) dst[1] = acc[CX ? 1 : 0][mt][nt][e];
          }
        }
      }
    }
  }
  cp_async_wait<0>();
}

template <typename T, bool SKEW, bool V16>
static int launch_flush_v(const State& st, Ctx& cx, cudaStream_t s) {
  using Cfg = FlushCfg<T>;
  const int tr = (st.n + Cfg::BM - 1) / Cfg::BM, tc = (st.n + Cfg::BN - 1) / Cfg::BN;
  int64_t tiles = (int64_t)tr * tc;
  if (SKEW) {
    tiles = 0;
    for (int R = 0; R < tr; ++R) tiles += tc - (R * Cfg::BM) / Cfg::BN;
  }
  const size_t smem = (size_t)Cfg::NS * Cfg::KC * (Cfg::LDB + Cfg::LDA) * sizeof(T);
  auto kern = flush_dmma_kernel<T, SKEW, V16>;
  constexpr int NTHR = Cfg::WR * Cfg::WC * 32;
  const int occ = cx.configure((const void*)kern, NTHR, smem);
  if (occ < 0) return -1;
  cx.name(LRUX_PROF_FLUSH, "flush_dmma_kernel");
  int64_t grid = (int64_t)cx.num_sms * occ;
  if (grid > st.W * tiles) grid = st.W * tiles;
  kern<<<(unsigned)grid, NTHR, smem, s>>>(st, tr, tc, (int)tiles);
  return 1;
}

template <typename T, bool SKEW>
static int launch_flush_t(const State& st, Ctx& cx, cudaStream_t s) {
  if (sizeof(T) == 16 || (st.n % 2) == 0) return launch_flush_v<T, SKEW, true>(st, cx, s);
  if constexpr (sizeof(T) == 8) return launch_flush_v<T, SKEW, false>(st, cx, s);
  return -1;
}

int launch_flush_dmma(const State& st, Ctx& cx, cudaStream_t s) {
  if (st.kind == KIND_PF)
    return st.dt == LRUX_F64 ? launch_flush_t<double, true>(st, cx, s)
                             : launch_flush_t<cplx, true>(st, cx, s);
  return st.dt == LRUX_F64 ? launch_flush_t<double, false>(st, cx, s)
                           : launch_flush_t<cplx, false>(st, cx, s);
}

}  // namespace lrux
