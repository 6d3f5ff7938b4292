// Flush of the delay buffers on the FP64 tensor-core path.
//
//   det:  Ti[j][i] -= sum_s Bbuf[s][j] Abuf[s][i]          (Eq. 12; Ti = A^-T)
//   pf :  Ti[i][j] += sum_s Bbuf[s][i] Abuf[s][j], j > i,  (Eq. 26)
//         Ti[j][i] = -Ti[i][j] exactly
// i.e. out[r][c] (-/+)= sum_s Bbuf[s][r] Abuf[s][c]: an (n x fill)(fill x n) contraction
// per flushed walker.  sm_100a has no tcgen05 kind for f64; the FP64 tensor path is the
// warp-level DMMA (mma.sync.m8n8k4.f64), fed from shared memory.
//
// Work item = (walker on the flush list, 64x64 output tile); persistent grid.  8 warps
// as 4 (rows) x 2 (cols), warp tile 16 x 32 = 2 x 4 MMA tiles.  The two buffer panels
// are staged s-major in shared memory (row stride 72 doubles: the 32 fragment loads
// of a warp then hit 32 distinct doubles).  complex128 is split into planar re/im
// planes while staging, so one complex MMA = 4 real DMMAs.
#include "lrux_common.cuh"
#include "lrux_internal.h"

namespace lrux {

__device__ __forceinline__ void dmma884(double& d0, double& d1, double a, double b) {
  asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
               : "+d"(d0), "+d"(d1)
               : "d"(a), "d"(b));
}

template <typename T>
struct FlushCfg;
template <>
struct FlushCfg<double> {
  static constexpr int NP = 1, KC = 32;
};
template <>
struct FlushCfg<cplx> {
  static constexpr int NP = 2, KC = 16;
};

__device__ __forceinline__ void split_store(double* p0, double*, int off, double v) { p0[off] = v; }
__device__ __forceinline__ void split_store(double* p0, double* p1, int off, cplx v) {
  p0[off] = v.re;
  p1[off] = v.im;
}

template <typename T, bool SKEW>
__global__ void __launch_bounds__(256) flush_dmma_kernel(State st, int t1) {
  using S = Sc<T>;
  constexpr int BT = 64, LD = 72;
  constexpr int NP = FlushCfg<T>::NP, KC = FlushCfg<T>::KC;
  constexpr bool CX = NP == 2;
  __shared__ __align__(16) double Bs[NP][KC][LD];
  __shared__ __align__(16) double As[NP][KC][LD];
  const int n = st.n, cap = st.cap;
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int wr = warp >> 1, wc = warp & 1;   // warp position in the 4 x 2 grid
  const int lm = lane >> 2, lk = lane & 3;   // fragment row / k index
  const int count = st.counters[1];
  const int tiles = SKEW ? t1 * (t1 + 1) / 2 : t1 * t1;
  for (int item = blockIdx.x; item < count * tiles; item += gridDim.x) {
    const int w = st.flist[item / tiles];
    int R, Cc;
    if (SKEW) {
      int rem = item % tiles;
      R = 0;
      while (rem >= t1 - R) { rem -= t1 - R; ++R; }
      Cc = R + rem;
    } else {
      R = (item % tiles) / t1;
      Cc = (item % tiles) % t1;
    }
    const int r0 = R * BT, c0 = Cc * BT;
    const int fill = st.fill[w];
    const T* Ab = (const T*)st.Abuf + (size_t)w * cap * n;
    const T* Bb = (const T*)st.Bbuf + (size_t)w * cap * n;
    T* Tw = (T*)st.Ti + (size_t)w * n * n;
    double acc[NP][2][4][2];
#pragma unroll
    for (int p = 0; p < NP; ++p)
#pragma unroll
      for (int mt = 0; mt < 2; ++mt)
#pragma unroll
        for (int nt = 0; nt < 4; ++nt) acc[p][mt][nt][0] = acc[p][mt][nt][1] = 0.0;
    // real case: issue the loads of the output tile now, consume them in the epilogue
    // (hides one global-memory latency per work item; the HBM-bound regime, Kk <~ 50)
    double tv[CX ? 1 : 2][CX ? 1 : 4][2];
    if (!CX) {
#pragma unroll
      for (int mt = 0; mt < 2; ++mt) {
        const int row = r0 + wr * 16 + mt * 8 + lm;
#pragma unroll
        for (int nt = 0; nt < 4; ++nt)
#pragma unroll
          for (int e = 0; e < 2; ++e) {
            const int col = c0 + wc * 32 + nt * 8 + 2 * lk + e;
            const bool need = row < n && col < n && (!SKEW || col > row);
            tv[CX ? 0 : mt][CX ? 0 : nt][e] = need ? ((const double*)Tw)[(size_t)row * n + col] : 0.0;
          }
      }
    }

    // register double buffering: the global loads of panel chunk s0+KC are in flight
    // while the DMMAs of chunk s0 run
    constexpr int EPT = KC * BT / 256;   // staged elements per thread and panel
    T rb[EPT], ra[EPT];
    auto fetch = [&](int s0) {
#pragma unroll
      for (int u = 0; u < EPT; ++u) {
        const int q = tid + 256 * u;
        const int kk = q / BT, c = q % BT;
        const bool sv = s0 + kk < fill;
        rb[u] = (sv && r0 + c < n) ? Bb[(size_t)(s0 + kk) * n + r0 + c] : S::zero();
        ra[u] = (sv && c0 + c < n) ? Ab[(size_t)(s0 + kk) * n + c0 + c] : S::zero();
      }
    };
    fetch(0);
    for (int s0 = 0; s0 < fill; s0 += KC) {
      __syncthreads();
#pragma unroll
      for (int u = 0; u < EPT; ++u) {
        const int q = tid + 256 * u;
        const int kk = q / BT, c = q % BT;
        split_store(&Bs[0][kk][0], &Bs[NP - 1][kk][0], c, rb[u]);
        split_store(&As[0][kk][0], &As[NP - 1][kk][0], c, ra[u]);
      }
      __syncthreads();
      if (s0 + KC < fill) fetch(s0 + KC);
      const int kend = min(KC, (fill - s0 + 3) & ~3);
      for (int k4 = 0; k4 < kend; k4 += 4) {
        double bf[NP][2], af[NP][4];
#pragma unroll
        for (int p = 0; p < NP; ++p) {
#pragma unroll
          for (int mt = 0; mt < 2; ++mt) bf[p][mt] = Bs[p][k4 + lk][wr * 16 + mt * 8 + lm];
#pragma unroll
          for (int nt = 0; nt < 4; ++nt) af[p][nt] = As[p][k4 + lk][wc * 32 + nt * 8 + lm];
        }
#pragma unroll
        for (int mt = 0; mt < 2; ++mt)
#pragma unroll
          for (int nt = 0; nt < 4; ++nt) {
            if (!CX) {
              dmma884(acc[0][mt][nt][0], acc[0][mt][nt][1], bf[0][mt], af[0][nt]);
            } else {
              // (br + i bi)(ar + i ai) = (br ar - bi ai) + i (br ai + bi ar)
              dmma884(acc[0][mt][nt][0], acc[0][mt][nt][1], bf[0][mt], af[0][nt]);
              dmma884(acc[0][mt][nt][0], acc[0][mt][nt][1], -bf[NP - 1][mt], af[NP - 1][nt]);
              dmma884(acc[NP - 1][mt][nt][0], acc[NP - 1][mt][nt][1], bf[0][mt], af[NP - 1][nt]);
              dmma884(acc[NP - 1][mt][nt][0], acc[NP - 1][mt][nt][1], bf[NP - 1][mt], af[0][nt]);
            }
          }
      }
    }
    // epilogue: accumulator (row lm, cols 2*lk, 2*lk+1) of each 8x8 tile
#pragma unroll
    for (int mt = 0; mt < 2; ++mt) {
      const int row = r0 + wr * 16 + mt * 8 + lm;
      if (row >= n) continue;
#pragma unroll
      for (int nt = 0; nt < 4; ++nt) {
#pragma unroll
        for (int e = 0; e < 2; ++e) {
          const int col = c0 + wc * 32 + nt * 8 + 2 * lk + e;
          if (col >= n) continue;
          T a;
          if (!CX) a = sc_from(acc[0][mt][nt][e], 0.0, T{});
          else a = sc_from(acc[0][mt][nt][e], acc[NP - 1][mt][nt][e], T{});
          T old;
          if (!CX) old = sc_from(tv[CX ? 0 : mt][CX ? 0 : nt][e], 0.0, T{});
          else if (!SKEW || col > row) old = Tw[(size_t)row * n + col];
          if (SKEW) {
            if (col > row) {
              const T v = S::add(old, a);
              Tw[(size_t)row * n + col] = v;
              Tw[(size_t)col * n + row] = S::neg(v);
            }
          } else {
            Tw[(size_t)row * n + col] = S::sub(old, a);
          }
        }
      }
    }
  }
}

template <typename T, bool SKEW>
static int launch_flush_t(const State& st, Ctx& cx, cudaStream_t s) {
  const int t1 = (st.n + 63) / 64;
  const int64_t tiles = SKEW ? (int64_t)t1 * (t1 + 1) / 2 : (int64_t)t1 * t1;
  const int occ = cx.configure((const void*)flush_dmma_kernel<T, SKEW>, 256, 0);
  if (occ < 0) return -1;
  cx.name(LRUX_PROF_FLUSH, "flush_dmma_kernel");
  int64_t grid = (int64_t)cx.num_sms * occ;
  if (grid > st.W * tiles) grid = st.W * tiles;
  flush_dmma_kernel<T, SKEW><<<(unsigned)grid, 256, 0, s>>>(st, t1);
  return 1;
}

int launch_flush_dmma(const State& st, Ctx& cx, cudaStream_t s) {
  if (st.kind == KIND_PF)
    return st.dt == LRUX_F64 ? launch_flush_t<double, true>(st, cx, s)
                             : launch_flush_t<cplx, true>(st, cx, s);
  return st.dt == LRUX_F64 ? launch_flush_t<double, false>(st, cx, s)
                           : launch_flush_t<cplx, false>(st, cx, s);
}

}  // namespace lrux
