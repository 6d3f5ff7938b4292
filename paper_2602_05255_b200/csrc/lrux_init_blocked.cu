// Step a0 for large matrices: blocked in-place Gauss-Jordan inversion with partial pivoting.
//
// The unblocked kernel (lrux_init.cu) sweeps the whole n x n matrix once per pivot:
// O(n^3) memory traffic.  Here the n pivots are processed in panels of 32 columns:
//   1. gj_panel_kernel      pivoting + elimination restricted to the 32 panel columns
//                           (all rows): after it the panel holds V = T[:, panel], the block's
//                           combined row transformation T = I + (V - E) E^T (in-place GJ keeps
//                           the transformed unit columns where the eliminated columns were)
//   2. gj_block_apply_kernel  the block's row swaps on the other columns, then
//                           U = M[pivot rows, other columns] and -(V - E) into scratch
//   3. flush_dmma_kernel    M[:, other] += (V - E) U  -- the (n x 32)(32 x n) contraction of
//                           the delayed-update flush (Eq. 12's shape), on the FP64 tensor path
// and at the end one gather undoes the row permutation.  Traffic drops to O(n^3 / 32).
#include "lrux_common.cuh"
#include "lrux_internal.h"

namespace lrux {

constexpr int kPanel = 32;   // = warp width: lane <-> panel column

struct ArgMaxB {
  double v;
  int i;
};
__device__ __forceinline__ ArgMaxB amax_combine(ArgMaxB a, ArgMaxB b) {
  if (b.v > a.v || (b.v == a.v && b.i < a.i)) return b;   // lowest index on ties
  return a;
}

template <typename T>
__device__ __forceinline__ T shfl_elem(T v, int src) { return Sc<T>::shfl(v, src); }

template <typename T>
__global__ void __launch_bounds__(256)
gj_panel_kernel(T* __restrict__ Mall, int n, int c0, int32_t* __restrict__ piv_all,
                T* __restrict__ phase_io, double* __restrict__ logabs_io,
                int32_t* __restrict__ info, int write_amp) {
  using S = Sc<T>;
  __shared__ T prow[kPanel];
  __shared__ ArgMaxB red[8];
  __shared__ int s_p;
  const int w = blockIdx.x, tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  if (info[w] & 1) return;
  T* M = Mall + (size_t)w * n * n;
  int32_t* piv = piv_all + (size_t)w * n;
  const int nbc = min(kPanel, n - c0);
  T phase = S::one();
  double logabs = 0.0;
  if (tid == 0 && write_amp && c0 > 0) { phase = phase_io[w]; logabs = logabs_io[w]; }
  for (int c = c0; c < c0 + nbc; ++c) {
    const int lc = c - c0;
    // ---- pivot: largest modulus in column c at or below the diagonal
    ArgMaxB best{-1.0, 0x7fffffff};
    for (int r = c + tid; r < n; r += 256) {
      double v = S::abs2(M[(size_t)r * n + c]);
      if (!(v == v)) v = -1.0;
      best = amax_combine(best, ArgMaxB{v, r});
    }
#pragma unroll
    for (int m = 16; m > 0; m >>= 1) {
      ArgMaxB o;
      o.v = __shfl_xor_sync(0xffffffffu, best.v, m);
      o.i = __shfl_xor_sync(0xffffffffu, best.i, m);
      best = amax_combine(best, o);
    }
    if (lane == 0) red[warp] = best;
    __syncthreads();
    if (tid == 0) {
      ArgMaxB b = red[0];
      for (int q = 1; q < 8; ++q) b = amax_combine(b, red[q]);
      s_p = (!(b.v > 0.0) || !isfinite(b.v)) ? -1 : b.i;
    }
    __syncthreads();
    const int p = s_p;
    if (p < 0) {   // singular: uniform exit
      if (tid == 0) {
        atomicOr(&info[w], 1);
        if (write_amp) { phase_io[w] = S::zero(); logabs_io[w] = -INFINITY; }
      }
      return;
    }
    // ---- swap rows c <-> p inside the panel, scale the pivot row
    if (warp == 0) {
      const bool on = lane < nbc;
      const T a = on ? M[(size_t)c * n + c0 + lane] : S::zero();
      const T b = on ? M[(size_t)p * n + c0 + lane] : S::zero();
      if (on && p != c) M[(size_t)p * n + c0 + lane] = a;
      const T d = shfl_elem(b, lc);
      const T dinv = S::inv(d);
      const T v = (lane == lc) ? dinv : S::mul(b, dinv);
      if (on) { prow[lane] = v; M[(size_t)c * n + c0 + lane] = v; }
      else prow[lane] = S::zero();
      if (lane == 0) {
        piv[c] = p;
        const double ad = S::abs(d);
        phase = S::mul(phase, S::unit(d, ad));
        if (p != c) phase = S::neg(phase);
        logabs += log(ad);
      }
    }
    __syncthreads();
    // ---- eliminate: every other row, 4 rows in flight per warp
    const T pv = prow[lane];
    for (int r0 = warp; r0 < n; r0 += 32) {
      T x[4];
#pragma unroll
      for (int u = 0; u < 4; ++u) {
        const int r = r0 + 8 * u;
        x[u] = (r < n && lane < nbc) ? M[(size_t)r * n + c0 + lane] : S::zero();
      }
#pragma unroll
      for (int u = 0; u < 4; ++u) {
        const int r = r0 + 8 * u;
        const T f = shfl_elem(x[u], lc);
        if (r < n && r != c && lane < nbc) {
          const T base = (lane == lc) ? S::zero() : x[u];
          M[(size_t)r * n + c0 + lane] = S::fnma(f, pv, base);
        }
      }
    }
    __syncthreads();
  }
  if (tid == 0 && write_amp) { phase_io[w] = phase; logabs_io[w] = logabs; }
}

// Thread per column j (grid (W, ceil(n/256))).  Also sets up the flush bookkeeping.
template <typename T>
__global__ void __launch_bounds__(256)
gj_block_apply_kernel(State st, int c0) {
  using S = Sc<T>;
  const int n = st.n;
  const int w = blockIdx.x, j = blockIdx.y * 256 + threadIdx.x;
  const int nbc = min(kPanel, n - c0);
  if (blockIdx.y == 0 && threadIdx.x == 0) {
    st.fill[w] = (st.info[w] & 1) ? 0 : nbc;
    st.flist[w] = w;
    if (w == 0) st.counters[1] = (int)st.W;
  }
  if ((st.info[w] & 1) || j >= n) return;
  T* M = (T*)st.Ti + (size_t)w * n * n;
  const int32_t* piv = st.init_piv + (size_t)w * n;
  T* Ab = (T*)st.Abuf + (size_t)w * st.cap * n;
  T* Bb = (T*)st.Bbuf + (size_t)w * st.cap * n;
  const bool in_panel = j >= c0 && j < c0 + nbc;
  if (!in_panel) {
    for (int s = 0; s < nbc; ++s) {
      const int c = c0 + s, p = piv[c];
      if (p != c) {
        const T a = M[(size_t)c * n + j];
        M[(size_t)c * n + j] = M[(size_t)p * n + j];
        M[(size_t)p * n + j] = a;
      }
    }
  }
  for (int s = 0; s < nbc; ++s) {
    Ab[(size_t)s * n + j] = in_panel ? S::zero() : M[(size_t)(c0 + s) * n + j];
    T v = M[(size_t)j * n + c0 + s];           // V[j][s]
    if (j == c0 + s) v = S::sub(v, S::one());
    Bb[(size_t)s * n + j] = S::neg(v);         // flush computes Ti -= Bbuf^T Abuf
  }
}

// newM[r][j] = M[r][arr[j]], arr = the column swaps (c <-> piv[c], c = n-1 .. 0) applied to
// the identity: undoes the row permutation of the elimination.  Grid (W, 8).
template <typename T>
__global__ void __launch_bounds__(256) gj_unpermute_kernel(State st) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const int n = st.n;
  T* buf = (T*)smem_raw;               // [n]
  int* arr = (int*)(buf + n);          // [n]
  const int w = blockIdx.x, tid = threadIdx.x;
  if (st.info[w] & 1) return;
  const int32_t* piv = st.init_piv + (size_t)w * n;
  for (int j = tid; j < n; j += 256) arr[j] = j;
  __syncthreads();
  if (tid == 0)
    for (int c = n - 1; c >= 0; --c) {
      const int p = piv[c];
      if (p != c) { const int t = arr[c]; arr[c] = arr[p]; arr[p] = t; }
    }
  __syncthreads();
  T* M = (T*)st.Ti + (size_t)w * n * n;
  for (int r = blockIdx.y; r < n; r += gridDim.y) {
    for (int j = tid; j < n; j += 256) buf[j] = M[(size_t)r * n + j];
    __syncthreads();
    for (int j = tid; j < n; j += 256) M[(size_t)r * n + j] = buf[arr[j]];
    __syncthreads();
  }
}

__global__ void clear_fill_kernel(State st) {
  const int64_t w = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (w < st.W) st.fill[w] = 0;
  if (w == 0) st.counters[1] = 0;
}

template <typename T>
static int gj_blocked_t(const State& st, bool write_amp, Ctx& cx, cudaStream_t s) {
  const int n = st.n;
  State st2 = st;          // the flush kernel sees the init scratch as a 32-deep delay buffer
  st2.Abuf = st.init_A;
  st2.Bbuf = st.init_B;
  st2.cap = kPanel;
  st2.kind = KIND_DET;
  int nl = 0;
  const dim3 gcol((unsigned)st.W, (unsigned)((n + 255) / 256));
  for (int c0 = 0; c0 < n; c0 += kPanel) {
    gj_panel_kernel<T><<<(unsigned)st.W, 256, 0, s>>>((T*)st.Ti, n, c0, st.init_piv, (T*)st.phase,
                                                      st.logabs, st.info, write_amp ? 1 : 0);
    gj_block_apply_kernel<T><<<gcol, 256, 0, s>>>(st2, c0);
    nl += 2 + launch_flush_dmma(st2, cx, s);
  }
  const size_t sm = (size_t)n * (sizeof(T) + 4);
  if (cx.configure((const void*)gj_unpermute_kernel<T>, 256, sm) < 0) return -1;
  gj_unpermute_kernel<T><<<dim3((unsigned)st.W, 8), 256, sm, s>>>(st2);
  clear_fill_kernel<<<(unsigned)((st.W + 255) / 256), 256, 0, s>>>(st2);
  nl += 2;
  return cudaGetLastError() == cudaSuccess ? nl : -1;
}

// In-place inverse of st.Ti (already loaded) for n >= kBlockedInitMin; 0 = not applicable.
int launch_gj_blocked(const State& st, bool write_amp, Ctx& cx, cudaStream_t s) {
  if (!st.init_A || !st.init_B || !st.init_piv) return 0;
  const char* keep = cx.last[LRUX_PROF_FLUSH];   // the trailing updates borrow the flush kernel
  const int r = st.dt == LRUX_F64 ? gj_blocked_t<double>(st, write_amp, cx, s)
                                  : gj_blocked_t<cplx>(st, write_amp, cx, s);
  cx.last[LRUX_PROF_FLUSH] = keep;
  return r;
}

}  // namespace lrux
