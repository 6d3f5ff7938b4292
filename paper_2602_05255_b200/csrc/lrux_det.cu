// Determinant hot path.
//
// New-rows-only forms used here (readings 5/5b), with P the k
// replaced row indices, N (k x n) the new rows, C = A^-1[:,P]:
//   R = 1 + u^T A^-1 v = N C                                  (Eq. 4)
//   u^T A^-1 = N A^-1 - I[P,:]  =: Wm
//   A'^-1 = A^-1 - C R^-1 Wm                                  (Eq. 5)
// State Ti = A^-T row-major, so C[:,a] is the contiguous row P[a] of Ti and column
// j of Wm depends only on row j of Ti: the update is a single pass over Ti.
#include "lrux_common.cuh"
#include "lrux_internal.h"

// smallest template rank (1, 2, 4, 8) from which real-valued updates take the DMMA kernel
#ifndef LRUX_DMMA_MIN_KT
#define LRUX_DMMA_MIN_KT 4
#endif
// ... and from which real-valued delayed appends take the row-dot DMMA pass
// rows of A0^-1 per work item of the register-row / complex-DMMA append
#ifndef LRUX_RATIO_FLY_MAX_KT
#define LRUX_RATIO_FLY_MAX_KT 4
#endif
// CTAs per SM the ratio kernel is compiled for (64 registers; complex k = 8 keeps 128: it would spill)
// 1: one warp per walker in the ratio for n <= 128; 2: also n <= 256 with k <= 2 and no delay buffer (configs[1]:
// ratio 22.5 -> 19.1 us per step, 18.88 M -> 19.10 M walker-updates/s; with K = 16 the CTA kernel is faster)
#ifndef LRUX_RATIO_WARP
#define LRUX_RATIO_WARP 2
#endif
#ifndef LRUX_RATIO_MINB
#define LRUX_RATIO_MINB 4
#endif
#ifndef LRUX_RATIO_FLY_MAX_KT_CX
#define LRUX_RATIO_FLY_MAX_KT_CX 2
#endif
#ifndef LRUX_APPEND_REAL_STREAM_MIN_K
#define LRUX_APPEND_REAL_STREAM_MIN_K 1
#endif
// per-warp copies of N in the real stream append up to this much shared memory (n <= 256 with k <= 4:
// n=128 k=2 0.49 of HBM against 0.40, n=256 k=4 0.57 / 0.55; beyond -- n=384, or k > 4 -- the shared copy wins)
#ifndef LRUX_APPEND_PW_SMEM_KB
#define LRUX_APPEND_PW_SMEM_KB 68
#endif
#ifndef LRUX_APPEND_TILE_ROWS
#define LRUX_APPEND_TILE_ROWS 128
#endif
#ifndef LRUX_APPEND_ROWDOT_MIN_KT
#define LRUX_APPEND_ROWDOT_MIN_KT 8
#endif

namespace lrux {

// ---------------------------------------------------------------- ratio (a1, a2, a5)
// Grid (W, nsplit): CTA (w, sp) owns the column slice [sp*256, sp*256+256) of walker w.
// Each thread owns EPT elements i of the k gathered columns C_eff = A_eff^-1[:,P] and
// walks the delay buffer ONCE for all of them:
//   a_tau = A0^-1 v - sum_t a_t (b_t^T v)                       (Eq. 14)
// (b_t^T v = Bbuf[s][P[a]] is a warp-uniform load).  C_eff and N are stashed for
// accept.  R = N C_eff (Eq. 4 / Eq. 13): every slice writes its partial k x k sum
// (accumulated on the fly), and the slice that finishes last adds the partials in slice
// order (deterministic) -- or, with KT = 8, forms R from the complete stash --
// and evaluates r = det R by a k x k LU in one thread.
template <typename T, int KT, int EPT>
__global__ void __launch_bounds__(256, (sizeof(T) == 16 && KT == 8) ? 2 : LRUX_RATIO_MINB)
det_ratio_kernel(State st, int k, const int32_t* __restrict__ idx, const T* __restrict__ rows,
                 T* __restrict__ ratio_out) {
  using S = Sc<T>;
  // k x k accumulators in registers up to k = 4; at k = 8 the 64 accumulators cost 161 registers
  // (one CTA per SM, 4.2 ms per step at n = 512, W = 8192): R comes from the complete stash instead
  // (complex: up to k = 2 -- at k = 4 the 32 accumulator doubles meant 102 registers, two CTAs per SM and
  // 6.9 waves for configs[3]: 180 us per step)
  constexpr bool FLY = KT <= (sizeof(T) == 8 ? LRUX_RATIO_FLY_MAX_KT : LRUX_RATIO_FLY_MAX_KT_CX);
  extern __shared__ __align__(16) unsigned char smem_raw[];
  T* Bp = (T*)smem_raw;  // [fill][KT]: b_t^T v = Bbuf[s][P[a]]
  __shared__ T Rs[kMaxK * kMaxK];
  __shared__ T Ri[kMaxK * kMaxK];
  // real k = 8: the slice's partial R by DMMA from the stash this CTA has just written (n even)
  constexpr bool DM = !FLY && sizeof(T) == 8 && KT == 8;
  __shared__ T red[8][(FLY || DM) ? KT * KT : 1];
  __shared__ int sP[KT];
  __shared__ int is_last;
  const int w = blockIdx.x, sp = blockIdx.y, nsplit = gridDim.y;
  const int tid = threadIdx.x, nt = blockDim.x;
  const int warp = tid >> 5, lane = tid & 31, nw = nt >> 5;
  const int n = st.n, kmax = st.kmax;
  if (w == 0 && sp == 0 && tid == 0) st.counters[0] = 0;
  int P[KT];
  bool bad = false;
#pragma unroll
  for (int a = 0; a < KT; ++a) {
    P[a] = a < k ? idx[(size_t)w * k + a] : -1 - a;
    if (a < k && (P[a] < 0 || P[a] >= n)) bad = true;
#pragma unroll
    for (int c = 0; c < a; ++c)
      if (a < k && P[c] == P[a]) bad = true;
  }
  if (bad) {   // uniform over the walker's CTAs
    if (sp == 0 && tid == 0) {
      ratio_out[w] = S::nan();
      ((T*)st.pend_ratio)[w] = S::nan();
      st.pend_ok[w] = 0;
      atomicOr(&st.info[w], 2);
    }
    return;
  }
  const int fill = st.cap ? st.fill[w] : 0;
  const T* Tw = (const T*)st.Ti + (size_t)w * n * n;
  const T* Ab = st.cap ? (const T*)st.Abuf + (size_t)w * st.cap * n : nullptr;
  const T* Bb = st.cap ? (const T*)st.Bbuf + (size_t)w * st.cap * n : nullptr;
  T* pC = (T*)st.pend_C + (size_t)w * kmax * n;
  T* pN = (T*)st.pend_N + (size_t)w * kmax * n;
  T racc[KT][KT];   // unused (and removed by the compiler) when !FLY
#pragma unroll
  for (int b = 0; b < KT; ++b)
#pragma unroll
    for (int a = 0; a < KT; ++a) racc[b][a] = S::zero();
  if (fill > 0) {
    if (tid == 0) {
#pragma unroll
      for (int a = 0; a < KT; ++a) sP[a] = a < k ? P[a] : P[0];
    }
    __syncthreads();
    for (int q = tid; q < fill * KT; q += nt) Bp[q] = Bb[(size_t)(q / KT) * n + sP[q % KT]];
    __syncthreads();
  }
  {
    const int i0 = sp * kRatioSlice;
    T c[KT][EPT];
#pragma unroll
    for (int e = 0; e < EPT; ++e) {
      const int i = i0 + tid + nt * e;
#pragma unroll
      for (int a = 0; a < KT; ++a)
        c[a][e] = (a < k && i < n) ? Tw[(size_t)P[a] * n + i] : S::zero();
    }
#pragma unroll 8
    for (int s = 0; s < fill; ++s) {
      T av[EPT];
#pragma unroll
      for (int e = 0; e < EPT; ++e) {
        const int i = i0 + tid + nt * e;
        av[e] = i < n ? Ab[(size_t)s * n + i] : S::zero();
      }
#pragma unroll
      for (int a = 0; a < KT; ++a) {
        const T bp = Bp[s * KT + a];
#pragma unroll
        for (int e = 0; e < EPT; ++e) c[a][e] = S::fnma(bp, av[e], c[a][e]);
      }
    }
#pragma unroll
    for (int e = 0; e < EPT; ++e) {
      const int i = i0 + tid + nt * e;
      if (i < n) {
#pragma unroll
        for (int b = 0; b < KT; ++b) {
          if (b < k) {
            const T x = rows[((size_t)w * k + b) * n + i];
            pN[(size_t)b * n + i] = x;
            pC[(size_t)b * n + i] = c[b][e];
            if constexpr (FLY) {
#pragma unroll
              for (int a = 0; a < KT; ++a) racc[b][a] = S::fma(x, c[a][e], racc[b][a]);
            }
          }
        }
      }
    }
  }
  T* part = (T*)st.pend_Rpart + ((size_t)w * nsplit + sp) * kmax * kmax;
  const bool dm = DM && (n & 1) == 0;
  if constexpr (DM) {
    if (dm) {
      // R[b][a] = sum_i N[b][i] C[a][i] over this slice's columns: lane (r, q) reads the 16-byte pairs
      // N[r][c + 2q, +1] and C[r][c + 2q, +1] (permuted contraction index), two DMMAs per 8 columns;
      // the warps take the slice's 8-column blocks in turn.  D fragment = R[r][2q, 2q + 1].
      __syncthreads();   // the CTA's own stores to pN / pC are visible to all of its threads
      const int r8 = lane >> 2, q = lane & 3;
      const int i0 = sp * kRatioSlice;
      double d0 = 0.0, d1 = 0.0, e0 = 0.0, e1 = 0.0;
      for (int c8 = warp * 8; c8 < kRatioSlice; c8 += nw * 8) {
        const int col = i0 + c8 + 2 * q;
        double2 nv = make_double2(0.0, 0.0), cv = nv;
        if (col < n && r8 < k) {
          nv = *(const double2*)((const double*)pN + (size_t)r8 * n + col);
          cv = *(const double2*)((const double*)pC + (size_t)r8 * n + col);
        }
        asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
                     : "+d"(d0), "+d"(d1) : "d"(nv.x), "d"(cv.x));
        asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
                     : "+d"(e0), "+d"(e1) : "d"(nv.y), "d"(cv.y));
      }
      ((double*)&red[warp][r8 * KT + 2 * q])[0] = d0 + e0;
      ((double*)&red[warp][r8 * KT + 2 * q + 1])[0] = d1 + e1;
    }
  }
  if constexpr (FLY) {
#pragma unroll
    for (int b = 0; b < KT; ++b)
#pragma unroll
      for (int a = 0; a < KT; ++a) {
        const T v = warp_sum(racc[b][a]);
        if (lane == 0) red[warp][b * KT + a] = v;
      }
  }
  if (FLY || dm) {
    __syncthreads();
    if (tid < KT * KT) {
      T v = red[0][tid];
      for (int q = 1; q < nw; ++q) v = S::add(v, red[q][tid]);
      if (nsplit == 1) Rs[(tid / KT) * kMaxK + (tid % KT)] = v;
      else if (tid / KT < k && tid % KT < k) part[(tid / KT) * kmax + (tid % KT)] = v;
    }
  }
  if (nsplit > 1 || !(FLY || dm)) {
    // make this slice's stash / partial visible, then find out whether we are last
    __threadfence();
    __syncthreads();
    if (tid == 0) {
      const int done = nsplit > 1 ? atomicAdd(&st.pend_cnt[w], 1) : 0;
      is_last = done == nsplit - 1;
      if (is_last && nsplit > 1) st.pend_cnt[w] = 0;
    }
    __syncthreads();
    if (!is_last) return;
    __threadfence();
    if (FLY || dm) {
      if (tid < KT * KT && tid / KT < k && tid % KT < k) {
        const T* p0 = (const T*)st.pend_Rpart + (size_t)w * nsplit * kmax * kmax +
                      (tid / KT) * kmax + (tid % KT);
        T v = S::zero();
        for (int q = 0; q < nsplit; ++q) {
          const double2* src = (const double2*)(p0 + (size_t)q * kmax * kmax);
          T x;
          if constexpr (sizeof(T) == 16) { const double2 t = __ldcg(src); x = sc_from(t.x, t.y, T{}); }
          else x = sc_from(__ldcg((const double*)src), 0.0, T{});
          v = S::add(v, x);
        }
        Rs[(tid / KT) * kMaxK + (tid % KT)] = v;
      }
    } else {
      for (int pr = warp; pr < k * k; pr += nw) {
        const int a = pr / k, b = pr % k;
        T acc = S::zero();
        for (int i = lane; i < n; i += 32) {
          T x, y;
          if constexpr (sizeof(T) == 16) {
            const double2 tx = __ldcg((const double2*)(pN + (size_t)a * n + i));
            const double2 ty = __ldcg((const double2*)(pC + (size_t)b * n + i));
            x = sc_from(tx.x, tx.y, T{}); y = sc_from(ty.x, ty.y, T{});
          } else {
            x = sc_from(__ldcg((const double*)(pN + (size_t)a * n + i)), 0.0, T{});
            y = sc_from(__ldcg((const double*)(pC + (size_t)b * n + i)), 0.0, T{});
          }
          acc = S::fma(x, y, acc);
        }
        acc = warp_sum(acc);
        if (lane == 0) Rs[a * kMaxK + b] = acc;
      }
    }
  }
  __syncthreads();
  if (warp == 0) {   // k x k elimination by one warp (bit-identical to the serial small_det_inv)
    bool ok;
    const T det = warp_det_inv<T, KT>(Rs, Ri, k, kMaxK, &ok, lane);
    if (lane == 0) {
      ratio_out[w] = det;
      ((T*)st.pend_ratio)[w] = det;
      st.pend_ok[w] = ok ? 1 : 0;
    }
    T* pR = (T*)st.pend_Rinv + (size_t)w * st.kc * st.kc;
    for (int q = lane; q < k * k; q += 32) pR[(q / k) * st.kc + (q % k)] = Ri[(q / k) * kMaxK + (q % k)];
#pragma unroll
    for (int a = 0; a < KT; ++a)
      if (lane == a && a < k) st.pend_idx[(size_t)w * kmax + a] = P[a];
  }
}

// Narrow matrices (n <= 128): ONE WARP per walker, 8 walkers per CTA.  With one CTA per walker the
// ratio had become the step at these sizes (n = 64, k = 8, W = 32768: 306 us of ratio for 77 us of
// update -- one small CTA, two barriers and a single-warp tail per walker).  Lane l owns the
// columns l, l + 32, ... (EPT of them) of the k gathered columns; the delay buffer is walked as in
// det_ratio_kernel (Eq. 14), C_eff and N are stashed, R = N C_eff comes from k^2 warp reductions
// and the elimination is warp_det_inv on the warp's own 2 x KT x KT doubles of shared memory.
template <typename T, int KT, int EPT>
__global__ void __launch_bounds__(256)
det_ratio_warp_kernel(State st, int k, const int32_t* __restrict__ idx, const T* __restrict__ rows,
                      T* __restrict__ ratio_out) {
  using S = Sc<T>;
  __shared__ T Rs[8][KT * KT];
  __shared__ T Ri[8][KT * KT];
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int64_t w = (int64_t)blockIdx.x * 8 + warp;
  const int n = st.n, kmax = st.kmax;
  if (blockIdx.x == 0 && threadIdx.x == 0) st.counters[0] = 0;
  if (w >= st.W) return;
  int P[KT];
  bool bad = false;
#pragma unroll
  for (int a = 0; a < KT; ++a) {
    P[a] = a < k ? idx[(size_t)w * k + a] : -1 - a;
    if (a < k && (P[a] < 0 || P[a] >= n)) bad = true;
#pragma unroll
    for (int c = 0; c < a; ++c)
      if (a < k && P[c] == P[a]) bad = true;
  }
  if (bad) {
    if (lane == 0) {
      ratio_out[w] = S::nan();
      ((T*)st.pend_ratio)[w] = S::nan();
      st.pend_ok[w] = 0;
      atomicOr(&st.info[w], 2);
    }
    return;
  }
  const int fill = st.cap ? st.fill[w] : 0;
  const T* Tw = (const T*)st.Ti + (size_t)w * n * n;
  const T* Ab = st.cap ? (const T*)st.Abuf + (size_t)w * st.cap * n : nullptr;
  const T* Bb = st.cap ? (const T*)st.Bbuf + (size_t)w * st.cap * n : nullptr;
  T* pC = (T*)st.pend_C + (size_t)w * kmax * n;
  T* pN = (T*)st.pend_N + (size_t)w * kmax * n;
  T c[KT][EPT];
#pragma unroll
  for (int e = 0; e < EPT; ++e) {
    const int i = lane + 32 * e;
#pragma unroll
    for (int a = 0; a < KT; ++a) c[a][e] = (a < k && i < n) ? Tw[(size_t)P[a] * n + i] : S::zero();
  }
  for (int s2 = 0; s2 < fill; ++s2) {
    T av[EPT];
#pragma unroll
    for (int e = 0; e < EPT; ++e) {
      const int i = lane + 32 * e;
      av[e] = i < n ? Ab[(size_t)s2 * n + i] : S::zero();
    }
#pragma unroll
    for (int a = 0; a < KT; ++a) {
      if (a < k) {
        const T bp = Bb[(size_t)s2 * n + P[a]];          // b_t^T v: the same address for the whole warp
#pragma unroll
        for (int e = 0; e < EPT; ++e) c[a][e] = S::fnma(bp, av[e], c[a][e]);
      }
    }
  }
#pragma unroll
  for (int e = 0; e < EPT; ++e) {
    const int i = lane + 32 * e;
    if (i < n) {
#pragma unroll
      for (int a = 0; a < KT; ++a)
        if (a < k) pC[(size_t)a * n + i] = c[a][e];
    }
  }
#pragma unroll
  for (int b = 0; b < KT; ++b) {
    if (b < k) {
      T x[EPT];
#pragma unroll
      for (int e = 0; e < EPT; ++e) {
        const int i = lane + 32 * e;
        x[e] = i < n ? rows[((size_t)w * k + b) * n + i] : S::zero();
        if (i < n) pN[(size_t)b * n + i] = x[e];
      }
#pragma unroll
      for (int a = 0; a < KT; ++a) {
        if (a < k) {
          T v = S::zero();
#pragma unroll
          for (int e = 0; e < EPT; ++e) v = S::fma(x[e], c[a][e], v);
          v = warp_sum(v);
          if (lane == 0) Rs[warp][b * KT + a] = v;
        }
      }
    }
  }
  __syncwarp();
  bool ok;
  const T det = warp_det_inv<T, KT>(Rs[warp], Ri[warp], k, KT, &ok, lane);
  if (lane == 0) {
    ratio_out[w] = det;
    ((T*)st.pend_ratio)[w] = det;
    st.pend_ok[w] = ok ? 1 : 0;
  }
  T* pR = (T*)st.pend_Rinv + (size_t)w * st.kc * st.kc;
  for (int q = lane; q < k * k; q += 32) pR[(q / k) * st.kc + (q % k)] = Ri[warp][(q / k) * KT + (q % k)];
#pragma unroll
  for (int a = 0; a < KT; ++a)
    if (lane == a && a < k) st.pend_idx[(size_t)w * kmax + a] = P[a];
}

// ---------------------------------------------------------------- select + amplitude (a8)
// Compacts the accepted walkers into st.list and multiplies the amplitude by r,
// kept as (phase, log|.|)  (detA *= r).
template <typename T>
__global__ void select_kernel(State st, const uint8_t* __restrict__ mask) {
  using S = Sc<T>;
  const int64_t w = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (w == 0) st.counters[1] = 0;
  if (w >= st.W) return;
  bool acc = mask[w] != 0;
  if (acc && !st.pend_ok[w]) {
    atomicOr(&st.info[w], 4);
    acc = false;
  }
  st.pend_ok[w] = 0;
  if (!acc) return;
  const int slot = atomicAdd(&st.counters[0], 1);
  st.list[slot] = (int32_t)w;
  const T r = ((const T*)st.pend_ratio)[w];
  const double ar = S::abs(r);
  st.logabs[w] += log(ar);
  T* ph = (T*)st.phase;
  ph[w] = S::mul(ph[w], S::unit(r, ar));
}
template __global__ void select_kernel<double>(State, const uint8_t*);
template __global__ void select_kernel<cplx>(State, const uint8_t*);

// ---------------------------------------------------------------- immediate update (a3)
// Work item = (accepted walker, tile of rows of Ti).  Persistent grid.  Each warp
// owns whole rows: row j is loaded once into registers, its k dot products with N
// give column j of Wm, and the row is written back once:
//   Ti[j][:] -= sum_a g[a] C[a][:],   g = R^-1 (N Ti[j][:] - [j == P])
// N, C (k x n each) are staged in shared memory once per item.
// VEC elements per 16-byte lane access; CH chunks of 32*VEC elements cover a row.
template <typename T, int VEC>
struct RowVec;
template <>
struct RowVec<double, 2> {
  using type = double2;
  static __device__ __forceinline__ double get(const double2& v, int e) { return e ? v.y : v.x; }
  static __device__ __forceinline__ void set(double2& v, int e, double x) { if (e) v.y = x; else v.x = x; }
};
template <>
struct RowVec<double, 1> {
  using type = double;
  static __device__ __forceinline__ double get(const double& v, int) { return v; }
  static __device__ __forceinline__ void set(double& v, int, double x) { v = x; }
};
template <>
struct RowVec<cplx, 1> {
  using type = double2;
  static __device__ __forceinline__ cplx get(const double2& v, int) { return cplx{v.x, v.y}; }
  static __device__ __forceinline__ void set(double2& v, int, cplx x) { v.x = x.re; v.y = x.im; }
};

template <typename T, int KT, int VEC, int CH, int RW>
__global__ void __launch_bounds__(256)
det_update_kernel(State st, int k, int tiles, int rows_per_tile) {
  using S = Sc<T>;
  using RV = RowVec<T, VEC>;
  using V = typename RV::type;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const int n = st.n, kmax = st.kmax;
  T* Ns = (T*)smem_raw;            // [k][n]
  T* Cs = Ns + (size_t)k * n;      // [k][n]
  __shared__ T Ri[KT * KT];
  __shared__ int sidx[KT];
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31, nw = blockDim.x >> 5;
  const int count = st.counters[0];
  const int nvec = n / VEC;  // vectors per row
  // Work unit = one pass of the CTA's warps (nw * RW rows); every CTA takes a CONTIGUOUS, equal
  // range of the units of the concatenated accepted list, so that N, C, R^-1 are staged once per
  // walker and CTA (they were staged per 64-row tile: 8 KB of staging per 128 KB of rows at
  // configs[1]) and the last wave is a fraction of a unit, not of a tile.
  (void)tiles; (void)rows_per_tile;
  const int rpu = nw * RW;
  const int upw = (n + rpu - 1) / rpu;
  const int64_t total = (int64_t)count * upw;
  const int64_t first = total * blockIdx.x / gridDim.x, last = total * (blockIdx.x + 1) / gridDim.x;
  int wi = (int)(first / upw), ul = (int)(first % upw);   // 32-bit running (walker, unit) from here on
  const int my = (int)(last - first);
  bool fresh = true;
  int w = my > 0 ? st.list[wi] : 0;
  for (int it = 0; it < my;) {
    if (ul == upw) { ul = 0; w = st.list[++wi]; fresh = true; }
    // up to 4 units of the same walker in an inner loop without a barrier (the compiler overlaps
    // their loads; one unit per barrier-carrying iteration cost 5 % at configs[1]: 0.87 of HBM
    // against 0.94); n <= 128 -- a walker is 4-8 units -- is faster one unit at a time (0.93 / 0.89
    // at n = 128 / 64 against 0.89 / 0.86)
    const int nun = min(min(n <= 128 ? 1 : 4, upw - ul), my - it);
    if (fresh) {
    fresh = false;
    __syncthreads();
    {
      const V* gN = (const V*)((const T*)st.pend_N + (size_t)w * kmax * n);
      const V* gC = (const V*)((const T*)st.pend_C + (size_t)w * kmax * n);
      for (int q = tid; q < k * nvec; q += blockDim.x) {
        ((V*)Ns)[q] = gN[q];
        ((V*)Cs)[q] = gC[q];
      }
      if (tid < KT * KT) {
        const int a = tid / KT, b = tid % KT;
        Ri[tid] = (a < k && b < k) ? ((const T*)st.pend_Rinv)[(size_t)w * st.kc * st.kc + a * st.kc + b]
                                   : S::zero();
      }
      if (tid < KT) sidx[tid] = tid < k ? st.pend_idx[(size_t)w * kmax + tid] : -1;
    }
    __syncthreads();
    }
    T* Tw = (T*)st.Ti + (size_t)w * n * n;
    const int j_end = min(n, (ul + nun) * rpu);
    const int j_beg = ul * rpu + warp * RW;
    ul += nun;
    it += nun;
    for (int j0 = j_beg; j0 < j_end; j0 += rpu) {
      V x[RW][CH];
      T d[RW][KT];
#pragma unroll
      for (int r = 0; r < RW; ++r) {
        const bool rv = j0 + r < j_end;
        const V* row = (const V*)(Tw + (size_t)(j0 + r) * n);
#pragma unroll
        for (int m = 0; m < CH; ++m) {
          const int q = lane + 32 * m;
          if (rv && q < nvec) x[r][m] = row[q];
          else { RV::set(x[r][m], 0, S::zero()); if (VEC == 2) RV::set(x[r][m], 1, S::zero()); }
        }
#pragma unroll
        for (int a = 0; a < KT; ++a) d[r][a] = S::zero();
      }
#pragma unroll
      for (int m = 0; m < CH; ++m) {
        const int q = lane + 32 * m;
        if (q < nvec) {
#pragma unroll
          for (int a = 0; a < KT; ++a) {
            if (a < k) {
              const V nv = ((const V*)(Ns + (size_t)a * n))[q];
#pragma unroll
              for (int e = 0; e < VEC; ++e)
#pragma unroll
                for (int r = 0; r < RW; ++r)
                  d[r][a] = S::fma(RV::get(x[r][m], e), RV::get(nv, e), d[r][a]);
            }
          }
        }
      }
      T g[RW][KT];
#pragma unroll
      for (int r = 0; r < RW; ++r) {
#pragma unroll
        for (int a = 0; a < KT; ++a) {
          d[r][a] = warp_sum(d[r][a]);
          if (j0 + r == sidx[a]) d[r][a] = S::sub(d[r][a], S::one());
        }
#pragma unroll
        for (int a = 0; a < KT; ++a) {
          T acc = S::zero();
#pragma unroll
          for (int b = 0; b < KT; ++b) acc = S::fma(Ri[a * KT + b], d[r][b], acc);
          g[r][a] = acc;
        }
      }
#pragma unroll
      for (int m = 0; m < CH; ++m) {
        const int q = lane + 32 * m;
        if (q < nvec) {
#pragma unroll
          for (int a = 0; a < KT; ++a) {
            if (a < k) {
              const V cv = ((const V*)(Cs + (size_t)a * n))[q];
#pragma unroll
              for (int e = 0; e < VEC; ++e)
#pragma unroll
                for (int r = 0; r < RW; ++r)
                  RV::set(x[r][m], e, S::fnma(g[r][a], RV::get(cv, e), RV::get(x[r][m], e)));
            }
          }
#pragma unroll
          for (int r = 0; r < RW; ++r)
            if (j0 + r < j_end) ((V*)(Tw + (size_t)(j0 + r) * n))[q] = x[r][m];
        }
      }
    }
  }
}

// Generic fallback for rows that do not fit in registers: the row is read twice
// (second read hits L1/L2), N and C come from global memory.
template <typename T, int KT>
__global__ void __launch_bounds__(256)
det_update_stream_kernel(State st, int k, int tiles, int rows_per_tile) {
  using S = Sc<T>;
  __shared__ T Ri[KT * KT];
  __shared__ int sidx[KT];
  const int n = st.n, kmax = st.kmax;
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31, nw = blockDim.x >> 5;
  const int count = st.counters[0];
  for (int item = blockIdx.x; item < count * tiles; item += gridDim.x) {
    const int w = st.list[item / tiles];
    const int tile = item % tiles;
    __syncthreads();
    if (tid < KT * KT) {
      const int a = tid / KT, b = tid % KT;
      Ri[tid] = (a < k && b < k) ? ((const T*)st.pend_Rinv)[(size_t)w * st.kc * st.kc + a * st.kc + b]
                                 : S::zero();
    }
    if (tid < KT) sidx[tid] = tid < k ? st.pend_idx[(size_t)w * kmax + tid] : -1;
    __syncthreads();
    const T* gN = (const T*)st.pend_N + (size_t)w * kmax * n;
    const T* gC = (const T*)st.pend_C + (size_t)w * kmax * n;
    T* Tw = (T*)st.Ti + (size_t)w * n * n;
    const int j_end = min(n, (tile + 1) * rows_per_tile);
    // RW rows per warp pass: every N / C element fetched from L1/L2 serves RW rows
    constexpr int RW = 4;
    for (int j0 = tile * rows_per_tile + warp * RW; j0 < j_end; j0 += nw * RW) {
      T d[RW][KT];
#pragma unroll
      for (int r = 0; r < RW; ++r)
#pragma unroll
        for (int a = 0; a < KT; ++a) d[r][a] = S::zero();
      for (int i = lane; i < n; i += 32) {
        T x[RW];
#pragma unroll
        for (int r = 0; r < RW; ++r) x[r] = j0 + r < j_end ? Tw[(size_t)(j0 + r) * n + i] : S::zero();
#pragma unroll
        for (int a = 0; a < KT; ++a) {
          if (a < k) {
            const T nv = gN[(size_t)a * n + i];
#pragma unroll
            for (int r = 0; r < RW; ++r) d[r][a] = S::fma(x[r], nv, d[r][a]);
          }
        }
      }
      T g[RW][KT];
#pragma unroll
      for (int r = 0; r < RW; ++r) {
#pragma unroll
        for (int a = 0; a < KT; ++a) {
          d[r][a] = warp_sum(d[r][a]);
          if (j0 + r == sidx[a]) d[r][a] = S::sub(d[r][a], S::one());
        }
#pragma unroll
        for (int a = 0; a < KT; ++a) {
          T acc = S::zero();
#pragma unroll
          for (int b = 0; b < KT; ++b) acc = S::fma(Ri[a * KT + b], d[r][b], acc);
          g[r][a] = acc;
        }
      }
      for (int i = lane; i < n; i += 32) {
        T x[RW];
#pragma unroll
        for (int r = 0; r < RW; ++r) x[r] = j0 + r < j_end ? Tw[(size_t)(j0 + r) * n + i] : S::zero();
#pragma unroll
        for (int a = 0; a < KT; ++a) {
          if (a < k) {
            const T cv = gC[(size_t)a * n + i];
#pragma unroll
            for (int r = 0; r < RW; ++r) x[r] = S::fnma(g[r][a], cv, x[r]);
          }
        }
#pragma unroll
        for (int r = 0; r < RW; ++r)
          if (j0 + r < j_end) Tw[(size_t)(j0 + r) * n + i] = x[r];
      }
    }
  }
}

// ---------------------------------------------------------------- rank split (a3, large k n)
// A rank-k row replacement is the rank-c replacement of its first c rows followed by
// the rank-(k-c) replacement of the rest in the once-updated matrix.  With
// R^-1 = [[X11, X12], [X21, X22]] (c | k-c blocks) everything the two steps need follows
// from the stash without touching A^-1:
//   first step :  C1, N1, P1,  R11^-1 = X11 - X12 X22^-1 X21
//   second step:  C2' = A1^-1[:,P2] = C2 + C1 X12 X22^-1,  N2, P2,  (Schur complement)^-1 = X22
// This kernel rewrites pend_Rinv[0:c,0:c] and pend_C[c:k] in place (per accepted walker);
// the second step then runs on pointer-shifted views of the same pending area, and may
// be split again.  Used when no TMA-staged instance exists for the full k (registers).
template <typename T>
__global__ void __launch_bounds__(256) det_split_prep_kernel(State st, int c, int k) {
  using S = Sc<T>;
  __shared__ T X22[kMaxK * kMaxK], Z[kMaxK * kMaxK], Q[kMaxK * kMaxK];
  const int n = st.n, kmax = st.kmax, kc = st.kc, m = k - c;
  const int tid = threadIdx.x;
  const int count = st.counters[0];
  for (int it = blockIdx.x; it < count; it += gridDim.x) {
    const int w = st.list[it];
    T* Ri = (T*)st.pend_Rinv + (size_t)w * kc * kc;
    __syncthreads();
    if (tid < m * m) X22[(tid / m) * kMaxK + tid % m] = Ri[(c + tid / m) * kc + c + tid % m];
    __syncthreads();
    if (tid == 0) {
      bool ok;
      small_det_inv(X22, Z, m, kMaxK, &ok);   // Z = X22^-1 (X22 is destroyed)
    }
    __syncthreads();
    if (tid < c * m) {   // Q = X12 Z   (c x m)
      const int a = tid / m, b = tid % m;
      T acc = S::zero();
      for (int q = 0; q < m; ++q) acc = S::fma(Ri[a * kc + c + q], Z[q * kMaxK + b], acc);
      Q[a * kMaxK + b] = acc;
    }
    __syncthreads();
    if (tid < c * c) {   // R11^-1 = X11 - Q X21 (each thread rewrites only its own X11 entry)
      const int a = tid / c, b = tid % c;
      T acc = Ri[a * kc + b];
      for (int q = 0; q < m; ++q) acc = S::fnma(Q[a * kMaxK + q], Ri[(c + q) * kc + b], acc);
      Ri[a * kc + b] = acc;
    }
    T* pC = (T*)st.pend_C + (size_t)w * kmax * n;
    for (int i = tid; i < n; i += 256) {
      T c1[kMaxK];
      for (int a = 0; a < c; ++a) c1[a] = pC[(size_t)a * n + i];
      for (int b = 0; b < m; ++b) {
        T v = pC[(size_t)(c + b) * n + i];
        for (int a = 0; a < c; ++a) v = S::fma(c1[a], Q[a * kMaxK + b], v);
        pC[(size_t)(c + b) * n + i] = v;
      }
    }
  }
}

// ---------------------------------------------------------------- delayed append (a6)
// prep: work item = (accepted walker, group of 8*RW buffer rows).  Each warp reads RW rows
// a_s of Abuf once and forms NA[b][s] = N_b . a_s for all b (-> pend_Y), so that one
// load of N from L2 serves RW buffer rows (with one row per warp the kernel moved four
// times more N than Abuf); group 0 also copies a_tau = C_eff into Abuf[fill .. fill+k)
// (Eq. 14).
constexpr int kPrepRows = 4;   // buffer rows per warp
template <typename T, int KT>
__global__ void __launch_bounds__(256) det_prep_kernel(State st, int k, int groups) {
  using S = Sc<T>;
  constexpr int RW = kPrepRows;
  const int n = st.n, kmax = st.kmax, cap = st.cap;
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int count = st.counters[0];
  for (int item = blockIdx.x; item < count * groups; item += gridDim.x) {
    const int w = st.list[item / groups];
    const int grp = item % groups;
    const int fill = st.fill[w];
    const T* gN = (const T*)st.pend_N + (size_t)w * kmax * n;
    T* Ab = (T*)st.Abuf + (size_t)w * cap * n;
    if (grp == 0) {
      const T* gC = (const T*)st.pend_C + (size_t)w * kmax * n;
      for (int q = tid; q < k * n; q += blockDim.x) Ab[(size_t)fill * n + q] = gC[q];
    }
    const int s0 = (grp * 8 + warp) * RW;
    if (s0 >= fill) continue;
    T acc[RW][KT];
#pragma unroll
    for (int r = 0; r < RW; ++r)
#pragma unroll
      for (int b = 0; b < KT; ++b) acc[r][b] = S::zero();
#pragma unroll 2
    for (int i = lane; i < n; i += 32) {
      T x[RW];
#pragma unroll
      for (int r = 0; r < RW; ++r) x[r] = s0 + r < fill ? Ab[(size_t)(s0 + r) * n + i] : S::zero();
#pragma unroll
      for (int b = 0; b < KT; ++b) {
        if (b < k) {
          const T nb = gN[(size_t)b * n + i];
#pragma unroll
          for (int r = 0; r < RW; ++r) acc[r][b] = S::fma(nb, x[r], acc[r][b]);
        }
      }
    }
    T* NA = (T*)st.pend_Y + (size_t)w * kmax * cap;
#pragma unroll
    for (int r = 0; r < RW; ++r) {
#pragma unroll
      for (int b = 0; b < KT; ++b) {
        if (b < k) {
          const T v = warp_sum(acc[r][b]);
          if (lane == 0 && s0 + r < fill) NA[(size_t)b * cap + s0 + r] = v;
        }
      }
    }
  }
}

// Second half of the append for one (walker, row tile): dsm[b][j] holds d = N A0^-1 - I[P,:]
// on entry; subtract (N Abuf) Bbuf^T, apply R^-1, write Bbuf[fill .. fill+k).
template <typename T, int KT>
__device__ __forceinline__ void append_finish(const State& st, int w, int k, int fill, int j_beg, int j_end,
                                              int rows_per_tile, T* dsm, const T* Ri) {
  using S = Sc<T>;
  const int n = st.n, kmax = st.kmax, cap = st.cap, tid = threadIdx.x;
  __syncthreads();
  // m[b][j] = d[b][j] - sum_s NA[b][s] Bbuf[s][j]: 4 groups of threads split the s range
  const T* NA = (const T*)st.pend_Y + (size_t)w * kmax * cap;
  T* Bb = (T*)st.Bbuf + (size_t)w * cap * n;
  const int nj = j_end - j_beg;
  const int jj = tid % rows_per_tile, sg = tid / rows_per_tile, nsg = blockDim.x / rows_per_tile;
  T m[KT];
#pragma unroll
  for (int b = 0; b < KT; ++b) m[b] = S::zero();
  if (jj < nj && sg < nsg) {
#pragma unroll 8
    for (int s = sg; s < fill; s += nsg) {
      const T bv = Bb[(size_t)s * n + j_beg + jj];
#pragma unroll
      for (int b = 0; b < KT; ++b)
        if (b < k) m[b] = S::fnma(NA[(size_t)b * cap + s], bv, m[b]);
    }
  }
  if (sg >= 1 && sg < nsg && jj < nj) {
#pragma unroll
    for (int b = 0; b < KT; ++b) dsm[(sg * KT + b) * rows_per_tile + jj] = m[b];
  }
  __syncthreads();
  if (sg == 0 && jj < nj) {
#pragma unroll
    for (int b = 0; b < KT; ++b) {
      T v = S::add(dsm[b * rows_per_tile + jj], m[b]);
      for (int g = 1; g < nsg; ++g) v = S::add(v, dsm[(g * KT + b) * rows_per_tile + jj]);
      dsm[b * rows_per_tile + jj] = v;
    }
  }
  __syncthreads();
  for (int q = tid; q < k * nj; q += blockDim.x) {
    const int a = q / nj, j2 = q % nj;
    T acc = S::zero();
#pragma unroll
    for (int b = 0; b < KT; ++b) acc = S::fma(Ri[a * KT + b], dsm[b * rows_per_tile + j2], acc);
    Bb[(size_t)(fill + a) * n + j_beg + j2] = acc;
  }
}

// append: b_tau^T = R^-1 (N A0^-1 - (N Abuf) Bbuf^T - I[P,:])   (Eq. 15 in new-rows form,
// PAPER.md:194; reading 5b) -> Bbuf[fill .. fill+k).  One read-only pass over
// Ti: work item = (accepted walker, tile of RPT rows); N staged in shared memory, each
// warp streams RW rows at a time with 16-byte loads.
template <typename T, int KT, int VEC, int RW>
__global__ void __launch_bounds__(256)
det_append_kernel(State st, int k, int tiles, int rows_per_tile, int n_in_smem) {
  using S = Sc<T>;
  using RV = RowVec<T, VEC>;
  using V = typename RV::type;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const int n = st.n, kmax = st.kmax, cap = st.cap;
  T* dsm = (T*)smem_raw;                         // [4][KT][rows_per_tile] partial sums
  T* Ns = dsm + 4 * KT * rows_per_tile;          // [k][n] (when it fits)
  __shared__ T Ri[KT * KT];
  __shared__ int sidx[KT];
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31, nw = blockDim.x >> 5;
  const int count = st.counters[0];
  const int nvec = n / VEC;
  // each CTA takes a CONTIGUOUS range of (walker, tile) items: N, R^-1 and P are staged once per
  // walker, not once per tile, so that small tiles (an even last wave) cost nothing extra
  const int total = count * tiles;
  const int first = (int)((int64_t)total * blockIdx.x / gridDim.x), last = (int)((int64_t)total * (blockIdx.x + 1) / gridDim.x);
  int cur_w = -1;
  for (int item = first; item < last; ++item) {
    const int w = st.list[item / tiles];
    const int tile = item % tiles;
    const int fill = st.fill[w];
    __syncthreads();
    if (w != cur_w) {
      cur_w = w;
      const V* gN = (const V*)((const T*)st.pend_N + (size_t)w * kmax * n);
      if (n_in_smem)
        for (int q = tid; q < k * nvec; q += blockDim.x) ((V*)Ns)[q] = gN[q];
      if (tid < KT * KT) {
        const int a = tid / KT, b = tid % KT;
        Ri[tid] = (a < k && b < k) ? ((const T*)st.pend_Rinv)[(size_t)w * st.kc * st.kc + a * st.kc + b]
                                   : S::zero();
      }
      if (tid < KT) sidx[tid] = tid < k ? st.pend_idx[(size_t)w * kmax + tid] : -1;
    }
    __syncthreads();
    const T* Np = n_in_smem ? Ns : (const T*)st.pend_N + (size_t)w * kmax * n;
    const T* Tw = (const T*)st.Ti + (size_t)w * n * n;
    const int j_beg = tile * rows_per_tile, j_end = min(n, j_beg + rows_per_tile);
    for (int j0 = j_beg + warp * RW; j0 < j_end; j0 += nw * RW) {
      T d[RW][KT];
#pragma unroll
      for (int r = 0; r < RW; ++r)
#pragma unroll
        for (int a = 0; a < KT; ++a) d[r][a] = S::zero();
      constexpr int U = sizeof(T) == 16 ? 8 : 4;   // 16-byte loads in flight per thread = U * RW
      for (int q0 = lane; q0 < nvec; q0 += 32 * U) {
        V x[U][RW];
#pragma unroll
        for (int u = 0; u < U; ++u) {
          const int q = q0 + 32 * u;
#pragma unroll
          for (int r = 0; r < RW; ++r) {
            if (q < nvec && j0 + r < j_end) x[u][r] = ((const V*)(Tw + (size_t)(j0 + r) * n))[q];
            else { RV::set(x[u][r], 0, S::zero()); if (VEC == 2) RV::set(x[u][r], 1, S::zero()); }
          }
        }
#pragma unroll
        for (int u = 0; u < U; ++u) {
          const int q = q0 + 32 * u;
          if (q < nvec) {
#pragma unroll
            for (int a = 0; a < KT; ++a) {
              if (a < k) {
                const V nv = ((const V*)(Np + (size_t)a * n))[q];
#pragma unroll
                for (int e = 0; e < VEC; ++e)
#pragma unroll
                  for (int r = 0; r < RW; ++r)
                    d[r][a] = S::fma(RV::get(x[u][r], e), RV::get(nv, e), d[r][a]);
              }
            }
          }
        }
      }
#pragma unroll
      for (int r = 0; r < RW; ++r)
#pragma unroll
        for (int a = 0; a < KT; ++a) {
          T v = warp_sum(d[r][a]);
          if (j0 + r == sidx[a]) v = S::sub(v, S::one());
          if (lane == 0 && j0 + r < j_end) dsm[a * rows_per_tile + (j0 + r - j_beg)] = v;
        }
    }
    append_finish<T, KT>(st, w, k, fill, j_beg, j_end, rows_per_tile, dsm, Ri);
  }
}

// The same dot products for complex128 with k <= 4 on the FP64 tensor pipe.  The k dot products
// per row are an (rows x n)(n x k) contraction: per warp, 8 rows x 4 columns of Ti form the A
// fragment of mma.sync.m8n8k4.f64 straight from the global loads (lane = (row, column): one
// 16-byte complex element, both halves used), and the 8 real columns [Re N | Im N] the B
// fragment, so that  A=Re Ti, B=[Re N | Im N]  and  A=Im Ti, B'=[-Im N | Re N]  accumulate
// [Re W | Im W] in two DMMAs per 8x4 complex elements.  Against the scalar pass: 2 tensor
// instructions instead of 32 DFMAs + shuffles, 4 accumulator registers per lane instead of
// 32, which leaves room for 16 loads of 16 bytes in flight per lane.
__device__ __forceinline__ void dmma884_acc(double& d0, double& d1, double a, double b) {
  asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
               : "+d"(d0), "+d"(d1)
               : "d"(a), "d"(b));
}

// The complex k <= 4 dot-product pass as a PURE STREAM.  Both contractions of the append have
// the same shape -- rows of a matrix against the k new rows N:
//     D[a][j]  = sum_i N[a][i] Ti[j][i] - [j == P_a]      (N A0^-1 - I[P,:], j < n)
//     NA[a][s] = sum_i N[a][i] Abuf[s][i]                 (N Abuf^T of Eq. 15, s < fill)
// so one kernel streams the n rows of Ti AND the fill rows of Abuf of every accepted walker
// (det_prep_kernel is not launched on this path).  D goes to the rows Bbuf[fill .. fill+k) that
// b_tau will occupy (free space), NA to pend_Y; det_append_finish_kernel then copies a_tau and
// does Eq. 15, so this kernel has no per-tile phases and no CTA barrier except when its range
// crosses into the next walker ([Re N | Im N] restaged).  Work is split in 16-row units, the
// ceil(cap/16) buffer units of a walker interleaved evenly among its ceil(n/16) inverse units
// (Bresenham), so that every contiguous range holds its share of both: CTA b takes units
// [total b / G, total (b+1) / G) of the concatenated accepted list -- with ~150 accepted
// walkers of 72 units over 296 CTAs that is 36.5 units each instead of 4 or 5 whole 128-row
// tiles (a 25 % tail) -- and warp (u - first) mod 8 takes unit u.
__global__ void __launch_bounds__(256, 2) det_append_dmma_stream_kernel(State st, int k) {
  using T = cplx;
  using S = Sc<T>;
  constexpr int UN = 8, MT = 2;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const int n = st.n, kmax = st.kmax, cap = st.cap;
  double* Bs = (double*)smem_raw;                // [n][8]  Re N (cols 0-3), Im N (cols 4-7)
  __shared__ int sidx[4];
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31, nw = blockDim.x >> 5;
  const int r8 = lane >> 2, kk = lane & 3;
  const int count = st.counters[0];
  const int upt = (n + 15) >> 4, upa = (cap + 15) >> 4, upw = upt + upa;
  const int64_t total = (int64_t)count * upw;
  const int64_t first = total * blockIdx.x / gridDim.x, last = total * (blockIdx.x + 1) / gridDim.x;
  for (int64_t u = first; u < last;) {
    const int wi = (int)(u / upw);
    const int w = st.list[wi];
    const int fill = st.fill[w];
    const int64_t seg_end = min(last, (int64_t)(wi + 1) * upw);
    __syncthreads();
    {
      const T* gN = (const T*)st.pend_N + (size_t)w * kmax * n;
      for (int q = tid; q < 4 * n; q += blockDim.x) {
        const int a = q / n, i = q % n;
        const T v = a < k ? gN[(size_t)a * n + i] : S::zero();
        Bs[i * 8 + a] = v.re;
        Bs[i * 8 + 4 + a] = v.im;
      }
      if (tid < 4) sidx[tid] = tid < k ? st.pend_idx[(size_t)w * kmax + tid] : -1;
    }
    __syncthreads();
    const int64_t u_mine = u + ((warp - (int)((u - first) % nw)) + nw) % nw;
    for (int64_t uu = u_mine; uu < seg_end; uu += nw) {
      const int ul = (int)(uu - (int64_t)wi * upw);          // unit within the walker
      const int a_before = (int)((int64_t)ul * upa / upw);
      const bool is_a = (int)((int64_t)(ul + 1) * upa / upw) > a_before;
      const int j0 = (is_a ? a_before : ul - a_before) * 16;
      const int rlim = is_a ? fill : n;                     // valid rows of this matrix
      if (j0 >= rlim) continue;                              // buffer unit past the fill
      const T* X = is_a ? (const T*)st.Abuf + (size_t)w * cap * n : (const T*)st.Ti + (size_t)w * n * n;
      double acc[2][2] = {{0.0, 0.0}, {0.0, 0.0}};
      const T* row0 = X + (size_t)min(j0 + r8, rlim - 1) * n + kk;         // rows past the end: clamped, discarded
      const T* row1 = X + (size_t)min(j0 + 8 + r8, rlim - 1) * n + kk;
      const double* bp = Bs + kk * 8 + r8;
      const double* bq = Bs + kk * 8 + (r8 ^ 4);
      const bool lo = r8 < 4;
      for (int i0 = 0; i0 < n; i0 += 4 * UN) {
        T x0[UN], x1[UN];
#pragma unroll
        for (int v = 0; v < UN; ++v) {
          const bool in = i0 + 4 * v < n;
          x0[v] = in ? row0[i0 + 4 * v] : S::zero();
          x1[v] = in ? row1[i0 + 4 * v] : S::zero();
        }
#pragma unroll
        for (int v = 0; v < UN; ++v) {
          if (i0 + 4 * v < n) {
            const double b = bp[(i0 + 4 * v) * 8];
            const double b2 = bq[(i0 + 4 * v) * 8];
            const double bm = lo ? -b2 : b2;          // B' = [-Im N | Re N]
            dmma884_acc(acc[0][0], acc[0][1], x0[v].re, b);
            dmma884_acc(acc[0][0], acc[0][1], x0[v].im, bm);
            dmma884_acc(acc[1][0], acc[1][1], x1[v].re, b);
            dmma884_acc(acc[1][0], acc[1][1], x1[v].im, bm);
          }
        }
      }
      // D fragment: row r8, columns 2*kk, 2*kk+1 of [Re | Im]
      T* outD = (T*)st.Bbuf + ((size_t)w * cap + fill) * n;                // [a][j], row stride n
      T* outNA = (T*)st.pend_Y + (size_t)w * kmax * cap;                   // [a][s], row stride cap
#pragma unroll
      for (int mt = 0; mt < MT; ++mt) {
        const int j = j0 + 8 * mt + r8;
#pragma unroll
        for (int e = 0; e < 2; ++e) {
          const int col = 2 * kk + e, a = col & 3;
          if (j < rlim && a < k) {
            double v = acc[mt][e];
            if (is_a) {
              ((double*)&outNA[(size_t)a * cap + j])[col >> 2] = v;
            } else {
              if (col < 4 && j == sidx[a]) v -= 1.0;
              ((double*)&outD[(size_t)a * n + j])[col >> 2] = v;
            }
          }
        }
      }
    }
    u = seg_end;
  }
}

// The same stream for float64 and every k <= 8.  Lane (r, q) loads the 16-byte pair
// X[j0+r][i0+2q, i0+2q+1] of its row and the same pair of N[a = r][.] from shared memory
// (permuted contraction index, as in lrux_rowdot.cu) and issues two DMMAs into two independent
// accumulator chains; D fragment = (row j0+r, a = 2q, 2q+1).  KS = rows of N kept in shared
// memory (4 for k <= 4, else 8: lanes with r >= KS contribute zeros), row stride 8 mod 16
// doubles: conflict-free.  Replaces det_prep_kernel + det_append_kernel and det_prep_kernel +
// rowdot_dmma_kernel on this path: no per-tile phases, balanced 16-row units, N Abuf^T folded in.
// Measured (append class, fraction of HBM for n^2 e per accepted walker, Metropolis): n=512 K=8:
// k=4 0.76 (was 0.62), k=8 0.65 (0.56); K=32: n=512 k=4 0.62 (0.45), n=1024 k=4 0.74 (0.61),
// k=8 0.64 (0.52), n=2048 k=4 0.81 (0.71); k=1: 0.95-0.98 (0.94-0.96).
// PW (small n: eight copies of N fit in shared memory): every WARP owns a contiguous range of
// units and its own copy of N -- no CTA barrier at all.  With one shared copy a walker of 18 units
// (n = 256) keeps the 8 warps busy for 2 or 3 units each between two barriers: 75 % at best.
template <int KS, bool PW>
__global__ void __launch_bounds__(256, 2) det_append_stream_real_kernel(State st, int k, int ldn) {
  constexpr int UN = 8, MT = 2;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const int n = st.n, kmax = st.kmax, cap = st.cap;
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31, nw = blockDim.x >> 5;
  double* Ns = (double*)smem_raw + (PW ? (size_t)warp * KS * ldn : 0);   // [KS][ldn] (per warp when PW)
  __shared__ int sidx_s[PW ? 8 : 1][8];
  int* sidx = sidx_s[PW ? warp : 0];
  const int r8 = lane >> 2, q = lane & 3;
  const int count = st.counters[0];
  const int upt = (n + 15) >> 4, upa = (cap + 15) >> 4, upw = upt + upa;
  const int64_t total = (int64_t)count * upw;
  const int64_t me = PW ? (int64_t)blockIdx.x * nw + warp : blockIdx.x, parts = PW ? (int64_t)gridDim.x * nw : gridDim.x;
  const int64_t first = total * me / parts, last = total * (me + 1) / parts;
  for (int64_t u = first; u < last;) {
    const int wi = (int)(u / upw);
    const int w = st.list[wi];
    const int fill = st.fill[w];
    const int64_t seg_end = min(last, (int64_t)(wi + 1) * upw);
    if (PW) __syncwarp(); else __syncthreads();
    {
      const double* gN = (const double*)st.pend_N + (size_t)w * kmax * n;
      for (int qd = PW ? lane : tid; qd < KS * (n >> 1); qd += PW ? 32 : blockDim.x) {
        const int a = qd / (n >> 1), i = 2 * (qd % (n >> 1));
        *(double2*)(Ns + (size_t)a * ldn + i) = a < k ? *(const double2*)(gN + (size_t)a * n + i) : make_double2(0.0, 0.0);
      }
      if ((PW ? lane : tid) < 8) sidx[PW ? lane : tid] = (PW ? lane : tid) < k ? st.pend_idx[(size_t)w * kmax + (PW ? lane : tid)] : -1;
    }
    if (PW) __syncwarp(); else __syncthreads();
    const int64_t u_mine = PW ? u : u + ((warp - (int)((u - first) % nw)) + nw) % nw;
    for (int64_t uu = u_mine; uu < seg_end; uu += PW ? 1 : nw) {
      const int ul = (int)(uu - (int64_t)wi * upw);          // unit within the walker
      const int a_before = (int)((int64_t)ul * upa / upw);
      const bool is_a = (int)((int64_t)(ul + 1) * upa / upw) > a_before;
      const int j0 = (is_a ? a_before : ul - a_before) * 16;
      const int rlim = is_a ? fill : n;                     // valid rows of this matrix
      if (j0 >= rlim) continue;                              // buffer unit past the fill
      const double* X = is_a ? (const double*)st.Abuf + (size_t)w * cap * n : (const double*)st.Ti + (size_t)w * n * n;
      double acc[MT][2][2] = {};
      const double* row0 = X + (size_t)min(j0 + r8, rlim - 1) * n + 2 * q;       // rows past the end: clamped, discarded
      const double* row1 = X + (size_t)min(j0 + 8 + r8, rlim - 1) * n + 2 * q;
      const double* bp = Ns + (size_t)(r8 < KS ? r8 : 0) * ldn + 2 * q;
      const bool bz = r8 >= KS;
      for (int i0 = 0; i0 < n; i0 += 8 * UN) {
        double2 x0[UN], x1[UN];
#pragma unroll
        for (int v = 0; v < UN; ++v) {
          const bool in = i0 + 8 * v + 2 * q < n;
          x0[v] = in ? *(const double2*)(row0 + i0 + 8 * v) : make_double2(0.0, 0.0);
          x1[v] = in ? *(const double2*)(row1 + i0 + 8 * v) : make_double2(0.0, 0.0);
        }
#pragma unroll
        for (int v = 0; v < UN; ++v) {
          if (i0 + 8 * v < n) {
            double2 b = (i0 + 8 * v + 2 * q < n) ? *(const double2*)(bp + i0 + 8 * v) : make_double2(0.0, 0.0);
            if (bz) b = make_double2(0.0, 0.0);
            dmma884_acc(acc[0][0][0], acc[0][0][1], x0[v].x, b.x);
            dmma884_acc(acc[0][1][0], acc[0][1][1], x0[v].y, b.y);
            dmma884_acc(acc[1][0][0], acc[1][0][1], x1[v].x, b.x);
            dmma884_acc(acc[1][1][0], acc[1][1][1], x1[v].y, b.y);
          }
        }
      }
      double* outD = (double*)st.Bbuf + ((size_t)w * cap + fill) * n;          // [a][j], row stride n
      double* outNA = (double*)st.pend_Y + (size_t)w * kmax * cap;             // [a][s], row stride cap
#pragma unroll
      for (int mt = 0; mt < MT; ++mt) {
        const int j = j0 + 8 * mt + r8;
#pragma unroll
        for (int e = 0; e < 2; ++e) {
          const int a = 2 * q + e;
          if (j < rlim && a < k) {
            double v = acc[mt][0][e] + acc[mt][1][e];
            if (is_a) {
              outNA[(size_t)a * cap + j] = v;
            } else {
              if (j == sidx[a]) v -= 1.0;
              outD[(size_t)a * n + j] = v;
            }
          }
        }
      }
    }
    u = seg_end;
  }
}

// Second half of the append as its own pass, for the tensor-pipe variant below: D = N A0^-1 -
// I[P,:] is already in the pending area (pend_C, free once det_prep_kernel has copied a_tau
// into the buffer).  b_tau^T = R^-1 (D - (N Abuf) Bbuf^T) -> Bbuf[fill .. fill+k)   (Eq. 15,
// PAPER.md:194; reading 5b).  Work item = (accepted walker, 64 columns); four groups of
// threads split the buffer rows (the loop over them is a chain of dependent loads) and meet in
// shared memory, summed in a fixed order.
// inplace = 1 (after det_append_dmma_stream_kernel, which ran without det_prep_kernel): D is
// read from the rows Bbuf[fill .. fill+k) it is about to overwrite (each thread reads its k
// values before it writes any), and a_tau = C_eff is copied into Abuf[fill .. fill+k) here.
template <typename T, int KT>
__global__ void __launch_bounds__(256) det_append_finish_kernel(State st, int k, int chunks, int inplace) {
  using S = Sc<T>;
  constexpr int CW = 64, SG = 4;               // columns per work item, groups that split the buffer rows
  extern __shared__ __align__(16) unsigned char smem_raw[];
  T* NAs = (T*)smem_raw;                       // [fill][KT]
  T* red = NAs + (size_t)st.cap * KT;          // [SG-1][KT][CW] partial sums of groups 1..SG-1
  __shared__ T Ri[KT * KT];
  const int n = st.n, kmax = st.kmax, cap = st.cap;
  const int tid = threadIdx.x, jj = tid & (CW - 1), sg = tid / CW;
  const int count = st.counters[0];
  for (int item = blockIdx.x; item < count * chunks; item += gridDim.x) {
    const int w = st.list[item / chunks];
    const int j = (item % chunks) * CW + jj;
    const int fill = st.fill[w];
    __syncthreads();
    const T* NA = (const T*)st.pend_Y + (size_t)w * kmax * cap;
    for (int q = tid; q < fill * KT; q += 256)
      NAs[q] = (q % KT) < k ? NA[(size_t)(q % KT) * cap + q / KT] : S::zero();
    if (tid < KT * KT) {
      const int a = tid / KT, b = tid % KT;
      Ri[tid] = (a < k && b < k) ? ((const T*)st.pend_Rinv)[(size_t)w * st.kc * st.kc + a * st.kc + b]
                                 : S::zero();
    }
    __syncthreads();
    T* Bb = (T*)st.Bbuf + (size_t)w * cap * n;
    const T* pC = (const T*)st.pend_C + (size_t)w * kmax * n;
    const T* D = inplace ? Bb + (size_t)fill * n : pC;
    T m[KT];
#pragma unroll
    for (int b = 0; b < KT; ++b) m[b] = (sg == 0 && b < k && j < n) ? D[(size_t)b * n + j] : S::zero();
    if (inplace && sg == 1 && j < n) {
      T* Ab = (T*)st.Abuf + ((size_t)w * cap + fill) * n;
#pragma unroll
      for (int b = 0; b < KT; ++b)
        if (b < k) Ab[(size_t)b * n + j] = pC[(size_t)b * n + j];
    }
    if (j < n) {
#pragma unroll 8
      for (int s = sg; s < fill; s += SG) {
        const T bv = Bb[(size_t)s * n + j];
#pragma unroll
        for (int b = 0; b < KT; ++b) m[b] = S::fnma(NAs[s * KT + b], bv, m[b]);
      }
    }
    if (sg > 0) {
#pragma unroll
      for (int b = 0; b < KT; ++b) red[((size_t)(sg - 1) * KT + b) * CW + jj] = m[b];
    }
    __syncthreads();
    if (sg == 0 && j < n) {
#pragma unroll
      for (int b = 0; b < KT; ++b)
#pragma unroll
        for (int g = 0; g < SG - 1; ++g) m[b] = S::add(m[b], red[((size_t)g * KT + b) * CW + jj]);
#pragma unroll
      for (int a = 0; a < KT; ++a) {
        if (a < k) {
          T acc = S::zero();
#pragma unroll
          for (int b = 0; b < KT; ++b) acc = S::fma(Ri[a * KT + b], m[b], acc);
          Bb[(size_t)(fill + a) * n + j] = acc;
        }
      }
    }
  }
}

// post: fill += k for accepted walkers; walkers whose depth reached K (or whose
// buffer cannot take another kmax columns) go to the flush list (reading 9).
__global__ void post_kernel(State st, int k) {
  const int it = blockIdx.x * blockDim.x + threadIdx.x;
  if (it >= st.counters[0]) return;
  const int w = st.list[it];
  const int f = st.fill[w] + k, u = st.nupd[w] + 1;
  st.fill[w] = f;
  st.nupd[w] = u;
  if (u >= st.K || f + st.kc > st.cap) st.flist[atomicAdd(&st.counters[1], 1)] = w;
}

// flush-all selection: every walker with a non-empty buffer.
__global__ void flush_all_select_kernel(State st) {
  const int64_t w = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (w >= st.W) return;
  if (st.fill[w] > 0) st.flist[atomicAdd(&st.counters[1], 1)] = (int32_t)w;
}
__global__ void reset_counter_kernel(State st, int which) { st.counters[which] = 0; }

__global__ void flush_clear_kernel(State st) {
  const int it = blockIdx.x * blockDim.x + threadIdx.x;
  if (it >= st.counters[1]) return;
  const int w = st.flist[it];
  // running totals for lrux_*_get_flush_count: [walker flushes, buffer columns folded]
  unsigned long long* tot = (unsigned long long*)(st.counters + 4);
  atomicAdd(&tot[0], 1ULL);
  atomicAdd(&tot[1], (unsigned long long)st.fill[w]);
  st.fill[w] = 0;
  st.nupd[w] = 0;
}

// ---------------------------------------------------------------- shared helpers
int launch_select(const State& st, const uint8_t* mask, cudaStream_t s) {
  const unsigned gw = (unsigned)((st.W + 255) / 256);
  if (st.dt == LRUX_F64) select_kernel<double><<<gw, 256, 0, s>>>(st, mask);
  else select_kernel<cplx><<<gw, 256, 0, s>>>(st, mask);
  return 1;
}
int launch_post(const State& st, int ncols, cudaStream_t s) {
  post_kernel<<<(unsigned)((st.W + 255) / 256), 256, 0, s>>>(st, ncols);
  return 1;
}
int launch_flush_select_all(const State& st, cudaStream_t s) {
  reset_counter_kernel<<<1, 1, 0, s>>>(st, 1);
  flush_all_select_kernel<<<(unsigned)((st.W + 255) / 256), 256, 0, s>>>(st);
  return 2;
}
int launch_flush_clear(const State& st, cudaStream_t s) {
  flush_clear_kernel<<<(unsigned)((st.W + 255) / 256), 256, 0, s>>>(st);
  return 1;
}

// ---------------------------------------------------------------- launchers
// Every choice below depends on the shape (dtype, n, k, K) only.
template <typename T, int KT, int VEC, int CH, int RW>
static int launch_update_reg(const State& st, int k, Ctx& cx, cudaStream_t s) {
  const int n = st.n;
  const size_t smem = 2 * (size_t)k * n * sizeof(T);
  auto kern = det_update_kernel<T, KT, VEC, CH, RW>;
  const int occ = cx.configure((const void*)kern, 256, smem);
  if (occ < 0) return -1;
  int rows_per_tile = 64;
  if (rows_per_tile > n) rows_per_tile = n;
  const int tiles = (n + rows_per_tile - 1) / rows_per_tile;
  const int grid = persistent_grid(cx.num_sms, occ, (int64_t)st.W * tiles);
  kern<<<grid, 256, smem, s>>>(st, k, tiles, rows_per_tile);
  cx.name(LRUX_PROF_UPDATE, "det_update_kernel");
  return 1;
}

template <typename T, int KT>
static int launch_update_kt(const State& st, int k, Ctx& cx, cudaStream_t s) {
  const int n = st.n;
  constexpr int VECMAX = sizeof(T) == 8 ? 2 : 1;
  if constexpr (sizeof(T) == 8 && KT >= LRUX_DMMA_MIN_KT) {
    // real data, k >= 3: 8-row strips on the FP64 tensor pipe (lrux_det_dmma.cu) -- the scalar
    // kernels below are bound by their operand traffic from k = 4 on.  Measured exception
    // (profiles/r02_sweep.md): k = 3, 4 at 1024 < n <= 2048, where the strips are split over a
    // 2-CTA cluster (0.73 of HBM) and the TMA-staged kernel still has a rank-4 instance (0.81-0.84).
    const bool tma_better = KT == 4 && n > 1024 && n <= 2048 && launch_det_update_tma(st, k, cx, s, true) == 1;
    if (!tma_better) {
      const int r = launch_det_update_dmma(st, k, cx, s);
      if (r != 0) return r;
    }
  }
  if ((size_t)n * sizeof(T) >= 8 * 1024) {
    // rows of >= 8 KB: TMA-staged kernel (lrux_det_tma.cu)
    const int r = launch_det_update_tma(st, k, cx, s);
    if (r != 0) return r;
    // no instance for the full rank (register budget): peel off chunks of the largest
    // rank that has one; each chunk is one full pass over A^-1
    int c = 0;
    for (int cand = 4; cand >= 1; cand >>= 1)
      if (cand < k && launch_det_update_tma(st, cand, cx, s, /*probe=*/true) == 1) { c = cand; break; }
    if (c > 0) {
      int nl = 0, rem = k;
      State v = st;   // view of the pending area, shifted past the chunks already applied
      const size_t e = sizeof(T);
      while (rem > 0) {
        const int cur = rem > c ? c : rem;
        if (rem > cur) {
          det_split_prep_kernel<T><<<persistent_grid(cx.num_sms, 4, st.W), 256, 0, s>>>(v, cur, rem);
          ++nl;
        }
        const int r2 = launch_det_update_tma(v, cur, cx, s);
        if (r2 <= 0) return -1;
        nl += r2;
        v.pend_idx += cur;
        v.pend_N = (char*)v.pend_N + (size_t)cur * n * e;
        v.pend_C = (char*)v.pend_C + (size_t)cur * n * e;
        v.pend_Rinv = (char*)v.pend_Rinv + ((size_t)cur * st.kc + cur) * e;
        rem -= cur;
      }
      return nl;
    }
  }
  const size_t smem = 2 * (size_t)k * n * sizeof(T);
  const bool vec_ok = (n % VECMAX) == 0;
  const int nvec = n / VECMAX;
  if (vec_ok && smem <= 160 * 1024) {
    if (nvec <= 32 * 1) return launch_update_reg<T, KT, VECMAX, 1, 2>(st, k, cx, s);
    if (nvec <= 32 * 2) return launch_update_reg<T, KT, VECMAX, 2, 2>(st, k, cx, s);
    if (nvec <= 32 * 4) return launch_update_reg<T, KT, VECMAX, 4, 2>(st, k, cx, s);
    if (nvec <= 32 * 8) return launch_update_reg<T, KT, VECMAX, 8, 1>(st, k, cx, s);
    if (nvec <= 32 * 16) return launch_update_reg<T, KT, VECMAX, 16, 1>(st, k, cx, s);
  }
  int rows_per_tile = 64;
  if (rows_per_tile > n) rows_per_tile = n;
  const int tiles = (n + rows_per_tile - 1) / rows_per_tile;
  const int grid = persistent_grid(cx.num_sms, 4, (int64_t)st.W * tiles);
  det_update_stream_kernel<T, KT><<<grid, 256, 0, s>>>(st, k, tiles, rows_per_tile);
  cx.name(LRUX_PROF_UPDATE, "det_update_stream_kernel");
  return 1;
}

template <typename T, int KT>
static int launch_append_kt(const State& st, int k, Ctx& cx, cudaStream_t s) {
  const int n = st.n;
  constexpr int VECMAX = sizeof(T) == 8 ? 2 : 1;
  if constexpr (sizeof(T) == 16 && KT <= 4) {
    // complex data, k <= 4: the dot products as a pure stream on the FP64 tensor pipe, Eq. 15 in a second pass
    if (n % 4 == 0 && n >= 1024 && (size_t)n * 64 <= 100 * 1024) {
      const size_t sms = (size_t)n * 64;
      const int occs = cx.configure((const void*)det_append_dmma_stream_kernel, 256, sms);
      if (occs < 0) return -1;
      det_append_dmma_stream_kernel<<<persistent_grid(cx.num_sms, occs, (int64_t)st.W * ((n + 15) / 16)), 256, sms, s>>>(st, k);
      const int chunks = (n + 63) / 64;
      const size_t smf = ((size_t)st.cap * KT + 3 * KT * 64) * sizeof(T);
      auto kf = det_append_finish_kernel<T, KT>;
      if (cx.configure((const void*)kf, 256, smf) < 0) return -1;
      kf<<<persistent_grid(cx.num_sms, 8, (int64_t)st.W * chunks), 256, smf, s>>>(st, k, chunks, 1);
      cx.name(LRUX_PROF_APPEND, "det_append_dmma_stream_kernel+det_append_finish_kernel");
      return 2;
    }
  }
  if constexpr (sizeof(T) == 8) {
    // real data, even n: the same stream for every k <= 8
    const int ks = k <= 4 ? 4 : 8;
    const int ldn = ((n + 15) & ~15) + 8;
    const bool pw = (size_t)8 * ks * ldn * sizeof(double) <= LRUX_APPEND_PW_SMEM_KB * 1024;   // a copy of N per warp
    const size_t sms = (size_t)(pw ? 8 : 1) * ks * ldn * sizeof(double);
    // (k <= 2 at 128 < n < 512 -- configs[1] with a delay -- stays on the register-row pass: 0.57-0.61 of HBM
    // against 0.56-0.58 for the stream)
    if ((n & 1) == 0 && (n >= 512 || n <= 128 || k >= 3) && k >= LRUX_APPEND_REAL_STREAM_MIN_K && sms <= 200 * 1024) {
      auto ksr = pw ? (ks == 4 ? det_append_stream_real_kernel<4, true> : det_append_stream_real_kernel<8, true>)
                    : (ks == 4 ? det_append_stream_real_kernel<4, false> : det_append_stream_real_kernel<8, false>);
      const int occs = cx.configure((const void*)ksr, 256, sms);
      if (occs < 0) return -1;
      ksr<<<persistent_grid(cx.num_sms, occs, (int64_t)st.W * ((n + 15) / 16)), 256, sms, s>>>(st, k, ldn);
      const int chunks = (n + 63) / 64;
      const size_t smf = ((size_t)st.cap * KT + 3 * KT * 64) * sizeof(T);
      auto kf = det_append_finish_kernel<T, KT>;
      if (cx.configure((const void*)kf, 256, smf) < 0) return -1;
      kf<<<persistent_grid(cx.num_sms, 8, (int64_t)st.W * chunks), 256, smf, s>>>(st, k, chunks, 1);
      cx.name(LRUX_PROF_APPEND, "det_append_stream_real_kernel+det_append_finish_kernel");
      return 2;
    }
  }
  int nl = 0;
  {
    const int groups = (st.cap + 8 * kPrepRows - 1) / (8 * kPrepRows);
    const int grid = persistent_grid(cx.num_sms, 8, (int64_t)st.W * groups);
    det_prep_kernel<T, KT><<<grid, 256, 0, s>>>(st, k, groups); ++nl;
  }
  // (... and whenever N does not fit beside the register-row pass in shared memory: k n e > 96 KB)
  if (sizeof(T) == 8 && (KT >= LRUX_APPEND_ROWDOT_MIN_KT || (size_t)k * n * sizeof(T) > 96 * 1024)) {
    // real data, k >= 5: the k dot products per row on the FP64 tensor pipe (one read-only pass,
    // lrux_rowdot.cu), then the buffer terms and R^-1 in a pass over the k x n result (measured
    // at n = 1024, K = 32: k = 8 0.46 of HBM against 0.40 for the register-row pass, k = 4
    // 0.63 against 0.67 -- so k <= 4 stays on the register-row pass)
    if ((n & 1) == 0) {
      RowdotArgs A{};
      A.X = (const double*)st.Ti;      A.x_stride = (size_t)n * n;          A.rows = n;  A.ldx = n;
      A.N = (const double*)st.pend_N;  A.n_stride = (size_t)st.kmax * n;   A.ldn = n;
      A.n = n;  A.k = k;
      A.out = (double*)st.pend_C;      A.o_stride = (size_t)st.kmax * n;   A.ldo = n;
      A.list = st.list;  A.count = st.counters;  A.W = st.W;
      A.idx = st.pend_idx;  A.idx_stride = st.kmax;
      const int r = launch_rowdot_dmma(A, cx, s);
      if (r < 0) return -1;
      if (r > 0) {
        const int chunks = (n + 63) / 64;
        const size_t smf = ((size_t)st.cap * KT + 3 * KT * 64) * sizeof(T);
        auto kf = det_append_finish_kernel<T, KT>;
        if (cx.configure((const void*)kf, 256, smf) < 0) return -1;
        kf<<<persistent_grid(cx.num_sms, 8, (int64_t)st.W * chunks), 256, smf, s>>>(st, k, chunks, 0);
        cx.name(LRUX_PROF_APPEND, "det_prep_kernel+rowdot_dmma_kernel+det_append_finish_kernel");
        return nl + r + 1;
      }
    }
  }
  const int rows_per_tile = LRUX_APPEND_TILE_ROWS;   // must divide the block size (256)
  const int tiles = (n + rows_per_tile - 1) / rows_per_tile;
  const int n_in_smem = (size_t)k * n * sizeof(T) <= 96 * 1024;
  const size_t smem = ((n_in_smem ? (size_t)k * n : 0) + 4 * (size_t)KT * rows_per_tile) * sizeof(T);
  const bool vec = (n % VECMAX) == 0 && VECMAX == 2;
  auto kern = vec ? det_append_kernel<T, KT, VECMAX, 2> : det_append_kernel<T, KT, 1, 2>;
  const int occ = cx.configure((const void*)kern, 256, smem);
  if (occ < 0) return -1;
  const int grid = persistent_grid(cx.num_sms, occ, (int64_t)st.W * tiles);
  kern<<<grid, 256, smem, s>>>(st, k, tiles, rows_per_tile, n_in_smem);
  cx.name(LRUX_PROF_APPEND, "det_prep_kernel+det_append_kernel");
  return nl + 1;
}

template <typename T>
static int flush_impl(const State& st, bool all, Ctx& cx, cudaStream_t s) {
  int nl = 0;
  const unsigned gw = (unsigned)((st.W + 255) / 256);
  if (all) {
    reset_counter_kernel<<<1, 1, 0, s>>>(st, 1); ++nl;
    flush_all_select_kernel<<<gw, 256, 0, s>>>(st); ++nl;
  }
  {
    ProfScope ps(&cx.prof, LRUX_PROF_FLUSH, s);
    nl += launch_flush_dmma(st, cx, s);   // Eq. 12 on the FP64 tensor path
  }
  flush_clear_kernel<<<gw, 256, 0, s>>>(st); ++nl;
  return cudaGetLastError() == cudaSuccess ? nl : -1;
}

template <typename T>
static int accept_impl(const State& st, int k, const uint8_t* mask, Ctx& cx, cudaStream_t s) {
  int nl = 0;
  const unsigned gw = (unsigned)((st.W + 255) / 256);
  select_kernel<T><<<gw, 256, 0, s>>>(st, mask); ++nl;
  const int kt = round_kt(k);
  int r = 0;
  if (st.K == 0) {
    ProfScope ps(&cx.prof, LRUX_PROF_UPDATE, s);
    switch (kt) {
      case 1: r = launch_update_kt<T, 1>(st, k, cx, s); break;
      case 2: r = launch_update_kt<T, 2>(st, k, cx, s); break;
      case 4: r = launch_update_kt<T, 4>(st, k, cx, s); break;
      default: r = launch_update_kt<T, 8>(st, k, cx, s); break;
    }
    if (r < 0) return -1;
    nl += r;
  } else {
    {
      ProfScope ps(&cx.prof, LRUX_PROF_APPEND, s);
      switch (kt) {
        case 1: r = launch_append_kt<T, 1>(st, k, cx, s); break;
        case 2: r = launch_append_kt<T, 2>(st, k, cx, s); break;
        case 4: r = launch_append_kt<T, 4>(st, k, cx, s); break;
        default: r = launch_append_kt<T, 8>(st, k, cx, s); break;
      }
    }
    if (r < 0) return -1;
    nl += r;
    post_kernel<<<gw, 256, 0, s>>>(st, k); ++nl;
    r = flush_impl<T>(st, false, cx, s);
    if (r < 0) return -1;
    nl += r;
  }
  return cudaGetLastError() == cudaSuccess ? nl : -1;
}

template <typename T, int KT>
static int launch_ratio_kt(const State& st, int k, const int32_t* d_idx, const void* d_rows,
                           void* d_ratio, Ctx& cx, cudaStream_t s) {
  // one CTA per 256-column slice: 128 threads x 2 elements (n <= 256: a single slice,
  // 1 element per thread when n <= 128), else 256 threads x 1 element
  const int n = st.n;
#if LRUX_RATIO_WARP
  // one warp per walker, 8 walkers per CTA: k <= 4 without a delay buffer, k <= 2 with one (measured at
  // n = 64 / 128, ratio time per step: k=1 0.38x / 0.49x, k=4 0.49x / 0.66x of the CTA kernel's; k=8 0.76x /
  // 0.93x -- not worth a second arithmetic order --; with K = 8: k=1 0.49x, k=4 1.29x)
  if ((n <= 128 && KT <= 4 && (st.cap == 0 || KT <= 2)) || (LRUX_RATIO_WARP >= 2 && n <= 256 && KT <= 2 && st.cap == 0)) {
    auto kw = n <= 32 ? det_ratio_warp_kernel<T, KT, 1> : n <= 64 ? det_ratio_warp_kernel<T, KT, 2>
            : n <= 128 ? det_ratio_warp_kernel<T, KT, 4> : det_ratio_warp_kernel<T, (KT <= 2 ? KT : 2), 8>;
    kw<<<(unsigned)((st.W + 7) / 8), 256, 0, s>>>(st, k, d_idx, (const T*)d_rows, (T*)d_ratio);
    return 1;
  }
#endif
  const int nsplit = (n + kRatioSlice - 1) / kRatioSlice;
  const dim3 grid((unsigned)st.W, (unsigned)nsplit);
  const size_t sm = (size_t)st.cap * KT * sizeof(T);   // <= kRatioCoefSmemMax (checked at init)
  auto kern = n <= 128 ? det_ratio_kernel<T, KT, 1> : n <= 256 ? det_ratio_kernel<T, KT, 2>
                                                               : det_ratio_kernel<T, KT, 1>;
  const int threads = n <= 256 ? 128 : 256;
  if (cx.configure((const void*)kern, threads, sm) < 0) return -1;
  kern<<<grid, threads, sm, s>>>(st, k, d_idx, (const T*)d_rows, (T*)d_ratio);
  return 1;
}

template <typename T>
static int launch_ratio_t(const State& st, int k, const int32_t* d_idx, const void* d_rows,
                          void* d_ratio, Ctx& cx, cudaStream_t s) {
  switch (round_kt(k)) {
    case 1: return launch_ratio_kt<T, 1>(st, k, d_idx, d_rows, d_ratio, cx, s);
    case 2: return launch_ratio_kt<T, 2>(st, k, d_idx, d_rows, d_ratio, cx, s);
    case 4: return launch_ratio_kt<T, 4>(st, k, d_idx, d_rows, d_ratio, cx, s);
    default: return launch_ratio_kt<T, 8>(st, k, d_idx, d_rows, d_ratio, cx, s);
  }
}

int launch_det_ratio(const State& st, int k, const int32_t* d_idx, const void* d_rows,
                     void* d_ratio, Ctx& cx, cudaStream_t s) {
  ProfScope ps(&cx.prof, LRUX_PROF_RATIO, s);
  cx.name(LRUX_PROF_RATIO, (LRUX_RATIO_WARP && ((st.n <= 128 && k <= 4 && (st.cap == 0 || k <= 2)) || (LRUX_RATIO_WARP >= 2 && st.n <= 256 && k <= 2 && st.cap == 0))) ? "det_ratio_warp_kernel" : "det_ratio_kernel");
  const int r = st.dt == LRUX_F64 ? launch_ratio_t<double>(st, k, d_idx, d_rows, d_ratio, cx, s)
                                  : launch_ratio_t<cplx>(st, k, d_idx, d_rows, d_ratio, cx, s);
  return (r > 0 && cudaGetLastError() == cudaSuccess) ? r : -1;
}

int launch_det_accept(const State& st, int k, const uint8_t* d_mask, Ctx& cx, cudaStream_t s) {
  return st.dt == LRUX_F64 ? accept_impl<double>(st, k, d_mask, cx, s)
                           : accept_impl<cplx>(st, k, d_mask, cx, s);
}

int launch_det_flush(const State& st, bool all, Ctx& cx, cudaStream_t s) {
  return st.dt == LRUX_F64 ? flush_impl<double>(st, all, cx, s) : flush_impl<cplx>(st, all, cx, s);
}

}  // namespace lrux
