// Pfaffian hot path.
//
// State Ti = A^-1 row-major, exactly skew.  New-rows-only forms (DESIGN.md §3,
// readings 5/5b), P the k replaced slots, N[a][:] the new row P[a] of A' (with
// N[a][P[a]] = 0), Aeff = A0^-1 + sum_s Bbuf[s][.] Abuf[s][.] the effective inverse:
//   C[a][i] = Aeff[i][P[a]]          Y[a][i] = sum_j Aeff[i][j] N[a][j]
//   R' = [[G, Tm], [-Tm^T, S]],  G[a][b] = N_a.Y_b + N[a][P[b]],  Tm[a][b] = N_a.C_b,
//        S[a][b] = Aeff[P[a]][P[b]]          (= J + u^T A^-1 u up to a congruence, Eq. 20)
//   r = (-1)^(k(k-1)/2) pf R'                                   (Eq. 19)
//   A'^-1 = Aeff + Y' R'^-1 Y'^T,  Y' = (Y + E_P, C)             (Eq. 21)
// R' is assembled from its strict upper triangle and mirrored, R'^-1 is skew
// projected, and the update writes the upper triangle and its exact negative, so
// the stored inverse stays exactly skew.
#include "lrux_common.cuh"
#include "lrux_internal.h"
#include "lrux_tma.cuh"
#include <cooperative_groups.h>
#include <algorithm>

#ifndef LRUX_PF_DMMA
#define LRUX_PF_DMMA 1
#endif
#ifndef LRUX_PF_Y_ROWDOT_MIN_K
#define LRUX_PF_Y_ROWDOT_MIN_K 3
#endif
#ifndef LRUX_PF_DMMA_MIN_K
#define LRUX_PF_DMMA_MIN_K 2
#endif

namespace lrux {

constexpr int kMaxC = 2 * kMaxK;  // largest core size

// ---------------------------------------------------------------- gather (+ ratio for k = 1)
template <typename T>
__global__ void __launch_bounds__(128)
pf_gather_kernel(State st, int k, const int32_t* __restrict__ idx, const T* __restrict__ rows,
                 T* __restrict__ ratio_out) {
  using S = Sc<T>;
  __shared__ int sidx[kMaxK];
  __shared__ int bad;
  __shared__ T red[4];
  const int w = blockIdx.x, tid = threadIdx.x, nt = blockDim.x;
  const int warp = tid >> 5, lane = tid & 31;
  const int n = st.n, kmax = st.kmax;
  if (w == 0 && tid == 0) st.counters[0] = 0;
  if (tid == 0) {
    int b = 0;
    for (int a = 0; a < k; ++a) {
      int p = idx[(size_t)w * k + a];
      sidx[a] = p;
      if (p < 0 || p >= n) b = 1;
      for (int c = 0; c < a; ++c)
        if (sidx[c] == p) b = 1;
    }
    bad = b;
  }
  __syncthreads();
  if (bad) {
    if (tid == 0) {
      ratio_out[w] = S::nan();
      ((T*)st.pend_ratio)[w] = S::nan();
      st.pend_ok[w] = 0;
      st.pend_idx[(size_t)w * kmax] = -1;
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
  T t1 = S::zero();
  for (int a = 0; a < k; ++a) {
    const int p = sidx[a];
    for (int i = tid; i < n; i += nt) {
      T c = S::neg(Tw[(size_t)p * n + i]);  // A0^-1[i][p] = -A0^-1[p][i]
      for (int s = 0; s < fill; ++s) c = S::fma(Bb[(size_t)s * n + i], Ab[(size_t)s * n + p], c);
      T x = (i == p) ? S::zero() : rows[((size_t)w * k + a) * n + i];
      pC[(size_t)a * n + i] = c;
      pN[(size_t)a * n + i] = x;
      if (k == 1) t1 = S::fma(x, c, t1);
    }
  }
  if (tid < k) st.pend_idx[(size_t)w * kmax + tid] = sidx[tid];
  if (k > 1) return;
  t1 = warp_sum(t1);
  if (lane == 0) red[warp] = t1;
  __syncthreads();
  if (tid == 0) {
    T t = red[0];
    for (int q = 1; q < (nt >> 5); ++q) t = S::add(t, red[q]);
    // k = 1: R' = [[0,t],[-t,0]], r = t; R'^-1 = [[0,-1/t],[1/t,0]]   (Eq. 22)
    ratio_out[w] = t;
    ((T*)st.pend_ratio)[w] = t;
    const bool ok = S::finite(t) && !S::is_zero(t);
    st.pend_ok[w] = ok ? 1 : 0;
    T* pR = (T*)st.pend_Rinv + (size_t)w * st.kc * st.kc;
    const T ti = ok ? S::inv(t) : S::zero();
    pR[0] = S::zero();
    pR[1] = S::neg(ti);
    pR[st.kc] = ti;
    pR[st.kc + 1] = S::zero();
  }
}

// ---------------------------------------------------------------- AN = N Abuf^T (delayed)
template <typename T>
__global__ void __launch_bounds__(256) pf_an_kernel(State st, int k, int use_list) {
  using S = Sc<T>;
  const int n = st.n, kmax = st.kmax, cap = st.cap;
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31, nw = blockDim.x >> 5;
  const int count = use_list ? st.counters[0] : (int)st.W;
  for (int it = blockIdx.x; it < count; it += gridDim.x) {
    const int w = use_list ? st.list[it] : it;
    if (st.pend_idx[(size_t)w * kmax] < 0) continue;
    const int fill = st.fill[w];
    const T* gN = (const T*)st.pend_N + (size_t)w * kmax * n;
    const T* Ab = (const T*)st.Abuf + (size_t)w * cap * n;
    T* AN = (T*)st.pend_AN + (size_t)w * kmax * cap;
    for (int pr = warp; pr < k * fill; pr += nw) {
      const int a = pr / fill, s = pr % fill;
      T acc = S::zero();
      for (int j = lane; j < n; j += 32) acc = S::fma(gN[(size_t)a * n + j], Ab[(size_t)s * n + j], acc);
      acc = warp_sum(acc);
      if (lane == 0) AN[(size_t)a * cap + s] = acc;
    }
  }
}

// ---------------------------------------------------------------- Y = Aeff N
// Work item = (walker, tile of rows).  One read-only pass over Ti.
template <typename T, int KT>
__global__ void __launch_bounds__(256)
pf_y_kernel(State st, int k, int tiles, int rows_per_tile, int use_list) {
  using S = Sc<T>;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  T* dsm = (T*)smem_raw;  // [KT][rows_per_tile]
  const int n = st.n, kmax = st.kmax, cap = st.cap;
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31, nw = blockDim.x >> 5;
  const int count = use_list ? st.counters[0] : (int)st.W;
  for (int item = blockIdx.x; item < count * tiles; item += gridDim.x) {
    const int w = use_list ? st.list[item / tiles] : item / tiles;
    const int tile = item % tiles;
    if (st.pend_idx[(size_t)w * kmax] < 0) continue;  // invalid proposal (uniform per CTA)
    const int fill = cap ? st.fill[w] : 0;
    const T* gN = (const T*)st.pend_N + (size_t)w * kmax * n;
    const T* Tw = (const T*)st.Ti + (size_t)w * n * n;
    const int i_beg = tile * rows_per_tile, i_end = min(n, i_beg + rows_per_tile);
    __syncthreads();
    // two rows per warp pass, 16-byte loads, 8 loads in flight per thread
    constexpr int RW = 2, U = 4;
    constexpr int VE = sizeof(T) == 8 ? 2 : 1;     // elements per 16-byte vector
    const bool vec = (n % VE) == 0;
    for (int i0 = i_beg + warp * RW; i0 < i_end; i0 += nw * RW) {
      T d[RW][KT];
#pragma unroll
      for (int r = 0; r < RW; ++r)
#pragma unroll
        for (int a = 0; a < KT; ++a) d[r][a] = S::zero();
      if (vec) {
        const int nvec = n / VE;
        for (int q0 = lane; q0 < nvec; q0 += 32 * U) {
          double2 x[U][RW];
#pragma unroll
          for (int u = 0; u < U; ++u)
#pragma unroll
            for (int r = 0; r < RW; ++r)
              x[u][r] = (q0 + 32 * u < nvec && i0 + r < i_end)
                            ? ((const double2*)(Tw + (size_t)(i0 + r) * n))[q0 + 32 * u]
                            : make_double2(0.0, 0.0);
#pragma unroll
          for (int u = 0; u < U; ++u) {
            const int q = q0 + 32 * u;
            if (q < nvec) {
#pragma unroll
              for (int a = 0; a < KT; ++a) {
                if (a < k) {
                  const double2 nv = ((const double2*)(gN + (size_t)a * n))[q];
#pragma unroll
                  for (int r = 0; r < RW; ++r) {
                    if constexpr (VE == 2) {
                      d[r][a] = S::fma(sc_from(x[u][r].x, 0.0, T{}), sc_from(nv.x, 0.0, T{}), d[r][a]);
                      d[r][a] = S::fma(sc_from(x[u][r].y, 0.0, T{}), sc_from(nv.y, 0.0, T{}), d[r][a]);
                    } else {
                      d[r][a] = S::fma(sc_from(x[u][r].x, x[u][r].y, T{}), sc_from(nv.x, nv.y, T{}), d[r][a]);
                    }
                  }
                }
              }
            }
          }
        }
      } else {
        for (int j = lane; j < n; j += 32) {
#pragma unroll
          for (int r = 0; r < RW; ++r) {
            if (i0 + r < i_end) {
              const T x = Tw[(size_t)(i0 + r) * n + j];
#pragma unroll
              for (int a = 0; a < KT; ++a)
                if (a < k) d[r][a] = S::fma(x, gN[(size_t)a * n + j], d[r][a]);
            }
          }
        }
      }
#pragma unroll
      for (int r = 0; r < RW; ++r)
#pragma unroll
        for (int a = 0; a < KT; ++a) {
          const T v = warp_sum(d[r][a]);
          if (lane == 0 && i0 + r < i_end) dsm[a * rows_per_tile + (i0 + r - i_beg)] = v;
        }
    }
    __syncthreads();
    const T* AN = cap ? (const T*)st.pend_AN + (size_t)w * kmax * cap : nullptr;
    const T* Bb = cap ? (const T*)st.Bbuf + (size_t)w * cap * n : nullptr;
    T* pY = (T*)st.pend_Y + (size_t)w * kmax * n;
    for (int ii = tid; ii < i_end - i_beg; ii += blockDim.x) {
      const int i = i_beg + ii;
      T y[KT];
#pragma unroll
      for (int a = 0; a < KT; ++a) y[a] = a < k ? dsm[a * rows_per_tile + ii] : S::zero();
      for (int s = 0; s < fill; ++s) {
        const T bv = Bb[(size_t)s * n + i];
#pragma unroll
        for (int a = 0; a < KT; ++a)
          if (a < k) y[a] = S::fma(bv, AN[(size_t)a * cap + s], y[a]);
      }
#pragma unroll
      for (int a = 0; a < KT; ++a)
        if (a < k) pY[(size_t)a * n + i] = y[a];
    }
  }
}

// ---------------------------------------------------------------- Y pass by column sums
// Y = A0^-1 N without a single warp reduction: A0^-1 is exactly skew, so
// Y[a][c] = -sum_j Ti[j][c] N[a][j] is a running sum DOWN the columns.  Work item = (walker,
// block of CW 16-byte column vectors); thread (cq, rg) owns one vector of columns and every
// RG-th row, streams its column slab with U row loads in flight (each warp load is 512
// contiguous bytes of a row), N[a][j] comes from shared memory as a broadcast.  Row groups
// (RG > 1 only when the matrix is narrower than the CTA) are combined through shared
// memory in a fixed order.  The buffer terms of the delayed path are added as in
// pf_y_kernel.  pf_y_kernel (row dot products, 5 shuffle stages per row and operand) ran
// at 0.36 of HBM at n = 512.
template <typename T, int KT>
__global__ void __launch_bounds__(256)
pf_y_colsum_kernel(State st, int k, int cblocks, int lg_cw, int use_list) {
  using S = Sc<T>;
  constexpr int VE = sizeof(T) == 8 ? 2 : 1;     // elements per 16-byte vector
  constexpr int U = 8;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const int n = st.n, kmax = st.kmax, cap = st.cap, nvec = n / VE;
  const int CW = 1 << lg_cw, RG = 256 >> lg_cw;
  T* Ns = (T*)smem_raw;                                   // [k][n]
  double2* part = (double2*)(Ns + (size_t)k * n);         // [RG][KT][CW]
  const int tid = threadIdx.x, cq = tid & (CW - 1), rg = tid >> lg_cw;
  const int count = use_list ? st.counters[0] : (int)st.W;
  for (int item = blockIdx.x; item < count * cblocks; item += gridDim.x) {
    const int w = use_list ? st.list[item / cblocks] : item / cblocks;
    const int cb = item % cblocks;
    if (st.pend_idx[(size_t)w * kmax] < 0) continue;  // invalid proposal (uniform per CTA)
    const int fill = cap ? st.fill[w] : 0;
    const T* gN = (const T*)st.pend_N + (size_t)w * kmax * n;
    const double2* Tw2 = (const double2*)((const T*)st.Ti + (size_t)w * n * n);
    __syncthreads();
    for (int q = tid; q < k * n; q += blockDim.x) Ns[q] = gN[q];
    __syncthreads();
    const int q = cb * CW + cq;
    const bool act = q < nvec;
    double2 acc[KT];
#pragma unroll
    for (int a = 0; a < KT; ++a) acc[a] = make_double2(0.0, 0.0);
    if (act) {
      for (int j0 = rg; j0 < n; j0 += RG * U) {
        double2 x[U];
#pragma unroll
        for (int u = 0; u < U; ++u) {
          const int j = j0 + u * RG;
          x[u] = j < n ? Tw2[(size_t)j * nvec + q] : make_double2(0.0, 0.0);
        }
#pragma unroll
        for (int u = 0; u < U; ++u) {
          const int j = j0 + u * RG;
          if (j < n) {
#pragma unroll
            for (int a = 0; a < KT; ++a) {
              if (a < k) {
                const T nv = Ns[(size_t)a * n + j];
                if constexpr (VE == 2) {
                  acc[a].x = fma(x[u].x, sc_re(nv), acc[a].x);
                  acc[a].y = fma(x[u].y, sc_re(nv), acc[a].y);
                } else {
                  const T r = S::fma(sc_from(x[u].x, x[u].y, T{}), nv, sc_from(acc[a].x, acc[a].y, T{}));
                  acc[a] = make_double2(sc_re(r), sc_im(r));
                }
              }
            }
          }
        }
      }
    }
    if (RG > 1) {
#pragma unroll
      for (int a = 0; a < KT; ++a)
        if (a < k) part[((size_t)rg * KT + a) * CW + cq] = acc[a];
      __syncthreads();
      if (rg == 0) {
#pragma unroll
        for (int a = 0; a < KT; ++a) {
          if (a < k) {
            for (int g = 1; g < RG; ++g) {
              const double2 t = part[((size_t)g * KT + a) * CW + cq];
              acc[a].x += t.x;
              acc[a].y += t.y;
            }
          }
        }
      }
    }
    if (rg == 0 && act) {
      const T* AN = cap ? (const T*)st.pend_AN + (size_t)w * kmax * cap : nullptr;
      const double2* Bb2 = cap ? (const double2*)((const T*)st.Bbuf + (size_t)w * cap * n) : nullptr;
      double2* pY2 = (double2*)((T*)st.pend_Y + (size_t)w * kmax * n);
      double2 y[KT];
#pragma unroll
      for (int a = 0; a < KT; ++a) y[a] = make_double2(-acc[a].x, -acc[a].y);
      for (int sft = 0; sft < fill; ++sft) {
        const double2 bv = Bb2[(size_t)sft * nvec + q];
#pragma unroll
        for (int a = 0; a < KT; ++a) {
          if (a < k) {
            const T an = AN[(size_t)a * cap + sft];
            if constexpr (VE == 2) {
              y[a].x = fma(bv.x, sc_re(an), y[a].x);
              y[a].y = fma(bv.y, sc_re(an), y[a].y);
            } else {
              const T r = S::fma(sc_from(bv.x, bv.y, T{}), an, sc_from(y[a].x, y[a].y, T{}));
              y[a] = make_double2(sc_re(r), sc_im(r));
            }
          }
        }
      }
#pragma unroll
      for (int a = 0; a < KT; ++a)
        if (a < k) pY2[(size_t)a * nvec + q] = y[a];
    }
  }
}

// ---------------------------------------------------------------- core (k >= 2)
// Builds the exactly skew 2k x 2k core R', r = (-1)^(k(k-1)/2) pf R', R'^-1.
template <typename T>
__global__ void __launch_bounds__(128)
pf_core_kernel(State st, int k, T* __restrict__ ratio_out) {
  using S = Sc<T>;
  __shared__ T R[kMaxC * kMaxC];
  __shared__ T R2[kMaxC * kMaxC];
  __shared__ T Ri[kMaxC * kMaxC];
  const int w = blockIdx.x, tid = threadIdx.x, nt = blockDim.x;
  const int warp = tid >> 5, lane = tid & 31, nw = nt >> 5;
  const int n = st.n, kmax = st.kmax, m = 2 * k;
  if (st.pend_idx[(size_t)w * kmax] < 0) return;
  const T* pC = (const T*)st.pend_C + (size_t)w * kmax * n;
  const T* pN = (const T*)st.pend_N + (size_t)w * kmax * n;
  const T* pY = (const T*)st.pend_Y + (size_t)w * kmax * n;
  const int32_t* P = st.pend_idx + (size_t)w * kmax;
  for (int q = tid; q < kMaxC * kMaxC; q += nt) R[q] = S::zero();
  __syncthreads();
  // upper-right block Tm (all a,b) and strict upper triangle of G
  for (int pr = warp; pr < 2 * k * k; pr += nw) {
    const bool isG = pr >= k * k;
    const int q = isG ? pr - k * k : pr;
    const int a = q / k, b = q % k;
    if (isG && a >= b) continue;
    const T* other = isG ? pY + (size_t)b * n : pC + (size_t)b * n;
    T acc = S::zero();
    for (int i = lane; i < n; i += 32) acc = S::fma(pN[(size_t)a * n + i], other[i], acc);
    acc = warp_sum(acc);
    if (lane == 0) {
      if (isG) {
        acc = S::add(acc, pN[(size_t)a * n + P[b]]);
        R[a * kMaxC + b] = acc;
        R[b * kMaxC + a] = S::neg(acc);
      } else {
        R[a * kMaxC + (k + b)] = acc;
        R[(k + b) * kMaxC + a] = S::neg(acc);
      }
    }
  }
  // S block: Aeff[P[a]][P[b]] = C[b][P[a]], strict upper triangle mirrored
  if (tid < k * k) {
    const int a = tid / k, b = tid % k;
    if (a < b) {
      const T v = pC[(size_t)b * n + P[a]];
      R[(k + a) * kMaxC + (k + b)] = v;
      R[(k + b) * kMaxC + (k + a)] = S::neg(v);
    }
  }
  __syncthreads();
  for (int q = tid; q < kMaxC * kMaxC; q += nt) R2[q] = R[q];
  __syncthreads();
  // warp 0: R'^-1 by Gauss-Jordan, warp 1: pf R' by Parlett-Reid, side by side (each bit-identical
  // to the serial small_det_inv / small_pf, which at k = 8 cost more than the update pass)
  __shared__ T pf_s;
  __shared__ int ok_s;
  if (warp == 0) {
    bool ok;
    warp_det_inv(R, Ri, m, kMaxC, &ok, lane);
    if (lane == 0) ok_s = ok ? 1 : 0;
  } else if (warp == 1) {
    T pfv = warp_pf(R2, m, kMaxC, lane);
    if ((k * (k - 1) / 2) & 1) pfv = S::neg(pfv);
    if (lane == 0) pf_s = pfv;
  }
  __syncthreads();
  const T pfv = pf_s;
  const bool ok = ok_s && S::finite(pfv) && !S::is_zero(pfv);
  if (tid == 0) {
    ratio_out[w] = pfv;
    ((T*)st.pend_ratio)[w] = pfv;
    st.pend_ok[w] = ok ? 1 : 0;
  }
  T* pR = (T*)st.pend_Rinv + (size_t)w * st.kc * st.kc;
  for (int q = tid; q < m * m; q += nt) {
    const int a = q / m, b = q % m;
    if (a == b) pR[a * st.kc + a] = S::zero();
    else if (a < b) {
      const T v = ok ? S::scale(S::sub(Ri[a * kMaxC + b], Ri[b * kMaxC + a]), 0.5) : S::zero();
      pR[a * st.kc + b] = v;
      pR[b * st.kc + a] = S::neg(v);
    }
  }
}

// Y'[alpha][i] for alpha in [0,2k): (Y + E_P, C)
template <typename T>
__device__ __forceinline__ T yprime(const T* pY, const T* pC, const int* P, int k, int n, int alpha,
                                    int i) {
  if (alpha < k) {
    T y = pY[(size_t)alpha * n + i];
    return (i == P[alpha]) ? Sc<T>::add(y, Sc<T>::one()) : y;
  }
  return pC[(size_t)(alpha - k) * n + i];
}

// ---------------------------------------------------------------- immediate update (a4)
// Work item = (accepted walker, upper tile pair I <= J of 32x32 tiles).
//   Ti[i][j] += sum_beta g[beta][i] Y'[beta][j],  g[beta][i] = sum_alpha Y'[alpha][i] R'^-1[alpha][beta]
// for j > i only; the mirrored entry receives the exact negative.
template <typename T>
__global__ void __launch_bounds__(256) pf_update_kernel(State st, int k, int t1) {
  using S = Sc<T>;
  constexpr int TS = 32;
  __shared__ T gI[kMaxC][TS];
  __shared__ T yJ[kMaxC][TS];
  __shared__ T tile[TS][TS + 1];
  __shared__ T Ri[kMaxC * kMaxC];
  __shared__ int P[kMaxK];
  const int n = st.n, kmax = st.kmax, m = 2 * k;
  const int tid = threadIdx.x, tx = tid & 31, ty = tid >> 5;
  const int count = st.counters[0];
  const int tiles = t1 * (t1 + 1) / 2;
  for (int item = blockIdx.x; item < count * tiles; item += gridDim.x) {
    const int w = st.list[item / tiles];
    int rem = item % tiles, I = 0;
    while (rem >= t1 - I) { rem -= t1 - I; ++I; }
    const int J = I + rem;
    const int i0 = I * TS, j0 = J * TS;
    const T* pC = (const T*)st.pend_C + (size_t)w * kmax * n;
    const T* pY = (const T*)st.pend_Y + (size_t)w * kmax * n;
    T* Tw = (T*)st.Ti + (size_t)w * n * n;
    __syncthreads();
    for (int q = tid; q < m * m; q += 256)
      Ri[(q / m) * kMaxC + (q % m)] = ((const T*)st.pend_Rinv)[(size_t)w * st.kc * st.kc + (q / m) * st.kc + (q % m)];
    if (tid < k) P[tid] = st.pend_idx[(size_t)w * kmax + tid];
    __syncthreads();
    for (int q = tid; q < m * TS; q += 256) {
      const int beta = q / TS, c = q % TS;
      const int j = j0 + c, i = i0 + c;
      yJ[beta][c] = j < n ? yprime(pY, pC, P, k, n, beta, j) : S::zero();
      T g = S::zero();
      if (i < n)
        for (int alpha = 0; alpha < m; ++alpha)
          g = S::fma(yprime(pY, pC, P, k, n, alpha, i), Ri[alpha * kMaxC + beta], g);
      gI[beta][c] = g;
    }
    __syncthreads();
    for (int r = ty; r < TS; r += 8) {
      const int i = i0 + r, j = j0 + tx;
      T v = S::zero();
      if (i < n && j < n && j > i) {
        v = Tw[(size_t)i * n + j];
        for (int beta = 0; beta < m; ++beta) v = S::fma(gI[beta][r], yJ[beta][tx], v);
        Tw[(size_t)i * n + j] = v;
      }
      tile[r][tx] = v;
    }
    __syncthreads();
    // mirrored write: Ti[j][i] = -new(i,j)
    for (int r = ty; r < TS; r += 8) {
      const int j = j0 + r, i = i0 + tx;  // element (j,i) <- -tile[tx][r]
      if (i < n && j < n && j > i) Tw[(size_t)j * n + i] = S::neg(tile[tx][r]);
    }
  }
}

// ---------------------------------------------------------------- streaming update (a4)
// Large walkers: work item = (accepted walker, tile of 64 rows).  Y' and g = Y' R'^-1
// (2k x n each) are staged in shared memory; each warp streams whole rows of Ti with
// coalesced loads and stores.  As in the resident kernel every element is produced by
// its own thread: below the diagonal the thread recomputes the mirrored upper value
// from -Ti[r][c] with the same operands in the same order and stores its negative
// (exact skewness, no transposed access).
template <typename T, int MT>   // MT >= 2k: size of the per-row factor arrays
__global__ void __launch_bounds__(256)
pf_update_stream_kernel(State st, int k, int tiles, int rows_per_tile) {
  using S = Sc<T>;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const int n = st.n, kmax = st.kmax, m = 2 * k;
  T* yv = (T*)smem_raw;          // [m][n]
  T* gv = yv + (size_t)m * n;    // [m][n]
  __shared__ T Ri[kMaxC * kMaxC];
  __shared__ int P[kMaxK];
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31, nw = blockDim.x >> 5;
  const int count = st.counters[0];
  for (int item = blockIdx.x; item < count * tiles; item += gridDim.x) {
    const int w = st.list[item / tiles];
    const int tile = item % tiles;
    const T* pC = (const T*)st.pend_C + (size_t)w * kmax * n;
    const T* pY = (const T*)st.pend_Y + (size_t)w * kmax * n;
    T* Tw = (T*)st.Ti + (size_t)w * n * n;
    __syncthreads();
    for (int q = tid; q < m * m; q += 256)
      Ri[(q / m) * kMaxC + (q % m)] =
          ((const T*)st.pend_Rinv)[(size_t)w * st.kc * st.kc + (q / m) * st.kc + (q % m)];
    if (tid < k) P[tid] = st.pend_idx[(size_t)w * kmax + tid];
    __syncthreads();
    for (int i = tid; i < n; i += 256) {
      T yp[kMaxC];
      for (int alpha = 0; alpha < m; ++alpha) {
        yp[alpha] = yprime(pY, pC, P, k, n, alpha, i);
        yv[(size_t)alpha * n + i] = yp[alpha];
      }
      for (int beta = 0; beta < m; ++beta) {
        T g = S::zero();
        for (int alpha = 0; alpha < m; ++alpha) g = S::fma(yp[alpha], Ri[alpha * kMaxC + beta], g);
        gv[(size_t)beta * n + i] = g;
      }
    }
    __syncthreads();
    const int r_end = min(n, (tile + 1) * rows_per_tile);
    for (int r = tile * rows_per_tile + warp; r < r_end; r += nw) {
      T* row = Tw + (size_t)r * n;
      // the row's own factors live in registers; one shared-memory operand per FMA
      T gr[MT], yr[MT];
#pragma unroll
      for (int beta = 0; beta < MT; ++beta) {
        gr[beta] = beta < m ? gv[(size_t)beta * n + r] : S::zero();
        yr[beta] = beta < m ? yv[(size_t)beta * n + r] : S::zero();
      }
#pragma unroll 2
      for (int c = lane; c < r; c += 32) {          // below the diagonal: -v(c, r)
        T v = S::neg(row[c]);
#pragma unroll
        for (int beta = 0; beta < MT; ++beta)
          if (beta < m) v = S::fma(gv[(size_t)beta * n + c], yr[beta], v);
        row[c] = S::neg(v);
      }
      if (lane == 0) row[r] = S::zero();
#pragma unroll 2
      for (int c = r + 1 + lane; c < n; c += 32) {   // above: v(r, c)
        T v = row[c];
#pragma unroll
        for (int beta = 0; beta < MT; ++beta)
          if (beta < m) v = S::fma(gr[beta], yv[(size_t)beta * n + c], v);
        row[c] = v;
      }
    }
  }
}

// One row of the on-chip rank-2k update (Eq. 21; k = 1: Eq. 22), done by one warp.  Every
// element is produced by its own lane: for r > c the mirrored upper value v(c,r) is
// recomputed from -row[c] with the same operands in the same order and stored negated,
// so the matrix stays exactly skew with no transposed access.
template <typename T>
__device__ __forceinline__ void pf_row_update(T* row, int r, int n, int m, const T* yv, const T* gv,
                                              int lane) {
  using S = Sc<T>;
  if constexpr (sizeof(T) == 8) {
    if (m == 2) {
      // fp64, k = 1 (Eq. 22): pairs of columns; a pair entirely below / above the
      // diagonal needs no per-element selection
      const double g0r = gv[r], g1r = gv[n + r], y0r = yv[r], y1r = yv[n + r];
      const double2* g0 = (const double2*)gv;
      const double2* g1 = (const double2*)(gv + n);
      const double2* y0 = (const double2*)yv;
      const double2* y1 = (const double2*)(yv + n);
      double2* row2 = (double2*)row;
      for (int q = lane; q < n / 2; q += 32) {
        const int c0 = 2 * q;
        double2 x = row2[q];
        if (c0 + 1 < r) {          // both below the diagonal: mirrored value, negated
          const double2 a = g0[q], b = g1[q];
          x.x = -fma(b.x, y1r, fma(a.x, y0r, -x.x));
          x.y = -fma(b.y, y1r, fma(a.y, y0r, -x.y));
        } else if (c0 > r) {       // both above
          const double2 a = y0[q], b = y1[q];
          x.x = fma(g1r, b.x, fma(g0r, a.x, x.x));
          x.y = fma(g1r, b.y, fma(g0r, a.y, x.y));
        } else {                   // the pair that holds the diagonal element
          double e[2] = {x.x, x.y};
#pragma unroll
          for (int t = 0; t < 2; ++t) {
            const int cc = c0 + t;
            if (cc == r) e[t] = 0.0;
            else if (cc < r) e[t] = -fma(gv[n + cc], y1r, fma(gv[cc], y0r, -e[t]));
            else e[t] = fma(g1r, yv[n + cc], fma(g0r, yv[cc], e[t]));
          }
          x.x = e[0];
          x.y = e[1];
        }
        row2[q] = x;
      }
      return;
    }
  }
  if (m == 2) {
    const T g0r = gv[r], g1r = gv[n + r], y0r = yv[r], y1r = yv[n + r];
    for (int cc = lane; cc < n; cc += 32) {
      const bool up = r < cc;
      const T x = row[cc];
      T v = up ? x : S::neg(x);
      v = S::fma(up ? g0r : gv[cc], up ? yv[cc] : y0r, v);
      v = S::fma(up ? g1r : gv[n + cc], up ? yv[n + cc] : y1r, v);
      row[cc] = (r == cc) ? S::zero() : (up ? v : S::neg(v));
    }
  } else {
    for (int cc = lane; cc < n; cc += 32) {
      const bool up = r < cc;
      const int i = up ? r : cc, j = up ? cc : r;
      const T x = row[cc];
      T v = up ? x : S::neg(x);
      for (int beta = 0; beta < m; ++beta) v = S::fma(gv[beta * n + i], yv[beta * n + j], v);
      row[cc] = (r == cc) ? S::zero() : (up ? v : S::neg(v));
    }
  }
}

// ---------------------------------------------------------------- cluster-resident update (a4)
// The same on-chip update with a walker's inverse spread over a thread-block CLUSTER:
// CTA `cr` of CL holds rows [cr*rpc, (cr+1)*rpc) (one bulk copy in, one bulk store out).
// A 32-row slab of C3 is 32 KB, so several CTAs share an SM and the load of one slab
// overlaps the arithmetic and the store of others without any in-CTA pipeline, and
// ~4x more work items than walkers even out the tail of the persistent grid.  The only
// cross-CTA data is Y = A^-1 N (k = 1): each CTA computes the entries of its own rows
// and writes them into every peer's shared memory (distributed shared memory), one
// cluster barrier per walker.  The Y' buffer alternates between two slots so that a
// peer that is one walker ahead never overwrites what this CTA still reads.
template <typename T>
__global__ void __launch_bounds__(256) pf_cluster_update_kernel(State st, int k, int need_y) {
  using S = Sc<T>;
  namespace cg = cooperative_groups;
  cg::cluster_group cluster = cg::this_cluster();
  extern __shared__ __align__(128) unsigned char smem_raw[];
  const int n = st.n, kmax = st.kmax, m = 2 * k;
  const int CL = (int)cluster.num_blocks(), cr = (int)cluster.block_rank();
  const int ncl = (int)gridDim.x / CL, cid = (int)blockIdx.x / CL;
  const int rpc = (n + CL - 1) / CL, r0 = cr * rpc, r1 = min(n, r0 + rpc);
  const int rows = max(0, r1 - r0);
  T* Ts = (T*)smem_raw;                  // [rpc][n]  this CTA's rows
  T* yvb = Ts + (size_t)rpc * n;         // [2][m][n] Y' (two slots)
  T* gv = yvb + (size_t)2 * m * n;       // [m][n]    Y' R'^-1
  T* nv = gv + (size_t)m * n;            // [n]       new row (k = 1)
  __shared__ T Ri[kMaxC * kMaxC];
  __shared__ int P[kMaxK];
  __shared__ __align__(8) uint64_t bar;
  const int tid = threadIdx.x, nt = blockDim.x, warp = tid >> 5, lane = tid & 31, nw = nt >> 5;
  const int count = st.counters[0];
  const uint32_t bytes = (uint32_t)((size_t)rows * n * sizeof(T));
  if (tid == 0) {
    tma::mbar_init(&bar, 1);
    tma::fence_barrier_init();
  }
  __syncthreads();
  auto load_rows = [&](int w) {   // thread 0 only
    if (rows <= 0) return;
    tma::mbar_arrive_expect_tx(&bar, bytes);
    tma::load(Ts, (const T*)st.Ti + (size_t)w * n * n + (size_t)r0 * n, bytes, &bar);
  };
  if (tid == 0 && cid < count) load_rows(st.list[cid]);
  uint32_t phase = 0;
  int slot = 0;
  for (int it = cid; it < count; it += ncl, slot ^= 1) {
    const int w = st.list[it];
    const int w_next = it + ncl < count ? st.list[it + ncl] : -1;
    T* yv = yvb + (size_t)slot * m * n;
    const T* pC = (const T*)st.pend_C + (size_t)w * kmax * n;
    const T* pY = (const T*)st.pend_Y + (size_t)w * kmax * n;
    const T* pN = (const T*)st.pend_N + (size_t)w * kmax * n;
    for (int q = tid; q < m * m; q += nt)
      Ri[(q / m) * kMaxC + (q % m)] =
          ((const T*)st.pend_Rinv)[(size_t)w * st.kc * st.kc + (q / m) * st.kc + (q % m)];
    if (tid < k) P[tid] = st.pend_idx[(size_t)w * kmax + tid];
    __syncthreads();
    for (int q = tid; q < k * n; q += nt) {
      const int a = q / n, i = q % n;
      yv[(size_t)(k + a) * n + i] = pC[q];
      if (need_y) nv[q] = pN[q];   // k == 1
      else yv[q] = (i == P[a]) ? S::add(pY[q], S::one()) : pY[q];
    }
    __syncthreads();
    if (rows > 0) tma::mbar_wait(&bar, phase);
    phase ^= 1;
    if (need_y) {
      // Y = A^-1 N for the rows held here, broadcast to every CTA of the cluster
      for (int i = r0 + warp; i < r1; i += nw) {
        const T* row = Ts + (size_t)(i - r0) * n;
        T acc = S::zero();
        for (int j = lane; j < n; j += 32) acc = S::fma(row[j], nv[j], acc);
        acc = warp_sum(acc);
        if (i == P[0]) acc = S::add(acc, S::one());
        if (lane < CL) cluster.map_shared_rank(yv, lane)[i] = acc;
      }
      cluster.sync();
    } else {
      __syncthreads();
    }
    for (int q = tid; q < m * n; q += nt) {
      const int beta = q / n, i = q % n;
      T g = S::zero();
      for (int alpha = 0; alpha < m; ++alpha)
        g = S::fma(yv[(size_t)alpha * n + i], Ri[alpha * kMaxC + beta], g);
      gv[q] = g;
    }
    __syncthreads();
    for (int r = r0 + warp; r < r1; r += nw)
      pf_row_update<T>(Ts + (size_t)(r - r0) * n, r, n, m, yv, gv, lane);
    tma::fence_proxy_async();
    __syncthreads();
    if (tid == 0 && rows > 0) {
      tma::store((T*)st.Ti + (size_t)w * n * n + (size_t)r0 * n, Ts, bytes);
      tma::store_commit();
      if (w_next >= 0) {
        tma::store_wait_read<0>();   // the slab has left shared memory
        load_rows(w_next);
      }
    }
  }
  if (tid == 0) tma::store_wait_all<0>();
}

// ---------------------------------------------------------------- cluster-resident update, fp64 k = 1
// Config C3's case (Eq. 22), laid out to minimise issued instructions (the generic kernel
// above is issue-bound at n = 128, not memory-bound): thread (q, rg) owns the COLUMN PAIR
// (2q, 2q+1) and every RG-th row of the slab, so that
//  * Y = A^-1 N needs no warp reduction: by skewness y[c] = -sum_j Ti[j][c] N[j], a running
//    sum down the thread's own columns; the partial sums of the row groups meet in shared
//    memory, those of the CL slabs in every peer's shared memory (DSMEM), and every CTA adds
//    them in the same order (identical Y everywhere: the mirror stays exact);
//  * the column factors y0,y1,-g0,-g1 of the pair stay in registers for the whole slab, the
//    row factors come from one 32-byte broadcast load per row;
//  * below the diagonal -fma(g1c, y1r, fma(g0c, y0r, -x)) is evaluated as
//    fma(-g1c, y1r, fma(-g0c, y0r, x)): the same value bit for bit (rounding is symmetric
//    under negation), without the two sign flips.
// LG > 0: n/2 = 2^LG column pairs and exactly RPT rows per thread (loops fully unrolled, RPT
// independent shared-memory loads in flight); LG = 0: sizes taken at run time.
template <int LG, int RPT>
__global__ void __launch_bounds__(256, 4) pf_cluster_k1_kernel(State st, int lg_dyn) {
  const int lg_nqp = LG > 0 ? LG : lg_dyn;
  namespace cg = cooperative_groups;
  cg::cluster_group cluster = cg::this_cluster();
  extern __shared__ __align__(128) unsigned char smem_raw[];
  const int n = LG > 0 ? (2 << LG) : st.n, kmax = st.kmax, NQ = n >> 1;
  const int CL = (int)cluster.num_blocks(), cr = (int)cluster.block_rank();
  const int ncl = (int)gridDim.x / CL, cid = (int)blockIdx.x / CL;
  const int rpc = (n + CL - 1) / CL, r0 = cr * rpc, r1 = min(n, r0 + rpc);
  const int rows = max(0, r1 - r0);
  const int RG = 256 >> lg_nqp;
  const int rpt = LG > 0 ? RPT                                               // rows of this thread
                         : (rows > (int)(threadIdx.x >> lg_nqp) ? (rows - 1 - (int)(threadIdx.x >> lg_nqp)) / RG + 1 : 0);
  const int tid = threadIdx.x, q = tid & ((1 << lg_nqp) - 1), rg = tid >> lg_nqp;
  const bool act = q < NQ;
  double* Ts = (double*)smem_raw;                          // [rpc][n]   this CTA's rows
  double2* Ts2 = (double2*)Ts;
  double2* part = (double2*)(Ts + (size_t)rpc * n);        // [RG][NQ]   column sums per row group
  double2* ysum = part + (size_t)RG * NQ;                  // [2][CL][NQ] column sums per slab (two slots)
  double2* rowc = ysum + (size_t)2 * CL * NQ;              // [n][2]     {g0,g1},{y0,y1} of row r
  double* nv = (double*)(rowc + (size_t)2 * n);            // [n]        new row
  __shared__ __align__(8) uint64_t bar;
  const int count = st.counters[0];
  const uint32_t bytes = (uint32_t)((size_t)rows * n * sizeof(double));
  if (tid == 0) {
    tma::mbar_init(&bar, 1);
    tma::fence_barrier_init();
  }
  __syncthreads();
  auto load_rows = [&](int w) {   // thread 0 only
    if (rows <= 0) return;
    tma::mbar_arrive_expect_tx(&bar, bytes);
    tma::load(Ts, (const double*)st.Ti + (size_t)w * n * n + (size_t)r0 * n, bytes, &bar);
  };
  if (tid == 0 && cid < count) load_rows(st.list[cid]);
  uint32_t phase = 0;
  int slot = 0;
  for (int it = cid; it < count; it += ncl, slot ^= 1) {
    const int w = st.list[it];
    const int w_next = it + ncl < count ? st.list[it + ncl] : -1;
    const double* pC = (const double*)st.pend_C + (size_t)w * kmax * n;
    const double* pN = (const double*)st.pend_N + (size_t)w * kmax * n;
    const double* Rw = (const double*)st.pend_Rinv + (size_t)w * st.kc * st.kc;
    const double Ri00 = Rw[0], Ri01 = Rw[1], Ri10 = Rw[st.kc], Ri11 = Rw[st.kc + 1];
    const int p0 = st.pend_idx[(size_t)w * kmax];
    const double2 y1q = act ? ((const double2*)pC)[q] : make_double2(0.0, 0.0);
    for (int i = tid; i < n; i += 256) nv[i] = pN[i];
    __syncthreads();
    if (rows > 0) tma::mbar_wait(&bar, phase);
    phase ^= 1;
    // ---- column sums over the slab's rows
    if (act) {
      double2 acc = make_double2(0.0, 0.0);
#pragma unroll
      for (int t = 0; t < (LG > 0 ? RPT : rpt); ++t) {
        const int rr = rg + RG * t;
        const double2 x = Ts2[rr * NQ + q];
        const double nr = nv[r0 + rr];
        acc.x = fma(x.x, nr, acc.x);
        acc.y = fma(x.y, nr, acc.y);
      }
      part[rg * NQ + q] = acc;
    }
    __syncthreads();
    if (act) {
      double2 sum = part[q];
      for (int g = 1; g < RG; ++g) {
        const double2 t = part[g * NQ + q];
        sum.x += t.x;
        sum.y += t.y;
      }
      for (int p = rg; p < CL; p += RG)
        cluster.map_shared_rank(ysum, p)[(size_t)(slot * CL + cr) * NQ + q] = sum;
    }
    cluster.sync();
    double2 y0q = make_double2(0.0, 0.0), g0q = y0q, g1q = y0q;
    if (act) {
      double2 sum = ysum[(size_t)(slot * CL) * NQ + q];
      for (int c = 1; c < CL; ++c) {
        const double2 t = ysum[(size_t)(slot * CL + c) * NQ + q];
        sum.x += t.x;
        sum.y += t.y;
      }
      y0q.x = (2 * q == p0) ? -sum.x + 1.0 : -sum.x;
      y0q.y = (2 * q + 1 == p0) ? -sum.y + 1.0 : -sum.y;
      g0q.x = fma(y1q.x, Ri10, y0q.x * Ri00);
      g0q.y = fma(y1q.y, Ri10, y0q.y * Ri00);
      g1q.x = fma(y1q.x, Ri11, y0q.x * Ri01);
      g1q.y = fma(y1q.y, Ri11, y0q.y * Ri01);
      if (rg == 0) {
        rowc[4 * q + 0] = make_double2(g0q.x, g1q.x);
        rowc[4 * q + 1] = make_double2(y0q.x, y1q.x);
        rowc[4 * q + 2] = make_double2(g0q.y, g1q.y);
        rowc[4 * q + 3] = make_double2(y0q.y, y1q.y);
      }
    }
    __syncthreads();
    // ---- rank-2 update of the slab (Eq. 22)
    if (act) {
      const double2 ng0 = make_double2(-g0q.x, -g0q.y), ng1 = make_double2(-g1q.x, -g1q.y);
      const int c0 = 2 * q;
#pragma unroll
      for (int t = 0; t < (LG > 0 ? RPT : rpt); ++t) {
        const int rr = rg + RG * t, r = r0 + rr;
        double2 x = Ts2[rr * NQ + q];
        const double2 gr = rowc[2 * r], yr = rowc[2 * r + 1];
        if (c0 + 1 < r) {            // both below the diagonal
          x.x = fma(ng1.x, yr.y, fma(ng0.x, yr.x, x.x));
          x.y = fma(ng1.y, yr.y, fma(ng0.y, yr.x, x.y));
        } else if (c0 > r) {         // both above
          x.x = fma(gr.y, y1q.x, fma(gr.x, y0q.x, x.x));
          x.y = fma(gr.y, y1q.y, fma(gr.x, y0q.y, x.y));
        } else if (c0 == r) {        // (r,r), (r,r+1)
          x.x = 0.0;
          x.y = fma(gr.y, y1q.y, fma(gr.x, y0q.y, x.y));
        } else {                     // (r,r-1), (r,r)
          x.x = fma(ng1.x, yr.y, fma(ng0.x, yr.x, x.x));
          x.y = 0.0;
        }
        Ts2[rr * NQ + q] = x;
      }
    }
    tma::fence_proxy_async();
    __syncthreads();
    if (tid == 0 && rows > 0) {
      tma::store((double*)st.Ti + (size_t)w * n * n + (size_t)r0 * n, Ts, bytes);
      tma::store_commit();
      if (w_next >= 0) {
        tma::store_wait_read<0>();   // the slab has left shared memory
        load_rows(w_next);
      }
    }
  }
  if (tid == 0) tma::store_wait_all<0>();
}

// ---------------------------------------------------------------- whole-walker resident update, fp64 k = 1
// The column-pair scheme of pf_cluster_k1_kernel with the whole inverse of a walker in ONE
// CTA of 1024 threads (C3's n = 128 is the unrolled instance): no cluster barrier, no DSMEM
// traffic, per-walker fixed costs paid once.  Everything the next walker needs is in flight
// while the current one is updated:
//  * the inverse moves in NCH row chunks through NB = NCH+1 rotating shared-memory buffers
//    (one bulk copy + mbarrier each): chunk c of the next walker lands in the buffer of
//    chunk c-1 of the current one as soon as that has been stored, chunk 0 in the spare;
//  * the walker's small operands (new row, gathered column, R'^-1, slot) are staged two-deep
//    with cp.async, the walker index is read two items ahead;
//  * the column sums of the 1024/2^LG row groups are combined in two levels (4-way each for
//    LG = 6) instead of every thread re-adding all of them: the kernel is bound by
//    shared-memory bandwidth, not by HBM, until these are trimmed.
__device__ __forceinline__ void cp_async16(void* smem_dst, const void* gsrc) {
  asm volatile("cp.async.ca.shared.global [%0], [%1], 16;" ::"r"(tma::smem_u32(smem_dst)), "l"(gsrc) : "memory");
}
__device__ __forceinline__ void cp_async4(void* smem_dst, const void* gsrc) {
  asm volatile("cp.async.ca.shared.global [%0], [%1], 4;" ::"r"(tma::smem_u32(smem_dst)), "l"(gsrc) : "memory");
}

template <int LG, int NB>
__global__ void __launch_bounds__(1024, 1) pf_resident_k1_kernel(State st, int lg_dyn) {
  constexpr int NCH = 4, SP = NB - NCH;   // SP spare buffers: the next walker's loads run SP chunks ahead
  extern __shared__ __align__(128) unsigned char smem_raw[];
  const int lg = LG > 0 ? LG : lg_dyn;
  const int n = LG > 0 ? (2 << LG) : st.n, kmax = st.kmax, NQ = n >> 1;
  const int RG = 1024 >> lg, R2 = RG >> 2;
  const int tid = threadIdx.x, q = tid & ((1 << lg) - 1), rg = tid >> lg;
  const bool act = q < NQ;
  const int rpc = (n + NCH - 1) / NCH;  // rows per chunk
  const int cstride2 = rpc * NQ;        // double2 per chunk buffer
  const int STG = 2 * n + 6;            // doubles per staging slot: N row, C row, R'^-1 (2x2), {slot index, next walker}
  double2* Tb2 = (double2*)smem_raw;                       // [NB][rpc][n/2]
  double2* part = Tb2 + (size_t)NB * cstride2;             // [RG][NQ]   column sums per row group
  double2* part2 = part + (size_t)RG * NQ;                 // [R2][NQ]   ... per four row groups
  double2* rowc = part2 + (size_t)R2 * NQ;                 // [n][2]     {g0,g1},{y0,y1} of row r
  double* stg = (double*)(rowc + (size_t)2 * n);           // [2][STG]
  __shared__ __align__(8) uint64_t bar[NB];
  const int count = st.counters[0], grid = (int)gridDim.x;
  if (tid == 0) {
    for (int c = 0; c < NB; ++c) tma::mbar_init(&bar[c], 1);
    tma::fence_barrier_init();
  }
  __syncthreads();
  auto load_chunk = [&](int w, int c, int g) {   // thread 0 only; g = position in the chunk sequence
    const int r0 = c * rpc, rows = min(rpc, n - r0);
    if (rows <= 0) return;
    const int b = g % NB;
    const uint32_t bytes = (uint32_t)((size_t)rows * n * sizeof(double));
    tma::mbar_arrive_expect_tx(&bar[b], bytes);
    tma::load(Tb2 + (size_t)b * cstride2, (const double*)st.Ti + (size_t)w * n * n + (size_t)r0 * n, bytes, &bar[b]);
  };
  auto stage = [&](int w, int slot, const int* next) {   // small operands of walker w -> staging slot
    double* d = stg + slot * STG;
    const double* Rw = (const double*)st.pend_Rinv + (size_t)w * st.kc * st.kc;
    if (tid < NQ) cp_async16(d + 2 * tid, (const double*)st.pend_N + (size_t)w * kmax * n + 2 * tid);
    else if (tid < 2 * NQ) cp_async16(d + n + 2 * (tid - NQ), (const double*)st.pend_C + (size_t)w * kmax * n + 2 * (tid - NQ));
    else if (tid == 2 * NQ) cp_async16(d + 2 * n, Rw);
    else if (tid == 2 * NQ + 1) cp_async16(d + 2 * n + 2, Rw + st.kc);
    else if (tid == 2 * NQ + 2) cp_async4(d + 2 * n + 4, st.pend_idx + (size_t)w * kmax);
    else if (tid == 2 * NQ + 3 && next) cp_async4((int*)(d + 2 * n + 4) + 1, next);   // walker after w in this CTA's sequence
  };
  int w = (int)blockIdx.x < count ? st.list[blockIdx.x] : -1;
  if (w >= 0) {
    if (tid == 0)
      for (int c = 0; c < NCH; ++c) load_chunk(w, c, c);
    stage(w, 0, (int)blockIdx.x + grid < count ? st.list + blockIdx.x + grid : nullptr);
  }
  asm volatile("cp.async.commit_group;" ::: "memory");
  int j = 0;
  for (int it = blockIdx.x; it < count; it += grid, ++j) {
    const int slot = j & 1, g0 = j * NCH;
    double* Tw = (double*)st.Ti + (size_t)w * n * n;
    asm volatile("cp.async.wait_group 0;" ::: "memory");
    __syncthreads();
    const double* sd = stg + slot * STG;
    // the next walker's index arrived with this walker's operands; its operands (and the index after
    // it) are requested now and have this whole item to land
    const int w1 = it + grid < count ? *((const int*)(sd + 2 * n + 4) + 1) : -1;
    if (w1 >= 0) stage(w1, slot ^ 1, it + 2 * grid < count ? st.list + it + 2 * grid : nullptr);
    asm volatile("cp.async.commit_group;" ::: "memory");
    const double* nv = sd;
    const double2 y1q = act ? ((const double2*)(sd + n))[q] : make_double2(0.0, 0.0);
    // ---- column sums, chunk by chunk as the bulk copies land: y[c] = -sum_j Ti[j][c] N[j]
    double2 acc = make_double2(0.0, 0.0);
#pragma unroll
    for (int c = 0; c < NCH; ++c) {
      const int r0 = c * rpc, r1 = min(n, r0 + rpc);
      if (r0 < n) {
        const int g = g0 + c, b = g % NB;
        tma::mbar_wait(&bar[b], (uint32_t)((g / NB) & 1));
        if (act) {
          const double2* Tc = Tb2 + (size_t)b * cstride2 - (size_t)r0 * NQ;
#pragma unroll 2
          for (int rr = r0 + rg; rr < r1; rr += RG) {
            const double2 x = Tc[rr * NQ + q];
            const double nr = nv[rr];
            acc.x = fma(x.x, nr, acc.x);
            acc.y = fma(x.y, nr, acc.y);
          }
        }
      }
    }
    if (act) part[rg * NQ + q] = acc;
    __syncthreads();
    // the spare buffers (last chunks of the previous walker, stored long ago) take the first chunks of the next walker
    if (tid == 0 && w1 >= 0) {
      tma::store_wait_read<0>();
      for (int c = 0; c < SP; ++c) load_chunk(w1, c, g0 + NCH + c);
    }
    if (act && rg < R2) {
      double2 sum = part[(4 * rg) * NQ + q];
#pragma unroll
      for (int g = 1; g < 4; ++g) {
        const double2 t = part[(4 * rg + g) * NQ + q];
        sum.x += t.x;
        sum.y += t.y;
      }
      part2[rg * NQ + q] = sum;
    }
    __syncthreads();
    double2 y0q = make_double2(0.0, 0.0), g0q = y0q, g1q = y0q;
    if (act) {
      const double Ri00 = sd[2 * n], Ri01 = sd[2 * n + 1], Ri10 = sd[2 * n + 2], Ri11 = sd[2 * n + 3];
      const int p0 = *(const int*)(sd + 2 * n + 4);
      double2 sum = part2[q];
      for (int g = 1; g < R2; ++g) {
        const double2 t = part2[g * NQ + q];
        sum.x += t.x;
        sum.y += t.y;
      }
      y0q.x = (2 * q == p0) ? -sum.x + 1.0 : -sum.x;
      y0q.y = (2 * q + 1 == p0) ? -sum.y + 1.0 : -sum.y;
      g0q.x = fma(y1q.x, Ri10, y0q.x * Ri00);
      g0q.y = fma(y1q.y, Ri10, y0q.y * Ri00);
      g1q.x = fma(y1q.x, Ri11, y0q.x * Ri01);
      g1q.y = fma(y1q.y, Ri11, y0q.y * Ri01);
      if (rg == 0) {
        rowc[4 * q + 0] = make_double2(g0q.x, g1q.x);
        rowc[4 * q + 1] = make_double2(y0q.x, y1q.x);
        rowc[4 * q + 2] = make_double2(g0q.y, g1q.y);
        rowc[4 * q + 3] = make_double2(y0q.y, y1q.y);
      }
    }
    __syncthreads();
    // ---- rank-2 update (Eq. 22) chunk by chunk; a finished chunk is stored at once, and the
    // buffer of the chunk stored before it is refilled with the next walker's data
    const double2 ng0 = make_double2(-g0q.x, -g0q.y), ng1 = make_double2(-g1q.x, -g1q.y);
    const int c0 = 2 * q;
#pragma unroll
    for (int c = 0; c < NCH; ++c) {
      const int r0 = c * rpc, r1 = min(n, r0 + rpc);
      if (r0 >= n) break;
      const int b = (g0 + c) % NB;
      double2* Tc = Tb2 + (size_t)b * cstride2 - (size_t)r0 * NQ;
      if (act) {
#pragma unroll 2
        for (int r = r0 + rg; r < r1; r += RG) {
          double2 x = Tc[r * NQ + q];
          const double2 gr = rowc[2 * r], yr = rowc[2 * r + 1];
          if (c0 + 1 < r) {            // both below the diagonal
            x.x = fma(ng1.x, yr.y, fma(ng0.x, yr.x, x.x));
            x.y = fma(ng1.y, yr.y, fma(ng0.y, yr.x, x.y));
          } else if (c0 > r) {         // both above
            x.x = fma(gr.y, y1q.x, fma(gr.x, y0q.x, x.x));
            x.y = fma(gr.y, y1q.y, fma(gr.x, y0q.y, x.y));
          } else if (c0 == r) {        // (r,r), (r,r+1)
            x.x = 0.0;
            x.y = fma(gr.y, y1q.y, fma(gr.x, y0q.y, x.y));
          } else {                     // (r,r-1), (r,r)
            x.x = fma(ng1.x, yr.y, fma(ng0.x, yr.x, x.x));
            x.y = 0.0;
          }
          Tc[r * NQ + q] = x;
        }
      }
      tma::fence_proxy_async();
      __syncthreads();
      if (tid == 0) {
        tma::store(Tw + (size_t)r0 * n, Tb2 + (size_t)b * cstride2, (uint32_t)((size_t)(r1 - r0) * n * sizeof(double)));
        tma::store_commit();
        if (w1 >= 0 && c >= 1 && c - 1 + SP < NCH) {
          tma::store_wait_read<1>();   // chunk c-1 has left shared memory: its buffer takes chunk c-1+SP of the next walker
          load_chunk(w1, c - 1 + SP, g0 + NCH + c - 1 + SP);
        }
      }
    }
    w = w1;
  }
  asm volatile("cp.async.wait_group 0;" ::: "memory");
  if (tid == 0) tma::store_wait_all<0>();
}

// ---------------------------------------------------------------- register-resident update, fp64 k = 1
// pf_resident_k1_kernel is bound by shared-memory bandwidth (every row crosses the LSU pipe
// three times: column sums, update load, update store, plus the bulk store reading it out
// again).  Here the inverse of a walker (N = 128: 128 KB = half the register file) is held
// in REGISTERS between the column sums and the update: 512 threads, lane l of warp rg owns
// the column pairs {l, l+32, ..} of rows rg, rg+16, ..  Shared memory is only the landing
// zone of the bulk loads: each row is read from it once, the updated row goes straight from
// registers to global memory with coalesced 16-byte stores, and the landing zone is free for
// the NEXT walker's bulk loads as soon as the column sums are done (they then have the whole
// reduction + update to arrive).  No barrier inside the update, no store staging.
template <int N>
__global__ void __launch_bounds__(512, 1) pf_regs_k1_kernel(State st) {
  constexpr int NQ = N / 2, QL = NQ / 32, RG = 16, RPT = N / RG, NCH = 4, RPC = N / NCH, TPC = RPT / NCH;
  constexpr int STG = 2 * N + 6;        // doubles per staging slot: N row, C row, R'^-1 (2x2), {slot index, next walker}
  extern __shared__ __align__(128) unsigned char smem_raw[];
  const int kmax = st.kmax;
  const int tid = threadIdx.x, lane = tid & 31, rg = tid >> 5;
  double2* Ts2 = (double2*)smem_raw;                       // [N][NQ]    landing zone
  double2* part = Ts2 + (size_t)N * NQ;                    // [RG][NQ]   column sums per row group
  double2* part2 = part + (size_t)RG * NQ;                 // [4][NQ]    ... per four row groups
  double2* rowc = part2 + (size_t)4 * NQ;                  // [N][2]     {g0,g1},{y0,y1} of row r
  double* stg = (double*)(rowc + (size_t)2 * N);           // [2][STG]
  __shared__ __align__(8) uint64_t bar[NCH];
  const int count = st.counters[0], grid = (int)gridDim.x;
  if (tid == 0) {
    for (int c = 0; c < NCH; ++c) tma::mbar_init(&bar[c], 1);
    tma::fence_barrier_init();
  }
  __syncthreads();
  auto load_walker = [&](int w) {   // thread 0 only
    constexpr uint32_t bytes = (uint32_t)(RPC * N * sizeof(double));
    for (int c = 0; c < NCH; ++c) {
      tma::mbar_arrive_expect_tx(&bar[c], bytes);
      tma::load(Ts2 + (size_t)c * RPC * NQ, (const double*)st.Ti + (size_t)w * N * N + (size_t)c * RPC * N, bytes, &bar[c]);
    }
  };
  auto stage = [&](int w, int slot, const int* next) {   // small operands of walker w -> staging slot
    double* d = stg + slot * STG;
    const double* Rw = (const double*)st.pend_Rinv + (size_t)w * st.kc * st.kc;
    if (tid < NQ) cp_async16(d + 2 * tid, (const double*)st.pend_N + (size_t)w * kmax * N + 2 * tid);
    else if (tid < 2 * NQ) cp_async16(d + N + 2 * (tid - NQ), (const double*)st.pend_C + (size_t)w * kmax * N + 2 * (tid - NQ));
    else if (tid == 2 * NQ) cp_async16(d + 2 * N, Rw);
    else if (tid == 2 * NQ + 1) cp_async16(d + 2 * N + 2, Rw + st.kc);
    else if (tid == 2 * NQ + 2) cp_async4(d + 2 * N + 4, st.pend_idx + (size_t)w * kmax);
    else if (tid == 2 * NQ + 3 && next) cp_async4((int*)(d + 2 * N + 4) + 1, next);   // walker after w in this CTA's sequence
  };
  int w = (int)blockIdx.x < count ? st.list[blockIdx.x] : -1;
  if (w >= 0) {
    if (tid == 0) load_walker(w);
    stage(w, 0, (int)blockIdx.x + grid < count ? st.list + blockIdx.x + grid : nullptr);
  }
  asm volatile("cp.async.commit_group;" ::: "memory");
  int j = 0;
  for (int it = blockIdx.x; it < count; it += grid, ++j) {
    const int slot = j & 1;
    double2* Tw2 = (double2*)((double*)st.Ti + (size_t)w * N * N);
    asm volatile("cp.async.wait_group 0;" ::: "memory");
    __syncthreads();
    const double* sd = stg + slot * STG;
    const int w1 = it + grid < count ? *((const int*)(sd + 2 * N + 4) + 1) : -1;
    if (w1 >= 0) stage(w1, slot ^ 1, it + 2 * grid < count ? st.list + it + 2 * grid : nullptr);
    asm volatile("cp.async.commit_group;" ::: "memory");
    double2 y1q[QL];
#pragma unroll
    for (int u = 0; u < QL; ++u) y1q[u] = ((const double2*)(sd + N))[lane + 32 * u];
    // ---- rows -> registers, chunk by chunk as the bulk copies land, with the column sums
    // y[c] = -sum_j Ti[j][c] N[j] taken on the way
    double2 x[RPT][QL], acc[QL];
#pragma unroll
    for (int u = 0; u < QL; ++u) acc[u] = make_double2(0.0, 0.0);
#pragma unroll
    for (int c = 0; c < NCH; ++c) {
      tma::mbar_wait(&bar[c], (uint32_t)(j & 1));
#pragma unroll
      for (int tt = 0; tt < TPC; ++tt) {
        const int t = c * TPC + tt, r = rg + RG * t;
        const double nr = sd[r];
#pragma unroll
        for (int u = 0; u < QL; ++u) {
          x[t][u] = Ts2[r * NQ + lane + 32 * u];
          acc[u].x = fma(x[t][u].x, nr, acc[u].x);
          acc[u].y = fma(x[t][u].y, nr, acc[u].y);
        }
      }
    }
#pragma unroll
    for (int u = 0; u < QL; ++u) part[rg * NQ + lane + 32 * u] = acc[u];
    __syncthreads();
    // every row is in registers: the landing zone takes the next walker
    if (tid == 0 && w1 >= 0) load_walker(w1);
    if (rg < 4) {
#pragma unroll
      for (int u = 0; u < QL; ++u) {
        const int q = lane + 32 * u;
        double2 sum = part[(4 * rg) * NQ + q];
#pragma unroll
        for (int g = 1; g < 4; ++g) {
          const double2 t = part[(4 * rg + g) * NQ + q];
          sum.x += t.x;
          sum.y += t.y;
        }
        part2[rg * NQ + q] = sum;
      }
    }
    __syncthreads();
    double2 y0q[QL], ng0[QL], ng1[QL];
    {
      const double Ri00 = sd[2 * N], Ri01 = sd[2 * N + 1], Ri10 = sd[2 * N + 2], Ri11 = sd[2 * N + 3];
      const int p0 = *(const int*)(sd + 2 * N + 4);
#pragma unroll
      for (int u = 0; u < QL; ++u) {
        const int q = lane + 32 * u;
        double2 sum = part2[q];
#pragma unroll
        for (int g = 1; g < 4; ++g) {
          const double2 t = part2[g * NQ + q];
          sum.x += t.x;
          sum.y += t.y;
        }
        y0q[u].x = (2 * q == p0) ? -sum.x + 1.0 : -sum.x;
        y0q[u].y = (2 * q + 1 == p0) ? -sum.y + 1.0 : -sum.y;
        double2 g0q, g1q;
        g0q.x = fma(y1q[u].x, Ri10, y0q[u].x * Ri00);
        g0q.y = fma(y1q[u].y, Ri10, y0q[u].y * Ri00);
        g1q.x = fma(y1q[u].x, Ri11, y0q[u].x * Ri01);
        g1q.y = fma(y1q[u].y, Ri11, y0q[u].y * Ri01);
        if (rg == 0) {
          rowc[4 * q + 0] = make_double2(g0q.x, g1q.x);
          rowc[4 * q + 1] = make_double2(y0q[u].x, y1q[u].x);
          rowc[4 * q + 2] = make_double2(g0q.y, g1q.y);
          rowc[4 * q + 3] = make_double2(y0q[u].y, y1q[u].y);
        }
        ng0[u] = make_double2(-g0q.x, -g0q.y);
        ng1[u] = make_double2(-g1q.x, -g1q.y);
      }
    }
    __syncthreads();
    // ---- rank-2 update (Eq. 22) in registers, rows stored straight to global memory
#pragma unroll
    for (int t = 0; t < RPT; ++t) {
      const int r = rg + RG * t;
      const double2 gr = rowc[2 * r], yr = rowc[2 * r + 1];
#pragma unroll
      for (int u = 0; u < QL; ++u) {
        const int q = lane + 32 * u, c0 = 2 * q;
        double2 v = x[t][u];
        if (c0 + 1 < r) {            // both below the diagonal
          v.x = fma(ng1[u].x, yr.y, fma(ng0[u].x, yr.x, v.x));
          v.y = fma(ng1[u].y, yr.y, fma(ng0[u].y, yr.x, v.y));
        } else if (c0 > r) {         // both above
          v.x = fma(gr.y, y1q[u].x, fma(gr.x, y0q[u].x, v.x));
          v.y = fma(gr.y, y1q[u].y, fma(gr.x, y0q[u].y, v.y));
        } else if (c0 == r) {        // (r,r), (r,r+1)
          v.x = 0.0;
          v.y = fma(gr.y, y1q[u].y, fma(gr.x, y0q[u].y, v.y));
        } else {                     // (r,r-1), (r,r)
          v.x = fma(ng1[u].x, yr.y, fma(ng0[u].x, yr.x, v.x));
          v.y = 0.0;
        }
        Tw2[r * NQ + q] = v;
      }
    }
    w = w1;
  }
  asm volatile("cp.async.wait_group 0;" ::: "memory");
}

// ---------------------------------------------------------------- delayed append (a6)
// Abuf[fill+alpha][:] = Y'[alpha][:]  (a'_tau, Eq. 28), Bbuf[fill+beta][:] = (a'_tau R'^-1)[:, beta].
template <typename T>
__global__ void __launch_bounds__(256) pf_append_kernel(State st, int k) {
  using S = Sc<T>;
  __shared__ T Ri[kMaxC * kMaxC];
  __shared__ int P[kMaxK];
  const int n = st.n, kmax = st.kmax, cap = st.cap, m = 2 * k;
  const int tid = threadIdx.x;
  const int count = st.counters[0];
  for (int it = blockIdx.x; it < count; it += gridDim.x) {
    const int w = st.list[it];
    const int fill = st.fill[w];
    __syncthreads();
    for (int q = tid; q < m * m; q += 256)
      Ri[(q / m) * kMaxC + (q % m)] = ((const T*)st.pend_Rinv)[(size_t)w * st.kc * st.kc + (q / m) * st.kc + (q % m)];
    if (tid < k) P[tid] = st.pend_idx[(size_t)w * kmax + tid];
    __syncthreads();
    const T* pC = (const T*)st.pend_C + (size_t)w * kmax * n;
    const T* pY = (const T*)st.pend_Y + (size_t)w * kmax * n;
    T* Ab = (T*)st.Abuf + (size_t)w * cap * n;
    T* Bb = (T*)st.Bbuf + (size_t)w * cap * n;
    for (int i = tid; i < n; i += 256) {
      T yp[kMaxC];
      for (int alpha = 0; alpha < m; ++alpha) {
        yp[alpha] = yprime(pY, pC, P, k, n, alpha, i);
        Ab[(size_t)(fill + alpha) * n + i] = yp[alpha];
      }
      for (int beta = 0; beta < m; ++beta) {
        T g = S::zero();
        for (int alpha = 0; alpha < m; ++alpha) g = S::fma(yp[alpha], Ri[alpha * kMaxC + beta], g);
        Bb[(size_t)(fill + beta) * n + i] = g;
      }
    }
  }
}

// ---------------------------------------------------------------- launchers
// Every choice below depends on the shape (dtype, n, k, K) only.
template <typename T>
static int launch_y(const State& st, int k, int use_list, Ctx& cx, cudaStream_t s) {
  ProfScope ps(&cx.prof, LRUX_PROF_YPASS, s);
  int nl = 0;
  if (st.cap) {
    pf_an_kernel<T><<<persistent_grid(cx.num_sms, 4, st.W), 256, 0, s>>>(st, k, use_list); ++nl;
  }
  const int kt = round_kt(k);
  if (sizeof(T) == 8 && !st.cap && k >= LRUX_PF_Y_ROWDOT_MIN_K && (st.n & 1) == 0) {
    // real data, K = 0, k >= 3: by skewness Y[a][i] = sum_j Ti[i][j] N[a][j] is the row-dot
    // contraction of lrux_rowdot.cu on the FP64 tensor pipe (the column-sum kernel spends k
    // DFMAs and k shared-memory operands per element: 0.68 of its k = 2 rate at k = 4)
    RowdotArgs A{};
    A.X = (const double*)st.Ti;      A.x_stride = (size_t)st.n * st.n;        A.rows = st.n;  A.ldx = st.n;
    A.N = (const double*)st.pend_N;  A.n_stride = (size_t)st.kmax * st.n;     A.ldn = st.n;
    A.n = st.n;  A.k = k;
    A.out = (double*)st.pend_Y;      A.o_stride = (size_t)st.kmax * st.n;     A.ldo = st.n;
    A.list = use_list ? st.list : nullptr;  A.count = use_list ? st.counters : nullptr;  A.W = st.W;
    A.idx = nullptr;  A.idx_stride = 0;
    const int r = launch_rowdot_dmma(A, cx, s);
    if (r < 0) return -1;
    if (r > 0) {
      cx.name(LRUX_PROF_YPASS, "rowdot_dmma_kernel");
      return nl + r;
    }
  }
  {
    // column sums (no warp reductions) whenever N fits in shared memory
    constexpr int VE = sizeof(T) == 8 ? 2 : 1;
    const int nvec = st.n / VE;
    int lg = 5;
    while ((1 << lg) < nvec && lg < 8) ++lg;
    const int CW = 1 << lg, RG = 256 >> lg, cblocks = (nvec + CW - 1) / CW;
    const size_t smy = (size_t)k * st.n * sizeof(T) + (RG > 1 ? (size_t)RG * kt * CW * 16 : 0);
    if (st.n % VE == 0 && smy <= 64 * 1024) {
      auto kern = kt == 1 ? pf_y_colsum_kernel<T, 1> : kt == 2 ? pf_y_colsum_kernel<T, 2>
                : kt == 4 ? pf_y_colsum_kernel<T, 4> : pf_y_colsum_kernel<T, 8>;
      if (cx.configure((const void*)kern, 256, smy) < 0) return -1;
      kern<<<persistent_grid(cx.num_sms, 8, (int64_t)st.W * cblocks), 256, smy, s>>>(st, k, cblocks, lg, use_list);
      cx.name(LRUX_PROF_YPASS, "pf_y_colsum_kernel");
      return nl + 1;
    }
  }
  int rpt = 64;
  if (rpt > st.n) rpt = st.n;
  const int tiles = (st.n + rpt - 1) / rpt;
  const int grid = persistent_grid(cx.num_sms, 4, (int64_t)st.W * tiles);
  const size_t smem = (size_t)kt * rpt * sizeof(T);
  switch (kt) {
    case 1: pf_y_kernel<T, 1><<<grid, 256, smem, s>>>(st, k, tiles, rpt, use_list); break;
    case 2: pf_y_kernel<T, 2><<<grid, 256, smem, s>>>(st, k, tiles, rpt, use_list); break;
    case 4: pf_y_kernel<T, 4><<<grid, 256, smem, s>>>(st, k, tiles, rpt, use_list); break;
    default: pf_y_kernel<T, 8><<<grid, 256, smem, s>>>(st, k, tiles, rpt, use_list); break;
  }
  cx.name(LRUX_PROF_YPASS, "pf_y_kernel");
  return nl + 1;
}

template <typename T>
static int pf_ratio_impl(const State& st, int k, const int32_t* idx, const void* rows, void* ratio,
                         Ctx& cx, cudaStream_t s) {
  int nl = 0;
  {
    ProfScope ps(&cx.prof, LRUX_PROF_RATIO, s);
    pf_gather_kernel<T><<<(unsigned)st.W, 128, 0, s>>>(st, k, idx, (const T*)rows, (T*)ratio); ++nl;
    cx.name(LRUX_PROF_RATIO, "pf_gather_kernel");
  }
  if (k > 1) {
    const int r = launch_y<T>(st, k, 0, cx, s);
    if (r < 0) return -1;
    nl += r;
    ProfScope ps(&cx.prof, LRUX_PROF_RATIO, s);
    pf_core_kernel<T><<<(unsigned)st.W, 128, 0, s>>>(st, k, (T*)ratio); ++nl;
    cx.name(LRUX_PROF_RATIO, "pf_gather_kernel+pf_core_kernel");
  }
  return cudaGetLastError() == cudaSuccess ? nl : -1;
}

template <typename T>
static int pf_flush_impl(const State& st, bool all, Ctx& cx, cudaStream_t s) {
  int nl = 0;
  if (all) nl += launch_flush_select_all(st, s);
  {
    ProfScope ps(&cx.prof, LRUX_PROF_FLUSH, s);
    const int r = launch_flush_dmma(st, cx, s);   // Eq. 26 on the FP64 tensor path
    if (r < 0) return -1;
    nl += r;
  }
  nl += launch_flush_clear(st, s);
  return cudaGetLastError() == cudaSuccess ? nl : -1;
}

// Immediate update (K = 0) with the walker resident on chip.  Returns the number of
// launches, 0 when no resident kernel fits this shape, -1 on a CUDA error.
template <typename T>
static int launch_pf_resident(const State& st, int k, Ctx& cx, cudaStream_t s) {
  const int n = st.n;
  if (sizeof(T) == 8 && k == 1) {
    if (n == 128 || n == 64) {
      // the walker's inverse in registers between the column sums and the update
      const size_t smr = (size_t)n * n * 8 + (size_t)20 * (n / 2) * 16 + (size_t)n * 32 + (size_t)2 * (2 * n + 6) * 8;
      auto kern = n == 128 ? pf_regs_k1_kernel<128> : pf_regs_k1_kernel<64>;
      if (cx.configure((const void*)kern, 512, smr) < 0) return -1;
      ProfScope ps(&cx.prof, LRUX_PROF_UPDATE, s);
      kern<<<persistent_grid(cx.num_sms, 1, st.W), 512, smr, s>>>(st);
      cx.name(LRUX_PROF_UPDATE, "pf_regs_k1_kernel");
      return 1;
    }
    // the whole inverse in one CTA's shared memory: column-pair kernel, 1024 threads
    int lg1 = 5;
    while ((1 << lg1) < n / 2) ++lg1;
    const int rg1 = 1024 >> lg1;
    const size_t smx = (size_t)(rg1 + rg1 / 4) * (n / 2) * 16 + (size_t)n * 32 + (size_t)2 * (2 * n + 6) * 8;
    const size_t chunk = (size_t)((n + 3) / 4) * n * 8;
    const int nb = (6 * chunk + smx <= 226 * 1024) ? 6 : 5;   // two spare chunk buffers when they fit
    const size_t sm1 = nb * chunk + smx;
    if (lg1 <= 7 && sm1 <= 226 * 1024) {
      const bool c3 = (2 << lg1) == n && lg1 == 6;
      auto kern = c3 ? (nb == 6 ? pf_resident_k1_kernel<6, 6> : pf_resident_k1_kernel<6, 5>)
                     : (nb == 6 ? pf_resident_k1_kernel<0, 6> : pf_resident_k1_kernel<0, 5>);
      if (cx.configure((const void*)kern, 1024, sm1) < 0) return -1;
      ProfScope ps(&cx.prof, LRUX_PROF_UPDATE, s);
      kern<<<persistent_grid(cx.num_sms, 1, st.W), 1024, sm1, s>>>(st, lg1);
      cx.name(LRUX_PROF_UPDATE, "pf_resident_k1_kernel");
      return 1;
    }
  }
  // cluster-resident: CL CTAs share a walker; taken when a slab leaves room for >= 2 CTAs per SM.
  // fp64 k = 1: the column-pair kernel (n/2 <= 256 threads' worth of column pairs)
  const bool k1 = sizeof(T) == 8 && k == 1 && n <= 512;
  int lg = 5;
  while ((1 << lg) < n / 2) ++lg;
  for (int CL = 4; CL <= 8; CL *= 2) {
    const int rpc = (n + CL - 1) / CL;
    const size_t smc = k1 ? (size_t)rpc * n * 8 + (size_t)((256 >> lg) + 2 * CL) * (n / 2) * 16 + (size_t)n * 40
                          : ((size_t)rpc * n + (size_t)(6 * k + 1) * n) * sizeof(T);
    if (smc > (size_t)(CL == 4 ? 56 : 111) * 1024) continue;
    // unrolled instance when n/2 is a power of two and the slab splits evenly over the row groups
    const bool even = k1 && (2 << lg) == n && n % CL == 0 && rpc % (256 >> lg) == 0;
    const int rpt = even ? rpc / (256 >> lg) : 0;
    const void* kern = !k1 ? (const void*)pf_cluster_update_kernel<T>
                     : (lg == 6 && rpt == 8) ? (const void*)pf_cluster_k1_kernel<6, 8>
                     : (lg == 7 && rpt == 16) ? (const void*)pf_cluster_k1_kernel<7, 16>
                     : (lg == 5 && rpt == 2) ? (const void*)pf_cluster_k1_kernel<5, 2>
                     : (const void*)pf_cluster_k1_kernel<0, 0>;
    const int ncl = cx.configure_cluster(kern, 256, smc, CL);   // co-resident clusters on the whole GPU
    if (ncl < 1) return 0;
    cudaLaunchConfig_t cfg = {};
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeClusterDimension;
    attr[0].val.clusterDim.x = CL;
    attr[0].val.clusterDim.y = 1;
    attr[0].val.clusterDim.z = 1;
    cfg.blockDim = dim3(256);
    cfg.dynamicSmemBytes = smc;
    cfg.stream = s;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    cfg.gridDim = dim3((unsigned)(CL * (int)std::min<int64_t>(st.W, ncl)));
    ProfScope ps(&cx.prof, LRUX_PROF_UPDATE, s);
    State stc = st;
    int a1 = k1 ? lg : k, a2 = k == 1 ? 1 : 0;
    void* args3[3] = {&stc, &a1, &a2};
    if (cudaLaunchKernelExC(&cfg, kern, args3) != cudaSuccess) return -1;
    cx.name(LRUX_PROF_UPDATE, k1 ? "pf_cluster_k1_kernel" : "pf_cluster_update_kernel");
    return 1;
  }
  return 0;
}

template <typename T>
static int pf_accept_impl(const State& st, int k, const uint8_t* mask, Ctx& cx, cudaStream_t s) {
  int nl = launch_select(st, mask, s);
#if LRUX_PF_DMMA
  if (st.K == 0 && sizeof(T) == 8 && k >= LRUX_PF_DMMA_MIN_K && launch_pf_update_dmma(st, k, cx, s, true) > 0) {
    // real data, k >= 2 (Y is already in the pending area): 8-row strips on the FP64 tensor pipe
    ProfScope ps(&cx.prof, LRUX_PROF_UPDATE, s);
    const int r = launch_pf_update_dmma(st, k, cx, s);
    if (r < 0) return -1;
    if (r > 0) return cudaGetLastError() == cudaSuccess ? nl + r : -1;
  }
#endif
  if (st.K == 0) {
    const int r = launch_pf_resident<T>(st, k, cx, s);
    if (r < 0) return -1;
    if (r > 0) return cudaGetLastError() == cudaSuccess ? nl + r : -1;
  }
  if (k == 1) {   // Y only for accepted walkers
    const int r = launch_y<T>(st, k, 1, cx, s);
    if (r < 0) return -1;
    nl += r;
  }
  if (st.K == 0) {
    ProfScope ps(&cx.prof, LRUX_PROF_UPDATE, s);
    const size_t sm = 4 * (size_t)k * st.n * sizeof(T);   // Y' and g
    int rd = 0;
#if LRUX_PF_DMMA
    if (sizeof(T) == 8 && k < LRUX_PF_DMMA_MIN_K && launch_pf_update_dmma(st, k, cx, s, true) > 0) {   // k = 1 beyond the resident kernels
      rd = launch_pf_update_dmma(st, k, cx, s);
      if (rd < 0) return -1;
      nl += rd;
    }
#endif
    if (rd > 0) {
    } else if (sm <= 160 * 1024) {
      auto kern = k <= 1 ? pf_update_stream_kernel<T, 2> : k <= 2 ? pf_update_stream_kernel<T, 4>
                : k <= 4 ? pf_update_stream_kernel<T, 8> : pf_update_stream_kernel<T, 16>;
      const int occ = cx.configure((const void*)kern, 256, sm);
      if (occ < 0) return -1;
      const int rpt = 64, tiles = (st.n + rpt - 1) / rpt;
      kern<<<persistent_grid(cx.num_sms, occ, (int64_t)st.W * tiles), 256, sm, s>>>(st, k, tiles, rpt); ++nl;
      cx.name(LRUX_PROF_UPDATE, "pf_update_stream_kernel");
    } else {
      const int t1 = (st.n + 31) / 32;
      const int grid = persistent_grid(cx.num_sms, 4, (int64_t)st.W * (t1 * (t1 + 1) / 2));
      pf_update_kernel<T><<<grid, 256, 0, s>>>(st, k, t1); ++nl;
      cx.name(LRUX_PROF_UPDATE, "pf_update_kernel");
    }
  } else {
    {
      ProfScope ps(&cx.prof, LRUX_PROF_APPEND, s);
      pf_append_kernel<T><<<persistent_grid(cx.num_sms, 4, st.W), 256, 0, s>>>(st, k); ++nl;
      cx.name(LRUX_PROF_APPEND, "pf_append_kernel");
    }
    nl += launch_post(st, 2 * k, s);
    int r = pf_flush_impl<T>(st, false, cx, s);
    if (r < 0) return -1;
    nl += r;
  }
  return cudaGetLastError() == cudaSuccess ? nl : -1;
}

int launch_pf_ratio(const State& st, int k, const int32_t* d_idx, const void* d_rows, void* d_ratio,
                    Ctx& cx, cudaStream_t s) {
  return st.dt == LRUX_F64 ? pf_ratio_impl<double>(st, k, d_idx, d_rows, d_ratio, cx, s)
                           : pf_ratio_impl<cplx>(st, k, d_idx, d_rows, d_ratio, cx, s);
}
int launch_pf_accept(const State& st, int k, const uint8_t* d_mask, Ctx& cx, cudaStream_t s) {
  return st.dt == LRUX_F64 ? pf_accept_impl<double>(st, k, d_mask, cx, s)
                           : pf_accept_impl<cplx>(st, k, d_mask, cx, s);
}
int launch_pf_flush(const State& st, bool all, Ctx& cx, cudaStream_t s) {
  return st.dt == LRUX_F64 ? pf_flush_impl<double>(st, all, cx, s) : pf_flush_impl<cplx>(st, all, cx, s);
}

}  // namespace lrux
