// Shared device helpers for the lrux sm_100a kernels: scalar traits for
// float64 / complex128, warp reductions, small dense solves, the counter RNG.
#pragma once
#include <cuda_runtime.h>
#include <math.h>
#include <stdint.h>

#include "lrux.h"

namespace lrux {

constexpr int kMaxK = 8;   // largest rank of the register / shared-memory kernels (k > 8: lrux_det_big.cu)

// ---------------------------------------------------------------- scalars
// 16-byte aligned: one LDG.128 / STG.128 per element instead of two 8-byte accesses (the ncu
// capture of the complex flush showed 8 of every 32-byte sector used per store instruction).
// Every complex array at the ABI must therefore be 16-byte aligned (include/lrux.h).
#ifndef LRUX_CPLX_ALIGN
#define LRUX_CPLX_ALIGN 16
#endif
struct __align__(LRUX_CPLX_ALIGN) cplx {
  double re, im;
};

__device__ __forceinline__ double sc_from(double re, double, double) { return re; }
__device__ __forceinline__ cplx sc_from(double re, double im, cplx) { return cplx{re, im}; }
__device__ __forceinline__ double sc_re(double x) { return x; }
__device__ __forceinline__ double sc_im(double) { return 0.0; }
__device__ __forceinline__ double sc_re(cplx x) { return x.re; }
__device__ __forceinline__ double sc_im(cplx x) { return x.im; }

template <typename T>
struct Sc;

template <>
struct Sc<double> {
  using vec2 = double2;  // two consecutive elements
  static __device__ __forceinline__ double zero() { return 0.0; }
  static __device__ __forceinline__ double one() { return 1.0; }
  static __device__ __forceinline__ double from_real(double x) { return x; }
  static __device__ __forceinline__ double mul(double a, double b) { return a * b; }
  static __device__ __forceinline__ double fma(double a, double b, double c) {
    return ::fma(a, b, c);
  }
  // c - a*b
  static __device__ __forceinline__ double fnma(double a, double b, double c) {
    return ::fma(-a, b, c);
  }
  static __device__ __forceinline__ double add(double a, double b) { return a + b; }
  static __device__ __forceinline__ double sub(double a, double b) { return a - b; }
  static __device__ __forceinline__ double neg(double a) { return -a; }
  static __device__ __forceinline__ double abs2(double a) { return a * a; }
  static __device__ __forceinline__ double abs(double a) { return fabs(a); }
  static __device__ __forceinline__ double inv(double a) { return 1.0 / a; }
  static __device__ __forceinline__ double div(double a, double b) { return a / b; }
  static __device__ __forceinline__ double scale(double a, double s) { return a * s; }
  // a / |a| given |a|: exactly +-1 for real data
  static __device__ __forceinline__ double unit(double a, double) { return copysign(1.0, a); }
  static __device__ __forceinline__ bool is_zero(double a) { return a == 0.0; }
  static __device__ __forceinline__ bool finite(double a) { return isfinite(a); }
  static __device__ __forceinline__ double nan() { return __longlong_as_double(0x7ff8000000000000LL); }
  static __device__ __forceinline__ double shfl_xor(double v, int m) {
    return __shfl_xor_sync(0xffffffffu, v, m);
  }
  static __device__ __forceinline__ double shfl(double v, int src) {
    return __shfl_sync(0xffffffffu, v, src);
  }
};

template <>
struct Sc<cplx> {
  static __device__ __forceinline__ cplx zero() { return cplx{0.0, 0.0}; }
  static __device__ __forceinline__ cplx one() { return cplx{1.0, 0.0}; }
  static __device__ __forceinline__ cplx from_real(double x) { return cplx{x, 0.0}; }
  static __device__ __forceinline__ cplx mul(cplx a, cplx b) {
    return cplx{::fma(a.re, b.re, -a.im * b.im), ::fma(a.re, b.im, a.im * b.re)};
  }
  static __device__ __forceinline__ cplx fma(cplx a, cplx b, cplx c) {
    return cplx{::fma(-a.im, b.im, ::fma(a.re, b.re, c.re)),
                ::fma(a.im, b.re, ::fma(a.re, b.im, c.im))};
  }
  static __device__ __forceinline__ cplx fnma(cplx a, cplx b, cplx c) {
    return cplx{::fma(a.im, b.im, ::fma(-a.re, b.re, c.re)),
                ::fma(-a.im, b.re, ::fma(-a.re, b.im, c.im))};
  }
  static __device__ __forceinline__ cplx add(cplx a, cplx b) { return cplx{a.re + b.re, a.im + b.im}; }
  static __device__ __forceinline__ cplx sub(cplx a, cplx b) { return cplx{a.re - b.re, a.im - b.im}; }
  static __device__ __forceinline__ cplx neg(cplx a) { return cplx{-a.re, -a.im}; }
  static __device__ __forceinline__ double abs2(cplx a) { return ::fma(a.re, a.re, a.im * a.im); }
  static __device__ __forceinline__ double abs(cplx a) { return hypot(a.re, a.im); }
  static __device__ __forceinline__ cplx inv(cplx a) {
    // Smith's algorithm: no spurious overflow
    if (fabs(a.re) >= fabs(a.im)) {
      double t = a.im / a.re, d = a.re + a.im * t;
      return cplx{1.0 / d, -t / d};
    }
    double t = a.re / a.im, d = a.re * t + a.im;
    return cplx{t / d, -1.0 / d};
  }
  static __device__ __forceinline__ cplx div(cplx a, cplx b) { return mul(a, inv(b)); }
  static __device__ __forceinline__ cplx scale(cplx a, double s) { return cplx{a.re * s, a.im * s}; }
  static __device__ __forceinline__ cplx unit(cplx a, double abs_a) {
    return cplx{a.re / abs_a, a.im / abs_a};
  }
  static __device__ __forceinline__ bool is_zero(cplx a) { return a.re == 0.0 && a.im == 0.0; }
  static __device__ __forceinline__ bool finite(cplx a) { return isfinite(a.re) && isfinite(a.im); }
  static __device__ __forceinline__ cplx nan() {
    double q = __longlong_as_double(0x7ff8000000000000LL);
    return cplx{q, q};
  }
  static __device__ __forceinline__ cplx shfl_xor(cplx v, int m) {
    return cplx{__shfl_xor_sync(0xffffffffu, v.re, m), __shfl_xor_sync(0xffffffffu, v.im, m)};
  }
  static __device__ __forceinline__ cplx shfl(cplx v, int src) {
    return cplx{__shfl_sync(0xffffffffu, v.re, src), __shfl_sync(0xffffffffu, v.im, src)};
  }
};

template <typename T>
__device__ __forceinline__ T warp_sum(T v) {
#pragma unroll
  for (int m = 16; m > 0; m >>= 1) v = Sc<T>::add(v, Sc<T>::shfl_xor(v, m));
  return v;
}

// ---------------------------------------------------------------- small dense
// In-place LU with partial pivoting of a k x k matrix (row-major, leading
// dimension ld) executed by ONE thread; returns det, leaves the inverse in `inv`
// (row-major, ld).  k <= 2*kMaxK.  ok=false when a pivot is zero / non-finite.
template <typename T>
__device__ inline T small_det_inv(T* a, T* inv, int k, int ld, bool* ok) {
  using S = Sc<T>;
  T det = S::one();
  *ok = true;
  for (int i = 0; i < k; ++i)
    for (int j = 0; j < k; ++j) inv[i * ld + j] = (i == j) ? S::one() : S::zero();
  for (int c = 0; c < k; ++c) {
    int p = c;
    double best = S::abs2(a[c * ld + c]);
    for (int r = c + 1; r < k; ++r) {
      double v = S::abs2(a[r * ld + c]);
      if (v > best) { best = v; p = r; }
    }
    if (!(best > 0.0) || !isfinite(best)) { *ok = false; return S::zero(); }
    if (p != c) {
      for (int j = 0; j < k; ++j) {
        T t = a[c * ld + j]; a[c * ld + j] = a[p * ld + j]; a[p * ld + j] = t;
        t = inv[c * ld + j]; inv[c * ld + j] = inv[p * ld + j]; inv[p * ld + j] = t;
      }
      det = S::neg(det);
    }
    T d = a[c * ld + c];
    det = S::mul(det, d);
    T di = S::inv(d);
    for (int j = 0; j < k; ++j) {
      a[c * ld + j] = S::mul(a[c * ld + j], di);
      inv[c * ld + j] = S::mul(inv[c * ld + j], di);
    }
    for (int r = 0; r < k; ++r) {
      if (r == c) continue;
      T f = a[r * ld + c];
      for (int j = 0; j < k; ++j) {
        a[r * ld + j] = S::fnma(f, a[c * ld + j], a[r * ld + j]);
        inv[r * ld + j] = S::fnma(f, inv[c * ld + j], inv[r * ld + j]);
      }
    }
  }
  if (!S::finite(det)) *ok = false;
  return det;
}

// The same elimination executed by ONE WARP (all 32 lanes call it; a, inv in shared memory):
// lane l < 2k owns column l of the augmented matrix [a | inv].  Every element goes through the
// operations of small_det_inv in the same order, so det and inv are bit-identical to the
// serial routine -- at k = 8 the serial one was the longest phase of the ratio kernel.
template <typename T, int KM = 2 * kMaxK>   // KM >= k: size of the per-lane multiplier array
__device__ inline T warp_det_inv(T* a, T* inv, int k, int ld, bool* ok, int lane) {
  using S = Sc<T>;
  const bool act = lane < 2 * k;
  T* col = lane < k ? a + lane : inv + (lane - k);   // this lane's column, stride ld
  if (act && lane >= k)
    for (int i = 0; i < k; ++i) col[i * ld] = (i == lane - k) ? S::one() : S::zero();
  __syncwarp();
  T det = S::one();
  bool good = true;
  for (int c = 0; c < k; ++c) {
    int p = c;
    double best = S::abs2(a[c * ld + c]);
    for (int r = c + 1; r < k; ++r) {
      const double v = S::abs2(a[r * ld + c]);
      if (v > best) { best = v; p = r; }
    }
    if (!(best > 0.0) || !isfinite(best)) { good = false; det = S::zero(); break; }   // uniform
    __syncwarp();
    if (p != c) {
      if (act) { const T t = col[c * ld]; col[c * ld] = col[p * ld]; col[p * ld] = t; }
      det = S::neg(det);
      __syncwarp();
    }
    const T d = a[c * ld + c];
    det = S::mul(det, d);
    const T di = S::inv(d);
    __syncwarp();                      // every lane has d before lane c rescales it
    if (act) col[c * ld] = S::mul(col[c * ld], di);
    __syncwarp();
    T f[KM];
#pragma unroll
    for (int r = 0; r < KM; ++r) f[r] = r < k ? a[r * ld + c] : S::zero();
    __syncwarp();                      // ... and the multipliers before column c is eliminated
    if (act) {
      const T pc = col[c * ld];
#pragma unroll
      for (int r = 0; r < KM; ++r)
        if (r < k && r != c) col[r * ld] = S::fnma(f[r], pc, col[r * ld]);
    }
    __syncwarp();
  }
  if (good && !S::finite(det)) good = false;
  *ok = good;
  return det;
}

// Pfaffian of an exactly skew m x m matrix (m even, m <= 2*kMaxK) by
// Parlett-Reid elimination with pivoting, ONE thread, destroys `a`.
template <typename T>
__device__ inline T small_pf(T* a, int m, int ld) {
  using S = Sc<T>;
  T pf = S::one();
  for (int j = 0; j + 1 < m; j += 2) {
    int p = j + 1;
    double best = S::abs2(a[(j + 1) * ld + j]);
    for (int r = j + 2; r < m; ++r) {
      double v = S::abs2(a[r * ld + j]);
      if (v > best) { best = v; p = r; }
    }
    if (!(best > 0.0)) return S::zero();
    if (p != j + 1) {
      for (int c = 0; c < m; ++c) {
        T t = a[(j + 1) * ld + c]; a[(j + 1) * ld + c] = a[p * ld + c]; a[p * ld + c] = t;
      }
      for (int r = 0; r < m; ++r) {
        T t = a[r * ld + j + 1]; a[r * ld + j + 1] = a[r * ld + p]; a[r * ld + p] = t;
      }
      pf = S::neg(pf);
    }
    T piv = a[j * ld + j + 1];
    pf = S::mul(pf, piv);
    T pi = S::inv(piv);
    for (int r = j + 2; r < m; ++r) {
      for (int c = r + 1; c < m; ++c) {
        // A[r][c] += tau_r * col_c - col_r * tau_c, tau = A[j][.]/piv, col = A[.][j+1]
        T tr = S::mul(a[j * ld + r], pi), tc = S::mul(a[j * ld + c], pi);
        T v = a[r * ld + c];
        v = S::fma(tr, a[c * ld + j + 1], v);
        v = S::fnma(a[r * ld + j + 1], tc, v);
        a[r * ld + c] = v;
        a[c * ld + r] = S::neg(v);
      }
    }
  }
  return pf;
}

// small_pf executed by ONE WARP (all 32 lanes call it; `a` in shared memory).  The (r, c)
// updates of one elimination step are independent of each other, and the swaps keep the
// serial order (rows, then columns): bit-identical to small_pf.
template <typename T>
__device__ inline T warp_pf(T* a, int m, int ld, int lane) {
  using S = Sc<T>;
  T pf = S::one();
  for (int j = 0; j + 1 < m; j += 2) {
    int p = j + 1;
    double best = S::abs2(a[(j + 1) * ld + j]);
    for (int r = j + 2; r < m; ++r) {
      const double v = S::abs2(a[r * ld + j]);
      if (v > best) { best = v; p = r; }
    }
    if (!(best > 0.0)) return S::zero();   // uniform
    __syncwarp();
    if (p != j + 1) {
      if (lane < m) { const T t = a[(j + 1) * ld + lane]; a[(j + 1) * ld + lane] = a[p * ld + lane]; a[p * ld + lane] = t; }
      __syncwarp();
      if (lane < m) { const T t = a[lane * ld + j + 1]; a[lane * ld + j + 1] = a[lane * ld + p]; a[lane * ld + p] = t; }
      __syncwarp();
      pf = S::neg(pf);
    }
    const T piv = a[j * ld + j + 1];
    pf = S::mul(pf, piv);
    const T pi = S::inv(piv);
    for (int r = j + 2; r < m; ++r) {
      const int c = r + 1 + lane;
      if (c < m) {
        const T tr = S::mul(a[j * ld + r], pi), tc = S::mul(a[j * ld + c], pi);
        T v = a[r * ld + c];
        v = S::fma(tr, a[c * ld + j + 1], v);
        v = S::fnma(a[r * ld + j + 1], tc, v);
        a[r * ld + c] = v;
        a[c * ld + r] = S::neg(v);
      }
    }
    __syncwarp();
  }
  return pf;
}

// ---------------------------------------------------------------- counter RNG
// Same integer function as paper_2602_05255_b200/workload.py (splitmix64 finaliser).
__host__ __device__ __forceinline__ uint64_t mix64(uint64_t z) {
  z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ULL;
  z = (z ^ (z >> 27)) * 0x94D049BB133111EBULL;
  return z ^ (z >> 31);
}
__host__ __device__ __forceinline__ uint64_t rnd64(uint64_t seed, uint64_t w, uint64_t stream,
                                                   uint64_t ctr) {
  uint64_t h = mix64(seed ^ (stream * 0xD1342543DE82EF95ULL));
  h = mix64(h + w * 0x9E3779B97F4A7C15ULL);
  return mix64(h + (ctr + 1) * 0x9E3779B97F4A7C15ULL);
}
__device__ __forceinline__ double to_uniform(uint64_t bits) {
  return (double)(bits >> 11) * 0x1.0p-53;
}
__device__ __forceinline__ uint32_t to_below(uint64_t bits, uint32_t m) {
  return (uint32_t)__umul64hi(bits, (uint64_t)m);
}

}  // namespace lrux
