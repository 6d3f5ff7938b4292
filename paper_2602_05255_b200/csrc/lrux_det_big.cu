// Determinant row replacement of rank 8 < k <= 64 (the effective rank of
// a low-rank update inside neural-network backflow = orbital changes + backflow rank,
// PAPER.md:19), float64, immediate updates.  At these ranks the work is dense contractions,
// so every O(n k^2) / O(n^2 k) step runs on the FP64 tensor pipe:
//
//   ratio   C = A^-1[:,P] (k rows of Ti, gathered), R = N C (Eq. 4):
//           rowdot_dmma_kernel with X = C;  r = det R and R^-1 by Gauss-Jordan elimination with
//           partial pivoting in shared memory (Eq. 3)
//   accept  D = N A^-1 - I[P,:] = u^T A^-1 : rowdot_dmma_kernel with X = Ti, one read-only pass;
//           B = R^-1 D;  A^-1 -= C^T-side product (Eq. 5) = the delay-buffer fold
//           of Eq. 12 with k columns: flush_dmma_kernel with the pending area as its panels.
// HBM traffic of an accepted update: 3 n^2 e (read, read, write) against the compulsory
// 2 n^2 e -- at k >= 16 the update is above the FP64 ridge (k/4 flop/B), not HBM-bound.
#include "lrux_common.cuh"
#include "lrux_internal.h"

namespace lrux {

// ---------------------------------------------------------------- gather + validation
template <typename T>
__global__ void __launch_bounds__(256)
big_gather_kernel(State st, int k, const int32_t* __restrict__ idx, const T* __restrict__ rows) {
  __shared__ int sP[kBigMaxK];
  __shared__ int bad;
  const int w = blockIdx.x, tid = threadIdx.x;
  const int n = st.n, kmax = st.kmax;
  if (w == 0 && tid == 0) st.counters[0] = 0;
  if (tid == 0) bad = 0;
  if (tid < k) sP[tid] = idx[(size_t)w * k + tid];
  __syncthreads();
  if (tid < k) {
    const int p = sP[tid];
    bool b = p < 0 || p >= n;
    for (int c = 0; c < tid; ++c) b = b || sP[c] == p;
    if (b) bad = 1;
  }
  __syncthreads();
  if (tid < k) st.pend_idx[(size_t)w * kmax + tid] = bad ? -1 : sP[tid];
  if (bad) return;
  const T* Tw = (const T*)st.Ti + (size_t)w * n * n;
  T* pC = (T*)st.pend_C + (size_t)w * kmax * n;
  T* pN = (T*)st.pend_N + (size_t)w * kmax * n;
  for (int a = 0; a < k; ++a) {
    const T* src = Tw + (size_t)sP[a] * n;
    for (int i = tid; i < n; i += 256) {
      pC[(size_t)a * n + i] = src[i];
      pN[(size_t)a * n + i] = rows[((size_t)w * k + a) * n + i];
    }
  }
}

// ---------------------------------------------------------------- k x k core: det, inverse
// One CTA per walker; R (k x k, leading dimension k, in pend_Rinv) is inverted in place in
// shared memory by Gauss-Jordan elimination with partial pivoting (largest modulus, lowest
// index on ties); r = product of the pivots with the sign of the row exchanges.
template <typename T>
__global__ void __launch_bounds__(256) big_core_kernel(State st, int k, T* __restrict__ ratio_out) {
  using S = Sc<T>;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const int ld = k + 1;
  T* M = (T*)smem_raw;                 // [k][ld]
  T* prow = M + (size_t)k * ld;        // [k]
  T* colf = prow + k;                  // [k]
  int* piv = (int*)(colf + k);         // [k]
  __shared__ double bestv[8];
  __shared__ int besti[8];
  __shared__ int s_p, singular;
  const int w = blockIdx.x, tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int kmax = st.kmax;
  T* Rw = (T*)st.pend_Rinv + (size_t)w * st.kc * st.kc;
  if (st.pend_idx[(size_t)w * kmax] < 0) {   // invalid proposal
    if (tid == 0) {
      ratio_out[w] = S::nan();
      ((T*)st.pend_ratio)[w] = S::nan();
      st.pend_ok[w] = 0;
      atomicOr(&st.info[w], 2);
    }
    return;
  }
  for (int e = tid; e < k * k; e += 256) M[(e / k) * ld + e % k] = Rw[e];
  if (tid == 0) singular = 0;
  __syncthreads();
  T det = S::one();
  for (int c = 0; c < k; ++c) {
    // pivot
    double v = -1.0;
    int bi = 0x7fffffff;
    if (tid < 64 && c + tid < k) {
      v = S::abs2(M[(c + tid) * ld + c]);
      if (!(v == v)) v = -1.0;
      bi = c + tid;
    }
    if (warp < 2) {
#pragma unroll
      for (int m = 16; m > 0; m >>= 1) {
        const double ov = __shfl_xor_sync(0xffffffffu, v, m);
        const int oi = __shfl_xor_sync(0xffffffffu, bi, m);
        if (ov > v || (ov == v && oi < bi)) { v = ov; bi = oi; }
      }
      if (lane == 0) { bestv[warp] = v; besti[warp] = bi; }
    }
    __syncthreads();
    if (tid == 0) {
      double bv = bestv[0];
      int p = besti[0];
      if (bestv[1] > bv || (bestv[1] == bv && besti[1] < p)) { bv = bestv[1]; p = besti[1]; }
      if (!(bv > 0.0) || !isfinite(bv)) singular = 1;
      s_p = p;
      piv[c] = p;
    }
    __syncthreads();
    if (singular) break;
    const int p = s_p;
    if (tid < k) {               // swap rows c <-> p, keep the pivot row and the pivot column
      const T a = M[c * ld + tid], b = M[p * ld + tid];
      if (p != c) M[p * ld + tid] = a;
      prow[tid] = b;
    }
    __syncthreads();
    const T d = prow[c];
    const T dinv = S::inv(d);
    det = S::mul(det, d);
    if (p != c) det = S::neg(det);
    if (tid < k) colf[tid] = M[tid * ld + c];
    __syncthreads();
    if (tid < k) {
      const T x = (tid == c) ? dinv : S::mul(prow[tid], dinv);
      prow[tid] = x;
      M[c * ld + tid] = x;
    }
    __syncthreads();
    for (int e = tid; e < k * k; e += 256) {
      const int r = e / k, j = e % k;
      if (r == c) continue;
      const T x = (j == c) ? S::zero() : M[r * ld + j];
      M[r * ld + j] = S::fnma(colf[r], prow[j], x);
    }
    __syncthreads();
  }
  if (!singular) {
    for (int c = k - 1; c >= 0; --c) {   // undo the row exchanges: column swaps in reverse order
      const int p = piv[c];
      if (p != c) {
        if (tid < k) {
          const T a = M[tid * ld + c];
          M[tid * ld + c] = M[tid * ld + p];
          M[tid * ld + p] = a;
        }
        __syncthreads();
      }
    }
  }
  const bool ok = !singular && S::finite(det) && !S::is_zero(det);
  for (int e = tid; e < k * k; e += 256) Rw[e] = ok ? M[(e / k) * ld + e % k] : S::zero();
  if (tid == 0) {
    const T r = singular ? S::zero() : det;
    ratio_out[w] = r;
    ((T*)st.pend_ratio)[w] = r;
    st.pend_ok[w] = ok ? 1 : 0;
  }
}

// ---------------------------------------------------------------- B = R^-1 D, in place
// Work item = (accepted walker, block of 64 columns j): D[0..k)[j0..j0+64) is staged in shared
// memory, each thread forms 16 of the 64 x k outputs.  Item 0 of a walker also puts it on the
// fold list with k columns.
template <typename T>
__global__ void __launch_bounds__(256) big_bprep_kernel(State st, int k, int cblocks) {
  using S = Sc<T>;
  constexpr int CB = 64;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  T* Ri = (T*)smem_raw;               // [k][k]
  T* Ds = Ri + (size_t)k * k;         // [k][CB]
  const int n = st.n, kmax = st.kmax, tid = threadIdx.x;
  const int count = st.counters[0];
  if (blockIdx.x == 0 && tid == 0) st.counters[1] = count;
  int cur = -1;
  for (int item = blockIdx.x; item < count * cblocks; item += gridDim.x) {
    const int it = item / cblocks, cb = item % cblocks;
    const int w = st.list[it];
    __syncthreads();
    if (w != cur) {
      const T* Rw = (const T*)st.pend_Rinv + (size_t)w * st.kc * st.kc;
      for (int e = tid; e < k * k; e += 256) Ri[e] = Rw[e];
      cur = w;
    }
    if (cb == 0 && tid == 0) {
      st.flist[it] = w;
      st.fill[w] = k;
    }
    T* D = (T*)st.pend_D + (size_t)w * kmax * n;
    const int j0 = cb * CB;
    for (int e = tid; e < k * CB; e += 256) {
      const int b = e / CB, j = j0 + e % CB;
      Ds[e] = j < n ? D[(size_t)b * n + j] : S::zero();
    }
    __syncthreads();
    const int jj = tid % CB;
    if (j0 + jj < n) {
      for (int a = tid / CB; a < k; a += 256 / CB) {
        T acc = S::zero();
        for (int b = 0; b < k; ++b) acc = S::fma(Ri[a * k + b], Ds[b * CB + jj], acc);
        D[(size_t)a * n + j0 + jj] = acc;
      }
    }
  }
}

__global__ void big_done_kernel(State st) {
  const int it = blockIdx.x * blockDim.x + threadIdx.x;
  if (it < st.counters[1]) st.fill[st.flist[it]] = 0;
}

// ---------------------------------------------------------------- launchers
int launch_det_ratio_big(const State& st, int k, const int32_t* d_idx, const void* d_rows, void* d_ratio,
                         Ctx& cx, cudaStream_t s) {
  ProfScope ps(&cx.prof, LRUX_PROF_RATIO, s);
  big_gather_kernel<double><<<(unsigned)st.W, 256, 0, s>>>(st, k, d_idx, (const double*)d_rows);
  RowdotArgs A{};
  A.X = (const double*)st.pend_C;  A.x_stride = (size_t)st.kmax * st.n;  A.rows = k;  A.ldx = st.n;
  A.N = (const double*)st.pend_N;  A.n_stride = (size_t)st.kmax * st.n;  A.ldn = st.n;
  A.n = st.n;  A.k = k;
  A.out = (double*)st.pend_Rinv;   A.o_stride = (size_t)st.kc * st.kc;   A.ldo = k;
  A.W = st.W;
  const int r = launch_rowdot_dmma(A, cx, s);
  if (r <= 0) return -1;
  const size_t sm = ((size_t)k * (k + 1) + 2 * k) * sizeof(double) + (size_t)k * sizeof(int);
  if (cx.configure((const void*)big_core_kernel<double>, 256, sm) < 0) return -1;
  big_core_kernel<double><<<(unsigned)st.W, 256, sm, s>>>(st, k, (double*)d_ratio);
  cx.name(LRUX_PROF_RATIO, "big_gather_kernel+rowdot_dmma_kernel+big_core_kernel");
  return cudaGetLastError() == cudaSuccess ? 3 : -1;
}

int launch_det_accept_big(const State& st, int k, const uint8_t* mask, Ctx& cx, cudaStream_t s) {
  int nl = launch_select(st, mask, s);
  {
    ProfScope ps(&cx.prof, LRUX_PROF_UPDATE, s);
    RowdotArgs A{};
    A.X = (const double*)st.Ti;      A.x_stride = (size_t)st.n * st.n;     A.rows = st.n;  A.ldx = st.n;
    A.N = (const double*)st.pend_N;  A.n_stride = (size_t)st.kmax * st.n;  A.ldn = st.n;
    A.n = st.n;  A.k = k;
    A.out = (double*)st.pend_D;      A.o_stride = (size_t)st.kmax * st.n;  A.ldo = st.n;
    A.list = st.list;  A.count = st.counters;  A.W = st.W;
    A.idx = st.pend_idx;  A.idx_stride = st.kmax;
    const int r = launch_rowdot_dmma(A, cx, s);
    if (r <= 0) return -1;
    nl += r;
    const int cblocks = (st.n + 63) / 64;
    const size_t sm = ((size_t)k * k + (size_t)k * 64) * sizeof(double);
    if (cx.configure((const void*)big_bprep_kernel<double>, 256, sm) < 0) return -1;
    big_bprep_kernel<double><<<persistent_grid(cx.num_sms, 4, (int64_t)st.W * cblocks), 256, sm, s>>>(st, k, cblocks);
    ++nl;
    State v = st;            // the fold kernel sees the pending area as a k-deep delay buffer
    v.Abuf = st.pend_C;      // a = A^-1[:,P]
    v.Bbuf = st.pend_D;      // b = R^-1 u^T A^-1
    v.cap = st.kmax;
    const char* keep = cx.last[LRUX_PROF_FLUSH];
    const int rf = launch_flush_dmma(v, cx, s);
    cx.last[LRUX_PROF_FLUSH] = keep;
    if (rf < 0) return -1;
    nl += rf;
    cx.name(LRUX_PROF_UPDATE, "rowdot_dmma_kernel+big_bprep_kernel+flush_dmma_kernel");
  }
  big_done_kernel<<<(unsigned)((st.W + 255) / 256), 256, 0, s>>>(st);
  ++nl;
  return cudaGetLastError() == cudaSuccess ? nl : -1;
}

}  // namespace lrux
