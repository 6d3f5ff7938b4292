// General rank-k determinant updates: A' = A + v u^T with each factor
// in the paper's tuple form -- kd dense columns followed by ke one-hot columns
// (Eq. 6-9; dense u, v as in Eq. 2-5).
//
//   UA  = u^T A^-1   (k x n)     dense column x:  UA[a][j]  = sum_i x[i] Ti[j][i]   (row dots, one pass)
//                                one-hot e_p:     UA[a][j]  = Ti[j][p]               (O(n) gather)
//   AVt = (A^-1 v)^T (k x n)     dense column y:  AVt[b][i] = sum_j Ti[j][i] y[j]   (column sums, one pass)
//                                one-hot e_p:     AVt[b][i] = Ti[p][i]               (a contiguous row)
//   R = 1 + UA v (Eq. 4), r = det R (Eq. 3)
//   accept:  A^-1 -= (A^-1 v) R^-1 (u^T A^-1)  (Eq. 5)  <=>  Ti[j][i] -= sum_s (R^-1 UA)[s][j] AVt[s][i]
// The update is exactly the shape of the delay-buffer fold (Eq. 12) with k columns, so it runs
// through flush_dmma_kernel on the FP64 tensor pipe with the pending area as its two panels.
// With dense factors the RATIO itself is an O(n^2 k) pass over the inverse.
#include "lrux_common.cuh"
#include "lrux_internal.h"

namespace lrux {

// ---------------------------------------------------------------- UA rows of dense u columns
// Work item = (walker, tile of 32 rows j); each warp takes 4 rows per pass so that one read of
// the x vectors (L1/L2) serves 4 rows.
template <typename T, int KD>
__global__ void __launch_bounds__(256)
gen_rowdot_kernel(State st, int kd, const T* __restrict__ dense, int tiles) {
  using S = Sc<T>;
  constexpr int RW = 4;
  const int n = st.n, kmax = st.kmax;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  for (int64_t item = blockIdx.x; item < st.W * tiles; item += gridDim.x) {
    const int w = (int)(item / tiles), tile = (int)(item % tiles);
    const T* Tw = (const T*)st.Ti + (size_t)w * n * n;
    const T* x = dense + (size_t)w * kd * n;
    T* UA = (T*)st.pend_N + (size_t)w * kmax * n;
    const int j0 = tile * 32 + warp * RW;
    if (j0 >= n) continue;
    T acc[RW][KD];
#pragma unroll
    for (int r = 0; r < RW; ++r)
#pragma unroll
      for (int a = 0; a < KD; ++a) acc[r][a] = S::zero();
    for (int i = lane; i < n; i += 32) {
      T t[RW];
#pragma unroll
      for (int r = 0; r < RW; ++r) t[r] = j0 + r < n ? Tw[(size_t)(j0 + r) * n + i] : S::zero();
#pragma unroll
      for (int a = 0; a < KD; ++a) {
        if (a < kd) {
          const T xv = x[(size_t)a * n + i];
#pragma unroll
          for (int r = 0; r < RW; ++r) acc[r][a] = S::fma(xv, t[r], acc[r][a]);
        }
      }
    }
#pragma unroll
    for (int r = 0; r < RW; ++r)
#pragma unroll
      for (int a = 0; a < KD; ++a) {
        if (a < kd) {
          const T v = warp_sum(acc[r][a]);
          if (lane == 0 && j0 + r < n) UA[(size_t)a * n + j0 + r] = v;
        }
      }
  }
}

// ---------------------------------------------------------------- AVt rows of dense v columns
// Work item = (walker, block of 256 columns i); thread per column, running sums down the
// rows (each warp load is a contiguous piece of a row), y broadcast from shared memory.
template <typename T, int KD>
__global__ void __launch_bounds__(256)
gen_colsum_kernel(State st, int kd, int k, const T* __restrict__ dense, int cblocks) {
  using S = Sc<T>;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  T* ys = (T*)smem_raw;   // [kd][n]
  const int n = st.n, kmax = st.kmax, tid = threadIdx.x;
  for (int64_t item = blockIdx.x; item < st.W * cblocks; item += gridDim.x) {
    const int w = (int)(item / cblocks), cb = (int)(item % cblocks);
    const T* Tw = (const T*)st.Ti + (size_t)w * n * n;
    const T* y = dense + (size_t)w * kd * n;
    T* AVt = (T*)st.pend_C + (size_t)w * kmax * n;
    __syncthreads();
    for (int qd = tid; qd < kd * n; qd += 256) ys[qd] = y[qd];
    __syncthreads();
    const int i = cb * 256 + tid;
    if (i >= n) continue;
    T acc[KD];
#pragma unroll
    for (int b = 0; b < KD; ++b) acc[b] = S::zero();
    constexpr int U = 4;
    for (int j0 = 0; j0 < n; j0 += U) {
      T t[U];
#pragma unroll
      for (int u = 0; u < U; ++u) t[u] = j0 + u < n ? Tw[(size_t)(j0 + u) * n + i] : S::zero();
#pragma unroll
      for (int u = 0; u < U; ++u) {
        if (j0 + u < n) {
#pragma unroll
          for (int b = 0; b < KD; ++b)
            if (b < kd) acc[b] = S::fma(t[u], ys[(size_t)b * n + j0 + u], acc[b]);
        }
      }
    }
#pragma unroll
    for (int b = 0; b < KD; ++b)
      if (b < kd) AVt[(size_t)b * n + i] = acc[b];
  }
  (void)k;
}

// ---------------------------------------------------------------- one-hot parts, core, ratio
// One CTA per walker: fills the UA / AVt rows of the one-hot columns, forms R = 1 + UA v
// (dense v column: a dot product over n; one-hot e_p: UA[a][p]), r = det R and R^-1.
template <typename T>
__global__ void __launch_bounds__(128)
gen_core_kernel(State st, int k, int u_kd, const int32_t* __restrict__ u_idx, int v_kd,
                const T* __restrict__ v_dense, const int32_t* __restrict__ v_idx,
                T* __restrict__ ratio_out) {
  using S = Sc<T>;
  __shared__ T Rs[kMaxK * kMaxK];
  __shared__ T Ri[kMaxK * kMaxK];
  __shared__ int pu[kMaxK], pv[kMaxK];
  __shared__ int bad;
  const int w = blockIdx.x, tid = threadIdx.x, nt = blockDim.x;
  const int warp = tid >> 5, lane = tid & 31, nw = nt >> 5;
  const int n = st.n, kmax = st.kmax;
  const int u_ke = k - u_kd, v_ke = k - v_kd;
  if (w == 0 && tid == 0) st.counters[0] = 0;
  if (tid == 0) {
    int b = 0;
    for (int a = 0; a < u_ke; ++a) {
      pu[a] = u_idx[(size_t)w * u_ke + a];
      if (pu[a] < 0 || pu[a] >= n) b = 1;
    }
    for (int a = 0; a < v_ke; ++a) {
      pv[a] = v_idx[(size_t)w * v_ke + a];
      if (pv[a] < 0 || pv[a] >= n) b = 1;
    }
    bad = b;
  }
  __syncthreads();
  if (bad) {
    if (tid == 0) {
      ratio_out[w] = S::nan();
      ((T*)st.pend_ratio)[w] = S::nan();
      st.pend_ok[w] = 0;
      atomicOr(&st.info[w], 2);
    }
    return;
  }
  const T* Tw = (const T*)st.Ti + (size_t)w * n * n;
  T* UA = (T*)st.pend_N + (size_t)w * kmax * n;
  T* AVt = (T*)st.pend_C + (size_t)w * kmax * n;
  for (int a = 0; a < u_ke; ++a)
    for (int j = tid; j < n; j += nt) UA[(size_t)(u_kd + a) * n + j] = Tw[(size_t)j * n + pu[a]];
  for (int b = 0; b < v_ke; ++b)
    for (int i = tid; i < n; i += nt) AVt[(size_t)(v_kd + b) * n + i] = Tw[(size_t)pv[b] * n + i];
  __syncthreads();   // this CTA's own global writes to UA are visible to its threads
  const T* y = v_kd ? v_dense + (size_t)w * v_kd * n : nullptr;
  for (int pr = warp; pr < k * k; pr += nw) {
    const int a = pr / k, b = pr % k;
    T acc = S::zero();
    if (b < v_kd) {
      for (int j = lane; j < n; j += 32) acc = S::fma(UA[(size_t)a * n + j], y[(size_t)b * n + j], acc);
      acc = warp_sum(acc);
    } else {
      acc = UA[(size_t)a * n + pv[b - v_kd]];
    }
    if (lane == 0) Rs[a * kMaxK + b] = a == b ? S::add(acc, S::one()) : acc;
  }
  __syncthreads();
  if (tid == 0) {
    bool ok;
    const T det = small_det_inv(Rs, Ri, k, kMaxK, &ok);
    ratio_out[w] = det;
    ((T*)st.pend_ratio)[w] = det;
    st.pend_ok[w] = ok ? 1 : 0;
    T* pR = (T*)st.pend_Rinv + (size_t)w * st.kc * st.kc;
    for (int a = 0; a < k; ++a)
      for (int b = 0; b < k; ++b) pR[a * st.kc + b] = Ri[a * kMaxK + b];
  }
}

// ---------------------------------------------------------------- accept
// Accepted walkers: UA <- R^-1 UA in place (column by column), and the walker is put on the
// fold list with k columns.
template <typename T>
__global__ void __launch_bounds__(256) gen_apply_prep_kernel(State st, int k) {
  using S = Sc<T>;
  __shared__ T Ri[kMaxK * kMaxK];
  const int n = st.n, kmax = st.kmax, tid = threadIdx.x;
  const int count = st.counters[0];
  if (blockIdx.x == 0 && tid == 0) st.counters[1] = count;
  for (int it = blockIdx.x; it < count; it += gridDim.x) {
    const int w = st.list[it];
    __syncthreads();
    if (tid < k * k) Ri[(tid / k) * kMaxK + tid % k] =
        ((const T*)st.pend_Rinv)[(size_t)w * st.kc * st.kc + (tid / k) * st.kc + tid % k];
    if (tid == 0) {
      st.flist[it] = w;
      st.fill[w] = k;
    }
    __syncthreads();
    T* UA = (T*)st.pend_N + (size_t)w * kmax * n;
    for (int j = tid; j < n; j += 256) {
      T d[kMaxK];
      for (int b = 0; b < k; ++b) d[b] = UA[(size_t)b * n + j];
      for (int a = 0; a < k; ++a) {
        T acc = S::zero();
        for (int b = 0; b < k; ++b) acc = S::fma(Ri[a * kMaxK + b], d[b], acc);
        UA[(size_t)a * n + j] = acc;
      }
    }
  }
}

// the fold list is reset by the next select / flush-all; only the column counts go back to 0
__global__ void gen_apply_done_kernel(State st) {
  const int it = blockIdx.x * blockDim.x + threadIdx.x;
  if (it < st.counters[1]) st.fill[st.flist[it]] = 0;
}

// ---------------------------------------------------------------- launchers
template <typename T>
static int ratio_general_t(const State& st, int k, int u_kd, const void* u_dense, const int32_t* u_idx,
                           int v_kd, const void* v_dense, const int32_t* v_idx, void* ratio, Ctx& cx,
                           cudaStream_t s) {
  ProfScope ps(&cx.prof, LRUX_PROF_RATIO, s);
  const int n = st.n;
  int nl = 0;
  if (u_kd > 0) {
    const int tiles = (n + 31) / 32;
    const int grid = persistent_grid(cx.num_sms, 8, (int64_t)st.W * tiles);
    switch (round_kt(u_kd)) {
      case 1: gen_rowdot_kernel<T, 1><<<grid, 256, 0, s>>>(st, u_kd, (const T*)u_dense, tiles); break;
      case 2: gen_rowdot_kernel<T, 2><<<grid, 256, 0, s>>>(st, u_kd, (const T*)u_dense, tiles); break;
      case 4: gen_rowdot_kernel<T, 4><<<grid, 256, 0, s>>>(st, u_kd, (const T*)u_dense, tiles); break;
      default: gen_rowdot_kernel<T, 8><<<grid, 256, 0, s>>>(st, u_kd, (const T*)u_dense, tiles); break;
    }
    ++nl;
  }
  if (v_kd > 0) {
    const int cblocks = (n + 255) / 256;
    const size_t sm = (size_t)v_kd * n * sizeof(T);
    const void* kern;
    switch (round_kt(v_kd)) {
      case 1: kern = (const void*)gen_colsum_kernel<T, 1>; break;
      case 2: kern = (const void*)gen_colsum_kernel<T, 2>; break;
      case 4: kern = (const void*)gen_colsum_kernel<T, 4>; break;
      default: kern = (const void*)gen_colsum_kernel<T, 8>; break;
    }
    const int occ = cx.configure(kern, 256, sm);
    if (occ < 0) return -1;
    State stc = st;
    int a1 = v_kd, a2 = k, a4 = cblocks;
    const void* dp = v_dense;
    void* args[5] = {&stc, &a1, &a2, &dp, &a4};
    if (cudaLaunchKernel(kern, dim3(persistent_grid(cx.num_sms, occ, (int64_t)st.W * cblocks)), dim3(256), args,
                         sm, s) != cudaSuccess)
      return -1;
    ++nl;
  }
  gen_core_kernel<T><<<(unsigned)st.W, 128, 0, s>>>(st, k, u_kd, u_idx, v_kd, (const T*)v_dense, v_idx, (T*)ratio);
  ++nl;
  cx.name(LRUX_PROF_RATIO, "gen_rowdot_kernel+gen_colsum_kernel+gen_core_kernel");
  return cudaGetLastError() == cudaSuccess ? nl : -1;
}

int launch_det_ratio_general(const State& st, int k, int u_kd, const void* u_dense, const int32_t* u_idx,
                             int v_kd, const void* v_dense, const int32_t* v_idx, void* ratio, Ctx& cx,
                             cudaStream_t s) {
  // dense-factor shared memory: v_kd * n elements per CTA
  if ((size_t)v_kd * st.n * (st.dt == LRUX_C128 ? 16 : 8) > 200 * 1024) return -2;
  return st.dt == LRUX_F64
             ? ratio_general_t<double>(st, k, u_kd, u_dense, u_idx, v_kd, v_dense, v_idx, ratio, cx, s)
             : ratio_general_t<cplx>(st, k, u_kd, u_dense, u_idx, v_kd, v_dense, v_idx, ratio, cx, s);
}

int launch_det_accept_general(const State& st, int k, const uint8_t* mask, Ctx& cx, cudaStream_t s) {
  int nl = launch_select(st, mask, s);
  {
    ProfScope ps(&cx.prof, LRUX_PROF_UPDATE, s);
    const int grid = persistent_grid(cx.num_sms, 4, st.W);
    if (st.dt == LRUX_F64) gen_apply_prep_kernel<double><<<grid, 256, 0, s>>>(st, k);
    else gen_apply_prep_kernel<cplx><<<grid, 256, 0, s>>>(st, k);
    ++nl;
    State v = st;            // the fold kernel sees the pending area as a k-deep delay buffer
    v.Abuf = st.pend_C;      // a = A^-1 v   (rows of AVt)
    v.Bbuf = st.pend_N;      // b = R^-1 u^T A^-1
    v.cap = st.kmax;
    v.kind = KIND_DET;
    const char* keep = cx.last[LRUX_PROF_FLUSH];
    const int r = launch_flush_dmma(v, cx, s);
    cx.last[LRUX_PROF_FLUSH] = keep;
    if (r < 0) return -1;
    nl += r;
    cx.name(LRUX_PROF_UPDATE, "gen_apply_prep_kernel+flush_dmma_kernel");
  }
  gen_apply_done_kernel<<<(unsigned)((st.W + 255) / 256), 256, 0, s>>>(st);
  ++nl;
  return cudaGetLastError() == cudaSuccess ? nl : -1;
}

}  // namespace lrux
