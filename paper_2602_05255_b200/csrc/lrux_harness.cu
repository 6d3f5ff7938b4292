// Monte-Carlo harness kernels (include/lrux_harness.h): proposal draws + row
// gather, Metropolis decision.  Integer RNG identical to workload.py.
#include "lrux_common.cuh"
#include "lrux_harness.h"

namespace lrux {

constexpr uint64_t STREAM_SLOT = 2, STREAM_ORB = 3, STREAM_ACCEPT = 4;
constexpr int kHMaxK = LRUX_MAX_K;   // proposals of up to this many rows

// k distinct values in [0,m): rho_a in [0,m-a) with counter step*k+a, skipping
// previously chosen values in ascending order (workload._distinct), i.e. the
// rho_a-th smallest value not chosen yet = least fixpoint of
// v = rho_a + #{c < a : out[c] <= v}.
__device__ __forceinline__ void draw_distinct(uint64_t seed, uint64_t w, uint64_t stream,
                                              uint64_t step, int k, int m, int* out) {
  for (int a = 0; a < k; ++a) {
    const int rho = (int)to_below(rnd64(seed, w, stream, step * (uint64_t)k + a), (uint32_t)(m - a));
    int v = rho;
    for (int it = 0; it <= a; ++it) {
      int cnt = 0;
      for (int c = 0; c < a; ++c) cnt += (out[c] <= v) ? 1 : 0;
      if (rho + cnt == v) break;
      v = rho + cnt;
    }
    out[a] = v;
  }
}

template <typename T>
__global__ void __launch_bounds__(128)
det_propose_kernel(uint64_t seed, int64_t w0, int64_t step, const int64_t* __restrict__ d_step, int n,
                   int M, int k, const T* __restrict__ Phi, const int32_t* __restrict__ occ,
                   const int32_t* __restrict__ unocc, int32_t* __restrict__ idx,
                   int32_t* __restrict__ upos, T* __restrict__ rows) {
  __shared__ int sq[kHMaxK];
  const int64_t w = blockIdx.x;
  if (d_step) step = d_step[0];
  if (threadIdx.x == 0) {
    int P[kHMaxK], J[kHMaxK];
    draw_distinct(seed, (uint64_t)(w0 + w), STREAM_SLOT, (uint64_t)step, k, n, P);
    draw_distinct(seed, (uint64_t)(w0 + w), STREAM_ORB, (uint64_t)step, k, M - n, J);
    for (int a = 0; a < k; ++a) {
      idx[w * k + a] = P[a];
      upos[w * k + a] = J[a];
      sq[a] = unocc[w * (M - n) + J[a]];
    }
  }
  __syncthreads();
  for (int a = 0; a < k; ++a) {
    const T* src = Phi + ((size_t)w * M + sq[a]) * n;
    T* dst = rows + ((size_t)w * k + a) * n;
    for (int i = threadIdx.x; i < n; i += blockDim.x) dst[i] = src[i];
  }
}

template <typename T>
__global__ void __launch_bounds__(128)
pf_propose_kernel(uint64_t seed, int64_t w0, int64_t step, const int64_t* __restrict__ d_step, int n,
                  int M, int k, const T* __restrict__ F, const int32_t* __restrict__ occ,
                  const int32_t* __restrict__ unocc, int32_t* __restrict__ idx,
                  int32_t* __restrict__ upos, T* __restrict__ rows) {
  __shared__ int sq[kHMaxK], sp[kHMaxK];
  const int64_t w = blockIdx.x;
  if (d_step) step = d_step[0];
  if (threadIdx.x == 0) {
    int P[kHMaxK], J[kHMaxK];
    draw_distinct(seed, (uint64_t)(w0 + w), STREAM_SLOT, (uint64_t)step, k, n, P);
    draw_distinct(seed, (uint64_t)(w0 + w), STREAM_ORB, (uint64_t)step, k, M - n, J);
    for (int a = 0; a < k; ++a) {
      idx[w * k + a] = P[a];
      upos[w * k + a] = J[a];
      sp[a] = P[a];
      sq[a] = unocc[w * (M - n) + J[a]];
    }
  }
  __syncthreads();
  for (int a = 0; a < k; ++a) {
    const T* src = F + ((size_t)w * M + sq[a]) * M;
    T* dst = rows + ((size_t)w * k + a) * n;
    for (int j = threadIdx.x; j < n; j += blockDim.x) {
      int o = occ[w * n + j];
      for (int b = 0; b < k; ++b)
        if (sp[b] == j) o = sq[b];  // proposed occupation
      dst[j] = src[o];
    }
  }
}

template <typename T>
__global__ void decide_kernel(uint64_t seed, int64_t w0, int64_t step, int64_t* __restrict__ d_step, int64_t W,
                              int n, int M, int k, const T* __restrict__ ratio,
                              const int32_t* __restrict__ idx, const int32_t* __restrict__ upos,
                              int32_t* __restrict__ occ, int32_t* __restrict__ unocc,
                              uint8_t* __restrict__ mask, unsigned long long* __restrict__ naccept) {
  const int64_t w = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (d_step) step = d_step[0];
  if (w < W) {
    const double xi = to_uniform(rnd64(seed, (uint64_t)(w0 + w), STREAM_ACCEPT, (uint64_t)step));
    const double a2 = Sc<T>::abs2(ratio[w]);
    const double p = fmin(1.0, a2);
    const bool acc = (a2 == a2) && xi < p;  // NaN rejects
    mask[w] = acc ? 1 : 0;
    if (acc) {
      for (int a = 0; a < k; ++a) {
        const int ps = idx[w * k + a], j = upos[w * k + a];
        const int o = occ[w * n + ps];
        occ[w * n + ps] = unocc[w * (M - n) + j];
        unocc[w * (M - n) + j] = o;
      }
      atomicAdd(naccept, 1ULL);
    }
  }
  if (d_step) {
    // device-side step counter (CUDA-graph replay): the block that finishes last advances it --
    // every block has read d_step[0] before it arrives here
    __syncthreads();
    if (threadIdx.x == 0) {
      __threadfence();
      const unsigned long long prev = atomicAdd((unsigned long long*)&d_step[1], 1ULL);
      if (prev == (unsigned long long)gridDim.x - 1) {
        d_step[1] = 0;
        d_step[0] = step + 1;
      }
    }
  }
}

}  // namespace lrux

using namespace lrux;

static bool bad_args(int64_t W, int n, int M, int k, int dt) {
  return W <= 0 || n <= 0 || M <= n || k < 1 || k > kHMaxK || k > n || k > M - n ||
         (dt != LRUX_F64 && dt != LRUX_C128);
}

extern "C" {

lrux_status_t lruxh_det_propose(uint64_t seed, int64_t w0, int64_t step, int64_t W, int32_t n,
                                int32_t M, int32_t k, lrux_dtype_t dt, const void* d_Phi,
                                const int32_t* d_occ, const int32_t* d_unocc, int32_t* d_idx,
                                int32_t* d_upos, void* d_rows, const int64_t* d_step, void* stream) {
  if (bad_args(W, n, M, k, dt) || !d_Phi || !d_occ || !d_unocc || !d_idx || !d_upos || !d_rows)
    return LRUX_EINVAL;
  cudaStream_t s = (cudaStream_t)stream;
  if (dt == LRUX_F64)
    det_propose_kernel<double><<<(unsigned)W, 128, 0, s>>>(seed, w0, step, d_step, n, M, k,
        (const double*)d_Phi, d_occ, d_unocc, d_idx, d_upos, (double*)d_rows);
  else
    det_propose_kernel<cplx><<<(unsigned)W, 128, 0, s>>>(seed, w0, step, d_step, n, M, k,
        (const cplx*)d_Phi, d_occ, d_unocc, d_idx, d_upos, (cplx*)d_rows);
  return cudaGetLastError() == cudaSuccess ? LRUX_OK : LRUX_ECUDA;
}

lrux_status_t lruxh_pf_propose(uint64_t seed, int64_t w0, int64_t step, int64_t W, int32_t n,
                               int32_t M, int32_t k, lrux_dtype_t dt, const void* d_F,
                               const int32_t* d_occ, const int32_t* d_unocc, int32_t* d_idx,
                               int32_t* d_upos, void* d_rows, const int64_t* d_step, void* stream) {
  if (bad_args(W, n, M, k, dt) || !d_F || !d_occ || !d_unocc || !d_idx || !d_upos || !d_rows)
    return LRUX_EINVAL;
  cudaStream_t s = (cudaStream_t)stream;
  if (dt == LRUX_F64)
    pf_propose_kernel<double><<<(unsigned)W, 128, 0, s>>>(seed, w0, step, d_step, n, M, k,
        (const double*)d_F, d_occ, d_unocc, d_idx, d_upos, (double*)d_rows);
  else
    pf_propose_kernel<cplx><<<(unsigned)W, 128, 0, s>>>(seed, w0, step, d_step, n, M, k,
        (const cplx*)d_F, d_occ, d_unocc, d_idx, d_upos, (cplx*)d_rows);
  return cudaGetLastError() == cudaSuccess ? LRUX_OK : LRUX_ECUDA;
}

lrux_status_t lruxh_decide(uint64_t seed, int64_t w0, int64_t step, int64_t W, int32_t n,
                           int32_t M, int32_t k, lrux_dtype_t dt, const void* d_ratio,
                           const int32_t* d_idx, const int32_t* d_upos, int32_t* d_occ,
                           int32_t* d_unocc, uint8_t* d_mask, int64_t* d_naccept, int64_t* d_step,
                           void* stream) {
  if (bad_args(W, n, M, k, dt) || !d_ratio || !d_idx || !d_upos || !d_occ || !d_unocc || !d_mask ||
      !d_naccept)
    return LRUX_EINVAL;
  cudaStream_t s = (cudaStream_t)stream;
  const unsigned g = (unsigned)((W + 255) / 256);
  if (dt == LRUX_F64)
    decide_kernel<double><<<g, 256, 0, s>>>(seed, w0, step, d_step, W, n, M, k, (const double*)d_ratio,
        d_idx, d_upos, d_occ, d_unocc, d_mask, (unsigned long long*)d_naccept);
  else
    decide_kernel<cplx><<<g, 256, 0, s>>>(seed, w0, step, d_step, W, n, M, k, (const cplx*)d_ratio, d_idx,
        d_upos, d_occ, d_unocc, d_mask, (unsigned long long*)d_naccept);
  return cudaGetLastError() == cudaSuccess ? LRUX_OK : LRUX_ECUDA;
}

}  // extern "C"
