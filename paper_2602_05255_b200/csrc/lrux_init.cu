// Step a0: batched initial factorisation, timed separately.
//   det: A^-T by in-place Gauss-Jordan elimination with partial pivoting on A^T,
//        (phase, log|det|) from the pivots
//   pf : (phase, log|pf|) by Parlett-Reid elimination with pivoting (PAPER.md:445
//        leaves the algorithm open), A^-1 by the same Gauss-Jordan kernel followed
//        by an exact skew projection.
// One CTA per walker, matrix resident in global memory / L2.
#include "lrux_common.cuh"
#include "lrux_internal.h"

namespace lrux {

// ---------------------------------------------------------------- load / store
// dst[w][r][c] = transpose ? src[w][c][r] : src[w][r][c];  skew: read only the strict
// upper triangle of src and mirror it.
template <typename T>
__global__ void copy_matrix_kernel(const T* __restrict__ src, T* __restrict__ dst, int n,
                                   bool transpose, bool skew) {
  __shared__ T tile[32][33];
  const size_t base = (size_t)blockIdx.z * n * n;
  const int r0 = blockIdx.y * 32, c0 = blockIdx.x * 32;
  // read the source tile whose transpose (or itself) lands at dst tile (r0,c0)
  for (int y = threadIdx.y; y < 32; y += blockDim.y) {
    int sr = (transpose ? c0 : r0) + y, sc = (transpose ? r0 : c0) + threadIdx.x;
    if (sr < n && sc < n) {
      T v;
      if (skew) {
        if (sr < sc) v = src[base + (size_t)sr * n + sc];
        else if (sr > sc) v = Sc<T>::neg(src[base + (size_t)sc * n + sr]);
        else v = Sc<T>::zero();
      } else {
        v = src[base + (size_t)sr * n + sc];
      }
      tile[y][threadIdx.x] = v;
    }
  }
  __syncthreads();
  for (int y = threadIdx.y; y < 32; y += blockDim.y) {
    int dr = r0 + y, dc = c0 + threadIdx.x;
    if (dr < n && dc < n)
      dst[base + (size_t)dr * n + dc] = transpose ? tile[threadIdx.x][y] : tile[y][threadIdx.x];
  }
}

template <typename T>
static void launch_copy(const void* src, void* dst, int64_t W, int n, bool transpose, bool skew,
                        cudaStream_t s) {
  dim3 grid((n + 31) / 32, (n + 31) / 32, (unsigned)W), block(32, 8);
  copy_matrix_kernel<T><<<grid, block, 0, s>>>((const T*)src, (T*)dst, n, transpose, skew);
}

// M <- (M - M^T)/2 exactly skew, zero diagonal.
template <typename T>
__global__ void skew_project_kernel(T* __restrict__ Mall, int n) {
  T* M = Mall + (size_t)blockIdx.z * n * n;
  int i = blockIdx.y * blockDim.y + threadIdx.y, j = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n || j >= n || i > j) return;
  if (i == j) { M[(size_t)i * n + i] = Sc<T>::zero(); return; }
  T v = Sc<T>::scale(Sc<T>::sub(M[(size_t)i * n + j], M[(size_t)j * n + i]), 0.5);
  M[(size_t)i * n + j] = v;
  M[(size_t)j * n + i] = Sc<T>::neg(v);
}

// ---------------------------------------------------------------- block argmax
struct ArgMax {
  double v;
  int i;
};
__device__ __forceinline__ ArgMax argmax_combine(ArgMax a, ArgMax b) {
  // larger value wins; lowest index on ties
  if (b.v > a.v || (b.v == a.v && b.i < a.i)) return b;
  return a;
}
__device__ inline ArgMax block_argmax(ArgMax x, ArgMax* red /*[32]*/) {
#pragma unroll
  for (int m = 16; m > 0; m >>= 1) {
    ArgMax o;
    o.v = __shfl_xor_sync(0xffffffffu, x.v, m);
    o.i = __shfl_xor_sync(0xffffffffu, x.i, m);
    x = argmax_combine(x, o);
  }
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, nw = blockDim.x >> 5;
  __syncthreads();
  if (lane == 0) red[warp] = x;
  __syncthreads();
  ArgMax r = red[0];
  for (int q = 1; q < nw; ++q) r = argmax_combine(r, red[q]);
  return r;
}

// ---------------------------------------------------------------- Gauss-Jordan
// In-place inverse of M (n x n, global memory) with partial (row) pivoting.
// write_amp: also write phase / logabs of det M.
template <typename T>
__global__ void __launch_bounds__(256)
gj_inverse_kernel(T* __restrict__ Mall, int n, T* __restrict__ phase_out,
                  double* __restrict__ logabs_out, int32_t* __restrict__ info, bool write_amp) {
  using S = Sc<T>;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  T* prow = (T*)smem_raw;          // [n] scaled pivot row
  T* colf = prow + n;              // [n] elimination factors
  int* piv = (int*)(colf + n);     // [n]
  __shared__ ArgMax red[32];
  __shared__ int singular;
  const int w = blockIdx.x, tid = threadIdx.x, nt = blockDim.x;
  const int warp = tid >> 5, lane = tid & 31, nw = nt >> 5;
  T* M = Mall + (size_t)w * n * n;
  T phase = S::one();
  double logabs = 0.0;
  if (tid == 0) singular = 0;
  __syncthreads();

  for (int c = 0; c < n; ++c) {
    ArgMax best{-1.0, 0x7fffffff};
    for (int r = c + tid; r < n; r += nt) {
      double v = S::abs2(M[(size_t)r * n + c]);
      if (!(v == v)) v = -1.0;  // NaN never wins
      best = argmax_combine(best, ArgMax{v, r});
    }
    best = block_argmax(best, red);
    const int p = best.i;
    if (!(best.v > 0.0) || !isfinite(best.v)) {
      if (tid == 0) singular = 1;
      break;  // uniform across the block
    }
    if (tid == 0) piv[c] = p;
    // swap rows c <-> p; the new pivot row goes to smem
    for (int j = tid; j < n; j += nt) {
      T a = M[(size_t)c * n + j];
      T b = M[(size_t)p * n + j];
      if (p != c) M[(size_t)p * n + j] = a;
      prow[j] = b;
    }
    __syncthreads();
    const T d = prow[c];
    const T dinv = S::inv(d);
    if (tid == 0) {
      double ad = S::abs(d);
      T u = S::unit(d, ad);
      phase = S::mul(phase, u);
      if (p != c) phase = S::neg(phase);
      logabs += log(ad);
    }
    for (int r = tid; r < n; r += nt) colf[r] = M[(size_t)r * n + c];
    __syncthreads();
    for (int j = tid; j < n; j += nt) {
      T v = (j == c) ? dinv : S::mul(prow[j], dinv);
      prow[j] = v;
      M[(size_t)c * n + j] = v;
    }
    __syncthreads();
    for (int r = warp; r < n; r += nw) {
      if (r == c) continue;
      const T f = colf[r];
      T* row = M + (size_t)r * n;
      for (int j = lane; j < n; j += 32) {
        T v = (j == c) ? S::zero() : row[j];
        row[j] = S::fnma(f, prow[j], v);
      }
    }
    __syncthreads();
  }
  __syncthreads();
  if (singular) {
    if (tid == 0) {
      atomicOr(&info[w], 1);
      if (write_amp) { phase_out[w] = S::zero(); logabs_out[w] = -INFINITY; }
    }
    return;
  }
  // undo the row permutation: columns swapped in reverse order
  for (int c = n - 1; c >= 0; --c) {
    const int p = piv[c];
    if (p != c) {
      for (int r = tid; r < n; r += nt) {
        T a = M[(size_t)r * n + c];
        M[(size_t)r * n + c] = M[(size_t)r * n + p];
        M[(size_t)r * n + p] = a;
      }
      __syncthreads();
    }
  }
  if (tid == 0 && write_amp) {
    phase_out[w] = phase;
    logabs_out[w] = logabs;
  }
}

// ---------------------------------------------------------------- Parlett-Reid
// Pfaffian of the skew matrix M (destroyed): (phase, log|pf|).
template <typename T>
__global__ void __launch_bounds__(256)
parlett_reid_kernel(T* __restrict__ Mall, int n, T* __restrict__ phase_out,
                    double* __restrict__ logabs_out, int32_t* __restrict__ info) {
  using S = Sc<T>;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  T* tau = (T*)smem_raw;  // [n]
  T* col = tau + n;       // [n]
  __shared__ ArgMax red[32];
  const int w = blockIdx.x, tid = threadIdx.x, nt = blockDim.x;
  const int warp = tid >> 5, lane = tid & 31, nw = nt >> 5;
  T* M = Mall + (size_t)w * n * n;
  T phase = S::one();
  double logabs = 0.0;
  bool zero = false;
  for (int j = 0; j + 1 < n; j += 2) {
    ArgMax best{-1.0, 0x7fffffff};
    for (int r = j + 1 + tid; r < n; r += nt) {
      double v = S::abs2(M[(size_t)r * n + j]);
      if (!(v == v)) v = -1.0;
      best = argmax_combine(best, ArgMax{v, r});
    }
    best = block_argmax(best, red);
    const int p = best.i;
    if (!(best.v > 0.0) || !isfinite(best.v)) { zero = true; break; }
    if (p != j + 1) {
      for (int c = tid; c < n; c += nt) {
        T a = M[(size_t)(j + 1) * n + c];
        M[(size_t)(j + 1) * n + c] = M[(size_t)p * n + c];
        M[(size_t)p * n + c] = a;
      }
      __syncthreads();
      for (int r = tid; r < n; r += nt) {
        T a = M[(size_t)r * n + j + 1];
        M[(size_t)r * n + j + 1] = M[(size_t)r * n + p];
        M[(size_t)r * n + p] = a;
      }
      __syncthreads();
      phase = S::neg(phase);
    }
    const T a = M[(size_t)j * n + j + 1];
    const T ainv = S::inv(a);
    {
      double ad = S::abs(a);
      phase = S::mul(phase, S::unit(a, ad));
      logabs += log(ad);
    }
    for (int c = j + 2 + tid; c < n; c += nt) {
      tau[c] = S::mul(M[(size_t)j * n + c], ainv);
      col[c] = M[(size_t)c * n + j + 1];
    }
    __syncthreads();
    for (int r = j + 2 + warp; r < n; r += nw) {
      const T tr = tau[r], cr = col[r];
      T* row = M + (size_t)r * n;
      for (int c = j + 2 + lane; c < n; c += 32) {
        T v = row[c];
        v = S::fma(tr, col[c], v);
        v = S::fnma(cr, tau[c], v);
        row[c] = v;
      }
    }
    __syncthreads();
  }
  if (tid == 0) {
    if (zero) {
      atomicOr(&info[w], 1);
      phase_out[w] = S::zero();
      logabs_out[w] = -INFINITY;
    } else {
      phase_out[w] = phase;
      logabs_out[w] = logabs;
    }
  }
}

// ---------------------------------------------------------------- launchers
// refresh: bit 1 (singular matrix) is re-evaluated, the other sticky bits stay
__global__ void info_clear_singular_kernel(int32_t* __restrict__ info, int64_t W) {
  const int64_t w = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (w < W) info[w] &= ~1;
}

template <typename T>
static int init_impl(const State& st, const void* d_A0, Ctx& cx, cudaStream_t s, bool refresh = false) {
  const int n = st.n;
  const size_t W = (size_t)st.W;
  int nl = 0;
  if (refresh) {
    info_clear_singular_kernel<<<(unsigned)((W + 255) / 256), 256, 0, s>>>(st.info, (int64_t)W); ++nl;
  } else {
    cudaMemsetAsync(st.info, 0, W * 4, s);
  }
  cudaMemsetAsync(st.fill, 0, W * 4, s);
  cudaMemsetAsync(st.nupd, 0, W * 4, s);
  cudaMemsetAsync(st.pend_ok, 0, W, s);
  cudaMemsetAsync(st.counters, 0, refresh ? 16 : 32, s);   // a refresh keeps the flush totals
  if (st.pend_cnt) cudaMemsetAsync(st.pend_cnt, 0, W * 4, s);
  const size_t smem_gj = 2 * (size_t)n * sizeof(T) + (size_t)n * 4;
  const size_t smem_pr = 2 * (size_t)n * sizeof(T);
  const bool blocked = n >= kBlockedInitMin;   // the unblocked kernels are configured only where they run
  if (!blocked && cx.configure((const void*)gj_inverse_kernel<T>, 256, smem_gj) < 0) return -1;
  if (st.kind == KIND_DET) {
    launch_copy<T>(d_A0, st.Ti, st.W, n, /*transpose=*/true, /*skew=*/false, s); ++nl;
    const int rb = blocked ? launch_gj_blocked(st, true, cx, s) : 0;
    if (rb < 0) return -1;
    if (rb > 0) nl += rb;
    else {
      gj_inverse_kernel<T><<<(unsigned)W, 256, smem_gj, s>>>((T*)st.Ti, n, (T*)st.phase, st.logabs,
                                                             st.info, true); ++nl;
    }
  } else {
    if (cx.configure((const void*)parlett_reid_kernel<T>, 256, smem_pr) < 0) return -1;
    launch_copy<T>(d_A0, st.Ti, st.W, n, false, /*skew=*/true, s); ++nl;
    parlett_reid_kernel<T><<<(unsigned)W, 256, smem_pr, s>>>((T*)st.Ti, n, (T*)st.phase, st.logabs,
                                                             st.info); ++nl;
    launch_copy<T>(d_A0, st.Ti, st.W, n, false, true, s); ++nl;
    const int rb = blocked ? launch_gj_blocked(st, false, cx, s) : 0;
    if (rb < 0) return -1;
    if (rb > 0) nl += rb;
    else {
      gj_inverse_kernel<T><<<(unsigned)W, 256, smem_gj, s>>>((T*)st.Ti, n, (T*)st.phase, st.logabs,
                                                             st.info, false); ++nl;
    }
    dim3 grid((n + 31) / 32, (n + 7) / 8, (unsigned)W), block(32, 8);
    skew_project_kernel<T><<<grid, block, 0, s>>>((T*)st.Ti, n); ++nl;
  }
  return cudaGetLastError() == cudaSuccess ? nl : -1;
}

int launch_det_init(const State& st, const void* d_A0, Ctx& cx, cudaStream_t s) {
  return st.dt == LRUX_F64 ? init_impl<double>(st, d_A0, cx, s) : init_impl<cplx>(st, d_A0, cx, s);
}
int launch_pf_init(const State& st, const void* d_A0, Ctx& cx, cudaStream_t s) {
  return st.dt == LRUX_F64 ? init_impl<double>(st, d_A0, cx, s) : init_impl<cplx>(st, d_A0, cx, s);
}

int launch_refresh(const State& st, const void* d_A, Ctx& cx, cudaStream_t s) {
  return st.dt == LRUX_F64 ? init_impl<double>(st, d_A, cx, s, true)
                           : init_impl<cplx>(st, d_A, cx, s, true);
}

int launch_get_amplitude(const State& st, void* d_phase, double* d_logabs, cudaStream_t s) {
  const size_t e = st.dt == LRUX_C128 ? 16 : 8;
  cudaMemcpyAsync(d_phase, st.phase, (size_t)st.W * e, cudaMemcpyDeviceToDevice, s);
  cudaMemcpyAsync(d_logabs, st.logabs, (size_t)st.W * 8, cudaMemcpyDeviceToDevice, s);
  return cudaGetLastError() == cudaSuccess ? 0 : -1;
}

int launch_get_inverse(const State& st, void* d_out, cudaStream_t s) {
  const bool tr = st.kind == KIND_DET;
  if (st.dt == LRUX_F64) launch_copy<double>(st.Ti, d_out, st.W, st.n, tr, false, s);
  else launch_copy<cplx>(st.Ti, d_out, st.W, st.n, tr, false, s);
  return cudaGetLastError() == cudaSuccess ? 1 : -1;
}

}  // namespace lrux
