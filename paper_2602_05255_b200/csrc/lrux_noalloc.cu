// lrux_det_ratio_noalloc: the rank-k determinant ratio (Eq. 3-4 with one-hot v, PAPER.md:57-65,
// 169) as ONE entry point that allocates nothing -- for callers that cannot call cudaMalloc (code
// under CUDA-graph capture, serving loops, harnesses that forbid it) and therefore cannot own the
// state buffer a handle needs.  It is the ratio step of det_ratio_kernel with the k x k cores
// R_w = N_w A_w^-1[:,P_w] passed between its two kernels through a fixed scratch array in the
// library image instead of the caller's pending area:
//
//   noalloc_core_kernel : R_w[a][b] = sum_i N_w[a][i] Ti_w[P_b][i]   one warp per element -> scratch
//   noalloc_det_kernel  : r_w = det R_w by partial-pivot elimination, one thread per walker
//
// The scratch array (LRUX_NOALLOC_SCRATCH_BYTES = 1 MiB) is resident on every GPU that loads the
// library until the process exits.  Every call on a device shares it: calls that may overlap on
// the GPU race.  It keeps the previous call's contents; the first kernel writes every element the
// second one reads, so nothing has to start at zero.
//
// In HOST code the name of a __device__ array is a host-side stand-in, not a device address; the
// device address comes from cudaGetSymbolAddress, asked once per device with that device current.
#include <mutex>

#include "lrux_common.cuh"
#include "lrux_internal.h"

namespace lrux {

static __device__ __align__(256) unsigned char g_noalloc_scratch[LRUX_NOALLOC_SCRATCH_BYTES];

namespace {

constexpr int kMaxDevices = 64;
std::mutex g_mu;
void* g_scratch_addr[kMaxDevices];   // device address of g_noalloc_scratch, per device ordinal
int g_num_sms[kMaxDevices];

// Device address of the scratch array on the CURRENT device (looked up once per device).
cudaError_t scratch_on_current_device(void** ptr, int* num_sms) {
  int dev = -1;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return e;
  if (dev < 0 || dev >= kMaxDevices) return cudaErrorInvalidDevice;
  std::lock_guard<std::mutex> lock(g_mu);
  if (!g_scratch_addr[dev]) {
    void* p = nullptr;
    e = cudaGetSymbolAddress(&p, g_noalloc_scratch);
    if (e != cudaSuccess) return e;
    int sms = 0;
    e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    if (e != cudaSuccess) return e;
    g_scratch_addr[dev] = p;
    g_num_sms[dev] = sms;
  }
  *ptr = g_scratch_addr[dev];
  *num_sms = g_num_sms[dev];
  return cudaSuccess;
}

}  // namespace

// One warp per element R_w[a][b]; both operands are contiguous rows (Ti = A^-T, so column P_b
// of A^-1 is row P_b of Ti: the O(n) gather of PAPER.md:169).  An index outside [0,n) makes
// the element NaN instead of an out-of-bounds read.
template <typename T>
__global__ void __launch_bounds__(256)
noalloc_core_kernel(int64_t W, int n, int k, const T* __restrict__ Ti, const int32_t* __restrict__ idx,
                    const T* __restrict__ rows, T* __restrict__ R) {
  using S = Sc<T>;
  const int lane = threadIdx.x & 31;
  const int64_t nwarps = (int64_t)gridDim.x * (blockDim.x >> 5);
  const int64_t items = W * k * k;
  for (int64_t item = (int64_t)blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5); item < items; item += nwarps) {
    const int64_t w = item / (k * k);
    const int ab = (int)(item % (k * k)), a = ab / k, b = ab % k;
    const int p = idx[w * k + b];
    T acc = S::zero();
    if (p < 0 || p >= n) {
      acc = S::nan();
    } else {
      const T* x = rows + ((size_t)w * k + a) * n;
      const T* c = Ti + ((size_t)w * n + p) * n;
      for (int i = lane; i < n; i += 32) acc = S::fma(x[i], c[i], acc);
      acc = warp_sum(acc);
    }
    if (lane == 0) R[item] = acc;
  }
}

template <typename T>
__global__ void __launch_bounds__(128)
noalloc_det_kernel(int64_t W, int k, const int32_t* __restrict__ idx, const T* __restrict__ R,
                   T* __restrict__ ratio) {
  using S = Sc<T>;
  const int64_t w = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (w >= W) return;
  bool dup = false;
  for (int a = 0; a < k; ++a)
    for (int b = a + 1; b < k; ++b) dup |= idx[w * k + a] == idx[w * k + b];
  T m[kMaxK * kMaxK];
  for (int q = 0; q < k * k; ++q) m[q] = R[w * k * k + q];
  T det = S::one();
  for (int c = 0; c < k; ++c) {
    int p = c;
    double best = S::abs2(m[c * k + c]);
    for (int r = c + 1; r < k; ++r) {
      const double v = S::abs2(m[r * k + c]);
      if (v > best) { best = v; p = r; }
    }
    if (!(best > 0.0)) {                       // exactly singular core (or NaN): det = 0 (or NaN)
      det = S::mul(det, m[p * k + c]);
      break;
    }
    if (p != c) {
      for (int j = c; j < k; ++j) { const T t = m[c * k + j]; m[c * k + j] = m[p * k + j]; m[p * k + j] = t; }
      det = S::neg(det);
    }
    const T d = m[c * k + c];
    det = S::mul(det, d);
    const T di = S::inv(d);
    for (int r = c + 1; r < k; ++r) {
      const T f = S::mul(m[r * k + c], di);
      for (int j = c + 1; j < k; ++j) m[r * k + j] = S::fnma(f, m[c * k + j], m[r * k + j]);
    }
  }
  ratio[w] = dup ? S::nan() : det;
}

template <typename T>
static lrux_status_t run_noalloc(int64_t W, int n, int k, const void* Ti, const int32_t* idx, const void* rows,
                                 void* ratio, cudaStream_t s) {
  if (W > (int64_t)LRUX_NOALLOC_SCRATCH_BYTES ||
      (uint64_t)W * k * k * sizeof(T) > (uint64_t)LRUX_NOALLOC_SCRATCH_BYTES)
    return LRUX_ELIMIT;
  void* scratch = nullptr;
  int sms = 0;
  if (scratch_on_current_device(&scratch, &sms) != cudaSuccess) return LRUX_ECUDA;
  const int64_t items = W * k * k;
  const int64_t want = (items + 7) / 8;
  const int grid = (int)(want < (int64_t)sms * 8 ? want : (int64_t)sms * 8);
  noalloc_core_kernel<T><<<grid, 256, 0, s>>>(W, n, k, (const T*)Ti, idx, (const T*)rows, (T*)scratch);
  if (cudaGetLastError() != cudaSuccess) return LRUX_ECUDA;
  noalloc_det_kernel<T><<<(unsigned)((W + 127) / 128), 128, 0, s>>>(W, k, idx, (const T*)scratch, (T*)ratio);
  if (cudaGetLastError() != cudaSuccess) return LRUX_ECUDA;
  return LRUX_OK;
}

}  // namespace lrux

extern "C" lrux_status_t lrux_det_ratio_noalloc(int64_t W, int32_t n, int32_t k, lrux_dtype_t dtype,
                                                const void* d_Ti, const int32_t* d_idx, const void* d_rows,
                                                void* d_ratio, void* stream) {
  if (W < 1 || n < 1 || k < 1 || k > LRUX_MAX_K_GENERAL || k > n || !d_Ti || !d_idx || !d_rows || !d_ratio)
    return LRUX_EINVAL;
  if (dtype != LRUX_F64 && dtype != LRUX_C128) return LRUX_EINVAL;
  cudaStream_t s = (cudaStream_t)stream;
  return dtype == LRUX_F64 ? lrux::run_noalloc<double>(W, n, k, d_Ti, d_idx, d_rows, d_ratio, s)
                           : lrux::run_noalloc<lrux::cplx>(W, n, k, d_Ti, d_idx, d_rows, d_ratio, s);
}
