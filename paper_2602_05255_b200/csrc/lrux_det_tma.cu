// Immediate Woodbury update for large rows: A^-1 streamed through
// TMA-staged shared-memory tiles exactly once per step.
//
//   Ti[j][:] -= sum_a g[a] C[a][:],   g = R^-1 (N Ti[j][:] - [j == P])      (Eq. 5)
//
// Rows of one walker are contiguous in memory, so a chunk of RC rows is ONE 1-D bulk
// asynchronous copy (cp.async.bulk, mbarrier completion).  Each CTA (one per SM) owns a
// contiguous range of chunks of the concatenated accepted-walker list and runs a ring of
// S stages: up to S-2 chunk loads in flight, one chunk being computed on, one being
// stored back with a bulk store.  Bytes in flight no longer depend on how many
// registers or warps the arithmetic needs -- which is what limits the register-row
// kernel (det_update_kernel) once a row or k gets large.
//
// Per chunk: every warp forms the partial dots of all RC rows over its interleaved column
// slice (rows from shared memory, its slices of N and C cached in registers), the
// partial sums meet in shared memory, g = R^-1 d, then the same lanes apply the rank-k
// update to their columns in place and the chunk goes back to HBM.
#include "lrux_common.cuh"
#include "lrux_internal.h"
#include "lrux_tma.cuh"

namespace lrux {

// Sum NV doubles across the warp with NV-1 + (5 - log2 NV) shuffles instead of 5 NV:
// at each halving step a lane keeps one half of its values and trades the other half.
// On return v[0] of lane L holds the total of value index multi_index<NV>(L).
template <int NV>
__device__ __forceinline__ void warp_reduce_multi(double (&v)[NV]) {
  const int lane = threadIdx.x & 31;
  int off = 16;
#pragma unroll
  for (int h = NV / 2; h >= 1; h >>= 1) {
    const bool hi = (lane & off) != 0;
#pragma unroll
    for (int i = 0; i < h; ++i) {
      const double send = hi ? v[i] : v[i + h];
      const double keep = hi ? v[i + h] : v[i];
      v[i] = keep + __shfl_xor_sync(0xffffffffu, send, off);
    }
    off >>= 1;
  }
  for (; off >= 1; off >>= 1) v[0] += __shfl_xor_sync(0xffffffffu, v[0], off);
}
template <int NV>
__device__ __forceinline__ int multi_index(int lane) {
  int idx = 0, off = 16;
#pragma unroll
  for (int h = NV / 2; h >= 1; h >>= 1) {
    if (lane & off) idx += h;
    off >>= 1;
  }
  return idx;
}
// lanes whose low bits (below the last trading offset) are zero publish the result
template <int NV>
__device__ __forceinline__ bool multi_writer(int lane) {
  int low = 32;
#pragma unroll
  for (int h = NV / 2; h >= 1; h >>= 1) low >>= 1;
  return (lane & (low - 1)) == 0;
}

template <typename T>
struct Vec16;   // 16-byte vector of T
template <>
struct Vec16<double> {
  static constexpr int N = 2;
  static __device__ __forceinline__ double get(const double2& v, int e) { return e ? v.y : v.x; }
  static __device__ __forceinline__ void set(double2& v, int e, double x) { if (e) v.y = x; else v.x = x; }
};
template <>
struct Vec16<cplx> {
  static constexpr int N = 1;
  static __device__ __forceinline__ cplx get(const double2& v, int) { return cplx{v.x, v.y}; }
  static __device__ __forceinline__ void set(double2& v, int, cplx x) { v.x = x.re; v.y = x.im; }
};
__device__ __forceinline__ void to_doubles(double x, double* o) { o[0] = x; }
__device__ __forceinline__ void to_doubles(cplx x, double* o) { o[0] = x.re; o[1] = x.im; }

// RC rows per chunk (one bulk copy), TV 16-byte vectors of every row per lane.  All NW
// warps split the columns of a chunk: lane owns the vectors q = warp*32 + lane + 32 NW t,
// t < TV, of EVERY row -- so its slices of N and C (k x TV vectors each) stay in
// registers for as long as the CTA works on one walker, and shared memory carries only
// the streamed rows.
template <typename T, int KT, int RC, int TV, int NW>
__global__ void __launch_bounds__(NW * 32, 1)
det_update_tma_kernel(State st, int k, int NS) {
  using S = Sc<T>;
  using V = Vec16<T>;
  constexpr int VEC = V::N;
  constexpr int ND = sizeof(T) / 8;          // doubles per element
  constexpr int NV = RC * KT * ND;           // values reduced per warp and chunk (<= 32)
  static_assert(NV <= 32, "too many partial sums per warp");
  extern __shared__ __align__(128) unsigned char smem_raw[];
  const int n = st.n, kmax = st.kmax;
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const size_t chunk_elems = (size_t)RC * n;
  T* stage_buf = (T*)smem_raw;                                   // [NS][RC][n]
  double* dpart0 = (double*)(stage_buf + (size_t)NS * chunk_elems);  // [2][NW][NV]
  double* dsum0 = dpart0 + 2 * NW * NV;                          // [2][NV]
  T* gsm = (T*)(dsum0 + 2 * NV);                                 // [RC][KT]
  uint64_t* full = (uint64_t*)(gsm + RC * KT);                   // [NS]
  __shared__ T Ri[KT * KT];
  __shared__ int sidx[KT];

  const int count = st.counters[0];
  const int cpw = (n + RC - 1) / RC;                             // chunks per walker
  const int64_t TC = (int64_t)count * cpw;
  const int64_t first = TC * blockIdx.x / gridDim.x, last = TC * (blockIdx.x + 1) / gridDim.x;
  const int my = (int)(last - first);
  if (my <= 0) return;
  if (tid == 0) {
    for (int q = 0; q < NS; ++q) tma::mbar_init(&full[q], 1);
    tma::fence_barrier_init();
  }
  __syncthreads();

  auto issue = [&](int li) {   // thread 0 only
    const int64_t cidx = first + li;
    const int w = st.list[cidx / cpw];
    const int j0 = (int)(cidx % cpw) * RC;
    const int rows = min(RC, n - j0);
    const uint32_t bytes = (uint32_t)((size_t)rows * n * sizeof(T));
    const int stg = li % NS;
    tma::mbar_arrive_expect_tx(&full[stg], bytes);
    tma::load(stage_buf + (size_t)stg * chunk_elems, (const T*)st.Ti + (size_t)w * n * n + (size_t)j0 * n,
              bytes, &full[stg]);
  };
  if (tid == 0)
    for (int li = 0; li < min(NS - 2, my); ++li) issue(li);

  const int nvec = n / VEC;
  double2 nreg[KT][TV], creg[KT][TV];
  int cur_w = -1;
  for (int li = 0; li < my; ++li) {
    const int64_t cidx = first + li;
    const int w = st.list[cidx / cpw];
    const int j0 = (int)(cidx % cpw) * RC;
    const int rows = min(RC, n - j0);
    const int stg = li % NS;
    if (w != cur_w) {
      __syncthreads();
      const double2* gN = (const double2*)((const T*)st.pend_N + (size_t)w * kmax * n);
      const double2* gC = (const double2*)((const T*)st.pend_C + (size_t)w * kmax * n);
#pragma unroll
      for (int a = 0; a < KT; ++a)
#pragma unroll
        for (int t = 0; t < TV; ++t) {
          const int q = warp * 32 + lane + 32 * NW * t;
          const bool ok = a < k && q < nvec;
          nreg[a][t] = ok ? gN[(size_t)a * nvec + q] : make_double2(0.0, 0.0);
          creg[a][t] = ok ? gC[(size_t)a * nvec + q] : make_double2(0.0, 0.0);
        }
      if (tid < KT * KT) {
        const int a = tid / KT, b = tid % KT;
        Ri[tid] = (a < k && b < k) ? ((const T*)st.pend_Rinv)[(size_t)w * st.kc * st.kc + a * st.kc + b]
                                   : S::zero();
      }
      if (tid < KT) sidx[tid] = tid < k ? st.pend_idx[(size_t)w * kmax + tid] : -1;
      cur_w = w;
      __syncthreads();
    }
    if (tid == 0 && li + NS - 2 < my) {
      tma::store_wait_read<1>();   // the stage consumed two chunks ago has been read out
      issue(li + NS - 2);
    }
    double* dpart = dpart0 + (li & 1) * NW * NV;   // double-buffered by chunk parity
    double* dsum = dsum0 + (li & 1) * NV;
    tma::mbar_wait(&full[stg], (uint32_t)((li / NS) & 1));
    T* xs = stage_buf + (size_t)stg * chunk_elems;

    // ---- partial dots d[r][a] = sum over this lane's columns of x[r][i] N[a][i]
    T d[RC][KT];
#pragma unroll
    for (int r = 0; r < RC; ++r)
#pragma unroll
      for (int a = 0; a < KT; ++a) d[r][a] = S::zero();
#pragma unroll
    for (int t = 0; t < TV; ++t) {
      const int q = warp * 32 + lane + 32 * NW * t;
      if (q < nvec) {
#pragma unroll
        for (int r = 0; r < RC; ++r) {
          const double2 xv = ((const double2*)(xs + (size_t)r * n))[q];
#pragma unroll
          for (int a = 0; a < KT; ++a)
#pragma unroll
            for (int e = 0; e < VEC; ++e)
              d[r][a] = S::fma(V::get(xv, e), V::get(nreg[a][t], e), d[r][a]);
        }
      }
    }
    {
      double v[NV];
#pragma unroll
      for (int r = 0; r < RC; ++r)
#pragma unroll
        for (int a = 0; a < KT; ++a) to_doubles(d[r][a], &v[(r * KT + a) * ND]);
      warp_reduce_multi<NV>(v);
      if (multi_writer<NV>(lane)) dpart[warp * NV + multi_index<NV>(lane)] = v[0];
    }
    __syncthreads();
    // ---- cross-warp sum of the partials: one thread per value, then (a second short
    // phase) g[r][a] = sum_b Ri[a][b] (d[r][b] - [j0 + r == P[b]])
    if (tid < NV) {
      double v = 0.0;
#pragma unroll
      for (int c = 0; c < NW; ++c) v += dpart[c * NV + tid];
      dsum[tid] = v;
    }
    __syncthreads();
    if (tid < RC * KT) {
      const int r = tid / KT, a = tid % KT;
      T acc = S::zero();
#pragma unroll
      for (int b = 0; b < KT; ++b) {
        T db = sc_from(dsum[(r * KT + b) * ND], dsum[(r * KT + b) * ND + ND - 1], T{});
        if (j0 + r == sidx[b]) db = S::sub(db, S::one());
        acc = S::fma(Ri[a * KT + b], db, acc);
      }
      gsm[r * KT + a] = acc;
    }
    __syncthreads();
    // ---- x[r][i] -= sum_a g[r][a] C[a][i] on this lane's columns, in place
    {
      T g[RC][KT];
#pragma unroll
      for (int r = 0; r < RC; ++r)
#pragma unroll
        for (int a = 0; a < KT; ++a) g[r][a] = gsm[r * KT + a];
#pragma unroll
      for (int t = 0; t < TV; ++t) {
        const int q = warp * 32 + lane + 32 * NW * t;
        if (q < nvec) {
#pragma unroll
          for (int r = 0; r < RC; ++r) {
            double2 xv = ((const double2*)(xs + (size_t)r * n))[q];
#pragma unroll
            for (int a = 0; a < KT; ++a)
#pragma unroll
              for (int e = 0; e < VEC; ++e)
                V::set(xv, e, S::fnma(g[r][a], V::get(creg[a][t], e), V::get(xv, e)));
            ((double2*)(xs + (size_t)r * n))[q] = xv;
          }
        }
      }
    }
    tma::fence_proxy_async();
    __syncthreads();
    if (tid == 0) {
      tma::store((T*)st.Ti + (size_t)w * n * n + (size_t)j0 * n, xs, (uint32_t)((size_t)rows * n * sizeof(T)));
      tma::store_commit();
    }
  }
  if (tid == 0) tma::store_wait_all<0>();
}

template <typename T, int KT, int RC, int TV, int NW>
static int launch_tma_inst(const State& st, int k, Ctx& cx, cudaStream_t s, bool probe) {
  constexpr int ND = sizeof(T) / 8;
  if constexpr (RC * KT * ND > 32 || KT * TV > (NW == 16 ? 8 : 16)) {
    return 0;   // too many partial sums / cached registers for this instance
  } else {
    const size_t row = (size_t)st.n * sizeof(T);
    const size_t fixed = 2 * (NW + 1) * (size_t)(RC * KT * ND) * 8 + (size_t)RC * KT * sizeof(T) + 64 + 256;
    int NS = (int)((220 * 1024 - fixed) / ((size_t)RC * row));
    if (NS > 8) NS = 8;
    if (NS < 3) return 0;
    const size_t smem = (size_t)NS * RC * row + fixed;
    if (probe) return 1;
    auto kern = det_update_tma_kernel<T, KT, RC, TV, NW>;
    if (cx.configure((const void*)kern, NW * 32, smem) < 0) return -1;
    kern<<<cx.num_sms, NW * 32, smem, s>>>(st, k, NS);
    cx.name(LRUX_PROF_UPDATE, "det_update_tma_kernel");
    return 1;
  }
}

// Returns the number of launches (1), 0 when this shape is not eligible (caller falls
// back to the register-row / generic kernels), -1 on a CUDA error.
template <typename T, int KT>
static int launch_update_tma_kt(const State& st, int k, Ctx& cx, cudaStream_t s, bool probe) {
  const size_t row = (size_t)st.n * sizeof(T);
  if (row % 16 != 0) return 0;
  const int nvec = (int)(row / 16);
  // rows per chunk: ~32 KB per bulk copy
  const int rc = row >= 32 * 1024 ? 1 : row >= 16 * 1024 ? 2 : 4;
  // 16 warps when a lane would otherwise own >= 2 vectors of a row: more warps to cover
  // the FP64 / shared-memory latency of the per-chunk arithmetic
  const int tv8 = (nvec + 255) / 256, tv16 = (nvec + 511) / 512;
#define LRUX_TMA_CASE(RC_, TV_, NW_)                                                       \
  if (rc == RC_ && (NW_ == 16 ? tv16 : tv8) <= TV_) {                                      \
    const int r_ = launch_tma_inst<T, KT, RC_, TV_, NW_>(st, k, cx, s, probe);             \
    if (r_ != 0) return r_;                                                                \
  }
  if (tv8 >= 2 && KT <= 2) {
    LRUX_TMA_CASE(4, 1, 16)
    LRUX_TMA_CASE(4, 2, 16)
    LRUX_TMA_CASE(2, 2, 16)
    LRUX_TMA_CASE(1, 2, 16)
    LRUX_TMA_CASE(1, 4, 16)
  }
  LRUX_TMA_CASE(4, 1, 8)
  LRUX_TMA_CASE(4, 2, 8)
  LRUX_TMA_CASE(4, 4, 8)
  LRUX_TMA_CASE(2, 2, 8)
  LRUX_TMA_CASE(2, 4, 8)
  LRUX_TMA_CASE(1, 4, 8)
  LRUX_TMA_CASE(1, 8, 8)
#undef LRUX_TMA_CASE
  return 0;
}

template <typename T>
static int launch_update_tma_t(const State& st, int k, Ctx& cx, cudaStream_t s, bool probe) {
  switch (round_kt(k)) {
    case 1: return launch_update_tma_kt<T, 1>(st, k, cx, s, probe);
    case 2: return launch_update_tma_kt<T, 2>(st, k, cx, s, probe);
    case 4: return launch_update_tma_kt<T, 4>(st, k, cx, s, probe);
    default: return launch_update_tma_kt<T, 8>(st, k, cx, s, probe);
  }
}

int launch_det_update_tma(const State& st, int k, Ctx& cx, cudaStream_t s, bool probe) {
  return st.dt == LRUX_F64 ? launch_update_tma_t<double>(st, k, cx, s, probe)
                           : launch_update_tma_t<cplx>(st, k, cx, s, probe);
}

}  // namespace lrux
