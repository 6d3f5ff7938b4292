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
#include <stdlib.h>

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
//
// APPEND = true is the delayed-update variant (row a6): the same streamed pass, read
// only -- it leaves D[a][j] = N_a . Ti[j][:] - [j == P[a]]  (= u^T A0^-1, Eq. 15) in the
// pending area (pend_C, free once det_prep_kernel has copied a_tau into the buffer) for
// det_append_finish_kernel; nothing is written back to A0^-1.
template <typename T, int KT, int RC, int TV, bool APPEND, int NW>
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
          if (!APPEND) creg[a][t] = ok ? gC[(size_t)a * nvec + q] : make_double2(0.0, 0.0);
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
      if (!APPEND) tma::store_wait_read<1>();   // the stage consumed two chunks ago has been read out
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
      if constexpr (APPEND) {
        if (a < k && r < rows) {
          T db = sc_from(dsum[(r * KT + a) * ND], dsum[(r * KT + a) * ND + ND - 1], T{});
          if (j0 + r == sidx[a]) db = S::sub(db, S::one());
          ((T*)st.pend_C)[((size_t)w * kmax + a) * n + j0 + r] = db;
        }
      } else {
        T acc = S::zero();
#pragma unroll
        for (int b = 0; b < KT; ++b) {
          T db = sc_from(dsum[(r * KT + b) * ND], dsum[(r * KT + b) * ND + ND - 1], T{});
          if (j0 + r == sidx[b]) db = S::sub(db, S::one());
          acc = S::fma(Ri[a * KT + b], db, acc);
        }
        gsm[r * KT + a] = acc;
      }
    }
    if constexpr (APPEND) continue;   // dsum / dpart are double-buffered by chunk parity
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
  if (!APPEND && tid == 0) tma::store_wait_all<0>();
}

// b_tau^T = R^-1 (D - (N Abuf) Bbuf^T) -> Bbuf[fill .. fill+k)   (Eq. 15, PAPER.md:194;
// DESIGN.md reading 5b).  Work item = (accepted walker, 256 columns); thread per column.
template <typename T, int KT>
__global__ void __launch_bounds__(256) det_append_finish_kernel(State st, int k, int chunks) {
  using S = Sc<T>;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  T* NAs = (T*)smem_raw;   // [fill][KT]
  __shared__ T Ri[KT * KT];
  const int n = st.n, kmax = st.kmax, cap = st.cap;
  const int tid = threadIdx.x;
  const int count = st.counters[0];
  for (int item = blockIdx.x; item < count * chunks; item += gridDim.x) {
    const int w = st.list[item / chunks];
    const int j = (item % chunks) * 256 + tid;
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
    if (j >= n) continue;
    const T* D = (const T*)st.pend_C + (size_t)w * kmax * n;
    T* Bb = (T*)st.Bbuf + (size_t)w * cap * n;
    T m[KT];
#pragma unroll
    for (int b = 0; b < KT; ++b) m[b] = b < k ? D[(size_t)b * n + j] : S::zero();
#pragma unroll 8
    for (int s = 0; s < fill; ++s) {
      const T bv = Bb[(size_t)s * n + j];
#pragma unroll
      for (int b = 0; b < KT; ++b) m[b] = S::fnma(NAs[s * KT + b], bv, m[b]);
    }
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

template <typename T, int KT, int RC, int TV, bool APPEND, int NW>
static int launch_tma_inst(const State& st, int k, int num_sms, cudaStream_t s) {
  constexpr int ND = sizeof(T) / 8;
  if constexpr (RC * KT * ND > 32 || KT * TV > (APPEND ? 16 : NW == 16 ? 8 : 16)) {
    return 0;   // too many partial sums / cached registers for this instance
  } else {
    const size_t row = (size_t)st.n * sizeof(T);
    const size_t fixed = 2 * (NW + 1) * (size_t)(RC * KT * ND) * 8 + (size_t)RC * KT * sizeof(T) + 64 + 256;
    int NS = (int)((220 * 1024 - fixed) / ((size_t)RC * row));
    if (NS > 8) NS = 8;
    if (NS < 3) return 0;
    const size_t smem = (size_t)NS * RC * row + fixed;
    if (num_sms <= 0) return 1;   // eligibility probe (launch_det_update_tma_ok)
    auto kern = det_update_tma_kernel<T, KT, RC, TV, APPEND, NW>;
    if (cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess)
      return -1;
    kern<<<num_sms, NW * 32, smem, s>>>(st, k, NS);
    if (!APPEND) return 1;
    const int chunks = (st.n + 255) / 256;
    int64_t grid = (int64_t)num_sms * 8;
    if (grid > st.W * chunks) grid = st.W * chunks;
    det_append_finish_kernel<T, KT><<<(unsigned)grid, 256, (size_t)st.cap * KT * sizeof(T), s>>>(st, k, chunks);
    return 2;
  }
}

// Returns the number of launches (1), 0 when this shape is not eligible (caller falls
// back to the register-row / generic kernels), -1 on a CUDA error.
template <typename T, int KT, bool APPEND>
static int launch_update_tma_kt(const State& st, int k, int num_sms, cudaStream_t s) {
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
    const int r_ = launch_tma_inst<T, KT, RC_, TV_, APPEND, NW_>(st, k, num_sms, s);       \
    if (r_ != 0) return r_;                                                                \
  }
  const char* warps_env = getenv("LRUX_TMA_WARPS");   // A-B measurements only
  if (tv8 >= 2 && KT <= 2 && !(warps_env && warps_env[0] == '8')) {
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

template <typename T, bool APPEND>
static int launch_update_tma_t(const State& st, int k, int num_sms, cudaStream_t s) {
  const int kt = k <= 1 ? 1 : k <= 2 ? 2 : k <= 4 ? 4 : 8;
  switch (kt) {
    case 1: return launch_update_tma_kt<T, 1, APPEND>(st, k, num_sms, s);
    case 2: return launch_update_tma_kt<T, 2, APPEND>(st, k, num_sms, s);
    case 4: return launch_update_tma_kt<T, 4, APPEND>(st, k, num_sms, s);
    default: return launch_update_tma_kt<T, 8, APPEND>(st, k, num_sms, s);
  }
}

int launch_det_update_tma(const State& st, int k, int num_sms, cudaStream_t s) {
  return st.dt == LRUX_F64 ? launch_update_tma_t<double, false>(st, k, num_sms, s)
                           : launch_update_tma_t<cplx, false>(st, k, num_sms, s);
}

// true when a rank-k immediate update of this shape has a TMA-staged instance
bool launch_det_update_tma_ok(const State& st, int k) {
  return launch_det_update_tma(st, k, 0, nullptr) == 1;
}

// delayed append through the same pass (after det_prep_kernel): 2 launches, 0 = not eligible
int launch_det_append_tma(const State& st, int k, int num_sms, cudaStream_t s) {
  return st.dt == LRUX_F64 ? launch_update_tma_t<double, true>(st, k, num_sms, s)
                           : launch_update_tma_t<cplx, true>(st, k, num_sms, s);
}

}  // namespace lrux
