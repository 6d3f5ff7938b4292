// Immediate Pfaffian update on the FP64 tensor pipe, real data.
//
//   A^-1 += Y' R'^-1 Y'^T   (Eq. 21; k = 1: Eq. 22),   Y' = (A^-1 N + E_P, C)   (n x 2k)
//   <=>  Ti[i][j] += sum_beta g[beta][i] y[beta][j],   y = Y'^T,  g[beta][i] = sum_alpha y[alpha][i] R'^-1[alpha][beta]
//
// a rank-2k outer-product accumulation into every element: the "apply" half of
// det_update_dmma_kernel without its dot products, so there is no reduction and no barrier
// between strips.  An 8-ROW STRIP of Ti is the M side of mma.sync.m8n8k4.f64: lane (r, q) loads
// the 16-byte pair Ti[j0+r][cb+2q, cb+2q+1] -- the accumulator layout -- and each 8 x 8 block
// takes 2k/4 DMMAs whose A fragment (g of the strip's rows) lives in registers for the whole
// strip and whose B fragment (y of the block's columns) comes from shared memory, against 2k
// shared-memory operands and 2k DFMAs PER ELEMENT in pf_update_stream_kernel.
//
// Exact skewness (reading 7): as in the scalar kernels every element is produced by
// its own thread, and an element below the diagonal is the exact negative of its mirror image
// because it is computed from the same operands in the same order: block (rows J, columns I)
// below the diagonal starts from -Ti[j][i] (= Ti[i][j] bit for bit), contracts A = y[.][j] with
// B = g[.][i] -- the products g[beta][i] y[beta][j] of the mirrored element, same beta order
// inside and across the DMMAs -- and stores the negative.  Diagonal blocks evaluate both forms
// and select per element; the diagonal itself is written as zero.
//
// Work = 8-row strips of the concatenated accepted list, a contiguous balanced range per CTA;
// y and g of the current walker (2k x n each, zero-padded to MH rows) staged in shared memory
// once per walker and CTA; the next strip's loads are in flight during the current strip's DMMAs.
#include "lrux_common.cuh"
#include "lrux_internal.h"

namespace lrux {

__device__ __forceinline__ void dmma884p(double& d0, double& d1, double a, double b) {
  asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
               : "+d"(d0), "+d"(d1)
               : "d"(a), "d"(b));
}

// NB = 8-column blocks per warp and strip, NW = warps per CTA (8 NB NW >= n), MQ = DMMAs per
// block (4 MQ >= 2k).  ld = row stride of yv / gv (>= n + 8, 8 mod 16 doubles: conflict-free).
template <int NB, int NW, int MQ>
__global__ void __launch_bounds__(NW * 32, NW <= 8 ? 2 : 1) pf_update_dmma_kernel(State st, int k, int ld) {
  constexpr int MH = 4 * MQ;
  constexpr int kMaxC = 2 * kMaxK;
  extern __shared__ __align__(128) unsigned char smem_raw[];
  const int n = st.n, kmax = st.kmax, m = 2 * k;
  double* yv = (double*)smem_raw;           // [MH][ld]
  double* gv = yv + (size_t)MH * ld;        // [MH][ld]
  __shared__ double Ri[kMaxC * kMaxC];
  __shared__ int P[kMaxK];
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int r8 = lane >> 2, q = lane & 3;

  const int count = st.counters[0];
  const int spw = (n + 7) >> 3;
  const int64_t S = (int64_t)count * spw;
  const int64_t first = S * blockIdx.x / gridDim.x, last = S * (blockIdx.x + 1) / gridDim.x;
  const int my = (int)(last - first);
  const int wi0 = (int)(first / spw), s00 = (int)(first % spw);
  const double* Ti = (const double*)st.Ti;

  auto load_strip = [&](int li, double2 (&x)[NB]) {
    const int sx = s00 + li;
    const int w = st.list[wi0 + sx / spw];
    const int j = min((sx % spw) * 8 + r8, n - 1);        // rows past the end: clamped, never stored
    const double* row = Ti + ((size_t)w * n + j) * n;
#pragma unroll
    for (int t = 0; t < NB; ++t) {
      const int c = 8 * (t * NW + warp) + 2 * q;
      x[t] = c < n ? *(const double2*)(row + c) : make_double2(0.0, 0.0);
    }
  };

  double2 xc[NB], xn[NB];
  if (my > 0) load_strip(0, xc);
  int cur_w = -1;
  for (int li = 0; li < my; ++li) {
    const int sx = s00 + li;
    const int w = st.list[wi0 + sx / spw];
    const int j0 = (sx % spw) * 8;
    if (w != cur_w) {
      __syncthreads();   // every warp is done with the previous walker's y, g
      for (int idx = tid; idx < m * m; idx += NW * 32)
        Ri[(idx / m) * kMaxC + (idx % m)] =
            ((const double*)st.pend_Rinv)[(size_t)w * st.kc * st.kc + (idx / m) * st.kc + (idx % m)];
      if (tid < k) P[tid] = st.pend_idx[(size_t)w * kmax + tid];
      __syncthreads();
      const double* pC = (const double*)st.pend_C + (size_t)w * kmax * n;
      const double* pY = (const double*)st.pend_Y + (size_t)w * kmax * n;
      for (int i = tid; i < ld; i += NW * 32) {
        double yp[MH];
#pragma unroll
        for (int a = 0; a < MH; ++a) {
          double v = 0.0;
          if (a < m && i < n) {
            v = a < k ? pY[(size_t)a * n + i] : pC[(size_t)(a - k) * n + i];
            if (a < k && i == P[a]) v += 1.0;
          }
          yp[a] = v;
          yv[(size_t)a * ld + i] = v;
        }
#pragma unroll 1
        for (int b = 0; b < MH; ++b) {
          double g = 0.0;
          if (b < m) {
#pragma unroll
            for (int a = 0; a < MH; ++a)
              if (a < m) g = fma(yp[a], Ri[a * kMaxC + b], g);
          }
          gv[(size_t)b * ld + i] = g;
        }
      }
      cur_w = w;
      __syncthreads();
    }
    if (li + 1 < my) load_strip(li + 1, xn);   // in flight during this strip's arithmetic

    double ag[MQ], ay[MQ];                      // A fragments: g / y of the strip's rows
#pragma unroll
    for (int s = 0; s < MQ; ++s) {
      ag[s] = gv[(size_t)(4 * s + q) * ld + j0 + r8];
      ay[s] = yv[(size_t)(4 * s + q) * ld + j0 + r8];
    }
    const int j = j0 + r8;
    double* orow = (double*)st.Ti + ((size_t)w * n + min(j, n - 1)) * n;
#pragma unroll
    for (int t = 0; t < NB; ++t) {
      const int cb = 8 * (t * NW + warp);
      if (cb < n) {
        double2 v = xc[t];
        if (cb > j0) {                          // above the diagonal: v(r, c)
#pragma unroll
          for (int s = 0; s < MQ; ++s) dmma884p(v.x, v.y, ag[s], yv[(size_t)(4 * s + q) * ld + cb + r8]);
        } else if (cb < j0) {                   // below: -v(c, r)
          v.x = -v.x;
          v.y = -v.y;
#pragma unroll
          for (int s = 0; s < MQ; ++s) dmma884p(v.x, v.y, ay[s], gv[(size_t)(4 * s + q) * ld + cb + r8]);
          v.x = -v.x;
          v.y = -v.y;
        } else {                                // the diagonal block: both forms, selected per element
          double2 lo = make_double2(-v.x, -v.y);
#pragma unroll
          for (int s = 0; s < MQ; ++s) {
            dmma884p(v.x, v.y, ag[s], yv[(size_t)(4 * s + q) * ld + cb + r8]);
            dmma884p(lo.x, lo.y, ay[s], gv[(size_t)(4 * s + q) * ld + cb + r8]);
          }
          const int c0 = cb + 2 * q;
          v.x = c0 > j ? v.x : c0 < j ? -lo.x : 0.0;
          v.y = c0 + 1 > j ? v.y : c0 + 1 < j ? -lo.y : 0.0;
        }
        const int c = cb + 2 * q;
        if (j < n && c < n) *(double2*)(orow + c) = v;
      }
    }
#pragma unroll
    for (int t = 0; t < NB; ++t) xc[t] = xn[t];
  }
}

template <int NB, int NW, int MQ>
static int launch_pf_dmma_inst(const State& st, int k, int ld, Ctx& cx, cudaStream_t s, bool probe) {
  const size_t smem = (size_t)2 * 4 * MQ * ld * sizeof(double);
  if (smem > 200 * 1024) return 0;
  if (probe) return 1;
  auto kern = pf_update_dmma_kernel<NB, NW, MQ>;
  const int occ = cx.configure((const void*)kern, NW * 32, smem);
  if (occ < 0) return -1;
  const int64_t strips = (int64_t)st.W * ((st.n + 7) / 8);
  kern<<<persistent_grid(cx.num_sms, occ, strips), NW * 32, smem, s>>>(st, k, ld);
  cx.name(LRUX_PROF_UPDATE, "pf_update_dmma_kernel");
  return 1;
}

// 1 = launched, 0 = shape not eligible (complex data, n > 1024, 2k x n panels beyond shared
// memory), -1 = CUDA error.  Expects Y in pend_Y (launch_y) and the accepted list (select).
int launch_pf_update_dmma(const State& st, int k, Ctx& cx, cudaStream_t s, bool probe) {
  const int n = st.n;
  if (st.dt != LRUX_F64 || (n & 1) || k > 8 || n > 1024) return 0;
  const int ld = ((n + 15) & ~15) + 8;
  const int blocks = (n + 7) / 8;
  const int mq = k <= 2 ? 1 : k <= 4 ? 2 : 4;
#define LRUX_PFD_CASE(NB_, NW_)                                                         \
  if (blocks <= NB_ * NW_)                                                              \
    return mq == 1 ? launch_pf_dmma_inst<NB_, NW_, 1>(st, k, ld, cx, s, probe)                 \
         : mq == 2 ? launch_pf_dmma_inst<NB_, NW_, 2>(st, k, ld, cx, s, probe)                 \
                   : launch_pf_dmma_inst<NB_, NW_, 4>(st, k, ld, cx, s, probe);
  LRUX_PFD_CASE(2, 8)
  LRUX_PFD_CASE(4, 8)
  LRUX_PFD_CASE(8, 8)
  LRUX_PFD_CASE(8, 16)
#undef LRUX_PFD_CASE
  return 0;
}

}  // namespace lrux
