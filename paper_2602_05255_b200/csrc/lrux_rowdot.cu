// Row-dot contraction on the FP64 tensor pipe, real data:
//
//     out[a][j] = sum_i N[a][i] X[j][i]   (- 1 where j == idx[a])          a < k, j < rows
//
// i.e. (k x n)(n x rows) with BOTH operands stored with the contraction index contiguous.
// It is what the method needs whenever a rank is too large for the register kernels:
//   * X = Ti (A^-T, rows = n), N = the new rows:  out = N A^-1 - I[P,:] = u^T A^-1 of Eq. 5
//      for a whole walker in one read-only pass -- the accept of ranks k > 8
//      and the dense u columns of a general update (f1);
//   * X = C = A^-1[:,P] (rows = k), N = the new rows:  out = R = N C (Eq. 4), the
//     k x k core of a rank-k ratio.
//
// Work item = (walker, tile of 128 rows of X); persistent grid, 8 warps, warp tile 16 rows x KT
// (2 x KT/8 m8n8k4 tiles).  X and N chunks of 32 columns move global -> shared with 16-byte
// cp.async through a ring of stages that runs across work items.  The contraction index of
// mma.sync.m8n8k4.f64 may be permuted freely as long as both fragments agree, so lane (r, q)
// reads the 16-byte pair [i0+2q, i0+2q+1] of its row of X and of its row of N and issues two
// DMMAs: half the fragment loads, all of them 16 bytes wide.  Row stride of the staged chunks =
// 40 doubles (64 B mod 128 B): conflict-free.
#include "lrux_common.cuh"
#include "lrux_internal.h"

namespace lrux {

__device__ __forceinline__ void dmma884r(double& d0, double& d1, double a, double b) {
  asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
               : "+d"(d0), "+d"(d1)
               : "d"(a), "d"(b));
}
__device__ __forceinline__ void rd_cp_async_16(void* smem_dst, const void* gsrc, int src_bytes) {
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;" ::"r"((uint32_t)__cvta_generic_to_shared(smem_dst)),
               "l"(gsrc), "r"(src_bytes)
               : "memory");
}

template <int KT>
__global__ void __launch_bounds__(256, 1) rowdot_dmma_kernel(RowdotArgs A) {
  constexpr int BM = 128, KC = 32, LD = KC + 8, NT = KT / 8, MT = 2;
  constexpr int NS = KT <= 16 ? 4 : 3;
  constexpr int STAGE = (BM + KT) * LD;            // doubles per stage: Xs[BM][LD] | Ns[KT][LD]
  extern __shared__ __align__(128) unsigned char smem_raw[];
  double* ring = (double*)smem_raw;
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int r8 = lane >> 2, q = lane & 3;
  const int n = A.n, rows = A.rows, k = A.k;
  const int count = A.count ? *A.count : (int)A.W;
  const int tiles = (rows + BM - 1) / BM;
  const int nch = (n + KC - 1) / KC;
  const int64_t total = (int64_t)count * tiles;
  const int G = (int)gridDim.x;
  if (total <= (int64_t)blockIdx.x) return;
  const int my_items = (int)((total - blockIdx.x + G - 1) / G);

  auto walker_of = [&](int i, int& tile) {
    const int64_t item = (int64_t)blockIdx.x + (int64_t)i * G;
    tile = (int)(item % tiles);
    const int wi = (int)(item / tiles);
    return A.list ? A.list[wi] : wi;
  };
  auto issue = [&](int w, int tile, int ch, int stage) {
    const double* X = A.X + (size_t)w * A.x_stride;
    const double* N = A.N + (size_t)w * A.n_stride;
    double* Xs = ring + (size_t)stage * STAGE;
    double* Ns = Xs + BM * LD;
    const int i0 = ch * KC;
#pragma unroll
    for (int u = 0; u < BM * (KC / 2) / 256; ++u) {
      const int qd = tid + 256 * u;
      const int r = qd / (KC / 2), c = (qd % (KC / 2)) * 2;
      const bool ok = tile * BM + r < rows && i0 + c < n;
      rd_cp_async_16(Xs + r * LD + c, X + (ok ? (size_t)(tile * BM + r) * A.ldx + i0 + c : 0), ok ? 16 : 0);
    }
#pragma unroll
    for (int u = 0; u < (KT * (KC / 2) + 255) / 256; ++u) {
      const int qd = tid + 256 * u;
      if (qd < KT * (KC / 2)) {
        const int r = qd / (KC / 2), c = (qd % (KC / 2)) * 2;
        const bool ok = r < k && i0 + c < n;
        rd_cp_async_16(Ns + r * LD + c, N + (ok ? (size_t)r * A.ldn + i0 + c : 0), ok ? 16 : 0);
      }
    }
  };

  int p_item = 0, p_ch = 0, p_tile = 0, issued = 0;
  int p_w = walker_of(0, p_tile);
  auto produce = [&]() {
    if (p_item < my_items) {
      issue(p_w, p_tile, p_ch, issued % NS);
      if (++p_ch == nch) {
        p_ch = 0;
        if (++p_item < my_items) p_w = walker_of(p_item, p_tile);
      }
    }
    ++issued;
    asm volatile("cp.async.commit_group;" ::: "memory");
  };
#pragma unroll 1
  for (int s = 0; s < NS - 1; ++s) produce();

  int consumed = 0;
#pragma unroll 1
  for (int i = 0; i < my_items; ++i) {
    int tile;
    const int w = walker_of(i, tile);
    double acc[MT][NT][2];
#pragma unroll
    for (int mt = 0; mt < MT; ++mt)
#pragma unroll
      for (int nt = 0; nt < NT; ++nt) acc[mt][nt][0] = acc[mt][nt][1] = 0.0;
#pragma unroll 1
    for (int ch = 0; ch < nch; ++ch) {
      asm volatile("cp.async.wait_group %0;" ::"n"(NS - 2) : "memory");
      __syncthreads();
      produce();
      const double* Xs = ring + (size_t)(consumed % NS) * STAGE;
      const double* Ns = Xs + BM * LD;
      ++consumed;
#pragma unroll
      for (int c8 = 0; c8 < KC; c8 += 8) {
        double2 af[MT], bf[NT];
#pragma unroll
        for (int mt = 0; mt < MT; ++mt) af[mt] = *(const double2*)(Xs + (warp * 16 + mt * 8 + r8) * LD + c8 + 2 * q);
#pragma unroll
        for (int nt = 0; nt < NT; ++nt) bf[nt] = *(const double2*)(Ns + (nt * 8 + r8) * LD + c8 + 2 * q);
#pragma unroll
        for (int mt = 0; mt < MT; ++mt)
#pragma unroll
          for (int nt = 0; nt < NT; ++nt) dmma884r(acc[mt][nt][0], acc[mt][nt][1], af[mt].x, bf[nt].x);
#pragma unroll
        for (int mt = 0; mt < MT; ++mt)
#pragma unroll
          for (int nt = 0; nt < NT; ++nt) dmma884r(acc[mt][nt][0], acc[mt][nt][1], af[mt].y, bf[nt].y);
      }
    }
    // accumulator of tile (mt, nt): row j = .. + r8 of X, columns a = nt*8 + 2q, +1 of N
    double* out = A.out + (size_t)w * A.o_stride;
    const int32_t* idx = A.idx ? A.idx + (size_t)w * A.idx_stride : nullptr;
#pragma unroll
    for (int mt = 0; mt < MT; ++mt) {
      const int j = tile * BM + warp * 16 + mt * 8 + r8;
      if (j >= rows) continue;
#pragma unroll
      for (int nt = 0; nt < NT; ++nt)
#pragma unroll
        for (int e = 0; e < 2; ++e) {
          const int a = nt * 8 + 2 * q + e;
          if (a < k) {
            double v = acc[mt][nt][e];
            if (idx && idx[a] == j) v -= 1.0;
            out[(size_t)a * A.ldo + j] = v;
          }
        }
    }
  }
  asm volatile("cp.async.wait_group 0;" ::: "memory");
}

// Requires 16-byte aligned rows: n, ldx, ldn even and even walker strides.  Returns the
// number of launches (1), 0 when the shape is not eligible, -1 on a CUDA error.
int launch_rowdot_dmma(const RowdotArgs& A, Ctx& cx, cudaStream_t s) {
  if ((A.n & 1) || (A.ldx & 1) || (A.ldn & 1) || (A.x_stride & 1) || (A.n_stride & 1) || A.k > 64) return 0;
  const int kt = A.k <= 8 ? 8 : A.k <= 16 ? 16 : A.k <= 32 ? 32 : 64;
  const void* kern = kt == 8 ? (const void*)rowdot_dmma_kernel<8> : kt == 16 ? (const void*)rowdot_dmma_kernel<16>
                   : kt == 32 ? (const void*)rowdot_dmma_kernel<32> : (const void*)rowdot_dmma_kernel<64>;
  const int ns = kt <= 16 ? 4 : 3;
  const size_t smem = (size_t)ns * (128 + kt) * 40 * sizeof(double);
  const int occ = cx.configure(kern, 256, smem);
  if (occ < 0) return -1;
  const int64_t items = A.W * ((A.rows + 127) / 128);
  RowdotArgs a = A;
  void* args[1] = {&a};
  if (cudaLaunchKernel(kern, dim3(persistent_grid(cx.num_sms, occ, items)), dim3(256), args, smem, s) != cudaSuccess)
    return -1;
  return 1;
}

}  // namespace lrux
