// C-ABI entry points (include/lrux.h): argument checks, state layout, dispatch.
#include <new>

#include "lrux_internal.h"

namespace lrux {

static inline size_t align_up(size_t x) { return (x + 255) & ~size_t(255); }

size_t state_layout(State* st, void* base, int64_t W, int32_t n, int32_t kmax, int32_t K,
                    int32_t dt, int32_t kind) {
  const size_t e = dt == LRUX_C128 ? 16 : 8;
  const size_t kc = kind == KIND_PF ? 2 * (size_t)kmax : (size_t)kmax;
  const size_t cap = (size_t)K * kc;
  size_t off = 0;
  char* b = (char*)base;
  auto take = [&](size_t bytes) {
    void* p = b ? (void*)(b + off) : nullptr;
    off = align_up(off + bytes);
    return p;
  };
  State s{};
  s.W = W; s.n = n; s.kmax = kmax; s.K = K; s.kc = (int32_t)kc; s.cap = (int32_t)cap;
  s.dt = dt; s.kind = kind;
  s.Ti = take((size_t)W * n * n * e);
  s.phase = take((size_t)W * e);
  s.logabs = (double*)take((size_t)W * 8);
  s.fill = (int32_t*)take((size_t)W * 4);
  s.nupd = (int32_t*)take((size_t)W * 4);
  s.pend_idx = (int32_t*)take((size_t)W * kmax * 4);
  s.pend_ok = (uint8_t*)take((size_t)W);
  s.pend_ratio = take((size_t)W * e);
  s.pend_Rinv = take((size_t)W * kc * kc * e);
  s.pend_C = take((size_t)W * kmax * n * e);
  s.pend_N = take((size_t)W * kmax * n * e);
  if (kind == KIND_DET && kmax > kSmallMaxK) s.pend_D = take((size_t)W * kmax * n * e);
  if (kind == KIND_DET) {
    const size_t nsplit = ((size_t)n + kRatioSlice - 1) / kRatioSlice;
    s.pend_Rpart = take((size_t)W * nsplit * kmax * kmax * e);
    s.pend_cnt = (int32_t*)take((size_t)W * 4);
  }
  if (kind == KIND_PF) {
    s.pend_Y = take((size_t)W * kmax * n * e);
    s.pend_AN = cap ? take((size_t)W * kmax * cap * e) : nullptr;
  } else {
    s.pend_Y = cap ? take((size_t)W * kmax * cap * e) : nullptr;
    s.pend_AN = nullptr;
  }
  s.Abuf = cap ? take((size_t)W * cap * n * e) : nullptr;
  s.Bbuf = cap ? take((size_t)W * cap * n * e) : nullptr;
  if (n >= kBlockedInitMin) {
    s.init_A = take((size_t)W * 32 * n * e);
    s.init_B = take((size_t)W * 32 * n * e);
    s.init_piv = (int32_t*)take((size_t)W * n * 4);
  }
  s.list = (int32_t*)take((size_t)W * 4);
  s.flist = (int32_t*)take((size_t)W * 4);
  s.counters = (int32_t*)take(8 * 4);   // [0] accepted, [1] to flush, [4..7] two uint64 flush totals
  if (st) *st = s;
  return off;
}

static lrux_status_t check_dims(int64_t W, int32_t n, int32_t kmax, int32_t K, int dt, int kind) {
  if (W <= 0 || n <= 0 || kmax <= 0 || kmax > LRUX_MAX_K || K < 0) return LRUX_EINVAL;
  if (dt != LRUX_F64 && dt != LRUX_C128) return LRUX_EINVAL;
  if (kind == KIND_PF && (n % 2 != 0)) return LRUX_EINVAL;
  if (kmax > n) return LRUX_EINVAL;
  // ranks above 8: float64 determinants with immediate updates and even n (tensor-pipe path)
  if (kmax > kSmallMaxK && (kind != KIND_DET || dt != LRUX_F64 || K != 0 || (n & 1))) return LRUX_EUNSUPPORTED;
  // the delayed determinant ratio stages K*kmax coefficients per proposal row in (opt-in)
  // dynamic shared memory; the Pfaffian path has no such limit
  const size_t kt = kmax <= 1 ? 1 : kmax <= 2 ? 2 : kmax <= 4 ? 4 : 8;   // kernels' template rank
  if (kind == KIND_DET && (size_t)K * kmax * kt * (dt == LRUX_C128 ? 16 : 8) > kRatioCoefSmemMax)
    return LRUX_EUNSUPPORTED;
  if (W > (int64_t)2000000000) return LRUX_EINVAL;
  if (n > kRatioSlice * kRatioSplitMax) return LRUX_EUNSUPPORTED;
  // initialisation scratch in one CTA's shared memory: a row + a pivot list (blocked
  // Gauss-Jordan), two rows (Parlett-Reid)
  const size_t e = dt == LRUX_C128 ? 16 : 8;
  if ((size_t)n * (e + 4) > 200 * 1024) return LRUX_EUNSUPPORTED;
  if (kind == KIND_PF && 2 * (size_t)n * e > 200 * 1024) return LRUX_EUNSUPPORTED;
  return LRUX_OK;
}

static lrux_status_t state_bytes(int64_t W, int32_t n, int32_t kmax, int32_t K, lrux_dtype_t dt,
                                 size_t* bytes, int kind) {
  if (!bytes) return LRUX_EINVAL;
  lrux_status_t s = check_dims(W, n, kmax, K, dt, kind);
  if (s != LRUX_OK) return s;
  *bytes = state_layout(nullptr, nullptr, W, n, kmax, K, dt, kind);
  return LRUX_OK;
}

// d_A0 == nullptr with attach == true: build the handle only (lrux_*_attach)
static lrux_status_t init(lrux_handle_t* h, int64_t W, int32_t n, int32_t kmax, int32_t K,
                          lrux_dtype_t dt, const void* d_A0, void* d_state, size_t sb,
                          int32_t* d_info, void* stream, int kind, bool attach = false) {
  if (!h || (!d_A0 && !attach) || !d_state || !d_info) return LRUX_EINVAL;
  lrux_status_t s = check_dims(W, n, kmax, K, dt, kind);
  if (s != LRUX_OK) return s;
  if (((uintptr_t)d_state & 255) != 0) return LRUX_EINVAL;
  size_t need = state_layout(nullptr, nullptr, W, n, kmax, K, dt, kind);
  if (sb < need) return LRUX_EWORKSPACE;
  int dev = 0, sms = 0, optin = 0;
  if (cudaGetDevice(&dev) != cudaSuccess) return LRUX_ECUDA;
  if (cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess ||
      cudaDeviceGetAttribute(&optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev) != cudaSuccess)
    return LRUX_ECUDA;
  lrux_handle_s* hh = new (std::nothrow) lrux_handle_s();
  if (!hh) return LRUX_EINVAL;
  state_layout(&hh->st, d_state, W, n, kmax, K, dt, kind);
  hh->st.info = d_info;
  hh->pending_k = 0;
  hh->launches = 0;
  hh->cx.num_sms = sms;
  hh->cx.smem_optin = optin;
  int nl = attach ? 0
           : kind == KIND_DET ? launch_det_init(hh->st, d_A0, hh->cx, (cudaStream_t)stream)
                              : launch_pf_init(hh->st, d_A0, hh->cx, (cudaStream_t)stream);
  if (nl < 0) {
    delete hh;
    return LRUX_ECUDA;
  }
  hh->launches += nl;
  *h = hh;
  return LRUX_OK;
}

// ---------------------------------------------------------------- launch context
// Static shared memory counts towards the 48 KiB default: opt in from 40 KiB of dynamic
// shared memory on, always to the most this kernel can have (device opt-in maximum minus its
// static part) -- a kernel attribute is shared by every handle of the process, so it must
// never be lowered to what one handle happens to need.
bool Ctx::optin(const void* fn, size_t smem) {
  if (smem <= 40 * 1024) return true;
  cudaFuncAttributes fa;
  if (cudaFuncGetAttributes(&fa, fn) != cudaSuccess) { cudaGetLastError(); return false; }
  const int most = smem_optin - (int)fa.sharedSizeBytes;
  if ((int)smem > most ||
      cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, most) != cudaSuccess) {
    cudaGetLastError();
    return false;
  }
  return true;
}

int Ctx::configure(const void* fn, int threads, size_t smem) {
  for (const Cfg& c : cfgs)
    if (c.fn == fn && c.threads == threads && c.smem == smem && c.cluster == 0) return c.occ;
  if (!optin(fn, smem)) return -1;
  int occ = 0;
  if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, fn, threads, smem) != cudaSuccess || occ < 1) {
    cudaGetLastError();
    return -1;
  }
  cfgs.push_back(Cfg{fn, threads, smem, 0, occ});
  return occ;
}

int Ctx::configure_cluster(const void* fn, int threads, size_t smem, int cluster) {
  for (const Cfg& c : cfgs)
    if (c.fn == fn && c.threads == threads && c.smem == smem && c.cluster == cluster) return c.occ;
  int ncl = 0;
  if (optin(fn, smem)) {
    cudaLaunchConfig_t cfg = {};
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeClusterDimension;
    attr[0].val.clusterDim.x = cluster;
    attr[0].val.clusterDim.y = 1;
    attr[0].val.clusterDim.z = 1;
    cfg.blockDim = dim3(threads);
    cfg.gridDim = dim3(cluster);
    cfg.dynamicSmemBytes = smem;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    if (cudaOccupancyMaxActiveClusters(&ncl, fn, &cfg) != cudaSuccess || ncl < 0) {
      cudaGetLastError();
      ncl = 0;
    }
  }
  cfgs.push_back(Cfg{fn, threads, smem, cluster, ncl});
  return ncl;
}

}  // namespace lrux

using namespace lrux;

#define LRUX_CHECK_HANDLE(h, KIND_)          \
  if (!(h)) return LRUX_EINVAL;              \
  if ((h)->st.kind != (KIND_)) return LRUX_ESTATE;

#define LRUX_COUNT(h, expr)          \
  do {                               \
    int nl__ = (expr);               \
    if (nl__ < 0) return LRUX_ECUDA; \
    (h)->launches += nl__;           \
  } while (0)

extern "C" {

lrux_status_t lrux_det_state_bytes(int64_t W, int32_t n, int32_t kmax, int32_t K, lrux_dtype_t dt,
                                   size_t* bytes) {
  return state_bytes(W, n, kmax, K, dt, bytes, KIND_DET);
}
lrux_status_t lrux_pf_state_bytes(int64_t W, int32_t n, int32_t kmax, int32_t K, lrux_dtype_t dt,
                                  size_t* bytes) {
  return state_bytes(W, n, kmax, K, dt, bytes, KIND_PF);
}

lrux_status_t lrux_det_init(lrux_handle_t* h, int64_t W, int32_t n, int32_t kmax, int32_t K,
                            lrux_dtype_t dt, const void* d_A0, void* d_state, size_t state_bytes,
                            int32_t* d_info, void* stream) {
  return init(h, W, n, kmax, K, dt, d_A0, d_state, state_bytes, d_info, stream, KIND_DET);
}
lrux_status_t lrux_pf_init(lrux_handle_t* h, int64_t W, int32_t n, int32_t kmax, int32_t K,
                           lrux_dtype_t dt, const void* d_A0, void* d_state, size_t state_bytes,
                           int32_t* d_info, void* stream) {
  return init(h, W, n, kmax, K, dt, d_A0, d_state, state_bytes, d_info, stream, KIND_PF);
}

lrux_status_t lrux_det_attach(lrux_handle_t* h, int64_t W, int32_t n, int32_t kmax, int32_t K,
                              lrux_dtype_t dt, void* d_state, size_t state_bytes, int32_t* d_info) {
  return init(h, W, n, kmax, K, dt, nullptr, d_state, state_bytes, d_info, nullptr, KIND_DET, true);
}
lrux_status_t lrux_pf_attach(lrux_handle_t* h, int64_t W, int32_t n, int32_t kmax, int32_t K,
                             lrux_dtype_t dt, void* d_state, size_t state_bytes, int32_t* d_info) {
  return init(h, W, n, kmax, K, dt, nullptr, d_state, state_bytes, d_info, nullptr, KIND_PF, true);
}

lrux_status_t lrux_det_ratio(lrux_handle_t h, int32_t k, const int32_t* d_idx, const void* d_rows,
                             void* d_ratio, void* stream) {
  LRUX_CHECK_HANDLE(h, KIND_DET);
  if (k < 1 || k > h->st.kmax || !d_idx || !d_rows || !d_ratio) return LRUX_EINVAL;
  if (k > kSmallMaxK)
    LRUX_COUNT(h, launch_det_ratio_big(h->st, k, d_idx, d_rows, d_ratio, h->cx, (cudaStream_t)stream));
  else
    LRUX_COUNT(h, launch_det_ratio(h->st, k, d_idx, d_rows, d_ratio, h->cx, (cudaStream_t)stream));
  h->pending_k = k;
  h->pending_general = false;
  return LRUX_OK;
}
lrux_status_t lrux_det_ratio_general(lrux_handle_t h, int32_t k, int32_t u_kd, const void* d_u_dense,
                                     const int32_t* d_u_idx, int32_t v_kd, const void* d_v_dense,
                                     const int32_t* d_v_idx, void* d_ratio, void* stream) {
  LRUX_CHECK_HANDLE(h, KIND_DET);
  if (k < 1 || k > h->st.kmax || k > LRUX_MAX_K_GENERAL || u_kd < 0 || u_kd > k || v_kd < 0 || v_kd > k || !d_ratio)
    return LRUX_EINVAL;
  if ((u_kd > 0 && !d_u_dense) || (u_kd < k && !d_u_idx) || (v_kd > 0 && !d_v_dense) || (v_kd < k && !d_v_idx))
    return LRUX_EINVAL;
  // the proposal is evaluated against, and applied to, the folded inverse
  if (h->st.K > 0) LRUX_COUNT(h, launch_det_flush(h->st, true, h->cx, (cudaStream_t)stream));
  const int nl = launch_det_ratio_general(h->st, k, u_kd, d_u_dense, d_u_idx, v_kd, d_v_dense, d_v_idx, d_ratio,
                                          h->cx, (cudaStream_t)stream);
  if (nl == -2) return LRUX_EUNSUPPORTED;
  if (nl < 0) return LRUX_ECUDA;
  h->launches += nl;
  h->pending_k = k;
  h->pending_general = true;
  return LRUX_OK;
}
lrux_status_t lrux_pf_ratio(lrux_handle_t h, int32_t k, const int32_t* d_idx, const void* d_rows,
                            void* d_ratio, void* stream) {
  LRUX_CHECK_HANDLE(h, KIND_PF);
  if (k < 1 || k > h->st.kmax || !d_idx || !d_rows || !d_ratio) return LRUX_EINVAL;
  LRUX_COUNT(h, launch_pf_ratio(h->st, k, d_idx, d_rows, d_ratio, h->cx, (cudaStream_t)stream));
  h->pending_k = k;
  return LRUX_OK;
}

lrux_status_t lrux_det_accept(lrux_handle_t h, const uint8_t* d_mask, void* stream) {
  LRUX_CHECK_HANDLE(h, KIND_DET);
  if (!d_mask) return LRUX_EINVAL;
  if (h->pending_k == 0) return LRUX_ESTATE;
  if (h->pending_general)
    LRUX_COUNT(h, launch_det_accept_general(h->st, h->pending_k, d_mask, h->cx, (cudaStream_t)stream));
  else if (h->pending_k > kSmallMaxK)
    LRUX_COUNT(h, launch_det_accept_big(h->st, h->pending_k, d_mask, h->cx, (cudaStream_t)stream));
  else
    LRUX_COUNT(h, launch_det_accept(h->st, h->pending_k, d_mask, h->cx, (cudaStream_t)stream));
  h->pending_k = 0;
  h->pending_general = false;
  return LRUX_OK;
}
lrux_status_t lrux_pf_accept(lrux_handle_t h, const uint8_t* d_mask, void* stream) {
  LRUX_CHECK_HANDLE(h, KIND_PF);
  if (!d_mask) return LRUX_EINVAL;
  if (h->pending_k == 0) return LRUX_ESTATE;
  LRUX_COUNT(h, launch_pf_accept(h->st, h->pending_k, d_mask, h->cx, (cudaStream_t)stream));
  h->pending_k = 0;
  return LRUX_OK;
}

lrux_status_t lrux_det_flush(lrux_handle_t h, void* stream) {
  LRUX_CHECK_HANDLE(h, KIND_DET);
  if (h->st.K == 0) return LRUX_OK;
  LRUX_COUNT(h, launch_det_flush(h->st, true, h->cx, (cudaStream_t)stream));
  return LRUX_OK;
}
lrux_status_t lrux_pf_flush(lrux_handle_t h, void* stream) {
  LRUX_CHECK_HANDLE(h, KIND_PF);
  if (h->st.K == 0) return LRUX_OK;
  LRUX_COUNT(h, launch_pf_flush(h->st, true, h->cx, (cudaStream_t)stream));
  return LRUX_OK;
}

lrux_status_t lrux_det_get_amplitude(lrux_handle_t h, void* d_phase, double* d_logabs,
                                     void* stream) {
  LRUX_CHECK_HANDLE(h, KIND_DET);
  if (!d_phase || !d_logabs) return LRUX_EINVAL;
  LRUX_COUNT(h, launch_get_amplitude(h->st, d_phase, d_logabs, (cudaStream_t)stream));
  return LRUX_OK;
}
lrux_status_t lrux_pf_get_amplitude(lrux_handle_t h, void* d_phase, double* d_logabs,
                                    void* stream) {
  LRUX_CHECK_HANDLE(h, KIND_PF);
  if (!d_phase || !d_logabs) return LRUX_EINVAL;
  LRUX_COUNT(h, launch_get_amplitude(h->st, d_phase, d_logabs, (cudaStream_t)stream));
  return LRUX_OK;
}

lrux_status_t lrux_det_get_inverse(lrux_handle_t h, void* d_out, void* stream) {
  LRUX_CHECK_HANDLE(h, KIND_DET);
  if (!d_out) return LRUX_EINVAL;
  if (h->st.K > 0) LRUX_COUNT(h, launch_det_flush(h->st, true, h->cx, (cudaStream_t)stream));
  LRUX_COUNT(h, launch_get_inverse(h->st, d_out, (cudaStream_t)stream));
  return LRUX_OK;
}
lrux_status_t lrux_pf_get_inverse(lrux_handle_t h, void* d_out, void* stream) {
  LRUX_CHECK_HANDLE(h, KIND_PF);
  if (!d_out) return LRUX_EINVAL;
  if (h->st.K > 0) LRUX_COUNT(h, launch_pf_flush(h->st, true, h->cx, (cudaStream_t)stream));
  LRUX_COUNT(h, launch_get_inverse(h->st, d_out, (cudaStream_t)stream));
  return LRUX_OK;
}

static lrux_status_t refresh(lrux_handle_t h, const void* d_A, void* stream) {
  if (!d_A) return LRUX_EINVAL;
  LRUX_COUNT(h, launch_refresh(h->st, d_A, h->cx, (cudaStream_t)stream));
  h->pending_k = 0;
  return LRUX_OK;
}
lrux_status_t lrux_det_refresh(lrux_handle_t h, const void* d_A, void* stream) {
  LRUX_CHECK_HANDLE(h, KIND_DET);
  return refresh(h, d_A, stream);
}
lrux_status_t lrux_pf_refresh(lrux_handle_t h, const void* d_A, void* stream) {
  LRUX_CHECK_HANDLE(h, KIND_PF);
  return refresh(h, d_A, stream);
}

lrux_status_t lrux_get_flush_count(lrux_handle_t h, int64_t* d_out, void* stream) {
  if (!h || !d_out) return LRUX_EINVAL;
  if (cudaMemcpyAsync(d_out, h->st.counters + 4, 16, cudaMemcpyDeviceToDevice,
                      (cudaStream_t)stream) != cudaSuccess)
    return LRUX_ECUDA;
  return LRUX_OK;
}

lrux_status_t lrux_launch_count(lrux_handle_t h, int64_t* count) {
  if (!h || !count) return LRUX_EINVAL;
  *count = h->launches;
  return LRUX_OK;
}

const char* lrux_kernel_name(lrux_handle_t h, int32_t cls) {
  if (!h || cls < 0 || cls >= LRUX_PROF_NCLASS || !h->cx.last[cls]) return "";
  return h->cx.last[cls];
}

lrux_status_t lrux_profile_enable(lrux_handle_t h, int32_t on) {
  if (!h) return LRUX_EINVAL;
  h->cx.prof.on = on != 0;
  return LRUX_OK;
}

lrux_status_t lrux_profile_read(lrux_handle_t h, int32_t cls, double* ms_total, int64_t* launches) {
  if (!h || !ms_total || !launches || cls < 0 || cls >= LRUX_PROF_NCLASS) return LRUX_EINVAL;
  double ms = 0.0;
  int64_t cnt = 0;
  for (auto& r : h->cx.prof.recs[cls]) {
    float t = 0.f;
    if (cudaEventSynchronize(r.b) != cudaSuccess || cudaEventElapsedTime(&t, r.a, r.b) != cudaSuccess)
      return LRUX_ECUDA;
    ms += t;
    ++cnt;
    h->cx.prof.pool.push_back(r);
  }
  h->cx.prof.recs[cls].clear();
  *ms_total = ms;
  *launches = cnt;
  return LRUX_OK;
}

lrux_status_t lrux_destroy(lrux_handle_t h) {
  if (!h) return LRUX_EINVAL;
  for (int c = 0; c < LRUX_PROF_NCLASS; ++c)
    for (auto& r : h->cx.prof.recs[c]) h->cx.prof.pool.push_back(r);
  for (auto& r : h->cx.prof.pool) { cudaEventDestroy(r.a); cudaEventDestroy(r.b); }
  delete h;
  return LRUX_OK;
}

const char* lrux_status_string(lrux_status_t s) {
  switch (s) {
    case LRUX_OK: return "LRUX_OK";
    case LRUX_EINVAL: return "LRUX_EINVAL: invalid argument";
    case LRUX_ESTATE: return "LRUX_ESTATE: call not valid in this state";
    case LRUX_EWORKSPACE: return "LRUX_EWORKSPACE: state buffer too small";
    case LRUX_EUNSUPPORTED: return "LRUX_EUNSUPPORTED";
    case LRUX_ECUDA: return "LRUX_ECUDA: CUDA error";
    case LRUX_ELIMIT: return "LRUX_ELIMIT: W*k*k*sizeof(elem) exceeds LRUX_NOALLOC_SCRATCH_BYTES (1 MiB)";
  }
  return "LRUX_?";
}

}  // extern "C"
