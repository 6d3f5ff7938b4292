// Host-side handle, state layout and kernel-launcher declarations.
#pragma once
#include <cuda_runtime.h>
#include <stddef.h>
#include <stdint.h>

#include <vector>

#include "lrux.h"

namespace lrux {

enum Kind { KIND_DET = 0, KIND_PF = 1 };
constexpr int kRatioSlice = 256;       // columns of A^-1[:,P] handled by one CTA of the det ratio
constexpr int kRatioSplitMax = 64;     // => n <= 16384
constexpr int kSmallMaxK = 8;          // largest rank of the register / shared-memory kernels (= kMaxK)
constexpr int kBigMaxK = 64;           // largest rank (float64 determinants, K = 0, k > 8: lrux_det_big.cu)
constexpr int kBlockedInitMin = 768;   // blocked (panel + DMMA) initialisation from this n on
constexpr size_t kRatioCoefSmemMax = 160 * 1024;   // det delayed ratio: K*kmax*KT coefficients staged per CTA

// Views into the caller-owned d_state buffer (all device pointers, 256 B aligned).
// Element type is double (LRUX_F64) or interleaved complex (LRUX_C128); sizes
// below are in elements of that type unless noted.
struct State {
  int64_t W;
  int32_t n, kmax, K, kc;  // kc = core size: kmax (det) or 2*kmax (pf)
  int32_t cap;             // delay-buffer capacity in columns: K*kmax (det), K*2*kmax (pf)
  int32_t dt, kind;
  // det: Ti[w][j][i] = (A^-1)[i][j]  (A^-T row-major);  pf: Ti[w] = A^-1 row-major
  void* Ti;
  void* phase;       // [W] elem
  double* logabs;    // [W]
  int32_t* fill;     // [W] columns in use in the delay buffer
  int32_t* nupd;     // [W] updates held in the delay buffer
  int32_t* pend_idx; // [W][kmax]
  uint8_t* pend_ok;  // [W] 1 = valid proposal with finite non-zero R
  void* pend_ratio;  // [W] elem
  void* pend_Rinv;   // [W][kc][kc]
  void* pend_C;      // [W][kmax][n]  det: effective A^-1[:,P] (= a_tau, Eq. 14); pf: A^-1[:,P]
  void* pend_N;      // [W][kmax][n]  new rows
  void* pend_Y;      // pf: [W][kmax][n]  A^-1 N ; det delayed: [W][kmax][cap] N * Abuf^T
  void* pend_AN;     // pf delayed: [W][kmax][cap]  N * Abuf^T
  void* pend_D;      // det, kmax > 8: [W][kmax][n]  N A^-1 - I[P,:], then R^-1 times it
  void* pend_Rpart;  // det: [W][kRatioSplitMax][kmax*kmax] partial R of each column slice
  int32_t* pend_cnt; // det: [W] slices of the current ratio call that have finished
  void* init_A;      // n >= kBlockedInitMin: [W][32][n] scratch of the blocked initialisation
  void* init_B;      //                       [W][32][n]
  int32_t* init_piv; //                       [W][n] pivot rows
  void* Abuf;        // [W][cap][n]  det: a_t (Eq. 10);  pf: a'_t (Eq. 25)
  void* Bbuf;        // [W][cap][n]  det: b_t (Eq. 11);  pf: a'_t R_t^-1
  int32_t* list;     // [W] accepted walkers (compacted)
  int32_t* flist;    // [W] walkers to flush (compacted)
  int32_t* counters; // [8]: 0 = accepted count, 1 = flush count
  int32_t* info;     // caller's d_info
};

// Optional per-class kernel timing (lrux_profile_*): event pairs recorded on the
// caller's stream around the library's own launches.
struct Prof {
  struct Rec { cudaEvent_t a, b; };
  bool on = false;
  std::vector<Rec> recs[LRUX_PROF_NCLASS];
  std::vector<Rec> pool;
  Rec get() {
    Rec r{};
    if (!pool.empty()) { r = pool.back(); pool.pop_back(); return r; }
    cudaEventCreate(&r.a);
    cudaEventCreate(&r.b);
    return r;
  }
};
struct ProfScope {
  Prof* p; int cls; cudaStream_t s; Prof::Rec r;
  ProfScope(Prof* p_, int cls_, cudaStream_t s_) : p(p_ && p_->on ? p_ : nullptr), cls(cls_), s(s_) {
    if (p) { r = p->get(); cudaEventRecord(r.a, s); }
  }
  ~ProfScope() {
    if (p) { cudaEventRecord(r.b, s); p->recs[cls].push_back(r); }
  }
};

// out[a][j] = sum_i N[a][i] X[j][i] (- 1 where j == idx[a]) on the FP64 tensor pipe
// (lrux_rowdot.cu); per-walker strides and leading dimensions in elements.
struct RowdotArgs {
  const double* X; size_t x_stride; int rows, ldx;
  const double* N; size_t n_stride; int ldn;
  int n, k;
  double* out; size_t o_stride; int ldo;
  const int32_t* list;    // walker list (nullptr: walkers 0..W-1)
  const int32_t* count;   // device count of listed walkers (nullptr: W)
  int64_t W;
  const int32_t* idx; int idx_stride;   // subtract 1 at out[a][idx[a]] (nullptr: nothing)
};

// Per-handle launch context (host only): what a launcher needs besides the state views.
// Kernel attributes and occupancy are queried ONCE per (kernel, block size, shared memory)
// and cached here, so that the per-step calls enqueue launches and do nothing else on
// the host; `last[cls]` names the kernel most recently enqueued for each class
// (lrux_kernel_name: kernels are selected by shape only, this is how tests and bench.py
// learn which one a shape takes).
struct Ctx {
  int num_sms = 0;
  int smem_optin = 0;                     // cudaDevAttrMaxSharedMemoryPerBlockOptin
  Prof prof;
  const char* last[LRUX_PROF_NCLASS] = {nullptr, nullptr, nullptr, nullptr, nullptr};
  struct Cfg { const void* fn; int threads; size_t smem; int cluster; int occ; };
  std::vector<Cfg> cfgs;
  // Resident CTAs per SM of `fn` at this block size / dynamic shared memory (>= 1), or
  // -1 on a CUDA error.  Opts the kernel into large dynamic shared memory when needed.
  int configure(const void* fn, int threads, size_t smem);
  // Co-resident clusters of `cluster` CTAs on the whole GPU (0: not launchable), cached.
  int configure_cluster(const void* fn, int threads, size_t smem, int cluster);
  bool optin(const void* fn, size_t smem);
  void name(int cls, const char* kernel) { last[cls] = kernel; }
};

}  // namespace lrux

struct lrux_handle_s {
  lrux::State st;
  lrux::Ctx cx;
  int32_t pending_k;  // 0 = nothing pending
  bool pending_general = false;   // the pending proposal came from lrux_det_ratio_general
  int64_t launches;
};

namespace lrux {

size_t state_layout(State* st, void* base, int64_t W, int32_t n, int32_t kmax, int32_t K,
                    int32_t dt, int32_t kind);

static inline int persistent_grid(int num_sms, int ctas_per_sm, int64_t max_items) {
  int64_t g = (int64_t)num_sms * ctas_per_sm;
  if (g > max_items) g = max_items;
  return g < 1 ? 1 : (int)g;
}
static inline int round_kt(int k) { return k <= 1 ? 1 : k <= 2 ? 2 : k <= 4 ? 4 : 8; }

// launchers (each returns the number of kernels it enqueued, or -1 on a CUDA error)
int launch_det_init(const State& st, const void* d_A0, Ctx& cx, cudaStream_t s);
int launch_pf_update_dmma(const State& st, int k, Ctx& cx, cudaStream_t s, bool probe = false);
int launch_pf_init(const State& st, const void* d_A0, Ctx& cx, cudaStream_t s);
int launch_refresh(const State& st, const void* d_A, Ctx& cx, cudaStream_t s);
// blocked in-place inverse of st.Ti (lrux_init_blocked.cu); 0 = not applicable
int launch_gj_blocked(const State& st, bool write_amp, Ctx& cx, cudaStream_t s);
int launch_det_ratio(const State& st, int k, const int32_t* d_idx, const void* d_rows,
                     void* d_ratio, Ctx& cx, cudaStream_t s);
int launch_det_accept(const State& st, int k, const uint8_t* d_mask, Ctx& cx, cudaStream_t s);
int launch_det_flush(const State& st, bool all, Ctx& cx, cudaStream_t s);
int launch_pf_ratio(const State& st, int k, const int32_t* d_idx, const void* d_rows,
                    void* d_ratio, Ctx& cx, cudaStream_t s);
int launch_pf_accept(const State& st, int k, const uint8_t* d_mask, Ctx& cx, cudaStream_t s);
int launch_pf_flush(const State& st, bool all, Ctx& cx, cudaStream_t s);
// TMA-staged immediate det update for large rows (lrux_det_tma.cu): 1 = launched,
// 0 = shape not eligible, -1 = CUDA error.  probe = true: eligibility only, nothing launched.
int launch_det_update_tma(const State& st, int k, Ctx& cx, cudaStream_t s, bool probe = false);
// immediate det update on the FP64 tensor pipe, real data (lrux_det_dmma.cu): same return codes
int launch_det_update_dmma(const State& st, int k, Ctx& cx, cudaStream_t s, bool probe = false);
// general update factors (lrux_general.cu); ratio: -2 = shape not supported
int launch_det_ratio_general(const State& st, int k, int u_kd, const void* u_dense, const int32_t* u_idx,
                             int v_kd, const void* v_dense, const int32_t* v_idx, void* ratio, Ctx& cx,
                             cudaStream_t s);
int launch_det_accept_general(const State& st, int k, const uint8_t* mask, Ctx& cx, cudaStream_t s);
int launch_rowdot_dmma(const RowdotArgs& A, Ctx& cx, cudaStream_t s);
// ranks 8 < k <= 64, float64, K = 0 (lrux_det_big.cu)
int launch_det_ratio_big(const State& st, int k, const int32_t* d_idx, const void* d_rows, void* d_ratio,
                         Ctx& cx, cudaStream_t s);
int launch_det_accept_big(const State& st, int k, const uint8_t* mask, Ctx& cx, cudaStream_t s);
// DMMA flush of the delay buffers, det and pf (lrux_flush.cu)
int launch_flush_dmma(const State& st, Ctx& cx, cudaStream_t s);
// shared between det and pf (defined in lrux_det.cu)
int launch_select(const State& st, const uint8_t* mask, cudaStream_t s);
int launch_post(const State& st, int ncols, cudaStream_t s);
int launch_flush_select_all(const State& st, cudaStream_t s);
int launch_flush_clear(const State& st, cudaStream_t s);
int launch_get_amplitude(const State& st, void* d_phase, double* d_logabs, cudaStream_t s);
int launch_get_inverse(const State& st, void* d_out, cudaStream_t s);

}  // namespace lrux
