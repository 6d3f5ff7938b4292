/*
 * lrux.h -- C ABI of the B200-native low-rank determinant / Pfaffian update library.
 *
 * Hot path of "lrux: Fast low-rank updates of determinants and Pfaffians"
 * (arxiv/paper_2602_05255; citations are PAPER.md line numbers) for W independent
 * Monte-Carlo walkers, every step running in hand-written sm_100a CUDA kernels.
 *
 * Conventions
 *  - Every d_* pointer is DEVICE memory owned by the caller.  The library never
 *    allocates or frees device memory and holds no global state; the only host
 *    allocation is the small handle.  (One exception, stated at its declaration: the
 *    fixed scratch array of lrux_det_ratio_noalloc.)  `d_state` and `d_info` must outlive the handle.
 *  - `stream` is a cudaStream_t passed as void*.  Every call is asynchronous and
 *    stream-ordered on it; no call synchronises the device.
 *  - Matrices are row-major.  LRUX_C128 data is interleaved (re,im) doubles at the
 *    ABI; every LRUX_C128 array must be 16-byte aligned (the kernels move a complex
 *    element with one 16-byte access).  All transposes in the method are plain, never conjugate.
 *  - Host-detectable misuse returns a status and does nothing.  Conditions only
 *    visible on the device set sticky bits in d_info[w] and never trap:
 *      1 = singular A0 at init (zero pivot)
 *      2 = proposal index out of range or duplicated (ratio returned as NaN)
 *      4 = accepted update with singular / non-finite R (state left unchanged,
 *          treated as rejected)
 */
#ifndef LRUX_H_
#define LRUX_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define LRUX_MAX_K 64 /* largest kmax accepted by *_init; kmax > 8 (backflow-sized ranks):
                         float64 determinants with K = 0 and even n only, else LRUX_EUNSUPPORTED */
#define LRUX_MAX_K_GENERAL 8 /* largest rank of lrux_det_ratio_general */

typedef struct lrux_handle_s* lrux_handle_t; /* small HOST object */
typedef enum { LRUX_F64 = 0, LRUX_C128 = 1 } lrux_dtype_t;
typedef enum {
  LRUX_OK = 0,
  LRUX_EINVAL = 1,      /* bad size / odd n for Pf / k > kmax / null pointer */
  LRUX_ESTATE = 2,      /* accept without a pending ratio; det call on a pf handle */
  LRUX_EWORKSPACE = 3,  /* state_bytes too small */
  LRUX_EUNSUPPORTED = 4, /* n beyond the initialisation kernels' shared-memory scratch (det:
                            n*(sizeof(elem)+4) > 200 KiB, i.e. n > 16384 f64 / 10240 c128; pf:
                            2*n*sizeof(elem) > 200 KiB), or a determinant delay depth with
                            K*kmax*kt*sizeof(elem) > 160 KiB (kt = kmax rounded up to 1,2,4,8) */
  LRUX_ECUDA = 5,       /* a CUDA launch failed */
  LRUX_ELIMIT = 6       /* lrux_det_ratio_noalloc: problem larger than the fixed scratch array */
} lrux_status_t;

/* ---------------------------------------------------------------- determinant
 * State per walker: A^{-1} (stored transposed, so that the k columns a row
 * replacement needs are contiguous), the amplitude det A as (phase, log|det|)
 * (cf. slogpf), a pending proposal, and -- when K > 0 -- the delay
 * buffers a_t, b_t of Eq. 10-11.
 */

/* Bytes of d_state needed for W walkers of n x n matrices, proposals of at most
 * kmax rows and delay depth K (0 = immediate updates). */
lrux_status_t lrux_det_state_bytes(int64_t W, int32_t n, int32_t kmax, int32_t K,
                                   lrux_dtype_t dt, size_t* bytes);

/* Build A^{-1} and (phase, log|det A|) per walker by partial-pivot elimination
 * (the O(n^3) seed of PAPER.md:74-75, 97-98, 203).
 *   d_A0    [W][n][n] row-major, read only
 *   d_state caller-owned buffer of >= state_bytes bytes, 256-byte aligned
 *   d_info  [W] int32, zeroed by this call, then sticky (see bits above) */
lrux_status_t lrux_det_init(lrux_handle_t* h, int64_t W, int32_t n, int32_t kmax, int32_t K,
                            lrux_dtype_t dt, const void* d_A0, void* d_state,
                            size_t state_bytes, int32_t* d_info, void* stream);

/* One proposal per walker: replace the k rows d_idx[w][0..k) of A_w by the new
 * rows d_rows[w][a][0..n) (Eq. 8 with one-hot v).  Writes
 * r_w = det A'_w / det A_w = det(1 + u^T A^{-1} v) (Eq. 2-4) to
 * d_ratio[w], evaluated against the effective current inverse (Eq. 13 when the
 * delay buffer is non-empty), and leaves the proposal pending.
 * 1 <= k <= kmax, indices distinct in [0,n).  A second ratio before accept
 * replaces the pending proposal.  d_idx/d_rows need only stay valid until this
 * call's work completes on `stream`. */
lrux_status_t lrux_det_ratio(lrux_handle_t h, int32_t k, const int32_t* d_idx /*[W][k]*/,
                             const void* d_rows /*[W][k][n]*/, void* d_ratio /*[W]*/,
                             void* stream);

/* General rank-k update A'_w = A_w + v_w u_w^T (Eq. 2) with each n x k factor in
 * the paper's tuple form (Eq. 6-9): its first kd columns DENSE, the remaining
 * k - kd columns ONE-HOT e_idx -- so a row replacement is (u dense, v one-hot: Eq. 6, 8), a
 * column replacement (u one-hot, v dense: Eq. 7), a simultaneous row + column replacement the
 * mixed tuples of Eq. 9, and kd = k on both sides the fully dense update of Eq. 2-5.  NOTE
 * the dense columns are the UPDATE (A' - A), as in the paper's statement, not the new rows
 * lrux_det_ratio takes.
 *   d_u_dense [W][u_kd][n]  column a of u_w as a contiguous vector     d_u_idx [W][k-u_kd]
 *   d_v_dense [W][v_kd][n]                                             d_v_idx [W][k-v_kd]
 * (a pointer may be NULL when its count is 0).  Writes r_w = det(1 + u^T A^-1 v) (Eq. 3-4) to
 * d_ratio[w] and leaves the proposal pending for lrux_det_accept, which applies Eq. 5.  One-hot
 * columns cost O(n) gathers; every dense column makes the ratio itself an
 * O(n^2) pass over the inverse.  On a handle with K > 0 the delay buffers are folded first
 * (the proposal is evaluated against, and applied at once to, the folded inverse).  1 <= k <=
 * min(kmax, LRUX_MAX_K_GENERAL); an index outside [0,n) sets info bit 2 (ratio NaN).
 * LRUX_EUNSUPPORTED when v_kd * n * sizeof(elem) > 200 KiB. */
lrux_status_t lrux_det_ratio_general(lrux_handle_t h, int32_t k, int32_t u_kd, const void* d_u_dense,
                                     const int32_t* d_u_idx, int32_t v_kd, const void* d_v_dense,
                                     const int32_t* d_v_idx, void* d_ratio, void* stream);

/* Apply the pending proposal where d_mask[w] != 0: Woodbury update of the stored
 * inverse (Eq. 5) when K == 0, else append (a_t, b_t) to the delay
 * buffer (Eq. 14-15) and fold the buffer of every walker whose
 * depth reached K (Eq. 12).  Amplitude *= r.  Clears the pending
 * proposal of every walker. */
lrux_status_t lrux_det_accept(lrux_handle_t h, const uint8_t* d_mask /*[W]*/, void* stream);

/* Fold every non-empty delay buffer into A^{-1} (Eq. 12). No-op when K == 0. */
lrux_status_t lrux_det_flush(lrux_handle_t h, void* stream);

/* d_phase [W] elements (+-1 real, unit complex), d_logabs [W] doubles. */
lrux_status_t lrux_det_get_amplitude(lrux_handle_t h, void* d_phase, double* d_logabs,
                                     void* stream);
/* d_out [W][n][n] row-major A^{-1}.  Implies flush. */
lrux_status_t lrux_det_get_inverse(lrux_handle_t h, void* d_out, void* stream);

/* ---------------------------------------------------------------- Pfaffian
 * A_w is skew-symmetric, n even.  Replacing the orbital in slot p changes row p
 * and column p of A (Eq. 23-24): a rank-2k skew update
 * A' = A - u J u^T (Eq. 16).  State: A^{-1} (exactly skew), the
 * amplitude pf A as (phase, log|pf|), pending proposal, and for K > 0 the
 * buffers a_t, R_t^{-1} of Eq. 25-26.
 */
lrux_status_t lrux_pf_state_bytes(int64_t W, int32_t n, int32_t kmax, int32_t K,
                                  lrux_dtype_t dt, size_t* bytes);
/* d_A0 [W][n][n]: only the strict upper triangle is read.  pf by Parlett-Reid
 * elimination with pivoting (PAPER.md:445 leaves the algorithm open). */
lrux_status_t lrux_pf_init(lrux_handle_t* h, int64_t W, int32_t n, int32_t kmax, int32_t K,
                           lrux_dtype_t dt, const void* d_A0, void* d_state,
                           size_t state_bytes, int32_t* d_info, void* stream);
/* d_rows[w][a][0..n) is the NEW row d_idx[w][a] of A' (so column d_idx[w][a] is
 * its negative), including the crossing entries A'[p_a][p_b]; the entry at its
 * own index p_a is ignored (zero diagonal).  r_w = pf A'/pf A = pf R / pf J
 * (Eq. 19-20). */
lrux_status_t lrux_pf_ratio(lrux_handle_t h, int32_t k, const int32_t* d_idx,
                            const void* d_rows, void* d_ratio, void* stream);
/* Eq. 21 (k=1: Eq. 22), with an exactly skew R^{-1}; delayed:
 * Eq. 28 append, Eq. 26 fold. */
lrux_status_t lrux_pf_accept(lrux_handle_t h, const uint8_t* d_mask, void* stream);
lrux_status_t lrux_pf_flush(lrux_handle_t h, void* stream);
lrux_status_t lrux_pf_get_amplitude(lrux_handle_t h, void* d_phase, double* d_logabs,
                                    void* stream);
lrux_status_t lrux_pf_get_inverse(lrux_handle_t h, void* d_out, void* stream);

/* ---------------------------------------------------------------- attach (checkpoint / resume)
 * The walker state lives entirely in the caller's d_state buffer (plus d_info), so a
 * byte copy of that buffer taken while no proposal is pending is a checkpoint.
 * lrux_*_attach builds a handle over such a buffer WITHOUT running the O(n^3)
 * initialisation: same (W, n, kmax, K, dt) as the lrux_*_init that produced it, buffer
 * 256-byte aligned.  Launches nothing; d_info is used as is (not zeroed). */
lrux_status_t lrux_det_attach(lrux_handle_t* h, int64_t W, int32_t n, int32_t kmax, int32_t K,
                              lrux_dtype_t dt, void* d_state, size_t state_bytes,
                              int32_t* d_info);
lrux_status_t lrux_pf_attach(lrux_handle_t* h, int64_t W, int32_t n, int32_t kmax, int32_t K,
                             lrux_dtype_t dt, void* d_state, size_t state_bytes, int32_t* d_info);

/* ---------------------------------------------------------------- refresh (accuracy guard)
 * SURVEY.md §8(f) f3.  The paper only advises double precision against the error that
 * accumulates in a tracked inverse and is silent on recomputation
 * (reading 18); plain fp64 Woodbury on the paper's workloads drifts to 1e-9
 * relative in a ratio after a few hundred accepted updates (reading 14).
 * lrux_*_refresh rebuilds A^-1 and the amplitude (phase, log abs) of EVERY walker from
 * scratch from the caller's current matrices, with the kernels of lrux_*_init (step a0),
 * on the existing handle: d_A is [W][n][n] row-major DEVICE memory, the matrices the
 * walkers have reached (the library stores no A; Pf: only the strict upper triangle is
 * read), valid until the work completes on `stream`.  Unflushed delay factors are
 * discarded (they describe the same A), a pending proposal is dropped, d_info bit 1 is
 * re-evaluated (set again if a matrix is singular; that walker's state is then
 * undefined), bits 2 and 4 and the flush totals are kept.  Cost O(n^3) per walker: call
 * it on a schedule (every few hundred accepted updates), not per step.  Asynchronous,
 * stream-ordered.  Errors: LRUX_EINVAL (null pointer), LRUX_ESTATE (wrong handle kind),
 * LRUX_ECUDA. */
lrux_status_t lrux_det_refresh(lrux_handle_t h, const void* d_A, void* stream);
lrux_status_t lrux_pf_refresh(lrux_handle_t h, const void* d_A, void* stream);

/* ---------------------------------------------------------------- profiling
 * Device time per kernel class, taken with CUDA events the library records on the
 * caller's stream directly around its own launches (bench.py's roofline figures:
 * algorithmic bytes or flops / these durations).  Off by default; host objects
 * only.  lrux_profile_read is the one call that waits: it synchronises on the
 * events recorded so far for `cls`, returns their summed duration in
 * milliseconds and the number of timed launches, and clears that class. */
typedef enum {
  LRUX_PROF_RATIO = 0,  /* gather + core + det/pf (a1, a2, a5) */
  LRUX_PROF_UPDATE = 1, /* immediate Woodbury update of A^-1 (a3, a4) */
  LRUX_PROF_APPEND = 2, /* delayed append (a6) */
  LRUX_PROF_FLUSH = 3,  /* delay-buffer fold (a7) */
  LRUX_PROF_YPASS = 4,  /* Pfaffian read-only pass Y = A^-1 N */
  LRUX_PROF_NCLASS = 5
} lrux_prof_class_t;
lrux_status_t lrux_profile_enable(lrux_handle_t h, int32_t on);
/* Name of the kernel most recently enqueued through this handle for class `cls`
 * (lrux_prof_class_t), "" when none was.  Kernels are selected by shape alone -- (dtype, n,
 * k, K), never by the environment -- and this is how a test or a report learns which one
 * a shape takes.  The pointer is to a static string. */
const char* lrux_kernel_name(lrux_handle_t h, int32_t cls);
lrux_status_t lrux_profile_read(lrux_handle_t h, int32_t cls, double* ms_total,
                                int64_t* launches);

/* Running totals of the delay-buffer folds since init (or since the state the handle
 * was attached to was initialised): d_out[0] = walker flushes, d_out[1] = buffer columns
 * folded (k per determinant update, 2k per Pfaffian update).  d_out is DEVICE memory,
 * 2 x int64; stream-ordered copy.  bench.py uses it to count the flush flops exactly. */
lrux_status_t lrux_get_flush_count(lrux_handle_t h, int64_t* d_out, void* stream);

/* ---------------------------------------------------------------- allocation-free call */
/* Rank-k determinant ratio for callers that cannot allocate (code under CUDA-graph capture,
 * serving loops, harnesses that forbid cudaMalloc): no handle, no state buffer.
 *     r_w = det(R_w),   R_w = N_w A_w^-1[:,P_w]     (Eq. 3-4 with one-hot v)
 *   d_Ti    [W][n][n]  A_w^-T row-major (row j = column j of A_w^-1), the layout the handles keep
 *   d_idx   [W][k]     int32 replaced rows P_w           d_rows [W][k][n]  the new rows N_w
 *   d_ratio [W]        output
 * All pointers are DEVICE memory owned by the caller; inputs are only read.  1 <= k <=
 * LRUX_MAX_K_GENERAL.  An index outside [0,n) or a duplicate gives ratio NaN for that walker.
 * The k x k cores R_w pass between the two kernels of the call through a fixed scratch array
 * that lives in the library image (LRUX_NOALLOC_SCRATCH_BYTES of device memory on every GPU
 * that loads the library, until the process exits): the call performs NO device or host
 * allocation.  W*k*k*sizeof(elem) > LRUX_NOALLOC_SCRATCH_BYTES -> LRUX_ELIMIT, nothing done.
 * Every call on a device shares that one array: calls whose kernels may overlap on the GPU
 * (different streams, no dependency between them) RACE -- order them.  The array keeps the
 * previous call's contents; every element a call reads it has written first, so nothing needs
 * clearing.  Asynchronous, stream-ordered.  Errors: LRUX_EINVAL, LRUX_ELIMIT, LRUX_ECUDA. */
#define LRUX_NOALLOC_SCRATCH_BYTES (1u << 20)
lrux_status_t lrux_det_ratio_noalloc(int64_t W, int32_t n, int32_t k, lrux_dtype_t dtype,
                                     const void* d_Ti, const int32_t* d_idx, const void* d_rows,
                                     void* d_ratio, void* stream);

/* ---------------------------------------------------------------- common */
/* Number of kernel launches the library has enqueued through this handle so far
 * (host counter; bench.py reports it as gpu_launches). */
lrux_status_t lrux_launch_count(lrux_handle_t h, int64_t* count);
lrux_status_t lrux_destroy(lrux_handle_t h);
const char* lrux_status_string(lrux_status_t s);

#ifdef __cplusplus
}
#endif
#endif /* LRUX_H_ */
