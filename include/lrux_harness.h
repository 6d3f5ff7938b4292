/*
 * lrux_harness.h -- device-side Monte-Carlo harness around lrux.h (the L3 "user
 * workflow" of the paper): proposal and Metropolis decision
 * kernels, so that a whole trajectory runs stream-ordered without host syncs.
 * Not part of the method; part of what bench.py times as one "step"
 * (propose -> lrux_*_ratio -> decide -> lrux_*_accept).
 *
 * Step counter.  Every call takes the step number `step` as a host argument; when `d_step`
 * is not NULL the step is read from DEVICE memory instead (d_step[0]; `step` is ignored), and
 * lruxh_decide advances it by one after use (d_step is int64[2]: [0] the step, [1] scratch
 * that must start at 0).  With the counter on the device, one step -- propose, lrux_*_ratio,
 * decide, lrux_*_accept -- is the same launch sequence every time and can be captured ONCE
 * into a CUDA graph and replayed (mc.Chain.capture), which removes the host launch cost.
 *
 * The random draws use the counter-based generator documented in
 * paper_2602_05255_b200/workload.py (integer arithmetic only, so host and device
 * produce identical draws).  Same pointer/stream conventions as lrux.h.
 */
#ifndef LRUX_HARNESS_H_
#define LRUX_HARNESS_H_

#include <stdint.h>

#include "lrux.h"

#ifdef __cplusplus
extern "C" {
#endif

/* Determinant proposal (BASELINE.json configs[0,1,3]): for walker w (global id
 * w0 + w) and step `step`, draw k distinct slots P and k distinct positions J in
 * the unoccupied list (streams 2, 3), write d_idx[w][a] = P[a],
 * d_upos[w][a] = J[a], and gather the new rows
 * d_rows[w][a][:] = d_Phi[w][ d_unocc[w][J[a]] ][:]   (Phi is [W][M][n]). */
lrux_status_t lruxh_det_propose(uint64_t seed, int64_t w0, int64_t step, int64_t W, int32_t n,
                                int32_t M, int32_t k, lrux_dtype_t dt, const void* d_Phi,
                                const int32_t* d_occ /*[W][n]*/,
                                const int32_t* d_unocc /*[W][M-n]*/, int32_t* d_idx /*[W][k]*/,
                                int32_t* d_upos /*[W][k]*/, void* d_rows /*[W][k][n]*/,
                                const int64_t* d_step /* NULL or int64[2] */, void* stream);

/* Pfaffian proposal (configs[2]): same draws; the new row of slot P[a] is
 * d_rows[w][a][j] = d_F[w][q_a][occ'[j]] with q_a = unocc[J[a]] and occ' the
 * proposed occupation (occ with occ[P[b]] = q_b).  F is [W][M][M] skew. */
lrux_status_t lruxh_pf_propose(uint64_t seed, int64_t w0, int64_t step, int64_t W, int32_t n,
                               int32_t M, int32_t k, lrux_dtype_t dt, const void* d_F,
                               const int32_t* d_occ, const int32_t* d_unocc, int32_t* d_idx,
                               int32_t* d_upos, void* d_rows, const int64_t* d_step, void* stream);

/* Metropolis decision: xi = uniform(stream 4, counter step);
 * d_mask[w] = xi < min(1, |r_w|^2) (strict; NaN rejects).  On accept swaps
 * d_occ[w][P[a]] <-> d_unocc[w][J[a]] and adds 1 to d_naccept[0] (int64). */
lrux_status_t lruxh_decide(uint64_t seed, int64_t w0, int64_t step, int64_t W, int32_t n,
                           int32_t M, int32_t k, lrux_dtype_t dt, const void* d_ratio,
                           const int32_t* d_idx, const int32_t* d_upos, int32_t* d_occ,
                           int32_t* d_unocc, uint8_t* d_mask, int64_t* d_naccept,
                           int64_t* d_step /* NULL or int64[2]; advanced by one */, void* stream);

#ifdef __cplusplus
}
#endif
#endif /* LRUX_HARNESS_H_ */
