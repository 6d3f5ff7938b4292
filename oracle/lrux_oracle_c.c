/*
 * lrux_oracle_c.c -- C restatement of the CPU oracle (TEST INFRASTRUCTURE ONLY).
 *
 * The same functions as oracle/lrux_oracle.py (partial-pivot LU, Parlett-Reid
 * Pfaffian, det_lru / pf_lru, the delayed carriers and the Metropolis trajectories),
 * written from /root/reference/PAPER.md as plain C loops in float64 / complex128:
 * host only, no BLAS/LAPACK, no CUDA, shares no code with the CUDA path and is not
 * linked into liblrux.so.  It exists because the numpy oracle's interpreter loops make
 * full-length trajectories (1000 steps at n = 256, 500 at n = 1024 complex) and an
 * all-cores CPU baseline unaffordable.  Only tests/,
 * __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may load
 * it (through oracle/c_oracle.py).
 *
 * Pins: tests/test_oracle_pins.py and tests/test_oracle_trajectory.py run every pin
 * (brute force n <= 8, the paper's closed forms Eq. A.2-A.3 and pf J, identities
 * A.4-A.9, numpy.linalg as a library special case, lemma vs from scratch,
 * A_t A_t^-1 = 1, telescoping product of ratios, delayed == immediate) against this
 * implementation as well as against the numpy one, and the two are compared with each
 * other.  No function is "parity unpinned".
 *
 * Build: gcc -O2 -fopenmp -shared -fPIC (oracle/build_oracle.py).
 */
#define _POSIX_C_SOURCE 199309L
#include <complex.h>
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

/* kind 0 = determinant, 1 = Pfaffian; see orc_trajectory_* in the body */
typedef struct {
  int32_t kind, n, M, k, steps, scratch_every, delay, final_scratch;
  int32_t mark_step;   /* timing only: steps >= mark_step are clocked (bench.py's cpu_baseline) */
} orc_cfg;

#include <time.h>
static double orc_now(void) {
  struct timespec ts;
  clock_gettime(CLOCK_MONOTONIC, &ts);
  return (double)ts.tv_sec + 1e-9 * (double)ts.tv_nsec;
}

#define T double
#define FN(name) name##_d
#define ABS(x) fabs(x)
#define REAL(x) (x)
#define IMAG(x) (0.0)
#include "lrux_oracle_body.h"
#undef T
#undef FN
#undef ABS
#undef REAL
#undef IMAG

#define T double _Complex
#define FN(name) name##_z
#define ABS(x) cabs(x)
#define REAL(x) creal(x)
#define IMAG(x) cimag(x)
#include "lrux_oracle_body.h"
#undef T
#undef FN
#undef ABS
#undef REAL
#undef IMAG

int orc_num_threads(void) {
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}
