/*
 * lrux_oracle_body.h -- type-generic body of the C oracle (TEST INFRASTRUCTURE ONLY).
 *
 * Included twice by lrux_oracle_c.c: with T = double (suffix _d) and with
 * T = double _Complex (suffix _z).  Plain loops, no BLAS/LAPACK, no blocking, no
 * reordering beyond what the cited definition states; every function names the
 * passage of /root/reference/PAPER.md it follows.  Shares nothing with the CUDA
 * path (paper_2602_05255_b200/csrc).  All "^T" are plain transposes, never
 * conjugate transposes, also for complex data.
 *
 * Matrices are row-major.  X(i,j,ld) = X[i*ld + j].
 */

/* ---------------------------------------------------------------- 1. partial-pivot LU
 * Pivot = largest modulus in the column at or below the diagonal, lowest index on
 * ties.  LU is overwritten with L (unit lower) and U,
 * perm[i] = source row of row i, *parity = +-1.  Returns 0 when a zero pivot was
 * met (singular A), else 1. */
static int FN(lu_factor)(int n, T* LU, int* perm, double* parity) {
  int ok = 1;
  *parity = 1.0;
  for (int i = 0; i < n; ++i) perm[i] = i;
  for (int c = 0; c < n; ++c) {
    int p = c;
    double best = ABS(LU[(size_t)c * n + c]);
    for (int r = c + 1; r < n; ++r) {
      double v = ABS(LU[(size_t)r * n + c]);
      if (v > best) { best = v; p = r; }
    }
    if (LU[(size_t)p * n + c] == 0) { ok = 0; continue; }
    if (p != c) {
      for (int j = 0; j < n; ++j) {
        T t = LU[(size_t)c * n + j];
        LU[(size_t)c * n + j] = LU[(size_t)p * n + j];
        LU[(size_t)p * n + j] = t;
      }
      int tp = perm[c]; perm[c] = perm[p]; perm[p] = tp;
      *parity = -*parity;
    }
    const T piv = LU[(size_t)c * n + c];
    for (int r = c + 1; r < n; ++r) {
      const T l = LU[(size_t)r * n + c] / piv;
      LU[(size_t)r * n + c] = l;
      for (int j = c + 1; j < n; ++j) LU[(size_t)r * n + j] -= l * LU[(size_t)c * n + j];
    }
  }
  return ok;
}

/* (phase, log|det A|): phase = parity * prod U_ii/|U_ii|, logabs = sum log|U_ii|.
 * Singular A gives (0, -inf) and returns 0. */
int FN(orc_slogdet)(int n, const T* A, T* phase, double* logabs) {
  if (n == 0) { *phase = 1; *logabs = 0.0; return 1; }
  T* LU = (T*)malloc((size_t)n * n * sizeof(T));
  int* perm = (int*)malloc((size_t)n * sizeof(int));
  memcpy(LU, A, (size_t)n * n * sizeof(T));
  double parity;
  int ok = FN(lu_factor)(n, LU, perm, &parity);
  for (int i = 0; i < n && ok; ++i)
    if (LU[(size_t)i * n + i] == 0) ok = 0;
  if (!ok) {
    *phase = 0; *logabs = -INFINITY;
  } else {
    T ph = parity;
    double la = 0.0;
    for (int i = 0; i < n; ++i) {
      const T d = LU[(size_t)i * n + i];
      const double a = ABS(d);
      ph *= d / a;
      la += log(a);
    }
    *phase = ph; *logabs = la;
  }
  free(LU); free(perm);
  return ok;
}

/* A^-1 by LU and n pairs of triangular solves (forward L Y = P I, backward U X = Y).
 * Returns 0 for a singular matrix (out undefined). */
int FN(orc_inv)(int n, const T* A, T* out) {
  T* LU = (T*)malloc((size_t)n * n * sizeof(T));
  T* Y = (T*)malloc((size_t)n * n * sizeof(T));
  int* perm = (int*)malloc((size_t)n * sizeof(int));
  memcpy(LU, A, (size_t)n * n * sizeof(T));
  double parity;
  int ok = FN(lu_factor)(n, LU, perm, &parity);
  for (int i = 0; i < n && ok; ++i)
    if (LU[(size_t)i * n + i] == 0) ok = 0;
  if (ok) {
    for (int i = 0; i < n; ++i) {             /* L Y = P I, row i of Y */
      for (int j = 0; j < n; ++j) Y[(size_t)i * n + j] = (perm[i] == j) ? 1 : 0;
      for (int m = 0; m < i; ++m) {
        const T l = LU[(size_t)i * n + m];
        for (int j = 0; j < n; ++j) Y[(size_t)i * n + j] -= l * Y[(size_t)m * n + j];
      }
    }
    for (int i = n - 1; i >= 0; --i) {        /* U X = Y, row i of X */
      for (int j = 0; j < n; ++j) out[(size_t)i * n + j] = Y[(size_t)i * n + j];
      for (int m = i + 1; m < n; ++m) {
        const T uim = LU[(size_t)i * n + m];
        for (int j = 0; j < n; ++j) out[(size_t)i * n + j] -= uim * out[(size_t)m * n + j];
      }
      const T d = LU[(size_t)i * n + i];
      for (int j = 0; j < n; ++j) out[(size_t)i * n + j] /= d;
    }
  }
  free(LU); free(Y); free(perm);
  return ok;
}

/* ---------------------------------------------------------------- 2. Pfaffian (Parlett-Reid)
 * (phase, log|pf A|) of a skew-symmetric matrix, cf. lrux.slogpf (the
 * paper leaves the algorithm open, reading 10).  For j = 0,2,4,...: pivot p in
 * [j+1,n) maximising |A[p][j]| (lowest index on ties); a simultaneous row+column
 * swap j+1 <-> p flips the sign (Eq. A.5 with B a transposition); pf
 * picks up the factor A[j][j+1] and the trailing block receives the Schur complement
 * of Eq. A.9: A[j+2:,j+2:] += tau (x) c - c (x) tau,
 * tau = A[j][j+2:]/a, c = A[j+2:][j+1]. */
int FN(orc_slogpf)(int n, const T* Ain, T* phase, double* logabs) {
  if (n == 0) { *phase = 1; *logabs = 0.0; return 1; }
  if (n % 2 == 1) { *phase = 0; *logabs = -INFINITY; return 0; }
  T* A = (T*)malloc((size_t)n * n * sizeof(T));
  T* tau = (T*)malloc((size_t)n * sizeof(T));
  T* cc = (T*)malloc((size_t)n * sizeof(T));
  memcpy(A, Ain, (size_t)n * n * sizeof(T));
  T ph = 1;
  double la = 0.0;
  int ok = 1;
  for (int j = 0; j < n - 1 && ok; j += 2) {
    int p = j + 1;
    double best = ABS(A[(size_t)(j + 1) * n + j]);
    for (int r = j + 2; r < n; ++r) {
      double v = ABS(A[(size_t)r * n + j]);
      if (v > best) { best = v; p = r; }
    }
    if (p != j + 1) {
      for (int c = 0; c < n; ++c) {
        T t = A[(size_t)(j + 1) * n + c];
        A[(size_t)(j + 1) * n + c] = A[(size_t)p * n + c];
        A[(size_t)p * n + c] = t;
      }
      for (int r = 0; r < n; ++r) {
        T t = A[(size_t)r * n + j + 1];
        A[(size_t)r * n + j + 1] = A[(size_t)r * n + p];
        A[(size_t)r * n + p] = t;
      }
      ph = -ph;
    }
    const T a = A[(size_t)j * n + j + 1];
    if (a == 0) { ok = 0; break; }
    const double aa = ABS(a);
    ph *= a / aa;
    la += log(aa);
    if (j + 2 < n) {
      for (int i = j + 2; i < n; ++i) {
        tau[i] = A[(size_t)j * n + i] / a;
        cc[i] = A[(size_t)i * n + j + 1];
      }
      for (int r = j + 2; r < n; ++r)
        for (int c = j + 2; c < n; ++c)
          A[(size_t)r * n + c] = A[(size_t)r * n + c] + tau[r] * cc[c] - cc[r] * tau[c];
    }
  }
  if (!ok) { *phase = 0; *logabs = -INFINITY; }
  else { *phase = ph; *logabs = la; }
  free(A); free(tau); free(cc);
  return ok;
}

/* small helpers: det / pf as a plain value */
static T FN(det_value)(int n, const T* A) {
  T ph; double la;
  FN(orc_slogdet)(n, A, &ph, &la);
  return ph * exp(la);
}
static T FN(pf_value)(int n, const T* A) {
  T ph; double la;
  FN(orc_slogpf)(n, A, &ph, &la);
  return ph * exp(la);
}
/* pf J = (-1)^(k(k-1)/2) */
static double FN(pf_skew_eye)(int k) { return ((k * (k - 1) / 2) % 2) ? -1.0 : 1.0; }

/* ---------------------------------------------------------------- 4. low-rank updates
 * lrux.det_lru.  A_t = A_{t-1} + v u^T, u and v are n x k.
 * R = 1 + u^T A^-1 v (Eq. 4), r = det R (Eq. 3); when `newinv` is not
 * NULL also A_t^-1 = A^-1 - A^-1 v R^-1 u^T A^-1 (Eq. 5). */
int FN(orc_det_lru)(int n, int k, const T* Ainv, const T* u, const T* v, T* r, T* newinv) {
  T* uA = (T*)calloc((size_t)k * n, sizeof(T));   /* u^T A^-1   (k x n) */
  T* R = (T*)malloc((size_t)k * k * sizeof(T));
  for (int a = 0; a < k; ++a)
    for (int i = 0; i < n; ++i) {
      const T ui = u[(size_t)i * k + a];
      for (int j = 0; j < n; ++j) uA[(size_t)a * n + j] += ui * Ainv[(size_t)i * n + j];
    }
  for (int a = 0; a < k; ++a)
    for (int b = 0; b < k; ++b) {
      T s = (a == b) ? 1 : 0;
      for (int j = 0; j < n; ++j) s += uA[(size_t)a * n + j] * v[(size_t)j * k + b];
      R[a * k + b] = s;
    }
  *r = FN(det_value)(k, R);
  int ok = 1;
  if (newinv) {
    T* Av = (T*)calloc((size_t)n * k, sizeof(T));   /* A^-1 v   (n x k) */
    T* Ri = (T*)malloc((size_t)k * k * sizeof(T));
    T* AvRi = (T*)malloc((size_t)n * k * sizeof(T));
    ok = FN(orc_inv)(k, R, Ri);
    for (int i = 0; i < n; ++i)
      for (int j = 0; j < n; ++j) {
        const T aij = Ainv[(size_t)i * n + j];
        for (int b = 0; b < k; ++b) Av[(size_t)i * k + b] += aij * v[(size_t)j * k + b];
      }
    for (int i = 0; i < n; ++i)
      for (int b = 0; b < k; ++b) {
        T s = 0;
        for (int a = 0; a < k; ++a) s += Av[(size_t)i * k + a] * Ri[a * k + b];
        AvRi[(size_t)i * k + b] = s;
      }
    for (int i = 0; i < n; ++i)
      for (int j = 0; j < n; ++j) {
        T s = 0;
        for (int b = 0; b < k; ++b) s += AvRi[(size_t)i * k + b] * uA[(size_t)b * n + j];
        newinv[(size_t)i * n + j] = Ainv[(size_t)i * n + j] - s;
      }
    free(Av); free(Ri); free(AvRi);
  }
  free(uA); free(R);
  return ok;
}

/* G (m x m) -> strict upper triangle of G minus its transpose: exactly skew (reading 8) */
static void FN(skew_from_upper)(int m, T* G) {
  for (int a = 0; a < m; ++a) {
    G[a * m + a] = 0;
    for (int b = a + 1; b < m; ++b) G[b * m + a] = -G[a * m + b];
  }
}

/* R^-1 of an exactly skew R, skew-projected: (X - X^T)/2 */
static int FN(skew_inv)(int m, const T* R, T* Ri) {
  T* X = (T*)malloc((size_t)m * m * sizeof(T));
  int ok = FN(orc_inv)(m, R, X);
  for (int a = 0; a < m; ++a)
    for (int b = 0; b < m; ++b) Ri[a * m + b] = (X[a * m + b] - X[b * m + a]) / 2;
  free(X);
  return ok;
}

/* lrux.pf_lru.  A_t = A_{t-1} - u J u^T (Eq. 16), u is n x 2k,
 * J = [[0,1],[-1,0]] (Eq. 17).  R = J + u^T A^-1 u (Eq. 20; Eq. 18 prints A without
 * the inverse: reading 1), r = pf R / pf J (Eq. 19).  R is built from its strict upper
 * triangle and mirrored (reading 8).  When `newinv` is not NULL also
 * A_t^-1 = A^-1 + (A^-1 u) R^-1 (A^-1 u)^T (Eq. 21) with an exactly skew
 * R^-1 and an exactly skew result. */
int FN(orc_pf_lru)(int n, int k, const T* Ainv, const T* u, T* r, T* newinv) {
  const int m = 2 * k;
  T* a = (T*)calloc((size_t)n * m, sizeof(T));    /* A^-1 u   (n x 2k) */
  T* R = (T*)malloc((size_t)m * m * sizeof(T));
  for (int i = 0; i < n; ++i)
    for (int j = 0; j < n; ++j) {
      const T aij = Ainv[(size_t)i * n + j];
      for (int b = 0; b < m; ++b) a[(size_t)i * m + b] += aij * u[(size_t)j * m + b];
    }
  for (int p = 0; p < m; ++p)
    for (int q = 0; q < m; ++q) {
      T s = 0;
      for (int i = 0; i < n; ++i) s += u[(size_t)i * m + p] * a[(size_t)i * m + q];
      R[p * m + q] = s;
    }
  FN(skew_from_upper)(m, R);
  for (int p = 0; p < k; ++p) { R[p * m + k + p] += 1; R[(k + p) * m + p] -= 1; }   /* + J */
  *r = FN(pf_value)(m, R) / FN(pf_skew_eye)(k);
  int ok = 1;
  if (newinv) {
    T* Ri = (T*)malloc((size_t)m * m * sizeof(T));
    T* aRi = (T*)malloc((size_t)n * m * sizeof(T));
    ok = FN(skew_inv)(m, R, Ri);
    for (int i = 0; i < n; ++i)
      for (int q = 0; q < m; ++q) {
        T s = 0;
        for (int p = 0; p < m; ++p) s += a[(size_t)i * m + p] * Ri[p * m + q];
        aRi[(size_t)i * m + q] = s;
      }
    for (int i = 0; i < n; ++i) {
      newinv[(size_t)i * n + i] = Ainv[(size_t)i * n + i];
      for (int j = i + 1; j < n; ++j) {
        T s = 0;
        for (int q = 0; q < m; ++q) s += aRi[(size_t)i * m + q] * a[(size_t)j * m + q];
        newinv[(size_t)i * n + j] = Ainv[(size_t)i * n + j] + s;
        newinv[(size_t)j * n + i] = Ainv[(size_t)j * n + i] - s;
      }
    }
    free(Ri); free(aRi);
  }
  free(a); free(R);
  return ok;
}

/* u = (x, e) for replacing the rows AND columns P of a skew matrix (Eq. 23-24,
 * PAPER.md:317-345).  old_rows[a] / new_rows[a] are row P[a] of A_{t-1} / A_t.
 * x[:,a] is the row delta; where replaced rows and columns cross, the delta is halved
 * (reading 5: -u J u^T = e x^T - x e^T counts that block twice); the diagonal entry
 * multiplies A^-1[p][p] = 0 (reading 6).  u is n x 2k. */
void FN(orc_pf_update_vectors)(int n, int k, const T* old_rows, const T* new_rows, const int32_t* P,
                               T* u) {
  const int m = 2 * k;
  for (int i = 0; i < n; ++i)
    for (int a = 0; a < k; ++a) {
      u[(size_t)i * m + a] = new_rows[(size_t)a * n + i] - old_rows[(size_t)a * n + i];
      u[(size_t)i * m + k + a] = (i == P[a]) ? 1 : 0;
    }
  for (int a = 0; a < k; ++a)
    for (int b = 0; b < k; ++b) u[(size_t)P[b] * m + a] = u[(size_t)P[b] * m + a] / 2;
}

/* ---------------------------------------------------------------- 5. delayed updates
 * Determinant carrier (lrux.init_det_carrier / det_lru_delayed):
 * A_0^-1 plus the delayed factors a_t (Eq. 10) and b_t (Eq. 11), each n x k.
 * Pfaffian carrier: A_0^-1, a_t (Eq. 25, n x 2k), R_t^-1. */
typedef struct {
  int n, max_delay, count;
  int* kk;        /* columns of update t (k for det, 2k for pf) */
  T* A0inv;
  T** a;
  T** b;          /* det: b_t (n x k);  pf: R_t^-1 (2k x 2k) */
} FN(carrier);

static void FN(carrier_init)(FN(carrier)* c, int n, int max_delay, const T* Ainv) {
  c->n = n; c->max_delay = max_delay; c->count = 0;
  c->kk = (int*)calloc((size_t)max_delay + 1, sizeof(int));
  c->a = (T**)calloc((size_t)max_delay + 1, sizeof(T*));
  c->b = (T**)calloc((size_t)max_delay + 1, sizeof(T*));
  c->A0inv = (T*)malloc((size_t)n * n * sizeof(T));
  memcpy(c->A0inv, Ainv, (size_t)n * n * sizeof(T));
}
static void FN(carrier_clear)(FN(carrier)* c) {
  for (int t = 0; t < c->count; ++t) { free(c->a[t]); free(c->b[t]); }
  c->count = 0;
}
static void FN(carrier_free)(FN(carrier)* c) {
  FN(carrier_clear)(c);
  free(c->kk); free(c->a); free(c->b); free(c->A0inv);
}

/* Eq. 12: A_tau^-1 = A_0^-1 - sum_t a_t b_t^T, written into out */
static void FN(det_carrier_inverse)(const FN(carrier)* c, T* out) {
  const int n = c->n;
  memcpy(out, c->A0inv, (size_t)n * n * sizeof(T));
  for (int t = 0; t < c->count; ++t) {
    const int k = c->kk[t];
    for (int i = 0; i < n; ++i)
      for (int j = 0; j < n; ++j) {
        T s = 0;
        for (int q = 0; q < k; ++q) s += c->a[t][(size_t)i * k + q] * c->b[t][(size_t)j * k + q];
        out[(size_t)i * n + j] -= s;
      }
  }
}
static void FN(det_carrier_flush)(FN(carrier)* c) {
  T* out = (T*)malloc((size_t)c->n * c->n * sizeof(T));
  FN(det_carrier_inverse)(c, out);
  memcpy(c->A0inv, out, (size_t)c->n * c->n * sizeof(T));
  free(out);
  FN(carrier_clear)(c);
}

/* det_lru_delayed: R_tau by Eq. 13; with `update` also a_tau (Eq. 14)
 * and b_tau (Eq. 15), appended; flush (Eq. 12) when tau = T. */
static int FN(det_carrier_lru)(FN(carrier)* c, int k, const T* u, const T* v, T* r, int update) {
  const int n = c->n;
  T* R = (T*)malloc((size_t)k * k * sizeof(T));
  T* uA = (T*)calloc((size_t)k * n, sizeof(T));
  for (int a = 0; a < k; ++a)
    for (int i = 0; i < n; ++i) {
      const T ui = u[(size_t)i * k + a];
      for (int j = 0; j < n; ++j) uA[(size_t)a * n + j] += ui * c->A0inv[(size_t)i * n + j];
    }
  for (int a = 0; a < k; ++a)
    for (int b = 0; b < k; ++b) {
      T s = (a == b) ? 1 : 0;
      for (int j = 0; j < n; ++j) s += uA[(size_t)a * n + j] * v[(size_t)j * k + b];
      R[a * k + b] = s;
    }
  for (int t = 0; t < c->count; ++t) {            /* - (u^T a_t)(b_t^T v) */
    const int kt = c->kk[t];
    T* ua = (T*)calloc((size_t)k * kt, sizeof(T));
    T* bv = (T*)calloc((size_t)kt * k, sizeof(T));
    for (int a = 0; a < k; ++a)
      for (int q = 0; q < kt; ++q)
        for (int i = 0; i < n; ++i) ua[a * kt + q] += u[(size_t)i * k + a] * c->a[t][(size_t)i * kt + q];
    for (int q = 0; q < kt; ++q)
      for (int b = 0; b < k; ++b)
        for (int i = 0; i < n; ++i) bv[q * k + b] += c->b[t][(size_t)i * kt + q] * v[(size_t)i * k + b];
    for (int a = 0; a < k; ++a)
      for (int b = 0; b < k; ++b) {
        T s = 0;
        for (int q = 0; q < kt; ++q) s += ua[a * kt + q] * bv[q * k + b];
        R[a * k + b] -= s;
      }
    free(ua); free(bv);
  }
  *r = FN(det_value)(k, R);
  int ok = 1;
  if (update) {
    T* an = (T*)calloc((size_t)n * k, sizeof(T));   /* a_tau = A_0^-1 v - sum a_t (b_t^T v)   Eq. 14 */
    T* bn = (T*)calloc((size_t)n * k, sizeof(T));   /* b_tau = [(A_0^-1)^T u - sum b_t (a_t^T u)] R^-T   Eq. 15 */
    for (int i = 0; i < n; ++i)
      for (int j = 0; j < n; ++j) {
        const T aij = c->A0inv[(size_t)i * n + j];
        for (int b = 0; b < k; ++b) an[(size_t)i * k + b] += aij * v[(size_t)j * k + b];
      }
    for (int j = 0; j < n; ++j)
      for (int a = 0; a < k; ++a) bn[(size_t)j * k + a] = uA[(size_t)a * n + j];
    for (int t = 0; t < c->count; ++t) {
      const int kt = c->kk[t];
      T* bv = (T*)calloc((size_t)kt * k, sizeof(T));
      T* au = (T*)calloc((size_t)kt * k, sizeof(T));
      for (int q = 0; q < kt; ++q)
        for (int b = 0; b < k; ++b)
          for (int i = 0; i < n; ++i) {
            bv[q * k + b] += c->b[t][(size_t)i * kt + q] * v[(size_t)i * k + b];
            au[q * k + b] += c->a[t][(size_t)i * kt + q] * u[(size_t)i * k + b];
          }
      for (int i = 0; i < n; ++i)
        for (int b = 0; b < k; ++b) {
          T s1 = 0, s2 = 0;
          for (int q = 0; q < kt; ++q) {
            s1 += c->a[t][(size_t)i * kt + q] * bv[q * k + b];
            s2 += c->b[t][(size_t)i * kt + q] * au[q * k + b];
          }
          an[(size_t)i * k + b] -= s1;
          bn[(size_t)i * k + b] -= s2;
        }
      free(bv); free(au);
    }
    T* Ri = (T*)malloc((size_t)k * k * sizeof(T));
    ok = FN(orc_inv)(k, R, Ri);
    T* bfin = (T*)malloc((size_t)n * k * sizeof(T));
    for (int i = 0; i < n; ++i)
      for (int a = 0; a < k; ++a) {               /* b R^-T: sum_q b[i][q] Ri[a][q] */
        T s = 0;
        for (int q = 0; q < k; ++q) s += bn[(size_t)i * k + q] * Ri[a * k + q];
        bfin[(size_t)i * k + a] = s;
      }
    free(bn); free(Ri);
    c->a[c->count] = an; c->b[c->count] = bfin; c->kk[c->count] = k;
    c->count++;
    if (c->count == c->max_delay) FN(det_carrier_flush)(c);      /* tau = T */
  }
  free(R); free(uA);
  return ok;
}

/* Eq. 26: A_tau^-1 = A_0^-1 + sum_t a_t R_t^-1 a_t^T (exactly skew) */
static void FN(pf_carrier_inverse)(const FN(carrier)* c, T* out) {
  const int n = c->n;
  memcpy(out, c->A0inv, (size_t)n * n * sizeof(T));
  for (int t = 0; t < c->count; ++t) {
    const int m = c->kk[t];
    T* aRi = (T*)malloc((size_t)n * m * sizeof(T));
    for (int i = 0; i < n; ++i)
      for (int q = 0; q < m; ++q) {
        T s = 0;
        for (int p = 0; p < m; ++p) s += c->a[t][(size_t)i * m + p] * c->b[t][p * m + q];
        aRi[(size_t)i * m + q] = s;
      }
    for (int i = 0; i < n; ++i)
      for (int j = i + 1; j < n; ++j) {
        T s = 0;
        for (int q = 0; q < m; ++q) s += aRi[(size_t)i * m + q] * c->a[t][(size_t)j * m + q];
        out[(size_t)i * n + j] += s;
        out[(size_t)j * n + i] -= s;
      }
    free(aRi);
  }
}
static void FN(pf_carrier_flush)(FN(carrier)* c) {
  T* out = (T*)malloc((size_t)c->n * c->n * sizeof(T));
  FN(pf_carrier_inverse)(c, out);
  memcpy(c->A0inv, out, (size_t)c->n * c->n * sizeof(T));
  free(out);
  FN(carrier_clear)(c);
}

/* pf_lru_delayed: R_tau by Eq. 27; with `update` also a_tau by Eq. 28
 * (with u_tau: reading 2) and R_tau^-1, appended; flush (Eq. 26) when tau = T. */
static int FN(pf_carrier_lru)(FN(carrier)* c, int k, const T* u, T* r, int update) {
  const int n = c->n, m = 2 * k;
  T* a = (T*)calloc((size_t)n * m, sizeof(T));     /* A_0^-1 u */
  T* G = (T*)malloc((size_t)m * m * sizeof(T));
  for (int i = 0; i < n; ++i)
    for (int j = 0; j < n; ++j) {
      const T aij = c->A0inv[(size_t)i * n + j];
      for (int b = 0; b < m; ++b) a[(size_t)i * m + b] += aij * u[(size_t)j * m + b];
    }
  for (int p = 0; p < m; ++p)
    for (int q = 0; q < m; ++q) {
      T s = 0;
      for (int i = 0; i < n; ++i) s += u[(size_t)i * m + p] * a[(size_t)i * m + q];
      G[p * m + q] = s;
    }
  for (int t = 0; t < c->count; ++t) {             /* + (u^T a_t) R_t^-1 (u^T a_t)^T */
    const int mt = c->kk[t];
    T* ua = (T*)calloc((size_t)m * mt, sizeof(T));
    T* uaRi = (T*)malloc((size_t)m * mt * sizeof(T));
    for (int p = 0; p < m; ++p)
      for (int q = 0; q < mt; ++q)
        for (int i = 0; i < n; ++i) ua[p * mt + q] += u[(size_t)i * m + p] * c->a[t][(size_t)i * mt + q];
    for (int p = 0; p < m; ++p)
      for (int q = 0; q < mt; ++q) {
        T s = 0;
        for (int x = 0; x < mt; ++x) s += ua[p * mt + x] * c->b[t][x * mt + q];
        uaRi[p * mt + q] = s;
      }
    for (int p = 0; p < m; ++p)
      for (int q = 0; q < m; ++q) {
        T s = 0;
        for (int x = 0; x < mt; ++x) s += uaRi[p * mt + x] * ua[q * mt + x];
        G[p * m + q] += s;
      }
    if (update) {                                  /* a += a_t R_t^-1 (u^T a_t)^T   Eq. 28 */
      for (int i = 0; i < n; ++i)
        for (int q = 0; q < m; ++q) {
          T s = 0;
          for (int x = 0; x < mt; ++x) {
            T ar = 0;
            for (int y = 0; y < mt; ++y) ar += c->a[t][(size_t)i * mt + y] * c->b[t][y * mt + x];
            s += ar * ua[q * mt + x];
          }
          a[(size_t)i * m + q] += s;
        }
    }
    free(ua); free(uaRi);
  }
  FN(skew_from_upper)(m, G);
  for (int p = 0; p < k; ++p) { G[p * m + k + p] += 1; G[(k + p) * m + p] -= 1; }
  *r = FN(pf_value)(m, G) / FN(pf_skew_eye)(k);
  int ok = 1;
  if (update) {
    T* Ri = (T*)malloc((size_t)m * m * sizeof(T));
    ok = FN(skew_inv)(m, G, Ri);
    c->a[c->count] = a; c->b[c->count] = Ri; c->kk[c->count] = m;
    c->count++;
    a = NULL;
    if (c->count == c->max_delay) FN(pf_carrier_flush)(c);
  }
  free(a); free(G);
  return ok;
}

/* ---------------------------------------------------------------- 6. Metropolis trajectories
 * One walker's chain (BASELINE.json configs; SURVEY.md §8(c) part 4).  kind 0:
 * determinant, A = Phi[occ,:] (Phi is M x n), step t puts orbital unocc[J[t][a]] into slot
 * P[t][a]: u = (new rows - old rows)^T, v = one-hot(P) (Eq. 8).  kind 1:
 * Pfaffian, A = F[occ][:,occ] (F is M x M skew), u from orc_pf_update_vectors.
 * r_lemma by the lemma against the tracked inverse (or the carrier when delay > 0),
 * r_scratch = amplitude(A')/amplitude(A) recomputed from scratch every `scratch_every`
 * steps and at the last step (NaN elsewhere; scratch_every = 0: never), accept iff
 * xi < min(1,|r_lemma|^2) strictly, NaN rejects (reading 12); accepted updates apply
 * Eq. 5 / Eq. 21 naively or go through the carrier.  The amplitude is tracked as
 * (phase, log|.|).  final_scratch: recompute the amplitude of the final A from scratch
 * (needed by the parity tests; left out by the timing runs). */
static void FN(gather_A)(int kind, int n, int M, const T* orb, const int32_t* occ, T* A) {
  for (int i = 0; i < n; ++i)
    for (int j = 0; j < n; ++j)
      A[(size_t)i * n + j] = kind == 0 ? orb[(size_t)occ[i] * n + j] : orb[(size_t)occ[i] * M + occ[j]];
}

int FN(orc_trajectory)(const orc_cfg* cfg, const T* orb, const int32_t* occ_in, const int32_t* unocc_in,
                       const int32_t* P, const int32_t* J, const double* xi,
                       T* r_lemma, T* r_scratch, uint8_t* accepted, uint8_t* near_tie, double* prob,
                       T* A_out, T* Ainv_out, int32_t* occ_out, int32_t* unocc_out,
                       T* amp /* [3]: tracked phase, scratch phase, initial phase */,
                       double* logs /* [3]: tracked, scratch, initial log|.| */,
                       double* dur /* seconds spent in steps >= cfg->mark_step, or NULL */) {
  const int kind = cfg->kind, n = cfg->n, M = cfg->M, k = cfg->k, steps = cfg->steps;
  const int m = kind == 0 ? k : 2 * k;
  int32_t* occ = (int32_t*)malloc((size_t)n * sizeof(int32_t));
  int32_t* unocc = (int32_t*)malloc((size_t)(M - n) * sizeof(int32_t));
  int32_t* occ_new = (int32_t*)malloc((size_t)n * sizeof(int32_t));
  memcpy(occ, occ_in, (size_t)n * sizeof(int32_t));
  memcpy(unocc, unocc_in, (size_t)(M - n) * sizeof(int32_t));
  T* A = (T*)malloc((size_t)n * n * sizeof(T));
  T* A_new = (T*)malloc((size_t)n * n * sizeof(T));
  T* Ainv = (T*)malloc((size_t)n * n * sizeof(T));
  T* Anext = (T*)malloc((size_t)n * n * sizeof(T));
  T* u = (T*)malloc((size_t)n * m * sizeof(T));
  T* v = (T*)malloc((size_t)n * k * sizeof(T));
  T* oldr = (T*)malloc((size_t)k * n * sizeof(T));
  T* newr = (T*)malloc((size_t)k * n * sizeof(T));
  FN(gather_A)(kind, n, M, orb, occ, A);
  T ph0; double la0;
  if (kind == 0) FN(orc_slogdet)(n, A, &ph0, &la0); else FN(orc_slogpf)(n, A, &ph0, &la0);
  T phase = ph0, s_ph = ph0;
  double logabs = la0, s_la = la0;
  int ok = FN(orc_inv)(n, A, Ainv);
  if (kind == 1)
    for (int i = 0; i < n; ++i) {
      Ainv[(size_t)i * n + i] = 0;                 /* (X - X^T)/2 on the diagonal */
      for (int j = i + 1; j < n; ++j) {
        const T s = (Ainv[(size_t)i * n + j] - Ainv[(size_t)j * n + i]) / 2;
        Ainv[(size_t)i * n + j] = s;
        Ainv[(size_t)j * n + i] = -s;
      }
    }
  FN(carrier) car;
  const int delayed = cfg->delay > 0;
  if (delayed) FN(carrier_init)(&car, n, cfg->delay, Ainv);
  const int se = cfg->scratch_every;
  double t_mark = 0.0;
  for (int t = 0; t < steps; ++t) {
    if (dur && t == cfg->mark_step) t_mark = orc_now();
    const int32_t* p = P + (size_t)t * k;
    const int32_t* jj = J + (size_t)t * k;
    /* proposed matrix A' and the update vectors */
    memcpy(A_new, A, (size_t)n * n * sizeof(T));
    if (kind == 0) {
      for (int a = 0; a < k; ++a) {
        const int q = unocc[jj[a]];
        for (int i = 0; i < n; ++i) A_new[(size_t)p[a] * n + i] = orb[(size_t)q * n + i];
      }
      for (int i = 0; i < n; ++i)
        for (int a = 0; a < k; ++a) {
          u[(size_t)i * k + a] = A_new[(size_t)p[a] * n + i] - A[(size_t)p[a] * n + i];
          v[(size_t)i * k + a] = (i == p[a]) ? 1 : 0;
        }
    } else {
      memcpy(occ_new, occ, (size_t)n * sizeof(int32_t));
      for (int a = 0; a < k; ++a) occ_new[p[a]] = unocc[jj[a]];
      FN(gather_A)(1, n, M, orb, occ_new, A_new);
      for (int a = 0; a < k; ++a)
        for (int i = 0; i < n; ++i) {
          oldr[(size_t)a * n + i] = A[(size_t)p[a] * n + i];
          newr[(size_t)a * n + i] = A_new[(size_t)p[a] * n + i];
        }
      FN(orc_pf_update_vectors)(n, k, oldr, newr, p, u);
    }
    T r;
    if (delayed) {
      if (kind == 0) FN(det_carrier_lru)(&car, k, u, v, &r, 0);
      else FN(pf_carrier_lru)(&car, k, u, &r, 0);
    } else {
      if (kind == 0) FN(orc_det_lru)(n, k, Ainv, u, v, &r, NULL);
      else FN(orc_pf_lru)(n, k, Ainv, u, &r, NULL);
    }
    r_lemma[t] = r;
    r_scratch[t] = NAN;
    T n_ph = 0; double n_la = 0.0;
    int have_new = 0;
    if (se && (t % se == 0 || t == steps - 1)) {
      if (kind == 0) FN(orc_slogdet)(n, A_new, &n_ph, &n_la); else FN(orc_slogpf)(n, A_new, &n_ph, &n_la);
      r_scratch[t] = (n_ph / s_ph) * exp(n_la - s_la);
      have_new = 1;
    }
    const double a2 = REAL(r) * REAL(r) + IMAG(r) * IMAG(r);
    int acc = 0;
    double pr = NAN;
    if (!isnan(a2)) { pr = a2 < 1.0 ? a2 : 1.0; acc = xi[t] < pr; }
    accepted[t] = (uint8_t)acc;
    prob[t] = pr;
    near_tie[t] = (uint8_t)(fabs(xi[t] - pr) < 1e-8);
    if (acc) {
      if (delayed) {
        T r2;
        if (kind == 0) FN(det_carrier_lru)(&car, k, u, v, &r2, 1);
        else FN(pf_carrier_lru)(&car, k, u, &r2, 1);
      } else {
        T r2;
        if (kind == 0) FN(orc_det_lru)(n, k, Ainv, u, v, &r2, Anext);
        else FN(orc_pf_lru)(n, k, Ainv, u, &r2, Anext);
        T* tmp = Ainv; Ainv = Anext; Anext = tmp;
      }
      T* tmp = A; A = A_new; A_new = tmp;
      if (se) {                 /* from-scratch amplitude of the current A */
        if (have_new) { s_ph = n_ph; s_la = n_la; }
        else if (kind == 0) FN(orc_slogdet)(n, A, &s_ph, &s_la);
        else FN(orc_slogpf)(n, A, &s_ph, &s_la);
      }
      const double ar = ABS(r);
      phase = phase * (r / ar);
      logabs = logabs + log(ar);
      for (int a = 0; a < k; ++a) {
        const int32_t o = occ[p[a]];
        occ[p[a]] = unocc[jj[a]];
        unocc[jj[a]] = o;
      }
    }
  }
  if (dur) *dur = (cfg->mark_step < steps) ? orc_now() - t_mark : 0.0;
  if (!se && cfg->final_scratch) {
    if (kind == 0) FN(orc_slogdet)(n, A, &s_ph, &s_la); else FN(orc_slogpf)(n, A, &s_ph, &s_la);
  }
  if (A_out) memcpy(A_out, A, (size_t)n * n * sizeof(T));
  if (Ainv_out) {
    if (delayed) {
      if (kind == 0) FN(det_carrier_inverse)(&car, Ainv_out); else FN(pf_carrier_inverse)(&car, Ainv_out);
    } else {
      memcpy(Ainv_out, Ainv, (size_t)n * n * sizeof(T));
    }
  }
  if (occ_out) memcpy(occ_out, occ, (size_t)n * sizeof(int32_t));
  if (unocc_out) memcpy(unocc_out, unocc, (size_t)(M - n) * sizeof(int32_t));
  amp[0] = phase; amp[1] = s_ph; amp[2] = ph0;
  logs[0] = logabs; logs[1] = s_la; logs[2] = la0;
  if (delayed) FN(carrier_free)(&car);
  free(occ); free(unocc); free(occ_new); free(A); free(A_new); free(Ainv); free(Anext);
  free(u); free(v); free(oldr); free(newr);
  return ok;
}

/* Many independent walkers: walker w uses the w-th slice of every array (P, J are
 * [W][steps][k], xi [W][steps]).  OpenMP `parallel for` over walkers, `threads`
 * workers (0 = all cores): the CPU baseline of bench.py and the parity tests. */
int FN(orc_batch)(const orc_cfg* cfg, int W, int threads, const T* orb, const int32_t* occ,
                  const int32_t* unocc, const int32_t* P, const int32_t* J, const double* xi,
                  T* r_lemma, T* r_scratch, uint8_t* accepted, uint8_t* near_tie, double* prob,
                  T* A_out, T* Ainv_out, int32_t* occ_out, int32_t* unocc_out, T* amp, double* logs,
                  double* dur /* [W] or NULL */) {
  const size_t n = cfg->n, M = cfg->M, k = cfg->k, steps = cfg->steps;
  const size_t orb_sz = cfg->kind == 0 ? M * n : M * M;
  int ok_all = 1;
#ifdef _OPENMP
  if (threads > 0) omp_set_num_threads(threads);
#endif
#pragma omp parallel for schedule(dynamic, 1) reduction(&& : ok_all)
  for (int w = 0; w < W; ++w) {
    const int ok = FN(orc_trajectory)(
        cfg, orb + w * orb_sz, occ + w * n, unocc + w * (M - n), P + w * steps * k, J + w * steps * k,
        xi + w * steps, r_lemma + w * steps, r_scratch + w * steps, accepted + w * steps,
        near_tie + w * steps, prob + w * steps, A_out ? A_out + w * n * n : NULL,
        Ainv_out ? Ainv_out + w * n * n : NULL, occ_out ? occ_out + w * n : NULL,
        unocc_out ? unocc_out + w * (M - n) : NULL, amp + w * 3, logs + w * 3, dur ? dur + w : NULL);
    ok_all = ok_all && ok;
  }
  return ok_all;
}
