/*
 * dmuon_oracle.c -- fp64 CPU oracle for the Muon optimizer step of DMuon (arxiv/paper_2606_27153).
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke() and the
 * cpu_baseline / --impl reference legs of bench.py may load it.  It shares no code, header,
 * table or helper with the CUDA path (paper_2606_27153_b200/csrc) and never calls it.
 *
 * What it computes, written out step by step in the paper's order and notation, all in fp64,
 * dense, with no blocking, no symmetry shortcut and no fusion:
 *
 *   NS_k (Eq. 2, in the Gram form of PAPER.md:170, section 3.3):
 *       G_i = X_i X_i^T ; P_i = a I + b G_i + c G_i^2 ; X_{i+1} = P_i X_i
 *     written here, as BASELINE.json:north_star does, as
 *       A = X X^T ; B = b A + c A A ; X <- a X + B X .
 *     "whenever m < n": the iteration runs on the orientation with rows <= cols;
 *     a tall input is transposed first and the result transposed back.
 *   Normalisation before NS: X_0 = U / (||U||_F + eps)    (reading N1/N2; paper silent)
 *   Muon step (Eq. 1; Algorithm 1 lines 12-15):
 *       M' = mu M + G ; U = G + mu M'          (Nesterov form, reading N3)
 *       U  <- RNE_bf16(U)                      (reading N15, the "bf16 cast" of north_star)
 *       O  = NS_k(U)
 *       W' = W - lr ( sqrt(max(1, rows/cols)) O + wd W )     (readings N4, N5)
 *
 * Pins (tests/test_oracle_pins.py, -m "not gpu"): scalar closed form p(s)=a s+b s^3+c s^5 iterated on
 * diagonal and orthogonal-times-diagonal inputs; SVD-derived polar structure on tiny matrices;
 * exact symmetry of A; singular values inside the quintic's invariant band; Eq. 2 evaluated
 * literally in long double; Eq. 4 G_{i+1} = P G P; the convergent cubic (1.5,-0.5,0) against the
 * exact polar factor; transpose equivariance; a hand-worked 2x3 Muon step.
 * Parity unpinned: the conventions N3 (momentum form), N4 (update scale), N5 (weight-decay form)
 * have no statement in the paper to pin them against; they are readings, listed in DESIGN.md.
 *
 *   AdamW for the non-matrix parameters (Alg. 1 l.16 "non-matrix params: sharded AdamW
 *   through the host stack"; decoupled weight decay is the paper's citation [16]).  The
 *   paper prints no formula; reading N17 takes the host stack's (PyTorch's) convention:
 *       m_t = beta1 m + (1 - beta1) g ;  v_t = beta2 v + (1 - beta2) g^2
 *       mhat = m_t / (1 - beta1^t) ;  vhat = v_t / (1 - beta2^t)
 *       p_t = p - lr ( mhat / (sqrt(vhat) + eps) + wd p )
 *   Pins: torch.optim.AdamW in float64 on the CPU over several steps (a library routine, not this
 *   file); the closed form of step 1 (mhat = g, vhat = g^2).
 */
#include <math.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define ORACLE_API __attribute__((visibility("default")))

ORACLE_API int oracle_num_threads(void) {
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}

/* Round a double to the nearest bfloat16 value (8 significant bits, exponent range of float),
 * ties to even; returned as a double.  Used at the two points where the method stores bf16:
 * the cast of U (reading N15) and the stored M', W'. */
ORACLE_API double oracle_round_bf16(double x) {
  if (x == 0.0 || isnan(x) || isinf(x)) return x;
  int e;
  (void)frexp(x, &e);                /* |x| = f * 2^e, f in [0.5, 1)  ->  leading bit at 2^(e-1) */
  int lead = e - 1;
  if (lead < -126) lead = -126;      /* bf16 subnormals share the quantum of the smallest normal */
  double q = ldexp(1.0, lead - 7);   /* spacing of bf16 values at this exponent (7 mantissa bits) */
  double r = nearbyint(x / q) * q;   /* x/q is exact (power of two); nearbyint is ties-to-even */
  const double BF16_MAX = 3.3895313892515355e38; /* 0x7F7F */
  if (fabs(r) > BF16_MAX) return x > 0 ? INFINITY : -INFINITY;
  return r;
}

ORACLE_API void oracle_round_bf16_array(const double* x, double* out, long long n) {
  for (long long i = 0; i < n; ++i) out[i] = oracle_round_bf16(x[i]);
}

static double* dalloc(size_t n) {
  double* p = (double*)malloc((n ? n : 1) * sizeof(double));
  return p;
}

/* C[p x q] = T^T for T[q x p] (plain transpose copy). */
static void transpose(const double* T, int q, int p, double* C) {
  for (int i = 0; i < q; ++i)
    for (int j = 0; j < p; ++j) C[(size_t)j * q + i] = T[(size_t)i * p + j];
}

/* C[m x n] = beta * D[m x n] + alpha * L[m x k] * R[k x n]   (D may be NULL when beta == 0).
 * Plain triple loop; each C[i][j] is sum over kk = 0..k-1 in ascending order. */
static void matmul(int m, int k, int n, double alpha, const double* L, const double* R,
                   double beta, const double* D, double* C) {
#pragma omp parallel for schedule(static)
  for (int i = 0; i < m; ++i) {
    double* c = C + (size_t)i * n;
    for (int j = 0; j < n; ++j) c[j] = 0.0;
    for (int kk = 0; kk < k; ++kk) {
      const double l = L[(size_t)i * k + kk];
      const double* r = R + (size_t)kk * n;
      for (int j = 0; j < n; ++j) c[j] += l * r[j];
    }
    if (D) {
      const double* d = D + (size_t)i * n;
      for (int j = 0; j < n; ++j) c[j] = beta * d[j] + alpha * c[j];
    } else {
      for (int j = 0; j < n; ++j) c[j] = alpha * c[j];
    }
  }
}

/* One Gram-form NS step on X[m x n], m <= n:  A = X X^T ; B = b A + c A A ;
 * X <- a X + B X.  If A_out / B_out are non-NULL the step's A and B are copied there. */
static int ns_step(double* X, int m, int n, double a, double b, double c, double* A_out,
                   double* B_out) {
  double* XT = dalloc((size_t)n * m);
  double* A = dalloc((size_t)m * m);
  double* B = dalloc((size_t)m * m);
  double* Xn = dalloc((size_t)m * n);
  if (!XT || !A || !B || !Xn) { free(XT); free(A); free(B); free(Xn); return -1; }
  transpose(X, m, n, XT);
  matmul(m, n, m, 1.0, X, XT, 0.0, NULL, A);  /* A = X X^T  (full dense; symmetric by construction) */
  matmul(m, m, m, c, A, A, b, A, B);          /* B = b A + c (A A) */
  matmul(m, m, n, 1.0, B, X, a, X, Xn);       /* X' = a X + B X */
  memcpy(X, Xn, (size_t)m * n * sizeof(double));
  if (A_out) memcpy(A_out, A, (size_t)m * m * sizeof(double));
  if (B_out) memcpy(B_out, B, (size_t)m * m * sizeof(double));
  free(XT); free(A); free(B); free(Xn);
  return 0;
}

/* Frobenius norm, plain ascending-order sum of squares. */
ORACLE_API double oracle_fro_norm(const double* X, long long count) {
  double s = 0.0;
  for (long long i = 0; i < count; ++i) s += X[i] * X[i];
  return sqrt(s);
}

/* NS_steps(X) in place.  X is rows x cols, row-major.  coeffs holds per_step ? steps*3 : 3 doubles
 * (a, b, c).  normalize != 0 divides by (||X||_F + eps) first (readings N1, N2).
 * A1_out, if non-NULL, receives the FIRST step's A (min(rows,cols)^2 doubles) for the symmetry pin.
 * Returns 0, or -1 on allocation failure / bad arguments. */
ORACLE_API int oracle_ns(double* X, int rows, int cols, int steps, const double* coeffs,
                         int per_step, int normalize, double eps, double* A1_out) {
  if (!X || rows <= 0 || cols <= 0 || steps < 0 || !coeffs) return -1;
  const int tall = rows > cols;              /* work in the smaller Gram dimension */
  const int m = tall ? cols : rows, n = tall ? rows : cols;
  double* Y = X;
  if (tall) {
    Y = dalloc((size_t)m * n);
    if (!Y) return -1;
    transpose(X, rows, cols, Y);
  }
  if (normalize) {
    const double s = oracle_fro_norm(Y, (long long)m * n) + eps;
    for (size_t i = 0; i < (size_t)m * n; ++i) Y[i] = Y[i] / s;
  }
  int rc = 0;
  for (int i = 0; i < steps && rc == 0; ++i) {
    const double* q = coeffs + (per_step ? 3 * i : 0);
    rc = ns_step(Y, m, n, q[0], q[1], q[2], i == 0 ? A1_out : NULL, NULL);
  }
  if (tall) {
    if (rc == 0) transpose(Y, m, n, X);
    free(Y);
  }
  return rc;
}

/* One Muon step for one rows x cols parameter (Eq. 1; Alg. 1 l.12-15 :232-238).
 * Inputs W, G, M: doubles holding the stored (bf16-exact) values.  lr, mu, wd: the values the
 * caller passes to the C ABI (floats widened to double).  u_cast != 0 applies reading N15.
 * Outputs (each rows*cols doubles, any may be NULL):
 *   M_out   = mu M + G                       (unrounded)
 *   U_out   = G + mu M_out, after the cast if u_cast
 *   O_out   = NS_steps(U_out)
 *   W_out   = W - lr ( sqrt(max(1, rows/cols)) O + wd W )   (unrounded)
 * The caller rounds M_out / W_out with oracle_round_bf16 to get the stored values. */
ORACLE_API int oracle_muon_step(const double* W, const double* G, const double* M, int rows, int cols,
                                double lr, double mu, double wd, int steps, const double* coeffs,
                                int per_step, double eps, int u_cast, double* M_out,
                                double* U_out, double* O_out, double* W_out) {
  if (!W || !G || !M || rows <= 0 || cols <= 0) return -1;
  const size_t cnt = (size_t)rows * cols;
  double* Mn = dalloc(cnt);
  double* U = dalloc(cnt);
  if (!Mn || !U) { free(Mn); free(U); return -1; }
  for (size_t i = 0; i < cnt; ++i) {
    Mn[i] = mu * M[i] + G[i];                 /* N3: M' = mu M + G */
    U[i] = G[i] + mu * Mn[i];                 /*     U  = G + mu M' (from the unrounded M') */
    if (u_cast) U[i] = oracle_round_bf16(U[i]); /* N15 */
  }
  if (U_out) memcpy(U_out, U, cnt * sizeof(double));
  int rc = oracle_ns(U, rows, cols, steps, coeffs, per_step, 1, eps, NULL);
  if (rc == 0) {
    const double ratio = (double)rows / (double)cols;
    const double scale = sqrt(ratio > 1.0 ? ratio : 1.0);   /* N4 */
    if (O_out) memcpy(O_out, U, cnt * sizeof(double));
    if (W_out)
      for (size_t i = 0; i < cnt; ++i) W_out[i] = W[i] - lr * (scale * U[i] + wd * W[i]); /* N5 */
    if (M_out) memcpy(M_out, Mn, cnt * sizeof(double));
  }
  free(Mn); free(U);
  return rc;
}

/* One decoupled-AdamW step over n elements (reading N17), all fp64.  step counts from 1.
 * Outputs (each n doubles): p_out (unrounded), m_out, v_out. */
ORACLE_API int oracle_adamw_step(const double* p, const double* g, const double* m, const double* v, long long n,
                                 double lr, double beta1, double beta2, double eps, double wd, int step,
                                 double* p_out, double* m_out, double* v_out) {
  if (!p || !g || !m || !v || !p_out || !m_out || !v_out || n < 0 || step < 1) return -1;
  const double bc1 = 1.0 - pow(beta1, (double)step);   /* bias corrections */
  const double bc2 = 1.0 - pow(beta2, (double)step);
  for (long long i = 0; i < n; ++i) {
    const double mt = beta1 * m[i] + (1.0 - beta1) * g[i];
    const double vt = beta2 * v[i] + (1.0 - beta2) * g[i] * g[i];
    const double mhat = mt / bc1;
    const double vhat = vt / bc2;
    p_out[i] = p[i] - lr * (mhat / (sqrt(vhat) + eps) + wd * p[i]);
    m_out[i] = mt;
    v_out[i] = vt;
  }
  return 0;
}
