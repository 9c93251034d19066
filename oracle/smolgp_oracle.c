/* smolgp_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, CPU-only restatement of what arXiv:2601.02527 ("Scalable GPs for
 * integrated and overlapping measurements via augmented state-space models")
 * computes.  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * --impl reference legs may load it.  It shares no code, header, table or
 * constant with the CUDA path under paper_2601_02527_b200/csrc/.
 *
 * P:<line> = line of /root/reference/PAPER.md.
 *
 * Two independent routes to the same posterior:
 *  (1) oracle_dense_*: the DEFINITION (Eq. 2.4 with the exposure-integrated
 *      kernel of Eq. 3.1): closed-form double integral of k over two exposures
 *      evaluated in __float128, Cholesky in REAL.  O(N^3); small N only.
 *  (2) oracle_ssm: the paper's sequential algorithm, step by step: augmented SSM
 *      (Eq. 3.3-3.10, 3.17-3.19), integrated Kalman filter (Eq. 3.13-3.15, 2.21-2.22),
 *      integrated RTS smoother (Eq. 2.23, 3.16), log-likelihood (Eq. 2.26) and
 *      Algorithm 1 with the readings listed in DESIGN.md.
 *      A second backward pass (two-filter / backward information form) is provided
 *      because the textbook RTS gain inverts a nearly singular P^-_{k+1} right after a
 *      reset; it is the parity reference for stiff cases (R7).
 *  (3) oracle_ssm_sqrt (Part 7): the same passes in square-root (Cholesky-factor) array form,
 *      the paper's named remedy for the conditioning of (2); pinned to (1) and (2)
 *      in tests/test_oracle_sqrt_pins.py.
 *
 * Compile twice: -DREAL_IS_LONG_DOUBLE (parity reference, x87 80-bit) and plain
 * double (the timed CPU baseline).  Pins: tests/test_oracle_*.py (-m "not gpu").
 * Parity status: every exported function is pinned; see DESIGN.md section "Oracle pins".
 */
#include <math.h>
#include <quadmath.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#include <time.h>

#ifdef REAL_IS_LONG_DOUBLE
typedef long double real;
#define R_EXP expl
#define R_SQRT sqrtl
#define R_LOG logl
#define R_FABS fabsl
#else
typedef double real;
#define R_EXP exp
#define R_SQRT sqrt
#define R_LOG log
#define R_FABS fabs
#endif

#define MAXN 40   /* max augmented state dimension n = d + N_inst */
#define MAXBD 4   /* max dimension of one block-diagonal block of F */
#define MAXBLK 32 /* max number of blocks */
#define MAXINST 16
#define PI_Q 3.14159265358979323846264338327950288Q
#define PI_R ((real)3.14159265358979323846264338327950288L)

enum { FAM_MATERN32 = 0, FAM_MATERN52 = 1, FAM_SHO = 2, FAM_MATERN32_X_PERIODIC = 3 };

/* one additive kernel component (App. C.1).  inst_mask bit i set <=> the
 * component enters instrument i's integrand H_i of Eq. 3.2.
 *   MATERN32 / MATERN52 : p0 = ell
 *   SHO                 : p0 = omega0, p1 = Q
 *   MATERN32_X_PERIODIC : p0 = ell, p1 = period, p2 = ell_periodic, order = J  */
typedef struct {
  int32_t family, order;
  uint32_t inst_mask;
  double sigma, p0, p1, p2;
} ocomp;

/* ------------------------------------------------------------------------------------------
 * Modified Bessel I_j(x) by its power series; series coefficients q_j^2 of the periodic
 * kernel exp(-2 sin^2(pi tau/P)/ell_p^2) = sum_j q_j^2 cos(j w tau)  (Solin & Sarkka 2014a,
 * cited P:47; the paper prints nothing: DESIGN.md reading R11).
 * ------------------------------------------------------------------------------------------ */
static long double bessel_i(int j, long double x) {
  long double term = 1.0L, sum;
  for (int m = 1; m <= j; ++m) term *= (x / 2) / m; /* (x/2)^j / j! */
  sum = term;
  for (int m = 1; m < 60; ++m) {
    term *= (x / 2) * (x / 2) / ((long double)m * (m + j));
    sum += term;
  }
  return sum;
}
static long double periodic_q2(int j, long double ell_p) {
  long double a = 1.0L / (ell_p * ell_p);
  return (j == 0 ? 1.0L : 2.0L) * bessel_i(j, a) * expl(-a);
}

/* ==========================================================================================
 * Part 1.  Scalar kernels as sums of  Re[(a0 + a1 tau + a2 tau^2) exp(-z tau)]  (complex z)
 * ========================================================================================== */
typedef struct {
  __complex128 z, a0, a1, a2;
  uint32_t mask;
} kterm;

static int build_terms(int ncomp, const ocomp *c, kterm *t, int maxt) {
  int nt = 0;
  for (int m = 0; m < ncomp; ++m) {
    __float128 s2 = (__float128)c[m].sigma * c[m].sigma;
    if (c[m].family == FAM_MATERN32 || c[m].family == FAM_MATERN52) {
      if (nt >= maxt) return -1;
      __float128 lam = sqrtq(c[m].family == FAM_MATERN32 ? 3.0Q : 5.0Q) / c[m].p0;
      t[nt].z = lam;
      t[nt].a0 = s2;
      t[nt].a1 = s2 * lam;
      t[nt].a2 = c[m].family == FAM_MATERN52 ? s2 * lam * lam / 3 : 0.0Q;
      t[nt++].mask = c[m].inst_mask;
    } else if (c[m].family == FAM_SHO) { /* (Kernel) P:753 */
      __float128 w0 = c[m].p0, Q = c[m].p1;
      __float128 a = w0 / (2 * Q);
      if (Q > 0.5Q) {
        __float128 eta = sqrtq(1 - 1 / (4 * Q * Q));
        if (nt >= maxt) return -1;
        __complex128 zz, aa;
        __real__ zz = a;   __imag__ zz = -eta * w0;
        __real__ aa = s2;  __imag__ aa = -s2 / (2 * eta * Q);
        t[nt].z = zz;
        t[nt].a0 = aa; /* Re[(1 - iA) e^{-a tau} e^{+i b tau}] = e^{-a tau}(cos + A sin) */
        t[nt].a1 = 0; t[nt].a2 = 0;
        t[nt++].mask = c[m].inst_mask;
      } else if (Q == 0.5Q) {
        if (nt >= maxt) return -1;
        t[nt].z = w0; t[nt].a0 = s2; t[nt].a1 = s2 * w0; t[nt].a2 = 0;
        t[nt++].mask = c[m].inst_mask;
      } else { /* cosh + A sinh = (1+A)/2 e^{b tau} + (1-A)/2 e^{-b tau} */
        __float128 eta = sqrtq(1 / (4 * Q * Q) - 1), b = eta * w0, A = 1 / (2 * eta * Q);
        if (nt + 2 > maxt) return -1;
        t[nt].z = a - b; t[nt].a0 = s2 * (1 + A) / 2; t[nt].a1 = 0; t[nt].a2 = 0;
        t[nt++].mask = c[m].inst_mask;
        t[nt].z = a + b; t[nt].a0 = s2 * (1 - A) / 2; t[nt].a1 = 0; t[nt].a2 = 0;
        t[nt++].mask = c[m].inst_mask;
      }
    } else if (c[m].family == FAM_MATERN32_X_PERIODIC) {
      __float128 lam = sqrtq(3.0Q) / c[m].p0, wp = 2 * PI_Q / c[m].p1;
      for (int j = 0; j <= c[m].order; ++j) {
        if (nt >= maxt) return -1;
        __float128 q2 = periodic_q2(j, c[m].p2);
        __complex128 zz;
        __real__ zz = lam; __imag__ zz = -j * wp;
        t[nt].z = zz;
        t[nt].a0 = s2 * q2; t[nt].a1 = s2 * q2 * lam; t[nt].a2 = 0;
        t[nt++].mask = c[m].inst_mask;
      }
    } else
      return -1;
  }
  return nt;
}

/* k(tau) restricted to the components seen by both instruments ia and ib */
static __float128 kern_q(const kterm *t, int nt, int ia, int ib, __float128 tau) {
  __float128 s = 0;
  tau = fabsq(tau);
  for (int i = 0; i < nt; ++i) {
    if (!((t[i].mask >> ia) & 1u) || !((t[i].mask >> ib) & 1u)) continue;
    s += crealq((t[i].a0 + t[i].a1 * tau + t[i].a2 * tau * tau) * cexpq(-t[i].z * tau));
  }
  return s;
}
/* G(u) = int_0^|u| (|u| - tau) k(tau) dtau   (even; G'' = k; G(0)=G'(0)=0).  Per term with
 * x = z u:  g0=(e^-x - 1 + x)/z^2, g1=(x-2+(x+2)e^-x)/z^3, g2=(2x-6+(x^2+4x+6)e^-x)/z^4. */
static __float128 G_q(const kterm *t, int nt, int ia, int ib, __float128 u) {
  __float128 s = 0;
  u = fabsq(u);
  for (int i = 0; i < nt; ++i) {
    if (!((t[i].mask >> ia) & 1u) || !((t[i].mask >> ib) & 1u)) continue;
    __complex128 z = t[i].z, x = z * u, e = cexpq(-x);
    __complex128 g0 = (e - 1 + x) / (z * z);
    __complex128 g1 = (x - 2 + (x + 2) * e) / (z * z * z);
    __complex128 g2 = (2 * x - 6 + (x * x + 4 * x + 6) * e) / (z * z * z * z);
    s += crealq(t[i].a0 * g0 + t[i].a1 * g1 + t[i].a2 * g2);
  }
  return s;
}
/* K1(u) = sign(u) int_0^|u| k */
static __float128 K1_q(const kterm *t, int nt, int ia, int ib, __float128 u) {
  __float128 s = 0, au = fabsq(u);
  for (int i = 0; i < nt; ++i) {
    if (!((t[i].mask >> ia) & 1u) || !((t[i].mask >> ib) & 1u)) continue;
    __complex128 z = t[i].z, x = z * au, e = cexpq(-x);
    __complex128 k0 = (1 - e) / z;
    __complex128 k1 = (1 - (1 + x) * e) / (z * z);
    __complex128 k2 = (2 - (x * x + 2 * x + 2) * e) / (z * z * z);
    s += crealq(t[i].a0 * k0 + t[i].a1 * k1 + t[i].a2 * k2);
  }
  return u < 0 ? -s : s;
}

/* k(tau) for the component set shared by instruments ia, ib (plain kernel, Eq. 2.20 check) */
int oracle_kernel(int ncomp, const ocomp *comp, int ia, int ib, int ntau, const double *tau,
                  double *out) {
  kterm t[64];
  int nt = build_terms(ncomp, comp, t, 64);
  if (nt < 0) return -1;
  for (int i = 0; i < ntau; ++i) out[i] = (double)kern_q(t, nt, ia, ib, tau[i]);
  return 0;
}

/* Exposure-integrated covariance, Eq. 3.1 with Eq. 3.2's H_n inside the integral:
 *   delta_n delta_m K_nm = G(e_n-s_m) + G(s_n-e_m) - G(e_n-e_m) - G(s_n-s_m)
 * (integrate G'' = k twice over the rectangle; covers every overlap case, incl. n = m).
 * Evaluated in __float128 because the four terms cancel heavily for slow kernels. */
static __float128 kff_q(const kterm *t, int nt, int ia, int ib, double sa, double ea, double sb,
                        double eb) {
  __float128 Sa = sa, Ea = ea, Sb = sb, Eb = eb;
  __float128 v = G_q(t, nt, ia, ib, Ea - Sb) + G_q(t, nt, ia, ib, Sa - Eb) -
                 G_q(t, nt, ia, ib, Ea - Eb) - G_q(t, nt, ia, ib, Sa - Sb);
  return v / ((Ea - Sa) * (Eb - Sb));
}

int oracle_kff(int ncomp, const ocomp *comp, int N, const double *ts, const double *te,
               const int32_t *inst, double *K /* N*N row-major */) {
  kterm t[64];
  int nt = build_terms(ncomp, comp, t, 64);
  if (nt < 0) return -1;
  for (int i = 0; i < N; ++i)
    for (int j = 0; j <= i; ++j) {
      double v = (double)kff_q(t, nt, inst[i], inst[j], ts[i], te[i], ts[j], te[j]);
      K[(size_t)i * N + j] = v;
      K[(size_t)j * N + i] = v;
    }
  return 0;
}

/* ==========================================================================================
 * Part 2.  Dense integrated-GP solver (the definition), Eq. 2.4, loglik P:258.
 * ========================================================================================== */
static int chol_lower(real *A, int N) { /* in place, row-major, lower */
  for (int j = 0; j < N; ++j) {
    real d = A[(size_t)j * N + j];
    for (int k = 0; k < j; ++k) d -= A[(size_t)j * N + k] * A[(size_t)j * N + k];
    if (!(d > 0)) return -1;
    d = R_SQRT(d);
    A[(size_t)j * N + j] = d;
    for (int i = j + 1; i < N; ++i) {
      real s = A[(size_t)i * N + j];
      for (int k = 0; k < j; ++k) s -= A[(size_t)i * N + k] * A[(size_t)j * N + k];
      A[(size_t)i * N + j] = s / d;
    }
  }
  return 0;
}
static void fwd_sub(const real *L, int N, real *b) { /* solve L x = b */
  for (int i = 0; i < N; ++i) {
    real s = b[i];
    for (int k = 0; k < i; ++k) s -= L[(size_t)i * N + k] * b[k];
    b[i] = s / L[(size_t)i * N + i];
  }
}
static void bwd_sub(const real *L, int N, real *b) { /* solve L^T x = b */
  for (int i = N - 1; i >= 0; --i) {
    real s = b[i];
    for (int k = i + 1; k < N; ++k) s -= L[(size_t)k * N + i] * b[k];
    b[i] = s / L[(size_t)i * N + i];
  }
}

/* loglik = -1/2 (y^T C^-1 y + log det C + N log 2 pi),  C = K + diag(sigma^2);
 * mean = K C^-1 y, var = diag(K - K C^-1 K)   (noise-free exposure averages);
 * queries: instantaneous latent of instrument query_inst, K*_qn = (1/delta_n) int k,
 * K** = k(0).  Returns 0, or -2 if C is not positive definite. */
int oracle_dense(int ncomp, const ocomp *comp, int N, const double *ts, const double *te,
                 const int32_t *inst, const double *y, const double *sigma, int M,
                 const double *tq, int query_inst, double *loglik, double *mean, double *var,
                 double *mq, double *vq) {
  kterm t[64];
  int nt = build_terms(ncomp, comp, t, 64);
  if (nt < 0) return -1;
  size_t NN = (size_t)N * N;
  real *K = malloc(NN * sizeof(real)), *L = malloc(NN * sizeof(real));
  real *a = malloc(N * sizeof(real)), *col = malloc(N * sizeof(real));
  if (!K || !L || !a || !col) return -4;
  for (int i = 0; i < N; ++i)
    for (int j = 0; j <= i; ++j) {
      real v = (real)kff_q(t, nt, inst[i], inst[j], ts[i], te[i], ts[j], te[j]);
      K[(size_t)i * N + j] = K[(size_t)j * N + i] = v;
    }
  memcpy(L, K, NN * sizeof(real));
  for (int i = 0; i < N; ++i) L[(size_t)i * N + i] += (real)sigma[i] * (real)sigma[i];
  if (chol_lower(L, N)) { free(K); free(L); free(a); free(col); return -2; }
  for (int i = 0; i < N; ++i) a[i] = y[i];
  fwd_sub(L, N, a);
  real quad = 0, logdet = 0;
  for (int i = 0; i < N; ++i) { quad += a[i] * a[i]; logdet += 2 * R_LOG(L[(size_t)i * N + i]); }
  if (loglik) *loglik = (double)(-0.5L * (quad + logdet + N * R_LOG((real)(2 * PI_R))));
  bwd_sub(L, N, a); /* a = C^-1 y */
  if (mean)
    for (int i = 0; i < N; ++i) {
      real s = 0;
      for (int j = 0; j < N; ++j) s += K[(size_t)i * N + j] * a[j];
      mean[i] = (double)s;
    }
  if (var)
    for (int i = 0; i < N; ++i) { /* var_i = K_ii - |L^-1 K_:i|^2 */
      for (int j = 0; j < N; ++j) col[j] = K[(size_t)j * N + i];
      fwd_sub(L, N, col);
      real s = 0;
      for (int j = 0; j < N; ++j) s += col[j] * col[j];
      var[i] = (double)(K[(size_t)i * N + i] - s);
    }
  for (int q = 0; q < M; ++q) {
    for (int j = 0; j < N; ++j) {
      __float128 T = tq[q];
      col[j] = (real)((K1_q(t, nt, query_inst, inst[j], T - (__float128)ts[j]) -
                       K1_q(t, nt, query_inst, inst[j], T - (__float128)te[j])) /
                      ((__float128)te[j] - (__float128)ts[j]));
    }
    real s = 0;
    for (int j = 0; j < N; ++j) s += col[j] * a[j];
    if (mq) mq[q] = (double)s;
    fwd_sub(L, N, col);
    real v = (real)kern_q(t, nt, query_inst, query_inst, 0);
    for (int j = 0; j < N; ++j) v -= col[j] * col[j];
    if (vq) vq[q] = (double)v;
  }
  free(K); free(L); free(a); free(col);
  return 0;
}

/* ==========================================================================================
 * Part 3.  State-space model: blocks (F, W = L Qc L^T, Pinf, H), sums (C2) and products (C6, C8)
 * ========================================================================================== */
typedef struct {
  int d;
  real F[MAXBD * MAXBD], W[MAXBD * MAXBD], P[MAXBD * MAXBD], H[MAXBD];
  uint32_t mask;
} block;

static void blk_zero(block *b, int d, uint32_t mask) {
  memset(b, 0, sizeof(*b));
  b->d = d;
  b->mask = mask;
}
/* Matern-3/2 (standard form, the paper cites Hartikainen & Sarkka 2010; reading R10) */
static void blk_matern32(block *b, real sigma, real ell, uint32_t mask) {
  real lam = R_SQRT((real)3) / ell, s2 = sigma * sigma;
  blk_zero(b, 2, mask);
  b->F[0 * 2 + 1] = 1; b->F[1 * 2 + 0] = -lam * lam; b->F[1 * 2 + 1] = -2 * lam;
  b->W[1 * 2 + 1] = 4 * lam * lam * lam * s2;
  b->P[0] = s2; b->P[3] = s2 * lam * lam;
  b->H[0] = 1;
}
static void blk_matern52(block *b, real sigma, real ell, uint32_t mask) {
  real lam = R_SQRT((real)5) / ell, s2 = sigma * sigma, l2 = lam * lam;
  blk_zero(b, 3, mask);
  b->F[0 * 3 + 1] = 1; b->F[1 * 3 + 2] = 1;
  b->F[2 * 3 + 0] = -l2 * lam; b->F[2 * 3 + 1] = -3 * l2; b->F[2 * 3 + 2] = -3 * lam;
  b->W[2 * 3 + 2] = 16 * s2 * l2 * l2 * lam / 3;
  b->P[0] = s2; b->P[0 * 3 + 2] = b->P[2 * 3 + 0] = -s2 * l2 / 3;
  b->P[1 * 3 + 1] = s2 * l2 / 3; b->P[2 * 3 + 2] = s2 * l2 * l2;
  b->H[0] = 1;
}
/* SHO: Eq. B6, B8 */
static void blk_sho(block *b, real sigma, real w0, real Q, uint32_t mask) {
  real s2 = sigma * sigma;
  blk_zero(b, 2, mask);
  b->F[0 * 2 + 1] = 1; b->F[1 * 2 + 0] = -w0 * w0; b->F[1 * 2 + 1] = -w0 / Q;
  b->W[1 * 2 + 1] = 2 * w0 * w0 * w0 * s2 / Q;
  b->P[0] = s2; b->P[3] = s2 * w0 * w0;
  b->H[0] = 1;
}
/* product of two blocks, Eq. C6 and C8 with L = I */
static int blk_kron(block *o, const block *a, const block *b) {
  int da = a->d, db = b->d, d = da * db;
  if (d > MAXBD) return -1;
  blk_zero(o, d, a->mask & b->mask);
  for (int i = 0; i < da; ++i)
    for (int j = 0; j < da; ++j)
      for (int k = 0; k < db; ++k)
        for (int l = 0; l < db; ++l) {
          int r = i * db + k, c = j * db + l;
          real Ib = (k == l), Ia = (i == j);
          o->F[r * d + c] = a->F[i * da + j] * Ib + Ia * b->F[k * db + l];
          o->P[r * d + c] = a->P[i * da + j] * b->P[k * db + l];
          o->W[r * d + c] = a->W[i * da + j] * b->P[k * db + l] + a->P[i * da + j] * b->W[k * db + l];
        }
  for (int i = 0; i < da; ++i)
    for (int k = 0; k < db; ++k) o->H[i * db + k] = a->H[i] * b->H[k];
  return 0;
}

typedef struct {
  int nblk, d, ninst, n;
  block blk[MAXBLK];
  int off[MAXBLK];
} model;

static int build_model(model *M, int ncomp, const ocomp *c, int ninst) {
  memset(M, 0, sizeof(*M));
  M->ninst = ninst;
  if (ninst < 1 || ninst > MAXINST) return -1;
  for (int m = 0; m < ncomp; ++m) {
    if (c[m].family == FAM_MATERN32) {
      if (M->nblk >= MAXBLK) return -1;
      blk_matern32(&M->blk[M->nblk++], c[m].sigma, c[m].p0, c[m].inst_mask);
    } else if (c[m].family == FAM_MATERN52) {
      if (M->nblk >= MAXBLK) return -1;
      blk_matern52(&M->blk[M->nblk++], c[m].sigma, c[m].p0, c[m].inst_mask);
    } else if (c[m].family == FAM_SHO) {
      if (M->nblk >= MAXBLK) return -1;
      blk_sho(&M->blk[M->nblk++], c[m].sigma, c[m].p0, c[m].p1, c[m].inst_mask);
    } else if (c[m].family == FAM_MATERN32_X_PERIODIC) {
      block env;
      blk_matern32(&env, c[m].sigma, c[m].p0, c[m].inst_mask);
      real wp = 2 * (real)PI_R / (real)c[m].p1;
      for (int j = 0; j <= c[m].order; ++j) {
        block per;
        real q2 = (real)periodic_q2(j, c[m].p2);
        if (j == 0) {
          blk_zero(&per, 1, c[m].inst_mask);
          per.P[0] = q2; per.H[0] = 1;
        } else {
          blk_zero(&per, 2, c[m].inst_mask);
          per.F[0 * 2 + 1] = -j * wp; per.F[1 * 2 + 0] = j * wp;
          per.P[0] = per.P[3] = q2;
          per.H[0] = 1;
        }
        if (M->nblk >= MAXBLK) return -1;
        if (blk_kron(&M->blk[M->nblk++], &env, &per)) return -1;
      }
    } else
      return -1;
  }
  int o = 0;
  for (int b = 0; b < M->nblk; ++b) { M->off[b] = o; o += M->blk[b].d; }
  M->d = o;
  M->n = o + ninst;
  return M->n <= MAXN ? 0 : -1;
}

int oracle_model_dim(int ncomp, const ocomp *comp, int ninst) {
  model M;
  if (build_model(&M, ncomp, comp, ninst)) return -1;
  return M.n;
}

/* Dense augmented continuous-time matrices (Eq. 3.17): Ft (n*n), Wt = Lt Qc Lt^T (n*n),
 * Pinf of the base state (d*d) and the integrand rows H_i (ninst*d).  Row z_i of Ft is H_i:
 * the printed "ones along the first column" generalised to multi-component kernels
 * as Eq. 3.2 requires (reading R2). */
int oracle_ssm_matrices(int ncomp, const ocomp *comp, int ninst, double *Ft, double *Wt,
                        double *Pinf, double *Hrows) {
  model M;
  if (build_model(&M, ncomp, comp, ninst)) return -1;
  int n = M.n, d = M.d;
  if (Ft) memset(Ft, 0, sizeof(double) * n * n);
  if (Wt) memset(Wt, 0, sizeof(double) * n * n);
  if (Pinf) memset(Pinf, 0, sizeof(double) * d * d);
  if (Hrows) memset(Hrows, 0, sizeof(double) * ninst * d);
  for (int b = 0; b < M.nblk; ++b) {
    const block *B = &M.blk[b];
    int o = M.off[b];
    for (int i = 0; i < B->d; ++i)
      for (int j = 0; j < B->d; ++j) {
        if (Ft) Ft[(o + i) * n + o + j] = (double)B->F[i * B->d + j];
        if (Wt) Wt[(o + i) * n + o + j] = (double)B->W[i * B->d + j];
        if (Pinf) Pinf[(o + i) * d + o + j] = (double)B->P[i * B->d + j];
      }
    for (int q = 0; q < ninst; ++q)
      if ((B->mask >> q) & 1u)
        for (int j = 0; j < B->d; ++j) {
          if (Ft) Ft[(d + q) * n + o + j] = (double)B->H[j];
          if (Hrows) Hrows[q * d + o + j] = (double)B->H[j];
        }
  }
  return 0;
}

/* ------------------------------------------------------------------------------------------
 * Discretisation over a step dt (Eq. 2.17-2.19; Eq. 3.7; Eq. 3.10):
 * per block on the augmented pair [x_b ; int H_b x_b] (dimension m = d_b + 1),
 *   Phi~(h) = sum_k F~^k h^k / k!,   Q~(h) = sum_{k>=1} Gamma_k h^k / k!,
 *   Gamma_1 = W~, Gamma_{k+1} = F~ Gamma_k + Gamma_k F~^T     (term-by-term integral of 3.10),
 * at h = dt / 2^s with |F~| h <= 1/2, followed by s doublings
 *   Q~(2h) = Q~(h) + Phi~(h) Q~(h) Phi~(h)^T,  Phi~(2h) = Phi~(h)^2     (semigroup property).
 * No growing exponentials appear, unlike the Van Loan form B13 which the paper itself
 * flags as unstable over long gaps.  Pinned to B10-B12, B19-B20 in tests.
 * ------------------------------------------------------------------------------------------ */
#define MB (MAXBD + 1)
static void disc_block(const block *B, real dt, real *Phi /* m*m */, real *Q /* m*m */) {
  int d = B->d, m = d + 1;
  real F[MB * MB] = {0}, W[MB * MB] = {0};
  for (int i = 0; i < d; ++i)
    for (int j = 0; j < d; ++j) { F[i * m + j] = B->F[i * d + j]; W[i * m + j] = B->W[i * d + j]; }
  for (int j = 0; j < d; ++j) F[d * m + j] = B->H[j];
  real nrm = 0;
  for (int i = 0; i < m; ++i) {
    real r = 0;
    for (int j = 0; j < m; ++j) r += R_FABS(F[i * m + j]);
    if (r > nrm) nrm = r;
  }
  int s = 0;
  real h = dt;
  while (nrm * h > 0.5) { h /= 2; ++s; }
  real Fk[MB * MB] = {0}, Gk[MB * MB], T[MB * MB];
  for (int i = 0; i < m; ++i) Fk[i * m + i] = 1; /* F^0 h^0/0! */
  memcpy(Gk, W, sizeof(Gk));                     /* Gamma_1 */
  memset(Phi, 0, sizeof(real) * m * m);
  memset(Q, 0, sizeof(real) * m * m);
  for (int i = 0; i < m * m; ++i) Phi[i] = Fk[i];
  real c = 1; /* h^k / k! */
  for (int k = 1; k <= 30; ++k) {
    c *= h / k;
    /* Fk <- F * Fk  (= F^k) */
    for (int i = 0; i < m; ++i)
      for (int j = 0; j < m; ++j) {
        real a = 0;
        for (int l = 0; l < m; ++l) a += F[i * m + l] * Fk[l * m + j];
        T[i * m + j] = a;
      }
    memcpy(Fk, T, sizeof(T));
    for (int i = 0; i < m * m; ++i) { Phi[i] += c * Fk[i]; Q[i] += c * Gk[i]; }
    /* Gk <- F Gk + Gk F^T */
    for (int i = 0; i < m; ++i)
      for (int j = 0; j < m; ++j) {
        real a = 0;
        for (int l = 0; l < m; ++l) a += F[i * m + l] * Gk[l * m + j] + Gk[i * m + l] * F[j * m + l];
        T[i * m + j] = a;
      }
    memcpy(Gk, T, sizeof(T));
  }
  for (int it = 0; it < s; ++it) {
    real PQ[MB * MB], N2[MB * MB];
    for (int i = 0; i < m; ++i)
      for (int j = 0; j < m; ++j) {
        real a = 0;
        for (int l = 0; l < m; ++l) a += Phi[i * m + l] * Q[l * m + j];
        PQ[i * m + j] = a;
      }
    for (int i = 0; i < m; ++i)
      for (int j = 0; j < m; ++j) {
        real a = 0;
        for (int l = 0; l < m; ++l) a += PQ[i * m + l] * Phi[j * m + l];
        N2[i * m + j] = Q[i * m + j] + a;
      }
    for (int i = 0; i < m; ++i)
      for (int j = 0; j < m; ++j) {
        real a = 0;
        for (int l = 0; l < m; ++l) a += Phi[i * m + l] * Phi[l * m + j];
        T[i * m + j] = a;
      }
    memcpy(Phi, T, sizeof(T));
    for (int i = 0; i < m; ++i)
      for (int j = 0; j < m; ++j) Q[i * m + j] = (N2[i * m + j] + N2[j * m + i]) / 2;
  }
}

/* assemble the n*n augmented A~ = [Phi 0; Phibar I] and Q~ of Eq. 3.17 from the blocks:
 *   A~[z_i, x_b] = Phibar_b  if b in instrument i's integrand;
 *   Q~[x_b, z_i] = Q12_b if b in i;  Q~[z_i, z_j] = sum_{b in i and j} Q22_b. */
static void disc_model(const model *M, real dt, real *A, real *Q) {
  int n = M->n, d = M->d;
  memset(A, 0, sizeof(real) * n * n);
  memset(Q, 0, sizeof(real) * n * n);
  for (int q = 0; q < M->ninst; ++q) A[(d + q) * n + d + q] = 1;
  for (int b = 0; b < M->nblk; ++b) {
    const block *B = &M->blk[b];
    int db = B->d, m = db + 1, o = M->off[b];
    real Ph[MB * MB], Qb[MB * MB];
    disc_block(B, dt, Ph, Qb);
    for (int i = 0; i < db; ++i)
      for (int j = 0; j < db; ++j) {
        A[(o + i) * n + o + j] = Ph[i * m + j];
        Q[(o + i) * n + o + j] = Qb[i * m + j];
      }
    for (int q = 0; q < M->ninst; ++q) {
      if (!((B->mask >> q) & 1u)) continue;
      for (int j = 0; j < db; ++j) {
        A[(d + q) * n + o + j] = Ph[db * m + j];
        Q[(d + q) * n + o + j] = Q[(o + j) * n + d + q] = Qb[db * m + j];
      }
      for (int r = 0; r < M->ninst; ++r)
        if ((B->mask >> r) & 1u) Q[(d + q) * n + d + r] += Qb[db * m + db];
    }
  }
}

int oracle_discretise(int ncomp, const ocomp *comp, int ninst, double dt, double *A, double *Q) {
  model M;
  if (build_model(&M, ncomp, comp, ninst)) return -1;
  real Ar[MAXN * MAXN], Qr[MAXN * MAXN];
  disc_model(&M, dt, Ar, Qr);
  for (int i = 0; i < M.n * M.n; ++i) { A[i] = (double)Ar[i]; Q[i] = (double)Qr[i]; }
  return 0;
}

/* ==========================================================================================
 * Part 4.  Small dense helpers (n <= MAXN), row-major, leading dimension n
 * ========================================================================================== */
static void mm(int n, const real *A, const real *B, real *C) { /* C = A B */
  for (int i = 0; i < n; ++i)
    for (int j = 0; j < n; ++j) {
      real s = 0;
      for (int k = 0; k < n; ++k) s += A[i * n + k] * B[k * n + j];
      C[i * n + j] = s;
    }
}
static void mmt(int n, const real *A, const real *B, real *C) { /* C = A B^T */
  for (int i = 0; i < n; ++i)
    for (int j = 0; j < n; ++j) {
      real s = 0;
      for (int k = 0; k < n; ++k) s += A[i * n + k] * B[j * n + k];
      C[i * n + j] = s;
    }
}
static void mtm(int n, const real *A, const real *B, real *C) { /* C = A^T B */
  for (int i = 0; i < n; ++i)
    for (int j = 0; j < n; ++j) {
      real s = 0;
      for (int k = 0; k < n; ++k) s += A[k * n + i] * B[k * n + j];
      C[i * n + j] = s;
    }
}
static void mv(int n, const real *A, const real *x, real *y) {
  for (int i = 0; i < n; ++i) {
    real s = 0;
    for (int k = 0; k < n; ++k) s += A[i * n + k] * x[k];
    y[i] = s;
  }
}
static void mtv(int n, const real *A, const real *x, real *y) { /* y = A^T x */
  for (int i = 0; i < n; ++i) {
    real s = 0;
    for (int k = 0; k < n; ++k) s += A[k * n + i] * x[k];
    y[i] = s;
  }
}
static void symmetrise(int n, real *A) {
  for (int i = 0; i < n; ++i)
    for (int j = 0; j < i; ++j) A[i * n + j] = A[j * n + i] = (A[i * n + j] + A[j * n + i]) / 2;
}
/* solve A X = B (n*n, nrhs columns) by LU with partial pivoting; A, B overwritten; X in B.
 * B is n * ldb row-major. Returns -1 if a pivot is exactly zero. */
static int lu_solve(int n, real *A, real *B, int nrhs) {
  for (int k = 0; k < n; ++k) {
    int p = k;
    real best = R_FABS(A[k * n + k]);
    for (int i = k + 1; i < n; ++i)
      if (R_FABS(A[i * n + k]) > best) { best = R_FABS(A[i * n + k]); p = i; }
    if (best == 0) return -1;
    if (p != k) {
      for (int j = 0; j < n; ++j) { real t = A[k * n + j]; A[k * n + j] = A[p * n + j]; A[p * n + j] = t; }
      for (int j = 0; j < nrhs; ++j) { real t = B[k * nrhs + j]; B[k * nrhs + j] = B[p * nrhs + j]; B[p * nrhs + j] = t; }
    }
    for (int i = k + 1; i < n; ++i) {
      real f = A[i * n + k] / A[k * n + k];
      if (f == 0) continue;
      for (int j = k; j < n; ++j) A[i * n + j] -= f * A[k * n + j];
      for (int j = 0; j < nrhs; ++j) B[i * nrhs + j] -= f * B[k * nrhs + j];
    }
  }
  for (int i = n - 1; i >= 0; --i)
    for (int j = 0; j < nrhs; ++j) {
      real s = B[i * nrhs + j];
      for (int k = i + 1; k < n; ++k) s -= A[i * n + k] * B[k * nrhs + j];
      B[i * nrhs + j] = s / A[i * n + i];
    }
  return 0;
}

/* ==========================================================================================
 * Part 5.  Events and the sequential integrated Kalman / RTS passes
 * ========================================================================================== */
typedef struct {
  double t;
  int kind; /* 0 = exposure end (observe), 1 = exposure start (reset): ends sort first (R5) */
  int inst, idx;
} event;
static int ev_cmp(const void *a, const void *b) {
  const event *x = a, *y = b;
  if (x->t != y->t) return x->t < y->t ? -1 : 1;
  if (x->kind != y->kind) return x->kind - y->kind;
  if (x->inst != y->inst) return x->inst - y->inst;
  return x->idx - y->idx;
}

/* sorted event table for callers that want to inspect it (tests of the CUDA event build) */
int oracle_events(int N, const double *ts, const double *te, const int32_t *inst, double *t_out,
                  int32_t *kind_out, int32_t *inst_out, int32_t *idx_out) {
  event *ev = malloc(sizeof(event) * 2 * (size_t)N);
  if (!ev) return -4;
  for (int i = 0; i < N; ++i) {
    ev[2 * i] = (event){ts[i], 1, inst[i], i};
    ev[2 * i + 1] = (event){te[i], 0, inst[i], i};
  }
  qsort(ev, 2 * (size_t)N, sizeof(event), ev_cmp);
  for (int k = 0; k < 2 * N; ++k) {
    t_out[k] = ev[k].t; kind_out[k] = ev[k].kind; inst_out[k] = ev[k].inst; idx_out[k] = ev[k].idx;
  }
  free(ev);
  return 0;
}

#define FLAG_IDLE_ZERO 1  /* also zero z_i at every event after which instrument i is idle (R6) */
#define FLAG_TWO_FILTER 2 /* backward pass in two-filter (information) form instead of RTS (R7) */

/* Instrumentation for bench.py's cpu_baseline split (discretisation and filter/smoother
 * time reported separately); no arithmetic.  Seconds spent inside disc_model during the last
 * oracle_ssm call made by the calling thread. */
static __thread double g_disc_seconds;
static double now_seconds(void) {
  struct timespec ts;
  clock_gettime(CLOCK_MONOTONIC, &ts);
  return (double)ts.tv_sec + 1e-9 * (double)ts.tv_nsec;
}
static void disc_model_timed(const model *M, real dt, real *A, real *Q) {
  double t0 = now_seconds();
  disc_model(M, dt, A, Q);
  g_disc_seconds += now_seconds() - t0;
}
double oracle_ssm_disc_seconds(void) { return g_disc_seconds; }

/* zero entry j of a mean and row+column j of a covariance: the reset R_i of Eq. 3.18 */
static void zero_state(int n, real *m, real *P, int j) {
  m[j] = 0;
  for (int i = 0; i < n; ++i) P[j * n + i] = P[i * n + j] = 0;
}

/* Sequential oracle.  y, sigma, ts, te, inst: exposure order as given.  Outputs in exposure
 * order.  zprior: value on the z-diagonal of P0 (Eq. 3.19 P:488 uses 1; results must not
 * depend on it).  Queries: instantaneous latent of instrument query_inst at tq[M]
 * (Algorithm 1, readings R8/R9).  Returns 0; -1 bad input; -2 same-instrument
 * overlap; -3 singular matrix met in a gain; -4 out of memory. */
int oracle_ssm(int ncomp, const ocomp *comp, int ninst, int N, const double *ts,
               const double *te, const int32_t *inst, const double *y, const double *sigma,
               int flags, double zprior, int M, const double *tq, int query_inst,
               double *loglik, double *mean, double *var, double *mq, double *vq) {
  model Md;
  g_disc_seconds = 0;
  if (build_model(&Md, ncomp, comp, ninst)) return -1;
  const int n = Md.n, d = Md.d, nn = n * n, K = 2 * N;
  const int want_smooth = (mean || var || M > 0);
  const int rts = !(flags & FLAG_TWO_FILTER);
  event *ev = malloc(sizeof(event) * (size_t)K);
  unsigned char *opst = malloc((size_t)K * ninst); /* instrument i exposing after event k? */
  if (!ev || !opst) { free(ev); free(opst); return -4; }
  for (int i = 0; i < N; ++i) {
    if (!(te[i] > ts[i]) || inst[i] < 0 || inst[i] >= ninst || !(sigma[i] > 0)) { free(ev); free(opst); return -1; }
    ev[2 * i] = (event){ts[i], 1, inst[i], i};
    ev[2 * i + 1] = (event){te[i], 0, inst[i], i};
  }
  qsort(ev, (size_t)K, sizeof(event), ev_cmp);
  { /* an instrument must not overlap itself: its events must alternate start, end */
    int open[MAXINST] = {0};
    for (int k = 0; k < K; ++k) {
      int i = ev[k].inst;
      if (ev[k].kind == open[i]) { free(ev); free(opst); return -2; }
      open[i] = ev[k].kind;
      for (int q = 0; q < ninst; ++q) opst[(size_t)k * ninst + q] = (unsigned char)open[q];
    }
  }
  /* stored per event: X_k = the state the smoother refines (filtered state at an end, pre-reset
   * predicted state at a start); predicted state (RTS only); smoothed state.  */
  size_t per = (size_t)n + nn;
  size_t n_ms = (M > 0) ? (size_t)K : 2;
  real *mx = want_smooth ? malloc(sizeof(real) * per * K) : NULL;
  real *mp = (want_smooth && rts) ? malloc(sizeof(real) * per * K) : NULL;
  real *ms = want_smooth ? malloc(sizeof(real) * per * n_ms) : NULL;
  if (want_smooth && (!mx || !ms || (rts && !mp))) { free(ev); free(opst); free(mx); free(mp); free(ms); return -4; }
#define MX(k) (mx + per * (size_t)(k))
#define PX_(k) (mx + per * (size_t)(k) + n)
#define MP(k) (mp + per * (size_t)(k))
#define PP(k) (mp + per * (size_t)(k) + n)
#define MS(k) (ms + per * ((size_t)(k) % n_ms))
#define PS(k) (ms + per * ((size_t)(k) % n_ms) + n)
  real m[MAXN] = {0}, P[MAXN * MAXN] = {0}, A[MAXN * MAXN], Q[MAXN * MAXN], T1[MAXN * MAXN], T2[MAXN * MAXN];
  /* init: m0 = 0, P0 = blkdiag(Pinf, zprior I) at the first event's time (Eq. 3.19) */
  for (int b = 0; b < Md.nblk; ++b)
    for (int i = 0; i < Md.blk[b].d; ++i)
      for (int j = 0; j < Md.blk[b].d; ++j)
        P[(Md.off[b] + i) * n + Md.off[b] + j] = Md.blk[b].P[i * Md.blk[b].d + j];
  for (int q = 0; q < ninst; ++q) P[(d + q) * n + d + q] = zprior;
  real ll = 0;
  /* ------------------------------ forward: integrated Kalman filter ---------------------- */
  for (int k = 0; k < K; ++k) {
    real dt = k == 0 ? 0 : (real)ev[k].t - (real)ev[k - 1].t;
    disc_model_timed(&Md, dt, A, Q);
    /* predict, Eq. 3.14 */
    mv(n, A, m, T1);
    memcpy(m, T1, sizeof(real) * n);
    mm(n, A, P, T1);
    mmt(n, T1, A, T2);
    for (int i = 0; i < nn; ++i) P[i] = T2[i] + Q[i];
    symmetrise(n, P);
    if (mp) { memcpy(MP(k), m, sizeof(real) * n); memcpy(PP(k), P, sizeof(real) * nn); }
    int zi = d + ev[k].inst;
    if (ev[k].kind == 1) { /* start: X_k = predicted; then m = R m-, P = R P- R^T, Eq. 3.15 */
      if (mx) { memcpy(MX(k), m, sizeof(real) * n); memcpy(PX_(k), P, sizeof(real) * nn); }
      zero_state(n, m, P, zi);
    } else { /* end: update with H~ = e_z / delta, Eq. 2.22, 3.12 */
      int e = ev[k].idx;
      real delta = (real)te[e] - (real)ts[e];
      real v = (real)y[e] - m[zi] / delta;
      real S = P[zi * n + zi] / (delta * delta) + (real)sigma[e] * (real)sigma[e];
      real Kg[MAXN];
      for (int i = 0; i < n; ++i) Kg[i] = P[i * n + zi] / delta / S;
      for (int i = 0; i < n; ++i) m[i] += Kg[i] * v;
      for (int i = 0; i < n; ++i)
        for (int j = 0; j < n; ++j) P[i * n + j] -= Kg[i] * S * Kg[j];
      symmetrise(n, P);
      ll += -(R_LOG(2 * (real)PI_R * S) + v * v / S) / 2; /* Eq. 2.26 */
      if (mx) { memcpy(MX(k), m, sizeof(real) * n); memcpy(PX_(k), P, sizeof(real) * nn); }
    }
    if (flags & FLAG_IDLE_ZERO)
      for (int q = 0; q < ninst; ++q)
        if (!opst[(size_t)k * ninst + q]) zero_state(n, m, P, d + q);
  }
  if (loglik) *loglik = (double)ll;

  int rc = 0;
  /* ------------------------------ backward ------------------------------------------------ */
  if (want_smooth && rts) {
    /* textbook integrated RTS, Eq. 2.23 and 3.16:
     *   G_k = P_X T_k^T [P-_{k+1}]^-1,  T_k = A~_k R  (R = the zeroing applied after event k),
     * where A~_k is the step from t_k to t_{k+1} (paper's indexing, Eq. 2.18). */
    memcpy(MS(K - 1), MX(K - 1), sizeof(real) * per); /* last event is an end: P:231 */
    for (int k = K - 2; k >= 0; --k) {
      real dt = (real)ev[k + 1].t - (real)ev[k].t;
      disc_model_timed(&Md, dt, A, Q);
      real Tm[MAXN * MAXN];
      memcpy(Tm, A, sizeof(real) * nn);
      for (int j = d; j < n; ++j) {
        int zeroed = (ev[k].kind == 1 && j == d + ev[k].inst) ||
                     ((flags & FLAG_IDLE_ZERO) && !opst[(size_t)k * ninst + (j - d)]);
        if (zeroed) for (int i = 0; i < n; ++i) Tm[i * n + j] = 0;
      }
      real Pm[MAXN * MAXN], Gt[MAXN * MAXN], G[MAXN * MAXN], D[MAXN * MAXN], dm[MAXN];
      memcpy(Pm, PP(k + 1), sizeof(real) * nn);
      mm(n, Tm, PX_(k), Gt); /* G^T = (P-_{k+1})^-1 T P_X */
      if (lu_solve(n, Pm, Gt, n)) { rc = -3; break; }
      for (int i = 0; i < n; ++i)
        for (int j = 0; j < n; ++j) G[i * n + j] = Gt[j * n + i];
      for (int i = 0; i < n; ++i) dm[i] = MS(k + 1)[i] - MP(k + 1)[i];
      for (int i = 0; i < nn; ++i) D[i] = PS(k + 1)[i] - PP(k + 1)[i];
      mv(n, G, dm, T1);
      for (int i = 0; i < n; ++i) MS(k)[i] = MX(k)[i] + T1[i];
      mm(n, G, D, T1);
      mmt(n, T1, G, T2);
      for (int i = 0; i < nn; ++i) PS(k)[i] = PX_(k)[i] + T2[i];
      symmetrise(n, PS(k));
      if (ev[k].kind == 0) {
        int e = ev[k].idx, zi = d + ev[k].inst;
        real delta = (real)te[e] - (real)ts[e];
        if (mean) mean[e] = (double)(MS(k)[zi] / delta);
        if (var) var[e] = (double)(PS(k)[zi * n + zi] / (delta * delta));
      }
    }
    if (rc == 0) { /* the last event's own output: H~ m^, H~ P^ H~^T */
      int k = K - 1, e = ev[k].idx, zi = d + ev[k].inst;
      real delta = (real)te[e] - (real)ts[e];
      if (mean) mean[e] = (double)(MX(k)[zi] / delta);
      if (var) var[e] = (double)(PX_(k)[zi * n + zi] / (delta * delta));
    }
  } else if (want_smooth) {
    /* two-filter form: (eta, J) = information about the state carried forward after event k
     * that all later data hold, p(y_{>k} | x) ~ exp(-x^T J x / 2 + eta^T x); combined with X_k:
     *   P^ = (I + P J)^-1 P,   m^ = (I + P J)^-1 (m + P eta)     (SG21's (eta, J); Fraser-Potter).
     * Going back over event k and then the step into it:  entries the forward pass zeroed carry
     * no information;  an end adds h h^T / r and h y / r (h = e_z / delta);
     *   J <- A^T (I + J Q)^-1 J A,   eta <- A^T (I + J Q)^-1 eta. */
    real J[MAXN * MAXN] = {0}, eta[MAXN] = {0};
    for (int k = K - 1; k >= 0; --k) {
      int zi = d + ev[k].inst;
      if (ev[k].kind == 1) zero_state(n, eta, J, zi);
      if (flags & FLAG_IDLE_ZERO)
        for (int q = 0; q < ninst; ++q)
          if (!opst[(size_t)k * ninst + q]) zero_state(n, eta, J, d + q);
      real Tm[MAXN * MAXN], R[MAXN * (MAXN + 1)], pe[MAXN];
      mm(n, PX_(k), J, Tm);
      for (int i = 0; i < n; ++i) Tm[i * n + i] += 1;
      mv(n, PX_(k), eta, pe);
      for (int i = 0; i < n; ++i) {
        for (int j = 0; j < n; ++j) R[i * (n + 1) + j] = PX_(k)[i * n + j];
        R[i * (n + 1) + n] = MX(k)[i] + pe[i];
      }
      if (lu_solve(n, Tm, R, n + 1)) { rc = -3; break; }
      for (int i = 0; i < n; ++i) {
        for (int j = 0; j < n; ++j) PS(k)[i * n + j] = R[i * (n + 1) + j];
        MS(k)[i] = R[i * (n + 1) + n];
      }
      symmetrise(n, PS(k));
      if (ev[k].kind == 0) {
        int e = ev[k].idx;
        real delta = (real)te[e] - (real)ts[e], r = (real)sigma[e] * (real)sigma[e];
        if (mean) mean[e] = (double)(MS(k)[zi] / delta);
        if (var) var[e] = (double)(PS(k)[zi * n + zi] / (delta * delta));
        J[zi * n + zi] += 1 / (delta * delta * r);
        eta[zi] += (real)y[e] / (delta * r);
      }
      real dt = k == 0 ? 0 : (real)ev[k].t - (real)ev[k - 1].t;
      disc_model_timed(&Md, dt, A, Q);
      real JA[MAXN * (MAXN + 1)], e2[MAXN];
      mm(n, J, Q, Tm);
      for (int i = 0; i < n; ++i) Tm[i * n + i] += 1;
      mm(n, J, A, T1);
      for (int i = 0; i < n; ++i) {
        for (int j = 0; j < n; ++j) JA[i * (n + 1) + j] = T1[i * n + j];
        JA[i * (n + 1) + n] = eta[i];
      }
      if (lu_solve(n, Tm, JA, n + 1)) { rc = -3; break; }
      for (int i = 0; i < n; ++i) {
        for (int j = 0; j < n; ++j) T1[i * n + j] = JA[i * (n + 1) + j];
        e2[i] = JA[i * (n + 1) + n];
      }
      mtm(n, A, T1, J);
      symmetrise(n, J);
      mtv(n, A, e2, eta);
    }
  }
  /* ------------------------------ Algorithm 1 -------------------------------- */
  if (rc == 0 && M > 0) {
    /* readings R8 (missing G^T on lines 9/20, "P_0"/"P_1^-" typos on line 18) and R9
     * (retrodiction on the x-block only).  Output H_q x, H_q = integrand row of query_inst. */
    real Hq[MAXN] = {0}, Pinf[MAXN * MAXN] = {0};
    for (int b = 0; b < Md.nblk; ++b) {
      if ((Md.blk[b].mask >> query_inst) & 1u)
        for (int j = 0; j < Md.blk[b].d; ++j) Hq[Md.off[b] + j] = Md.blk[b].H[j];
      for (int i = 0; i < Md.blk[b].d; ++i)
        for (int j = 0; j < Md.blk[b].d; ++j)
          Pinf[(Md.off[b] + i) * n + Md.off[b] + j] = Md.blk[b].P[i * Md.blk[b].d + j];
    }
    for (int q = 0; q < M && rc == 0; ++q) {
      real ms_[MAXN], Ps_[MAXN * MAXN], Gt[MAXN * MAXN], G[MAXN * MAXN], dm[MAXN], D[MAXN * MAXN];
      double t = tq[q];
      if (t < ev[0].t) { /* lines 3-9, on the x-block: m* = 0, P* = Pinf, P_1^- = Pinf */
        disc_model_timed(&Md, (real)ev[0].t - (real)t, A, Q);
        real Ax[MAXN * MAXN] = {0}, Ppred[MAXN * MAXN];
        for (int i = 0; i < d; ++i)
          for (int j = 0; j < d; ++j) Ax[i * n + j] = A[i * n + j];
        memcpy(Ppred, Pinf, sizeof(Ppred));
        for (int i = d; i < n; ++i) Ppred[i * n + i] = 1; /* keep the embedded system regular */
        mm(n, Ax, Pinf, Gt);                              /* G0^T = Pinf^-1 Phi Pinf */
        if (lu_solve(n, Ppred, Gt, n)) { rc = -3; break; }
        for (int i = 0; i < n; ++i)
          for (int j = 0; j < n; ++j) G[i * n + j] = Gt[j * n + i];
        memset(dm, 0, sizeof(dm));
        memset(D, 0, sizeof(D));
        for (int i = 0; i < d; ++i) dm[i] = MS(0)[i];
        for (int i = 0; i < d; ++i)
          for (int j = 0; j < d; ++j) D[i * n + j] = PS(0)[i * n + j] - Pinf[i * n + j];
        mv(n, G, dm, ms_);
        mm(n, G, D, T1);
        mmt(n, T1, G, T2);
        for (int i = 0; i < nn; ++i) Ps_[i] = Pinf[i] + T2[i];
      } else {
        int kp; /* last event with t_k <= t */
        if (t >= ev[K - 1].t) kp = K - 1;
        else {
          int lo = 0, hi = K - 1;
          while (hi - lo > 1) { int mid = (lo + hi) / 2; if (ev[mid].t <= t) lo = mid; else hi = mid; }
          kp = lo;
        }
        /* filtered state carried forward from kp: X_kp with the forward pass's zeroing */
        real mc[MAXN], Pc[MAXN * MAXN], mstar[MAXN], Pstar[MAXN * MAXN];
        memcpy(mc, MX(kp), sizeof(real) * n);
        memcpy(Pc, PX_(kp), sizeof(real) * nn);
        if (ev[kp].kind == 1) zero_state(n, mc, Pc, d + ev[kp].inst);
        if (flags & FLAG_IDLE_ZERO)
          for (int qq = 0; qq < ninst; ++qq)
            if (!opst[(size_t)kp * ninst + qq]) zero_state(n, mc, Pc, d + qq);
        disc_model_timed(&Md, (real)t - (real)ev[kp].t, A, Q); /* lines 14-18 / 23-27 */
        mv(n, A, mc, mstar);
        mm(n, A, Pc, T1);
        mmt(n, T1, A, T2);
        for (int i = 0; i < nn; ++i) Pstar[i] = T2[i] + Q[i];
        if (kp == K - 1) { /* extrapolate */
          memcpy(ms_, mstar, sizeof(real) * n);
          memcpy(Ps_, Pstar, sizeof(real) * nn);
        } else { /* interpolate: one smoothing step from the next state's (smoothed, predicted) */
          int kn = kp + 1;
          real Ppn[MAXN * MAXN], mpn[MAXN], Pm[MAXN * MAXN];
          disc_model_timed(&Md, (real)ev[kn].t - (real)t, A, Q);
          mv(n, A, mstar, mpn);
          mm(n, A, Pstar, T1);
          mmt(n, T1, A, T2);
          for (int i = 0; i < nn; ++i) Ppn[i] = T2[i] + Q[i];
          mm(n, A, Pstar, Gt); /* G*^T = (P-_next)^-1 A_next P* */
          memcpy(Pm, Ppn, sizeof(real) * nn);
          if (lu_solve(n, Pm, Gt, n)) { rc = -3; break; }
          for (int i = 0; i < n; ++i)
            for (int j = 0; j < n; ++j) G[i * n + j] = Gt[j * n + i];
          /* MS(kn) is the smoothed X_kn: at a start that is the pre-reset pair (R8) */
          for (int i = 0; i < n; ++i) dm[i] = MS(kn)[i] - mpn[i];
          for (int i = 0; i < nn; ++i) D[i] = PS(kn)[i] - Ppn[i];
          mv(n, G, dm, T1);
          for (int i = 0; i < n; ++i) ms_[i] = mstar[i] + T1[i];
          mm(n, G, D, T1);
          mmt(n, T1, G, T2);
          for (int i = 0; i < nn; ++i) Ps_[i] = Pstar[i] + T2[i];
        }
      }
      real mu = 0, vv = 0;
      for (int i = 0; i < n; ++i) {
        mu += Hq[i] * ms_[i];
        for (int j = 0; j < n; ++j) vv += Hq[i] * Ps_[i * n + j] * Hq[j];
      }
      if (mq) mq[q] = (double)mu;
      if (vq) vq[q] = (double)vv;
    }
  }
  free(ev); free(opst); free(mx); free(mp); free(ms);
  return rc;
}

/* ==========================================================================================
 * Part 6.  Instantaneous data (the paper's section 2: K = N states, no integral state).
 *   oracle_dense_instant : the definition, Eq. 2.4 with K_ij = k(|t_i - t_j|) restricted to the
 *                          components shared by the two samples' instruments; loglik as Eq. 2.26.
 *   oracle_ssm_instant   : the sequential algorithm of section 2, step by step: Kalman filter Eq. 2.21-2.22
 *                          (P:212-225), RTS smoother Eq. 2.23, log-likelihood Eq. 2.24-2.26
 *                          (P:246-260), prediction at arbitrary times Algorithm 1 in its printed,
 *                          non-augmented form.  State = the base state x (dimension d), H = the integrand row
 *                          H_i of the sample's instrument.
 * Pins (tests/test_oracle_instant_pins.py): dense_instant <- numpy on the pinned oracle_kernel; ssm_instant <-
 * dense_instant on tiny N (Fig. 1's claim: SSM = GP on instantaneous data to machine precision); the
 * exposure-integrated oracle with delta -> 0 converges to it with second order.
 * ========================================================================================== */
int oracle_dense_instant(int ncomp, const ocomp *comp, int N, const double *tt, const int32_t *inst,
                         const double *y, const double *sigma, int M, const double *tq, int query_inst,
                         double *loglik, double *mean, double *var, double *mq, double *vq) {
  kterm t[64];
  int nt = build_terms(ncomp, comp, t, 64);
  if (nt < 0) return -1;
  size_t NN = (size_t)N * N;
  real *K = malloc(NN * sizeof(real)), *L = malloc(NN * sizeof(real));
  real *a = malloc(N * sizeof(real)), *col = malloc(N * sizeof(real));
  if (!K || !L || !a || !col) return -4;
  for (int i = 0; i < N; ++i)
    for (int j = 0; j <= i; ++j) {
      real v = (real)kern_q(t, nt, inst[i], inst[j], (__float128)tt[i] - (__float128)tt[j]);
      K[(size_t)i * N + j] = K[(size_t)j * N + i] = v;
    }
  memcpy(L, K, NN * sizeof(real));
  for (int i = 0; i < N; ++i) L[(size_t)i * N + i] += (real)sigma[i] * (real)sigma[i];
  if (chol_lower(L, N)) { free(K); free(L); free(a); free(col); return -2; }
  for (int i = 0; i < N; ++i) a[i] = y[i];
  fwd_sub(L, N, a);
  real quad = 0, logdet = 0;
  for (int i = 0; i < N; ++i) { quad += a[i] * a[i]; logdet += 2 * R_LOG(L[(size_t)i * N + i]); }
  if (loglik) *loglik = (double)(-0.5L * (quad + logdet + N * R_LOG((real)(2 * PI_R))));
  bwd_sub(L, N, a);
  if (mean)
    for (int i = 0; i < N; ++i) {
      real s = 0;
      for (int j = 0; j < N; ++j) s += K[(size_t)i * N + j] * a[j];
      mean[i] = (double)s;
    }
  if (var)
    for (int i = 0; i < N; ++i) {
      for (int j = 0; j < N; ++j) col[j] = K[(size_t)j * N + i];
      fwd_sub(L, N, col);
      real s = 0;
      for (int j = 0; j < N; ++j) s += col[j] * col[j];
      var[i] = (double)(K[(size_t)i * N + i] - s);
    }
  for (int q = 0; q < M; ++q) {
    for (int j = 0; j < N; ++j) col[j] = (real)kern_q(t, nt, query_inst, inst[j], (__float128)tq[q] - (__float128)tt[j]);
    real s = 0;
    for (int j = 0; j < N; ++j) s += col[j] * a[j];
    if (mq) mq[q] = (double)s;
    fwd_sub(L, N, col);
    real v = (real)kern_q(t, nt, query_inst, query_inst, 0);
    for (int j = 0; j < N; ++j) v -= col[j] * col[j];
    if (vq) vq[q] = (double)v;
  }
  free(K); free(L); free(a); free(col);
  return 0;
}

/* base transition Phi (d x d) and process noise Q (d x d) of one step: the x-block of the augmented pair */
static void disc_base(const model *M, real dt, real *Phi, real *Q) {
  real A[MAXN * MAXN], Qa[MAXN * MAXN];
  disc_model(M, dt, A, Qa);
  const int n = M->n, d = M->d;
  for (int i = 0; i < d; ++i)
    for (int j = 0; j < d; ++j) { Phi[i * d + j] = A[i * n + j]; Q[i * d + j] = Qa[i * n + j]; }
}

int oracle_ssm_instant(int ncomp, const ocomp *comp, int ninst, int N, const double *tt, const int32_t *inst,
                       const double *y, const double *sigma, int M, const double *tq, int query_inst,
                       double *loglik, double *mean, double *var, double *mq, double *vq) {
  model Md;
  if (build_model(&Md, ncomp, comp, ninst)) return -1;
  const int d = Md.d, dd = d * d;
  /* measurement rows: H_i = sum of the H_m of the components in instrument i's mask (Eq. 3.2's H_n; P:86 for one instrument) */
  real H[32][MAXN] = {{0}};
  for (int q = 0; q < 32; ++q)
    for (int b = 0; b < Md.nblk; ++b)
      if ((Md.blk[b].mask >> q) & 1u)
        for (int j = 0; j < Md.blk[b].d; ++j) H[q][Md.off[b] + j] = Md.blk[b].H[j];
  event *ev = malloc(sizeof(event) * (size_t)N);
  if (!ev) return -4;
  for (int i = 0; i < N; ++i) {
    if (inst[i] < 0 || inst[i] >= ninst || !(sigma[i] > 0)) { free(ev); return -1; }
    ev[i] = (event){tt[i], 0, inst[i], i};
  }
  qsort(ev, (size_t)N, sizeof(event), ev_cmp);
  const int want_smooth = (mean || var || M > 0);
  size_t per = (size_t)d + dd;
  real *pr = malloc(sizeof(real) * per * N), *fi = malloc(sizeof(real) * per * N), *sm = want_smooth ? malloc(sizeof(real) * per * N) : NULL;
  if (!pr || !fi || (want_smooth && !sm)) { free(ev); free(pr); free(fi); free(sm); return -4; }
#define IM(a, k) ((a) + per * (size_t)(k))
#define IP(a, k) ((a) + per * (size_t)(k) + d)
  real m[MAXN] = {0}, P[MAXN * MAXN] = {0}, Phi[MAXN * MAXN], Q[MAXN * MAXN], T1[MAXN * MAXN], T2[MAXN * MAXN], Pinf[MAXN * MAXN] = {0};
  for (int b = 0; b < Md.nblk; ++b)
    for (int i = 0; i < Md.blk[b].d; ++i)
      for (int j = 0; j < Md.blk[b].d; ++j) Pinf[(Md.off[b] + i) * d + Md.off[b] + j] = Md.blk[b].P[i * Md.blk[b].d + j];
  memcpy(P, Pinf, sizeof(real) * dd); /* m0 = 0, P0 = Pinf */
  real ll = 0;
  int rc = 0;
  for (int k = 0; k < N; ++k) {
    real dt = k == 0 ? 0 : (real)ev[k].t - (real)ev[k - 1].t;
    disc_base(&Md, dt, Phi, Q);
    mv(d, Phi, m, T1); /* predict, Eq. 2.21 */
    memcpy(m, T1, sizeof(real) * d);
    mm(d, Phi, P, T1);
    mmt(d, T1, Phi, T2);
    for (int i = 0; i < dd; ++i) P[i] = T2[i] + Q[i];
    symmetrise(d, P);
    memcpy(IM(pr, k), m, sizeof(real) * d); memcpy(IP(pr, k), P, sizeof(real) * dd);
    const real *h = H[ev[k].inst]; /* update, Eq. 2.22 */
    int e = ev[k].idx;
    real v = (real)y[e], S = (real)sigma[e] * (real)sigma[e], Ph[MAXN];
    for (int i = 0; i < d; ++i) v -= h[i] * m[i];
    for (int i = 0; i < d; ++i) { real s = 0; for (int j = 0; j < d; ++j) s += P[i * d + j] * h[j]; Ph[i] = s; }
    for (int i = 0; i < d; ++i) S += h[i] * Ph[i];
    for (int i = 0; i < d; ++i) m[i] += Ph[i] / S * v;
    for (int i = 0; i < d; ++i)
      for (int j = 0; j < d; ++j) P[i * d + j] -= Ph[i] * Ph[j] / S;
    symmetrise(d, P);
    ll += -(R_LOG(2 * (real)PI_R * S) + v * v / S) / 2; /* Eq. 2.26 */
    memcpy(IM(fi, k), m, sizeof(real) * d); memcpy(IP(fi, k), P, sizeof(real) * dd);
  }
  if (loglik) *loglik = (double)ll;
  if (want_smooth) { /* RTS, Eq. 2.23 */
    memcpy(IM(sm, N - 1), IM(fi, N - 1), sizeof(real) * per);
    for (int k = N - 2; k >= 0 && rc == 0; --k) {
      real dt = (real)ev[k + 1].t - (real)ev[k].t;
      disc_base(&Md, dt, Phi, Q);
      real Pm[MAXN * MAXN], Gt[MAXN * MAXN], G[MAXN * MAXN], D[MAXN * MAXN], dm[MAXN];
      memcpy(Pm, IP(pr, k + 1), sizeof(real) * dd);
      mm(d, Phi, IP(fi, k), Gt); /* G^T = (P-_{k+1})^-1 Phi P_k */
      if (lu_solve(d, Pm, Gt, d)) { rc = -3; break; }
      for (int i = 0; i < d; ++i)
        for (int j = 0; j < d; ++j) G[i * d + j] = Gt[j * d + i];
      for (int i = 0; i < d; ++i) dm[i] = IM(sm, k + 1)[i] - IM(pr, k + 1)[i];
      for (int i = 0; i < dd; ++i) D[i] = IP(sm, k + 1)[i] - IP(pr, k + 1)[i];
      mv(d, G, dm, T1);
      for (int i = 0; i < d; ++i) IM(sm, k)[i] = IM(fi, k)[i] + T1[i];
      mm(d, G, D, T1);
      mmt(d, T1, G, T2);
      for (int i = 0; i < dd; ++i) IP(sm, k)[i] = IP(fi, k)[i] + T2[i];
      symmetrise(d, IP(sm, k));
    }
    for (int k = 0; k < N && rc == 0; ++k) {
      const real *h = H[ev[k].inst];
      real mu = 0, vv = 0;
      for (int i = 0; i < d; ++i) { mu += h[i] * IM(sm, k)[i]; for (int j = 0; j < d; ++j) vv += h[i] * IP(sm, k)[i * d + j] * h[j]; }
      if (mean) mean[ev[k].idx] = (double)mu;
      if (var) var[ev[k].idx] = (double)vv;
    }
  }
  /* Algorithm 1 as printed, with the missing G^T of lines 9/20 restored (reading c7) */
  for (int q = 0; q < M && rc == 0; ++q) {
    const real *h = H[query_inst];
    real ms_[MAXN], Ps_[MAXN * MAXN], Gt[MAXN * MAXN], G[MAXN * MAXN], dm[MAXN], D[MAXN * MAXN], Pm[MAXN * MAXN];
    double t = tq[q];
    if (t < ev[0].t) { /* retrodict: m* = m0 = 0, P* = Pinf; next = state 1 predicted from t* */
      disc_base(&Md, (real)ev[0].t - (real)t, Phi, Q);
      mm(d, Phi, Pinf, T1);
      mmt(d, T1, Phi, T2);
      for (int i = 0; i < dd; ++i) Pm[i] = T2[i] + Q[i]; /* P-_1 seen from t* (= Pinf: the prior is stationary) */
      mm(d, Phi, Pinf, Gt);
      if (lu_solve(d, Pm, Gt, d)) { rc = -3; break; }
      for (int i = 0; i < d; ++i)
        for (int j = 0; j < d; ++j) G[i * d + j] = Gt[j * d + i];
      mm(d, Phi, Pinf, T1); mmt(d, T1, Phi, T2);
      for (int i = 0; i < d; ++i) dm[i] = IM(sm, 0)[i];
      for (int i = 0; i < dd; ++i) D[i] = IP(sm, 0)[i] - (T2[i] + Q[i]);
      mv(d, G, dm, ms_);
      mm(d, G, D, T1); mmt(d, T1, G, T2);
      for (int i = 0; i < dd; ++i) Ps_[i] = Pinf[i] + T2[i];
    } else {
      int kp;
      if (t >= ev[N - 1].t) kp = N - 1;
      else { int lo = 0, hi = N - 1; while (hi - lo > 1) { int mid = (lo + hi) / 2; if (ev[mid].t <= t) lo = mid; else hi = mid; } kp = lo; }
      real mstar[MAXN], Pstar[MAXN * MAXN];
      disc_base(&Md, (real)t - (real)ev[kp].t, Phi, Q);
      mv(d, Phi, IM(fi, kp), mstar);
      mm(d, Phi, IP(fi, kp), T1); mmt(d, T1, Phi, T2);
      for (int i = 0; i < dd; ++i) Pstar[i] = T2[i] + Q[i];
      if (kp == N - 1) { memcpy(ms_, mstar, sizeof(real) * d); memcpy(Ps_, Pstar, sizeof(real) * dd); }
      else {
        int kn = kp + 1;
        real mpn[MAXN];
        disc_base(&Md, (real)ev[kn].t - (real)t, Phi, Q);
        mv(d, Phi, mstar, mpn);
        mm(d, Phi, Pstar, T1); mmt(d, T1, Phi, T2);
        for (int i = 0; i < dd; ++i) Pm[i] = T2[i] + Q[i];
        real Ppn[MAXN * MAXN];
        memcpy(Ppn, Pm, sizeof(real) * dd);
        mm(d, Phi, Pstar, Gt);
        if (lu_solve(d, Pm, Gt, d)) { rc = -3; break; }
        for (int i = 0; i < d; ++i)
          for (int j = 0; j < d; ++j) G[i * d + j] = Gt[j * d + i];
        for (int i = 0; i < d; ++i) dm[i] = IM(sm, kn)[i] - mpn[i];
        for (int i = 0; i < dd; ++i) D[i] = IP(sm, kn)[i] - Ppn[i];
        mv(d, G, dm, T1);
        for (int i = 0; i < d; ++i) ms_[i] = mstar[i] + T1[i];
        mm(d, G, D, T1); mmt(d, T1, G, T2);
        for (int i = 0; i < dd; ++i) Ps_[i] = Pstar[i] + T2[i];
      }
    }
    real mu = 0, vv = 0;
    for (int i = 0; i < d; ++i) { mu += h[i] * ms_[i]; for (int j = 0; j < d; ++j) vv += h[i] * Ps_[i * d + j] * h[j]; }
    if (mq) mq[q] = (double)mu;
    if (vq) vq[q] = (double)vv;
  }
  free(ev); free(pr); free(fi); free(sm);
  return rc;
}

/* ==========================================================================================
 * Part 7.  Square-root (Cholesky-factor) form of the sequential passes.
 *
 * The paper names it as the remedy for the conditioning of the covariance recursions ("numerical
 * instabilities ... square-root"; Yaghoobi et al. 2025) and prints no algorithm:
 * what it must compute is the SAME posterior as Part 5 (and as the dense definition of Part 2), so
 * Parts 2 and 5 are its pins (tests/test_oracle_sqrt_pins.py).  Written here in the textbook ARRAY
 * form (Kailath, Sayed & Hassibi, "Linear Estimation", ch. 12): every covariance P is carried as a
 * factor S with P = S S^T, every information matrix J as Z with J = Z Z^T, and every step is
 * "stack the factors side by side, re-triangularise":  tria(M) = the lower-triangular L with
 * L L^T = M M^T.  No covariance is ever formed, nothing is subtracted, nothing ill-conditioned is
 * inverted.
 *   predict (Eq. 3.14)     S^- = tria([A S | G]),  G G^T = Q~  (G from the blocks' own
 *                                Cholesky factors -- Q~ itself is singular)
 *   reset (Eq. 3.15 / 3.18)      zero row z_i of S and m_zi
 *   update (Eq. 2.22)      tria([[sqrt r, h^T S^-], [0, S^-]]) = [[sqrt s, 0], [K sqrt s, S^+]]
 *   backward, two-filter form of Part 5 (reading R7) with J = Z Z^T:
 *     smoothed   P^ = S (I + S^T J S)^-1 S^T,  m^ = m + S (I + S^T J S)^-1 S^T (eta - J m)
 *     end event  Z <- tria([Z | h / sqrt r]),  eta += h y / r
 *     step       (J^-1 + Q)^-1 = Z (I + Z^T Q Z)^-1 Z^T:  T = tria([I | Z^T G]),  Z <- A^T Z T^-T,
 *                eta <- A^T (eta - Z (T T^T)^-1 Z^T Q eta)
 * ========================================================================================== */
#define MAXQ (MAXN + MAXBLK) /* columns of G: d + nblk */

/* L (n x n, lower, row-major) with L L^T = M M^T, M n x m row-major (destroyed): Householder reflections
 * applied from the right, one per row */
static void tria(int n, int m, real *M, real *L) {
  for (int j = 0; j < n; ++j) {
    real *rj = M + (size_t)j * m;
    real ss = 0;
    for (int c = j; c < m; ++c) ss += rj[c] * rj[c];
    real sig = R_SQRT(ss);
    if (sig > 0 && j < m) {
      /* reflector v = u - alpha e_j with alpha = -sign(u_j) |u|, used in the scale-free form v / |u| so that
       * rows of any magnitude (the information factors span hundreds of orders) neither overflow nor vanish */
      real alpha = rj[j] > 0 ? -sig : sig;
      real v0 = (rj[j] - alpha) / sig;
      real beta = 1 / (1 + R_FABS(rj[j]) / sig);
      for (int c = j + 1; c < m; ++c) rj[c] /= sig;
      for (int i = j + 1; i < n; ++i) {
        real *ri = M + (size_t)i * m;
        real dsum = ri[j] * v0;
        for (int c = j + 1; c < m; ++c) dsum += ri[c] * rj[c];
        real w = beta * dsum;
        ri[j] -= w * v0;
        for (int c = j + 1; c < m; ++c) ri[c] -= w * rj[c];
      }
      rj[j] = alpha;
      for (int c = j + 1; c < m; ++c) rj[c] = 0;
    }
  }
  for (int i = 0; i < n; ++i)
    for (int j = 0; j < n; ++j) L[i * n + j] = (j <= i && j < m) ? M[(size_t)i * m + j] : 0;
}

/* lower Cholesky factor of a positive SEMI-definite m x m matrix (row-major): a pivot that rounding
 * has driven to <= 0 (or below 2^-44 of its diagonal entry) gives a zero column */
static void chol_psd(int m, const real *A, real *L) {
  memset(L, 0, sizeof(real) * m * m);
  for (int j = 0; j < m; ++j) {
    real p = A[j * m + j];
    for (int k = 0; k < j; ++k) p -= L[j * m + k] * L[j * m + k];
    if (!(p > A[j * m + j] * (real)5.7e-14)) continue;
    real r = R_SQRT(p);
    L[j * m + j] = r;
    for (int i = j + 1; i < m; ++i) {
      real a = A[i * m + j];
      for (int k = 0; k < j; ++k) a -= L[i * m + k] * L[j * m + k];
      L[i * m + j] = a / r;
    }
  }
}

/* A~ (n x n) as disc_model, and G (n x nq, nq = d + nblk) with G G^T = Q~ of Eq. 3.17: block b's
 * augmented Q_b = [Qxx q12; q12^T q22] is factored on its own, L_b L_b^T = Q_b, and placed like Q_b itself:
 * x rows of the block in its own columns, the integral row into z_i for every instrument i that integrates it */
static void disc_model_factor(const model *M, real dt, real *A, real *G, int *nq_out) {
  int n = M->n, d = M->d, nq = d + M->nblk;
  memset(A, 0, sizeof(real) * n * n);
  memset(G, 0, sizeof(real) * n * nq);
  for (int q = 0; q < M->ninst; ++q) A[(d + q) * n + d + q] = 1;
  for (int b = 0; b < M->nblk; ++b) {
    const block *B = &M->blk[b];
    int db = B->d, m = db + 1, o = M->off[b], c0 = o + b; /* first column of block b in G */
    real Ph[MB * MB], Qb[MB * MB], Lb[MB * MB];
    disc_block(B, dt, Ph, Qb);
    chol_psd(m, Qb, Lb);
    for (int i = 0; i < db; ++i) {
      for (int j = 0; j < db; ++j) A[(o + i) * n + o + j] = Ph[i * m + j];
      for (int j = 0; j < m; ++j) G[(o + i) * nq + c0 + j] = Lb[i * m + j];
    }
    for (int q = 0; q < M->ninst; ++q) {
      if (!((B->mask >> q) & 1u)) continue;
      for (int j = 0; j < db; ++j) A[(d + q) * n + o + j] = Ph[db * m + j];
      for (int j = 0; j < m; ++j) G[(d + q) * nq + c0 + j] = Lb[db * m + j];
    }
  }
  *nq_out = nq;
}

/* solve L x = b in place (L lower n x n, zero pivots give x_i = 0: the direction carries nothing) */
static void lsolve(int n, const real *L, real *b) {
  for (int i = 0; i < n; ++i) {
    real a = b[i];
    for (int k = 0; k < i; ++k) a -= L[i * n + k] * b[k];
    b[i] = (L[i * n + i] != 0) ? a / L[i * n + i] : 0;
  }
}
static void ltsolve(int n, const real *L, real *b) { /* L^T x = b */
  for (int i = n - 1; i >= 0; --i) {
    real a = b[i];
    for (int k = i + 1; k < n; ++k) a -= L[k * n + i] * b[k];
    b[i] = (L[i * n + i] != 0) ? a / L[i * n + i] : 0;
  }
}

/* Same contract as oracle_ssm with flags = IDLE_ZERO | TWO_FILTER (readings R6, R7), no query times.
 * Returns 0; -1 bad input; -2 same-instrument overlap; -4 out of memory. */
int oracle_ssm_sqrt(int ncomp, const ocomp *comp, int ninst, int N, const double *ts, const double *te,
                    const int32_t *inst, const double *y, const double *sigma, double zprior,
                    double *loglik, double *mean, double *var) {
  model Md;
  if (build_model(&Md, ncomp, comp, ninst)) return -1;
  const int n = Md.n, d = Md.d, nn = n * n, K = 2 * N;
  const int want_smooth = (mean || var);
  event *ev = malloc(sizeof(event) * (size_t)K);
  unsigned char *opst = malloc((size_t)K * ninst);
  if (!ev || !opst) { free(ev); free(opst); return -4; }
  for (int i = 0; i < N; ++i) {
    if (!(te[i] > ts[i]) || inst[i] < 0 || inst[i] >= ninst || !(sigma[i] > 0)) { free(ev); free(opst); return -1; }
    ev[2 * i] = (event){ts[i], 1, inst[i], i};
    ev[2 * i + 1] = (event){te[i], 0, inst[i], i};
  }
  qsort(ev, (size_t)K, sizeof(event), ev_cmp);
  {
    int open[MAXINST] = {0};
    for (int k = 0; k < K; ++k) {
      int i = ev[k].inst;
      if (ev[k].kind == open[i]) { free(ev); free(opst); return -2; }
      open[i] = ev[k].kind;
      for (int q = 0; q < ninst; ++q) opst[(size_t)k * ninst + q] = (unsigned char)open[q];
    }
  }
  /* stored per END event (exposure index): the filtered factor and mean the smoother refines */
  size_t per = (size_t)n + nn;
  real *sx = want_smooth ? malloc(sizeof(real) * per * (size_t)N) : NULL;
  if (want_smooth && !sx) { free(ev); free(opst); return -4; }
  real m[MAXN] = {0}, S[MAXN * MAXN] = {0}, A[MAXN * MAXN], G[MAXN * MAXQ];
  static __thread real W[(MAXN + 1) * (2 * MAXN + MAXQ + 1)];
  for (int b = 0; b < Md.nblk; ++b) { /* S0 = blkdiag(chol Pinf_b, sqrt(zprior) I) */
    int db = Md.blk[b].d, o = Md.off[b];
    real Lb[MAXBD * MAXBD];
    chol_psd(db, Md.blk[b].P, Lb);
    for (int i = 0; i < db; ++i)
      for (int j = 0; j < db; ++j) S[(o + i) * n + o + j] = Lb[i * db + j];
  }
  for (int q = 0; q < ninst; ++q) S[(d + q) * n + d + q] = R_SQRT((real)zprior);
  real ll = 0;
  int nq = 0;
  for (int k = 0; k < K; ++k) {
    real dt = k == 0 ? 0 : (real)ev[k].t - (real)ev[k - 1].t;
    disc_model_factor(&Md, dt, A, G, &nq);
    { /* predict: m <- A m, S <- tria([A S | G]) */
      real t1[MAXN];
      mv(n, A, m, t1);
      memcpy(m, t1, sizeof(real) * n);
      int mc = n + nq;
      for (int i = 0; i < n; ++i) {
        for (int j = 0; j < n; ++j) {
          real a = 0;
          for (int l = 0; l < n; ++l) a += A[i * n + l] * S[l * n + j];
          W[i * mc + j] = a;
        }
        for (int j = 0; j < nq; ++j) W[i * mc + n + j] = G[i * nq + j];
      }
      tria(n, mc, W, S);
    }
    int zi = d + ev[k].inst;
    if (ev[k].kind == 1) { /* start: reset, Eq. 3.15 */
      m[zi] = 0;
      for (int j = 0; j < n; ++j) S[zi * n + j] = 0;
    } else { /* end: array update with h = e_z / delta */
      int e = ev[k].idx;
      real delta = (real)te[e] - (real)ts[e], sg = (real)sigma[e];
      int mc = n + 1;
      real Lw[(MAXN + 1) * (MAXN + 1)];
      memset(W, 0, sizeof(real) * (size_t)(n + 1) * mc);
      W[0] = sg;
      for (int j = 0; j < n; ++j) W[1 + j] = S[zi * n + j] / delta; /* h^T S */
      for (int i = 0; i < n; ++i)
        for (int j = 0; j < n; ++j) W[(size_t)(i + 1) * mc + 1 + j] = S[i * n + j];
      /* tria of the (n+1) x (n+1) pre-array, written into an (n+1)-square L */
      {
        real Mw[(MAXN + 1) * (MAXN + 1)];
        memcpy(Mw, W, sizeof(real) * (size_t)(n + 1) * mc);
        int n1 = n + 1;
        /* tria() is written for leading dimension = column count: here both are n + 1 */
        tria(n1, n1, Mw, Lw);
      }
      int n1 = n + 1;
      real rs = Lw[0]; /* +- sqrt(s) */
      real s = rs * rs;
      real v = (real)y[e] - m[zi] / delta;
      for (int i = 0; i < n; ++i) m[i] += Lw[(i + 1) * n1] / rs * v; /* K = Kbar / sqrt(s) */
      for (int i = 0; i < n; ++i)
        for (int j = 0; j < n; ++j) S[i * n + j] = Lw[(i + 1) * n1 + 1 + j];
      ll += -(R_LOG(2 * (real)PI_R * s) + v * v / s) / 2;
      if (sx) { memcpy(sx + per * (size_t)e, m, sizeof(real) * n); memcpy(sx + per * (size_t)e + n, S, sizeof(real) * nn); }
    }
    for (int q = 0; q < ninst; ++q)
      if (!opst[(size_t)k * ninst + q]) { m[d + q] = 0; for (int j = 0; j < n; ++j) S[(d + q) * n + j] = 0; }
  }
  if (loglik) *loglik = (double)ll;
  if (want_smooth) {
    real Z[MAXN * MAXN] = {0}, eta[MAXN] = {0};
    for (int k = K - 1; k >= 0; --k) {
      int zi = d + ev[k].inst;
      if (ev[k].kind == 1) { eta[zi] = 0; for (int j = 0; j < n; ++j) Z[zi * n + j] = 0; }
      for (int q = 0; q < ninst; ++q)
        if (!opst[(size_t)k * ninst + q]) { eta[d + q] = 0; for (int j = 0; j < n; ++j) Z[(d + q) * n + j] = 0; }
      if (ev[k].kind == 0) {
        int e = ev[k].idx;
        const real *mf = sx + per * (size_t)e, *Sf = mf + n;
        real delta = (real)te[e] - (real)ts[e], r = (real)sigma[e] * (real)sigma[e];
        /* U U^T = I + V V^T, V = S^T Z */
        real U[MAXN * MAXN];
        int mc = 2 * n;
        for (int i = 0; i < n; ++i)
          for (int j = 0; j < n; ++j) {
            real a = 0;
            for (int l = 0; l < n; ++l) a += Sf[l * n + i] * Z[l * n + j];
            W[i * mc + j] = (i == j) ? 1 : 0;
            W[i * mc + n + j] = a;
          }
        tria(n, mc, W, U);
        real w[MAXN], gvec[MAXN], zt[MAXN], u[MAXN];
        for (int j = 0; j < n; ++j) w[j] = Sf[zi * n + j]; /* S^T e_z */
        lsolve(n, U, w);
        mtv(n, Z, mf, zt); /* Z^T m */
        mv(n, Z, zt, gvec);
        for (int i = 0; i < n; ++i) gvec[i] = eta[i] - gvec[i]; /* eta - J m */
        mtv(n, Sf, gvec, u);
        lsolve(n, U, u);
        real vv = 0, mu = mf[zi];
        for (int j = 0; j < n; ++j) { vv += w[j] * w[j]; mu += w[j] * u[j]; }
        if (mean) mean[e] = (double)(mu / delta);
        if (var) var[e] = (double)(vv / (delta * delta));
        /* the exposure's own information: Z <- tria([Z | h / sqrt r]), eta += h y / r */
        mc = n + 1;
        for (int i = 0; i < n; ++i) {
          for (int j = 0; j < n; ++j) W[i * mc + j] = Z[i * n + j];
          W[i * mc + n] = (i == zi) ? 1 / (delta * R_SQRT(r)) : 0;
        }
        tria(n, mc, W, Z);
        eta[zi] += (real)y[e] / (delta * r);
      }
      real dt = k == 0 ? 0 : (real)ev[k].t - (real)ev[k - 1].t;
      disc_model_factor(&Md, dt, A, G, &nq);
      { /* T T^T = I + Y Y^T, Y = Z^T G;  Z <- A^T Z T^-T;  eta <- A^T (eta - Z (T T^T)^-1 Y G^T eta) */
        real T[MAXN * MAXN], Y[MAXN * MAXQ], ge[MAXQ], ye[MAXN], Zp[MAXN * MAXN];
        int mc = n + nq;
        for (int i = 0; i < n; ++i) {
          for (int j = 0; j < nq; ++j) {
            real a = 0;
            for (int l = 0; l < n; ++l) a += Z[l * n + i] * G[l * nq + j];
            Y[i * nq + j] = a;
          }
          for (int j = 0; j < n; ++j) W[i * mc + j] = (i == j) ? 1 : 0;
          for (int j = 0; j < nq; ++j) W[i * mc + n + j] = Y[i * nq + j];
        }
        tria(n, mc, W, T);
        for (int j = 0; j < nq; ++j) {
          real a = 0;
          for (int l = 0; l < n; ++l) a += G[l * nq + j] * eta[l];
          ge[j] = a;
        }
        for (int i = 0; i < n; ++i) {
          real a = 0;
          for (int j = 0; j < nq; ++j) a += Y[i * nq + j] * ge[j];
          ye[i] = a;
        }
        lsolve(n, T, ye);
        ltsolve(n, T, ye);
        real e2[MAXN];
        mv(n, Z, ye, e2);
        for (int i = 0; i < n; ++i) e2[i] = eta[i] - e2[i];
        /* rows of Z T^-T: for each row z of Z solve T x = z^T */
        for (int i = 0; i < n; ++i) {
          real x[MAXN];
          for (int j = 0; j < n; ++j) x[j] = Z[i * n + j];
          lsolve(n, T, x);
          for (int j = 0; j < n; ++j) Zp[i * n + j] = x[j];
        }
        mtm(n, A, Zp, Z);
        mtv(n, A, e2, eta);
      }
    }
  }
  free(ev); free(opst); free(sx);
  return 0;
}
