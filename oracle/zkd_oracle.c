/* oracle/zkd_oracle.c — TEST INFRASTRUCTURE ONLY.
 *
 * Plain, slow, obviously-correct CPU oracle for the hot path of arxiv 2402.11868:
 * "diagonalizing N x N Hermitian matrix with random elements. The 768-bit precision was used"
 * (section 2.1; the routine is diag_H / zkcm_omp::diag_H / zkcm_cus::cus_diag_H).
 * The paper gives no algorithm beyond one sentence on RQI; the GPU method reaches the
 * plain result "real ascending lambda, unitary X with A X = X diag(lambda)" by a faster route, so the
 * oracle is that definition computed by the textbook method BASELINE.json fixes: cyclic Jacobi on MPFR
 * (followed here in that order and notation).
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may call this.
 * It shares no code with paper_2402_11868_b200/ (the CUDA path) and does not include include/zkd.h:
 * the number layout is restated below from DESIGN.md section "API number layout".
 *
 * API real number (little-endian, 16 + prec/8 bytes; 112 bytes at 768 bit):
 *   int32 sign (-1, 0, +1); int32 flags (must be 0); int64 exp; uint64 limb[prec/64] (little-endian limbs)
 *   value = sign * (sum_k limb[k] 2^(64k)) * 2^(exp - prec); nonzero => top bit of limb[L-1] set
 *   (mantissa in [1/2,1), the MPFR convention); zero => all fields zero.
 * Complex = (re, im) consecutive.  Matrices row-major A[i][j]; eigvecs[i][j] = component i of vector j.
 *
 * Pins (tests/test_oracle_pins.py, -m "not gpu"): 2x2 closed form, Hermitian tridiagonal Toeplitz spectrum and
 * vectors, Q diag(lambda) Q^H with chosen lambda, trace / Frobenius identities, characteristic-polynomial
 * roots at N <= 4, the paper's epsilon = 2^-(n-1) example, degenerate cases, ordering and
 * guard-precision independence.  All pin values are computed in the tests with mpmath, not with this file.
 */
#include "mpfr_abi.h"

#include <math.h>
#include <omp.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#define RN MPFR_RNDN

/* ------------------------------------------------------------------------------------------------ */
/* number format                                                                                    */
/* ------------------------------------------------------------------------------------------------ */

static size_t api_real_bytes(int prec) { return 16 + (size_t)prec / 8; }

/* returns 0 ok, 3 malformed.  tmp must have precision exactly prec (a multiple of 64). */
static int api_get(mpfr_ptr dst, const uint8_t *src, int prec, mpfr_ptr tmp) {
  int32_t sign, flags;
  int64_t e;
  int L = prec / 64;
  memcpy(&sign, src, 4);
  memcpy(&flags, src + 4, 4);
  memcpy(&e, src + 8, 8);
  if (flags != 0 || sign < -1 || sign > 1) return 3;
  if (sign == 0) {
    mpfr_set_zero(dst, +1);
    return 0;
  }
  uint64_t top;
  memcpy(&top, src + 16 + 8 * (size_t)(L - 1), 8);
  if (!(top >> 63)) return 3;
  memcpy(tmp->_mpfr_d, src + 16, 8 * (size_t)L);
  tmp->_mpfr_sign = sign;
  tmp->_mpfr_exp = (mpfr_exp_t)e;
  mpfr_set(dst, tmp, RN); /* exact when prec(dst) >= prec */
  return 0;
}

/* rounds src to prec bits (RNDN) and writes the API layout. */
static void api_put(uint8_t *dst, mpfr_srcptr src, int prec, mpfr_ptr tmp) {
  int L = prec / 64;
  memset(dst, 0, api_real_bytes(prec));
  mpfr_set(tmp, src, RN);
  if (mpfr_zero_p(tmp)) return;
  int32_t sign = mpfr_sgn(tmp) < 0 ? -1 : 1;
  int64_t e = (int64_t)mpfr_get_exp(tmp);
  memcpy(dst, &sign, 4);
  memcpy(dst + 8, &e, 8);
  memcpy(dst + 16, tmp->_mpfr_d, 8 * (size_t)L);
}

/* ------------------------------------------------------------------------------------------------ */
/* small helpers on arrays of mpfr                                                                  */
/* ------------------------------------------------------------------------------------------------ */

static __mpfr_struct *vec_alloc(size_t n, long prec) {
  __mpfr_struct *v = (__mpfr_struct *)malloc(n * sizeof(__mpfr_struct));
  for (size_t i = 0; i < n; ++i) {
    mpfr_init2(&v[i], prec);
    mpfr_set_zero(&v[i], +1);
  }
  return v;
}
static void vec_free(__mpfr_struct *v, size_t n) {
  for (size_t i = 0; i < n; ++i) mpfr_clear(&v[i]);
  free(v);
}

/* complex matrix: re and im planes, row-major */
typedef struct {
  int n;
  __mpfr_struct *re, *im;
} cmat;
static cmat cmat_alloc(int n, long prec) {
  cmat m;
  m.n = n;
  m.re = vec_alloc((size_t)n * n, prec);
  m.im = vec_alloc((size_t)n * n, prec);
  return m;
}
static void cmat_free(cmat *m) {
  vec_free(m->re, (size_t)m->n * m->n);
  vec_free(m->im, (size_t)m->n * m->n);
}
#define RE(m, i, j) (&(m).re[(size_t)(i) * (m).n + (j)])
#define IM(m, i, j) (&(m).im[(size_t)(i) * (m).n + (j)])

/* ------------------------------------------------------------------------------------------------ */
/* one Jacobi rotation                                                       */
/* ------------------------------------------------------------------------------------------------ */

typedef struct {
  mpfr_t c, sr, si; /* c real, sigma = sr + i si */
  mpfr_t absb, zeta, t, w1, w2, w3, w4;
  mpfr_t npr, npi, nqr, nqi; /* new values */
  int active;
} rot_t;

static void rot_init(rot_t *r, long prec) {
  mpfr_init2(r->c, prec); mpfr_init2(r->sr, prec); mpfr_init2(r->si, prec);
  mpfr_init2(r->absb, prec); mpfr_init2(r->zeta, prec); mpfr_init2(r->t, prec);
  mpfr_init2(r->w1, prec); mpfr_init2(r->w2, prec); mpfr_init2(r->w3, prec); mpfr_init2(r->w4, prec);
  mpfr_init2(r->npr, prec); mpfr_init2(r->npi, prec); mpfr_init2(r->nqr, prec); mpfr_init2(r->nqi, prec);
  r->active = 0;
}
static void rot_clear(rot_t *r) {
  mpfr_clear(r->c); mpfr_clear(r->sr); mpfr_clear(r->si);
  mpfr_clear(r->absb); mpfr_clear(r->zeta); mpfr_clear(r->t);
  mpfr_clear(r->w1); mpfr_clear(r->w2); mpfr_clear(r->w3); mpfr_clear(r->w4);
  mpfr_clear(r->npr); mpfr_clear(r->npi); mpfr_clear(r->nqr); mpfr_clear(r->nqi);
}

/* beta = a_pq, alpha = a_pp, gamma = a_qq.  Skip if |beta| <= thr.
 * zeta = (gamma - alpha) / (2|beta|);  t = sgn(zeta) / (|zeta| + sqrt(1 + zeta^2)), sgn(0) = +1;
 * c = 1/sqrt(1 + t^2);  s = t c;  sigma = s beta / |beta|. */
static void rot_params(rot_t *r, const cmat *A, int p, int q, mpfr_srcptr thr) {
  mpfr_srcptr br = RE(*A, p, q), bi = IM(*A, p, q);
  mpfr_sqr(r->w1, br, RN);
  mpfr_sqr(r->w2, bi, RN);
  mpfr_add(r->w1, r->w1, r->w2, RN);
  mpfr_sqrt(r->absb, r->w1, RN); /* |beta| */
  if (mpfr_cmp(r->absb, thr) <= 0) {
    r->active = 0;
    return;
  }
  r->active = 1;
  mpfr_sub(r->w1, RE(*A, q, q), RE(*A, p, p), RN); /* gamma - alpha */
  mpfr_mul_2si(r->w2, r->absb, 1, RN);              /* 2|beta| */
  mpfr_div(r->zeta, r->w1, r->w2, RN);
  int neg = mpfr_sgn(r->zeta) < 0;
  mpfr_sqr(r->w1, r->zeta, RN);
  mpfr_add_ui(r->w1, r->w1, 1, RN);
  mpfr_sqrt(r->w1, r->w1, RN); /* sqrt(1+zeta^2) */
  mpfr_abs(r->w2, r->zeta, RN);
  mpfr_add(r->w1, r->w1, r->w2, RN);
  mpfr_ui_div(r->t, 1, r->w1, RN);
  if (neg) mpfr_neg(r->t, r->t, RN);
  mpfr_sqr(r->w1, r->t, RN);
  mpfr_add_ui(r->w1, r->w1, 1, RN);
  mpfr_sqrt(r->w1, r->w1, RN);
  mpfr_ui_div(r->c, 1, r->w1, RN);    /* c = 1/sqrt(1+t^2) */
  mpfr_mul(r->w2, r->t, r->c, RN);    /* s = t c */
  mpfr_div(r->w2, r->w2, r->absb, RN);/* s/|beta| */
  mpfr_mul(r->sr, r->w2, br, RN);
  mpfr_mul(r->si, r->w2, bi, RN);
}

/* (x_p, x_q) <- (c x_p - conj(sg) x_q, sg x_p + c x_q), with sg = sr + i*sgn_i*si.
 * sgn_i = +1: column form (A J, V J);  sgn_i = -1: row form (J^H A), i.e. sigma -> conj(sigma). */
static void rot_apply(rot_t *r, mpfr_ptr pr, mpfr_ptr pi, mpfr_ptr qr, mpfr_ptr qi, int sgn_i) {
  /* conj(sg) x_q = (sr qr + s' qi) + i (sr qi - s' qr),  s' = sgn_i * si */
  /* sg x_p       = (sr pr - s' pi) + i (sr pi + s' pr) */
  if (sgn_i > 0) {
    mpfr_fmma(r->w1, r->sr, qr, r->si, qi, RN); /* Re conj(sg) x_q */
    mpfr_fmms(r->w2, r->sr, qi, r->si, qr, RN); /* Im conj(sg) x_q */
    mpfr_fmms(r->w3, r->sr, pr, r->si, pi, RN); /* Re sg x_p */
    mpfr_fmma(r->w4, r->sr, pi, r->si, pr, RN); /* Im sg x_p */
  } else {
    mpfr_fmms(r->w1, r->sr, qr, r->si, qi, RN);
    mpfr_fmma(r->w2, r->sr, qi, r->si, qr, RN);
    mpfr_fmma(r->w3, r->sr, pr, r->si, pi, RN);
    mpfr_fmms(r->w4, r->sr, pi, r->si, pr, RN);
  }
  mpfr_fms(r->npr, r->c, pr, r->w1, RN); /* c pr - w1 */
  mpfr_fms(r->npi, r->c, pi, r->w2, RN);
  mpfr_fma(r->nqr, r->c, qr, r->w3, RN); /* c qr + w3 */
  mpfr_fma(r->nqi, r->c, qi, r->w4, RN);
  mpfr_swap(pr, r->npr);
  mpfr_swap(pi, r->npi);
  mpfr_swap(qr, r->nqr);
  mpfr_swap(qi, r->nqi);
}

static void rot_columns(rot_t *r, cmat *A, cmat *V, int p, int q) {
  int n = A->n;
  for (int k = 0; k < n; ++k) rot_apply(r, RE(*A, k, p), IM(*A, k, p), RE(*A, k, q), IM(*A, k, q), +1);
  for (int k = 0; k < n; ++k) rot_apply(r, RE(*V, k, p), IM(*V, k, p), RE(*V, k, q), IM(*V, k, q), +1);
}
static void rot_rows(rot_t *r, cmat *A, int p, int q) {
  int n = A->n;
  for (int k = 0; k < n; ++k) rot_apply(r, RE(*A, p, k), IM(*A, p, k), RE(*A, q, k), IM(*A, q, k), -1);
  mpfr_set_zero(RE(*A, p, q), +1); mpfr_set_zero(IM(*A, p, q), +1);
  mpfr_set_zero(RE(*A, q, p), +1); mpfr_set_zero(IM(*A, q, p), +1);
  mpfr_set_zero(IM(*A, p, p), +1); mpfr_set_zero(IM(*A, q, q), +1);
}

/* off(A)^2 = sum_{i != j} |a_ij|^2 */
static void off_norm2(mpfr_ptr out, const cmat *A, mpfr_ptr w) {
  int n = A->n;
  mpfr_set_zero(out, +1);
  for (int i = 0; i < n; ++i)
    for (int j = 0; j < n; ++j) {
      if (i == j) continue;
      mpfr_sqr(w, RE(*A, i, j), RN); mpfr_add(out, out, w, RN);
      mpfr_sqr(w, IM(*A, i, j), RN); mpfr_add(out, out, w, RN);
    }
}

/* ------------------------------------------------------------------------------------------------ */
/* the oracle                                                                                       */
/* ------------------------------------------------------------------------------------------------ */

/* Cyclic Jacobi eigendecomposition of one Hermitian matrix.
 *   ordering 0 = row-cyclic, serial;  1 = round-robin (tournament), OpenMP over the disjoint pairs of a round.
 *   guard_bits: working precision P_o = prec + guard_bits (128 is the documented default, reading A6).
 *   max_rotations > 0: stop after that many rotations (bench sampling hook; result then NOT converged).
 *   info[0] = sweeps, info[1] = rotations applied, info[2] = status (0 ok, 2 not converged, 3 malformed input)
 * Returns info[2]. */
int zkd_oracle_diag_herm(int N, int prec, int guard_bits, int ordering, int nthreads, long max_rotations,
                         const uint8_t *A_api, uint8_t *eigvals_api, uint8_t *eigvecs_api, long *info) {
  const long Po = (long)prec + guard_bits;
  const size_t rb = api_real_bytes(prec);
  long sweeps = 0, rotations = 0;
  int status = 0;
  if (nthreads < 1) nthreads = 1;
  if (info) info[0] = info[1] = info[2] = 0;
  if (N < 1 || prec < 64 || prec % 64) { if (info) info[2] = 3; return 3; }

  mpfr_t tmpP, F, thr, offtol, w, off2;
  mpfr_init2(tmpP, prec); mpfr_init2(F, Po); mpfr_init2(thr, Po); mpfr_init2(offtol, Po);
  mpfr_init2(w, Po); mpfr_init2(off2, Po);
  cmat A = cmat_alloc(N, Po), V = cmat_alloc(N, Po);

  /* step 1: copy A, upper triangle authoritative, a_ji = conj(a_ij), Im a_ii = 0; V = I; F = ||A||_F */
  for (int i = 0; i < N && !status; ++i)
    for (int j = i; j < N; ++j) {
      const uint8_t *src = A_api + ((size_t)i * N + j) * 2 * rb;
      if (api_get(RE(A, i, j), src, prec, tmpP) || api_get(IM(A, i, j), src + rb, prec, tmpP)) { status = 3; break; }
      if (i == j) mpfr_set_zero(IM(A, i, j), +1);
      else { mpfr_set(RE(A, j, i), RE(A, i, j), RN); mpfr_neg(IM(A, j, i), IM(A, i, j), RN); }
    }
  if (status) goto done;
  for (int i = 0; i < N; ++i) mpfr_set_ui(RE(V, i, i), 1, RN);
  mpfr_set_zero(F, +1);
  for (int i = 0; i < N; ++i)
    for (int j = 0; j < N; ++j) {
      mpfr_sqr(w, RE(A, i, j), RN); mpfr_add(F, F, w, RN);
      mpfr_sqr(w, IM(A, i, j), RN); mpfr_add(F, F, w, RN);
    }
  mpfr_sqrt(F, F, RN);
  /* rotation skip threshold 2^-(Po+16) F / N; convergence off(A) <= 2^-(prec+64) F */
  mpfr_div_2si(thr, F, Po + 16, RN); mpfr_div_ui(thr, thr, (unsigned long)N, RN);
  mpfr_div_2si(offtol, F, prec + 64, RN);

  {
    int nt = ordering == 1 ? nthreads : 1;
    int M = N + (N & 1); /* round-robin players (one dummy if N odd) */
    rot_t *rots = (rot_t *)malloc(sizeof(rot_t) * (size_t)(M / 2 > 0 ? M / 2 : 1));
    for (int i = 0; i < (M / 2 > 0 ? M / 2 : 1); ++i) rot_init(&rots[i], Po);
    int *perm = (int *)malloc(sizeof(int) * (size_t)(M > 0 ? M : 1));
    int *pp = (int *)malloc(sizeof(int) * (size_t)(M / 2 + 1)), *qq = (int *)malloc(sizeof(int) * (size_t)(M / 2 + 1));

    /* step 2: sweeps until off(A) <= 2^-(P+64) F, or a sweep skipped every rotation; fail after 80 */
    for (;;) {
      off_norm2(off2, &A, w);
      mpfr_sqrt(off2, off2, RN);
      if (mpfr_cmp(off2, offtol) <= 0) break;
      if (sweeps >= 80) { status = 2; break; }
      if (max_rotations > 0 && rotations >= max_rotations) { status = 2; break; }
      long applied = 0;
      if (ordering == 0) {
        /* step 3: row-cyclic sweep */
        for (int p = 0; p < N - 1; ++p)
          for (int q = p + 1; q < N; ++q) {
            if (max_rotations > 0 && rotations + applied >= max_rotations) continue;
            rot_params(&rots[0], &A, p, q, thr);
            if (!rots[0].active) continue;
            rot_columns(&rots[0], &A, &V, p, q);
            rot_rows(&rots[0], &A, p, q);
            ++applied;
          }
      } else {
        /* step 5: round-robin ordering, M-1 rounds of M/2 disjoint pairs; column phase then row phase */
        for (int i = 0; i < M; ++i) perm[i] = i;
        for (int round = 0; round < M - 1; ++round) {
          if (max_rotations > 0 && rotations + applied >= max_rotations) break;
          int np = 0;
          for (int i = 0; i < M / 2; ++i) {
            int a = perm[i], b = perm[M - 1 - i];
            if (a >= N || b >= N) continue;
            pp[np] = a < b ? a : b; qq[np] = a < b ? b : a; ++np;
          }
#pragma omp parallel for num_threads(nt) schedule(dynamic, 1)
          for (int i = 0; i < np; ++i) rot_params(&rots[i], &A, pp[i], qq[i], thr);
#pragma omp parallel for num_threads(nt) schedule(dynamic, 1)
          for (int i = 0; i < np; ++i) if (rots[i].active) rot_columns(&rots[i], &A, &V, pp[i], qq[i]);
#pragma omp parallel for num_threads(nt) schedule(dynamic, 1)
          for (int i = 0; i < np; ++i) if (rots[i].active) rot_rows(&rots[i], &A, pp[i], qq[i]);
          for (int i = 0; i < np; ++i) applied += rots[i].active;
          /* rotate players 1..M-1, player 0 fixed */
          int last = perm[M - 1];
          for (int i = M - 1; i > 1; --i) perm[i] = perm[i - 1];
          if (M > 1) perm[1] = last;
        }
      }
      rotations += applied;
      ++sweeps;
      if (applied == 0) break;
    }
    for (int i = 0; i < (M / 2 > 0 ? M / 2 : 1); ++i) rot_clear(&rots[i]);
    free(rots); free(perm); free(pp); free(qq);
  }

  /* step 4: lambda_j = Re a_jj; stable ascending sort; permute V; renormalise; phase-normalise (A9); round */
  {
    int *ord = (int *)malloc(sizeof(int) * (size_t)N);
    for (int i = 0; i < N; ++i) ord[i] = i;
    for (int i = 1; i < N; ++i) { /* insertion sort: stable */
      int k = ord[i], j = i - 1;
      while (j >= 0 && mpfr_cmp(RE(A, ord[j], ord[j]), RE(A, k, k)) > 0) { ord[j + 1] = ord[j]; --j; }
      ord[j + 1] = k;
    }
    mpfr_t nrm, best, m2, ur, ui, xr, xi;
    mpfr_init2(nrm, Po); mpfr_init2(best, Po); mpfr_init2(m2, Po);
    mpfr_init2(ur, Po); mpfr_init2(ui, Po); mpfr_init2(xr, Po); mpfr_init2(xi, Po);
    for (int jj = 0; jj < N; ++jj) {
      int j = ord[jj];
      if (eigvals_api) api_put(eigvals_api + (size_t)jj * rb, RE(A, j, j), prec, tmpP);
      if (!eigvecs_api) continue;
      /* unit 2-norm */
      mpfr_set_zero(nrm, +1);
      int kstar = 0;
      mpfr_set_si(best, -1, RN);
      for (int k = 0; k < N; ++k) {
        mpfr_sqr(m2, RE(V, k, j), RN); mpfr_sqr(w, IM(V, k, j), RN); mpfr_add(m2, m2, w, RN);
        mpfr_add(nrm, nrm, m2, RN);
        if (mpfr_cmp(m2, best) > 0) { mpfr_set(best, m2, RN); kstar = k; } /* first index attaining the max */
      }
      mpfr_sqrt(nrm, nrm, RN);
      /* phase: multiply by conj(x_k*) / |x_k*|, and divide by the norm */
      mpfr_sqrt(best, best, RN);
      mpfr_mul(w, best, nrm, RN);
      mpfr_div(ur, RE(V, kstar, j), w, RN);
      mpfr_div(ui, IM(V, kstar, j), w, RN);
      mpfr_neg(ui, ui, RN); /* u = conj(x_k*) / (|x_k*| ||x||) */
      for (int k = 0; k < N; ++k) {
        mpfr_fmms(xr, RE(V, k, j), ur, IM(V, k, j), ui, RN);
        mpfr_fmma(xi, RE(V, k, j), ui, IM(V, k, j), ur, RN);
        if (k == kstar) mpfr_set_zero(xi, +1);
        uint8_t *dst = eigvecs_api + ((size_t)k * N + jj) * 2 * rb;
        api_put(dst, xr, prec, tmpP);
        api_put(dst + rb, xi, prec, tmpP);
      }
    }
    mpfr_clear(nrm); mpfr_clear(best); mpfr_clear(m2);
    mpfr_clear(ur); mpfr_clear(ui); mpfr_clear(xr); mpfr_clear(xi);
    free(ord);
  }

done:
  cmat_free(&A); cmat_free(&V);
  mpfr_clear(tmpP); mpfr_clear(F); mpfr_clear(thr); mpfr_clear(offtol); mpfr_clear(w); mpfr_clear(off2);
  if (info) { info[0] = sweeps; info[1] = rotations; info[2] = status; }
  return status;
}

/* ------------------------------------------------------------------------------------------------ */
/* comparator (SURVEY.md 8(c) "Comparator"; well-conditioned difference formulas only)               */
/* ------------------------------------------------------------------------------------------------ */

static void load_cmat(cmat *M, const uint8_t *api, int n, int prec, mpfr_ptr tmpP, int herm_upper) {
  size_t rb = api_real_bytes(prec);
  for (int i = 0; i < n; ++i)
    for (int j = 0; j < n; ++j) {
      const uint8_t *src = api + ((size_t)i * n + j) * 2 * rb;
      api_get(RE(*M, i, j), src, prec, tmpP);
      api_get(IM(*M, i, j), src + rb, prec, tmpP);
    }
  if (herm_upper)
    for (int i = 0; i < n; ++i) {
      mpfr_set_zero(IM(*M, i, i), +1);
      for (int j = i + 1; j < n; ++j) { mpfr_set(RE(*M, j, i), RE(*M, i, j), RN); mpfr_neg(IM(*M, j, i), IM(*M, i, j), RN); }
    }
}

static double log2_mpfr(mpfr_srcptr x) {
  if (mpfr_zero_p(x)) return -1.0e9;
  long e;
  double m = mpfr_get_d_2exp(&e, x, RN);
  return log2(fabs(m)) + (double)e;
}

/* Compare a candidate decomposition (lam, X) of A against invariants and (optionally) a reference (lam0, X0).
 *  cols/ncols: columns on which residual and orthogonality are evaluated (NULL => all N).
 *  lam0, X0 may be NULL (then (i)/(iv) are skipped).
 *  out[0] = log2 max_j |lam_j - lam0_j| / F                          (i)
 *  out[1] = log2 max_{j in cols} ||A x_j - lam_j x_j||_2 / F         (ii)
 *  out[2] = log2 max_{j in cols, all i} |x_i^H x_j - delta_ij|       (iii)
 *  out[3] = max over groups of  log2 ||E_G||_F - log2 (2^-(prec-38) F / gap_G)   (iv)  (<= 0 passes; 2^-730 at 768 bit)
 *  out[4] = log2 F;  out[5] = number of groups;  out[6] = largest group;  out[7] = log2 of worst ||E_G||_F
 * Groups (reading A10): reference eigenvalues sorted ascending; a new group starts where the gap exceeds
 * 2^-(prec-102) F (2^-666 F at 768 bit; the two constants follow the precision for the paper's 256- and 128-bit
 * settings, PAPER.md:61, :65 - DESIGN.md section 3, reading A18; at 768 bit nothing changes).  gap_G = distance from the group's extreme members to the nearest eigenvalue outside.
 * E_G = X_G - X0_G (X0_G^H X_G)  (= ||sin Theta||_F; for |G| = 1 the phase-aligned difference). */
int zkd_oracle_compare(int N, int prec, int nthreads, const uint8_t *A_api, const uint8_t *lam_api,
                       const uint8_t *X_api, const uint8_t *lam0_api, const uint8_t *X0_api, const int *cols,
                       int ncols, double *out) {
  const long Pc = (long)prec + 256;
  const size_t rb = api_real_bytes(prec);
  if (nthreads < 1) nthreads = 1;
  mpfr_t tmpP, F, w, acc;
  mpfr_init2(tmpP, prec); mpfr_init2(F, Pc); mpfr_init2(w, Pc); mpfr_init2(acc, Pc);
  cmat A = cmat_alloc(N, Pc), X = cmat_alloc(N, Pc);
  load_cmat(&A, A_api, N, prec, tmpP, 1);
  load_cmat(&X, X_api, N, prec, tmpP, 0);
  __mpfr_struct *lam = vec_alloc((size_t)N, Pc);
  for (int j = 0; j < N; ++j) api_get(&lam[j], lam_api + (size_t)j * rb, prec, tmpP);
  mpfr_set_zero(F, +1);
  for (int i = 0; i < N; ++i)
    for (int j = 0; j < N; ++j) {
      mpfr_sqr(w, RE(A, i, j), RN); mpfr_add(F, F, w, RN);
      mpfr_sqr(w, IM(A, i, j), RN); mpfr_add(F, F, w, RN);
    }
  mpfr_sqrt(F, F, RN);
  double lF = log2_mpfr(F);
  for (int i = 0; i < 8; ++i) out[i] = -1.0e9;
  out[4] = lF;
  int nc = cols ? ncols : N;

  /* (ii) residuals and (iii) orthogonality on the chosen columns */
  double *res = (double *)malloc(sizeof(double) * (size_t)nc), *orth = (double *)malloc(sizeof(double) * (size_t)nc);
#pragma omp parallel num_threads(nthreads)
  {
    mpfr_t sr, si, t1, t2, r2, d;
    mpfr_init2(sr, Pc); mpfr_init2(si, Pc); mpfr_init2(t1, Pc); mpfr_init2(t2, Pc); mpfr_init2(r2, Pc); mpfr_init2(d, Pc);
#pragma omp for schedule(dynamic, 1)
    for (int c = 0; c < nc; ++c) {
      int j = cols ? cols[c] : c;
      mpfr_set_zero(r2, +1);
      for (int i = 0; i < N; ++i) {
        mpfr_set_zero(sr, +1); mpfr_set_zero(si, +1);
        for (int k = 0; k < N; ++k) { /* (A x_j)_i */
          mpfr_fmms(t1, RE(A, i, k), RE(X, k, j), IM(A, i, k), IM(X, k, j), RN);
          mpfr_fmma(t2, RE(A, i, k), IM(X, k, j), IM(A, i, k), RE(X, k, j), RN);
          mpfr_add(sr, sr, t1, RN); mpfr_add(si, si, t2, RN);
        }
        mpfr_mul(t1, &lam[j], RE(X, i, j), RN); mpfr_sub(sr, sr, t1, RN);
        mpfr_mul(t2, &lam[j], IM(X, i, j), RN); mpfr_sub(si, si, t2, RN);
        mpfr_sqr(t1, sr, RN); mpfr_sqr(t2, si, RN);
        mpfr_add(r2, r2, t1, RN); mpfr_add(r2, r2, t2, RN);
      }
      mpfr_sqrt(r2, r2, RN);
      res[c] = log2_mpfr(r2) - lF;
      double worst = -1.0e9;
      for (int i = 0; i < N; ++i) { /* x_i^H x_j */
        mpfr_set_zero(sr, +1); mpfr_set_zero(si, +1);
        for (int k = 0; k < N; ++k) {
          mpfr_fmma(t1, RE(X, k, i), RE(X, k, j), IM(X, k, i), IM(X, k, j), RN);
          mpfr_fmms(t2, RE(X, k, i), IM(X, k, j), IM(X, k, i), RE(X, k, j), RN);
          mpfr_add(sr, sr, t1, RN); mpfr_add(si, si, t2, RN);
        }
        if (i == j) mpfr_sub_ui(sr, sr, 1, RN);
        mpfr_sqr(t1, sr, RN); mpfr_sqr(t2, si, RN); mpfr_add(d, t1, t2, RN); mpfr_sqrt(d, d, RN);
        double l = log2_mpfr(d);
        if (l > worst) worst = l;
      }
      orth[c] = worst;
    }
    mpfr_clear(sr); mpfr_clear(si); mpfr_clear(t1); mpfr_clear(t2); mpfr_clear(r2); mpfr_clear(d);
  }
  for (int c = 0; c < nc; ++c) { if (res[c] > out[1]) out[1] = res[c]; if (orth[c] > out[2]) out[2] = orth[c]; }
  free(res); free(orth);

  if (lam0_api) {
    __mpfr_struct *lam0 = vec_alloc((size_t)N, Pc);
    for (int j = 0; j < N; ++j) api_get(&lam0[j], lam0_api + (size_t)j * rb, prec, tmpP);
    /* (i) */
    for (int j = 0; j < N; ++j) {
      mpfr_sub(w, &lam[j], &lam0[j], RN);
      double l = log2_mpfr(w) - lF;
      if (l > out[0]) out[0] = l;
    }
    if (X0_api) {
      /* (iv) groups on the reference spectrum */
      cmat X0 = cmat_alloc(N, Pc);
      load_cmat(&X0, X0_api, N, prec, tmpP, 0);
      mpfr_t gthr, gap, g2;
      mpfr_init2(gthr, Pc); mpfr_init2(gap, Pc); mpfr_init2(g2, Pc);
      mpfr_div_2si(gthr, F, prec - 102, RN);
      int *gstart = (int *)malloc(sizeof(int) * (size_t)(N + 1));
      int ng = 0;
      gstart[ng++] = 0;
      for (int j = 0; j + 1 < N; ++j) {
        mpfr_sub(w, &lam0[j + 1], &lam0[j], RN);
        if (mpfr_cmp(w, gthr) > 0) gstart[ng++] = j + 1;
      }
      gstart[ng] = N;
      out[5] = ng;
      double *margin = (double *)malloc(sizeof(double) * (size_t)ng), *eabs = (double *)malloc(sizeof(double) * (size_t)ng);
      int maxg = 0;
      for (int g = 0; g < ng; ++g) if (gstart[g + 1] - gstart[g] > maxg) maxg = gstart[g + 1] - gstart[g];
      out[6] = maxg;
#pragma omp parallel num_threads(nthreads)
      {
        mpfr_t sr, si, t1, t2, e2, gp, g3;
        mpfr_init2(sr, Pc); mpfr_init2(si, Pc); mpfr_init2(t1, Pc); mpfr_init2(t2, Pc); mpfr_init2(e2, Pc);
        mpfr_init2(gp, Pc); mpfr_init2(g3, Pc);
#pragma omp for schedule(dynamic, 1)
        for (int g = 0; g < ng; ++g) {
          int a = gstart[g], b = gstart[g + 1], m = b - a;
          /* gap to the nearest eigenvalue outside */
          int have = 0;
          if (a > 0) { mpfr_sub(gp, &lam0[a], &lam0[a - 1], RN); have = 1; }
          if (b < N) {
            mpfr_sub(g3, &lam0[b], &lam0[b - 1], RN);
            if (!have || mpfr_cmp(g3, gp) < 0) mpfr_set(gp, g3, RN);
            have = 1;
          }
          /* M = X0_G^H X_G (m x m), E = X_G - X0_G M */
          cmat Mm = cmat_alloc(m, Pc);
          for (int p = 0; p < m; ++p)
            for (int q = 0; q < m; ++q) {
              mpfr_set_zero(sr, +1); mpfr_set_zero(si, +1);
              for (int k = 0; k < N; ++k) {
                mpfr_fmma(t1, RE(X0, k, a + p), RE(X, k, a + q), IM(X0, k, a + p), IM(X, k, a + q), RN);
                mpfr_fmms(t2, RE(X0, k, a + p), IM(X, k, a + q), IM(X0, k, a + p), RE(X, k, a + q), RN);
                mpfr_add(sr, sr, t1, RN); mpfr_add(si, si, t2, RN);
              }
              mpfr_set(RE(Mm, p, q), sr, RN); mpfr_set(IM(Mm, p, q), si, RN);
            }
          mpfr_set_zero(e2, +1);
          for (int k = 0; k < N; ++k)
            for (int q = 0; q < m; ++q) {
              mpfr_set(sr, RE(X, k, a + q), RN); mpfr_set(si, IM(X, k, a + q), RN);
              for (int p = 0; p < m; ++p) {
                mpfr_fmms(t1, RE(X0, k, a + p), RE(Mm, p, q), IM(X0, k, a + p), IM(Mm, p, q), RN);
                mpfr_fmma(t2, RE(X0, k, a + p), IM(Mm, p, q), IM(X0, k, a + p), RE(Mm, p, q), RN);
                mpfr_sub(sr, sr, t1, RN); mpfr_sub(si, si, t2, RN);
              }
              mpfr_sqr(t1, sr, RN); mpfr_sqr(t2, si, RN);
              mpfr_add(e2, e2, t1, RN); mpfr_add(e2, e2, t2, RN);
            }
          mpfr_sqrt(e2, e2, RN);
          eabs[g] = log2_mpfr(e2);
          double ltol = have ? (-(double)(prec - 38) + lF - log2_mpfr(gp)) : 1.0e9; /* single group spanning everything: any basis */
          margin[g] = eabs[g] - ltol;
          cmat_free(&Mm);
        }
        mpfr_clear(sr); mpfr_clear(si); mpfr_clear(t1); mpfr_clear(t2); mpfr_clear(e2); mpfr_clear(gp); mpfr_clear(g3);
      }
      for (int g = 0; g < ng; ++g) { if (margin[g] > out[3]) out[3] = margin[g]; if (eabs[g] > out[7]) out[7] = eabs[g]; }
      free(margin); free(eabs); free(gstart);
      mpfr_clear(gthr); mpfr_clear(gap); mpfr_clear(g2);
      cmat_free(&X0);
    }
    vec_free(lam0, (size_t)N);
  }
  vec_free(lam, (size_t)N);
  cmat_free(&A); cmat_free(&X);
  mpfr_clear(tmpP); mpfr_clear(F); mpfr_clear(w); mpfr_clear(acc);
  return 0;
}

/* number-format round trip helpers used by the tests */
double zkd_oracle_api_to_double(const uint8_t *src, int prec) {
  mpfr_t t, d;
  mpfr_init2(t, prec); mpfr_init2(d, prec);
  double r = NAN;
  if (api_get(d, src, prec, t) == 0) r = mpfr_get_d(d, RN);
  mpfr_clear(t); mpfr_clear(d);
  return r;
}
void zkd_oracle_api_from_double(uint8_t *dst, int prec, double v) {
  mpfr_t t, d;
  mpfr_init2(t, prec); mpfr_init2(d, prec);
  mpfr_set_d(d, v, RN);
  api_put(dst, d, prec, t);
  mpfr_clear(t); mpfr_clear(d);
}
const char *zkd_oracle_mpfr_version(void) { return mpfr_get_version(); }
int zkd_oracle_max_threads(void) { return omp_get_max_threads(); }

/* ================================================================================================ */
/* Singular value decomposition                                              */
/* ================================================================================================ */
/* PAPER.md:31, :33 (section 2): ZKCM_CUS ships two routines, Hermitian diagonalisation and "singular value decomposition";
 * PAPER.md:49 (section 2.2): ZKCM_QC switches both.  Result definition (plain): for A in C^{M x N}, K = min(M, N):
 * sigma_1 >= ... >= sigma_K >= 0, U (M x K) and V (N x K) with orthonormal columns, A V = U diag(sigma),
 * A^H U = V diag(sigma).  Computed by the textbook one-sided Jacobi method (Hestenes) on MPFR:
 *   1. working precision P_o = prec + guard_bits.  If M < N work on A^H and swap U and V at the end.  B = A, W = I (N x N).
 *   2. sweeps over all column pairs p < q (row-cyclic): alpha = ||b_p||^2, beta = ||b_q||^2, gamma = b_p^H b_q;
 *      skip if |gamma| <= 2^-(P_o-8) sqrt(alpha beta) (the computed gamma carries rounding noise of about 2^-P_o sqrt(alpha
 *      beta): a threshold below that would rotate on noise for ever); else rotate with the SAME formulas as the eigenvalue oracle applied
 *      to the 2 x 2 Gram matrix [[alpha, gamma], [conj gamma, beta]]:  zeta = (beta - alpha) / (2|gamma|),
 *      t = sgn(zeta) / (|zeta| + sqrt(1 + zeta^2)), c = 1/sqrt(1 + t^2), s = t c, sg = s gamma/|gamma|,
 *      (b_p, b_q) <- (c b_p - conj(sg) b_q, sg b_p + c b_q), same on (w_p, w_q).
 *      Stop when a sweep applied no rotation; fail after 80 sweeps.
 *   3. sigma_j = ||b_j||; sort descending (stable); v_j = w_j; u_j = b_j / sigma_j; when sigma_j <= 2^-(prec+32) F the
 *      direction of b_j is noise: sigma_j is kept as computed and u_j is completed by Gram-Schmidt (twice) of the unit
 *      vectors e_0, e_1, ... against the columns already fixed.
 *   4. phase: the first component of largest modulus of v_j is made real positive (the same factor on u_j); unit norm;
 *      round to prec bits.
 * Layout: A[i][j] row-major complex (M x N); S[j] real; U[i][j] (M x K), V[i][j] (N x K) row-major complex.
 * info[0] = sweeps, info[1] = rotations, info[2] = status (0 ok, 2 not converged, 3 malformed).
 * Parity status: pinned (tests/test_oracle_pins.py, section "SVD": 2 x 2 closed form, constructed U S V^H, sigma^2 =
 * eigenvalues of A^H A by the eigenvalue oracle, ||A||_F^2 = sum sigma^2, diagonal / rank-deficient / zero inputs,
 * mpmath.svd_c as a third opinion). */

typedef struct { int r, c; __mpfr_struct *re, *im; } rmat;
static rmat rmat_alloc(int r, int c, long prec) {
  rmat m; m.r = r; m.c = c;
  m.re = vec_alloc((size_t)r * c, prec); m.im = vec_alloc((size_t)r * c, prec);
  return m;
}
static void rmat_free(rmat *m) { vec_free(m->re, (size_t)m->r * m->c); vec_free(m->im, (size_t)m->r * m->c); }
#define RRE(m, i, j) (&(m).re[(size_t)(i) * (m).c + (j)])
#define RIM(m, i, j) (&(m).im[(size_t)(i) * (m).c + (j)])

/* acc <- x_p^H x_q over the rows of m (ar + i ai) */
static void col_dot(mpfr_ptr ar, mpfr_ptr ai, const rmat *m, int p, int q, mpfr_ptr w) {
  mpfr_set_zero(ar, +1); mpfr_set_zero(ai, +1);
  for (int k = 0; k < m->r; ++k) {
    /* conj(x_p) x_q = (pr qr + pi qi) + i (pr qi - pi qr) */
    mpfr_fmma(w, RRE(*m, k, p), RRE(*m, k, q), RIM(*m, k, p), RIM(*m, k, q), RN); mpfr_add(ar, ar, w, RN);
    mpfr_fmms(w, RRE(*m, k, p), RIM(*m, k, q), RIM(*m, k, p), RRE(*m, k, q), RN); mpfr_add(ai, ai, w, RN);
  }
}

int zkd_oracle_svd(int M, int N, int prec, int guard_bits, const uint8_t *A_api, uint8_t *S_api, uint8_t *U_api,
                   uint8_t *V_api, long *info) {
  const long Po = (long)prec + guard_bits;
  const size_t rb = api_real_bytes(prec);
  long sweeps = 0, rotations = 0;
  int status = 0;
  if (info) info[0] = info[1] = info[2] = 0;
  if (M < 1 || N < 1 || prec < 64 || prec % 64) { if (info) info[2] = 3; return 3; }
  const int tr = M < N;              /* work on A^H */
  const int R = tr ? N : M, C = tr ? M : N, K = C;
  mpfr_t tmpP, F, w, al, be, gr, gi, thr2, zt;
  mpfr_init2(tmpP, prec); mpfr_init2(F, Po); mpfr_init2(w, Po); mpfr_init2(al, Po); mpfr_init2(be, Po);
  mpfr_init2(gr, Po); mpfr_init2(gi, Po); mpfr_init2(thr2, Po); mpfr_init2(zt, Po);
  rmat B = rmat_alloc(R, C, Po), W = rmat_alloc(C, C, Po), Uo = rmat_alloc(R, K, Po);
  __mpfr_struct *sig = vec_alloc((size_t)C, Po);
  rot_t rt; rot_init(&rt, Po);
  int *ord = (int *)malloc(sizeof(int) * (size_t)C);

  for (int i = 0; i < M && !status; ++i)
    for (int j = 0; j < N; ++j) {
      const uint8_t *src = A_api + ((size_t)i * N + j) * 2 * rb;
      mpfr_ptr dr = tr ? RRE(B, j, i) : RRE(B, i, j), di = tr ? RIM(B, j, i) : RIM(B, i, j);
      if (api_get(dr, src, prec, tmpP) || api_get(di, src + rb, prec, tmpP)) { status = 3; break; }
      if (tr) mpfr_neg(di, di, RN);
    }
  if (status) goto done;
  for (int i = 0; i < C; ++i) mpfr_set_ui(RRE(W, i, i), 1, RN);
  mpfr_set_zero(F, +1);
  for (int i = 0; i < R; ++i)
    for (int j = 0; j < C; ++j) {
      mpfr_sqr(w, RRE(B, i, j), RN); mpfr_add(F, F, w, RN);
      mpfr_sqr(w, RIM(B, i, j), RN); mpfr_add(F, F, w, RN);
    }
  mpfr_sqrt(F, F, RN);

  /* step 2 */
  for (;;) {
    if (sweeps >= 80) { status = 2; break; }
    long applied = 0;
    for (int p = 0; p < C - 1; ++p)
      for (int q = p + 1; q < C; ++q) {
        col_dot(al, w, &B, p, p, zt);
        col_dot(be, w, &B, q, q, zt);
        col_dot(gr, gi, &B, p, q, zt);
        /* skip if |gamma|^2 <= 2^-(2 Po - 16) alpha beta */
        mpfr_sqr(rt.w1, gr, RN); mpfr_sqr(rt.w2, gi, RN); mpfr_add(rt.w1, rt.w1, rt.w2, RN); /* |gamma|^2 */
        mpfr_mul(thr2, al, be, RN); mpfr_div_2si(thr2, thr2, 2 * Po - 16, RN);
        if (mpfr_zero_p(rt.w1) || mpfr_cmp(rt.w1, thr2) <= 0) continue;
        mpfr_sqrt(rt.absb, rt.w1, RN);
        mpfr_sub(rt.w1, be, al, RN);
        mpfr_mul_2si(rt.w2, rt.absb, 1, RN);
        mpfr_div(rt.zeta, rt.w1, rt.w2, RN);
        int neg = mpfr_sgn(rt.zeta) < 0;
        mpfr_sqr(rt.w1, rt.zeta, RN); mpfr_add_ui(rt.w1, rt.w1, 1, RN); mpfr_sqrt(rt.w1, rt.w1, RN);
        mpfr_abs(rt.w2, rt.zeta, RN); mpfr_add(rt.w1, rt.w1, rt.w2, RN);
        mpfr_ui_div(rt.t, 1, rt.w1, RN);
        if (neg) mpfr_neg(rt.t, rt.t, RN);
        mpfr_sqr(rt.w1, rt.t, RN); mpfr_add_ui(rt.w1, rt.w1, 1, RN); mpfr_sqrt(rt.w1, rt.w1, RN);
        mpfr_ui_div(rt.c, 1, rt.w1, RN);
        mpfr_mul(rt.w2, rt.t, rt.c, RN); mpfr_div(rt.w2, rt.w2, rt.absb, RN);
        mpfr_mul(rt.sr, rt.w2, gr, RN); mpfr_mul(rt.si, rt.w2, gi, RN);
        for (int k = 0; k < R; ++k) rot_apply(&rt, RRE(B, k, p), RIM(B, k, p), RRE(B, k, q), RIM(B, k, q), +1);
        for (int k = 0; k < C; ++k) rot_apply(&rt, RRE(W, k, p), RIM(W, k, p), RRE(W, k, q), RIM(W, k, q), +1);
        ++applied;
      }
    rotations += applied;
    ++sweeps;
    if (applied == 0) break;
  }

  /* step 3 */
  for (int j = 0; j < C; ++j) { col_dot(&sig[j], w, &B, j, j, zt); mpfr_sqrt(&sig[j], &sig[j], RN); ord[j] = j; }
  for (int i = 1; i < C; ++i) { /* insertion sort, descending, stable */
    int k = ord[i], j = i - 1;
    while (j >= 0 && mpfr_cmp(&sig[ord[j]], &sig[k]) < 0) { ord[j + 1] = ord[j]; --j; }
    ord[j + 1] = k;
  }
  mpfr_div_2si(thr2, F, prec + 32, RN); /* directions of columns shorter than this are noise */
  {
    int next_e = 0;
    for (int jj = 0; jj < K; ++jj) {
      int j = ord[jj];
      if (mpfr_cmp(&sig[j], thr2) > 0) {
        for (int k = 0; k < R; ++k) { mpfr_div(RRE(Uo, k, jj), RRE(B, k, j), &sig[j], RN); mpfr_div(RIM(Uo, k, jj), RIM(B, k, j), &sig[j], RN); }
        continue;
      }
      for (; next_e < R; ++next_e) { /* complete by Gram-Schmidt of unit vectors (only reached for rank-deficient input) */
        for (int k = 0; k < R; ++k) { mpfr_set_zero(RRE(Uo, k, jj), +1); mpfr_set_zero(RIM(Uo, k, jj), +1); }
        mpfr_set_ui(RRE(Uo, next_e, jj), 1, RN);
        for (int pass = 0; pass < 2; ++pass)
          for (int c2 = 0; c2 < K; ++c2) {
            /* orthogonalise against every column already fixed: earlier ones and all later non-noise ones */
            int fixed = c2 < jj || (c2 > jj && mpfr_cmp(&sig[ord[c2]], thr2) > 0);
            if (!fixed) continue;
            if (c2 > jj) { /* later non-noise column: its u is b / sigma, not stored yet */
              for (int k = 0; k < R; ++k) { mpfr_div(RRE(Uo, k, c2), RRE(B, k, ord[c2]), &sig[ord[c2]], RN); mpfr_div(RIM(Uo, k, c2), RIM(B, k, ord[c2]), &sig[ord[c2]], RN); }
            }
            col_dot(gr, gi, &Uo, c2, jj, zt); /* u_c2^H x */
            for (int k = 0; k < R; ++k) {
              mpfr_fmms(w, RRE(Uo, k, c2), gr, RIM(Uo, k, c2), gi, RN); mpfr_sub(RRE(Uo, k, jj), RRE(Uo, k, jj), w, RN);
              mpfr_fmma(w, RRE(Uo, k, c2), gi, RIM(Uo, k, c2), gr, RN); mpfr_sub(RIM(Uo, k, jj), RIM(Uo, k, jj), w, RN);
            }
          }
        col_dot(al, w, &Uo, jj, jj, zt);
        if (mpfr_cmp_d(al, 0.25) > 0) {
          mpfr_sqrt(al, al, RN);
          for (int k = 0; k < R; ++k) { mpfr_div(RRE(Uo, k, jj), RRE(Uo, k, jj), al, RN); mpfr_div(RIM(Uo, k, jj), RIM(Uo, k, jj), al, RN); }
          ++next_e;
          break;
        }
      }
    }
  }
  /* step 4: phase from v_j (in the caller's orientation: V is W unless the problem was transposed, then V is Uo) */
  for (int jj = 0; jj < K; ++jj) {
    int j = ord[jj];
    const rmat *Vsrc = tr ? &Uo : &W;
    int vcol = tr ? jj : j, vrows = tr ? R : C;
    int kstar = 0;
    mpfr_set_si(be, -1, RN);
    mpfr_set_zero(al, +1);
    for (int k = 0; k < vrows; ++k) {
      mpfr_sqr(gr, RRE(*Vsrc, k, vcol), RN); mpfr_sqr(w, RIM(*Vsrc, k, vcol), RN); mpfr_add(gr, gr, w, RN);
      mpfr_add(al, al, gr, RN);
      if (mpfr_cmp(gr, be) > 0) { mpfr_set(be, gr, RN); kstar = k; }
    }
    mpfr_sqrt(be, be, RN);
    /* phase factor f = conj(x_k*) / |x_k*| */
    mpfr_div(gr, RRE(*Vsrc, kstar, vcol), be, RN);
    mpfr_div(gi, RIM(*Vsrc, kstar, vcol), be, RN); mpfr_neg(gi, gi, RN);
    if (S_api) api_put(S_api + (size_t)jj * rb, &sig[j], prec, tmpP);
    for (int side = 0; side < 2; ++side) {
      /* side 0: the caller's U, side 1: the caller's V */
      const int from_uo = tr ? side == 1 : side == 0;
      const rmat *src = from_uo ? &Uo : &W;
      const int col = from_uo ? jj : j, rows = from_uo ? R : C;
      uint8_t *dst0 = side == 0 ? U_api : V_api;
      if (!dst0) continue;
      col_dot(al, w, src, col, col, zt); mpfr_sqrt(al, al, RN); /* unit norm */
      for (int k = 0; k < rows; ++k) {
        mpfr_fmms(be, RRE(*src, k, col), gr, RIM(*src, k, col), gi, RN); mpfr_div(be, be, al, RN);
        mpfr_fmma(w, RRE(*src, k, col), gi, RIM(*src, k, col), gr, RN); mpfr_div(w, w, al, RN);
        if (side == 1 && k == kstar) mpfr_set_zero(w, +1);
        uint8_t *dst = dst0 + ((size_t)k * K + jj) * 2 * rb;
        api_put(dst, be, prec, tmpP);
        api_put(dst + rb, w, prec, tmpP);
      }
    }
  }

done:
  rmat_free(&B); rmat_free(&W); rmat_free(&Uo); vec_free(sig, (size_t)C); rot_clear(&rt); free(ord);
  mpfr_clear(tmpP); mpfr_clear(F); mpfr_clear(w); mpfr_clear(al); mpfr_clear(be); mpfr_clear(gr); mpfr_clear(gi);
  mpfr_clear(thr2); mpfr_clear(zt);
  if (info) { info[0] = sweeps; info[1] = rotations; info[2] = status; }
  return status;
}

static void load_rmat(rmat *m, const uint8_t *api, int prec, mpfr_ptr tmpP) {
  size_t rb = api_real_bytes(prec);
  for (int i = 0; i < m->r; ++i)
    for (int j = 0; j < m->c; ++j) {
      const uint8_t *src = api + ((size_t)i * m->c + j) * 2 * rb;
      api_get(RRE(*m, i, j), src, prec, tmpP);
      api_get(RIM(*m, i, j), src + rb, prec, tmpP);
    }
}

/* ||X_G - X0_G (X0_G^H X_G)||_F^2 over the columns [g0, g1) (the projector distance of comparator (iv)); X, X0: rows x K */
static void proj_dist2(mpfr_ptr out, const rmat *X, const rmat *X0, int g0, int g1, long Pc) {
  const int m = g1 - g0, rows = X->r;
  mpfr_t sr, si, t1, t2;
  mpfr_init2(sr, Pc); mpfr_init2(si, Pc); mpfr_init2(t1, Pc); mpfr_init2(t2, Pc);
  rmat Mm = rmat_alloc(m, m, Pc);
  for (int a = 0; a < m; ++a)
    for (int b = 0; b < m; ++b) {
      mpfr_set_zero(sr, +1); mpfr_set_zero(si, +1);
      for (int k = 0; k < rows; ++k) { /* conj(X0[k][g0+a]) X[k][g0+b] */
        mpfr_fmma(t1, RRE(*X0, k, g0 + a), RRE(*X, k, g0 + b), RIM(*X0, k, g0 + a), RIM(*X, k, g0 + b), RN); mpfr_add(sr, sr, t1, RN);
        mpfr_fmms(t1, RRE(*X0, k, g0 + a), RIM(*X, k, g0 + b), RIM(*X0, k, g0 + a), RRE(*X, k, g0 + b), RN); mpfr_add(si, si, t1, RN);
      }
      mpfr_set(RRE(Mm, a, b), sr, RN); mpfr_set(RIM(Mm, a, b), si, RN);
    }
  mpfr_set_zero(out, +1);
  for (int k = 0; k < rows; ++k)
    for (int b = 0; b < m; ++b) {
      mpfr_set(sr, RRE(*X, k, g0 + b), RN); mpfr_set(si, RIM(*X, k, g0 + b), RN);
      for (int a = 0; a < m; ++a) {
        mpfr_fmms(t1, RRE(*X0, k, g0 + a), RRE(Mm, a, b), RIM(*X0, k, g0 + a), RIM(Mm, a, b), RN); mpfr_sub(sr, sr, t1, RN);
        mpfr_fmma(t1, RRE(*X0, k, g0 + a), RIM(Mm, a, b), RIM(*X0, k, g0 + a), RRE(Mm, a, b), RN); mpfr_sub(si, si, t1, RN);
      }
      mpfr_sqr(t1, sr, RN); mpfr_sqr(t2, si, RN); mpfr_add(out, out, t1, RN); mpfr_add(out, out, t2, RN);
    }
  rmat_free(&Mm);
  mpfr_clear(sr); mpfr_clear(si); mpfr_clear(t1); mpfr_clear(t2);
}

/* Comparator for a candidate SVD (S, U, V) of A, optionally against a reference (S0, U0, V0).  K = min(M, N).
 *  out[0] = log2 max_j |sigma_j - sigma0_j| / F
 *  out[1] = log2 max_j max(||A v_j - sigma_j u_j||_2, ||A^H u_j - sigma_j v_j||_2) / F
 *  out[2] = log2 max(max |U^H U - I|, max |V^H V - I|)
 *  out[3] = max over groups of log2 err_G - log2 (2^-(prec-38) F / gap_G)      (<= 0 passes)
 *  out[4] = log2 F;  out[5] = groups;  out[6] = largest group;  out[7] = worst log2 err_G
 * Groups: reference sigma sorted descending, a new group where the gap exceeds 2^-(prec-102) F (the rule of
 * zkd_oracle_compare).  For a group of nonzero sigma the pairs are compared as stacked vectors z_j = (u_j; v_j)/sqrt 2 -
 * the eigenvectors of [[0, A], [A^H, 0]] for +sigma_j, so that the common phase of (u_j, v_j) is aligned by the projector -
 * with gap_G = min(distance to the nearest sigma outside the group, 2 sigma_min(G)) (the mirrored eigenvalue -sigma).  For
 * the group of sigma <= 2^-(prec-102) F, u and v decouple: the spans of V_G (when N <= M) and of U_G (when M <= N) are
 * compared separately, gap_G = distance to the smallest sigma outside the group. */
int zkd_oracle_svd_compare(int M, int N, int prec, const uint8_t *A_api, const uint8_t *S_api, const uint8_t *U_api,
                           const uint8_t *V_api, const uint8_t *S0_api, const uint8_t *U0_api, const uint8_t *V0_api,
                           double *out) {
  const long Pc = (long)prec + 256;
  const size_t rb = api_real_bytes(prec);
  const int K = M < N ? M : N;
  mpfr_t tmpP, F, w, sr, si, acc, worst, t1;
  mpfr_init2(tmpP, prec); mpfr_init2(F, Pc); mpfr_init2(w, Pc); mpfr_init2(sr, Pc); mpfr_init2(si, Pc);
  mpfr_init2(acc, Pc); mpfr_init2(worst, Pc); mpfr_init2(t1, Pc);
  rmat A = rmat_alloc(M, N, Pc), U = rmat_alloc(M, K, Pc), V = rmat_alloc(N, K, Pc);
  __mpfr_struct *S = vec_alloc((size_t)K, Pc);
  load_rmat(&A, A_api, prec, tmpP); load_rmat(&U, U_api, prec, tmpP); load_rmat(&V, V_api, prec, tmpP);
  for (int j = 0; j < K; ++j) api_get(&S[j], S_api + (size_t)j * rb, prec, tmpP);
  for (int i = 0; i < 8; ++i) out[i] = -1.0e9;
  mpfr_set_zero(F, +1);
  for (int i = 0; i < M; ++i)
    for (int j = 0; j < N; ++j) {
      mpfr_sqr(w, RRE(A, i, j), RN); mpfr_add(F, F, w, RN);
      mpfr_sqr(w, RIM(A, i, j), RN); mpfr_add(F, F, w, RN);
    }
  mpfr_sqrt(F, F, RN);
  const double lF = log2_mpfr(F);
  out[4] = lF;
  /* (ii) residuals */
  mpfr_set_zero(worst, +1);
  for (int j = 0; j < K; ++j) {
    mpfr_set_zero(acc, +1);
    for (int i = 0; i < M; ++i) { /* (A v_j - sigma_j u_j)_i */
      mpfr_set_zero(sr, +1); mpfr_set_zero(si, +1);
      for (int k = 0; k < N; ++k) {
        mpfr_fmms(t1, RRE(A, i, k), RRE(V, k, j), RIM(A, i, k), RIM(V, k, j), RN); mpfr_add(sr, sr, t1, RN);
        mpfr_fmma(t1, RRE(A, i, k), RIM(V, k, j), RIM(A, i, k), RRE(V, k, j), RN); mpfr_add(si, si, t1, RN);
      }
      mpfr_mul(t1, &S[j], RRE(U, i, j), RN); mpfr_sub(sr, sr, t1, RN);
      mpfr_mul(t1, &S[j], RIM(U, i, j), RN); mpfr_sub(si, si, t1, RN);
      mpfr_sqr(t1, sr, RN); mpfr_add(acc, acc, t1, RN); mpfr_sqr(t1, si, RN); mpfr_add(acc, acc, t1, RN);
    }
    if (mpfr_cmp(acc, worst) > 0) mpfr_set(worst, acc, RN);
    mpfr_set_zero(acc, +1);
    for (int k = 0; k < N; ++k) { /* (A^H u_j - sigma_j v_j)_k */
      mpfr_set_zero(sr, +1); mpfr_set_zero(si, +1);
      for (int i = 0; i < M; ++i) { /* conj(a_ik) u_ij */
        mpfr_fmma(t1, RRE(A, i, k), RRE(U, i, j), RIM(A, i, k), RIM(U, i, j), RN); mpfr_add(sr, sr, t1, RN);
        mpfr_fmms(t1, RRE(A, i, k), RIM(U, i, j), RIM(A, i, k), RRE(U, i, j), RN); mpfr_add(si, si, t1, RN);
      }
      mpfr_mul(t1, &S[j], RRE(V, k, j), RN); mpfr_sub(sr, sr, t1, RN);
      mpfr_mul(t1, &S[j], RIM(V, k, j), RN); mpfr_sub(si, si, t1, RN);
      mpfr_sqr(t1, sr, RN); mpfr_add(acc, acc, t1, RN); mpfr_sqr(t1, si, RN); mpfr_add(acc, acc, t1, RN);
    }
    if (mpfr_cmp(acc, worst) > 0) mpfr_set(worst, acc, RN);
  }
  mpfr_sqrt(worst, worst, RN);
  out[1] = log2_mpfr(worst) - lF;
  /* (iii) orthonormality */
  mpfr_set_zero(worst, +1);
  for (int side = 0; side < 2; ++side) {
    const rmat *X = side ? &V : &U;
    for (int a = 0; a < K; ++a)
      for (int b = a; b < K; ++b) {
        mpfr_set_zero(sr, +1); mpfr_set_zero(si, +1);
        for (int k = 0; k < X->r; ++k) {
          mpfr_fmma(t1, RRE(*X, k, a), RRE(*X, k, b), RIM(*X, k, a), RIM(*X, k, b), RN); mpfr_add(sr, sr, t1, RN);
          mpfr_fmms(t1, RRE(*X, k, a), RIM(*X, k, b), RIM(*X, k, a), RRE(*X, k, b), RN); mpfr_add(si, si, t1, RN);
        }
        if (a == b) mpfr_sub_ui(sr, sr, 1, RN);
        mpfr_abs(sr, sr, RN); mpfr_abs(si, si, RN);
        if (mpfr_cmp(sr, worst) > 0) mpfr_set(worst, sr, RN);
        if (mpfr_cmp(si, worst) > 0) mpfr_set(worst, si, RN);
      }
  }
  out[2] = log2_mpfr(worst);
  if (S0_api) {
    __mpfr_struct *S0 = vec_alloc((size_t)K, Pc);
    for (int j = 0; j < K; ++j) api_get(&S0[j], S0_api + (size_t)j * rb, prec, tmpP);
    mpfr_set_zero(worst, +1);
    for (int j = 0; j < K; ++j) { mpfr_sub(w, &S[j], &S0[j], RN); mpfr_abs(w, w, RN); if (mpfr_cmp(w, worst) > 0) mpfr_set(worst, w, RN); }
    out[0] = log2_mpfr(worst) - lF;
    if (U0_api && V0_api) {
      rmat U0 = rmat_alloc(M, K, Pc), V0 = rmat_alloc(N, K, Pc);
      load_rmat(&U0, U0_api, prec, tmpP); load_rmat(&V0, V0_api, prec, tmpP);
      /* stacked vectors (u; v), norm^2 = 2 */
      rmat Z = rmat_alloc(M + N, K, Pc), Z0 = rmat_alloc(M + N, K, Pc);
      for (int j = 0; j < K; ++j) {
        for (int i = 0; i < M; ++i) { mpfr_set(RRE(Z, i, j), RRE(U, i, j), RN); mpfr_set(RIM(Z, i, j), RIM(U, i, j), RN);
                                      mpfr_set(RRE(Z0, i, j), RRE(U0, i, j), RN); mpfr_set(RIM(Z0, i, j), RIM(U0, i, j), RN); }
        for (int i = 0; i < N; ++i) { mpfr_set(RRE(Z, M + i, j), RRE(V, i, j), RN); mpfr_set(RIM(Z, M + i, j), RIM(V, i, j), RN);
                                      mpfr_set(RRE(Z0, M + i, j), RRE(V0, i, j), RN); mpfr_set(RIM(Z0, M + i, j), RIM(V0, i, j), RN); }
      }
      /* scale the stacked vectors by 1/sqrt(2) so that proj_dist2's X0 X0^H is a projector */
      mpfr_set_ui(w, 2, RN); mpfr_sqrt(w, w, RN);
      for (size_t e = 0; e < (size_t)(M + N) * K; ++e) {
        mpfr_div(&Z.re[e], &Z.re[e], w, RN); mpfr_div(&Z.im[e], &Z.im[e], w, RN);
        mpfr_div(&Z0.re[e], &Z0.re[e], w, RN); mpfr_div(&Z0.im[e], &Z0.im[e], w, RN);
      }
      mpfr_t gthr, gap, g2, e2;
      mpfr_init2(gthr, Pc); mpfr_init2(gap, Pc); mpfr_init2(g2, Pc); mpfr_init2(e2, Pc);
      mpfr_div_2si(gthr, F, prec - 102, RN);
      int ng = 0, maxg = 0;
      double worst_margin = -1.0e9, worst_err = -1.0e9;
      int g0 = 0;
      while (g0 < K) {
        int g1 = g0 + 1;
        while (g1 < K) { mpfr_sub(w, &S0[g1 - 1], &S0[g1], RN); if (mpfr_cmp(w, gthr) > 0) break; ++g1; }
        ++ng; if (g1 - g0 > maxg) maxg = g1 - g0;
        const int zero_group = mpfr_cmp(&S0[g0], gthr) <= 0; /* its largest member is (numerically) zero */
        int have = 0;
        if (g0 > 0) { mpfr_sub(gap, &S0[g0 - 1], &S0[g0], RN); have = 1; }
        if (g1 < K) { mpfr_sub(g2, &S0[g1 - 1], &S0[g1], RN); if (!have || mpfr_cmp(g2, gap) < 0) mpfr_set(gap, g2, RN); have = 1; }
        double err;
        if (!zero_group) {
          mpfr_mul_2si(g2, &S0[g1 - 1], 1, RN); /* distance to the mirrored -sigma */
          if (!have || mpfr_cmp(g2, gap) < 0) mpfr_set(gap, g2, RN);
          have = 1;
          proj_dist2(e2, &Z, &Z0, g0, g1, Pc);
          mpfr_sqrt(e2, e2, RN);
          err = log2_mpfr(e2);
        } else {
          err = -1.0e9;
          if (N <= M) { proj_dist2(e2, &V, &V0, g0, g1, Pc); mpfr_sqrt(e2, e2, RN); if (log2_mpfr(e2) > err) err = log2_mpfr(e2); }
          if (M <= N) { proj_dist2(e2, &U, &U0, g0, g1, Pc); mpfr_sqrt(e2, e2, RN); if (log2_mpfr(e2) > err) err = log2_mpfr(e2); }
        }
        const double ltol = have ? (-(double)(prec - 38) + lF - log2_mpfr(gap)) : 1.0e9;
        if (err - ltol > worst_margin) worst_margin = err - ltol;
        if (err > worst_err) worst_err = err;
        g0 = g1;
      }
      out[3] = worst_margin; out[5] = ng; out[6] = maxg; out[7] = worst_err;
      mpfr_clear(gthr); mpfr_clear(gap); mpfr_clear(g2); mpfr_clear(e2);
      rmat_free(&U0); rmat_free(&V0); rmat_free(&Z); rmat_free(&Z0);
    }
    vec_free(S0, (size_t)K);
  }
  rmat_free(&A); rmat_free(&U); rmat_free(&V); vec_free(S, (size_t)K);
  mpfr_clear(tmpP); mpfr_clear(F); mpfr_clear(w); mpfr_clear(sr); mpfr_clear(si); mpfr_clear(acc); mpfr_clear(worst); mpfr_clear(t1);
  return 0;
}

/* ================================================================================================ */
/* Linear solve by Gaussian elimination (8(a) S4a')                           */
/* ================================================================================================ */
/* PAPER.md:31 (section 2): ZKCM_OMP's main routines include "Gaussian elimination, LU decomposition".  Result definition
 * (plain): X with A X = B for a nonsingular complex N x N matrix A and N x nrhs right-hand sides B.  Computed by the
 * textbook method at working precision P_o = prec + guard_bits:
 *   for k = 0 .. N-1: p = first row index >= k attaining max |a_ik|^2 (partial pivoting); swap rows k and p of A and B;
 *                     for i > k: l = a_ik / a_kk; row_i(A) -= l row_k(A) (columns > k); row_i(B) -= l row_k(B);
 *   back substitution: x_i = (b_i - sum_{j>i} a_ij x_j) / a_ii, i = N-1 .. 0;  round to prec bits.
 * Layout: A[i][j] (N x N), B[i][j], X[i][j] (N x nrhs) row-major complex API numbers.
 * Returns 0, 1 when a pivot is exactly zero (singular to working precision), 3 for malformed input.
 * Parity status: pinned (tests/test_oracle_lu_pins.py: 2 x 2 Cramer closed form, B = A X0 with chosen X0, residual, exact
 * permutation / diagonal / triangular cases, mpmath.lu_solve as a third opinion). */
int zkd_oracle_lu_solve(int N, int nrhs, int prec, int guard_bits, const uint8_t *A_api, const uint8_t *B_api, uint8_t *X_api) {
  const long Po = (long)prec + guard_bits;
  const size_t rb = api_real_bytes(prec);
  if (N < 1 || nrhs < 1 || prec < 64 || prec % 64) return 3;
  int status = 0;
  mpfr_t tmpP, best, m2, w, lr, li, dr, di, t1, t2;
  mpfr_init2(tmpP, prec); mpfr_init2(best, Po); mpfr_init2(m2, Po); mpfr_init2(w, Po); mpfr_init2(lr, Po); mpfr_init2(li, Po);
  mpfr_init2(dr, Po); mpfr_init2(di, Po); mpfr_init2(t1, Po); mpfr_init2(t2, Po);
  rmat A = rmat_alloc(N, N, Po), B = rmat_alloc(N, nrhs, Po);
  for (int i = 0; i < N && !status; ++i) {
    for (int j = 0; j < N; ++j) {
      const uint8_t *src = A_api + ((size_t)i * N + j) * 2 * rb;
      if (api_get(RRE(A, i, j), src, prec, tmpP) || api_get(RIM(A, i, j), src + rb, prec, tmpP)) { status = 3; break; }
    }
    for (int j = 0; j < nrhs && !status; ++j) {
      const uint8_t *src = B_api + ((size_t)i * nrhs + j) * 2 * rb;
      if (api_get(RRE(B, i, j), src, prec, tmpP) || api_get(RIM(B, i, j), src + rb, prec, tmpP)) { status = 3; break; }
    }
  }
  /* (x + i y) / (c + i d) = ((x c + y d) + i (y c - x d)) / (c^2 + d^2) */
#define CDIV(outr, outi, xr, xi, cr, ci)                                   \
  do {                                                                     \
    mpfr_sqr(t1, cr, RN); mpfr_sqr(t2, ci, RN); mpfr_add(w, t1, t2, RN);   \
    mpfr_fmma(t1, xr, cr, xi, ci, RN); mpfr_fmms(t2, xi, cr, xr, ci, RN);  \
    mpfr_div(outr, t1, w, RN); mpfr_div(outi, t2, w, RN);                  \
  } while (0)
  for (int k = 0; k < N && !status; ++k) {
    int p = k;
    mpfr_set_si(best, -1, RN);
    for (int i = k; i < N; ++i) {
      mpfr_sqr(m2, RRE(A, i, k), RN); mpfr_sqr(w, RIM(A, i, k), RN); mpfr_add(m2, m2, w, RN);
      if (mpfr_cmp(m2, best) > 0) { mpfr_set(best, m2, RN); p = i; }
    }
    if (mpfr_zero_p(best)) { status = 1; break; }
    if (p != k) {
      for (int j = 0; j < N; ++j) { mpfr_swap(RRE(A, k, j), RRE(A, p, j)); mpfr_swap(RIM(A, k, j), RIM(A, p, j)); }
      for (int j = 0; j < nrhs; ++j) { mpfr_swap(RRE(B, k, j), RRE(B, p, j)); mpfr_swap(RIM(B, k, j), RIM(B, p, j)); }
    }
    for (int i = k + 1; i < N; ++i) {
      CDIV(lr, li, RRE(A, i, k), RIM(A, i, k), RRE(A, k, k), RIM(A, k, k));
      for (int j = k + 1; j < N; ++j) {
        mpfr_fmms(t1, lr, RRE(A, k, j), li, RIM(A, k, j), RN); mpfr_sub(RRE(A, i, j), RRE(A, i, j), t1, RN);
        mpfr_fmma(t1, lr, RIM(A, k, j), li, RRE(A, k, j), RN); mpfr_sub(RIM(A, i, j), RIM(A, i, j), t1, RN);
      }
      for (int j = 0; j < nrhs; ++j) {
        mpfr_fmms(t1, lr, RRE(B, k, j), li, RIM(B, k, j), RN); mpfr_sub(RRE(B, i, j), RRE(B, i, j), t1, RN);
        mpfr_fmma(t1, lr, RIM(B, k, j), li, RRE(B, k, j), RN); mpfr_sub(RIM(B, i, j), RIM(B, i, j), t1, RN);
      }
      mpfr_set_zero(RRE(A, i, k), +1); mpfr_set_zero(RIM(A, i, k), +1);
    }
  }
  if (!status)
    for (int c = 0; c < nrhs; ++c)
      for (int i = N - 1; i >= 0; --i) {
        mpfr_set(dr, RRE(B, i, c), RN); mpfr_set(di, RIM(B, i, c), RN);
        for (int j = i + 1; j < N; ++j) {
          mpfr_fmms(t1, RRE(A, i, j), RRE(B, j, c), RIM(A, i, j), RIM(B, j, c), RN); mpfr_sub(dr, dr, t1, RN);
          mpfr_fmma(t1, RRE(A, i, j), RIM(B, j, c), RIM(A, i, j), RRE(B, j, c), RN); mpfr_sub(di, di, t1, RN);
        }
        CDIV(lr, li, dr, di, RRE(A, i, i), RIM(A, i, i));
        mpfr_set(RRE(B, i, c), lr, RN); mpfr_set(RIM(B, i, c), li, RN); /* x_i overwrites b_i */
      }
#undef CDIV
  if (!status)
    for (int i = 0; i < N; ++i)
      for (int j = 0; j < nrhs; ++j) {
        uint8_t *dst = X_api + ((size_t)i * nrhs + j) * 2 * rb;
        api_put(dst, RRE(B, i, j), prec, tmpP);
        api_put(dst + rb, RIM(B, i, j), prec, tmpP);
      }
  rmat_free(&A); rmat_free(&B);
  mpfr_clear(tmpP); mpfr_clear(best); mpfr_clear(m2); mpfr_clear(w); mpfr_clear(lr); mpfr_clear(li);
  mpfr_clear(dr); mpfr_clear(di); mpfr_clear(t1); mpfr_clear(t2);
  return status;
}

/* ================================================================================================ */
/* CPU restatement of the paper's own route: fp64 eigendecomposition + Rayleigh quotient iteration   */
/* ================================================================================================ */
/* PAPER.md:33 (section 2): "the Rayleigh quotient iteration was employed to recover the precision from the result of
 * double-precision calculations".  Used ONLY as a timed CPU baseline beside the GPU numbers (bench.py) and cross-checked
 * against the Jacobi oracle in tests/test_oracle_pins.py (P12); the checker of the CUDA path stays the Jacobi oracle.
 * For every eigenpair j in [first, first + count): start x = column j of the supplied fp64 eigenvector matrix; repeat `iters`
 * times: sigma = x^H A x (x has unit norm); solve (A - sigma I) y = x by Gaussian elimination with partial pivoting at
 * P_o = prec + guard_bits (a pivot that is exactly zero - sigma has converged to the working precision - is replaced by
 * 2^-P_o ||A||_F, the usual inverse-iteration safeguard); x = y / ||y||.  Output lambda_j = x^H A x and x, phase-normalised like
 * the Jacobi oracle (first component of largest modulus real positive).  Isolated eigenvalues only.
 *   max_pivots > 0: every elimination stops after that many pivot columns (bench sampling hook: the result is then
 *   meaningless; the caller extrapolates the time by the flop count sum_{k < max_pivots} (N-1-k)^2 / sum_{k < N-1} (N-1-k)^2).
 * OpenMP over eigenpairs.  Layout: V64[i][j] complex double, row-major (component i of vector j); lam_api[count],
 * X_api[i][c] (N x count) row-major complex API numbers.  Returns 0, or 3 for malformed input. */
int zkd_oracle_rqi(int N, int prec, int guard_bits, const uint8_t *A_api, const double *V64, int first, int count, int iters,
                   int max_pivots, int nthreads, uint8_t *lam_api, uint8_t *X_api) {
  const long Po = (long)prec + guard_bits;
  const size_t rb = api_real_bytes(prec);
  if (N < 1 || count < 1 || first < 0 || first + count > N || prec < 64 || prec % 64) return 3;
  if (nthreads < 1) nthreads = 1;
  int status = 0;
  mpfr_t tmpP0, F, w0;
  mpfr_init2(tmpP0, prec); mpfr_init2(F, Po); mpfr_init2(w0, Po);
  cmat A = cmat_alloc(N, Po);
  for (int i = 0; i < N && !status; ++i)
    for (int j = i; j < N; ++j) {
      const uint8_t *src = A_api + ((size_t)i * N + j) * 2 * rb;
      if (api_get(RE(A, i, j), src, prec, tmpP0) || api_get(IM(A, i, j), src + rb, prec, tmpP0)) { status = 3; break; }
      if (i == j) mpfr_set_zero(IM(A, i, j), +1);
      else { mpfr_set(RE(A, j, i), RE(A, i, j), RN); mpfr_neg(IM(A, j, i), IM(A, i, j), RN); }
    }
  mpfr_set_zero(F, +1);
  for (int i = 0; i < N && !status; ++i)
    for (int j = 0; j < N; ++j) {
      mpfr_sqr(w0, RE(A, i, j), RN); mpfr_add(F, F, w0, RN);
      mpfr_sqr(w0, IM(A, i, j), RN); mpfr_add(F, F, w0, RN);
    }
  mpfr_sqrt(F, F, RN);
  if (!status) {
#pragma omp parallel for num_threads(nthreads) schedule(dynamic, 1)
    for (int c = 0; c < count; ++c) {
      const int j = first + c;
      mpfr_t tmpP, sg, best, m2, w, lr, li, t1, t2, nr;
      mpfr_init2(tmpP, prec); mpfr_init2(sg, Po); mpfr_init2(best, Po); mpfr_init2(m2, Po); mpfr_init2(w, Po);
      mpfr_init2(lr, Po); mpfr_init2(li, Po); mpfr_init2(t1, Po); mpfr_init2(t2, Po); mpfr_init2(nr, Po);
      rmat M = rmat_alloc(N, N, Po), x = rmat_alloc(N, 1, Po), y = rmat_alloc(N, 1, Po);
      for (int i = 0; i < N; ++i) {
        mpfr_set_d(RRE(x, i, 0), V64[((size_t)i * N + j) * 2], RN);
        mpfr_set_d(RIM(x, i, 0), V64[((size_t)i * N + j) * 2 + 1], RN);
      }
      for (int it = 0; it <= iters; ++it) {
        /* unit norm, then sigma = x^H A x */
        col_dot(nr, w, &x, 0, 0, t1);
        mpfr_sqrt(nr, nr, RN);
        for (int i = 0; i < N; ++i) { mpfr_div(RRE(x, i, 0), RRE(x, i, 0), nr, RN); mpfr_div(RIM(x, i, 0), RIM(x, i, 0), nr, RN); }
        mpfr_set_zero(sg, +1);
        for (int i = 0; i < N; ++i) {
          mpfr_set_zero(lr, +1); mpfr_set_zero(li, +1); /* (A x)_i */
          for (int k = 0; k < N; ++k) {
            mpfr_fmms(t1, RE(A, i, k), RRE(x, k, 0), IM(A, i, k), RIM(x, k, 0), RN); mpfr_add(lr, lr, t1, RN);
            mpfr_fmma(t1, RE(A, i, k), RIM(x, k, 0), IM(A, i, k), RRE(x, k, 0), RN); mpfr_add(li, li, t1, RN);
          }
          mpfr_fmma(t1, RRE(x, i, 0), lr, RIM(x, i, 0), li, RN); /* Re conj(x_i) (A x)_i */
          mpfr_add(sg, sg, t1, RN);
        }
        if (it == iters) break;
        /* M = A - sigma I, y = x; Gaussian elimination with partial pivoting (same steps as zkd_oracle_lu_solve) */
        for (int i = 0; i < N; ++i) {
          for (int k = 0; k < N; ++k) { mpfr_set(RRE(M, i, k), RE(A, i, k), RN); mpfr_set(RIM(M, i, k), IM(A, i, k), RN); }
          mpfr_sub(RRE(M, i, i), RRE(M, i, i), sg, RN);
          mpfr_set(RRE(y, i, 0), RRE(x, i, 0), RN); mpfr_set(RIM(y, i, 0), RIM(x, i, 0), RN);
        }
#define CDIV2(outr, outi, xr, xi, cr, ci)                                  \
  do {                                                                     \
    mpfr_sqr(t1, cr, RN); mpfr_sqr(t2, ci, RN); mpfr_add(w, t1, t2, RN);   \
    mpfr_fmma(t1, xr, cr, xi, ci, RN); mpfr_fmms(t2, xi, cr, xr, ci, RN);  \
    mpfr_div(outr, t1, w, RN); mpfr_div(outi, t2, w, RN);                  \
  } while (0)
        const int kmax = (max_pivots > 0 && max_pivots < N) ? max_pivots : N;
        for (int k = 0; k < kmax; ++k) {
          int p = k;
          mpfr_set_si(best, -1, RN);
          for (int i = k; i < N; ++i) {
            mpfr_sqr(m2, RRE(M, i, k), RN); mpfr_sqr(w, RIM(M, i, k), RN); mpfr_add(m2, m2, w, RN);
            if (mpfr_cmp(m2, best) > 0) { mpfr_set(best, m2, RN); p = i; }
          }
          if (mpfr_zero_p(best)) { mpfr_div_2si(RRE(M, k, k), F, Po, RN); mpfr_set_zero(RIM(M, k, k), +1); p = k; }
          if (p != k) {
            for (int c2 = 0; c2 < N; ++c2) { mpfr_swap(RRE(M, k, c2), RRE(M, p, c2)); mpfr_swap(RIM(M, k, c2), RIM(M, p, c2)); }
            mpfr_swap(RRE(y, k, 0), RRE(y, p, 0)); mpfr_swap(RIM(y, k, 0), RIM(y, p, 0));
          }
          for (int i = k + 1; i < N; ++i) {
            CDIV2(lr, li, RRE(M, i, k), RIM(M, i, k), RRE(M, k, k), RIM(M, k, k));
            for (int c2 = k + 1; c2 < N; ++c2) {
              mpfr_fmms(t1, lr, RRE(M, k, c2), li, RIM(M, k, c2), RN); mpfr_sub(RRE(M, i, c2), RRE(M, i, c2), t1, RN);
              mpfr_fmma(t1, lr, RIM(M, k, c2), li, RRE(M, k, c2), RN); mpfr_sub(RIM(M, i, c2), RIM(M, i, c2), t1, RN);
            }
            mpfr_fmms(t1, lr, RRE(y, k, 0), li, RIM(y, k, 0), RN); mpfr_sub(RRE(y, i, 0), RRE(y, i, 0), t1, RN);
            mpfr_fmma(t1, lr, RIM(y, k, 0), li, RRE(y, k, 0), RN); mpfr_sub(RIM(y, i, 0), RIM(y, i, 0), t1, RN);
          }
        }
        if (kmax == N) {
          for (int i = N - 1; i >= 0; --i) {
            mpfr_set(lr, RRE(y, i, 0), RN); mpfr_set(li, RIM(y, i, 0), RN);
            for (int c2 = i + 1; c2 < N; ++c2) {
              mpfr_fmms(t1, RRE(M, i, c2), RRE(y, c2, 0), RIM(M, i, c2), RIM(y, c2, 0), RN); mpfr_sub(lr, lr, t1, RN);
              mpfr_fmma(t1, RRE(M, i, c2), RIM(y, c2, 0), RIM(M, i, c2), RRE(y, c2, 0), RN); mpfr_sub(li, li, t1, RN);
            }
            CDIV2(RRE(y, i, 0), RIM(y, i, 0), lr, li, RRE(M, i, i), RIM(M, i, i));
          }
          /* scale by 2^-exp of the largest component before the norm (y is huge once sigma has converged) */
          long emax = LONG_MIN;
          for (int i = 0; i < N; ++i) {
            if (!mpfr_zero_p(RRE(y, i, 0)) && mpfr_get_exp(RRE(y, i, 0)) > emax) emax = mpfr_get_exp(RRE(y, i, 0));
            if (!mpfr_zero_p(RIM(y, i, 0)) && mpfr_get_exp(RIM(y, i, 0)) > emax) emax = mpfr_get_exp(RIM(y, i, 0));
          }
          for (int i = 0; i < N; ++i) {
            mpfr_div_2si(RRE(x, i, 0), RRE(y, i, 0), emax, RN); mpfr_div_2si(RIM(x, i, 0), RIM(y, i, 0), emax, RN);
          }
        }
#undef CDIV2
      }
      /* output: lambda_j = sigma; x phase-normalised (first component of largest modulus real positive), unit norm */
      if (lam_api) api_put(lam_api + (size_t)c * rb, sg, prec, tmpP);
      if (X_api) {
        int kstar = 0;
        mpfr_set_si(best, -1, RN);
        for (int i = 0; i < N; ++i) {
          mpfr_sqr(m2, RRE(x, i, 0), RN); mpfr_sqr(w, RIM(x, i, 0), RN); mpfr_add(m2, m2, w, RN);
          if (mpfr_cmp(m2, best) > 0) { mpfr_set(best, m2, RN); kstar = i; }
        }
        mpfr_sqrt(best, best, RN);
        mpfr_div(lr, RRE(x, kstar, 0), best, RN); mpfr_div(li, RIM(x, kstar, 0), best, RN); mpfr_neg(li, li, RN);
        for (int i = 0; i < N; ++i) {
          mpfr_fmms(t1, RRE(x, i, 0), lr, RIM(x, i, 0), li, RN);
          mpfr_fmma(t2, RRE(x, i, 0), li, RIM(x, i, 0), lr, RN);
          if (i == kstar) mpfr_set_zero(t2, +1);
          uint8_t *dst = X_api + ((size_t)i * count + c) * 2 * rb;
          api_put(dst, t1, prec, tmpP);
          api_put(dst + rb, t2, prec, tmpP);
        }
      }
      rmat_free(&M); rmat_free(&x); rmat_free(&y);
      mpfr_clear(tmpP); mpfr_clear(sg); mpfr_clear(best); mpfr_clear(m2); mpfr_clear(w); mpfr_clear(lr); mpfr_clear(li);
      mpfr_clear(t1); mpfr_clear(t2); mpfr_clear(nr);
    }
  }
  cmat_free(&A);
  mpfr_clear(tmpP0); mpfr_clear(F); mpfr_clear(w0);
  return status;
}
