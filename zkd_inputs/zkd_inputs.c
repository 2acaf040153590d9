/* zkd_inputs/zkd_inputs.c — seeded synthetic input generators (shared by tests of the oracle and of the CUDA path).
 *
 * Holds none of the method's arithmetic: no eigensolver, no refinement, no comparison.  It only *builds inputs*:
 *   (1) N x N complex Hermitian matrices "with random elements", elements uniform[-1,1]
 *       with all 768 mantissa bits random (reading A2);
 *   (2) A = Q diag(lambda) Q^H with Q a product of R seeded 768-bit Householder reflectors and a chosen
 *       spectrum (BASELINE.json configs 4 and 5; readings A12-A14), formed at prec+256 bits with
 *       MPFR and rounded to prec, so that lambda and the columns of Q are the answer *by construction*.
 *
 * Random bits: a counter-based generator, word(seed, stream, idx) = splitmix64 finaliser of a linear
 * combination of the three; no state, so any element can be regenerated independently.
 *
 * API number layout (restated): int32 sign; int32 flags=0; int64 exp; uint64 limb[prec/64] LE;
 * value = sign * limbs * 2^(exp-prec); top bit of the top limb set when nonzero.
 *
 * MPFR is linked through hand-declared prototypes (the image has libmpfr.so.6 but no mpfr.h).
 */
#include <limits.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

/* ---- MPFR interface declaration (this module's own copy; nothing is shared with oracle/ or the CUDA path) ---- */
typedef long mpfr_prec_t;
typedef int mpfr_sign_t;
typedef long mpfr_exp_t;
typedef unsigned long mp_limb_t;
typedef struct { mpfr_prec_t _mpfr_prec; mpfr_sign_t _mpfr_sign; mpfr_exp_t _mpfr_exp; mp_limb_t *_mpfr_d; } __mpfr_struct;
typedef __mpfr_struct mpfr_t[1];
typedef __mpfr_struct *mpfr_ptr;
typedef const __mpfr_struct *mpfr_srcptr;
typedef enum { MPFR_RNDN = 0 } mpfr_rnd_t;
void mpfr_init2(mpfr_ptr, mpfr_prec_t);
void mpfr_clear(mpfr_ptr);
int mpfr_set(mpfr_ptr, mpfr_srcptr, mpfr_rnd_t);
int mpfr_set_ui(mpfr_ptr, unsigned long, mpfr_rnd_t);
void mpfr_set_zero(mpfr_ptr, int);
int mpfr_add(mpfr_ptr, mpfr_srcptr, mpfr_srcptr, mpfr_rnd_t);
int mpfr_sub(mpfr_ptr, mpfr_srcptr, mpfr_srcptr, mpfr_rnd_t);
int mpfr_mul(mpfr_ptr, mpfr_srcptr, mpfr_srcptr, mpfr_rnd_t);
int mpfr_sqr(mpfr_ptr, mpfr_srcptr, mpfr_rnd_t);
int mpfr_neg(mpfr_ptr, mpfr_srcptr, mpfr_rnd_t);
int mpfr_ui_div(mpfr_ptr, unsigned long, mpfr_srcptr, mpfr_rnd_t);
int mpfr_fmma(mpfr_ptr, mpfr_srcptr, mpfr_srcptr, mpfr_srcptr, mpfr_srcptr, mpfr_rnd_t);
int mpfr_fmms(mpfr_ptr, mpfr_srcptr, mpfr_srcptr, mpfr_srcptr, mpfr_srcptr, mpfr_rnd_t);
int mpfr_sgn(mpfr_srcptr);
int mpfr_zero_p(mpfr_srcptr);
mpfr_exp_t mpfr_get_exp(mpfr_srcptr);
#define RN MPFR_RNDN

static size_t rbytes(int prec) { return 16 + (size_t)prec / 8; }

/* ---- counter-based generator ---- */
static uint64_t mix64(uint64_t z) {
  z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ULL;
  z = (z ^ (z >> 27)) * 0x94D049BB133111EBULL;
  return z ^ (z >> 31);
}
uint64_t zkd_inputs_word(uint64_t seed, uint64_t stream, uint64_t idx) {
  return mix64(mix64(seed * 0x9E3779B97F4A7C15ULL + 0x632BE59BD9B4E019ULL) ^ mix64(stream * 0xD1342543DE82EF95ULL + 0x2545F4914F6CDD1DULL) ^
               (idx * 0x9E3779B97F4A7C15ULL + 0x1234567887654321ULL));
}

/* One uniform[-1,1) real with every mantissa bit random: value = (U - 2^(prec-1)) / 2^(prec-1), U a uniform
 * prec-bit integer drawn most-significant word first from counters idx0 .. idx0 + prec/64 - 1. */
static void uniform_real(uint8_t *dst, int prec, uint64_t seed, uint64_t stream, uint64_t idx0) {
  int L = prec / 64;
  uint64_t m[64];
  for (int k = 0; k < L; ++k) m[L - 1 - k] = zkd_inputs_word(seed, stream, idx0 + (uint64_t)k);
  int32_t sign;
  /* mag = |U - 2^(prec-1)| */
  if (m[L - 1] >> 63) {
    sign = 1;
    m[L - 1] &= ~(1ULL << 63);
  } else {
    sign = -1; /* mag = 2^(prec-1) - U: two's complement negate of U within prec bits, then clear... */
    uint64_t carry = 1;
    for (int k = 0; k < L; ++k) {
      uint64_t v = ~m[k] + carry;
      carry = (carry && v == 0) ? 1 : 0;
      m[k] = v;
    } /* m = 2^prec - U ; subtract 2^(prec-1) */
    m[L - 1] -= (1ULL << 63);
  }
  int allz = 1;
  for (int k = 0; k < L; ++k) if (m[k]) allz = 0;
  memset(dst, 0, rbytes(prec));
  if (allz) return;
  /* normalise */
  int sh = 0;
  while (!(m[L - 1] >> 63)) {
    int lw = 0;
    if (m[L - 1] == 0) { /* whole-limb shift */
      for (int k = L - 1; k > 0; --k) m[k] = m[k - 1];
      m[0] = 0; sh += 64; lw = 1;
    }
    if (!lw) {
      int z = __builtin_clzll(m[L - 1]);
      for (int k = L - 1; k > 0; --k) m[k] = (m[k] << z) | (m[k - 1] >> (64 - z));
      m[0] <<= z; sh += z;
    }
  }
  int64_t e = 1 - (int64_t)sh; /* value = mant * 2^(-sh-(prec-1)) = mant * 2^(e-prec) */
  memcpy(dst, &sign, 4);
  memcpy(dst + 8, &e, 8);
  memcpy(dst + 16, m, 8 * (size_t)L);
}

/* Hermitian matrix with random elements (reading A2).  Draw order: for i: a_ii, then for j>i:
 * Re a_ij, Im a_ij.  A[j][i] = conj(A[i][j]); Im a_ii = 0. */
int zkd_inputs_random_herm(int N, int prec, uint64_t seed, uint64_t stream, uint8_t *A_api) {
  if (N < 1 || prec < 64 || prec % 64 || prec > 4096) return -1;
  size_t rb = rbytes(prec);
  uint64_t L = (uint64_t)prec / 64, ctr = 0;
  for (int i = 0; i < N; ++i) {
    uint8_t *d = A_api + ((size_t)i * N + i) * 2 * rb;
    uniform_real(d, prec, seed, stream, ctr); ctr += L;
    memset(d + rb, 0, rb);
    for (int j = i + 1; j < N; ++j) {
      uint8_t *u = A_api + ((size_t)i * N + j) * 2 * rb, *l = A_api + ((size_t)j * N + i) * 2 * rb;
      uniform_real(u, prec, seed, stream, ctr); ctr += L;
      uniform_real(u + rb, prec, seed, stream, ctr); ctr += L;
      memcpy(l, u, 2 * rb);
      int32_t s;
      memcpy(&s, l + rb, 4); s = -s; memcpy(l + rb, &s, 4);
    }
  }
  return 0;
}

/* ---- API <-> MPFR (this module's own) ---- */
static void get_api(mpfr_ptr dst, const uint8_t *src, int prec, mpfr_ptr tmpP) {
  int32_t sign; int64_t e;
  memcpy(&sign, src, 4); memcpy(&e, src + 8, 8);
  if (sign == 0) { mpfr_set_zero(dst, +1); return; }
  memcpy(tmpP->_mpfr_d, src + 16, (size_t)prec / 8);
  tmpP->_mpfr_sign = sign; tmpP->_mpfr_exp = (mpfr_exp_t)e;
  mpfr_set(dst, tmpP, RN);
}
static void put_api(uint8_t *dst, mpfr_srcptr src, int prec, mpfr_ptr tmpP) {
  memset(dst, 0, rbytes(prec));
  mpfr_set(tmpP, src, RN);
  if (mpfr_zero_p(tmpP)) return;
  int32_t sign = mpfr_sgn(tmpP) < 0 ? -1 : 1; int64_t e = (int64_t)mpfr_get_exp(tmpP);
  memcpy(dst, &sign, 4); memcpy(dst + 8, &e, 8); memcpy(dst + 16, tmpP->_mpfr_d, (size_t)prec / 8);
}

/* A = Q diag(lambda) Q^H, Q = H_1 ... H_R, H_r = I - 2 u_r u_r^H / (u_r^H u_r), u_r in C^N with Re/Im
 * uniform[-1,1) at prec bits drawn from (seed, stream*65536 + r).  Reflectors are applied two-sidedly to
 * diag(lambda) (r = R..1) at prec+256 bits; the upper triangle is rounded to prec bits and mirrored.
 * Q_api (optional) receives Q rounded to prec bits: its columns are the eigenvectors by construction. */
int zkd_inputs_qdq(int N, int prec, uint64_t seed, uint64_t stream, int R, const uint8_t *lambda_api, uint8_t *A_api,
                   uint8_t *Q_api) {
  if (N < 1 || prec < 64 || prec % 64 || prec > 4096 || R < 0) return -1;
  const long Pw = (long)prec + 256;
  size_t rb = rbytes(prec), nn = (size_t)N * N;
  mpfr_t tmpP, tau, t1, t2, sr, si;
  mpfr_init2(tmpP, prec); mpfr_init2(tau, Pw); mpfr_init2(t1, Pw); mpfr_init2(t2, Pw); mpfr_init2(sr, Pw); mpfr_init2(si, Pw);
  __mpfr_struct *Mr = malloc(nn * sizeof *Mr), *Mi = malloc(nn * sizeof *Mi), *Qr = NULL, *Qi = NULL;
  __mpfr_struct *ur = malloc((size_t)N * sizeof *ur), *ui = malloc((size_t)N * sizeof *ui);
  __mpfr_struct *pr = malloc((size_t)N * sizeof *pr), *pi = malloc((size_t)N * sizeof *pi);
  for (size_t k = 0; k < nn; ++k) { mpfr_init2(&Mr[k], Pw); mpfr_init2(&Mi[k], Pw); mpfr_set_zero(&Mr[k], 1); mpfr_set_zero(&Mi[k], 1); }
  if (Q_api) {
    Qr = malloc(nn * sizeof *Qr); Qi = malloc(nn * sizeof *Qi);
    for (size_t k = 0; k < nn; ++k) { mpfr_init2(&Qr[k], Pw); mpfr_init2(&Qi[k], Pw); mpfr_set_zero(&Qr[k], 1); mpfr_set_zero(&Qi[k], 1); }
    for (int i = 0; i < N; ++i) mpfr_set_ui(&Qr[(size_t)i * N + i], 1, RN);
  }
  for (int i = 0; i < N; ++i) { mpfr_init2(&ur[i], Pw); mpfr_init2(&ui[i], Pw); mpfr_init2(&pr[i], Pw); mpfr_init2(&pi[i], Pw); }
  for (int i = 0; i < N; ++i) get_api(&Mr[(size_t)i * N + i], lambda_api + (size_t)i * rb, prec, tmpP);

  uint8_t *buf = malloc(rb);
  for (int r = R; r >= 1; --r) {
    uint64_t st = stream * 65536ULL + (uint64_t)r, L = (uint64_t)prec / 64;
    mpfr_set_zero(t1, 1);
    for (int i = 0; i < N; ++i) {
      uniform_real(buf, prec, seed, st, (uint64_t)(2 * i) * L); get_api(&ur[i], buf, prec, tmpP);
      uniform_real(buf, prec, seed, st, (uint64_t)(2 * i + 1) * L); get_api(&ui[i], buf, prec, tmpP);
      mpfr_sqr(t2, &ur[i], RN); mpfr_add(t1, t1, t2, RN);
      mpfr_sqr(t2, &ui[i], RN); mpfr_add(t1, t1, t2, RN);
    }
    mpfr_ui_div(tau, 2, t1, RN); /* tau = 2 / (u^H u) */
    /* M <- M H :  p = M u ; M -= tau p u^H */
    for (int pass = 0; pass < (Q_api ? 3 : 2); ++pass) {
      /* pass 0: M <- M H.  pass 1: M <- H M.  pass 2: Q <- H Q. */
      __mpfr_struct *Xr = pass == 2 ? Qr : Mr, *Xi = pass == 2 ? Qi : Mi;
      if (pass == 0) {
#pragma omp parallel for
        for (int i = 0; i < N; ++i) { /* p_i = sum_k M_ik u_k */
          mpfr_t a, b, c, d;
          mpfr_init2(a, Pw); mpfr_init2(b, Pw); mpfr_init2(c, Pw); mpfr_init2(d, Pw);
          mpfr_set_zero(a, 1); mpfr_set_zero(b, 1);
          for (int k = 0; k < N; ++k) {
            mpfr_fmms(c, &Xr[(size_t)i * N + k], &ur[k], &Xi[(size_t)i * N + k], &ui[k], RN);
            mpfr_fmma(d, &Xr[(size_t)i * N + k], &ui[k], &Xi[(size_t)i * N + k], &ur[k], RN);
            mpfr_add(a, a, c, RN); mpfr_add(b, b, d, RN);
          }
          mpfr_mul(&pr[i], a, tau, RN); mpfr_mul(&pi[i], b, tau, RN); /* tau p */
          mpfr_clear(a); mpfr_clear(b); mpfr_clear(c); mpfr_clear(d);
        }
#pragma omp parallel for
        for (int i = 0; i < N; ++i) { /* M_ij -= (tau p_i) conj(u_j) */
          mpfr_t c, d;
          mpfr_init2(c, Pw); mpfr_init2(d, Pw);
          for (int j = 0; j < N; ++j) {
            mpfr_fmma(c, &pr[i], &ur[j], &pi[i], &ui[j], RN); /* Re p conj(u) */
            mpfr_fmms(d, &pi[i], &ur[j], &pr[i], &ui[j], RN); /* Im p conj(u) */
            mpfr_sub(&Xr[(size_t)i * N + j], &Xr[(size_t)i * N + j], c, RN);
            mpfr_sub(&Xi[(size_t)i * N + j], &Xi[(size_t)i * N + j], d, RN);
          }
          mpfr_clear(c); mpfr_clear(d);
        }
      } else {
#pragma omp parallel for
        for (int j = 0; j < N; ++j) { /* q_j = sum_k conj(u_k) X_kj */
          mpfr_t a, b, c, d;
          mpfr_init2(a, Pw); mpfr_init2(b, Pw); mpfr_init2(c, Pw); mpfr_init2(d, Pw);
          mpfr_set_zero(a, 1); mpfr_set_zero(b, 1);
          for (int k = 0; k < N; ++k) {
            mpfr_fmma(c, &ur[k], &Xr[(size_t)k * N + j], &ui[k], &Xi[(size_t)k * N + j], RN);
            mpfr_fmms(d, &ur[k], &Xi[(size_t)k * N + j], &ui[k], &Xr[(size_t)k * N + j], RN);
            mpfr_add(a, a, c, RN); mpfr_add(b, b, d, RN);
          }
          mpfr_mul(&pr[j], a, tau, RN); mpfr_mul(&pi[j], b, tau, RN); /* tau q */
          mpfr_clear(a); mpfr_clear(b); mpfr_clear(c); mpfr_clear(d);
        }
#pragma omp parallel for
        for (int i = 0; i < N; ++i) { /* X_ij -= u_i (tau q_j) */
          mpfr_t c, d;
          mpfr_init2(c, Pw); mpfr_init2(d, Pw);
          for (int j = 0; j < N; ++j) {
            mpfr_fmms(c, &ur[i], &pr[j], &ui[i], &pi[j], RN);
            mpfr_fmma(d, &ur[i], &pi[j], &ui[i], &pr[j], RN);
            mpfr_sub(&Xr[(size_t)i * N + j], &Xr[(size_t)i * N + j], c, RN);
            mpfr_sub(&Xi[(size_t)i * N + j], &Xi[(size_t)i * N + j], d, RN);
          }
          mpfr_clear(c); mpfr_clear(d);
        }
      }
    }
  }
  for (int i = 0; i < N; ++i) {
    uint8_t *d = A_api + ((size_t)i * N + i) * 2 * rb;
    put_api(d, &Mr[(size_t)i * N + i], prec, tmpP); memset(d + rb, 0, rb);
    for (int j = i + 1; j < N; ++j) {
      uint8_t *u = A_api + ((size_t)i * N + j) * 2 * rb, *l = A_api + ((size_t)j * N + i) * 2 * rb;
      put_api(u, &Mr[(size_t)i * N + j], prec, tmpP); put_api(u + rb, &Mi[(size_t)i * N + j], prec, tmpP);
      memcpy(l, u, 2 * rb);
      int32_t s; memcpy(&s, l + rb, 4); s = -s; memcpy(l + rb, &s, 4);
    }
  }
  if (Q_api)
    for (size_t k = 0; k < nn; ++k) { put_api(Q_api + k * 2 * rb, &Qr[k], prec, tmpP); put_api(Q_api + k * 2 * rb + rb, &Qi[k], prec, tmpP); }

  free(buf);
  for (size_t k = 0; k < nn; ++k) { mpfr_clear(&Mr[k]); mpfr_clear(&Mi[k]); if (Q_api) { mpfr_clear(&Qr[k]); mpfr_clear(&Qi[k]); } }
  for (int i = 0; i < N; ++i) { mpfr_clear(&ur[i]); mpfr_clear(&ui[i]); mpfr_clear(&pr[i]); mpfr_clear(&pi[i]); }
  free(Mr); free(Mi); free(Qr); free(Qi); free(ur); free(ui); free(pr); free(pi);
  mpfr_clear(tmpP); mpfr_clear(tau); mpfr_clear(t1); mpfr_clear(t2); mpfr_clear(sr); mpfr_clear(si);
  return 0;
}

/* one uniform real, exported for tests of the generator itself */
void zkd_inputs_uniform_real(uint8_t *dst, int prec, uint64_t seed, uint64_t stream, uint64_t idx0) {
  uniform_real(dst, prec, seed, stream, idx0);
}
