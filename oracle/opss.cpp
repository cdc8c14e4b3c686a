/*
 * opss.cpp — CPU ORACLE for the semi-implicit pseudo-spectral SPDE step of cuPSS
 * (arXiv 2405.02410).  TEST INFRASTRUCTURE ONLY — see opss.h for who may load it.
 *
 * Written from PAPER.md alone; plain double arithmetic (std::complex<double>), its own
 * recursive radix-2 FFT, its own Philox4x32-10.  No blocking, fusion or reordering: one time
 * step is the paper's list executed in that order, each nonlinear term
 * transformed separately exactly as Eq. 15 is written.  OpenMP is used only over
 * independent 1-D transform lines and over independent modes/sites of pointwise loops.
 *
 * Readings of silent/ambiguous points (A1..A20) are those of DESIGN.md section "Readings".
 *
 * parity unpinned: the active-nematic workload (BASELINE config 4) has no equations in the
 * paper; only the invariants listed in DESIGN.md (P12) pin it.
 */
#include "opss.h"

#include <cmath>
#include <complex>
#include <cstdio>
#include <cstring>
#include <string>
#include <vector>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef std::complex<double> cplx;
static const long double PI_L = 3.14159265358979323846264338327950288L;
static const double PI_D = 3.14159265358979323846;

/* ------------------------------------------------------------------------------------------
 * FFT: textbook recursive decimation-in-time radix-2 (even/odd split), unnormalised.
 *   X[k] = sum_n x[n] exp(sign * 2 pi i n k / N)
 * tw[j] = exp(sign * 2 pi i j / N) for j < N/2, from long-double cos/sin.
 * ------------------------------------------------------------------------------------------ */
static void make_twiddles(std::vector<cplx> &tw, int64_t n, int sign) {
  tw.resize(n / 2 > 0 ? n / 2 : 1);
  for (int64_t j = 0; j < n / 2; ++j) {
    long double a = 2.0L * PI_L * (long double)j / (long double)n;
    tw[j] = cplx((double)cosl(a), (double)(sign * sinl(a)));
  }
}

/* out[0..n) = DFT of in[0], in[stride], in[2 stride], ...  (tw is the table for length N_top,
 * tws = N_top / n its stride for this level) */
static void fft_rec(const cplx *in, int64_t stride, cplx *out, int64_t n, const cplx *tw,
                    int64_t tws) {
  if (n == 1) {
    out[0] = in[0];
    return;
  }
  const int64_t h = n / 2;
  fft_rec(in, 2 * stride, out, h, tw, 2 * tws);              /* even samples */
  fft_rec(in + stride, 2 * stride, out + h, h, tw, 2 * tws); /* odd samples  */
  for (int64_t k = 0; k < h; ++k) {
    const cplx e = out[k];
    const cplx t = tw[k * tws] * out[k + h];
    out[k] = e + t;
    out[k + h] = e - t;
  }
}

static bool is_pow2(int64_t n) { return n >= 1 && (n & (n - 1)) == 0; }

/* transform `count` lines in place; line l starts at base(l) = (l / inner) * outer_stride +
 * (l % inner) * 1 ... expressed by the caller through a lambda-free (start, stride) table */
struct LineSet {
  int64_t n;       /* line length          */
  int64_t stride;  /* element stride       */
  int64_t count;   /* number of lines      */
  int64_t inner;   /* lines per outer block */
  int64_t inner_step, outer_step; /* start = (l % inner) * inner_step + (l / inner) * outer_step */
};

static void fft_lines(cplx *data, const LineSet &ls, int sign, int nthreads) {
  if (ls.n == 1) return;
  std::vector<cplx> tw;
  make_twiddles(tw, ls.n, sign);
#pragma omp parallel num_threads(nthreads)
  {
    std::vector<cplx> tmp(ls.n);
#pragma omp for schedule(static)
    for (int64_t l = 0; l < ls.count; ++l) {
      cplx *p = data + (l % ls.inner) * ls.inner_step + (l / ls.inner) * ls.outer_step;
      fft_rec(p, ls.stride, tmp.data(), ls.n, tw.data(), 1);
      for (int64_t k = 0; k < ls.n; ++k) p[k * ls.stride] = tmp[k];
    }
  }
}

struct Dims {
  int ndim;
  int64_t n[3];  /* padded with 1 */
  int64_t nxh;   /* n[0]/2 + 1    */
  int64_t nsites() const { return n[0] * n[1] * n[2]; }
  int64_t nmodes() const { return nxh * n[1] * n[2]; }
};

/* R2C: forward DFT of a real array, keep kx = 0..Nx/2 (unnormalised).  x is transformed as a
 * full complex line of the real data; y and z as complex lines of the half-spectrum. */
static void r2c(const std::vector<double> &re, std::vector<cplx> &half, const Dims &d, int nth) {
  const int64_t nx = d.n[0], ny = d.n[1], nz = d.n[2], nxh = d.nxh;
  half.assign(d.nmodes(), cplx(0, 0));
  std::vector<cplx> tw;
  make_twiddles(tw, nx, -1);
#pragma omp parallel num_threads(nth)
  {
    std::vector<cplx> in(nx), out(nx);
#pragma omp for schedule(static)
    for (int64_t l = 0; l < ny * nz; ++l) {
      for (int64_t x = 0; x < nx; ++x) in[x] = cplx(re[l * nx + x], 0.0);
      fft_rec(in.data(), 1, out.data(), nx, tw.data(), 1);
      for (int64_t k = 0; k < nxh; ++k) half[l * nxh + k] = out[k];
    }
  }
  if (d.ndim >= 2) {
    LineSet ls = {ny, nxh, nxh * nz, nxh, 1, nxh * ny};
    fft_lines(half.data(), ls, -1, nth);
  }
  if (d.ndim >= 3) {
    LineSet ls = {nz, nxh * ny, nxh * ny, nxh * ny, 1, 0};
    fft_lines(half.data(), ls, -1, nth);
  }
}

/* C2R: inverse of the above, including the 1/N.  Along x the half line is extended by
 * X[Nx-k] = conj X[k] (0 < k < Nx/2), transformed as a full complex line, and the real part kept. */
static void c2r(const std::vector<cplx> &half_in, std::vector<double> &re, const Dims &d, int nth) {
  const int64_t nx = d.n[0], ny = d.n[1], nz = d.n[2], nxh = d.nxh;
  std::vector<cplx> half(half_in);
  if (d.ndim >= 3) {
    LineSet ls = {nz, nxh * ny, nxh * ny, nxh * ny, 1, 0};
    fft_lines(half.data(), ls, +1, nth);
  }
  if (d.ndim >= 2) {
    LineSet ls = {ny, nxh, nxh * nz, nxh, 1, nxh * ny};
    fft_lines(half.data(), ls, +1, nth);
  }
  re.assign(d.nsites(), 0.0);
  std::vector<cplx> tw;
  make_twiddles(tw, nx, +1);
  const double inv = 1.0 / (double)d.nsites();
#pragma omp parallel num_threads(nth)
  {
    std::vector<cplx> in(nx), out(nx);
#pragma omp for schedule(static)
    for (int64_t l = 0; l < ny * nz; ++l) {
      for (int64_t k = 0; k < nxh; ++k) in[k] = half[l * nxh + k];
      for (int64_t k = 1; k < nx - nxh + 1; ++k) in[nx - k] = std::conj(half[l * nxh + k]);
      fft_rec(in.data(), 1, out.data(), nx, tw.data(), 1);
      for (int64_t x = 0; x < nx; ++x) re[l * nx + x] = out[x].real() * inv;
    }
  }
}

/* ------------------------------------------------------------------------------------------
 * Philox4x32-10 (Salmon, Moraes, Dror, Shaw, SC'11), from the published constants.
 * ------------------------------------------------------------------------------------------ */
static void philox4x32_10(const uint32_t c_in[4], const uint32_t k_in[2], uint32_t out[4]) {
  const uint32_t M0 = 0xD2511F53u, M1 = 0xCD9E8D57u, W0 = 0x9E3779B9u, W1 = 0xBB67AE85u;
  uint32_t c0 = c_in[0], c1 = c_in[1], c2 = c_in[2], c3 = c_in[3];
  uint32_t k0 = k_in[0], k1 = k_in[1];
  for (int r = 0; r < 10; ++r) {
    const uint64_t p0 = (uint64_t)M0 * c0;
    const uint64_t p1 = (uint64_t)M1 * c2;
    const uint32_t hi0 = (uint32_t)(p0 >> 32), lo0 = (uint32_t)p0;
    const uint32_t hi1 = (uint32_t)(p1 >> 32), lo1 = (uint32_t)p1;
    const uint32_t n0 = hi1 ^ c1 ^ k0;
    const uint32_t n1 = lo1;
    const uint32_t n2 = hi0 ^ c3 ^ k1;
    const uint32_t n3 = lo0;
    c0 = n0; c1 = n1; c2 = n2; c3 = n3;
    k0 += W0; k1 += W1;
  }
  out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

/* ------------------------------------------------------------------------------------------
 * The field system: dynamic fields with an implicit operator L_i, auxiliary
 * ("intermediate") fields defined as operators applied to other fields, a list of rhs terms.
 * ------------------------------------------------------------------------------------------ */
struct Def { opss_op op; int src; };
struct ATerm { opss_op outer; std::vector<int> factors; };
struct Frame { int axis; int64_t lo_w, hi_w; double lo_v, hi_v; };
struct Field {
  std::string name;
  bool dynamic;
  std::vector<Def> defs;      /* aux only: psi_q = sum coef Op(q) src_q          */
  std::vector<opss_op> alhs;  /* aux only: its own lhs, den(q) psi_q = rhs; empty = the bare field */
  std::vector<ATerm> aterms;  /* aux only: rhs terms that are products of fields                  */
  std::vector<opss_op> lhs;   /* dynamic only: dt phi + sum coef Op(q) phi = rhs */
  bool noisy; double D; int qpow;
  std::vector<Frame> frames;  /* dynamic only: Dirichlet buffer zones set at the end of every step */
  std::vector<cplx> hat;      /* half-spectrum, unnormalised forward DFT         */
};
struct Term { int field; opss_op outer; std::vector<int> factors; };

struct opss_system {
  Dims d;
  double dx[3];
  double dt;
  int prec;
  uint64_t seed;
  int dealias;
  int nthreads;
  bool finalized;
  uint64_t step;
  std::vector<Field> fields;
  std::vector<Term> terms;
};

static int max_threads() {
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}

static bool op_ok(const opss_system *s, const opss_op *op) {
  if (!op) return false;
  if (op->q2_pow < 0 || op->invq_pow < 0) return false;
  for (int j = 0; j < 3; ++j) {
    if (op->iq_pow[j] < 0) return false;
    if (j >= s->d.ndim && op->iq_pow[j] != 0) return false;
  }
  return std::isfinite(op->coef);
}

static inline int64_t signed_index(int64_t k, int64_t n) { return (k <= n / 2) ? k : k - n; }

/* q_j = 2 pi s(k_j) / (N_j dx_j)  (Delta q = 2 pi / (N Delta x)) */
static inline double qcomp(const opss_system *s, int j, int64_t k) {
  if (j >= s->d.ndim) return 0.0;
  return 2.0 * PI_D * (double)signed_index(k, s->d.n[j]) / ((double)s->d.n[j] * s->dx[j]);
}

/* Op(k) = coef (q^2)^m |q|^-p prod_j (i q_j)^a_j ;  |q|^-p := 0 at q = 0 (A10);
 * a monomial with odd a_j vanishes at the Nyquist index k_j = N_j/2 (A9). */
static cplx op_eval(const opss_system *s, const opss_op &op, const int64_t k[3]) {
  double q[3], q2 = 0.0;
  for (int j = 0; j < 3; ++j) { q[j] = qcomp(s, j, k[j]); q2 += q[j] * q[j]; }
  for (int j = 0; j < s->d.ndim; ++j)
    if ((op.iq_pow[j] & 1) && s->d.n[j] > 1 && k[j] == s->d.n[j] / 2) return cplx(0, 0);
  cplx v(op.coef, 0.0);
  for (int i = 0; i < op.q2_pow; ++i) v *= q2;
  if (op.invq_pow > 0) {
    if (q2 == 0.0) return cplx(0, 0);
    const double inv = 1.0 / std::sqrt(q2);
    for (int i = 0; i < op.invq_pow; ++i) v *= inv;
  }
  for (int j = 0; j < 3; ++j)
    for (int i = 0; i < op.iq_pow[j]; ++i) v *= cplx(0.0, q[j]);
  return v;
}

static inline void mode_of(const Dims &d, int64_t m, int64_t k[3]) {
  k[0] = m % d.nxh;
  k[1] = (m / d.nxh) % d.n[1];
  k[2] = m / (d.nxh * d.n[1]);
}
static inline int64_t index_of(const Dims &d, const int64_t k[3]) {
  return (k[2] * d.n[1] + k[1]) * d.nxh + k[0];
}

/* highest order of a product (>= 2 factors) the field takes part in; 0 if none */
static int max_order(const opss_system *s, int f) {
  int nmax = 0;
  for (const Term &t : s->terms) {
    if (t.factors.size() < 2) continue;
    for (int g : t.factors)
      if (g == f && (int)t.factors.size() > nmax) nmax = (int)t.factors.size();
  }
  /* products that define intermediate fields count as well ("fields that form part of nonlinearities") */
  for (const Field &F : s->fields)
    for (const ATerm &t : F.aterms) {
      if (t.factors.size() < 2) continue;
      for (int g : t.factors)
        if (g == f && (int)t.factors.size() > nmax) nmax = (int)t.factors.size();
    }
  return nmax;
}

/* keep iff (n+1) |s(k_j)| < N_j on every axis (readings A4, A5, A6) */
static bool keep_mode(const opss_system *s, int order, const int64_t k[3]) {
  if (s->dealias == OPSS_DEALIAS_OFF) return true;
  const int n = (s->dealias == OPSS_DEALIAS_TWO_THIRDS) ? 2 : order;
  for (int j = 0; j < s->d.ndim; ++j) {
    int64_t a = signed_index(k[j], s->d.n[j]);
    if (a < 0) a = -a;
    if ((int64_t)(n + 1) * a >= s->d.n[j]) return false;
  }
  return true;
}

/* ------------------------------------------------------------------------------------------
 * Noise (Eq. 16, 134, 194; readings A1, A13 and the generator of DESIGN.md).
 * ------------------------------------------------------------------------------------------ */
static void noise_block(const opss_system *s, int field, uint64_t step, int64_t m, uint32_t w[4]) {
  const uint32_t ctr[4] = {(uint32_t)((uint64_t)m & 0xffffffffu), (uint32_t)((uint64_t)m >> 32),
                           (uint32_t)(step & 0xffffffffu),
                           (uint32_t)((((step >> 32) & 0xffffu) << 16) | ((uint32_t)field & 0xffffu))};
  const uint32_t key[2] = {(uint32_t)(s->seed & 0xffffffffu), (uint32_t)(s->seed >> 32)};
  philox4x32_10(ctr, key, w);
}

static void gauss_pair(const opss_system *s, const uint32_t w[4], double &g1, double &g2) {
  double u1, u2;
  if (s->prec == OPSS_F32) {
    u1 = (double)((w[0] >> 8) + 1u) * (1.0 / 16777216.0);          /* (0,1] , 24 bits */
    u2 = (double)(w[1] >> 8) * (1.0 / 16777216.0);                 /* [0,1)           */
  } else {
    const uint64_t a = (((uint64_t)(w[0] >> 5)) << 26) | (uint64_t)(w[1] >> 6);
    const uint64_t b = (((uint64_t)(w[2] >> 5)) << 26) | (uint64_t)(w[3] >> 6);
    u1 = (double)(a + 1) * (1.0 / 9007199254740992.0);             /* (0,1] , 53 bits */
    u2 = (double)b * (1.0 / 9007199254740992.0);
  }
  const double r = std::sqrt(-2.0 * std::log(u1));                 /* Box-Muller */
  g1 = r * std::cos(2.0 * PI_D * u2);
  g2 = r * std::sin(2.0 * PI_D * u2);
}

/* unit-variance Hermitian complex Gaussian at mode k */
static cplx noise_z(const opss_system *s, int field, uint64_t step, const int64_t k[3]) {
  const Dims &d = s->d;
  const int64_t m = index_of(d, k);
  uint32_t w[4];
  double g1, g2;
  const bool on_plane = (k[0] == 0) || (2 * k[0] == d.n[0]);
  if (!on_plane) {
    noise_block(s, field, step, m, w);
    gauss_pair(s, w, g1, g2);
    return cplx(g1, g2) * std::sqrt(0.5);
  }
  const int64_t kp[3] = {k[0], (d.n[1] - k[1]) % d.n[1], (d.n[2] - k[2]) % d.n[2]};
  const int64_t mp = index_of(d, kp);
  if (mp == m) { /* self-conjugate: real, variance 1 */
    noise_block(s, field, step, m, w);
    gauss_pair(s, w, g1, g2);
    return cplx(g1, 0.0);
  }
  const int64_t mc = (m < mp) ? m : mp; /* canonical member draws */
  noise_block(s, field, step, mc, w);
  gauss_pair(s, w, g1, g2);
  const cplx z = cplx(g1, g2) * std::sqrt(0.5);
  return (m < mp) ? z : std::conj(z);
}

/* sqrt(2 D |q|^a dt N / dV)  (reading A1) */
static double noise_amp(const opss_system *s, const Field &f, const int64_t k[3]) {
  double q2 = 0.0, dV = 1.0;
  for (int j = 0; j < 3; ++j) { const double q = qcomp(s, j, k[j]); q2 += q * q; }
  for (int j = 0; j < s->d.ndim; ++j) dV *= s->dx[j];
  double qa = 1.0;
  if (f.qpow != 0) {
    const double q = std::sqrt(q2);
    const int a = f.qpow < 0 ? -f.qpow : f.qpow;
    if (f.qpow < 0 && q2 == 0.0) return 0.0;
    for (int i = 0; i < a; ++i) qa *= q;
    if (f.qpow < 0) qa = 1.0 / qa;
  }
  return std::sqrt(2.0 * f.D * qa * s->dt * (double)s->d.nsites() / dV);
}

/* ------------------------------------------------------------------------------------------
 * One time step: PAPER.md:128-135 in order, Eq. 18 at the end.
 * ------------------------------------------------------------------------------------------ */
static void one_step(opss_system *s) {
  const Dims &d = s->d;
  const int64_t M = d.nmodes(), NS = d.nsites();
  const int nth = s->nthreads;
  const int nf = (int)s->fields.size();

  /* de-aliased copy of field f in real space, made once its spectrum is final for this step */
  std::vector<std::vector<double>> real(nf);
  auto to_real = [&](int f) {
    if (!real[f].empty()) return;
    const int order = max_order(s, f);
    std::vector<cplx> masked(s->fields[f].hat);
#pragma omp parallel for num_threads(nth) schedule(static)
    for (int64_t m = 0; m < M; ++m) {
      int64_t k[3]; mode_of(d, m, k);
      if (!keep_mode(s, order, k)) masked[m] = cplx(0, 0);
    }
    c2r(masked, real[f], d, nth);
  };

  /* 1. intermediate fields psi_k, creation order, from time-t values (A12) */
  for (int a = 0; a < nf; ++a) {
    Field &fa = s->fields[a];
    if (fa.dynamic) continue;
    fa.hat.assign(M, cplx(0, 0));
    for (const Def &df : fa.defs) {
      const std::vector<cplx> &src = s->fields[df.src].hat;
#pragma omp parallel for num_threads(nth) schedule(static)
      for (int64_t m = 0; m < M; ++m) {
        int64_t k[3]; mode_of(d, m, k);
        fa.hat[m] += op_eval(s, df.op, k) * src[m];
      }
    }
    /* rhs terms that are products: the factors (dynamic or earlier intermediate fields) are final */
    for (const ATerm &t : fa.aterms) {
      std::vector<double> P(NS, 1.0);
      for (int g : t.factors) {
        to_real(g);
        const std::vector<double> &r = real[g];
#pragma omp parallel for num_threads(nth) schedule(static)
        for (int64_t x = 0; x < NS; ++x) P[x] *= r[x];
      }
      std::vector<cplx> Ph;
      r2c(P, Ph, d, nth);
#pragma omp parallel for num_threads(nth) schedule(static)
      for (int64_t m = 0; m < M; ++m) {
        int64_t k[3]; mode_of(d, m, k);
        fa.hat[m] += op_eval(s, t.outer, k) * Ph[m];
      }
    }
    /* its own lhs: den(q) psi_q = rhs_q, psi_q = 0 where den(q) = 0 (as 1/q at q = 0, A10) */
    if (!fa.alhs.empty()) {
#pragma omp parallel for num_threads(nth) schedule(static)
      for (int64_t m = 0; m < M; ++m) {
        int64_t k[3]; mode_of(d, m, k);
        cplx den(0, 0);
        for (const opss_op &o : fa.alhs) den += op_eval(s, o, k);
        fa.hat[m] = (den == cplx(0, 0)) ? cplx(0, 0) : fa.hat[m] / den;
      }
    }
  }

  /* 2.+3. de-aliased copies of the factor fields, to real space */
  for (int f = 0; f < nf; ++f) {
    const int order = max_order(s, f);
    if (order < 2) continue;
    to_real(f);
  }

  /* 3.+4.+5a. N_i(q) = sum_t outer_t(q) F[prod factors](q)  + explicit linear terms (Eq. 15) */
  std::vector<std::vector<cplx>> N(nf);
  for (int f = 0; f < nf; ++f)
    if (s->fields[f].dynamic) N[f].assign(M, cplx(0, 0));
  for (const Term &t : s->terms) {
    std::vector<cplx> &Ni = N[t.field];
    if (t.factors.size() == 1) { /* linear in another (or the same) field: no transform (A8) */
      const std::vector<cplx> &src = s->fields[t.factors[0]].hat;
#pragma omp parallel for num_threads(nth) schedule(static)
      for (int64_t m = 0; m < M; ++m) {
        int64_t k[3]; mode_of(d, m, k);
        Ni[m] += op_eval(s, t.outer, k) * src[m];
      }
      continue;
    }
    std::vector<double> P(NS, 1.0);
    for (int g : t.factors) {
      const std::vector<double> &r = real[g];
#pragma omp parallel for num_threads(nth) schedule(static)
      for (int64_t x = 0; x < NS; ++x) P[x] *= r[x];
    }
    std::vector<cplx> Ph;
    r2c(P, Ph, d, nth);
#pragma omp parallel for num_threads(nth) schedule(static)
    for (int64_t m = 0; m < M; ++m) {
      int64_t k[3]; mode_of(d, m, k);
      Ni[m] += op_eval(s, t.outer, k) * Ph[m];
    }
  }

  /* 5.+6. noise and the semi-implicit update, Eq. 18, all from time-t values */
  for (int f = 0; f < nf; ++f) {
    Field &F = s->fields[f];
    if (!F.dynamic) continue;
    std::vector<cplx> &Ni = N[f];
#pragma omp parallel for num_threads(nth) schedule(static)
    for (int64_t m = 0; m < M; ++m) {
      int64_t k[3]; mode_of(d, m, k);
      cplx L(0, 0);
      for (const opss_op &op : F.lhs) L -= op_eval(s, op, k); /* dt phi + lhs = rhs  =>  L = -lhs (A3) */
      cplx num = F.hat[m] + s->dt * Ni[m];
      if (F.noisy) num += noise_amp(s, F, k) * noise_z(s, f, s->step, k);
      Ni[m] = num / (cplx(1.0, 0.0) - s->dt * L);
    }
  }
  for (int f = 0; f < nf; ++f)
    if (s->fields[f].dynamic) s->fields[f].hat.swap(N[f]);
  /* callback at the end of the time step: the field in real space, a frame of fixed values around the
   * boundary ("a buffer zone of infinite stiffness", Fig. 2), back to Fourier space */
  for (int f = 0; f < nf; ++f) {
    Field &F = s->fields[f];
    if (!F.dynamic || F.frames.empty()) continue;
    std::vector<double> r;
    c2r(F.hat, r, d, nth);
    for (const Frame &fr : F.frames) {
      for (int64_t x = 0; x < NS; ++x) {
        int64_t c[3] = {x % d.n[0], (x / d.n[0]) % d.n[1], x / (d.n[0] * d.n[1])};
        if (c[fr.axis] < fr.lo_w) r[x] = fr.lo_v;
        else if (c[fr.axis] >= d.n[fr.axis] - fr.hi_w) r[x] = fr.hi_v;
      }
    }
    r2c(r, F.hat, d, nth);
  }
  s->step += 1;
}

/* ------------------------------------------------------------------------------------------
 * C ABI
 * ------------------------------------------------------------------------------------------ */
extern "C" {

int opss_create(opss_system **out, int ndim, const int64_t n[3], const double dx[3], double dt,
                int prec, uint64_t seed) {
  if (!out || !n || !dx) return OPSS_EINVAL;
  *out = nullptr;
  if (ndim < 1) return OPSS_EINVAL;
  if (ndim > 3) return OPSS_EUNSUPPORTED;
  if (prec != OPSS_F32 && prec != OPSS_F64) return OPSS_EINVAL;
  if (!(dt > 0.0) || !std::isfinite(dt)) return OPSS_EINVAL;
  for (int j = 0; j < ndim; ++j) {
    if (n[j] < 1 || !(dx[j] > 0.0) || !std::isfinite(dx[j])) return OPSS_EINVAL;
    if (!is_pow2(n[j]) || n[j] < 2) return OPSS_EUNSUPPORTED; /* A17 */
  }
  opss_system *s = new opss_system();
  s->d.ndim = ndim;
  for (int j = 0; j < 3; ++j) { s->d.n[j] = j < ndim ? n[j] : 1; s->dx[j] = j < ndim ? dx[j] : 1.0; }
  s->d.nxh = s->d.n[0] / 2 + 1;
  s->dt = dt; s->prec = prec; s->seed = seed;
  s->dealias = OPSS_DEALIAS_PAPER;
  s->nthreads = max_threads();
  s->finalized = false; s->step = 0;
  *out = s;
  return OPSS_OK;
}

int opss_add_field(opss_system *s, const char *name, int dynamic, int *field_id) {
  if (!s || !name) return OPSS_EINVAL;
  if (s->finalized) return OPSS_ESTATE;
  if (s->fields.size() >= 65536) return OPSS_EUNSUPPORTED;
  for (const Field &f : s->fields) if (f.name == name) return OPSS_EINVAL;
  Field f; f.name = name; f.dynamic = dynamic != 0; f.noisy = false; f.D = 0; f.qpow = 0;
  s->fields.push_back(f);
  if (field_id) *field_id = (int)s->fields.size() - 1;
  return OPSS_OK;
}

static bool fid_ok(const opss_system *s, int f) { return f >= 0 && f < (int)s->fields.size(); }

int opss_add_linear(opss_system *s, int field, const opss_op *op) {
  if (!s) return OPSS_EINVAL;
  if (s->finalized) return OPSS_ESTATE;
  if (!fid_ok(s, field) || !op_ok(s, op)) return OPSS_EINVAL;
  if (!s->fields[field].dynamic) return OPSS_EINVAL; /* implicit term on an aux field */
  s->fields[field].lhs.push_back(*op);
  return OPSS_OK;
}

int opss_add_aux_def(opss_system *s, int aux, const opss_op *op, int src) {
  if (!s) return OPSS_EINVAL;
  if (s->finalized) return OPSS_ESTATE;
  if (!fid_ok(s, aux) || !fid_ok(s, src) || !op_ok(s, op)) return OPSS_EINVAL;
  if (s->fields[aux].dynamic) return OPSS_EINVAL;
  /* a definition may use dynamic fields and EARLIER aux fields only (A12) */
  if (!s->fields[src].dynamic && src >= aux) return OPSS_EINVAL;
  Def d; d.op = *op; d.src = src;
  s->fields[aux].defs.push_back(d);
  return OPSS_OK;
}

int opss_set_frame(opss_system *s, int field, int axis, int64_t lo_width, double lo_value, int64_t hi_width, double hi_value) {
  if (!s) return OPSS_EINVAL;
  if (s->finalized) return OPSS_ESTATE;
  if (!fid_ok(s, field) || !s->fields[field].dynamic) return OPSS_EINVAL;
  if (axis < 0 || axis >= s->d.ndim) return OPSS_EINVAL;
  if (lo_width < 0 || hi_width < 0 || lo_width + hi_width > s->d.n[axis]) return OPSS_EINVAL;
  if (!std::isfinite(lo_value) || !std::isfinite(hi_value)) return OPSS_EINVAL;
  Frame fr; fr.axis = axis; fr.lo_w = lo_width; fr.hi_w = hi_width; fr.lo_v = lo_value; fr.hi_v = hi_value;
  s->fields[field].frames.push_back(fr);
  return OPSS_OK;
}

int opss_add_aux_lhs(opss_system *s, int aux, const opss_op *op) {
  if (!s) return OPSS_EINVAL;
  if (s->finalized) return OPSS_ESTATE;
  if (!fid_ok(s, aux) || !op_ok(s, op)) return OPSS_EINVAL;
  if (s->fields[aux].dynamic) return OPSS_EINVAL;
  s->fields[aux].alhs.push_back(*op);
  return OPSS_OK;
}

int opss_add_aux_term(opss_system *s, int aux, const opss_op *outer, int nfactors, const int *factor_fields) {
  if (!s) return OPSS_EINVAL;
  if (s->finalized) return OPSS_ESTATE;
  if (!fid_ok(s, aux) || !op_ok(s, outer) || !factor_fields) return OPSS_EINVAL;
  if (s->fields[aux].dynamic) return OPSS_EINVAL;
  if (nfactors < 2) return OPSS_EINVAL; /* one factor is opss_add_aux_def */
  if (nfactors > 4) return OPSS_EUNSUPPORTED;
  ATerm t; t.outer = *outer;
  for (int i = 0; i < nfactors; ++i) {
    const int g = factor_fields[i];
    if (!fid_ok(s, g)) return OPSS_EINVAL;
    if (!s->fields[g].dynamic && g >= aux) return OPSS_EINVAL; /* dynamic or EARLIER intermediate fields only (A12) */
    t.factors.push_back(g);
  }
  s->fields[aux].aterms.push_back(t);
  return OPSS_OK;
}

int opss_add_term(opss_system *s, int field, const opss_op *outer, int nfactors,
                  const int *factor_fields) {
  if (!s) return OPSS_EINVAL;
  if (s->finalized) return OPSS_ESTATE;
  if (!fid_ok(s, field) || !op_ok(s, outer) || !factor_fields) return OPSS_EINVAL;
  if (!s->fields[field].dynamic) return OPSS_EINVAL;
  if (nfactors < 1) return OPSS_EINVAL;
  if (nfactors > 4) return OPSS_EUNSUPPORTED;
  Term t; t.field = field; t.outer = *outer;
  for (int i = 0; i < nfactors; ++i) {
    if (!fid_ok(s, factor_fields[i])) return OPSS_EINVAL;
    t.factors.push_back(factor_fields[i]);
  }
  s->terms.push_back(t);
  return OPSS_OK;
}

int opss_set_noise(opss_system *s, int field, double D, int q_power) {
  if (!s) return OPSS_EINVAL;
  if (s->finalized) return OPSS_ESTATE;
  if (!fid_ok(s, field) || !s->fields[field].dynamic) return OPSS_EINVAL;
  if (!(D >= 0.0) || !std::isfinite(D)) return OPSS_EINVAL;
  if (q_power < -8 || q_power > 8) return OPSS_EINVAL;
  Field &f = s->fields[field];
  f.noisy = D > 0.0; f.D = D; f.qpow = q_power;
  return OPSS_OK;
}

int opss_set_dealias(opss_system *s, int rule) {
  if (!s) return OPSS_EINVAL;
  if (s->finalized) return OPSS_ESTATE;
  if (rule < OPSS_DEALIAS_PAPER || rule > OPSS_DEALIAS_OFF) return OPSS_EINVAL;
  s->dealias = rule;
  return OPSS_OK;
}

int opss_finalize(opss_system *s, size_t *workspace_bytes) {
  if (!s) return OPSS_EINVAL;
  if (s->finalized) return OPSS_ESTATE;
  int ndyn = 0;
  for (const Field &f : s->fields) ndyn += f.dynamic ? 1 : 0;
  if (ndyn == 0) return OPSS_EINVAL;
  for (size_t a = 0; a < s->fields.size(); ++a)
    if (!s->fields[a].dynamic && s->fields[a].defs.empty() && s->fields[a].aterms.empty()) return OPSS_EINVAL; /* undefined aux */
  for (Field &f : s->fields) f.hat.assign(s->d.nmodes(), cplx(0, 0));
  s->finalized = true;
  if (workspace_bytes) *workspace_bytes = 0; /* the oracle owns its memory */
  return OPSS_OK;
}

int opss_set_threads(opss_system *s, int nthreads) {
  if (!s || nthreads < 0) return OPSS_EINVAL;
  s->nthreads = nthreads == 0 ? max_threads() : nthreads;
  return OPSS_OK;
}

int opss_set_field(opss_system *s, int field, const void *real_xfastest) {
  if (!s || !real_xfastest) return OPSS_EINVAL;
  if (!s->finalized) return OPSS_ESTATE;
  if (!fid_ok(s, field) || !s->fields[field].dynamic) return OPSS_EINVAL;
  const int64_t NS = s->d.nsites();
  std::vector<double> re(NS);
  if (s->prec == OPSS_F32) { const float *p = (const float *)real_xfastest; for (int64_t i = 0; i < NS; ++i) re[i] = (double)p[i]; }
  else { const double *p = (const double *)real_xfastest; for (int64_t i = 0; i < NS; ++i) re[i] = p[i]; }
  r2c(re, s->fields[field].hat, s->d, s->nthreads);
  return OPSS_OK;
}

int opss_step(opss_system *s, int64_t nsteps) {
  if (!s || nsteps < 0) return OPSS_EINVAL;
  if (!s->finalized) return OPSS_ESTATE;
  for (int64_t i = 0; i < nsteps; ++i) one_step(s);
  return OPSS_OK;
}

int opss_get_field(opss_system *s, int field, void *real_out) {
  if (!s || !real_out) return OPSS_EINVAL;
  if (!s->finalized) return OPSS_ESTATE;
  if (!fid_ok(s, field) || !s->fields[field].dynamic) return OPSS_EINVAL;
  std::vector<double> re;
  c2r(s->fields[field].hat, re, s->d, s->nthreads);
  const int64_t NS = s->d.nsites();
  if (s->prec == OPSS_F32) { float *p = (float *)real_out; for (int64_t i = 0; i < NS; ++i) p[i] = (float)re[i]; }
  else { double *p = (double *)real_out; for (int64_t i = 0; i < NS; ++i) p[i] = re[i]; }
  return OPSS_OK;
}

int opss_get_field_fourier_f64(opss_system *s, int field, double *out) {
  if (!s || !out) return OPSS_EINVAL;
  if (!s->finalized) return OPSS_ESTATE;
  if (!fid_ok(s, field) || !s->fields[field].dynamic) return OPSS_EINVAL;
  const std::vector<cplx> &h = s->fields[field].hat;
  for (size_t m = 0; m < h.size(); ++m) { out[2 * m] = h[m].real(); out[2 * m + 1] = h[m].imag(); }
  return OPSS_OK;
}

int opss_get_field_fourier(opss_system *s, int field, void *out) {
  if (!s || !out) return OPSS_EINVAL;
  if (!s->finalized) return OPSS_ESTATE;
  if (!fid_ok(s, field) || !s->fields[field].dynamic) return OPSS_EINVAL;
  if (s->prec == OPSS_F64) return opss_get_field_fourier_f64(s, field, (double *)out);
  const std::vector<cplx> &h = s->fields[field].hat;
  float *p = (float *)out;
  for (size_t m = 0; m < h.size(); ++m) { p[2 * m] = (float)h[m].real(); p[2 * m + 1] = (float)h[m].imag(); }
  return OPSS_OK;
}

int opss_debug_noise(opss_system *s, int field, uint64_t step, uint32_t *bits, double *z) {
  if (!s) return OPSS_EINVAL;
  if (!s->finalized) return OPSS_ESTATE;
  if (!fid_ok(s, field)) return OPSS_EINVAL;
  const int64_t M = s->d.nmodes();
#pragma omp parallel for num_threads(s->nthreads) schedule(static)
  for (int64_t m = 0; m < M; ++m) {
    int64_t k[3]; mode_of(s->d, m, k);
    if (bits) noise_block(s, field, step, m, bits + 4 * m);
    if (z) { const cplx v = noise_z(s, field, step, k); z[2 * m] = v.real(); z[2 * m + 1] = v.imag(); }
  }
  return OPSS_OK;
}

uint64_t opss_step_count(const opss_system *s) { return s ? s->step : 0; }

const char *opss_strerror(int code) {
  switch (code) {
    case OPSS_OK: return "ok";
    case OPSS_EINVAL: return "invalid argument";
    case OPSS_EUNSUPPORTED: return "unsupported configuration";
    case OPSS_ESTATE: return "call made in the wrong state";
    default: return "unknown error";
  }
}

void opss_destroy(opss_system *s) { delete s; }

int opss_debug_fft_lines(double *data, int64_t n, int64_t howmany, int sign) {
  if (!data || !is_pow2(n) || howmany < 0 || (sign != 1 && sign != -1)) return OPSS_EINVAL;
  LineSet ls = {n, 1, howmany, howmany > 0 ? howmany : 1, n, 0};
  fft_lines(reinterpret_cast<cplx *>(data), ls, sign, max_threads());
  return OPSS_OK;
}

static int make_dims(Dims &d, int ndim, const int64_t n[3]) {
  if (ndim < 1 || ndim > 3 || !n) return OPSS_EINVAL;
  d.ndim = ndim;
  for (int j = 0; j < 3; ++j) { d.n[j] = j < ndim ? n[j] : 1; if (!is_pow2(d.n[j])) return OPSS_EUNSUPPORTED; }
  d.nxh = d.n[0] / 2 + 1;
  return OPSS_OK;
}

int opss_debug_r2c(const double *real_in, double *half_out, int ndim, const int64_t n[3]) {
  Dims d; int rc = make_dims(d, ndim, n); if (rc) return rc;
  std::vector<double> re(real_in, real_in + d.nsites());
  std::vector<cplx> h;
  r2c(re, h, d, max_threads());
  for (size_t m = 0; m < h.size(); ++m) { half_out[2 * m] = h[m].real(); half_out[2 * m + 1] = h[m].imag(); }
  return OPSS_OK;
}

int opss_debug_c2r(const double *half_in, double *real_out, int ndim, const int64_t n[3]) {
  Dims d; int rc = make_dims(d, ndim, n); if (rc) return rc;
  std::vector<cplx> h(d.nmodes());
  for (size_t m = 0; m < h.size(); ++m) h[m] = cplx(half_in[2 * m], half_in[2 * m + 1]);
  std::vector<double> re;
  c2r(h, re, d, max_threads());
  std::memcpy(real_out, re.data(), sizeof(double) * re.size());
  return OPSS_OK;
}

int opss_debug_op(const opss_system *s, const opss_op *op, const int64_t k[3], double out[2]) {
  if (!s || !op || !k || !out || !op_ok(s, op)) return OPSS_EINVAL;
  const cplx v = op_eval(s, *op, k);
  out[0] = v.real(); out[1] = v.imag();
  return OPSS_OK;
}

int opss_debug_mask(opss_system *s, int field, uint8_t *mask) {
  if (!s || !mask || !fid_ok(s, field)) return OPSS_EINVAL;
  const int order = max_order(s, field);
  if (order < 2) return 1; /* not a factor of any product */
  const int64_t M = s->d.nmodes();
  for (int64_t m = 0; m < M; ++m) { int64_t k[3]; mode_of(s->d, m, k); mask[m] = keep_mode(s, order, k) ? 1 : 0; }
  return OPSS_OK;
}

void opss_debug_philox(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]) {
  philox4x32_10(ctr, key, out);
}

} /* extern "C" */
