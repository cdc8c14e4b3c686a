/*
 * pss_pointwise.cuh — the per-mode arithmetic of the step: wavevectors, operator monomials,
 * the de-aliasing test, and the Philox4x32-10 + Box-Muller Hermitian noise.
 *
 * Citations are PAPER.md lines; A-numbers are the readings listed in DESIGN.md.
 */
#ifndef PSS_POINTWISE_CUH
#define PSS_POINTWISE_CUH
#include "pss_fft.cuh"

/* wavevector of one mode, q_j = 2 pi s(k_j)/(n_j dx_j) */
template <typename T> struct ModeQ {
  T q[3];
  T q2;
  T rq;    /* 1/|q| (0 at q = 0, A10); filled only when the program has a 1/q keyword (Program::any_invq) */
  int nyq; /* bit j set: k_j is the Nyquist index of axis j */
};

__device__ __forceinline__ int signed_index(int k, int n) { return (k <= (n >> 1)) ? k : k - n; }

template <typename T> __device__ __forceinline__ ModeQ<T> make_mode(const Program &P, int k0, int k1, int k2) {
  ModeQ<T> mq;
  const int kk[3] = {k0, k1, k2};
  mq.q2 = (T)0;
  mq.nyq = 0;
#pragma unroll
  for (int j = 0; j < 3; ++j) {
    if (j < P.ndim) {
      mq.q[j] = (T)P.qs[j] * (T)signed_index(kk[j], P.n[j]);
      if (P.n[j] > 1 && 2 * kk[j] == P.n[j]) mq.nyq |= 1 << j;
    } else {
      mq.q[j] = (T)0;
    }
    mq.q2 += mq.q[j] * mq.q[j];
  }
  mq.rq = (P.any_invq && mq.q2 > (T)0) ? (T)1 / sqrt(mq.q2) : (T)0;
  return mq;
}

/* value of one operator monomial without its denominator (A9, A10) */
template <typename T> __device__ __forceinline__ typename cplx_of<T>::type eval_op_nd(const DOp &op, const ModeQ<T> &mq) {
  typedef typename cplx_of<T>::type C;
  if ((op.zflags & 7 & mq.nyq) || ((op.zflags & 8) && mq.q2 == (T)0)) return mk<C, T>((T)0, (T)0);
  T r = (T)op.coef;
  {
    T bq = mq.q2;
    for (int m = op.m; m > 0; m >>= 1) { if (m & 1) r *= bq; bq *= bq; }
  }
  if (op.p > 0) {
    T bq = mq.rq;
    for (int m = op.p; m > 0; m >>= 1) { if (m & 1) r *= bq; bq *= bq; }
  }
  int s = 0;
#pragma unroll
  for (int j = 0; j < 3; ++j) {
    T bq = mq.q[j];
    for (int m = op.a[j]; m > 0; m >>= 1) { if (m & 1) r *= bq; bq *= bq; }
    s += op.a[j];
  }
  switch (s & 3) {
    case 0: return mk<C, T>(r, (T)0);
    case 1: return mk<C, T>((T)0, r);
    case 2: return mk<C, T>(-r, (T)0);
    default: return mk<C, T>((T)0, -r);
  }
}

/* 1/den(q) of the lhs polynomial `id` of an intermediate field; 0 where den vanishes (A10) */
template <typename T> __device__ __forceinline__ T eval_rden(const Program &P, int id, const ModeQ<T> &mq) {
  T d = (T)0;
  for (int e = P.den[id].beg; e < P.den[id].end; ++e) d += eval_op_nd<T>(P.lin[e], mq).x;
  return (d == (T)0) ? (T)0 : (T)1 / d;
}
/* value of one operator monomial, denominator included (evaluated only by the monomials that carry one) */
template <typename T> __device__ __forceinline__ typename cplx_of<T>::type eval_op(const Program &P, const DOp &op, const ModeQ<T> &mq) {
  typename cplx_of<T>::type v = eval_op_nd<T>(op, mq);
  if (op.den) {
    const T r = eval_rden<T>(P, op.den - 1, mq);
    v.x *= r;
    v.y *= r;
  }
  return v;
}

/* keep iff (n+1)|s(k)| < N on this axis (A4, A5, A6) */
__device__ __forceinline__ bool keep_axis(int dealias, int order, int k, int n) {
  if (dealias == 2) return true;
  const int nn = (dealias == 1) ? 2 : order;
  int a = signed_index(k, n);
  a = a < 0 ? -a : a;
  return (nn + 1) * a < n;
}

/* ---- Philox4x32-10 (Salmon, Moraes, Dror, Shaw, SC'11), published constants ---- */
__device__ __forceinline__ void philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3, uint32_t k0,
                                              uint32_t k1, uint32_t w[4]) {
#pragma unroll
  for (int r = 0; r < 10; ++r) {
    const uint32_t hi0 = __umulhi(0xD2511F53u, c0), lo0 = 0xD2511F53u * c0;
    const uint32_t hi1 = __umulhi(0xCD9E8D57u, c2), lo1 = 0xCD9E8D57u * c2;
    const uint32_t n0 = hi1 ^ c1 ^ k0, n2 = hi0 ^ c3 ^ k1;
    c0 = n0; c1 = lo1; c2 = n2; c3 = lo0;
    k0 += 0x9E3779B9u; k1 += 0xBB67AE85u;
  }
  w[0] = c0; w[1] = c1; w[2] = c2; w[3] = c3;
}

/* counter = (m_lo, m_hi, step_lo, ((step_hi & 0xffff) << 16) | field), key = seed */
/* replica r of an ensemble is the system with seed + r (pss_set_replicas) */
__device__ __forceinline__ unsigned long long replica_seed(const Program &P, unsigned rep) {
  return ((((unsigned long long)P.seed_hi) << 32) | (unsigned long long)P.seed_lo) + (unsigned long long)rep;
}
__device__ __forceinline__ void noise_block(const Program &P, unsigned rep, int field, unsigned long long step, long long m,
                                            uint32_t w[4]) {
  const unsigned long long sd = replica_seed(P, rep);
  philox4x32_10((uint32_t)((unsigned long long)m & 0xffffffffu), (uint32_t)((unsigned long long)m >> 32),
                (uint32_t)(step & 0xffffffffu),
                (uint32_t)((((step >> 32) & 0xffffu) << 16) | ((uint32_t)field & 0xffffu)), (uint32_t)(sd & 0xffffffffu),
                (uint32_t)(sd >> 32), w);
}

__device__ __forceinline__ void gauss_pair(const uint32_t w[4], float &g1, float &g2) {
  const float u1 = (float)((w[0] >> 8) + 1u) * (1.0f / 16777216.0f); /* (0,1], exact */
  const float u2 = (float)(w[1] >> 8) * (1.0f / 16777216.0f);        /* [0,1), exact */
  const float r = sqrtf(-2.0f * logf(u1));
  float s, c;
  sincospif(2.0f * u2, &s, &c);
  g1 = r * c;
  g2 = r * s;
}
__device__ __forceinline__ void gauss_pair(const uint32_t w[4], double &g1, double &g2) {
  const unsigned long long a = (((unsigned long long)(w[0] >> 5)) << 26) | (unsigned long long)(w[1] >> 6);
  const unsigned long long b = (((unsigned long long)(w[2] >> 5)) << 26) | (unsigned long long)(w[3] >> 6);
  const double u1 = (double)(a + 1ull) * (1.0 / 9007199254740992.0);
  const double u2 = (double)b * (1.0 / 9007199254740992.0);
  const double r = sqrt(-2.0 * log(u1));
  double s, c;
  sincospi(2.0 * u2, &s, &c);
  g1 = r * c;
  g2 = r * s;
}

/* ---- noise (Eq. 16): Philox4x32-10 + Box-Muller, lean fp32 path: only the two words the
 * fp32 uniforms use (same counter, same words, same uniforms as noise_block/gauss_pair), the step-invariant half of
 * round 1 left to the compiler to hoist, and own fp32 ln / sin / cos kernels
 * (coefficients fitted for this file; each within ~1 ulp of the exact value over all 2^24 inputs). ---- */
struct NoiseKey {
  uint32_t c2, c3;   /* counter words 2, 3: step_lo, ((step_hi & 0xffff) << 16) | field */
  uint32_t k0, k1;   /* key = seed */
};

__device__ __forceinline__ void philox_w01(uint32_t c0, uint32_t c1, const NoiseKey &K, uint32_t &w0, uint32_t &w1) {
  uint32_t c2 = K.c2, c3 = K.c3, k0 = K.k0, k1 = K.k1;
#pragma unroll
  for (int r = 0; r < 10; ++r) {
    const uint32_t hi0 = __umulhi(0xD2511F53u, c0), lo0 = 0xD2511F53u * c0;
    const uint32_t hi1 = __umulhi(0xCD9E8D57u, c2), lo1 = 0xCD9E8D57u * c2;
    const uint32_t n0 = hi1 ^ c1 ^ k0, n2 = hi0 ^ c3 ^ k1;
    c0 = n0; c1 = lo1; c2 = n2; c3 = lo0;
    k0 += 0x9E3779B9u; k1 += 0xBB67AE85u;
  }
  w0 = c0; w1 = c1;
}

/* sqrt(-ln u1) * (cos 2 pi u2, sin 2 pi u2) with u1 = ((w0>>8)+1) 2^-24 in (0,1], u2 = (w1>>8) 2^-24 in [0,1):
 * this is (g1 + i g2)/sqrt(2) of the Box-Muller pair g = sqrt(-2 ln u1) (cos, sin). */
__device__ __forceinline__ float2 box_muller_half(uint32_t w0, uint32_t w1) {
  /* ln u1: u1 = m 2^e, m in [2/3, 4/3); ln m = f - f^2/2 + f^3 P(f), f = m - 1 */
  const float u1 = (float)((w0 >> 8) + 1u) * (1.0f / 16777216.0f);
  const int iu = __float_as_int(u1);
  const int e = (iu - 0x3f2aaaab) & 0xff800000;
  const float f = __int_as_float(iu - e) - 1.0f;
  const float fe = (float)e * 1.1920928955078125e-07f;
  float p = -0.12429866194725037f;
  p = fmaf(p, f, 0.13433773815631866f);
  p = fmaf(p, f, -0.12287236750125885f);
  p = fmaf(p, f, 0.14116978645324707f);
  p = fmaf(p, f, -0.166733980178833f);
  p = fmaf(p, f, 0.2000383585691452f);
  p = fmaf(p, f, -0.24999943375587463f);
  p = fmaf(p, f, 0.33333319425582886f);
  const float f2 = f * f;
  const float lnm = fmaf(p * f, f2, -0.5f * f2) + f;
  const float x = -fmaf(fe, 0.693147182464599609375f, lnm);          /* -ln u1 >= 0 */
  /* sqrt by rsqrt + one Newton step; x = 0 (u1 = 1) gives 0 */
  const float y = rsqrtf(fmaxf(x, 1e-30f));
  float r = x * y;
  r = fmaf(0.5f * y, fmaf(-r, r, x), r);
  /* angle 2 pi j / 2^24: nearest quadrant q, remainder phi in [-pi/4, pi/4) exactly representable */
  const uint32_t j = w1 >> 8;
  const uint32_t qq = (j + (1u << 21)) >> 22;
  const int rem = (int)j - (int)(qq << 22);
  const float phi = (float)rem * 3.7450702829191576e-07f;             /* 2 pi / 2^24 */
  const float u = phi * phi;
  float sp = 2.7249941467744065e-06f, cp = -4.133496076974552e-06f;
  sp = fmaf(sp, u, -0.00019840087043121457f);
  cp = fmaf(cp, u, 2.896795376727823e-05f);
  sp = fmaf(sp, u, 0.008333331905305386f);
  cp = fmaf(cp, u, -0.0013901740312576294f);
  sp = fmaf(sp, u, -0.1666666716337204f);
  cp = fmaf(cp, u, 0.04166676476597786f);
  const float sn = fmaf(phi * u, sp, phi);
  const float cn = fmaf(u * u, cp, fmaf(-0.5f, u, 1.0f));
  const float ca = (qq & 1u) ? sn : cn, sa = (qq & 1u) ? cn : sn;     /* |cos|, |sin| carriers */
  const float c = ((qq + 1u) & 2u) ? -ca : ca;                        /* q = 1, 2 -> negative cosine */
  const float sgn = (qq & 2u) ? -sa : sa;                             /* q = 2, 3 -> negative sine   */
  return make_float2(r * c, r * sgn);
}

/* unit-variance Hermitian complex Gaussian at logical mode (k0,k1,k2)  (Eq. 16, 134) */
template <typename T>
__device__ __forceinline__ typename cplx_of<T>::type noise_z(const Program &P, unsigned rep, int field, unsigned long long step,
                                                             int k0, int k1, int k2) {
  typedef typename cplx_of<T>::type C;
  const long long n1 = P.n[1], n2 = P.n[2], nxh = P.nxh;
  const long long m = ((long long)k2 * n1 + k1) * nxh + k0;
  uint32_t w[4];
  T g1, g2;
  const bool on_plane = (k0 == 0) || (2 * k0 == P.n[0]);
  if (!on_plane) {
    noise_block(P, rep, field, step, m, w);
    gauss_pair(w, g1, g2);
    const T h = (T)0.70710678118654752440;
    return mk<C, T>(g1 * h, g2 * h);
  }
  const long long p1 = (n1 - k1) % n1, p2 = (n2 - k2) % n2;
  const long long mp = (p2 * n1 + p1) * nxh + k0;
  noise_block(P, rep, field, step, m < mp ? m : mp, w);
  gauss_pair(w, g1, g2);
  if (mp == m) return mk<C, T>(g1, (T)0);
  const T h = (T)0.70710678118654752440;
  return mk<C, T>(g1 * h, (m < mp) ? g2 * h : -(g2 * h));
}

/* fp32: the same stream through the lean path (two words, own ln/sin/cos) */
template <>
__device__ __forceinline__ float2 noise_z<float>(const Program &P, unsigned rep, int field, unsigned long long step, int k0, int k1, int k2) {
  const long long n1 = P.n[1], n2 = P.n[2], nxh = P.nxh;
  /* 32-bit index arithmetic whenever the half-spectrum has fewer than 2^31 modes */
  const bool small = (long long)P.nxh * P.n[1] * P.n[2] < 0x7fffffffLL;
  long long m = small ? (long long)(unsigned)(((unsigned)k2 * (unsigned)P.n[1] + (unsigned)k1) * (unsigned)P.nxh + (unsigned)k0)
                      : ((long long)k2 * n1 + k1) * nxh + k0;
  const unsigned long long sd = replica_seed(P, rep);
  NoiseKey K;
  K.k0 = (uint32_t)(sd & 0xffffffffu);
  K.k1 = (uint32_t)(sd >> 32);
  K.c2 = (uint32_t)(step & 0xffffffffu);
  K.c3 = (uint32_t)((((step >> 32) & 0xffffu) << 16) | ((uint32_t)field & 0xffffu));
  const bool on_plane = (k0 == 0) || (2 * k0 == P.n[0]);
  bool self = false, other = false;
  if (on_plane) {
    const long long p1 = (k1 == 0) ? 0 : n1 - k1, p2 = (k2 == 0) ? 0 : n2 - k2;
    const long long mp = (p2 * n1 + p1) * nxh + k0;
    self = (mp == m);
    other = (mp < m);
    m = other ? mp : m;
  }
  uint32_t w0, w1;
  philox_w01((uint32_t)((unsigned long long)m & 0xffffffffu), (uint32_t)((unsigned long long)m >> 32), K, w0, w1);
  float2 z = box_muller_half(w0, w1);
  if (self) z = make_float2(z.x * 1.41421356237309504880f, 0.f);
  else if (other) z.y = -z.y;
  return z;
}

/* sqrt(2 D |q|^a dt N / dV)  (A1) */
template <typename T> __device__ __forceinline__ T noise_amp(const DDyn &d, const ModeQ<T> &mq) {
  T qa = (T)1;
  if (d.noise_qpow != 0) {
    if (d.noise_qpow < 0 && mq.q2 == (T)0) return (T)0;
    const T q = sqrt(mq.q2);
    const int a = d.noise_qpow < 0 ? -d.noise_qpow : d.noise_qpow;
    for (int i = 0; i < a; ++i) qa *= q;
    if (d.noise_qpow < 0) qa = (T)1 / qa;
  }
  return sqrt((T)d.noise_c * qa);
}

/* v[i] for a run-time i without local-memory indexing (v lives in registers) */
template <int NS, typename C> __device__ __forceinline__ C sel_src(const C *v, int i) {
  C r = v[0];
#pragma unroll
  for (int j = 1; j < NS; ++j)
    if (i == j) r = v[j];
  return r;
}

#endif
