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
  return mq;
}

/* value of one operator monomial (A9, A10) */
template <typename T> __device__ __forceinline__ typename cplx_of<T>::type eval_op(const DOp &op, const ModeQ<T> &mq) {
  typedef typename cplx_of<T>::type C;
  if ((op.zflags & 7 & mq.nyq) || ((op.zflags & 8) && mq.q2 == (T)0)) return mk<C, T>((T)0, (T)0);
  T r = (T)op.coef;
  for (int i = 0; i < op.m; ++i) r *= mq.q2;
  if (op.p > 0) {
    const T inv = (T)1 / sqrt(mq.q2);
    for (int i = 0; i < op.p; ++i) r *= inv;
  }
  int s = 0;
#pragma unroll
  for (int j = 0; j < 3; ++j) {
    for (int i = 0; i < op.a[j]; ++i) r *= mq.q[j];
    s += op.a[j];
  }
  switch (s & 3) {
    case 0: return mk<C, T>(r, (T)0);
    case 1: return mk<C, T>((T)0, r);
    case 2: return mk<C, T>(-r, (T)0);
    default: return mk<C, T>((T)0, -r);
  }
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
__device__ __forceinline__ void noise_block(const Program &P, int field, unsigned long long step, long long m,
                                            uint32_t w[4]) {
  philox4x32_10((uint32_t)((unsigned long long)m & 0xffffffffu), (uint32_t)((unsigned long long)m >> 32),
                (uint32_t)(step & 0xffffffffu),
                (uint32_t)((((step >> 32) & 0xffffu) << 16) | ((uint32_t)field & 0xffffu)), P.seed_lo, P.seed_hi, w);
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

/* unit-variance Hermitian complex Gaussian at logical mode (k0,k1,k2)  (Eq. 16, 134) */
template <typename T>
__device__ __forceinline__ typename cplx_of<T>::type noise_z(const Program &P, int field, unsigned long long step,
                                                             int k0, int k1, int k2) {
  typedef typename cplx_of<T>::type C;
  const long long n1 = P.n[1], n2 = P.n[2], nxh = P.nxh;
  const long long m = ((long long)k2 * n1 + k1) * nxh + k0;
  uint32_t w[4];
  T g1, g2;
  const bool on_plane = (k0 == 0) || (2 * k0 == P.n[0]);
  if (!on_plane) {
    noise_block(P, field, step, m, w);
    gauss_pair(w, g1, g2);
    const T h = (T)0.70710678118654752440;
    return mk<C, T>(g1 * h, g2 * h);
  }
  const long long p1 = (n1 - k1) % n1, p2 = (n2 - k2) % n2;
  const long long mp = (p2 * n1 + p1) * nxh + k0;
  noise_block(P, field, step, m < mp ? m : mp, w);
  gauss_pair(w, g1, g2);
  if (mp == m) return mk<C, T>(g1, (T)0);
  const T h = (T)0.70710678118654752440;
  return mk<C, T>(g1 * h, (m < mp) ? g2 * h : -(g2 * h));
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

template <typename C> __device__ __forceinline__ C sel4(const C *v, int i) {
  C r = v[0];
  if (i == 1) r = v[1];
  if (i == 2) r = v[2];
  if (i == 3) r = v[3];
  return r;
}

#endif
