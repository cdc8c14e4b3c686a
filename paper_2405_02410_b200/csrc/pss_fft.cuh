/*
 * pss_fft.cuh — in-shared-memory FFT building blocks (sm_100a).
 *
 * A line of n = prod R_i complex points lives in shared memory, W lines interleaved:
 * element (j, c) at buf[geo_pad(j)*W + c] (rows padded against bank conflicts, see Geo).  Transforms are done IN PLACE without any reordering pass:
 *   fft_dif : natural order in  -> digit-reversed order out   (decimation in frequency)
 *   fft_dit : digit-reversed in -> natural order out           (its exact transpose)
 * The callers pair them so the digit-reversed order only ever meets pointwise work, which does
 * not care about order (transform, multiply pointwise, transform back).
 * Radix-R butterflies (R in 2,4,8,16) run in registers; one __syncthreads between passes.
 * Twiddles come from a table tw[j] = exp(-2 pi i j / n) computed on the host in long double.
 */
#ifndef PSS_FFT_CUH
#define PSS_FFT_CUH
#include <cuda_runtime.h>
#include "pss_program.h"

template <typename T> struct cplx_of;
template <> struct cplx_of<float> { typedef float2 type; };
template <> struct cplx_of<double> { typedef double2 type; };

template <typename C, typename T> __device__ __forceinline__ C mk(T x, T y) { C r; r.x = x; r.y = y; return r; }
template <typename C> __device__ __forceinline__ C cadd(C a, C b) { a.x += b.x; a.y += b.y; return a; }
template <typename C> __device__ __forceinline__ C csub(C a, C b) { a.x -= b.x; a.y -= b.y; return a; }
/* fp32: Blackwell's packed FADD2 (add.f32x2 / sub.f32x2) does a complex add in ONE issue slot; the halves of the
 * 64-bit register pair stay directly usable by scalar instructions (no moves in SASS). */
template <> __device__ __forceinline__ float2 cadd<float2>(float2 a, float2 b) {
  unsigned long long r;
  asm("add.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(*reinterpret_cast<unsigned long long *>(&a)), "l"(*reinterpret_cast<unsigned long long *>(&b)));
  return *reinterpret_cast<float2 *>(&r);
}
template <> __device__ __forceinline__ float2 csub<float2>(float2 a, float2 b) {
  unsigned long long r;
  asm("sub.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(*reinterpret_cast<unsigned long long *>(&a)), "l"(*reinterpret_cast<unsigned long long *>(&b)));
  return *reinterpret_cast<float2 *>(&r);
}
template <typename C> __device__ __forceinline__ C cmul(C a, C b) {
  C r; r.x = a.x * b.x - a.y * b.y; r.y = a.x * b.y + a.y * b.x; return r;
}
/* a * conj(b) */
template <typename C> __device__ __forceinline__ C cmulc(C a, C b) {
  C r; r.x = a.x * b.x + a.y * b.y; r.y = a.y * b.x - a.x * b.y; return r;
}

/* multiply by exp(SGN * 2 pi i * J / LEN) for compile-time J, LEN (LEN <= 16) */
template <int SGN, typename C> __device__ __forceinline__ C mul_root16(C d, int idx16) {
  /* idx16 = J * 16 / LEN in [0, 8) */
  typedef decltype(d.x) T;
  const T c1 = (T)0.92387953251128675613, s1 = (T)0.38268343236508977173, h = (T)0.70710678118654752440;
  T wr, wi;
  switch (idx16) {
    case 0: return d;
    case 4: { C r; if (SGN < 0) { r.x = d.y; r.y = -d.x; } else { r.x = -d.y; r.y = d.x; } return r; }
    case 1: wr = c1; wi = s1; break;
    case 2: wr = h; wi = h; break;
    case 3: wr = s1; wi = c1; break;
    case 5: wr = -s1; wi = c1; break;
    case 6: wr = -h; wi = h; break;
    default: wr = -c1; wi = s1; break; /* 7 */
  }
  if (SGN < 0) wi = -wi;
  C r; r.x = d.x * wr - d.y * wi; r.y = d.x * wi + d.y * wr; return r;
}

__host__ __device__ constexpr int bitrev_c(int i, int bits) {
  int r = 0;
  for (int b = 0; b < bits; ++b) r |= ((i >> b) & 1) << (bits - 1 - b);
  return r;
}

/* R-point DFT in registers, natural in -> natural out, X[m] = sum_k v[k] exp(SGN 2 pi i m k / R) */
template <int LGR, int SGN, typename C> __device__ __forceinline__ void dft_reg(C *v) {
  constexpr int R = 1 << LGR;
#pragma unroll
  for (int len = R; len >= 2; len >>= 1) {
    const int half = len >> 1;
#pragma unroll
    for (int blk = 0; blk < R; blk += len) {
#pragma unroll
      for (int j = 0; j < half; ++j) {
        const C a = v[blk + j], b = v[blk + j + half];
        v[blk + j] = cadd(a, b);
        v[blk + j + half] = mul_root16<SGN>(csub(a, b), j * (16 / len));
      }
    }
  }
  C t[R];
#pragma unroll
  for (int i = 0; i < R; ++i) t[bitrev_c(i, LGR)] = v[i];
#pragma unroll
  for (int i = 0; i < R; ++i) v[i] = t[i];
}

/* digit reversal between smem slot p and frequency/time index f (see header) */
__device__ __forceinline__ int geo_rev(const Geo &g, int p) { /* slot -> index */
  int f = 0, sh = 0, lgrem = 0;
#pragma unroll
  for (int q = 0; q < 4; ++q) if (q < g.nr) lgrem += g.lg[q];
#pragma unroll
  for (int q = 0; q < 4; ++q) {
    if (q < g.nr) {
      lgrem -= g.lg[q];
      const int m = (p >> lgrem) & ((1 << g.lg[q]) - 1);
      f |= m << sh;
      sh += g.lg[q];
    }
  }
  return f;
}
__device__ __forceinline__ int geo_slot(const Geo &g, int f) { /* index -> slot */
  int p = 0, lgrem = 0;
#pragma unroll
  for (int q = 0; q < 4; ++q) if (q < g.nr) lgrem += g.lg[q];
#pragma unroll
  for (int q = 0; q < 4; ++q) {
    if (q < g.nr) {
      lgrem -= g.lg[q];
      const int m = f & ((1 << g.lg[q]) - 1);
      f >>= g.lg[q];
      p |= m << lgrem;
    }
  }
  return p;
}

/* padded shared-memory row of slot p (see Geo) */
__device__ __forceinline__ int geo_pad(const Geo &g, int p) { return p + (p >> g.sh[0]) + (p >> g.sh[1]) + (p >> g.sh[2]); }
/* padded row stride of the digit whose field starts at slot bit lo (lo is 0 or one of g.sh) */
__device__ __forceinline__ int geo_stride(const Geo &g, int lo) {
  int w = 1 << lo;
#pragma unroll
  for (int i = 0; i < 3; ++i) if (g.sh[i] <= lo) w += 1 << (lo - g.sh[i]);
  return w;
}

/* branch-free digit reversal (same maps as geo_slot / geo_rev) */
__device__ __forceinline__ int geo_slot_fast(const Geo &g, int f) {
  return (((f >> g.fs[0]) & g.fm[0]) << g.ps[0]) | (((f >> g.fs[1]) & g.fm[1]) << g.ps[1]) |
         (((f >> g.fs[2]) & g.fm[2]) << g.ps[2]) | (((f >> g.fs[3]) & g.fm[3]) << g.ps[3]);
}
__device__ __forceinline__ int geo_rev_fast(const Geo &g, int p) {
  return (((p >> g.ps[0]) & g.fm[0]) << g.fs[0]) | (((p >> g.ps[1]) & g.fm[1]) << g.fs[1]) |
         (((p >> g.ps[2]) & g.fm[2]) << g.fs[2]) | (((p >> g.ps[3]) & g.fm[3]) << g.fs[3]);
}

/* one radix-2^LGR pass over `ncol` interleaved columns: element (j, c) at buf[j*rs + c], c < ncol <= rs
 * (several buffers of W columns each sit side by side in one row of rs columns).  lgL = log2 of the current sub-length L, lgn = log2 n.
 * DIT = false: butterfly then twiddle (DIF).  DIT = true: twiddle then butterfly. */
template <int LGR, int SGN, bool DIT, typename T>
__device__ __forceinline__ void fft_pass(const Geo &g, typename cplx_of<T>::type *buf, const typename cplx_of<T>::type *__restrict__ tw,
                                         int lgn, int lgL, int ncol, int rs, int twoff) {
  typedef typename cplx_of<T>::type C;
  constexpr int R = 1 << LGR;
  const int lgLs = lgL - LGR;          /* log2 of the leg stride L/R */
  const int nb = (1 << (lgn - LGR));   /* butterflies per column     */
  const int total = nb * ncol;
  const int ls = rs * geo_stride(g, lgLs); /* padded leg stride */
  const bool notw = (lgLs == 0);                       /* every twiddle of this pass is w^0 = 1 */
  const int lgc = (ncol & (ncol - 1)) ? -1 : (31 - __clz(ncol)); /* ncol a power of two: shifts */
  for (int idx = threadIdx.x; idx < total; idx += blockDim.x) {
    const int c = (lgc >= 0) ? (idx & (ncol - 1)) : (idx % ncol);
    const int b = (lgc >= 0) ? (idx >> lgc) : (idx / ncol);
    const int i = b & ((1 << lgLs) - 1);
    const int blk = b >> lgLs;
    C *p = buf + (size_t)geo_pad(g, (blk << lgL) + i) * rs + c;
    const C *twp = tw + twoff + i;     /* w_L^(m i) at twp[(m - 1) << lgLs] */
    C v[R];
#pragma unroll
    for (int k = 0; k < R; ++k) v[k] = p[k * ls];
    if (DIT && !notw) {
#pragma unroll
      for (int m = 1; m < R; ++m) {
        const C w = __ldg(twp + ((m - 1) << lgLs));
        v[m] = (SGN < 0) ? cmul(v[m], w) : cmulc(v[m], w);
      }
    }
    dft_reg<LGR, SGN>(v);
    if (!DIT && !notw) {
#pragma unroll
      for (int m = 1; m < R; ++m) {
        const C w = __ldg(twp + ((m - 1) << lgLs));
        v[m] = (SGN < 0) ? cmul(v[m], w) : cmulc(v[m], w);
      }
    }
#pragma unroll
    for (int k = 0; k < R; ++k) p[k * ls] = v[k];
  }
}

template <int SGN, bool DIT, typename T>
__device__ __forceinline__ void fft_pass_any(const Geo &g, int lgr, typename cplx_of<T>::type *buf,
                                             const typename cplx_of<T>::type *__restrict__ tw, int lgn, int lgL, int ncol, int rs, int twoff) {
  switch (lgr) {
    case 1: fft_pass<1, SGN, DIT, T>(g, buf, tw, lgn, lgL, ncol, rs, twoff); break;
    case 2: fft_pass<2, SGN, DIT, T>(g, buf, tw, lgn, lgL, ncol, rs, twoff); break;
    case 3: fft_pass<3, SGN, DIT, T>(g, buf, tw, lgn, lgL, ncol, rs, twoff); break;
    default: fft_pass<4, SGN, DIT, T>(g, buf, tw, lgn, lgL, ncol, rs, twoff); break;
  }
}

/* natural -> digit-reversed.  Caller guarantees a __syncthreads() before; one is issued after. */
template <int SGN, typename T>
__device__ __forceinline__ void fft_dif(const Geo &g, typename cplx_of<T>::type *buf,
                                        const typename cplx_of<T>::type *__restrict__ tw, int ncol, int rs) {
  int lgn = 0;
  for (int q = 0; q < g.nr; ++q) lgn += g.lg[q];
  int lgL = lgn;
  for (int q = 0; q < g.nr; ++q) {
    fft_pass_any<SGN, false, T>(g, g.lg[q], buf, tw, lgn, lgL, ncol, rs, g.twoff[q]);
    lgL -= g.lg[q];
    __syncthreads();
  }
}

/* digit-reversed -> natural.  Caller guarantees a __syncthreads() before; one is issued after. */
template <int SGN, typename T>
__device__ __forceinline__ void fft_dit(const Geo &g, typename cplx_of<T>::type *buf,
                                        const typename cplx_of<T>::type *__restrict__ tw, int ncol, int rs) {
  int lgn = 0;
  for (int q = 0; q < g.nr; ++q) lgn += g.lg[q];
  int lgL = 0;
  for (int q = g.nr - 1; q >= 0; --q) {
    lgL += g.lg[q];
    fft_pass_any<SGN, true, T>(g, g.lg[q], buf, tw, lgn, lgL, ncol, rs, g.twoff[q]);
    __syncthreads();
  }
}

/* ---- first DIF pass fed straight from global memory / last DIT pass written straight to global memory ----
 * The outermost pass (sub-length L = n) touches legs j = k*(n/R) + i: with the butterfly index i fastest across the
 * threads, leg k of a warp is one contiguous run in the line, so the pass can take its input from (or deliver its
 * output to) global memory directly and the separate copy loop and its barrier disappear.
 *   load(cc, j)       -> element j of column cc        store(cc, j, v): element j (natural order) of column cc */
template <int LGR, int SGN, typename T, typename LD>
__device__ __forceinline__ void fft_first_from(const Geo &g, typename cplx_of<T>::type *buf, const typename cplx_of<T>::type *__restrict__ tw,
                                               int lgn, int ncol, int rs, LD load) {
  typedef typename cplx_of<T>::type C;
  constexpr int R = 1 << LGR;
  const int lgLs = lgn - LGR, nb = 1 << lgLs;
  const int ls = rs * geo_stride(g, lgLs);
  const bool notw = (lgLs == 0);
  for (int idx = threadIdx.x; idx < nb * ncol; idx += blockDim.x) {
    const int i = idx & (nb - 1), cc = idx >> lgLs;
    C v[R];
#pragma unroll
    for (int k = 0; k < R; ++k) v[k] = load(cc, (k << lgLs) + i);
    dft_reg<LGR, SGN>(v);
    if (!notw) {
      const C *twp = tw + g.twoff[0] + i;
#pragma unroll
      for (int m = 1; m < R; ++m) {
        const C w = __ldg(twp + ((m - 1) << lgLs));
        v[m] = (SGN < 0) ? cmul(v[m], w) : cmulc(v[m], w);
      }
    }
    C *p = buf + (size_t)geo_pad(g, i) * rs + cc;
#pragma unroll
    for (int k = 0; k < R; ++k) p[k * ls] = v[k];
  }
}
template <int LGR, int SGN, typename T, typename ST>
__device__ __forceinline__ void fft_last_to(const Geo &g, const typename cplx_of<T>::type *buf, const typename cplx_of<T>::type *__restrict__ tw,
                                            int lgn, int ncol, int rs, ST store) {
  typedef typename cplx_of<T>::type C;
  constexpr int R = 1 << LGR;
  const int lgLs = lgn - LGR, nb = 1 << lgLs;
  const int ls = rs * geo_stride(g, lgLs);
  const bool notw = (lgLs == 0);
  for (int idx = threadIdx.x; idx < nb * ncol; idx += blockDim.x) {
    const int i = idx & (nb - 1), cc = idx >> lgLs;
    const C *p = buf + (size_t)geo_pad(g, i) * rs + cc;
    C v[R];
#pragma unroll
    for (int k = 0; k < R; ++k) v[k] = p[k * ls];
    if (!notw) {
      const C *twp = tw + g.twoff[0] + i;
#pragma unroll
      for (int m = 1; m < R; ++m) {
        const C w = __ldg(twp + ((m - 1) << lgLs));
        v[m] = (SGN < 0) ? cmul(v[m], w) : cmulc(v[m], w);
      }
    }
    dft_reg<LGR, SGN>(v);
#pragma unroll
    for (int k = 0; k < R; ++k) store(cc, (k << lgLs) + i, v[k]);
  }
}

/* fft_dif whose input comes from load(cc, j) instead of shared memory.  The caller guarantees that nobody still
 * reads the buffer; a __syncthreads() is issued after every pass (as fft_dif). */
template <int SGN, typename T, typename LD>
__device__ __forceinline__ void fft_dif_from(const Geo &g, typename cplx_of<T>::type *buf, const typename cplx_of<T>::type *__restrict__ tw,
                                             int ncol, int rs, LD load) {
  int lgn = 0;
  for (int q = 0; q < g.nr; ++q) lgn += g.lg[q];
  switch (g.lg[0]) {
    case 1: fft_first_from<1, SGN, T>(g, buf, tw, lgn, ncol, rs, load); break;
    case 2: fft_first_from<2, SGN, T>(g, buf, tw, lgn, ncol, rs, load); break;
    case 3: fft_first_from<3, SGN, T>(g, buf, tw, lgn, ncol, rs, load); break;
    default: fft_first_from<4, SGN, T>(g, buf, tw, lgn, ncol, rs, load); break;
  }
  __syncthreads();
  int lgL = lgn - g.lg[0];
  for (int q = 1; q < g.nr; ++q) {
    fft_pass_any<SGN, false, T>(g, g.lg[q], buf, tw, lgn, lgL, ncol, rs, g.twoff[q]);
    lgL -= g.lg[q];
    __syncthreads();
  }
}
/* fft_dit whose natural-order output goes to store(cc, j, v) instead of shared memory.  Caller guarantees a
 * __syncthreads() before; NO barrier is issued after the last pass (it only reads the buffer). */
template <int SGN, typename T, typename ST>
__device__ __forceinline__ void fft_dit_to(const Geo &g, typename cplx_of<T>::type *buf, const typename cplx_of<T>::type *__restrict__ tw,
                                           int ncol, int rs, ST store) {
  int lgn = 0;
  for (int q = 0; q < g.nr; ++q) lgn += g.lg[q];
  int lgL = 0;
  for (int q = g.nr - 1; q >= 1; --q) {
    lgL += g.lg[q];
    fft_pass_any<SGN, true, T>(g, g.lg[q], buf, tw, lgn, lgL, ncol, rs, g.twoff[q]);
    __syncthreads();
  }
  switch (g.lg[0]) {
    case 1: fft_last_to<1, SGN, T>(g, buf, tw, lgn, ncol, rs, store); break;
    case 2: fft_last_to<2, SGN, T>(g, buf, tw, lgn, ncol, rs, store); break;
    case 3: fft_last_to<3, SGN, T>(g, buf, tw, lgn, ncol, rs, store); break;
    default: fft_last_to<4, SGN, T>(g, buf, tw, lgn, ncol, rs, store); break;
  }
}

#endif
