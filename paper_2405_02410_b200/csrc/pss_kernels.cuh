/*
 * pss_kernels.cuh — the kernels of the time step on the internal layout.
 *
 * INTERNAL LAYOUT (x slowest, last axis fastest):  arr[kx][y][z] (3D), arr[kx][y] (2D), with
 * kx = 0..nx/2.  "rows" below are the r = y*nz + z positions that share one kx.  The state phi_q is
 * kept in Fourier space; real space exists only inside k_rows' shared memory.
 *
 * One 2D step is two kernels:
 *   k_rows   : for a tile of rows: C2R along x of every de-aliased factor (two real rows ride one
 *              complex transform), the real-space products summed per group, R2C
 *              along x.
 *   k_update : for a tile of contiguous last-axis lines: forward FFT of the groups, outer operators
 *              + explicit linear terms (Eq. 15), noise (Eq. 16), the implicit update (Eq. 18), then
 *              for the NEXT step the factor operators, the de-aliasing mask
 *               and the inverse FFT along the last axis.
 * 3D adds k_mid (the y axis) between them in each direction.
 */
#ifndef PSS_KERNELS_CUH
#define PSS_KERNELS_CUH
#include "pss_pointwise.cuh"

/* programmatic dependent launch: block until the previous kernel of the stream has completed and its writes are
 * visible (a no-op when the launch carries no such dependency) */
/* (an early griddepcontrol.launch_dependents was measured slower and is not used) */
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }

#ifndef PSS_MINB
#define PSS_MINB 3 /* fp32 k_rows / k_update: resident CTAs per SM the register budget is tuned for */
#endif

template <typename T> struct UpdArgs {
  typename cplx_of<T>::type *state; /* [ndyn][M] */
  typename cplx_of<T>::type *psix;  /* [nfac][M] */
  typename cplx_of<T>::type *phat;  /* [ngrp][M] */
  const typename cplx_of<T>::type *tw;
  long long M;
  int n, lgn;   /* last-axis length (a power of two) */
  int nlines;   /* nxh (2D) or nxh*ny (3D) */
  int W, lgW;   /* lines per block (a power of two) */
  int lg_ny;    /* 3D: log2 ny */
  int prologue;
  unsigned long long step;
  Geo geo;
};

/* wavevector pieces shared by all modes of one last-axis line */
template <typename T> struct LineQ {
  T q0, q1, q2line;
  int k0, k1, nyq;
};
template <typename T> __device__ __forceinline__ LineQ<T> make_line(const Program &P, int line, int lg_ny) {
  LineQ<T> l;
  if (P.ndim == 3) { l.k0 = line >> lg_ny; l.k1 = line & ((1 << lg_ny) - 1); } else { l.k0 = line; l.k1 = 0; }
  l.q0 = (T)P.qs[0] * (T)signed_index(l.k0, P.n[0]);
  l.nyq = (P.n[0] > 1 && 2 * l.k0 == P.n[0]) ? 1 : 0;
  l.q2line = l.q0 * l.q0;
  l.q1 = (T)0;
  if (P.ndim == 3) {
    l.q1 = (T)P.qs[1] * (T)signed_index(l.k1, P.n[1]);
    if (P.n[1] > 1 && 2 * l.k1 == P.n[1]) l.nyq |= 2;
    l.q2line += l.q1 * l.q1;
  }
  return l;
}
/* the mode (line, k) with k along the last axis; same arithmetic order as make_mode */
template <typename T> __device__ __forceinline__ ModeQ<T> line_mode(const Program &P, const LineQ<T> &l, int k, int n, T qs_last) {
  ModeQ<T> mq;
  const T ql = qs_last * (T)signed_index(k, n);
  const int last_nyq = (2 * k == n) ? 1 : 0;
  mq.q[0] = l.q0;
  if (P.ndim == 3) { mq.q[1] = l.q1; mq.q[2] = ql; mq.nyq = l.nyq | (last_nyq << 2); }
  else { mq.q[1] = ql; mq.q[2] = (T)0; mq.nyq = l.nyq | (last_nyq << 1); }
  mq.q2 = l.q2line + ql * ql;
  mq.rq = (P.any_invq && mq.q2 > (T)0) ? (T)1 / sqrt(mq.q2) : (T)0;
  return mq;
}
template <typename T> __device__ __forceinline__ T horner4(const T (&c)[5], T x) {
  return c[0] + x * (c[1] + x * (c[2] + x * (c[3] + x * c[4])));
}

/* ------------------------------------------------------------------------------------------ */
/* RAD: the "radial" fast path of pss_program.h: 0 = generic term interpreter, 1 = every coefficient a polynomial in
 * q^2 (Model B, diffusion), 2 = factors carry a derivative monomial on top (KPZ) */
/* NS: upper bound of the number of spectral sources (register arrays of the generic path); 1 for the radial paths */
template <typename T, int RAD, int NS>
__global__ void __launch_bounds__(256, sizeof(T) == 4 ? PSS_MINB : 2) k_update(const __grid_constant__ Program P, const UpdArgs<T> A) {
  typedef typename cplx_of<T>::type C;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  C *sm = reinterpret_cast<C *>(smem_raw);
  pdl_wait();
  const int n = A.n, W = A.W, lgn = A.lgn, lgW = A.lgW;
  const int line0 = blockIdx.x * W;
  const unsigned rep = blockIdx.y; /* ensemble replica: arrays [replica][field][M] */
  C *const st_base = A.state + (size_t)rep * P.ndyn * A.M;
  C *const psix_base = A.psix + (size_t)rep * P.nfac * A.M;
  const C *const phat_base = A.phat + (size_t)rep * P.ngrp * A.M;
  const int nl = min(W, A.nlines - line0);
  const int nb0 = max(P.ngrp, P.ndyn);
  const int RS = (nb0 + (P.nfac > 1 ? 1 : 0)) * W; /* columns per smem row */
  const int tid = threadIdx.x, nt = blockDim.x;
  const T qs_last = (T)P.qs[P.ndim - 1];
  const T dt = (T)P.dt, invN = (T)P.invN;
  const C zero = mk<C, T>((T)0, (T)0);
  T radL[5], radO[5];
#pragma unroll
  for (int i = 0; i < 5; ++i) { radL[i] = (T)P.rad_L[i]; radO[i] = (T)P.rad_O[i]; }

  /* ---- phase A: forward FFT of the groups along the last axis ---- */
  if (!A.prologue && P.ngrp > 0) {
    /* the first pass reads the groups straight from global memory (column cc = g*W + c) */
    fft_dif_from<-1, T>(A.geo, sm, A.tw, P.ngrp * W, RS, [&](int cc, int j) -> C {
      const int g = cc >> lgW, c = cc & (W - 1);
      return (c < nl) ? phat_base[(size_t)g * A.M + (size_t)(line0 + c) * n + j] : zero;
    });
  }
  /* ---- phase B: Eq. 15 + Eq. 16 + Eq. 18 per mode, natural order over k (coalesced state access) ---- */
  for (int c = 0; c < nl; ++c) {
    const int line = line0 + c;
    const LineQ<T> lq = make_line<T>(P, line, A.lg_ny);
#pragma unroll 2
    for (int k = tid; k < n; k += nt) {
      C *srow = sm + (size_t)geo_pad(A.geo, geo_slot_fast(A.geo, k)) * RS + c;
      const size_t gi = (size_t)line * n + k;
      if (RAD) {
        const C phi = st_base[gi];
        if (!A.prologue) {
          const ModeQ<T> mq = line_mode<T>(P, lq, k, n, qs_last);
          C num = phi;
          if (P.ngrp > 0) {
            const T o = dt * horner4<T>(radO, mq.q2);
            const C pq = srow[0];
            num.x += o * pq.x;
            num.y += o * pq.y;
          }
          const DDyn &d = P.dyn[0];
          if (d.noisy) {
            const T q4 = mq.q2 * mq.q2; /* (q^2)^nhp, nhp <= 4, branch-free */
            T qa = (T)d.noise_c;
            qa *= (P.rad_nhp & 1) ? mq.q2 : (T)1;
            qa *= (P.rad_nhp & 2) ? q4 : (T)1;
            qa *= (P.rad_nhp & 4) ? q4 * q4 : (T)1;
            const T amp = sqrt(qa);
            const C z = noise_z<T>(P, rep, d.field_id, A.step, lq.k0, P.ndim == 3 ? lq.k1 : k, P.ndim == 3 ? k : 0);
            num.x += amp * z.x;
            num.y += amp * z.y;
          }
          const T inv = (T)1 / ((T)1 - dt * horner4<T>(radL, mq.q2));
          const C out = mk<C, T>(num.x * inv, num.y * inv);
          st_base[gi] = out;
          srow[0] = out;
        } else {
          srow[0] = phi;
        }
      } else {
      C phi[NS];
#pragma unroll
      for (int i = 0; i < NS; ++i) phi[i] = (i < P.ndyn) ? st_base[(size_t)i * A.M + gi] : zero;
      if (!A.prologue) {
        const ModeQ<T> mq = line_mode<T>(P, lq, k, n, qs_last);
        C out[NS];
#pragma unroll
        for (int i = 0; i < NS; ++i) {
          if (i < P.ndyn && P.dyn[i].kind != PSS_SLOT_STEP) {
            /* an intermediate field defined by products: (re)assigned in its own round, else kept */
            const DDyn &d = P.dyn[i];
            out[i] = phi[i];
            if (d.kind == PSS_SLOT_ASSIGN) {
              C N = zero;
              for (int g = 0; g < P.ngrp; ++g)
                if (P.grp[g].target == i) N = cadd(N, cmul(eval_op<T>(P, P.grp[g].outer, mq), srow[g * W]));
              for (int e = d.lin_beg; e < d.lin_end; ++e) N = cadd(N, cmul(eval_op<T>(P, P.lin[e], mq), sel_src<NS>(phi, P.lin[e].src)));
              const T rd = d.den ? eval_rden<T>(P, d.den - 1, mq) : (T)1;
              out[i] = mk<C, T>(N.x * rd, N.y * rd);
            }
          } else if (i < P.ndyn) {
            const DDyn &d = P.dyn[i];
            C N = zero;
            for (int g = 0; g < P.ngrp; ++g)
              if (P.grp[g].target == i) N = cadd(N, cmul(eval_op<T>(P, P.grp[g].outer, mq), srow[g * W]));
            for (int e = d.lin_beg; e < d.lin_end; ++e) N = cadd(N, cmul(eval_op<T>(P, P.lin[e], mq), sel_src<NS>(phi, P.lin[e].src)));
            C L = zero;
            for (int e = d.lhs_beg; e < d.lhs_end; ++e) L = csub(L, eval_op<T>(P, P.lin[e], mq));
            C num = mk<C, T>(phi[i].x + dt * N.x, phi[i].y + dt * N.y);
            if (d.noisy) {
              const T amp = noise_amp<T>(d, mq);
              const C z = noise_z<T>(P, rep, d.field_id, A.step, lq.k0, P.ndim == 3 ? lq.k1 : k, P.ndim == 3 ? k : 0);
              num.x += amp * z.x;
              num.y += amp * z.y;
            }
            const C den = mk<C, T>((T)1 - dt * L.x, -dt * L.y);
            const T id = (T)1 / (den.x * den.x + den.y * den.y);
            const C q = cmulc(num, den);
            out[i] = mk<C, T>(q.x * id, q.y * id);
          } else {
            out[i] = zero;
          }
        }
#pragma unroll
        for (int i = 0; i < NS; ++i)
          if (i < P.ndyn) {
            if (P.dyn[i].kind != PSS_SLOT_KEEP) st_base[(size_t)i * A.M + gi] = out[i];
            srow[i * W] = out[i];
          }
      } else {
#pragma unroll
        for (int i = 0; i < NS; ++i)
          if (i < P.ndyn) srow[i * W] = phi[i];
      }
      }
    }
  }
  __syncthreads();
  /* ---- phase C: factor operators + mask + inverse FFT along the last axis, one factor at a time ---- */
  for (int f = 0; f < P.nfac; ++f) {
    const DFactor &F = P.fac[f];
    const int wb = (f == P.nfac - 1) ? 0 : nb0; /* work buffer; the last factor may overwrite buffer 0 */
    /* which of this block's lines survive the mask on their own (slow) axes? (block-uniform) */
    unsigned keepmask = 0;
    for (int c = 0; c < nl; ++c) {
      const int line = line0 + c;
      bool kp;
      if (P.ndim == 3) {
        const int k0 = line >> A.lg_ny, k1 = line & ((1 << A.lg_ny) - 1);
        kp = keep_axis(P.dealias, F.order, k0, P.n[0]) && keep_axis(P.dealias, F.order, k1, P.n[1]);
      } else {
        kp = keep_axis(P.dealias, F.order, line, P.n[0]);
      }
      if (kp) keepmask |= 1u << c;
    }
    if (keepmask == 0) continue; /* the whole tile is masked: psix stays zero (zeroed at bind) */
    T radF[5];
#pragma unroll
    for (int i = 0; i < 5; ++i) radF[i] = RAD ? (T)P.rad_F[f][i] : (T)0;
    const int ra0 = (RAD == 2) ? P.rad_a[f][0] : 0, ra1 = (RAD == 2) ? P.rad_a[f][1] : 0, ra2 = (RAD == 2) ? P.rad_a[f][2] : 0,
              ra3 = (RAD == 2) ? P.rad_a[f][3] : 0;
    for (int idx = tid; idx < (n << lgW); idx += nt) {
      const int c = idx & (W - 1), s = idx >> lgW;
      C *srow = sm + (size_t)geo_pad(A.geo, s) * RS + c;
      C v = zero;
      if ((keepmask >> c) & 1u) {
        const int k = geo_rev_fast(A.geo, s);
        if (keep_axis(P.dealias, F.order, k, n)) {
          const LineQ<T> lq = make_line<T>(P, line0 + c, A.lg_ny);
          const ModeQ<T> mq = line_mode<T>(P, lq, k, n, qs_last);
          if (RAD) {
            /* factor f = rad_F[f](q^2) * prod_j (i q_j)^a_j  (pss_program.h) */
            T fc = horner4<T>(radF, mq.q2) * invN;
            const C ph = srow[0];
            if (RAD == 1) {
              v = mk<C, T>(ph.x * fc, ph.y * fc);
            } else {
              if (ra3 & mq.nyq) fc = (T)0;
#pragma unroll
              for (int j = 0; j < 3; ++j) {
                const int aj = (j == 0) ? ra0 : (j == 1 ? ra1 : ra2);
                const T qj = mq.q[j];
                fc *= (aj & 1) ? qj : (T)1;
                fc *= (aj & 2) ? qj * qj : (T)1;
              }
              const int sph = (ra0 + ra1 + ra2) & 3; /* i^s */
              const T re = ph.x * fc, im = ph.y * fc;
              v = (sph == 0) ? mk<C, T>(re, im) : (sph == 1) ? mk<C, T>(-im, re) : (sph == 2) ? mk<C, T>(-re, -im) : mk<C, T>(im, -re);
            }
          } else {
            C phi[NS];
#pragma unroll
            for (int i = 0; i < NS; ++i) phi[i] = (i < P.ndyn) ? srow[i * W] : zero;
            for (int e = F.lin_beg; e < F.lin_end; ++e) v = cadd(v, cmul(eval_op<T>(P, P.lin[e], mq), sel_src<NS>(phi, P.lin[e].src)));
            v.x *= invN;
            v.y *= invN;
          }
        }
      }
      srow[wb * W] = v;
    }
    __syncthreads();
    /* the last pass writes the kept lines straight to global memory (natural order) */
    C *dst = psix_base + (size_t)f * A.M + (size_t)line0 * n;
    fft_dit_to<+1, T>(A.geo, sm + wb * W, A.tw, W, RS, [&](int c, int j, C val) {
      if ((keepmask >> c) & 1u) dst[(size_t)c * n + j] = val;
    });
    __syncthreads();
  }
}

/* ------------------------------------------------------------------------------------------ */
/* two consecutive rows of one kx: element index kx*R + 2c is even and the arrays are 256-byte aligned */
template <typename C> struct __align__(16) CPair { C a, b; };

template <typename T> struct RowArgs {
  const typename cplx_of<T>::type *psix; /* [nfac][M]  (kx, r) */
  typename cplx_of<T>::type *phat;       /* [ngrp][M]           */
  const typename cplx_of<T>::type *tw;
  long long M;
  long long R; /* rows per kx: ny*nz */
  int nx;
  int Wc;      /* complex columns per block = row pairs */
  Geo geo;
};

/* BIG: one CTA per SM (tile > half of the shared memory): 512 threads, else 256 threads and 3 CTAs per SM */
template <typename T, bool BIG>
__global__ void __launch_bounds__(BIG ? 512 : 256, (!BIG && sizeof(T) == 4) ? PSS_MINB : 1) k_rows(const __grid_constant__ Program P, const RowArgs<T> A) {
  typedef typename cplx_of<T>::type C;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  C *sm = reinterpret_cast<C *>(smem_raw);
  pdl_wait();
  const int nx = A.nx, nxh = nx / 2 + 1, Wc = A.Wc, lgWc = 31 - __clz(Wc); /* Wc is a power of two */
  const int RS = (P.nfac + (P.ngrp > 1 ? 1 : 0)) * Wc;
  const long long r0 = (long long)blockIdx.x * (2 * Wc);
  const C *const psix_base = A.psix + (size_t)blockIdx.y * P.nfac * A.M; /* ensemble replica blockIdx.y */
  C *const phat_base = A.phat + (size_t)blockIdx.y * P.ngrp * A.M;
  const int tid = threadIdx.x, nt = blockDim.x;
  const C zero = mk<C, T>((T)0, (T)0);

  /* zero, then Hermitian-extend the kept part of every factor: Z_k = A_k + i B_k (rows r, r+1) */
  for (int idx = tid; idx < A.geo.npad * RS; idx += nt) sm[idx] = zero;
  __syncthreads();
  for (int f = 0; f < P.nfac; ++f) {
    int cut = nxh; /* number of kept kx */
    if (P.dealias != 2) {
      const int nn = (P.dealias == 1 ? 2 : P.fac[f].order) + 1;
      cut = (nx + nn - 1) / nn; /* kx kept iff nn*kx < nx */
      if (cut > nxh) cut = nxh;
    }
    const C *src = psix_base + (size_t)f * A.M + r0;
#pragma unroll 4
    for (int idx = tid; idx < cut * Wc; idx += nt) {
      const int c = idx & (Wc - 1), kx = idx >> lgWc;
      const CPair<C> pr = *reinterpret_cast<const CPair<C> *>(src + (size_t)kx * A.R + 2 * c); /* rows r, r+1: one 16-byte access (fp32) */
      C a = pr.a, b = pr.b;
      if (kx == 0 || 2 * kx == nx) { a.y = (T)0; b.y = (T)0; } /* C2R keeps the real part there */
      sm[(size_t)geo_pad(A.geo, kx) * RS + f * Wc + c] = mk<C, T>(a.x - b.y, a.y + b.x);
      if (kx > 0 && 2 * kx < nx) sm[(size_t)geo_pad(A.geo, nx - kx) * RS + f * Wc + c] = mk<C, T>(a.x + b.y, b.x - a.y);
    }
  }
  __syncthreads();
  if (P.nfac > 0) fft_dif<+1, T>(A.geo, sm, A.tw, P.nfac * Wc, RS);
  T pc2 = (T)0, pc3 = (T)0, pc4 = (T)0;
  const bool poly1 = P.rad_ok && P.ngrp == 1 && P.nfac == 1; /* one factor field: the product is a polynomial of it */
  if (poly1)
    for (int t = P.grp[0].term_beg; t < P.grp[0].term_end; ++t) {
      const T cf = (T)P.term[t].coef;
      if (P.term[t].nf == 2) pc2 += cf;
      else if (P.term[t].nf == 3) pc3 += cf;
      else pc4 += cf;
    }
  /* real-space products per group, forward transform, Hermitian split */
  for (int g = 0; g < P.ngrp; ++g) {
    const DGroup &G = P.grp[g];
    const int wb = (g == P.ngrp - 1) ? 0 : P.nfac;
    for (int idx = tid; idx < nx * Wc; idx += nt) {
      const int c = idx & (Wc - 1), s = idx >> lgWc;
      const int sp = geo_pad(A.geo, s);
      const C *srow = sm + (size_t)sp * RS + c;
      T pa = (T)0, pb = (T)0;
      if (poly1) {
        /* one factor field: sum_t coef_t r^nf_t = r^2 (c2 + r (c3 + r c4))  (Eq. 11 with one psi) */
        const C v = srow[0];
        pa = v.x * v.x * (pc2 + v.x * (pc3 + v.x * pc4));
        pb = v.y * v.y * (pc2 + v.y * (pc3 + v.y * pc4));
      } else
      for (int t = G.term_beg; t < G.term_end; ++t) {
        const DTerm &tm = P.term[t];
        T ta = (T)tm.coef, tb = (T)tm.coef;
        for (int i = 0; i < tm.nf; ++i) {
          const C v = srow[tm.f[i] * Wc];
          ta *= v.x;
          tb *= v.y;
        }
        pa += ta;
        pb += tb;
      }
      sm[(size_t)sp * RS + wb * Wc + c] = mk<C, T>(pa, pb);
    }
    __syncthreads();
    fft_dit<-1, T>(A.geo, sm + wb * Wc, A.tw, Wc, RS);
    C *dst = phat_base + (size_t)g * A.M + r0;
    for (int idx = tid; idx < nxh * Wc; idx += nt) {
      const int c = idx & (Wc - 1), kx = idx >> lgWc;
      const C z = sm[(size_t)geo_pad(A.geo, kx) * RS + wb * Wc + c];
      const C zm = sm[(size_t)geo_pad(A.geo, (nx - kx) & (nx - 1)) * RS + wb * Wc + c];
      const T h = (T)0.5;
      CPair<C> pr;
      pr.a = mk<C, T>(h * (z.x + zm.x), h * (z.y - zm.y));
      pr.b = mk<C, T>(h * (z.y + zm.y), h * (zm.x - z.x));
      *reinterpret_cast<CPair<C> *>(dst + (size_t)kx * A.R + 2 * c) = pr;
    }
    __syncthreads();
  }
}

/* ------------------------------------------------------------------------------------------ */
/* middle (y) axis of 3D arrays arr[b][kx][y][z]: tile = (kx, W contiguous z), in place, natural order */
template <typename T> struct MidArgs {
  typename cplx_of<T>::type *arr;
  const typename cplx_of<T>::type *tw;
  long long M;
  int ny, nz, W;
  int kx_count; /* lines with kx >= kx_count are skipped (de-aliased away) */
  int nbatch;   /* arrays per replica */
  int nx;
  int nn[PSS_P_MAX_FAC]; /* per batch entry: order+1 of the de-aliasing rule, 0 = no mask.  Rows ky and lines
                            kx outside the kept band were never written by k_update: read them as zero */
  Geo geo;
};

template <int SGN, typename T> __global__ void __launch_bounds__(256) k_mid(const MidArgs<T> A) {
  typedef typename cplx_of<T>::type C;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  C *sm = reinterpret_cast<C *>(smem_raw);
  pdl_wait();
  const int W = A.W, ny = A.ny;
  const int kx = blockIdx.y;
  if (kx >= A.kx_count) return;
  const int nn = A.nn[blockIdx.z % A.nbatch]; /* blockIdx.z runs over [replica][array] */
  if (nn && nn * kx >= A.nx) return;
  C *base = A.arr + (size_t)blockIdx.z * A.M + (size_t)kx * ny * A.nz + (size_t)blockIdx.x * W;
  const int lgW = 31 - __clz(W); /* W is a power of two (planner) */
  if (sizeof(C) == 8 && W >= 2) {
    /* fp32: two complex numbers per 16-byte access (W, nz and every offset above are even) */
    const int lgH = lgW - 1;
#pragma unroll 8
    for (int idx = threadIdx.x; idx < (ny << lgH); idx += blockDim.x) {
      const int c = (idx & ((W >> 1) - 1)) << 1, j = idx >> lgH;
      int a = signed_index(j, ny);
      a = a < 0 ? -a : a;
      CPair<C> pr;
      pr.a = pr.b = mk<C, T>((T)0, (T)0);
      if (!(nn && nn * a >= ny)) pr = *reinterpret_cast<const CPair<C> *>(base + (size_t)j * A.nz + c);
      C *d = sm + geo_pad(A.geo, j) * W + c;
      d[0] = pr.a;
      d[1] = pr.b;
    }
    __syncthreads();
    fft_dif<SGN, T>(A.geo, sm, A.tw, W, W);
#pragma unroll 8
    for (int idx = threadIdx.x; idx < (ny << lgH); idx += blockDim.x) {
      const int c = (idx & ((W >> 1) - 1)) << 1, s = idx >> lgH;
      const C *q = sm + geo_pad(A.geo, s) * W + c;
      CPair<C> pr;
      pr.a = q[0];
      pr.b = q[1];
      *reinterpret_cast<CPair<C> *>(base + (size_t)geo_rev_fast(A.geo, s) * A.nz + c) = pr;
    }
    return;
  }
  for (int idx = threadIdx.x; idx < (ny << lgW); idx += blockDim.x) {
    const int c = idx & (W - 1), j = idx >> lgW;
    int a = signed_index(j, ny);
    a = a < 0 ? -a : a;
    sm[geo_pad(A.geo, j) * W + c] = (nn && nn * a >= ny) ? mk<C, T>((T)0, (T)0) : base[(size_t)j * A.nz + c];
  }
  __syncthreads();
  fft_dif<SGN, T>(A.geo, sm, A.tw, W, W);
  for (int idx = threadIdx.x; idx < (ny << lgW); idx += blockDim.x) {
    const int c = idx & (W - 1), s = idx >> lgW;
    base[(size_t)geo_rev_fast(A.geo, s) * A.nz + c] = sm[geo_pad(A.geo, s) * W + c];
  }
}

/* last axis, contiguous lines, in place, natural order (set/get paths only) */
template <typename T> struct LastArgs {
  typename cplx_of<T>::type *arr;
  const typename cplx_of<T>::type *tw;
  int n, nlines;
  Geo geo;
};

template <int SGN, typename T> __global__ void __launch_bounds__(256) k_last(const LastArgs<T> A) {
  typedef typename cplx_of<T>::type C;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  C *sm = reinterpret_cast<C *>(smem_raw);
  const int n = A.n;
  C *base = A.arr + (size_t)blockIdx.x * n;
  for (int j = threadIdx.x; j < n; j += blockDim.x) sm[geo_pad(A.geo, j)] = base[j];
  __syncthreads();
  fft_dif<SGN, T>(A.geo, sm, A.tw, 1, 1);
  for (int j = threadIdx.x; j < n; j += blockDim.x) base[j] = sm[geo_pad(A.geo, geo_slot(A.geo, j))];
}

/* ------------------------------------------------------------------------------------------ */
/* x axis between the USER layout (real, x fastest, then y, then z) and the internal layout.
 * One block per pair of user rows (ndim >= 2) or per single row (1D).  DIR = -1: R2C, +1: C2R. */
template <typename T> struct UserArgs {
  T *real;                                /* user array               */
  typename cplx_of<T>::type *arr;         /* internal [kx][y][z]      */
  const typename cplx_of<T>::type *tw;
  int nx, ny, nz, single;
  double scale;
  Geo geo;
};

template <int DIR, typename T> __global__ void __launch_bounds__(256) k_user_x(const UserArgs<T> A) {
  typedef typename cplx_of<T>::type C;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  C *sm = reinterpret_cast<C *>(smem_raw);
  const int nx = A.nx, nxh = nx / 2 + 1;
  const long long R = (long long)A.ny * A.nz;
  const long long ra = A.single ? blockIdx.x : 2ll * blockIdx.x, rb = ra + 1; /* user row ids z*ny + y */
  const long long ia = (ra % A.ny) * A.nz + ra / A.ny;                          /* internal y*nz + z    */
  const long long ib = A.single ? ia : (rb % A.ny) * A.nz + rb / A.ny;
  if (DIR < 0) {
    for (int x = threadIdx.x; x < nx; x += blockDim.x)
      sm[geo_pad(A.geo, x)] = mk<C, T>(A.real[ra * nx + x], A.single ? (T)0 : A.real[rb * nx + x]);
    __syncthreads();
    fft_dif<-1, T>(A.geo, sm, A.tw, 1, 1);
    for (int kx = threadIdx.x; kx < nxh; kx += blockDim.x) {
      const C z = sm[geo_pad(A.geo, geo_slot(A.geo, kx))];
      const C zm = sm[geo_pad(A.geo, geo_slot(A.geo, (nx - kx) & (nx - 1)))];
      const T h = (T)0.5;
      A.arr[(size_t)kx * R + ia] = mk<C, T>(h * (z.x + zm.x), h * (z.y - zm.y));
      if (!A.single) A.arr[(size_t)kx * R + ib] = mk<C, T>(h * (z.y + zm.y), h * (zm.x - z.x));
    }
  } else {
    for (int kx = threadIdx.x; kx < nxh; kx += blockDim.x) {
      C a = A.arr[(size_t)kx * R + ia];
      C b = A.single ? mk<C, T>((T)0, (T)0) : A.arr[(size_t)kx * R + ib];
      if (kx == 0 || 2 * kx == nx) { a.y = (T)0; b.y = (T)0; }
      sm[geo_pad(A.geo, kx)] = mk<C, T>(a.x - b.y, a.y + b.x);
      if (kx > 0 && 2 * kx < nx) sm[geo_pad(A.geo, nx - kx)] = mk<C, T>(a.x + b.y, b.x - a.y);
    }
    __syncthreads();
    fft_dif<+1, T>(A.geo, sm, A.tw, 1, 1);
    const T sc = (T)A.scale;
    for (int x = threadIdx.x; x < nx; x += blockDim.x) {
      const C z = sm[geo_pad(A.geo, geo_slot(A.geo, x))];
      A.real[ra * nx + x] = z.x * sc;
      if (!A.single) A.real[rb * nx + x] = z.y * sc;
    }
  }
}

/* internal [kx][r] -> logical [r'][kx] (r' = z*ny + y) for pss_get_field_fourier */
template <typename T>
__global__ void k_to_logical(const typename cplx_of<T>::type *arr, typename cplx_of<T>::type *out, int nxh, int ny, int nz) {
  const long long total = (long long)nxh * ny * nz;
  for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < total; i += (long long)gridDim.x * blockDim.x) {
    const int kx = (int)(i % nxh);
    const long long rp = i / nxh;
    const long long y = rp % ny, z = rp / ny;
    out[i] = arr[(size_t)kx * ny * nz + y * nz + z];
  }
}

/* logical [r'][kx] -> internal [kx][r] for pss_set_field_fourier (checkpoint restore) */
template <typename T>
__global__ void k_from_logical(const typename cplx_of<T>::type *in, typename cplx_of<T>::type *arr, int nxh, int ny, int nz) {
  const long long total = (long long)nxh * ny * nz;
  for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < total; i += (long long)gridDim.x * blockDim.x) {
    const int kx = (int)(i % nxh);
    const long long rp = i / nxh;
    const long long y = rp % ny, z = rp / ny;
    arr[(size_t)kx * ny * nz + y * nz + z] = in[i];
  }
}

/* noise test hook: Philox words and z per logical mode */
template <typename T>
__global__ void k_debug_noise(const __grid_constant__ Program P, unsigned rep, int field, unsigned long long step, uint32_t *bits,
                              typename cplx_of<T>::type *z) {
  const long long total = (long long)P.nxh * P.n[1] * P.n[2];
  for (long long m = blockIdx.x * (long long)blockDim.x + threadIdx.x; m < total; m += (long long)gridDim.x * blockDim.x) {
    const int k0 = (int)(m % P.nxh);
    const long long rp = m / P.nxh;
    const int k1 = (int)(rp % P.n[1]), k2 = (int)(rp / P.n[1]);
    if (bits) {
      uint32_t w[4];
      noise_block(P, rep, field, step, m, w);
      bits[4 * m] = w[0]; bits[4 * m + 1] = w[1]; bits[4 * m + 2] = w[2]; bits[4 * m + 3] = w[3];
    }
    if (z) z[m] = noise_z<T>(P, rep, field, step, k0, k1, k2);
  }
}

/* ------------------------------------------------------------------------------------------ */
/* 1D: the whole lattice fits one CTA; nsteps full steps per launch, state in
 * global memory (nxh complex per dynamic field), everything else in shared memory. */
template <typename T> struct Step1dArgs {
  typename cplx_of<T>::type *state; /* [ndyn][nxh] */
  const typename cplx_of<T>::type *tw;
  long long M;
  int nx;
  long long nsteps;
  unsigned long long step0;
  Geo geo;
};

template <typename T>
__global__ void __launch_bounds__(256) k_step1d(const __grid_constant__ Program P, const Step1dArgs<T> A) {
  typedef typename cplx_of<T>::type C;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  C *sm = reinterpret_cast<C *>(smem_raw);
  const int nx = A.nx, nxh = nx / 2 + 1;
  const int RS = P.nfac + P.ngrp;
  const int tid = threadIdx.x, nt = blockDim.x;
  const C zero = mk<C, T>((T)0, (T)0);
  C *const st1 = A.state + (size_t)blockIdx.x * P.ndyn * A.M; /* one CTA per ensemble replica */
  for (long long st = 0; st < A.nsteps; ++st) {
    /* steps 1-3: factor operators, mask, C2R (imaginary row unused) */
    for (int idx = tid; idx < A.geo.npad * RS; idx += nt) sm[idx] = zero;
    __syncthreads();
    for (int kx = tid; kx < nxh; kx += nt) {
      const ModeQ<T> mq = make_mode<T>(P, kx, 0, 0);
      C phi[PSS_P_MAX_DYN];
#pragma unroll
      for (int i = 0; i < PSS_P_MAX_DYN; ++i) phi[i] = (i < P.ndyn) ? st1[(size_t)i * A.M + kx] : zero;
      for (int f = 0; f < P.nfac; ++f) {
        const DFactor &F = P.fac[f];
        if (!keep_axis(P.dealias, F.order, kx, nx)) continue;
        C v = zero;
        for (int e = F.lin_beg; e < F.lin_end; ++e) v = cadd(v, cmul(eval_op<T>(P, P.lin[e], mq), sel_src<PSS_P_MAX_DYN>(phi, P.lin[e].src)));
        v.x *= (T)P.invN;
        v.y *= (T)P.invN;
        if (kx == 0 || 2 * kx == nx) v.y = (T)0;
        sm[(size_t)geo_pad(A.geo, kx) * RS + f] = v;
        if (kx > 0 && 2 * kx < nx) sm[(size_t)geo_pad(A.geo, nx - kx) * RS + f] = mk<C, T>(v.x, -v.y);
      }
    }
    __syncthreads();
    if (P.nfac > 0) fft_dif<+1, T>(A.geo, sm, A.tw, P.nfac, RS);
    /* steps 3-4: products and R2C */
    for (int idx = tid; idx < nx; idx += nt) {
      C *srow = sm + (size_t)geo_pad(A.geo, idx) * RS;
      for (int g = 0; g < P.ngrp; ++g) {
        const DGroup &G = P.grp[g];
        T pa = (T)0;
        for (int t = G.term_beg; t < G.term_end; ++t) {
          const DTerm &tm = P.term[t];
          T ta = (T)tm.coef;
          for (int i = 0; i < tm.nf; ++i) ta *= srow[tm.f[i]].x;
          pa += ta;
        }
        srow[P.nfac + g] = mk<C, T>(pa, (T)0);
      }
    }
    __syncthreads();
    if (P.ngrp > 0) fft_dit<-1, T>(A.geo, sm + P.nfac, A.tw, P.ngrp, RS);
    /* steps 5-6: noise and Eq. 18 */
    for (int kx = tid; kx < nxh; kx += nt) {
      const ModeQ<T> mq = make_mode<T>(P, kx, 0, 0);
      const C *srow = sm + (size_t)geo_pad(A.geo, kx) * RS + P.nfac;
      C phi[PSS_P_MAX_DYN], out[PSS_P_MAX_DYN];
#pragma unroll
      for (int i = 0; i < PSS_P_MAX_DYN; ++i) phi[i] = (i < P.ndyn) ? st1[(size_t)i * A.M + kx] : zero;
#pragma unroll
      for (int i = 0; i < PSS_P_MAX_DYN; ++i) {
        out[i] = zero;
        if (i < P.ndyn) {
          const DDyn &d = P.dyn[i];
          C N = zero;
          for (int g = 0; g < P.ngrp; ++g)
            if (P.grp[g].target == i) N = cadd(N, cmul(eval_op<T>(P, P.grp[g].outer, mq), srow[g]));
          for (int e = d.lin_beg; e < d.lin_end; ++e) N = cadd(N, cmul(eval_op<T>(P, P.lin[e], mq), sel_src<PSS_P_MAX_DYN>(phi, P.lin[e].src)));
          C L = zero;
          for (int e = d.lhs_beg; e < d.lhs_end; ++e) L = csub(L, eval_op<T>(P, P.lin[e], mq));
          C num = mk<C, T>(phi[i].x + (T)P.dt * N.x, phi[i].y + (T)P.dt * N.y);
          if (d.noisy) {
            const T amp = noise_amp<T>(d, mq);
            const C z = noise_z<T>(P, blockIdx.x, d.field_id, A.step0 + (unsigned long long)st, kx, 0, 0);
            num.x += amp * z.x;
            num.y += amp * z.y;
          }
          const C den = mk<C, T>((T)1 - (T)P.dt * L.x, -(T)P.dt * L.y);
          const T id = (T)1 / (den.x * den.x + den.y * den.y);
          const C q = cmulc(num, den);
          out[i] = mk<C, T>(q.x * id, q.y * id);
        }
      }
#pragma unroll
      for (int i = 0; i < PSS_P_MAX_DYN; ++i)
        if (i < P.ndyn) st1[(size_t)i * A.M + kx] = out[i];
    }
    __syncthreads();
  }
}

#endif
