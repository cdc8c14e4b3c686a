/*
 * pss_fused2d.cuh — the whole time step of a 1024 x 1024 fp32 single-field system as ONE
 * persistent cooperative kernel that runs nsteps steps per launch: 64 threads per 1024-point line, 16 values per
 * thread, the Fourier state phi_q in REGISTERS for the whole launch.
 *
 * Why: at 1024^2 the state (4.2 MB) and both intermediates are L2-resident, so a step is bound by launch gaps,
 * synchronisation and instruction issue, not by DRAM.  A first design with one warp per line (32 values per thread,
 * profiles/r1_v2_summary.md) was bound by the latency chain of ONE warp per scheduler (issue active 27 %, DRAM
 * idle).  Here every line is spread over 64 threads (8 transform warps per CTA, two per scheduler), which halves the
 * per-line critical path and gives the schedulers a second transform warp to hide shared-memory and dependency
 * latency; the noise is drawn by 8 further warps, decoupled from the grid barrier (named-barrier producer/consumer
 * hand-off, one step ahead); setmaxnreg moves registers from the noise warps (64) to the transform warps (184).
 *
 * Transform.  1024 = 16 x 16 x 4, three register passes around two shared-memory exchanges.
 *   index digits   natural   n = 64 n1 + 4 n2 + n3        (n1, n2 in [0,16), n3 in [0,4))
 *                  spectral  k = k1 + 16 k2 + 256 k3      (k1, k2 in [0,16), k3 in [0,4))
 *   n k mod 1024 = 64 n1 k1 + (4 n2 + n3) k1 + 64 n2 k2 + 16 n3 k2 + 256 n3 k3
 *   "D_nat"  : thread tq (0..63) holds x[64 a + tq], a = 0..15                 (register index a = n1)
 *   "D_spec" : thread tq = k1 + 16 c holds X[k1 + 16 (4 c + j) + 256 k3] at register r = j + 4 k3
 *   fwd_dif : D_nat -> D_spec  (radix 16 over n1, twiddle T1, radix 16 over n2, twiddle T2, radix 4 over n3)
 *   fwd_dit : D_spec -> D_nat  (the transposed graph: radix 4 over k3, T2, radix 16 over k2, T1, radix 16 over k1)
 *   Both are FORWARD transforms (the DFT matrix is symmetric); inverses are conj(fwd_dit(conj(.))), so one copy of
 *   each graph serves the four transforms of a step:
 *     phase R (rows, x axis):     E -> [dit] real space, product -> [dif] -> Z
 *     phase C (columns, y axis):  Z -> [dif] -> Eq. 15/16/18 on the register-resident state -> [dit] -> E
 *
 * Thread map (both phases): transform thread tid in [0,256): L = tid & 3 is the line of this CTA (4 packed rows in
 * phase R, 4 columns in phase C), tq = tid >> 2 its slot in the line.  A warp therefore holds 8 consecutive tq of
 * all four lines: every global access of a warp is 4 segments of 64 B or one run of 256 B, and the shared-memory
 * exchanges are conflict-free with row pitch 65 and line pitch = 4 mod 16 (8-byte units).
 *
 * Exchange arrays in L2 (float2), laid out for their consumer:
 *   Z [kx' in 0..1023][p in 0..511]      written by phase R, read by phase C      (p = packed row pair (p, p+512))
 *   E [p/4][kx' in 0..1023][p%4]         written by phase C, read by phase R
 *   state [kx in 0..512][ky in 0..1023]  the library's internal layout; lives in registers during the launch
 */
#ifndef PSS_FUSED2D_CUH
#define PSS_FUSED2D_CUH
#include "pss_pointwise.cuh"

namespace f2d {

constexpr int N = 1024;
constexpr int NP = 512;
constexpr int TT = 256;               /* transform threads (warps 0-7)                     */
constexpr int NT = 256;               /* noise threads (warps 8-15)                        */
constexpr int THREADS = TT + NT;
constexpr int NCTA = 129;             /* 128 CTAs own 4 packed rows + 4 columns; CTA 128 owns column kx = 512 */
constexpr int PITCH = 65;             /* k1-row pitch of an exchange buffer (float2)       */
constexpr int BUF = 16 * PITCH + 4;   /* one line's exchange buffer; = 4 mod 16            */
constexpr size_t SMEM_BYTES = (size_t)(4 * BUF + 2 * 16 * TT) * sizeof(float2) + (size_t)16 * TT * sizeof(float4);


struct Args {
  float2 *state;
  float2 *E;
  float2 *Z;
  const float2 *tw;              /* tw[j] = exp(-2 pi i j / 1024) */
  unsigned long long *bar;       /* grid barrier counter, monotonically increasing */
  unsigned long long bar_base;   /* its value when this launch starts              */
  long long nsteps;
  unsigned long long step0;
  int prologue;                  /* 1: E is stale (after pss_set_field): rebuild it from the state first */
  long long rep_stride;          /* k_fused2d_pair: elements between the arrays of replica r and r+1 (state, E, Z alike) */
};

__device__ __forceinline__ float2 ldcg2(const float2 *p) { return __ldcg(p); }

/* unit Hermitian complex Gaussian of logical mode (kx, ky) on the 1024 x 513 half-spectrum; `plane`: kx is 0 or 512.
 * Same stream as noise_z<float>() of pss_pointwise.cuh (Eq. 16, 134). */
__device__ __forceinline__ float2 noise_mode(const NoiseKey &K, int kx, int ky, bool plane) {
  uint32_t m = (uint32_t)(ky * (N / 2 + 1) + kx);
  bool self = false, other = false;
  if (plane) {
    const int kyp = (N - ky) & (N - 1);
    const uint32_t mp = (uint32_t)(kyp * (N / 2 + 1) + kx);
    self = (mp == m);
    other = (mp < m);
    m = other ? mp : m;
  }
  uint32_t w0, w1;
  philox_w01(m, 0u, K, w0, w1);
  float2 z = box_muller_half(w0, w1);
  if (plane) {
    if (self) z = make_float2(z.x * 1.41421356237309504880f, 0.f);
    else if (other) z.y = -z.y;
  }
  return z;
}

/* barrier ids: 1 = the 256 transform threads; 2,3 = z buffer full; 4,5 = z buffer empty (512 threads each) */
__device__ __forceinline__ void tsync() { asm volatile("bar.sync 1, 256;" ::: "memory"); }
__device__ __forceinline__ void nb_sync(int id) { asm volatile("bar.sync %0, 512;" ::"r"(id) : "memory"); }
__device__ __forceinline__ void nb_arrive(int id) {
  __threadfence_block();
  asm volatile("bar.arrive %0, 512;" ::"r"(id) : "memory");
}

__device__ __forceinline__ float2 cmulf(float2 a, float2 w) {
  return make_float2(a.x * w.x - a.y * w.y, a.x * w.y + a.y * w.x);
}

/* 4-point forward DFT, natural in, natural out */
__device__ __forceinline__ void dft4(float2 &x0, float2 &x1, float2 &x2, float2 &x3) {
  const float2 s02 = cadd(x0, x2), d02 = csub(x0, x2);
  const float2 s13 = cadd(x1, x3), d13 = csub(x1, x3);
  x0 = cadd(s02, s13);
  x2 = csub(s02, s13);
  x1 = make_float2(d02.x + d13.y, d02.y - d13.x); /* d02 - i d13 */
  x3 = make_float2(d02.x - d13.y, d02.y + d13.x); /* d02 + i d13 */
}

struct Lane {
  float2 *xl;       /* this line's exchange buffer                 */
  float2 t1[16];    /* t1[k1] = w1024^(k1 tq)   (registers)        */
  float2 t2[16];    /* t2[k2] = w64^(k2 (tq & 3))                  */
  int tq;
};

/* D_nat -> D_spec.  The caller guarantees that nobody still reads the exchange buffer (tsync before). */
__device__ __forceinline__ void fwd_dif(float2 (&v)[16], const Lane &ln) {
  dft_reg<4, -1>(v);
#pragma unroll
  for (int k1 = 0; k1 < 16; ++k1) {
    float2 x = v[k1];
    if (k1 > 0) x = cmulf(x, ln.t1[k1]);
    ln.xl[k1 * PITCH + ln.tq] = x;
  }
  tsync();
  float2 *base = ln.xl + (ln.tq >> 2) * PITCH + (ln.tq & 3);
#pragma unroll
  for (int n2 = 0; n2 < 16; ++n2) v[n2] = base[4 * n2];
  dft_reg<4, -1>(v);
#pragma unroll
  for (int k2 = 0; k2 < 16; ++k2) {
    float2 x = v[k2];
    if (k2 > 0) x = cmulf(x, ln.t2[k2]);
    base[4 * k2] = x;
  }
  tsync();
  const float2 *b2 = ln.xl + (ln.tq & 15) * PITCH + 16 * (ln.tq >> 4);
#pragma unroll
  for (int j = 0; j < 4; ++j) {
    float2 a0 = b2[4 * j], a1 = b2[4 * j + 1], a2 = b2[4 * j + 2], a3 = b2[4 * j + 3];
    dft4(a0, a1, a2, a3);
    v[j] = a0; v[j + 4] = a1; v[j + 8] = a2; v[j + 12] = a3;
  }
}

/* D_spec -> D_nat (also a forward transform).  Same guarantee as fwd_dif. */
__device__ __forceinline__ void fwd_dit(float2 (&v)[16], const Lane &ln) {
  float2 *b2 = ln.xl + (ln.tq & 15) * PITCH + 16 * (ln.tq >> 4);
#pragma unroll
  for (int j = 0; j < 4; ++j) {
    float2 a0 = v[j], a1 = v[j + 4], a2 = v[j + 8], a3 = v[j + 12];
    dft4(a0, a1, a2, a3);
    b2[4 * j] = a0; b2[4 * j + 1] = a1; b2[4 * j + 2] = a2; b2[4 * j + 3] = a3;
  }
  tsync();
  float2 *base = ln.xl + (ln.tq >> 2) * PITCH + (ln.tq & 3);
#pragma unroll
  for (int k2 = 0; k2 < 16; ++k2) {
    float2 x = base[4 * k2];
    if (k2 > 0) x = cmulf(x, ln.t2[k2]);
    v[k2] = x;
  }
  dft_reg<4, -1>(v);
#pragma unroll
  for (int n2 = 0; n2 < 16; ++n2) base[4 * n2] = v[n2];
  tsync();
#pragma unroll
  for (int k1 = 0; k1 < 16; ++k1) {
    float2 x = ln.xl[k1 * PITCH + ln.tq];
    if (k1 > 0) x = cmulf(x, ln.t1[k1]);
    v[k1] = x;
  }
  dft_reg<4, -1>(v);
}

/* grid barrier over the transform threads of all CTAs (the noise warps never take part): one monotonically
 * increasing 64-bit counter.  Thread 0 arrives with a release reduction once the CTA's 256 threads have passed
 * tsync (their data stores happen-before it through the CTA barrier) and polls with acquire loads; data crossing the
 * barrier is read with ld.global.cg. */
__device__ __forceinline__ void grid_barrier(unsigned long long *ctr, unsigned long long target) {
  tsync();
  if ((threadIdx.x & (TT - 1)) == 0) {
    asm volatile("red.release.gpu.global.add.u64 [%0], 1;" ::"l"(ctr) : "memory");
    unsigned long long v, t0 = 0;
    unsigned spins = 0;
    for (;;) {
      asm volatile("ld.acquire.gpu.global.u64 %0, [%1];" : "=l"(v) : "l"(ctr) : "memory");
      if (v >= target) break;
      if (((++spins) & 0x3fffu) == 0) { /* watchdog on the wall clock (30 s): fail the launch instead of hanging the GPU */
        unsigned long long t;
        asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t));
        if (t0 == 0) t0 = t;
        else if (t - t0 > 30000000000ull) __trap();
      }
    }
  }
  tsync();
}

/* ------------------------------------------------------------------------------------------ */
template <bool PRUNE>
__global__ void __launch_bounds__(THREADS, 1) k_fused2d(const __grid_constant__ Program P, const Args A) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  float2 *xs = reinterpret_cast<float2 *>(smem_raw);           /* [4][BUF] exchange buffers                 */
  float2 *zbuf = xs + 4 * BUF;                                 /* [2][16 r][256 tid] unit noise z           */
  float4 *tab = reinterpret_cast<float4 *>(zbuf + 2 * 16 * TT); /* [16 r][256 tid] per-mode coefficients     */

  const int tid = threadIdx.x & (TT - 1);
  const bool noisew = threadIdx.x >= TT;
  const int L = tid & 3, tq = tid >> 2;
  const int b = blockIdx.x;
  /* phase C ownership: column of line L; spectral index of register r: ky = kyb + 16 j + 256 k3, r = j + 4 k3 */
  int kx;
  if (b < 128) kx = (L < 2) ? (2 * b + L) : (256 + 2 * b + (L - 2));
  else kx = (L == 0) ? 512 : -1;
  const bool colw = kx >= 0;
  const int kxm = colw ? ((N - kx) & (N - 1)) : 0;
  const bool selfc = (kx == 0) || (kx == 512);
  const int kyb = (tq & 15) + 64 * (tq >> 4);
  const DDyn &D0 = P.dyn[0];
  const bool noisy = D0.noisy != 0;
  const long long nphase = A.nsteps + (A.prologue ? 1 : 0);

  if (noisew) {
    asm volatile("setmaxnreg.dec.sync.aligned.u32 64;"); /* hand registers to the transform warps */
    /* ============ noise warps: z(step s+1) is drawn while the transform warps work on step s ============ */
    if (!noisy || A.nsteps <= 0) return;
    NoiseKey K;
    K.k0 = P.seed_lo;
    K.k1 = P.seed_hi;
#pragma unroll 1
    for (long long s = 0; s < A.nsteps; ++s) {
      const unsigned long long step = A.step0 + (unsigned long long)s;
      K.c2 = (uint32_t)(step & 0xffffffffu);
      K.c3 = (uint32_t)((((step >> 32) & 0xffffu) << 16) | ((uint32_t)D0.field_id & 0xffffu));
      const int buf = (int)(s & 1);
      if (s >= 2) nb_sync(4 + buf); /* the transform warps have consumed z(s-2) */
      if (colw) {
        float2 *zw = zbuf + (size_t)buf * 16 * TT + tid;
#pragma unroll 2
        for (int r = 0; r < 16; ++r)
          zw[r * TT] = noise_mode(K, kx, kyb + 16 * (r & 3) + 256 * (r >> 2), selfc);
      }
      nb_arrive(2 + buf);
    }
    return;
  }

  /* ================= transform warps ================= */
  asm volatile("setmaxnreg.inc.sync.aligned.u32 184;"); /* 8 x 32 x (64 + 184) = 63488 <= 65536 registers */
  const bool need_inv = colw && keep_axis(P.dealias, P.fac[0].order, kx, N);
  const bool roww = b < 128;
  Lane ln;
  ln.xl = xs + L * BUF;
  ln.tq = tq;
#pragma unroll
  for (int i = 0; i < 16; ++i) {
    ln.t1[i] = A.tw[(i * tq) & (N - 1)];
    ln.t2[i] = A.tw[(16 * i * (tq & 3)) & (N - 1)];
  }

  /* per-mode coefficients: (dt*outer, 1/(1 - dt L), noise amplitude, factor op * mask / N), and the state */
  float2 st[16];
  {
    const float dt = (float)P.dt, invN = (float)P.invN;
#pragma unroll 1
    for (int r = 0; r < 16; ++r) {
      float4 t = make_float4(0.f, 0.f, 0.f, 0.f);
      if (colw) {
        const int ky = kyb + 16 * (r & 3) + 256 * (r >> 2);
        const ModeQ<float> mq = make_mode<float>(P, kx, ky, 0);
        t.x = dt * eval_op<float>(P, P.grp[0].outer, mq).x;
        float Lq = 0.f;
        for (int e = D0.lhs_beg; e < D0.lhs_end; ++e) Lq -= eval_op<float>(P, P.lin[e], mq).x;
        t.y = 1.0f / (1.0f - dt * Lq);
        t.z = noisy ? noise_amp<float>(D0, mq) : 0.f;
        float fc = 0.f;
        if (need_inv && keep_axis(P.dealias, P.fac[0].order, ky, N)) {
          for (int e = P.fac[0].lin_beg; e < P.fac[0].lin_end; ++e) fc += eval_op<float>(P, P.lin[e], mq).x;
          fc *= invN;
        }
        t.w = fc;
      }
      tab[r * TT + tid] = t;
      if (!noisy) {
        zbuf[r * TT + tid] = make_float2(0.f, 0.f);
        zbuf[16 * TT + r * TT + tid] = make_float2(0.f, 0.f);
      }
    }
#pragma unroll
    for (int r = 0; r < 16; ++r)
      st[r] = colw ? A.state[(size_t)kx * N + kyb + 16 * (r & 3) + 256 * (r >> 2)] : make_float2(0.f, 0.f);
  }
  /* sum_t coef_t r^nf_t = r^2 (c2 + r (c3 + r c4)): the product terms of the single group (Eq. 11) */
  float c2 = 0.f, c3 = 0.f, c4 = 0.f;
  for (int t = P.grp[0].term_beg; t < P.grp[0].term_end; ++t) {
    const float c = (float)P.term[t].coef;
    if (P.term[t].nf == 2) c2 += c;
    else if (P.term[t].nf == 3) c3 += c;
    else c4 += c;
  }
  unsigned long long bar_target = A.bar_base;
  tsync();

  float2 v[16];
#pragma unroll 1
  for (long long it = 0; it < nphase; ++it) {
    const bool pro = A.prologue && it == 0;
    const long long ls = it - (A.prologue ? 1 : 0);
    const int zb = (int)(ls & 1);
    if (pro) {
#pragma unroll
      for (int r = 0; r < 16; ++r) {
        const float fc = tab[r * TT + tid].w;
        v[r] = make_float2(st[r].x * fc, -st[r].y * fc);
      }
    }
    /* t = 0: inverse-x of E   t = 1: forward-x of the product   (phase R)
     * t = 2: forward-y of Z   t = 3: inverse-y of the next factor (phase C) */
#pragma unroll 1
    for (int t = pro ? 3 : 0; t < 4; ++t) {
      if (t == 0) {
        if (roww) {
          const float2 *Eb = A.E + ((size_t)b * N) * 4 + L + (size_t)kyb * 4;
#pragma unroll
          for (int r = 0; r < 16; ++r) {
            if (!PRUNE || (r >> 2) == 0 || (r >> 2) == 3) {
              const float2 e = ldcg2(Eb + (size_t)(16 * (r & 3) + 256 * (r >> 2)) * 4);
              v[r] = make_float2(e.x, -e.y);
            } else {
              v[r] = make_float2(0.f, 0.f);
            }
          }
        }
      } else if (t == 2) {
        if (colw) {
          const float2 *Z1 = A.Z + (size_t)kx * NP + tq, *Z2 = A.Z + (size_t)kxm * NP + tq;
#pragma unroll
          for (int a = 0; a < 8; ++a) {
            const float2 za = ldcg2(Z1 + 64 * a), zc = ldcg2(Z2 + 64 * a);
            v[a] = make_float2(0.5f * (za.x + zc.x), 0.5f * (za.y - zc.y));     /* row y = 64 a + tq       */
            v[a + 8] = make_float2(0.5f * (za.y + zc.y), 0.5f * (zc.x - za.x)); /* row y = 64 a + tq + 512 */
          }
        } else {
#pragma unroll
          for (int a = 0; a < 16; ++a) v[a] = make_float2(0.f, 0.f);
        }
      }
      if (t == 0 || t == 3) fwd_dit(v, ln); else fwd_dif(v, ln);
      if (t == 0) {
        /* conj(v[a]) = a(x) + i b(x) at x = 64 a + tq: rows p and p + 512 in real space */
#pragma unroll
        for (int a = 0; a < 16; ++a) {
          const float ra = v[a].x, rb = -v[a].y;
          v[a] = make_float2(ra * ra * (c2 + ra * (c3 + ra * c4)), rb * rb * (c2 + rb * (c3 + rb * c4)));
        }
        tsync(); /* everybody has left fwd_dit's last exchange read before fwd_dif writes */
      } else if (t == 1) {
        if (roww) {
          float2 *Zb = A.Z + (size_t)kyb * NP + 4 * b + L;
#pragma unroll
          for (int r = 0; r < 16; ++r) Zb[(size_t)(16 * (r & 3) + 256 * (r >> 2)) * NP] = v[r];
        }
        bar_target += NCTA;
        grid_barrier(A.bar, bar_target);
      } else if (t == 2) {
        /* v[r] = P_q at ky(r): Eq. 15 + Eq. 16 + Eq. 18, then the next factor's (conjugated) input */
        if (noisy) nb_sync(2 + zb);
        const float2 *myz = zbuf + (size_t)zb * 16 * TT + tid;
#pragma unroll
        for (int r = 0; r < 16; ++r) {
          const float4 tt = tab[r * TT + tid];
          const float2 z = myz[r * TT];
          const float2 pq = v[r];
          const float nx = (st[r].x + tt.x * pq.x) + tt.z * z.x;
          const float ny = (st[r].y + tt.x * pq.y) + tt.z * z.y;
          st[r] = make_float2(nx * tt.y, ny * tt.y);
          v[r] = make_float2(st[r].x * tt.w, -st[r].y * tt.w);
        }
        if (noisy && ls + 2 < A.nsteps) nb_arrive(4 + zb);
        tsync();
      } else {
        /* conj(v[a]) = psi_x[kx][y = 64 a + tq]; pack rows y (A) and y + 512 (B) */
        if (need_inv) {
#pragma unroll
          for (int a = 0; a < 8; ++a) {
            const float2 av = make_float2(v[a].x, -v[a].y);
            const float2 bv = make_float2(v[a + 8].x, -v[a + 8].y);
            const int p = 64 * a + tq;
            float2 *e = A.E + ((size_t)(p >> 2) * N) * 4 + (p & 3);
            if (selfc) {
              e[(size_t)kx * 4] = make_float2(av.x, bv.x);                  /* the C2R keeps the real part there */
            } else {
              e[(size_t)kx * 4] = make_float2(av.x - bv.y, av.y + bv.x);    /* A + iB              */
              e[(size_t)kxm * 4] = make_float2(av.x + bv.y, bv.x - av.y);   /* conj(A) + i conj(B) */
            }
          }
        }
        bar_target += NCTA;
        grid_barrier(A.bar, bar_target);
      }
    }
  }

  if (colw && A.nsteps > 0) {
#pragma unroll
    for (int r = 0; r < 16; ++r) A.state[(size_t)kx * N + kyb + 16 * (r & 3) + 256 * (r >> 2)] = st[r];
  }
}

/* ------------------------------------------------------------------------------------------ */
/* TWO ensemble replicas (seed, seed + 1; pss_set_replicas) in one persistent launch.  A single system cannot
 * overlap its two bulk-synchronous L2 exchanges with anything but the noise; two independent replicas can: the
 * loads of replica 1 are in flight while replica 0 is transformed, the stores of replica 0 drain while replica 1
 * is transformed, and each grid barrier is paid once per two replica-steps.  Per replica the arithmetic is exactly
 * that of k_fused2d (bit-identical results).  Differences in storage: the states live in shared memory (the
 * registers hold the prefetched loads instead) and z is single-buffered per replica. */
constexpr int NRE = 2;
constexpr size_t SMEM_BYTES_PAIR = (size_t)(4 * BUF + 2 * NRE * 16 * TT) * sizeof(float2) + (size_t)16 * TT * sizeof(float4);

template <bool PRUNE>
__global__ void __launch_bounds__(THREADS, 1) k_fused2d_pair(const __grid_constant__ Program P, const Args A) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  float2 *xs = reinterpret_cast<float2 *>(smem_raw);                  /* [4][BUF] exchange buffers            */
  float2 *zbuf = xs + 4 * BUF;                                        /* [NRE][16 r][256 tid] unit noise z    */
  float2 *stS = zbuf + NRE * 16 * TT;                                 /* [NRE][16 r][256 tid] state phi_q     */
  float4 *tab = reinterpret_cast<float4 *>(stS + NRE * 16 * TT);      /* [16 r][256 tid] per-mode coefficients */

  const int tid = threadIdx.x & (TT - 1);
  const bool noisew = threadIdx.x >= TT;
  const int L = tid & 3, tq = tid >> 2;
  const int b = blockIdx.x;
  int kx;
  if (b < 128) kx = (L < 2) ? (2 * b + L) : (256 + 2 * b + (L - 2));
  else kx = (L == 0) ? 512 : -1;
  const bool colw = kx >= 0;
  const int kxm = colw ? ((N - kx) & (N - 1)) : 0;
  const bool selfc = (kx == 0) || (kx == 512);
  const int kyb = (tq & 15) + 64 * (tq >> 4);
  const DDyn &D0 = P.dyn[0];
  const bool noisy = D0.noisy != 0;

  if (noisew) {
    asm volatile("setmaxnreg.dec.sync.aligned.u32 64;");
    if (!noisy || A.nsteps <= 0) return;
    const unsigned long long sd0 = (((unsigned long long)P.seed_hi) << 32) | (unsigned long long)P.seed_lo;
#pragma unroll 1
    for (long long s = 0; s < A.nsteps; ++s) {
      const unsigned long long step = A.step0 + (unsigned long long)s;
#pragma unroll 1
      for (int r = 0; r < NRE; ++r) {
        NoiseKey K;
        const unsigned long long sd = sd0 + (unsigned long long)r;
        K.k0 = (uint32_t)(sd & 0xffffffffu);
        K.k1 = (uint32_t)(sd >> 32);
        K.c2 = (uint32_t)(step & 0xffffffffu);
        K.c3 = (uint32_t)((((step >> 32) & 0xffffu) << 16) | ((uint32_t)D0.field_id & 0xffffu));
        if (s >= 1) nb_sync(4 + r); /* the transform warps have consumed z_r(s-1) */
        if (colw) {
          float2 *zw = zbuf + (size_t)r * 16 * TT + tid;
#pragma unroll 2
          for (int i = 0; i < 16; ++i)
            zw[i * TT] = noise_mode(K, kx, kyb + 16 * (i & 3) + 256 * (i >> 2), selfc);
        }
        nb_arrive(2 + r);
      }
    }
    return;
  }

  asm volatile("setmaxnreg.inc.sync.aligned.u32 184;");
  const bool need_inv = colw && keep_axis(P.dealias, P.fac[0].order, kx, N);
  const bool roww = b < 128;
  Lane ln;
  ln.xl = xs + L * BUF;
  ln.tq = tq;
#pragma unroll
  for (int i = 0; i < 16; ++i) {
    ln.t1[i] = A.tw[(i * tq) & (N - 1)];
    ln.t2[i] = A.tw[(16 * i * (tq & 3)) & (N - 1)];
  }
  {
    const float dt = (float)P.dt, invN = (float)P.invN;
#pragma unroll 1
    for (int i = 0; i < 16; ++i) {
      float4 t = make_float4(0.f, 0.f, 0.f, 0.f);
      const int ky = kyb + 16 * (i & 3) + 256 * (i >> 2);
      if (colw) {
        const ModeQ<float> mq = make_mode<float>(P, kx, ky, 0);
        t.x = dt * eval_op<float>(P, P.grp[0].outer, mq).x;
        float Lq = 0.f;
        for (int e = D0.lhs_beg; e < D0.lhs_end; ++e) Lq -= eval_op<float>(P, P.lin[e], mq).x;
        t.y = 1.0f / (1.0f - dt * Lq);
        t.z = noisy ? noise_amp<float>(D0, mq) : 0.f;
        float fc = 0.f;
        if (need_inv && keep_axis(P.dealias, P.fac[0].order, ky, N)) {
          for (int e = P.fac[0].lin_beg; e < P.fac[0].lin_end; ++e) fc += eval_op<float>(P, P.lin[e], mq).x;
          fc *= invN;
        }
        t.w = fc;
      }
      tab[i * TT + tid] = t;
      for (int r = 0; r < NRE; ++r) {
        stS[(size_t)r * 16 * TT + i * TT + tid] =
            colw ? A.state[(size_t)r * A.rep_stride + (size_t)kx * N + ky] : make_float2(0.f, 0.f);
        if (!noisy) zbuf[(size_t)r * 16 * TT + i * TT + tid] = make_float2(0.f, 0.f);
      }
    }
  }
  float c2 = 0.f, c3 = 0.f, c4 = 0.f;
  for (int t = P.grp[0].term_beg; t < P.grp[0].term_end; ++t) {
    const float c = (float)P.term[t].coef;
    if (P.term[t].nf == 2) c2 += c;
    else if (P.term[t].nf == 3) c3 += c;
    else c4 += c;
  }
  unsigned long long bar_target = A.bar_base;
  const long long nphase = A.nsteps + (A.prologue ? 1 : 0);
  tsync();

  float2 v[16], nx[16];
#pragma unroll 1
  for (long long it = 0; it < nphase; ++it) {
    const bool pro = A.prologue && it == 0;
    const long long ls = it - (A.prologue ? 1 : 0);
    /* ph = 0: rows (inverse-x, product, forward-x)   ph = 1: columns (forward-y, Eq. 15/16/18, inverse-y) */
#pragma unroll 1
    for (int ph = pro ? 1 : 0; ph < 2; ++ph) {
#pragma unroll 1
      for (int r = 0; r <= NRE; ++r) {
        /* software pipeline: issue the loads of replica r (into nx) before transforming replica r - 1 (in v) */
        const bool have_prev = r > 0;
        if (have_prev) {
          /* nx holds the raw loads of replica r - 1: turn them into the transform input */
          if (ph == 0) {
#pragma unroll
            for (int i = 0; i < 16; ++i) v[i] = make_float2(nx[i].x, -nx[i].y);
          } else if (!pro) {
#pragma unroll
            for (int a = 0; a < 8; ++a) {
              const float2 za = nx[a], zc = nx[a + 8];
              v[a] = make_float2(0.5f * (za.x + zc.x), 0.5f * (za.y - zc.y));
              v[a + 8] = make_float2(0.5f * (za.y + zc.y), 0.5f * (zc.x - za.x));
            }
          }
        }
        if (r < NRE && !pro) {
          if (ph == 0) {
            if (roww) {
              const float2 *Eb = A.E + (size_t)r * A.rep_stride + ((size_t)b * N) * 4 + L + (size_t)kyb * 4;
#pragma unroll
              for (int i = 0; i < 16; ++i) {
                if (!PRUNE || (i >> 2) == 0 || (i >> 2) == 3) nx[i] = ldcg2(Eb + (size_t)(16 * (i & 3) + 256 * (i >> 2)) * 4);
                else nx[i] = make_float2(0.f, 0.f);
              }
            } else {
#pragma unroll
              for (int i = 0; i < 16; ++i) nx[i] = make_float2(0.f, 0.f);
            }
          } else {
            if (colw) {
              const float2 *Z1 = A.Z + (size_t)r * A.rep_stride + (size_t)kx * NP + tq;
              const float2 *Z2 = A.Z + (size_t)r * A.rep_stride + (size_t)kxm * NP + tq;
#pragma unroll
              for (int a = 0; a < 8; ++a) { nx[a] = ldcg2(Z1 + 64 * a); nx[a + 8] = ldcg2(Z2 + 64 * a); }
            } else {
#pragma unroll
              for (int a = 0; a < 16; ++a) nx[a] = make_float2(0.f, 0.f);
            }
          }
        }
        if (!have_prev) continue;
        const int rr = r - 1; /* the replica being transformed */
        float2 *myst = stS + (size_t)rr * 16 * TT + tid;
        if (ph == 0) {
          fwd_dit(v, ln);
#pragma unroll
          for (int a = 0; a < 16; ++a) {
            const float ra = v[a].x, rb = -v[a].y;
            v[a] = make_float2(ra * ra * (c2 + ra * (c3 + ra * c4)), rb * rb * (c2 + rb * (c3 + rb * c4)));
          }
          tsync();
          fwd_dif(v, ln);
          if (roww) {
            float2 *Zb = A.Z + (size_t)rr * A.rep_stride + (size_t)kyb * NP + 4 * b + L;
#pragma unroll
            for (int i = 0; i < 16; ++i) Zb[(size_t)(16 * (i & 3) + 256 * (i >> 2)) * NP] = v[i];
          }
          tsync();
        } else {
          if (!pro) {
            fwd_dif(v, ln);
            if (noisy) nb_sync(2 + rr);
            const float2 *myz = zbuf + (size_t)rr * 16 * TT + tid;
#pragma unroll
            for (int i = 0; i < 16; ++i) {
              const float4 tt = tab[i * TT + tid];
              const float2 z = myz[i * TT];
              const float2 pq = v[i];
              const float2 so = myst[i * TT];
              const float nxr = (so.x + tt.x * pq.x) + tt.z * z.x;
              const float nyr = (so.y + tt.x * pq.y) + tt.z * z.y;
              const float2 sn = make_float2(nxr * tt.y, nyr * tt.y);
              myst[i * TT] = sn;
              v[i] = make_float2(sn.x * tt.w, -sn.y * tt.w);
            }
            if (noisy && ls + 1 < A.nsteps) nb_arrive(4 + rr);
            tsync();
          } else {
#pragma unroll
            for (int i = 0; i < 16; ++i) {
              const float fc = tab[i * TT + tid].w;
              const float2 so = myst[i * TT];
              v[i] = make_float2(so.x * fc, -so.y * fc);
            }
          }
          fwd_dit(v, ln);
          if (need_inv) {
#pragma unroll
            for (int a = 0; a < 8; ++a) {
              const float2 av = make_float2(v[a].x, -v[a].y);
              const float2 bv = make_float2(v[a + 8].x, -v[a + 8].y);
              const int p = 64 * a + tq;
              float2 *e = A.E + (size_t)rr * A.rep_stride + ((size_t)(p >> 2) * N) * 4 + (p & 3);
              if (selfc) {
                e[(size_t)kx * 4] = make_float2(av.x, bv.x);
              } else {
                e[(size_t)kx * 4] = make_float2(av.x - bv.y, av.y + bv.x);
                e[(size_t)kxm * 4] = make_float2(av.x + bv.y, bv.x - av.y);
              }
            }
          }
          tsync();
        }
      }
      bar_target += NCTA;
      grid_barrier(A.bar, bar_target);
    }
  }

  if (colw && A.nsteps > 0) {
    for (int r = 0; r < NRE; ++r)
#pragma unroll
      for (int i = 0; i < 16; ++i)
        A.state[(size_t)r * A.rep_stride + (size_t)kx * N + kyb + 16 * (i & 3) + 256 * (i >> 2)] = stS[(size_t)r * 16 * TT + i * TT + tid];
  }
}

}  // namespace f2d
#endif
