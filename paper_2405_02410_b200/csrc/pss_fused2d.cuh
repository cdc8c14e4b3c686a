/*
 * pss_fused2d.cuh — the whole time step of a 1024 x 1024 fp32 single-field system as ONE
 * persistent cooperative kernel that runs nsteps steps per launch.
 *
 * Why: at 1024^2 the state (4.2 MB) and both intermediates are L2-resident and the 148 SMs each own only
 * ~7 rows / ~3.5 columns, so a step is bound by launch gaps, synchronisation and instruction issue, not by
 * DRAM.  This kernel keeps the Fourier state phi_q in REGISTERS for the whole launch, exchanges only the two
 * transposes per step through L2, and separates the two phases of a step with a hand-rolled grid barrier.
 *
 * Decomposition.  A 1024-point line transform is two radix-32 passes done entirely in registers (32 complex
 * values per thread) with one shared-memory exchange in between; no transposes are written.
 *
 *   phase C ("columns", fixed kx, transform along y; one warp per column, lane = y mod 32 / ky mod 32):
 *       read Z[kx], Z[N-kx]  ->  un-tangle the two real rows that rode one complex x-transform
 *       -> forward FFT-y -> outer operator, noise, Eq. 18 (state in registers)
 *       -> factor operator + de-aliasing mask + 1/N -> inverse FFT-y (input-pruned)
 *       -> write E[kx] = A + iB and E[N-kx] = conj(A) + i conj(B)   (rows y and y+512 packed)
 *   phase R ("rows", fixed packed row p = rows (p, p+512), transform along x; 4 packed rows per CTA,
 *            thread = (row, butterfly slot)):
 *       read E[p] -> inverse FFT-x (input-pruned) -> real-space product on the real and on the imaginary part
 *       -> forward FFT-x -> write Z[.][p]
 *
 *   Packing two real rows a, b as a + ib makes phase R a pure complex transform pair: all Hermitian
 *   bookkeeping (the extension for the C2R, the split after the R2C) is thread-local arithmetic in phase C,
 *   because a thread of phase C holds y and y+512 of its column in the same registers.
 *
 * Layouts (float2 elements).  Each exchange array is laid out for its CONSUMER (all loads fully coalesced);
 * producers write whole 32-byte sectors:
 *   Z [kx' in 0..1023][p in 0..511]           written by phase R (8 sectors per warp store), read by phase C
 *   E [p/4][kx' in 0..1023][p%4]              written by phase C (8 sectors per warp store), read by phase R
 *   state [kx in 0..512][ky in 0..1023]       the library's internal layout (set/get paths unchanged)
 *
 * Per-mode coefficients (dt*outer(q), 1/(1-dt L(q)), noise amplitude, factor operator * mask / N) do not
 * change from step to step: they are evaluated once per launch with the generic operator code and kept in
 * shared memory as one float4 per mode.
 */
#ifndef PSS_FUSED2D_CUH
#define PSS_FUSED2D_CUH
#include "pss_pointwise.cuh"

namespace f2d {

constexpr int N = 1024;          /* lattice points per axis          */
constexpr int NP = 512;          /* packed row pairs (p, p+512)      */
constexpr int PITCH = 33;        /* exchange row pitch (complex)     */
constexpr int XBUF = 32 * PITCH + 8; /* one exchange region; +64 B so that neighbouring regions differ by 16 banks */
constexpr int THREADS = 256;     /* warps 0-3 transform, warps 4-7 draw the next step's noise concurrently */
constexpr int NCTA = 129;        /* 128 CTAs own 4 packed rows and 4 columns each; CTA 128 owns column kx = 512 */
constexpr size_t SMEM_BYTES = (size_t)(N + 2 * 4 * XBUF + 2 * 4 * N) * sizeof(float2) + (size_t)4 * N * sizeof(float4);

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
  int dbg;                       /* timing experiments only (PSS_DBG): 1 no barrier wait, 2 no FFT, 4 no global ld/st, 8 no noise */
};

__device__ __forceinline__ float2 ldcg2(const float2 *p) { return __ldcg(p); }

/* d * exp(SGN * 2 pi i * j / 32), j in [0, 16) a compile-time constant after unrolling */
template <int SGN> __device__ __forceinline__ float2 mul_w32(float2 d, int j) {
  const float c1 = 0.98078528040323044913f, s1 = 0.19509032201612826785f;
  const float c2 = 0.92387953251128675613f, s2 = 0.38268343236508977173f;
  const float c3 = 0.83146961230254523708f, s3 = 0.55557023301960222474f;
  const float h = 0.70710678118654752440f;
  float wr, wi;
  switch (j) {
    case 0: return d;
    case 8: { float2 r; if (SGN < 0) { r.x = d.y; r.y = -d.x; } else { r.x = -d.y; r.y = d.x; } return r; }
    case 1: wr = c1; wi = s1; break;
    case 2: wr = c2; wi = s2; break;
    case 3: wr = c3; wi = s3; break;
    case 4: wr = h; wi = h; break;
    case 5: wr = s3; wi = c3; break;
    case 6: wr = s2; wi = c2; break;
    case 7: wr = s1; wi = c1; break;
    case 9: wr = -s1; wi = c1; break;
    case 10: wr = -s2; wi = c2; break;
    case 11: wr = -s3; wi = c3; break;
    case 12: wr = -h; wi = h; break;
    case 13: wr = -c3; wi = s3; break;
    case 14: wr = -c2; wi = s2; break;
    default: wr = -c1; wi = s1; break; /* 15 */
  }
  if (SGN < 0) wi = -wi;
  float2 r;
  r.x = d.x * wr - d.y * wi;
  r.y = d.x * wi + d.y * wr;
  return r;
}

__host__ __device__ constexpr int brev5(int i) {
  return ((i & 1) << 4) | ((i & 2) << 2) | (i & 4) | ((i & 8) >> 2) | ((i & 16) >> 4);
}

/* 32-point forward DFT in registers, decimation in frequency: natural order in,
 * X[k] = sum_n v[n] exp(-2 pi i n k/32) left at v[brev5(k)].  The inverse transforms are taken as
 * conj(FFT(conj(x))), so that the step loop holds ONE copy of this code (instruction-cache footprint). */
__device__ __forceinline__ void fft32(float2 (&v)[32]) {
#pragma unroll
  for (int len = 32; len >= 2; len >>= 1) {
    const int half = len >> 1;
#pragma unroll
    for (int blk = 0; blk < 32; blk += len) {
#pragma unroll
      for (int j = 0; j < half; ++j) {
        const float2 a = v[blk + j], b = v[blk + j + half];
        v[blk + j] = make_float2(a.x + b.x, a.y + b.y);
        v[blk + j + half] = mul_w32<-1>(make_float2(a.x - b.x, a.y - b.y), j * (32 / len));
      }
    }
  }
}

/* the four transform warps only (named barrier 1) */
__device__ __forceinline__ void fft_warps_sync() { asm volatile("bar.sync 1, 128;" ::: "memory"); }

/* one 1024-point forward transform of the line this thread group holds: thread `me` (0..31) enters with
 * v[n1] = x[32 n1 + me] and leaves with X[me + 32 k2] at v[brev5(k2)].  Two radix-32 passes around one
 * shared-memory exchange; tws[a*32+b] = exp(-2 pi i a b / 1024).  `cta_sync`: the 32 threads of the line
 * sit in different warps (phase R) -> barrier over the four transform warps, else (phase C, one warp per line) __syncwarp. */
__device__ __forceinline__ void fft1024(float2 (&v)[32], float2 *xs, const float2 *tws, int me, bool cta_sync) {
#pragma unroll 1
  for (int h = 0; h < 2; ++h) {
    fft32(v);
    if (h == 0) {
#pragma unroll
      for (int i = 0; i < 32; ++i) {
        float2 x = v[brev5(i)];
        if (i > 0) {
          const float2 w = tws[i * 32 + me];
          x = make_float2(x.x * w.x - x.y * w.y, x.x * w.y + x.y * w.x);
        }
        xs[i * PITCH + me] = x;
      }
      if (cta_sync) fft_warps_sync(); else __syncwarp();
#pragma unroll
      for (int i = 0; i < 32; ++i) v[i] = xs[me * PITCH + i];
    }
  }
}

/* unit Hermitian complex Gaussian of logical mode (kx, ky) on the 1024 x 513 half-spectrum; `plane`: kx is 0 or 512 */
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

__device__ __forceinline__ unsigned long long ld_relaxed_u64(const unsigned long long *p) {
  unsigned long long v;
  asm volatile("ld.relaxed.gpu.global.u64 %0, [%1];" : "=l"(v) : "l"(p) : "memory");
  return v;
}

/* grid barrier over all CTAs of the (cooperative, co-resident) grid, split in two.  `target` = counter value
 * once all arrived.  Data crossing the barrier is written with plain stores (made visible by the fence before
 * the arrival) and read with ld.global.cg, so the L1 never has to be invalidated while polling. */
__device__ __forceinline__ void grid_arrive(unsigned long long *ctr) {
  __syncthreads();
  if (threadIdx.x == 0) {
    __threadfence();
    atomicAdd(ctr, 1ULL);
  }
}
__device__ __forceinline__ void grid_wait(const unsigned long long *ctr, unsigned long long target) {
  if (threadIdx.x == 0) {
    while (ld_relaxed_u64(ctr) < target) { }
    __threadfence();
  }
  __syncthreads();
}
/* ------------------------------------------------------------------------------------------ */
template <bool PRUNE>
__global__ void __launch_bounds__(THREADS, 1) k_fused2d(const __grid_constant__ Program P, const Args A) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  float2 *tws = reinterpret_cast<float2 *>(smem_raw);          /* [32][32]                          */
  float2 *xa = tws + N;                                        /* [4][XBUF] exchange, inverse       */
  float2 *xb = xa + 4 * XBUF;                                  /* [4][XBUF] exchange, forward       */
  float2 *zbuf = xb + 4 * XBUF;                                /* [2][4][32 k2][32 k1] noise z      */
  float4 *tab = reinterpret_cast<float4 *>(zbuf + 2 * 4 * N);  /* [4][32 k2][32 k1] coefficients    */

  const int tid = threadIdx.x, lane = tid & 31, w = (tid >> 5) & 3;
  const bool noisew = tid >= 128;
  const int b = blockIdx.x;
  /* phase C ownership: one column per transform warp (and per noise warp) */
  int kx;
  if (b < 128) kx = (w < 2) ? (2 * b + w) : (256 + 2 * b + (w - 2));
  else kx = (w == 0) ? 512 : -1;
  const bool colw = kx >= 0;
  const int kxm = colw ? ((N - kx) & (N - 1)) : 0;
  const bool selfc = (kx == 0) || (kx == 512);
  const DDyn &D0 = P.dyn[0];
  const long long nphase = A.nsteps + (A.prologue ? 1 : 0);
  unsigned long long bar_target = A.bar_base;

  if (noisew) {
    /* ================= noise warps: z(step + 1) while the transform warps work on `step` ================= */
    const bool draw = colw && D0.noisy;
    NoiseKey K;
    K.k0 = P.seed_lo;
    K.k1 = P.seed_hi;
    float2 *zw = zbuf + (size_t)w * N + lane;
    if (draw && A.nsteps > 0) {
      K.c2 = (uint32_t)(A.step0 & 0xffffffffu);
      K.c3 = (uint32_t)((((A.step0 >> 32) & 0xffffu) << 16) | ((uint32_t)D0.field_id & 0xffffu));
#pragma unroll 2
      for (int k2 = 0; k2 < 32; ++k2) zw[k2 * 32] = noise_mode(K, kx, lane + 32 * k2, selfc);
    }
    __syncthreads();
#pragma unroll 1
    for (long long it = 0; it < nphase; ++it) {
      const bool pro = A.prologue && it == 0;
      const long long ls = it - (A.prologue ? 1 : 0);
      const bool more = draw && !pro && (ls + 1 < A.nsteps);
      const unsigned long long nstep = A.step0 + (unsigned long long)(ls + 1);
      K.c2 = (uint32_t)(nstep & 0xffffffffu);
      K.c3 = (uint32_t)((((nstep >> 32) & 0xffffu) << 16) | ((uint32_t)D0.field_id & 0xffffu));
      float2 *zn = zw + (size_t)((ls + 1) & 1) * 4 * N;
      if (!pro) {
        if (more) {
#pragma unroll 2
          for (int k2 = 0; k2 < 16; ++k2) zn[k2 * 32] = noise_mode(K, kx, lane + 32 * k2, selfc);
        }
        grid_arrive(A.bar);
        bar_target += NCTA;
        grid_wait(A.bar, bar_target);
        if (more) {
#pragma unroll 2
          for (int k2 = 16; k2 < 32; ++k2) zn[k2 * 32] = noise_mode(K, kx, lane + 32 * k2, selfc);
        }
      }
      grid_arrive(A.bar);
      bar_target += NCTA;
      grid_wait(A.bar, bar_target);
    }
    return;
  }

  /* ================= transform warps ================= */
  const bool need_inv = colw && keep_axis(P.dealias, P.fac[0].order, kx, N);
  /* phase R ownership: thread = (packed row pl of this CTA, butterfly slot) */
  const int s8 = lane & 7, pl = lane >> 3, slot = 8 * w + s8;
  const bool roww = b < 128;

  for (int i = tid; i < N; i += 128) tws[i] = A.tw[((i >> 5) * (i & 31)) & (N - 1)];

  /* per-mode coefficients of this warp's column: (dt*outer, 1/(1 - dt L), noise amplitude, factor op * mask / N) */
  float2 st[32];
  float4 *mytab = tab + (size_t)w * N;
  if (colw) {
    const float dt = (float)P.dt, invN = (float)P.invN;
    const bool keepx = keep_axis(P.dealias, P.fac[0].order, kx, N);
#pragma unroll 1
    for (int k2 = 0; k2 < 32; ++k2) {
      const int ky = lane + 32 * k2;
      const ModeQ<float> mq = make_mode<float>(P, kx, ky, 0);
      float4 t;
      t.x = dt * eval_op<float>(P.grp[0].outer, mq).x;
      float L = 0.f;
      for (int e = D0.lhs_beg; e < D0.lhs_end; ++e) L -= eval_op<float>(P.lin[e], mq).x;
      t.y = 1.0f / (1.0f - dt * L);
      t.z = D0.noisy ? noise_amp<float>(D0, mq) : 0.f;
      float fc = 0.f;
      if (keepx && keep_axis(P.dealias, P.fac[0].order, ky, N)) {
        for (int e = P.fac[0].lin_beg; e < P.fac[0].lin_end; ++e) fc += eval_op<float>(P.lin[e], mq).x;
        fc *= invN;
      }
      t.w = fc;
      mytab[k2 * 32 + lane] = t;
      if (!D0.noisy) {
        zbuf[(size_t)w * N + k2 * 32 + lane] = make_float2(0.f, 0.f);
        zbuf[(size_t)(4 + w) * N + k2 * 32 + lane] = make_float2(0.f, 0.f);
      }
    }
#pragma unroll
    for (int k2 = 0; k2 < 32; ++k2) st[k2] = A.state[(size_t)kx * N + lane + 32 * k2];
  }
  /* the product terms of the single group are powers of the one factor field: sum_t coef_t r^nf_t is the
   * polynomial r^2 (c2 + r (c3 + r c4))  (Eq. 11 with one psi) */
  float c2 = 0.f, c3 = 0.f, c4 = 0.f;
  for (int t = P.grp[0].term_beg; t < P.grp[0].term_end; ++t) {
    const float c = (float)P.term[t].coef;
    if (P.term[t].nf == 2) c2 += c;
    else if (P.term[t].nf == 3) c3 += c;
    else c4 += c;
  }
  __syncthreads();

  float2 v[32];
#pragma unroll 1
  for (long long it = 0; it < nphase; ++it) {
    const bool pro = A.prologue && it == 0;
    const long long ls = it - (A.prologue ? 1 : 0);
    const float2 *myz = zbuf + (size_t)(ls & 1) * 4 * N + (size_t)w * N + lane;
    if (pro && need_inv) {
#pragma unroll
      for (int k2 = 0; k2 < 32; ++k2) {
        const float fc = mytab[k2 * 32 + lane].w;
        v[k2] = make_float2(st[k2].x * fc, -st[k2].y * fc);
      }
    }
    /* four 1024-point transforms per step, one copy of the transform code:
     *   t = 0: inverse-x of E      t = 1: forward-x of the product     (phase R)
     *   t = 2: forward-y of Z      t = 3: inverse-y of the next factor (phase C)   */
#pragma unroll 1
    for (int t = pro ? 3 : 0; t < 4; ++t) {
      const bool rowsT = t < 2;
      const bool active = rowsT ? roww : (t == 2 ? colw : need_inv);
      if (active) {
        if (t == 0) {
          const float2 *Eb = A.E + ((size_t)b * N) * 4 + pl;
#pragma unroll
          for (int n1 = 0; n1 < 32; ++n1) {
            if (!PRUNE || n1 < 8 || n1 >= 24) {
              const float2 e = ldcg2(Eb + (size_t)(32 * n1 + slot) * 4);
              v[n1] = make_float2(e.x, -e.y);
            } else {
              v[n1] = make_float2(0.f, 0.f);
            }
          }
        } else if (t == 2) {
          const float2 *Z1 = A.Z + (size_t)kx * NP + lane, *Z2 = A.Z + (size_t)kxm * NP + lane;
#pragma unroll
          for (int m = 0; m < 16; ++m) {
            const float2 a = ldcg2(Z1 + 32 * m), c = ldcg2(Z2 + 32 * m);
            v[m] = make_float2(0.5f * (a.x + c.x), 0.5f * (a.y - c.y));        /* row y = 32 m + lane       */
            v[m + 16] = make_float2(0.5f * (a.y + c.y), 0.5f * (c.x - a.x));   /* row y = 32 m + lane + 512 */
          }
        }
        float2 *xs = ((t & 1) ? xb : xa) + (rowsT ? pl : w) * XBUF;
        fft1024(v, xs, tws, rowsT ? slot : lane, rowsT);
        if (t == 0) {
          /* conj(v[brev5(x1)]) = a(x) + i b(x) at x = 32 x1 + slot: rows p and p+512 in real space;
           * the product of each row becomes the input of the forward transform */
          float2 c[32];
#pragma unroll
          for (int x1 = 0; x1 < 32; ++x1) {
            const float ra = v[brev5(x1)].x, rb = -v[brev5(x1)].y;
            c[x1] = make_float2(ra * ra * (c2 + ra * (c3 + ra * c4)), rb * rb * (c2 + rb * (c3 + rb * c4)));
          }
#pragma unroll
          for (int x1 = 0; x1 < 32; ++x1) v[x1] = c[x1];
        } else if (t == 1) {
          float2 *Zb = A.Z + (size_t)slot * NP + 4 * b + pl;
#pragma unroll
          for (int k2 = 0; k2 < 32; ++k2) Zb[(size_t)(32 * k2) * NP] = v[brev5(k2)];
        } else if (t == 2) {
          /* v[brev5(k2)] = P_q at ky = lane + 32 k2: Eq. 15 + Eq. 16 + Eq. 18, then the next factor's input */
          float2 c[32];
#pragma unroll
          for (int k2 = 0; k2 < 32; ++k2) {
            const float4 tt = mytab[k2 * 32 + lane];
            const float2 z = myz[k2 * 32];
            const float2 pq = v[brev5(k2)];
            const float nx = (st[k2].x + tt.x * pq.x) + tt.z * z.x;
            const float ny = (st[k2].y + tt.x * pq.y) + tt.z * z.y;
            st[k2] = make_float2(nx * tt.y, ny * tt.y);
            c[k2] = make_float2(st[k2].x * tt.w, -st[k2].y * tt.w);
          }
#pragma unroll
          for (int k2 = 0; k2 < 32; ++k2) v[k2] = c[k2];
        } else {
          /* conj(v[brev5(y1)]) = psi_x[kx][y = 32 y1 + lane]; pack rows y (A) and y + 512 (B) */
#pragma unroll
          for (int y1 = 0; y1 < 16; ++y1) {
            const float2 a = make_float2(v[brev5(y1)].x, -v[brev5(y1)].y);
            const float2 bb = make_float2(v[brev5(y1 + 16)].x, -v[brev5(y1 + 16)].y);
            const int p = 32 * y1 + lane;
            float2 *e = A.E + ((size_t)(p >> 2) * N) * 4 + (p & 3);
            if (selfc) {
              e[(size_t)kx * 4] = make_float2(a.x, bb.x);                 /* the C2R keeps the real part there */
            } else {
              e[(size_t)kx * 4] = make_float2(a.x - bb.y, a.y + bb.x);    /* A + iB              */
              e[(size_t)kxm * 4] = make_float2(a.x + bb.y, bb.x - a.y);   /* conj(A) + i conj(B) */
            }
          }
        }
      }
      if (t == 1 || t == 3) {
        grid_arrive(A.bar);
        bar_target += NCTA;
        grid_wait(A.bar, bar_target);
      }
    }
  }

  if (colw && A.nsteps > 0) {
#pragma unroll
    for (int k2 = 0; k2 < 32; ++k2) A.state[(size_t)kx * N + lane + 32 * k2] = st[k2];
  }
}

}  // namespace f2d
#endif
