/*
 * pss_persist2d.cuh — the whole time step of a 1024 x 1024 fp32 single-field system with a cubic
 * (cutoff <= N/4) de-aliasing mask as ONE persistent cooperative kernel, second generation.
 *
 * What changed against pss_fused2d.cuh (which stays for the other de-aliasing rules).  The
 * timeline of that kernel (globaltimer stamps, profiles/r2_summary.md) showed half of the step in the two all-to-all
 * exchanges, and its per-thread 8-byte global accesses touching 4-8 different 128-byte lines per warp instruction.
 * Here
 *   - each exchange array is laid out per CONSUMER CTA as one contiguous block made of 128-byte chunks, one chunk per
 *     producer: the producer writes whole lines (16 bytes per lane), the consumer reads its block with fully
 *     coalesced 16-byte loads; the transposition happens in shared memory on both sides (scatter into a staging tile /
 *     gather out of it) with an in-chunk rotation that makes every half-warp access hit 16 different banks;
 *   - the consumer fetches its block with 16-byte asynchronous copies (cp.async.cg, global -> shared, no registers)
 *     issued by all 256 transform threads as soon as the one polling thread has seen the grid barrier open;
 *   - the noise warps draw z(s+1) while the transform warps WAIT (grid barrier in flight, block being fetched) and
 *     pause while they compute: the step is issue-bound in its compute phases and latency-bound in its exchanges, so
 *     the third of the instructions that is noise goes where the issue slots are free;
 *   - a CTA's 256 transform threads are two independent 128-thread groups (2 lines each) with their own named
 *     barriers, so one group's exchange traffic overlaps the other's transforms; group 0 owns the two de-aliased
 *     (kept) columns, whose inverse transform feeds the next exchange, and runs first in phase C; group 1 owns the two
 *     columns outside the mask (no inverse transform): it arrives at barrier B with a relaxed reduction as soon as its
 *     input block is fetched and transforms while that barrier is in flight.
 * Bulk asynchronous copies (cp.async.bulk + mbarrier) and two flag-in-data protocols without a grid barrier were built
 * and measured for these exchanges and were not faster (profiles/r2_summary.md).
 *
 * Transform.  1024 = 16 x 16 x 4, three register passes around two shared-memory exchanges (as pss_fused2d.cuh):
 *   natural n = 64 n1 + 4 n2 + n3, spectral k = k1 + 16 k2 + 256 k3
 *   "D_nat"  : thread tq (0..63) holds x[64 a + tq], a = 0..15
 *   "D_spec" : thread tq = k1 + 16 c holds X[k1 + 16 (4 c + j) + 256 k3] at register r = j + 4 k3
 *   Pass 2 is done by thread (k1 = tq & 15, n3 = tq >> 4), pass 3 by thread (k1 = tq & 15, k2 = 4 (tq >> 4) + j):
 *   with a half-warp = 16 consecutive tq of ONE line every shared-memory access of the transform walks 16 rows of odd
 *   pitch or 16 consecutive columns: conflict-free.
 *
 * Thread map: transform thread tid in [0,256): group g = tid >> 7; inside the group warp w = (tid >> 5) & 3, lane
 * l = tid & 31: line L = l >> 4, slot tq = 16 w + (l & 15).
 *   phase R (rows, x axis):    group (b, g) owns the packed row pairs p = 4 b + 2 g + L        ("bg" = 2 b + g)
 *   phase C (columns, y axis): group (c, gc) owns the columns kx = 256 gc + 2 c + L;  CTA 128 owns kx = 512
 *
 * Exchange arrays (float2):
 *   Zg [c in 0..127][bg in 0..255][16]   chunk (bg -> c): Z[k'][p] for p = 2 bg + L and the eight k' CTA c consumes,
 *       element (gc, L, s) at (8 gc + 4 L + s + 2 c + rho(bg)) & 15, s = 0,1: kx = 256 gc + 2 c + s, s = 2,3: its
 *       mirror 1024 - kx;  rho(bg) = (bg & 3) | ((bg & 4) << 1).   Z512[p] for column 512 follows the 128 blocks.
 *   Eg [b in 0..127][c in 0..127][16]    chunk (c -> b): E[p][k'] for p = 4 b + pl and kx = 2 c + s (s = 0,1) and the
 *       mirrors (s = 2,3), element (pl, s) at (4 pl + s + 2 c + b) & 15.
 *   Producers: lanes walk consecutive k (2 c + s) -> 16 banks.  Consumers of Z: lanes walk (bg, L) -> 4 L + rho(bg);
 *   consumers of E: lanes walk consecutive k again.  Every staging index below is a thread constant plus a
 *   compile-time multiple of a chunk stride.
 */
#ifndef PSS_PERSIST2D_CUH
#define PSS_PERSIST2D_CUH
#include "pss_pointwise.cuh"

namespace p2d {

constexpr int N = 1024;
constexpr int TT = 256;               /* transform threads (two groups of 128)             */
constexpr int GT = 128;               /* threads of one group (2 lines x 64)               */
constexpr int NT = 256;               /* noise threads                                     */
constexpr int THREADS = TT + NT;
constexpr int NCTA = 129;             /* 128 CTAs own 4 packed rows + 4 columns; CTA 128 owns column kx = 512 */
constexpr int PITCH = 65;             /* k1-row pitch of an exchange buffer (float2), odd  */
constexpr int BUF = 16 * PITCH;       /* one line's exchange buffer                        */
constexpr int REGA = 4096;            /* staging A (float2): Z out (two groups x 2048) in phase R, Z in (4096) in phase C */
constexpr int REGB = 2048;            /* staging B (float2): E in (phase R), E out (phase C, group 0)                     */
constexpr size_t SMEM_BYTES = (size_t)(4 * BUF + REGA + REGB + 16 * TT) * sizeof(float2) + (size_t)16 * TT * sizeof(float4) + 16;
constexpr size_t Z512_OFF = (size_t)128 * 256 * 16;   /* float2 offset of Z512[512] inside the Z array (fits one half-spectrum array) */
constexpr int NARRIVE = 2 * NCTA;                     /* every group of every CTA arrives at every grid barrier           */

struct Args {
  float2 *state;
  float2 *Eg;
  float2 *Zg;
  const float2 *tw;              /* tw[j] = exp(-2 pi i j / 1024) */
  unsigned long long *bar;       /* bar[0]: counter of barrier A (Z complete), bar[16]: barrier B (E complete); zero at launch */
  long long nsteps;
  unsigned long long step0;
  int prologue;                  /* 1: E is stale (after pss_set_field): rebuild it from the state first */
  int prio;                      /* 1: in phase C group 1 waits for group 0's transforms (PSS_P2D_PRIO=0 disables) */
  int gate;                      /* > 0: the noise warps pause while their group computes, polling every `gate` ns (PSS_NOISE_GATE=0 disables) */
  int dbg;                       /* timing experiments only (-DPSS_P2D_DEBUG): 1 = skip the transforms, 2 = skip the noise */
  long long *ts;                 /* timing experiments only (-DPSS_P2D_DEBUG): globaltimer stamps [cta][group][32] of the last-but-one step */
};
#ifdef PSS_P2D_DEBUG
#define TS(i) do { if (A.ts && ls == A.nsteps - 2 && (tid & 127) == 0) { unsigned long long t_; asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t_)); A.ts[(blockIdx.x * 2 + g) * 32 + (i)] = (long long)t_; } } while (0)
#else
#define TS(i) do {} while (0)
#endif
#ifdef PSS_P2D_DEBUG
#define P2D_DBG(bit) ((A.dbg >> (bit)) & 1)
#else
#define P2D_DBG(bit) 0
#endif

__device__ __forceinline__ int rho(int bg) { return (bg & 3) | ((bg & 4) << 1); }
__device__ __forceinline__ int zidx(int gc, int L, int s, int c, int bg) { return (8 * gc + 4 * L + s + 2 * c + rho(bg)) & 15; }
__device__ __forceinline__ int eidx(int pl, int s, int c, int b) { return (4 * pl + s + 2 * c + b) & 15; }

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

/* named barriers: 1 + g = the 128 transform threads of group g; 3 + g = z of group g full; 5 + g = z of group g empty
 * (256 threads each: the group and its 128 noise threads) */
__device__ __forceinline__ void gsync(int g) { asm volatile("bar.sync %0, 128;" ::"r"(1 + g) : "memory"); }
__device__ __forceinline__ void nb_sync(int id) { asm volatile("bar.sync %0, 256;" ::"r"(id) : "memory"); }
__device__ __forceinline__ void nb_arrive(int id) {
  __threadfence_block();
  asm volatile("bar.arrive %0, 256;" ::"r"(id) : "memory");
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
  float2 t2[16];    /* t2[k2] = w64^(k2 (tq >> 4))                 */
  int tq, g;
};

/* D_nat -> D_spec.  The caller guarantees that nobody of the group still reads the exchange buffer. */
__device__ __forceinline__ void fwd_dif(float2 (&v)[16], const Lane &ln) {
  dft_reg<4, -1>(v);
#pragma unroll
  for (int k1 = 0; k1 < 16; ++k1) {
    float2 x = v[k1];
    if (k1 > 0) x = cmulf(x, ln.t1[k1]);
    ln.xl[k1 * PITCH + ln.tq] = x;
  }
  gsync(ln.g);
  float2 *base = ln.xl + (ln.tq & 15) * PITCH + (ln.tq >> 4);   /* row k1 = tq & 15, column 4 n2 + (n3 = tq >> 4) */
#pragma unroll
  for (int n2 = 0; n2 < 16; ++n2) v[n2] = base[4 * n2];
  dft_reg<4, -1>(v);
#pragma unroll
  for (int k2 = 0; k2 < 16; ++k2) {
    float2 x = v[k2];
    if (k2 > 0) x = cmulf(x, ln.t2[k2]);
    base[4 * k2] = x;
  }
  gsync(ln.g);
  const float2 *b2 = ln.xl + (ln.tq & 15) * PITCH + 16 * (ln.tq >> 4);
#pragma unroll
  for (int j = 0; j < 4; ++j) {
    float2 a0 = b2[4 * j], a1 = b2[4 * j + 1], a2 = b2[4 * j + 2], a3 = b2[4 * j + 3];
    dft4(a0, a1, a2, a3);
    v[j] = a0; v[j + 4] = a1; v[j + 8] = a2; v[j + 12] = a3;
  }
}

/* D_spec -> D_nat (also a forward transform; the DFT matrix is symmetric).  Same guarantee as fwd_dif. */
__device__ __forceinline__ void fwd_dit(float2 (&v)[16], const Lane &ln) {
  float2 *b2 = ln.xl + (ln.tq & 15) * PITCH + 16 * (ln.tq >> 4);
#pragma unroll
  for (int j = 0; j < 4; ++j) {
    float2 a0 = v[j], a1 = v[j + 4], a2 = v[j + 8], a3 = v[j + 12];
    dft4(a0, a1, a2, a3);
    b2[4 * j] = a0; b2[4 * j + 1] = a1; b2[4 * j + 2] = a2; b2[4 * j + 3] = a3;
  }
  gsync(ln.g);
  float2 *base = ln.xl + (ln.tq & 15) * PITCH + (ln.tq >> 4);
#pragma unroll
  for (int k2 = 0; k2 < 16; ++k2) {
    float2 x = base[4 * k2];
    if (k2 > 0) x = cmulf(x, ln.t2[k2]);
    v[k2] = x;
  }
  dft_reg<4, -1>(v);
#pragma unroll
  for (int n2 = 0; n2 < 16; ++n2) base[4 * n2] = v[n2];
  gsync(ln.g);
#pragma unroll
  for (int k1 = 0; k1 < 16; ++k1) {
    float2 x = ln.xl[k1 * PITCH + ln.tq];
    if (k1 > 0) x = cmulf(x, ln.t1[k1]);
    v[k1] = x;
  }
  dft_reg<4, -1>(v);
}

/* all 256 transform threads */
__device__ __forceinline__ void tsync_all() { asm volatile("bar.sync 7, 256;" ::: "memory"); }
__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void st_cg16(void *p, uint4 v) {
  asm volatile("st.global.cg.v4.u32 [%0], {%1, %2, %3, %4};" ::"l"(p), "r"(v.x), "r"(v.y), "r"(v.z), "r"(v.w) : "memory");
}

/* ---- grid barrier: one monotonically increasing counter per barrier kind, zeroed by the host before the launch.
 * A group arrives with a release reduction by one thread after its own bar.sync (the group's global stores
 * happen-before it through the CTA barrier).  Only thread 0 of a CTA polls (acquire loads); everybody else waits at a
 * CTA barrier for it, then fetches the block. ---- */
__device__ __forceinline__ void grid_arrive(unsigned long long *ctr) {
  asm volatile("red.release.gpu.global.add.u64 [%0], 1;" ::"l"(ctr) : "memory");
}
/* Arrival of a group that wrote nothing the other CTAs read: it only reports that its input block has been fetched, so
 * that the producers may overwrite that block in their next phase (a write-after-read dependency).
 *
 * Ordering.  In the PTX memory model a relaxed reduction gives the producers' acquire poll nothing to
 * synchronise with, so the model does not order the fetch before the overwrite.  The hardware does: the fetch is
 * cp.async.cg, and the group executes cp.async.wait_all and its named barrier before the one arriving thread issues the
 * reduction; wait_all returns only when the copied bytes are in shared memory, i.e. the reads of the block have
 * completed at L2 and can no longer observe a later store.  A read that has returned its data cannot be reordered
 * after anything.  What the relaxed form drops is the MEMBAR.GPU of a release (the wait for the acknowledgement of
 * the group's own earlier stores, of which there are none that matter here).
 * Cost of the formally ordered form, measured (round 3, B200, bench.py --steps 40, A/B/A/B on one box): 10.005 us per
 * step with red.release.gpu here against 9.595 us with red.relaxed.gpu (+0.41 us, 4.3 %).  The product keeps the
 * relaxed form; -DPSS_P2D_ARRIVE_RELEASE (PSS_NVCC_EXTRA) builds the other, bit-identical in its results.
 * tests/test_gpu_soak.py runs 10^6 steps and compares bit for bit with the first-generation kernel (PSS_PERSIST=0),
 * whose barriers are all release/acquire. */
__device__ __forceinline__ void grid_arrive_relaxed(unsigned long long *ctr) {
#ifdef PSS_P2D_ARRIVE_RELEASE
  asm volatile("red.release.gpu.global.add.u64 [%0], 1;" ::"l"(ctr) : "memory");
#else
  asm volatile("red.relaxed.gpu.global.add.u64 [%0], 1;" ::"l"(ctr) : "memory");
#endif
}
__device__ __forceinline__ void grid_poll(const unsigned long long *ctr, unsigned long long target) {
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
/* 16 bytes global (L2) -> shared, asynchronous, no register staging */
__device__ __forceinline__ void cp_async16(uint32_t dst, const void *src) {
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(dst), "l"(src) : "memory");
}
/* the CTA's contiguous input block (N16 x 256 x 16 bytes) into a staging tile, all 256 transform threads */
template <int N16> __device__ __forceinline__ void load_block(float2 *dst, const float2 *src, int tid) {
  const uint32_t d = smem_u32(dst) + tid * 16;
  const char *sp = reinterpret_cast<const char *>(src) + tid * 16;
#pragma unroll
  for (int i = 0; i < N16; ++i) cp_async16(d + i * 4096, sp + i * 4096);
  asm volatile("cp.async.wait_all;" ::: "memory");
}

/* ------------------------------------------------------------------------------------------ */
__global__ void __launch_bounds__(THREADS, 1) k_persist2d(const __grid_constant__ Program P, const Args A) {
  extern __shared__ __align__(128) unsigned char smem_raw[];
  float2 *xs = reinterpret_cast<float2 *>(smem_raw);            /* [4][BUF] exchange buffers               */
  float2 *regA = xs + 4 * BUF;                                  /* staging A                               */
  float2 *regB = regA + REGA;                                   /* staging B                               */
  float2 *zbuf = regB + REGB;                                   /* [16 r][256 tid] unit noise z            */
  float4 *tab = reinterpret_cast<float4 *>(zbuf + 16 * TT);     /* [16 r][256 tid] per-mode coefficients   */
  volatile int *hold = reinterpret_cast<volatile int *>(tab + 16 * TT); /* [2]: group g is computing: its noise warps pause */

  const int tid = threadIdx.x & (TT - 1);
  const bool noisew = threadIdx.x >= TT;
  const int g = tid >> 7, lane = tid & 31, L = lane >> 4, tq = 16 * ((tid >> 5) & 3) + (lane & 15);
  const int b = blockIdx.x;
  const bool roww = b < 128;
  /* phase C ownership: column of (group, line); spectral index of register r: ky = kyb + 16 j + 256 k3, r = j + 4 k3 */
  const int kx = roww ? (256 * g + 2 * b + L) : ((g == 0 && L == 0) ? 512 : -1);
  const bool colw = kx >= 0;
  const bool selfc = (kx == 0) || (kx == 512);
  const bool kept = roww && g == 0;           /* |kx| < 256: the masked factor is non-zero, inverse transform + E */
  const int kyb = (tq & 15) + 64 * (tq >> 4);
  const DDyn &D0 = P.dyn[0];
  const bool noisy = D0.noisy != 0;
  const long long nphase = A.nsteps + (A.prologue ? 1 : 0);

  if (threadIdx.x < 2) hold[threadIdx.x] = 0;
  __syncthreads();

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
      if (s >= 1) nb_sync(5 + g); /* the group has consumed z(s-1) */
      if (colw && !P2D_DBG(1)) {
        float2 *zw = zbuf + tid;
#pragma unroll 1
        for (int r = 0; r < 16; r += 2) {
          /* pause while the group's transform warps compute; they clear the flag when they wait (exchange in flight,
           * or z itself needed) */
          if (A.gate) while (hold[g]) __nanosleep(A.gate);
          zw[r * TT] = noise_mode(K, kx, kyb + 16 * (r & 3) + 256 * (r >> 2), selfc);
          zw[(r + 1) * TT] = noise_mode(K, kx, kyb + 16 * ((r + 1) & 3) + 256 * ((r + 1) >> 2), selfc);
        }
      }
      nb_arrive(3 + g);
    }
    return;
  }

  /* ================= transform warps ================= */
  asm volatile("setmaxnreg.inc.sync.aligned.u32 184;"); /* 8 x 32 x (64 + 184) = 63488 <= 65536 registers */
  Lane ln;
  ln.xl = xs + (2 * g + L) * BUF;
  ln.tq = tq;
  ln.g = g;
#pragma unroll
  for (int i = 0; i < 16; ++i) {
    ln.t1[i] = A.tw[(i * tq) & (N - 1)];
    ln.t2[i] = A.tw[(16 * i * (tq >> 4)) & (N - 1)];
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
        if (kept && keep_axis(P.dealias, P.fac[0].order, kx, N) && keep_axis(P.dealias, P.fac[0].order, ky, N)) {
          for (int e = P.fac[0].lin_beg; e < P.fac[0].lin_end; ++e) fc += eval_op<float>(P, P.lin[e], mq).x;
          fc *= invN;
        }
        t.w = fc;
      }
      tab[r * TT + tid] = t;
      if (!noisy) zbuf[r * TT + tid] = make_float2(0.f, 0.f);
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
  const int bg = 2 * b + g, pl = 2 * g + L;
  float2 *zout = regA + g * 2048;      /* this group's Z staging tile: [128 c][16]           */
  /* staging indices: every access below is one of these bases plus a compile-time multiple of a chunk stride */
  const int k00 = (tq & 15) + 64 * (tq >> 4);                                   /* k of register j = 0, k3 = 0 */
  const int eg0 = (k00 >> 1) * 16 + ((k00 + 4 * pl + b) & 15);                   /* E gather, k3 = 0: + 128 j    */
  const int eg3 = ((256 - k00) >> 1) * 16 + ((2 + 256 - k00 + 4 * pl + b) & 15); /* E gather, k3 = 3: - 128 j    */
  const int zs0 = (k00 >> 1) * 16 + ((4 * L + k00 + rho(bg)) & 15);              /* Z scatter, k3 = 0: + 128 j   */
  const int zs1 = (k00 >> 1) * 16 + ((8 + 4 * L + k00 + rho(bg)) & 15);          /* k3 = 1                       */
  const int zs2 = ((256 - k00) >> 1) * 16 + ((8 + 4 * L + 2 + 256 - k00 + rho(bg)) & 15); /* k3 = 2: - 128 j     */
  const int zs3 = ((256 - k00) >> 1) * 16 + ((4 * L + 2 + 256 - k00 + rho(bg)) & 15);     /* k3 = 3: - 128 j     */
  const int zg0 = (tq >> 1) * 16 + zidx(g, tq & 1, L, b, tq >> 1);               /* Z gather, direct: + 512 a    */
  const int zg1 = selfc ? zg0 : (tq >> 1) * 16 + zidx(g, tq & 1, 2 + L, b, tq >> 1); /* mirror                  */
  const int es0 = (tq >> 2) * 16 + eidx(tq & 3, L, b, tq >> 2);                  /* E scatter, direct: + 256 a   */
  const int es1 = (tq >> 2) * 16 + eidx(tq & 3, 2 + L, b, tq >> 2);              /* mirror                       */
  const int gt = tid & (GT - 1), cq = gt & 7;                                    /* copy-out: lane cq of chunk (gt >> 3) + 16 i */
  unsigned long long *ctrA = A.bar, *ctrB = A.bar + 16;
  unsigned long long nA = 0, nB = 0;   /* barriers of each kind this thread has been through */
  gsync(g);

  /* first phase R of a launch that finds E valid: no barrier to wait for */
  if (!A.prologue && roww && nphase > 0) {
    load_block<4>(regB, A.Eg + (size_t)b * 2048, tid);
    tsync_all();
  }

  float2 v[16];
#pragma unroll 1
  for (long long it = 0; it < nphase; ++it) {
    const bool pro = A.prologue && it == 0;
    const long long ls = it - (A.prologue ? 1 : 0);
    if (!pro) {
      /* ======================= phase R: inverse-x of E, product, forward-x -> Z ======================= */
      if (roww) {
        if (gt == 0) hold[g] = 1;
        TS(0);
        /* D_spec input, conjugated (inverse transform = conj o forward o conj); only |k| < 256 is non-zero:
         * k3 = 0 reads column kx = k00 + 16 j (chunk +8 per j), k3 = 3 the mirror slot of kx = 256 - k00 - 16 j */
#pragma unroll
        for (int j = 0; j < 4; ++j) {
          const float2 e0 = regB[eg0 + 128 * j];
          float2 e3 = regB[eg3 - 128 * j];
          if (j == 0 && tq == 0) e3 = make_float2(0.f, 0.f);         /* k = 768: outside the mask */
          v[j] = make_float2(e0.x, -e0.y);
          v[j + 4] = make_float2(0.f, 0.f);
          v[j + 8] = make_float2(0.f, 0.f);
          v[j + 12] = make_float2(e3.x, -e3.y);
        }
        if (!P2D_DBG(0)) fwd_dit(v, ln);
        TS(2);
        /* conj(v[a]) = a(x) + i b(x) at x = 64 a + tq: rows p and p + 512 in real space */
#pragma unroll
        for (int a = 0; a < 16; ++a) {
          const float ra = v[a].x, rb = -v[a].y;
          v[a] = make_float2(ra * ra * (c2 + ra * (c3 + ra * c4)), rb * rb * (c2 + rb * (c3 + rb * c4)));
        }
        /* no barrier here: fwd_dit's last pass read column tq of the exchange buffer and fwd_dif's first pass writes
         * the same addresses, both by this thread */
        if (!P2D_DBG(0)) fwd_dif(v, ln);
        TS(3);
        /* scatter Z[k][p] into the staging tile, one 16-element chunk per consumer CTA: k = k00 + 16 j + 256 k3;
         * k3 = 0, 1: direct slots of kx = k (groups 0, 1 of CTA (k & 255) >> 1); k3 = 2, 3: mirror slots of
         * kx = 1024 - k (groups 1, 0).  In-chunk positions do not depend on j. */
#pragma unroll
        for (int j = 0; j < 4; ++j) {
          zout[zs0 + 128 * j] = v[j];
          zout[zs1 + 128 * j] = v[j + 4];
          if (j == 0 && tq == 0) {
            A.Zg[Z512_OFF + 2 * bg + L] = v[8];                      /* k = 512: column 512 itself          */
            zout[zidx(1, L, 2, 0, bg)] = v[12];                      /* k = 768: mirror of kx = 256 (group 1 of CTA 0) */
          } else {
            zout[zs2 - 128 * j] = v[j + 8];
            zout[zs3 - 128 * j] = v[j + 12];
          }
        }
        gsync(g);
        TS(4);
        /* copy-out: 128 chunks of 128 bytes, 8 lanes per chunk, whole lines */
        {
          const uint4 *src = reinterpret_cast<const uint4 *>(zout);
          uint4 *dst = reinterpret_cast<uint4 *>(A.Zg);
#pragma unroll
          for (int i = 0; i < 8; ++i) {
            const int c = (gt >> 3) + 16 * i;
            st_cg16(dst + ((size_t)c * 256 + bg) * 8 + cq, src[c * 8 + cq]);
          }
        }
        TS(5);
      }
      gsync(g);
      if (gt == 0) {
        hold[g] = 0;
        if (roww) grid_arrive(ctrA);
        else grid_arrive_relaxed(ctrA);
      }
      nA += 1;
      TS(6);
      /* ======================= phase C: forward-y of Z, Eq. 15/16/18, inverse-y -> E ======================= */
      if (tid == 0) grid_poll(ctrA, nA * NARRIVE);
      tsync_all();
      TS(7);
      if (roww) load_block<8>(regA, A.Zg + (size_t)b * 4096, tid);
      else load_block<1>(regA, A.Zg + Z512_OFF, tid);
      tsync_all();
      TS(8);
      /* the kept columns are the critical path (their inverse transform feeds the next exchange): group 1 starts its
       * forward transform when group 0 has finished both of its own, and runs while barrier B is in flight */
      if (roww && g == 1 && A.prio) asm volatile("bar.sync 8, 256;" ::: "memory");
      if (gt == 0) hold[g] = 1;
      if (colw) {
#pragma unroll
        for (int a = 0; a < 8; ++a) {
          float2 za, zc;
          if (roww) {
            za = regA[zg0 + 512 * a];
            zc = regA[zg1 + 512 * a];
          } else {
            za = regA[64 * a + tq];
            zc = za;
          }
          v[a] = make_float2(0.5f * (za.x + zc.x), 0.5f * (za.y - zc.y));     /* row y = 64 a + tq       */
          v[a + 8] = make_float2(0.5f * (za.y + zc.y), 0.5f * (zc.x - za.x)); /* row y = 64 a + tq + 512 */
        }
      } else {
#pragma unroll
        for (int a = 0; a < 16; ++a) v[a] = make_float2(0.f, 0.f);
      }
      if (!kept) { /* nothing of this group feeds E: arrive as soon as the input tile has been consumed */
        gsync(g);
        if (gt == 0) grid_arrive_relaxed(ctrB);
      }
      if (!P2D_DBG(0)) fwd_dif(v, ln);
      TS(10);
      /* v[r] = P_q at ky(r): Eq. 15 + Eq. 16 + Eq. 18, then the next factor's (conjugated) input */
      if (noisy) {
        if (gt == 0) hold[g] = 0;      /* z is needed now: let the noise warps finish */
        nb_sync(3 + g);
        if (gt == 0 && kept) hold[g] = 1;
      }
#pragma unroll
      for (int r = 0; r < 16; ++r) {
        const float4 tt = tab[r * TT + tid];
        const float2 z = zbuf[r * TT + tid];
        const float2 pq = v[r];
        const float nx = (st[r].x + tt.x * pq.x) + tt.z * z.x;
        const float ny = (st[r].y + tt.x * pq.y) + tt.z * z.y;
        st[r] = make_float2(nx * tt.y, ny * tt.y);
        v[r] = make_float2(st[r].x * tt.w, -st[r].y * tt.w);
      }
      if (noisy && ls + 1 < A.nsteps) nb_arrive(5 + g);
      if (!noisy && gt == 0 && !kept) hold[g] = 0;
      TS(11);
      /* no barrier before fwd_dit: its first pass writes the 16 slots this thread read last in fwd_dif */
    } else {
      if (kept) {
#pragma unroll
        for (int r = 0; r < 16; ++r) {
          const float fc = tab[r * TT + tid].w;
          v[r] = make_float2(st[r].x * fc, -st[r].y * fc);
        }
      } else {
        gsync(g);
        if (gt == 0) grid_arrive_relaxed(ctrB);
      }
    }
    if (kept) {
      if (!P2D_DBG(0)) fwd_dit(v, ln);
      if (!pro && A.prio) asm volatile("bar.arrive 8, 256;" ::: "memory");
      TS(12);
      /* conj(v[a]) = psi_x[kx][y = 64 a + tq]; pack rows y (A) and y + 512 (B); chunk per consumer CTA p >> 2 */
#pragma unroll
      for (int a = 0; a < 8; ++a) {
        const float2 av = make_float2(v[a].x, -v[a].y);
        const float2 bv = make_float2(v[a + 8].x, -v[a + 8].y);
        if (selfc) {
          regB[es0 + 256 * a] = make_float2(av.x, bv.x);                       /* the C2R keeps the real part there */
        } else {
          regB[es0 + 256 * a] = make_float2(av.x - bv.y, av.y + bv.x);          /* A + iB              */
          regB[es1 + 256 * a] = make_float2(av.x + bv.y, bv.x - av.y);          /* conj(A) + i conj(B) */
        }
      }
      gsync(g);
      TS(13);
      {
        const uint4 *src = reinterpret_cast<const uint4 *>(regB);
        uint4 *dst = reinterpret_cast<uint4 *>(A.Eg);
#pragma unroll
        for (int i = 0; i < 8; ++i) {
          const int bp = (gt >> 3) + 16 * i;
          st_cg16(dst + ((size_t)bp * 128 + b) * 8 + cq, src[bp * 8 + cq]);
        }
      }
      TS(14);
      gsync(g);
      if (gt == 0) { hold[g] = 0; grid_arrive(ctrB); }
      TS(15);
    }
    nB += 1;
    /* entry of the next phase R: the CTA's E block (16 KB) as soon as barrier B is open */
    if (it + 1 < nphase && roww) {
      if (tid == 0) grid_poll(ctrB, nB * NARRIVE);
      tsync_all();
      TS(16);
      load_block<4>(regB, A.Eg + (size_t)b * 2048, tid);
      tsync_all();
      TS(17);
    }
  }

  if (colw && A.nsteps > 0) {
#pragma unroll
    for (int r = 0; r < 16; ++r) A.state[(size_t)kx * N + kyb + 16 * (r & 3) + 256 * (r >> 2)] = st[r];
  }
}

}  // namespace p2d
#endif
