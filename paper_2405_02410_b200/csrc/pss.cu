/*
 * pss.cu — host side of libpss.so: the C ABI of include/pss.h, the term-list compiler
 * (field system -> Program), the launch plan and the step loop.
 *
 * No CPU compute path exists here: every transform, product, operator, noise draw and update
 * runs in the kernels of pss_kernels.cuh.  The host only validates, flattens the term list and
 * launches.
 */
#include "../../include/pss.h"

#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <mutex>
#include <string>
#include <vector>

#include "pss_kernels.cuh"
#include "pss_fused2d.cuh"
#include "pss_persist2d.cuh"

namespace {

struct DefH { pss_op op; int src; };
struct ATermH { pss_op outer; std::vector<int> factors; };
struct FrameH { int axis; long long lo_w, hi_w; double lo_v, hi_v; };
struct FieldH {
  std::string name;
  bool dynamic;
  std::vector<DefH> defs;
  std::vector<pss_op> lhs;    /* dynamic: implicit terms; intermediate: its own lhs */
  std::vector<ATermH> aterms; /* intermediate: rhs terms that are products          */
  std::vector<FrameH> frames; /* dynamic: Dirichlet buffer zones set at the end of every step */
  bool noisy;
  double D;
  int qpow;
};
struct TermH { int field; pss_op outer; std::vector<int> factors; };

struct Plan {
  Geo geo[3];
  int upd_W, upd_threads; size_t upd_smem; int upd_blocks;
  int row_Wc, row_threads; size_t row_smem; int row_blocks;
  int mid_W, mid_threads; size_t mid_smem;
  int one_threads; size_t one_smem; /* 1D */
  int kx_keep_max;                  /* max over factors of the number of kept kx */
  int fused;                        /* 1: the persistent 1024^2 fp32 kernel of pss_fused2d.cuh runs the steps (PSS_FUSED=0 disables) */
  int fused_prune;                  /* its input-pruned instantiation (mask cutoff <= n/4 on both axes)       */
  int pdl;                          /* programmatic dependent launch between the step kernels (PSS_PDL=0 disables) */
  int fused_pair;                   /* ensembles: two replicas per launch (k_fused2d_pair)                    */
  int persist;                      /* 1: pss_persist2d.cuh's kernel (cutoff <= N/4; cp.async.cg block fetches behind two grid-barrier counters) runs the steps, one launch per replica (PSS_PERSIST=0 disables) */
};

}  // namespace

struct pss_system {
  int ndim;
  int64_t n[3];
  double dx[3];
  double dt;
  int prec;
  uint64_t seed;
  int dealias;
  int nrep, sel; /* ensemble: replicas of the same field system (replica r = seed + r), selected replica for set/get */
  bool finalized, bound, psix_valid;
  uint64_t step;
  int64_t herm_period; /* the state is projected onto Hermitian symmetry whenever step % herm_period == 0 (plan_hermitian) */
  std::vector<FieldH> fields;
  std::vector<TermH> terms;
  std::vector<int> dyn_slot; /* field -> spectral source slot (dynamic fields, then product-defined intermediate fields), else -1 */
  Program P;                 /* the launch program of the last round: groups of the dynamic equations, Eq. 18, factors of the first round */
  /* systems with product-defined intermediate fields run one extra round of the two step kernels per dependency level:
   * PR[k] = (factors, groups, terms) of round k for k_rows; PU[k] = (groups, slot kinds of round k, factors of the next
   * round) for k_update.  Round nround - 1 is the dynamic equations'.  Without such fields nround = 1 and PR[0] = PU[0] = P. */
  int nround;
  std::vector<Program> PR, PU;
  int nfac_max, ngrp_max; /* over the rounds: array counts and tile sizes are planned for the largest round */
  Plan plan;
  size_t csize, rsize;
  int64_t M, N; /* modes (half-spectrum), sites */
  /* workspace carve-up (byte offsets) */
  size_t off_state, off_psix, off_phat, off_scratch, off_ureal, off_tw[3], off_bar, ws_need;
  unsigned long long bar_count; /* value of the fused kernel's grid-barrier counter */
  char *ws;
  int dev; /* device that owns the workspace (pss_bind); made current inside every entry point that launches */
  cudaStream_t stream;
  std::string cuda_msg;
  bool cuda_bad;
  uint64_t launches;
  /* pss_profile_step: one event pair per launch */
  bool prof_on;
  std::vector<cudaEvent_t> prof_ev;
  std::vector<int> prof_kind;
};

namespace {

bool is_pow2(int64_t v) { return v >= 1 && (v & (v - 1)) == 0; }
int ilog2(int64_t v) { int l = 0; while ((1ll << l) < v) ++l; return l; }

bool op_ok(const pss_system *s, const pss_op *op) {
  if (!op) return false;
  if (op->q2_pow < 0 || op->invq_pow < 0 || op->q2_pow > 24 || op->invq_pow > 24) return false;
  for (int j = 0; j < 3; ++j) {
    if (op->iq_pow[j] < 0 || op->iq_pow[j] > 24) return false;
    if (j >= s->ndim && op->iq_pow[j] != 0) return false;
  }
  return std::isfinite(op->coef);
}
bool fid_ok(const pss_system *s, int f) { return f >= 0 && f < (int)s->fields.size(); }

int cuda_fail(pss_system *s, cudaError_t e, const char *what) {
  s->cuda_bad = true;
  s->cuda_msg = std::string(what) + ": " + cudaGetErrorString(e);
  return PSS_ECUDA;
}
#define CK(call)                                                   \
  do {                                                             \
    cudaError_t e_ = (call);                                       \
    if (e_ != cudaSuccess) return cuda_fail(s, e_, #call);         \
  } while (0)
#define CKL(name)                                                  \
  do {                                                             \
    cudaError_t e_ = cudaGetLastError();                           \
    if (e_ != cudaSuccess) return cuda_fail(s, e_, name);          \
    s->launches += 1;                                              \
  } while (0)

/* makes the workspace's device current for the duration of an entry point and restores the caller's device */
struct DeviceGuard {
  int prev;
  bool switched;
  explicit DeviceGuard(int dev) : prev(-1), switched(false) {
    if (dev >= 0 && cudaGetDevice(&prev) == cudaSuccess && prev != dev) switched = (cudaSetDevice(dev) == cudaSuccess);
  }
  ~DeviceGuard() { if (switched) cudaSetDevice(prev); }
};

int env_int(const char *name, int dflt) {
  const char *v = std::getenv(name);
  return (v && *v) ? std::atoi(v) : dflt;
}

/* ---- term-list compiler ---------------------------------------------------------------- */
DOp link_op(const pss_system *s, const pss_op &op, int src_slot) {
  DOp d;
  std::memset(&d, 0, sizeof(d));
  d.coef = op.coef;
  d.m = (int8_t)op.q2_pow;
  d.p = (int8_t)op.invq_pow;
  uint8_t z = 0;
  for (int j = 0; j < 3; ++j) {
    d.a[j] = (int8_t)op.iq_pow[j];
    if (j < s->ndim && (op.iq_pow[j] & 1) && s->n[j] > 1) z |= (uint8_t)(1u << j);
  }
  if (op.invq_pow > 0) z |= 8u;
  d.zflags = z;
  d.src = (int8_t)src_slot;
  return d;
}
bool real_op(const DOp &d) { return ((d.a[0] + d.a[1] + d.a[2]) & 1) == 0; }
bool compose(const DOp &outer, const DOp &inner, DOp &r) {
  r = inner;
  r.coef = outer.coef * inner.coef;
  const int m = outer.m + inner.m, p = outer.p + inner.p;
  if (m > 100 || p > 100) return false;
  r.m = (int8_t)m;
  r.p = (int8_t)p;
  for (int j = 0; j < 3; ++j) {
    const int a = outer.a[j] + inner.a[j];
    if (a > 100) return false;
    r.a[j] = (int8_t)a;
  }
  r.zflags = outer.zflags | inner.zflags;
  if (outer.den && inner.den) return false; /* one denominator per monomial */
  r.den = outer.den ? outer.den : inner.den;
  return true;
}
bool same_monomial(const DOp &a, const DOp &b) {
  return a.m == b.m && a.p == b.p && a.a[0] == b.a[0] && a.a[1] == b.a[1] && a.a[2] == b.a[2] &&
         a.zflags == b.zflags && a.src == b.src && a.den == b.den;
}
void push_merged(std::vector<DOp> &v, const DOp &d) {
  for (DOp &e : v)
    if (same_monomial(e, d)) { e.coef += d.coef; return; }
  v.push_back(d);
}

/* field -> sum of monomials acting on spectral sources.  Dynamic fields and product-defined intermediate fields ARE
 * sources; the other intermediate fields are linear in earlier fields and flatten onto them, each link
 * carrying its Nyquist / q = 0 zero rules (A9, A10) and the denominator of a field with its own lhs. */
bool flatten(const pss_system *s, const std::vector<int> &den_of, std::vector<std::vector<DOp>> &flat) {
  const int nf = (int)s->fields.size();
  flat.assign(nf, std::vector<DOp>());
  for (int f = 0; f < nf; ++f) {
    const FieldH &F = s->fields[f];
    if (s->dyn_slot[f] >= 0) {
      pss_op one = {1.0, 0, 0, {0, 0, 0}};
      flat[f].push_back(link_op(s, one, s->dyn_slot[f]));
      continue;
    }
    for (const DefH &d : F.defs) {
      DOp l = link_op(s, d.op, 0);
      l.den = (int8_t)den_of[f];
      for (const DOp &e : flat[d.src]) {
        DOp r;
        if (!compose(l, e, r)) return false;
        push_merged(flat[f], r);
      }
    }
  }
  return true;
}

/* (factors, groups, terms) of one round: the product terms `terms` (field = target source slot) */
struct RoundH {
  std::vector<DFactor> fac;
  std::vector<DGroup> grp;
  std::vector<DTerm> term;
};
struct PTermH { int target; pss_op outer; std::vector<int> factors; };

int build_round(const pss_system *s, const std::vector<PTermH> &terms, const std::vector<std::vector<DOp>> &flat,
                const std::vector<int> &order_of, std::vector<DOp> &lin, RoundH &R) {
  const int nf = (int)s->fields.size();
  std::vector<int> fac_slot(nf, -1);
  for (int f = 0; f < nf; ++f) {
    bool used = false;
    for (const PTermH &t : terms)
      for (int g : t.factors) if (g == f) used = true;
    if (!used) continue;
    if ((int)R.fac.size() >= PSS_P_MAX_FAC) return PSS_EUNSUPPORTED;
    DFactor F;
    std::memset(&F, 0, sizeof(F));
    F.lin_beg = (int16_t)lin.size();
    for (const DOp &e : flat[f]) lin.push_back(e);
    F.lin_end = (int16_t)lin.size();
    F.order = (int16_t)order_of[f];
    fac_slot[f] = (int)R.fac.size();
    R.fac.push_back(F);
  }
  /* groups of product terms: same target, same outer monomial (coef moves into the term) */
  std::vector<std::vector<DTerm>> gterms;
  for (const PTermH &t : terms) {
    DOp o = link_op(s, t.outer, t.target);
    o.coef = 1.0;
    int g = -1;
    for (size_t i = 0; i < R.grp.size(); ++i)
      if (R.grp[i].target == t.target && same_monomial(R.grp[i].outer, o)) g = (int)i;
    if (g < 0) {
      if ((int)R.grp.size() >= PSS_P_MAX_GRP) return PSS_EUNSUPPORTED;
      DGroup G;
      std::memset(&G, 0, sizeof(G));
      G.outer = o;
      G.target = (int16_t)t.target;
      g = (int)R.grp.size();
      R.grp.push_back(G);
      gterms.push_back(std::vector<DTerm>());
    }
    DTerm dt;
    std::memset(&dt, 0, sizeof(dt));
    dt.coef = t.outer.coef;
    dt.nf = (int8_t)t.factors.size();
    for (size_t i = 0; i < t.factors.size(); ++i) dt.f[i] = (int8_t)fac_slot[t.factors[i]];
    gterms[(size_t)g].push_back(dt);
  }
  for (size_t g = 0; g < R.grp.size(); ++g) {
    R.grp[g].term_beg = (int16_t)R.term.size();
    for (const DTerm &dt : gterms[g]) R.term.push_back(dt);
    R.grp[g].term_end = (int16_t)R.term.size();
  }
  if ((int)R.term.size() > PSS_P_MAX_TERM) return PSS_EUNSUPPORTED;
  return PSS_OK;
}

void put_round(Program &P, const RoundH &facs, const RoundH &grps) {
  P.nfac = (int32_t)facs.fac.size();
  for (size_t i = 0; i < facs.fac.size(); ++i) P.fac[i] = facs.fac[i];
  P.ngrp = (int32_t)grps.grp.size();
  for (size_t i = 0; i < grps.grp.size(); ++i) P.grp[i] = grps.grp[i];
  P.nterm = (int32_t)grps.term.size();
  for (size_t i = 0; i < grps.term.size(); ++i) P.term[i] = grps.term[i];
}

int build_program(pss_system *s) {
  Program base;
  std::memset(&base, 0, sizeof(base));
  base.ndim = s->ndim;
  double dV = 1.0;
  for (int j = 0; j < 3; ++j) {
    base.n[j] = (int32_t)s->n[j];
    base.qs[j] = (j < s->ndim) ? 2.0 * 3.14159265358979323846 / ((double)s->n[j] * s->dx[j]) : 0.0;
    if (j < s->ndim) dV *= s->dx[j];
  }
  base.nxh = (int32_t)(s->n[0] / 2 + 1);
  base.dealias = s->dealias;
  base.dt = s->dt;
  base.invN = 1.0 / (double)s->N;
  base.seed_lo = (uint32_t)(s->seed & 0xffffffffu);
  base.seed_hi = (uint32_t)(s->seed >> 32);

  const int nf = (int)s->fields.size();
  /* spectral sources: dynamic fields first, then the intermediate fields that are defined by products */
  s->dyn_slot.assign(nf, -1);
  int nsrc = 0, ndyn = 0;
  for (int f = 0; f < nf; ++f)
    if (s->fields[f].dynamic) { s->dyn_slot[f] = nsrc++; ++ndyn; }
  for (int f = 0; f < nf; ++f)
    if (!s->fields[f].dynamic && !s->fields[f].aterms.empty()) s->dyn_slot[f] = nsrc++;
  if (nsrc > PSS_P_MAX_DYN) return PSS_EUNSUPPORTED;
  base.ndyn = nsrc;
  const bool multi = nsrc > ndyn;
  if (multi && (s->ndim == 1 || s->nrep != 1)) return PSS_EUNSUPPORTED; /* rounds: 2D/3D single systems */

  std::vector<DOp> lin;
  /* denominators of the intermediate fields with their own lhs: real-valued monomials only */
  std::vector<int> den_of(nf, 0);
  for (int f = 0; f < nf; ++f) {
    const FieldH &F = s->fields[f];
    if (F.dynamic || F.lhs.empty()) continue;
    if (base.nden >= PSS_P_MAX_DEN) return PSS_EUNSUPPORTED;
    DDen &D = base.den[base.nden];
    D.beg = (int16_t)lin.size();
    std::vector<DOp> tmp;
    for (const pss_op &op : F.lhs) {
      DOp d = link_op(s, op, 0);
      if (!real_op(d)) return PSS_EUNSUPPORTED;
      push_merged(tmp, d);
    }
    for (const DOp &e : tmp) lin.push_back(e);
    D.end = (int16_t)lin.size();
    den_of[f] = ++base.nden;
  }
  std::vector<std::vector<DOp>> flat;
  if (!flatten(s, den_of, flat)) return PSS_EUNSUPPORTED;

  /* highest product order every field appears in, over ALL products */
  std::vector<int> order_of(nf, 0);
  auto see = [&](const std::vector<int> &factors) {
    if (factors.size() < 2) return;
    for (int g : factors) if ((int)factors.size() > order_of[g]) order_of[g] = (int)factors.size();
  };
  for (const TermH &t : s->terms) see(t.factors);
  for (const FieldH &F : s->fields) for (const ATermH &t : F.aterms) see(t.factors);

  /* dependency level of every field: sources of level l are assigned in round l (dynamic fields: level 0, stepped last) */
  std::vector<int> level(nf, 0);
  int lmax = 0;
  for (int f = 0; f < nf; ++f) {
    const FieldH &F = s->fields[f];
    if (F.dynamic) continue;
    int lv = 0;
    for (const DefH &d : F.defs) lv = std::max(lv, level[d.src]);
    if (!F.aterms.empty()) {
      for (const ATermH &t : F.aterms) for (int g : t.factors) lv = std::max(lv, level[g]);
      lv += 1;
    }
    level[f] = lv;
    lmax = std::max(lmax, lv);
  }
  s->nround = lmax + 1;

  /* rounds 0 .. lmax-1: the product-defined intermediate fields of level round + 1; round lmax: the dynamic equations */
  std::vector<RoundH> R((size_t)s->nround);
  for (int k = 0; k < s->nround; ++k) {
    std::vector<PTermH> pt;
    if (k < lmax) {
      for (int f = 0; f < nf; ++f)
        if (s->dyn_slot[f] >= 0 && !s->fields[f].dynamic && level[f] == k + 1)
          for (const ATermH &t : s->fields[f].aterms) { PTermH x; x.target = s->dyn_slot[f]; x.outer = t.outer; x.factors = t.factors; pt.push_back(x); }
    } else {
      for (const TermH &t : s->terms)
        if (t.factors.size() >= 2) { PTermH x; x.target = s->dyn_slot[t.field]; x.outer = t.outer; x.factors = t.factors; pt.push_back(x); }
    }
    const int rc = build_round(s, pt, flat, order_of, lin, R[(size_t)k]);
    if (rc != PSS_OK) return rc;
  }

  /* per source slot: lhs, explicit linear terms, noise (dynamic) / linear part of the definition, denominator (intermediate) */
  std::vector<DDyn> slots((size_t)nsrc);
  std::vector<int> slot_level((size_t)nsrc, 0);
  for (int f = 0; f < nf; ++f) {
    if (s->dyn_slot[f] < 0) continue;
    const FieldH &F = s->fields[f];
    DDyn &d = slots[(size_t)s->dyn_slot[f]];
    std::memset(&d, 0, sizeof(d));
    d.field_id = f;
    slot_level[(size_t)s->dyn_slot[f]] = level[f];
    d.lhs_beg = (int16_t)lin.size();
    if (F.dynamic) {
      std::vector<DOp> tmp;
      for (const pss_op &op : F.lhs) push_merged(tmp, link_op(s, op, s->dyn_slot[f]));
      for (const DOp &e : tmp) lin.push_back(e);
    }
    d.lhs_end = (int16_t)lin.size();
    d.lin_beg = (int16_t)lin.size();
    {
      std::vector<DOp> tmp;
      if (F.dynamic) {
        for (const TermH &t : s->terms) {
          if (t.field != f || t.factors.size() != 1) continue;
          const DOp l = link_op(s, t.outer, 0);
          for (const DOp &e : flat[t.factors[0]]) {
            DOp r;
            if (!compose(l, e, r)) return PSS_EUNSUPPORTED;
            push_merged(tmp, r);
          }
        }
      } else {
        for (const DefH &df : F.defs) { /* linear part of a product-defined intermediate field; its den applies to the whole sum */
          const DOp l = link_op(s, df.op, 0);
          for (const DOp &e : flat[df.src]) {
            DOp r;
            if (!compose(l, e, r)) return PSS_EUNSUPPORTED;
            push_merged(tmp, r);
          }
        }
        d.den = (int16_t)den_of[f];
      }
      for (const DOp &e : tmp) lin.push_back(e);
    }
    d.lin_end = (int16_t)lin.size();
    d.noisy = (F.dynamic && F.noisy) ? 1 : 0;
    d.noise_qpow = (int16_t)F.qpow;
    d.noise_c = 2.0 * F.D * s->dt * (double)s->N / dV;
  }
  if (lin.size() > PSS_P_MAX_LIN) return PSS_EUNSUPPORTED;
  for (size_t i = 0; i < lin.size(); ++i) base.lin[i] = lin[i];
  base.nlin = (int32_t)lin.size();
  base.any_invq = 0;
  for (const DOp &d : lin) if (d.p > 0) base.any_invq = 1;
  for (const RoundH &r : R) for (const DGroup &g : r.grp) if (g.outer.p > 0) base.any_invq = 1;

  /* launch programs */
  s->PR.assign((size_t)s->nround, base);
  s->PU.assign((size_t)s->nround, base);
  for (int k = 0; k < s->nround; ++k) {
    put_round(s->PR[(size_t)k], R[(size_t)k], R[(size_t)k]);
    put_round(s->PU[(size_t)k], R[(size_t)((k + 1) % s->nround)], R[(size_t)k]);
    for (int i = 0; i < nsrc; ++i) {
      DDyn d = slots[(size_t)i];
      const bool is_dyn = s->fields[(size_t)d.field_id].dynamic;
      if (k == lmax) d.kind = is_dyn ? PSS_SLOT_STEP : PSS_SLOT_KEEP;
      else d.kind = (!is_dyn && slot_level[(size_t)i] == k + 1) ? PSS_SLOT_ASSIGN : PSS_SLOT_KEEP;
      s->PR[(size_t)k].dyn[i] = d;
      s->PU[(size_t)k].dyn[i] = d;
    }
  }
  s->P = s->PU[(size_t)lmax];
  Program &P = s->P;
  /* radial fast path (pss_program.h): L and the outer operator polynomials in q^2, every factor a polynomial in q^2
   * times one derivative monomial */
  {
    auto radial = [](const DOp &d) { return d.p == 0 && d.a[0] == 0 && d.a[1] == 0 && d.a[2] == 0 && d.zflags == 0 && d.m <= 4 && d.den == 0; };
    bool ok = env_int("PSS_RADIAL", 1) != 0 && !multi && P.nden == 0 && P.ndyn == 1 && P.ngrp <= 1 && P.dyn[0].lin_beg == P.dyn[0].lin_end;
    if (ok && P.dyn[0].noisy && (P.dyn[0].noise_qpow < 0 || (P.dyn[0].noise_qpow & 1) || P.dyn[0].noise_qpow > 14)) ok = false;
    for (int e = P.dyn[0].lhs_beg; ok && e < P.dyn[0].lhs_end; ++e) ok = radial(P.lin[e]);
    if (ok && P.ngrp == 1) ok = radial(P.grp[0].outer);
    for (int f = 0; ok && f < P.nfac; ++f) {
      const DOp &d0 = P.lin[P.fac[f].lin_beg];
      for (int e = P.fac[f].lin_beg; ok && e < P.fac[f].lin_end; ++e) {
        const DOp &d = P.lin[e];
        ok = d.p == 0 && d.m <= 4 && d.den == 0 && (d.zflags & 8) == 0 && d.a[0] == d0.a[0] && d.a[1] == d0.a[1] && d.a[2] == d0.a[2] &&
             d.zflags == d0.zflags && d.a[0] <= 3 && d.a[1] <= 3 && d.a[2] <= 3;
      }
      if (P.fac[f].lin_beg == P.fac[f].lin_end) ok = false;
    }
    if (ok) {
      for (int e = P.dyn[0].lhs_beg; e < P.dyn[0].lhs_end; ++e) P.rad_L[P.lin[e].m] -= P.lin[e].coef;
      if (P.ngrp == 1) P.rad_O[P.grp[0].outer.m] += P.grp[0].outer.coef;
      for (int f = 0; f < P.nfac; ++f) {
        const DOp &d0 = P.lin[P.fac[f].lin_beg];
        for (int e = P.fac[f].lin_beg; e < P.fac[f].lin_end; ++e) P.rad_F[f][P.lin[e].m] += P.lin[e].coef;
        for (int j = 0; j < 3; ++j) P.rad_a[f][j] = d0.a[j];
        P.rad_a[f][3] = (int8_t)(d0.zflags & 7);
      }
      P.rad_nhp = P.dyn[0].noisy ? P.dyn[0].noise_qpow / 2 : 0;
    }
    P.rad_ok = 0;
    if (ok) {
      P.rad_ok = 1; /* 2: some factor carries a derivative monomial */
      for (int f = 0; f < P.nfac; ++f)
        if (P.rad_a[f][0] | P.rad_a[f][1] | P.rad_a[f][2]) P.rad_ok = 2;
    }
  }
  if (!multi) { s->PR[0] = P; s->PU[0] = P; }
  s->nfac_max = s->ngrp_max = 0;
  for (const Program &X : s->PR) { s->nfac_max = std::max(s->nfac_max, (int)X.nfac); s->ngrp_max = std::max(s->ngrp_max, (int)X.ngrp); }
  return PSS_OK;
}

/* ---- launch plan ----------------------------------------------------------------------- */
/* entries of one axis' twiddle array: tw[n] followed by the per-pass tables (Geo::twoff) */
long long tw_entries(const Geo &g) {
  long long e = g.n;
  int lgL = 0;
  for (int q = 0; q < g.nr; ++q) lgL += g.lg[q];
  for (int q = 0; q < g.nr; ++q) { e += (long long)((1 << g.lg[q]) - 1) << (lgL - g.lg[q]); lgL -= g.lg[q]; }
  return e;
}

int geo_pad_h(const Geo &g, int p) { return p + (p >> g.sh[0]) + (p >> g.sh[1]) + (p >> g.sh[2]); }

Geo make_geo(int64_t n) {
  Geo g;
  std::memset(&g, 0, sizeof(g));
  g.n = (int32_t)n;
  const int lg = ilog2(n);
  const int np = (lg + 3) / 4;
  g.nr = np;
  for (int q = 0; q < np; ++q) g.lg[q] = lg / np + (q < lg % np ? 1 : 0);
  /* pad rows at the digit boundaries of the slot index (the last pass's digit sits in the low bits) */
  int b = 0, k = 0;
  for (int i = 0; i < 3; ++i) g.sh[i] = 31;
  for (int q = np - 1; q >= 1; --q) { b += g.lg[q]; g.sh[k++] = b; }
  g.npad = geo_pad_h(g, (int)n - 1) + 1;
  /* digit fields: the first pass's digit is the LOW digit of the frequency and the HIGH digit of the slot */
  int fs = 0, rem = lg;
  for (int q = 0; q < 4; ++q) {
    if (q < np) {
      rem -= g.lg[q];
      g.fs[q] = fs; g.ps[q] = rem; g.fm[q] = (1 << g.lg[q]) - 1;
      fs += g.lg[q];
    } else {
      g.fs[q] = 0; g.ps[q] = 0; g.fm[q] = 0;
    }
  }
  {
    long long off = n;
    int lgL = lg;
    for (int q = 0; q < 4; ++q) {
      g.twoff[q] = (int32_t)off;
      if (q < np) { off += (long long)((1 << g.lg[q]) - 1) << (lgL - g.lg[q]); lgL -= g.lg[q]; }
    }
  }
  return g;
}

const size_t SMEM_MAX = 227 * 1024;
const size_t SMEM_SOFT = 100 * 1024; /* leaves room for two CTAs per SM */

int round_threads(long long work) {
  long long t = ((work + 31) / 32) * 32;
  if (t < 64) t = 64;
  if (t > 256) t = 256;
  return (int)t;
}

/* the persistent kernel of pss_fused2d.cuh: one real-coefficient field with one product group on 1024^2 fp32 */
bool fused2d_eligible(const pss_system *s) {
  const Program &P = s->P;
  if (env_int("PSS_FUSED", 1) == 0) return false;
  if (s->ndim != 2 || s->prec != PSS_F32 || s->n[0] != f2d::N || s->n[1] != f2d::N) return false;
  if (P.ndyn != 1 || P.nfac != 1 || P.ngrp != 1) return false;
  if (P.dyn[0].lin_beg != P.dyn[0].lin_end) return false;
  if (!real_op(P.grp[0].outer)) return false;
  for (int e = P.dyn[0].lhs_beg; e < P.dyn[0].lhs_end; ++e) if (!real_op(P.lin[e])) return false;
  for (int e = P.fac[0].lin_beg; e < P.fac[0].lin_end; ++e) if (!real_op(P.lin[e])) return false;
  return true;
}

int make_plan(pss_system *s) {
  Plan &pl = s->plan;
  std::memset(&pl, 0, sizeof(pl));
  Program Pm = s->P; /* counts of the largest round */
  Pm.nfac = s->nfac_max;
  Pm.ngrp = s->ngrp_max;
  const Program &P = Pm;
  for (int j = 0; j < 3; ++j) pl.geo[j] = make_geo(s->n[j]);
  const size_t cs = s->csize;
  const int nxh = P.nxh;
  pl.kx_keep_max = 0;
  for (const Program &X : s->PR)
    for (int f = 0; f < X.nfac; ++f) {
      int cut = nxh;
      if (P.dealias != PSS_DEALIAS_OFF) {
        const int nn = (P.dealias == PSS_DEALIAS_TWO_THIRDS ? 2 : X.fac[f].order) + 1;
        cut = (int)((s->n[0] + nn - 1) / nn);
        if (cut > nxh) cut = nxh;
      }
      if (cut > pl.kx_keep_max) pl.kx_keep_max = cut;
    }
  pl.pdl = env_int("PSS_PDL", 1);
  pl.fused = fused2d_eligible(s) ? 1 : 0;
  if (pl.fused) {
    const int nn = (P.dealias == PSS_DEALIAS_OFF) ? 1 : ((P.dealias == PSS_DEALIAS_TWO_THIRDS ? 2 : P.fac[0].order) + 1);
    pl.fused_prune = (nn >= 4) ? 1 : 0;
  }
  if (s->ndim == 1) {
    const size_t bufs = (size_t)(P.nfac + P.ngrp);
    pl.one_smem = bufs * (size_t)pl.geo[0].npad * cs;
    if (pl.one_smem > SMEM_MAX) return PSS_EUNSUPPORTED;
    if (pl.one_smem < 16) pl.one_smem = 16;
    pl.one_threads = round_threads(s->n[0] / 4);
    return PSS_OK;
  }
  /* k_update: W contiguous last-axis lines per CTA */
  {
    const int64_t n = s->n[s->ndim - 1];
    const int64_t nlines = (s->ndim == 3) ? (int64_t)nxh * s->n[1] : nxh;
    const int nb0 = P.ngrp > P.ndyn ? P.ngrp : P.ndyn;
    const size_t per = (size_t)(nb0 + (P.nfac > 1 ? 1 : 0)) * (size_t)pl.geo[s->ndim - 1].npad * cs;
    if (per > SMEM_MAX) return PSS_EUNSUPPORTED;
    int W = 1;
    for (int cand = 8; cand >= 1; cand >>= 1) {
      if (per * cand > 40 * 1024 && cand > 1) continue; /* measured: small tiles win once a line fills ~32 KB */
      if ((nlines + cand - 1) / cand < 2 * 148 && cand > 1) continue;
      W = cand;
      break;
    }
    W = env_int("PSS_UPD_W", W);
    if (W < 1) W = 1;
    if (W > 32) W = 32; /* the kernel keeps one keep-bit per line in a 32-bit mask */
    while (W & (W - 1)) W &= W - 1; /* a power of two (the kernel indexes with shifts) */
    while (W > 1 && per * W > SMEM_MAX) W >>= 1;
    pl.upd_W = W;
    pl.upd_smem = per * W;
    pl.upd_blocks = (int)((nlines + W - 1) / W);
    pl.upd_threads = round_threads((n / 8) * W * (P.ngrp > 0 ? P.ngrp : 1));
    /* short lines in a big grid (3D): one thread per radix-16 butterfly and more, smaller CTAs per SM (measured) */
    if ((n / 16) * W * (P.ngrp > 0 ? P.ngrp : 1) <= 128 && pl.upd_blocks >= 12 * 148 && pl.upd_threads > 128) pl.upd_threads = 128;
    /* small lattices are latency-bound: at least n/2 threads (128..256) for the pointwise stage (measured) */
    if (n <= 512 && pl.upd_threads < 128) pl.upd_threads = (n >= 512) ? 256 : 128;
    pl.upd_threads = env_int("PSS_UPD_T", pl.upd_threads);
    if (pl.upd_threads < 32) pl.upd_threads = 32;
    if (pl.upd_threads > 256) pl.upd_threads = 256; /* __launch_bounds__(256) */
    pl.upd_threads &= ~31;
  }
  /* k_rows: Wc pairs of rows per CTA (2*Wc contiguous rows of every kx) */
  if (P.ngrp > 0) {
    const int64_t nx = s->n[0];
    const int64_t R = s->N / nx;
    const size_t per = (size_t)(P.nfac + (P.ngrp > 1 ? 1 : 0)) * (size_t)pl.geo[0].npad * cs;
    if (per > SMEM_MAX) return PSS_EUNSUPPORTED;
    const int wc_sector = (cs == 8) ? 2 : 1; /* 2*Wc complex = one 32-byte sector */
    int Wc = 1;
    for (int cand = 8; cand >= 1; cand >>= 1) {
      if (2 * cand > R) continue;
      if (per * cand > SMEM_SOFT && cand > wc_sector) continue; /* whole 32-byte sectors first, then occupancy */
      if (per * cand > SMEM_MAX) continue;
      if (R / (2 * cand) < 2 * 148 && cand > wc_sector) continue;
      Wc = cand;
      break;
    }
    Wc = env_int("PSS_ROW_WC", Wc);
    if (Wc < 1) Wc = 1;
    while (Wc & (Wc - 1)) Wc &= Wc - 1; /* a power of two (the kernel indexes with shifts) */
    while (Wc > 1 && (per * Wc > SMEM_MAX || 2 * Wc > R || R % (2 * Wc) != 0)) Wc >>= 1;
    pl.row_Wc = Wc;
    pl.row_smem = per * Wc;
    pl.row_blocks = (int)(R / (2 * Wc));
    pl.row_threads = round_threads((nx / 8) * Wc * (P.nfac > 0 ? P.nfac : 1));
    if ((nx / 16) * Wc * (P.nfac > 0 ? P.nfac : 1) <= 128 && pl.row_blocks >= 12 * 148 && pl.row_threads > 128) pl.row_threads = 128;
    /* a tile that leaves room for one CTA per SM only gets 512 threads (fp32; the fp64 butterflies need the registers) */
    if (pl.row_smem > 113 * 1024 && cs == 8 && (nx / 16) * Wc * (P.nfac > 0 ? P.nfac : 1) >= 512) pl.row_threads = 512;
    pl.row_threads = env_int("PSS_ROW_T", pl.row_threads);
    if (pl.row_threads > 512) pl.row_threads = 512;
    if (pl.row_threads < 32) pl.row_threads = 32;
    pl.row_threads &= ~31;
  }
  if (s->ndim == 3) {
    int W = env_int("PSS_MID_W", (int)(128 / cs));
    if (W < 1) W = 1;
    while (W & (W - 1)) W &= W - 1; /* a power of two, so that it divides nz */
    if (W > s->n[2]) W = (int)s->n[2];
    while ((size_t)W * pl.geo[1].npad * cs > SMEM_MAX && W > 1) W >>= 1;
    if ((size_t)W * pl.geo[1].npad * cs > SMEM_MAX) return PSS_EUNSUPPORTED;
    pl.mid_W = W;
    pl.mid_smem = (size_t)W * pl.geo[1].npad * cs;
    pl.mid_threads = env_int("PSS_MID_T", round_threads((s->n[1] / 32) * W)); /* two radix-16 butterflies per thread (measured) */
    if (pl.mid_threads < 32) pl.mid_threads = 32;
    if (pl.mid_threads > 256) pl.mid_threads = 256; /* __launch_bounds__(256) */
    pl.mid_threads &= ~31;
  }
  return PSS_OK;
}

size_t align_up(size_t v, size_t a) { return (v + a - 1) / a * a; }

void carve_workspace(pss_system *s) {
  const Program &P = s->P;
  size_t off = 0;
  const size_t arr = align_up((size_t)s->M * s->csize, 256);
  const size_t R = (size_t)s->nrep; /* arrays of one kind: [replica][field][M] */
  s->off_state = off; off += arr * (size_t)P.ndyn * R;
  s->off_psix = off;  off += arr * (size_t)s->nfac_max * R;
  s->off_phat = off;  off += arr * (size_t)s->ngrp_max * R;
  s->off_scratch = off; off += arr;
  s->off_ureal = off; off += align_up((size_t)s->N * s->rsize, 256);
  for (int j = 0; j < 3; ++j) { s->off_tw[j] = off; off += align_up((size_t)tw_entries(s->plan.geo[j]) * s->csize, 256); }
  s->off_bar = off; off += 512; /* first-generation counter | the two counters of pss_persist2d.cuh */
  s->ws_need = off;
}

template <typename T> typename cplx_of<T>::type *carr(pss_system *s, size_t off, int idx) {
  const size_t arr = align_up((size_t)s->M * s->csize, 256);
  return reinterpret_cast<typename cplx_of<T>::type *>(s->ws + off + arr * (size_t)idx);
}
/* NOTE: arrays of one kind are spaced by the ALIGNED size; kernels take M_stride = arr / csize */
long long arr_stride(const pss_system *s) { return (long long)(align_up((size_t)s->M * s->csize, 256) / s->csize); }

template <typename T> const typename cplx_of<T>::type *twp(pss_system *s, int axis) {
  return reinterpret_cast<const typename cplx_of<T>::type *>(s->ws + s->off_tw[axis]);
}

template <typename T> int set_attrs(pss_system *s) {
  CK(cudaFuncSetAttribute(k_update<T, 0, 2>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)SMEM_MAX));
  CK(cudaFuncSetAttribute(k_update<T, 0, PSS_P_MAX_DYN>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)SMEM_MAX));
  CK(cudaFuncSetAttribute(k_update<T, 1, 1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)SMEM_MAX));
  CK(cudaFuncSetAttribute(k_update<T, 2, 1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)SMEM_MAX));
  CK(cudaFuncSetAttribute(k_rows<T, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)SMEM_MAX));
  CK(cudaFuncSetAttribute(k_rows<T, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)SMEM_MAX));
  CK(cudaFuncSetAttribute(k_mid<-1, T>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)SMEM_MAX));
  CK(cudaFuncSetAttribute(k_mid<+1, T>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)SMEM_MAX));
  CK(cudaFuncSetAttribute(k_last<-1, T>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)SMEM_MAX));
  CK(cudaFuncSetAttribute(k_last<+1, T>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)SMEM_MAX));
  CK(cudaFuncSetAttribute(k_user_x<-1, T>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)SMEM_MAX));
  CK(cudaFuncSetAttribute(k_user_x<+1, T>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)SMEM_MAX));
  CK(cudaFuncSetAttribute(k_step1d<T>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)SMEM_MAX));
  return PSS_OK;
}

/* the persistent kernel needs every CTA co-resident (its phases are separated by a grid barrier): check that a
 * cooperative launch of f2d::NCTA CTAs fits this device, else fall back to the two-kernel path. */
int setup_fused(pss_system *s) {
  if (!s->plan.fused) return PSS_OK;
  int dev = 0, coop = 0, nsm = 0, occ = 0;
  CK(cudaGetDevice(&dev));
  CK(cudaDeviceGetAttribute(&coop, cudaDevAttrCooperativeLaunch, dev));
  CK(cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, dev));
  CK(cudaFuncSetAttribute(f2d::k_fused2d<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)f2d::SMEM_BYTES));
  CK(cudaFuncSetAttribute(f2d::k_fused2d<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)f2d::SMEM_BYTES));
  if (s->plan.fused_prune)
    CK(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, f2d::k_fused2d<true>, f2d::THREADS, f2d::SMEM_BYTES));
  else
    CK(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, f2d::k_fused2d<false>, f2d::THREADS, f2d::SMEM_BYTES));
  if (!coop || (long long)occ * nsm < f2d::NCTA) s->plan.fused = 0;
  s->plan.persist = 0;
  if (s->plan.fused && s->plan.fused_prune && env_int("PSS_PERSIST", 1) != 0) {
    int occ3 = 0;
    CK(cudaFuncSetAttribute(p2d::k_persist2d, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)p2d::SMEM_BYTES));
    CK(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ3, p2d::k_persist2d, p2d::THREADS, p2d::SMEM_BYTES));
    if ((long long)occ3 * nsm >= p2d::NCTA) s->plan.persist = 1;
  }

  /* ensembles: the two-replica kernel needs more shared memory; fall back to one launch per replica if it does not fit */
  s->plan.fused_pair = 0;
  if (s->plan.fused && s->nrep >= 2 && env_int("PSS_FUSED_PAIR", 1) != 0) {
    int occ2 = 0;
    CK(cudaFuncSetAttribute(f2d::k_fused2d_pair<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)f2d::SMEM_BYTES_PAIR));
    CK(cudaFuncSetAttribute(f2d::k_fused2d_pair<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)f2d::SMEM_BYTES_PAIR));
    if (s->plan.fused_prune)
      CK(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ2, f2d::k_fused2d_pair<true>, f2d::THREADS, f2d::SMEM_BYTES_PAIR));
    else
      CK(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ2, f2d::k_fused2d_pair<false>, f2d::THREADS, f2d::SMEM_BYTES_PAIR));
    if ((long long)occ2 * nsm >= f2d::NCTA) s->plan.fused_pair = 1;
  }
  return PSS_OK;
}

template <typename T> int upload_twiddles(pss_system *s) {
  typedef typename cplx_of<T>::type C;
  for (int j = 0; j < s->ndim; ++j) {
    std::vector<C> tw((size_t)s->n[j]);
    const long double PI_L = 3.14159265358979323846264338327950288L;
    for (int64_t i = 0; i < s->n[j]; ++i) {
      const long double a = 2.0L * PI_L * (long double)i / (long double)s->n[j];
      tw[(size_t)i].x = (T)cosl(a);
      tw[(size_t)i].y = (T)(-sinl(a));
    }
    /* per-pass tables: the same numbers, re-ordered so that consecutive butterflies read consecutive entries */
    const Geo &g = s->plan.geo[j];
    int lgn = 0;
    for (int q = 0; q < g.nr; ++q) lgn += g.lg[q];
    tw.resize((size_t)tw_entries(g));
    int lgL = lgn;
    for (int q = 0; q < g.nr; ++q) {
      const int R = 1 << g.lg[q], lgLs = lgL - g.lg[q];
      for (int m = 1; m < R; ++m)
        for (int i = 0; i < (1 << lgLs); ++i)
          tw[(size_t)g.twoff[q] + ((size_t)(m - 1) << lgLs) + i] = tw[((size_t)m * i) << (lgn - lgL)];
      lgL -= g.lg[q];
    }
    CK(cudaMemcpyAsync(s->ws + s->off_tw[j], tw.data(), tw.size() * sizeof(C), cudaMemcpyHostToDevice, s->stream));
    CK(cudaStreamSynchronize(s->stream)); /* tw is a stack-lifetime host buffer */
  }
  return PSS_OK;
}

/* ---- launches -------------------------------------------------------------------------- */
enum { KIND_ROWS = 0, KIND_UPDATE = 1, KIND_MID = 2, KIND_FUSED = 3, KIND_COUNT = 4 };
void prof_mark(pss_system *s, int kind, bool begin) {
  if (!s->prof_on) return;
  cudaEvent_t e;
  if (cudaEventCreate(&e) != cudaSuccess) return;
  cudaEventRecord(e, s->stream);
  s->prof_ev.push_back(e);
  if (begin) s->prof_kind.push_back(kind);
}

/* Programmatic dependent launch: the next kernel of the step is launched while the previous one drains; every step
 * kernel starts with griddepcontrol.wait, so nothing is read or written before the previous grid has completed. */
template <typename... KArgs, typename... Args>
cudaError_t launch_pdl(void (*kernel)(KArgs...), dim3 grid, unsigned threads, size_t smem, cudaStream_t stream, bool pdl, Args... args) {
  cudaLaunchConfig_t cfg;
  std::memset(&cfg, 0, sizeof(cfg));
  cfg.gridDim = grid;
  cfg.blockDim = dim3(threads);
  cfg.dynamicSmemBytes = smem;
  cfg.stream = stream;
  cudaLaunchAttribute at[1];
  at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  at[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = at;
  cfg.numAttrs = pdl ? 1 : 0;
  return cudaLaunchKernelEx(&cfg, kernel, args...);
}

template <typename T> int launch_mid(pss_system *s, int sgn, size_t off, int nbatch, int kx_count, const Program *Pf = nullptr, int nrep = 1) {
  MidArgs<T> a;
  std::memset(&a, 0, sizeof(a));
  a.nx = (int)s->n[0];
  if (Pf && Pf->dealias != PSS_DEALIAS_OFF) /* Pf: the program whose factor list is being transformed (mask per factor) */
    for (int f = 0; f < nbatch; ++f) a.nn[f] = (Pf->dealias == PSS_DEALIAS_TWO_THIRDS ? 2 : Pf->fac[f].order) + 1;
  a.arr = carr<T>(s, off, 0);
  a.tw = twp<T>(s, 1);
  a.M = arr_stride(s);
  a.ny = (int)s->n[1];
  a.nz = (int)s->n[2];
  a.W = s->plan.mid_W;
  a.kx_count = kx_count;
  a.nbatch = nbatch;
  a.geo = s->plan.geo[1];
  dim3 grid((unsigned)(s->n[2] / s->plan.mid_W), (unsigned)kx_count, (unsigned)(nbatch * nrep));
  prof_mark(s, KIND_MID, true);
  if (sgn < 0) launch_pdl(k_mid<-1, T>, grid, s->plan.mid_threads, s->plan.mid_smem, s->stream, s->plan.pdl != 0, a);
  else launch_pdl(k_mid<+1, T>, grid, s->plan.mid_threads, s->plan.mid_smem, s->stream, s->plan.pdl != 0, a);
  prof_mark(s, KIND_MID, false);
  CKL("k_mid");
  return PSS_OK;
}

template <typename T> int launch_update(pss_system *s, int prologue, uint64_t step, const Program &P) {
  UpdArgs<T> a;
  a.state = carr<T>(s, s->off_state, 0);
  a.psix = carr<T>(s, s->off_psix, 0);
  a.phat = carr<T>(s, s->off_phat, 0);
  a.tw = twp<T>(s, s->ndim - 1);
  a.M = arr_stride(s);
  a.n = (int)s->n[s->ndim - 1];
  a.lgn = ilog2(a.n);
  a.nlines = (s->ndim == 3) ? (int)(P.nxh * s->n[1]) : P.nxh;
  a.W = s->plan.upd_W;
  a.lgW = ilog2(a.W);
  a.lg_ny = ilog2(s->n[1]);
  a.prologue = prologue;
  a.step = step;
  a.geo = s->plan.geo[s->ndim - 1];
  prof_mark(s, KIND_UPDATE, true);
  const dim3 grid((unsigned)s->plan.upd_blocks, (unsigned)s->nrep);
  const bool pdl = s->plan.pdl != 0;
  if (P.rad_ok == 1) launch_pdl(k_update<T, 1, 1>, grid, s->plan.upd_threads, s->plan.upd_smem, s->stream, pdl, P, a);
  else if (P.rad_ok == 2) launch_pdl(k_update<T, 2, 1>, grid, s->plan.upd_threads, s->plan.upd_smem, s->stream, pdl, P, a);
  else if (P.ndyn <= 2) launch_pdl(k_update<T, 0, 2>, grid, s->plan.upd_threads, s->plan.upd_smem, s->stream, pdl, P, a);
  else launch_pdl(k_update<T, 0, PSS_P_MAX_DYN>, grid, s->plan.upd_threads, s->plan.upd_smem, s->stream, pdl, P, a);
  prof_mark(s, KIND_UPDATE, false);
  CKL("k_update");
  if (s->ndim == 3 && P.nfac > 0) return launch_mid<T>(s, +1, s->off_psix, P.nfac, s->plan.kx_keep_max, &P, s->nrep);
  return PSS_OK;
}

template <typename T> int launch_rows(pss_system *s, const Program &P) {
  RowArgs<T> a;
  a.psix = carr<T>(s, s->off_psix, 0);
  a.phat = carr<T>(s, s->off_phat, 0);
  a.tw = twp<T>(s, 0);
  a.M = arr_stride(s);
  a.R = s->N / s->n[0];
  a.nx = (int)s->n[0];
  a.Wc = s->plan.row_Wc;
  a.geo = s->plan.geo[0];
  prof_mark(s, KIND_ROWS, true);
  const dim3 grid((unsigned)s->plan.row_blocks, (unsigned)s->nrep);
  const bool pdl = s->plan.pdl != 0;
  if (s->plan.row_threads > 256) launch_pdl(k_rows<T, true>, grid, s->plan.row_threads, s->plan.row_smem, s->stream, pdl, P, a);
  else launch_pdl(k_rows<T, false>, grid, s->plan.row_threads, s->plan.row_smem, s->stream, pdl, P, a);
  prof_mark(s, KIND_ROWS, false);
  CKL("k_rows");
  if (s->ndim == 3) return launch_mid<T>(s, -1, s->off_phat, P.ngrp, P.nxh, nullptr, s->nrep);
  return PSS_OK;
}

/* nsteps steps (plus the E-rebuilding prologue when the state was just set) in one cooperative launch */
int launch_fused(pss_system *s, int64_t nsteps) {
  const int prologue = s->psix_valid ? 0 : 1;
  const void *fn1 = s->plan.fused_prune ? (const void *)f2d::k_fused2d<true> : (const void *)f2d::k_fused2d<false>;
  const void *fn2 = s->plan.fused_prune ? (const void *)f2d::k_fused2d_pair<true> : (const void *)f2d::k_fused2d_pair<false>;
  /* replica r: arrays [r], seed + r.  With the second-generation kernel (plan.persist, the default rule) every replica
   * gets its own launch; only the first-generation fallback pairs them (k_fused2d_pair overlaps one replica's L2
   * exchanges with the other's transforms, a last odd one alone) */
  for (int r = 0; r < s->nrep;) {
    /* (the second-generation kernel runs the replicas one launch each: as fast per replica-step as the pair kernel) */
    const bool pair = s->plan.fused_pair && !s->plan.persist && r + 1 < s->nrep;
    Program Pr = s->P;
    const uint64_t sd = s->seed + (uint64_t)r;
    Pr.seed_lo = (uint32_t)(sd & 0xffffffffu);
    Pr.seed_hi = (uint32_t)(sd >> 32);
    f2d::Args a;
    a.state = carr<float>(s, s->off_state, r * Pr.ndyn);
    a.E = carr<float>(s, s->off_psix, r * Pr.nfac);
    a.Z = carr<float>(s, s->off_phat, r * Pr.ngrp);
    a.tw = twp<float>(s, 0);
    a.bar = reinterpret_cast<unsigned long long *>(s->ws + s->off_bar);
    a.bar_base = s->bar_count;
    a.nsteps = nsteps;
    a.step0 = s->step;
    a.prologue = prologue;
    a.rep_stride = arr_stride(s); /* ndyn = nfac = ngrp = 1: consecutive replicas are one array apart */
    void *params[2] = {(void *)&Pr, (void *)&a};
    cudaError_t e;
    if (!pair && s->plan.persist) {
      /* second-generation kernel (pss_persist2d.cuh): two grid-barrier counters (bar[0], bar[16]; zeroed before every launch),
       * exchange blocks fetched with cp.async.cg; an ensemble gets one launch per replica */
      p2d::Args pa;
      pa.state = a.state;
      pa.Eg = a.E; /* the factor array and the group array hold the two exchange arrays */
      pa.Zg = a.Z;
      pa.tw = a.tw;
      pa.bar = a.bar + 32; /* 256 bytes past the first-generation counter; its two counters start from zero in every launch */
      pa.nsteps = nsteps; pa.step0 = s->step; pa.prologue = prologue;
      pa.gate = std::min(std::max(env_int("PSS_NOISE_GATE", 200), 0), 100000); /* poll interval in ns, 0 = gate off */
      pa.prio = env_int("PSS_P2D_PRIO", 1) != 0 ? 1 : 0;
      pa.dbg = 0; /* knock-out switches and time stamps exist in -DPSS_P2D_DEBUG builds only */
      pa.ts = nullptr;
#ifdef PSS_P2D_DEBUG
      pa.dbg = env_int("PSS_P2D_DBG", 0);
      pa.ts = env_int("PSS_P2D_TS", 0) ? reinterpret_cast<long long *>(s->ws + s->off_scratch) : nullptr;
#endif
      CK(cudaMemsetAsync(pa.bar, 0, 256, s->stream));
      void *pparams[2] = {(void *)&Pr, (void *)&pa};
      prof_mark(s, KIND_FUSED, true);
      e = cudaLaunchCooperativeKernel((const void *)p2d::k_persist2d, dim3(p2d::NCTA), dim3(p2d::THREADS), pparams, p2d::SMEM_BYTES, s->stream);
      prof_mark(s, KIND_FUSED, false);
      if (e != cudaSuccess) return cuda_fail(s, e, "k_persist2d");
      CKL("k_persist2d");
#ifdef PSS_P2D_DEBUG
      if (pa.ts && nsteps >= 3) { /* timing experiment: globaltimer stamps, min / median / max over all groups */
        std::vector<long long> h(129 * 2 * 32);
        cudaStreamSynchronize(s->stream);
        cudaMemcpy(h.data(), pa.ts, h.size() * sizeof(long long), cudaMemcpyDeviceToHost);
        long long t00 = -1;
        for (int c = 0; c < 128; ++c) for (int g = 0; g < 2; ++g) { const long long v = h[(c * 2 + g) * 32]; if (v && (t00 < 0 || v < t00)) t00 = v; }
        for (int i = 0; i < 18; ++i) {
          std::vector<long long> v;
          for (int c = 0; c < 129; ++c) for (int g = 0; g < 2; ++g) if (h[(c * 2 + g) * 32 + i]) v.push_back(h[(c * 2 + g) * 32 + i] - t00);
          if (v.empty()) continue;
          std::sort(v.begin(), v.end());
          std::printf("stamp %2d: n=%3d min %6lld med %6lld max %6lld ns\n", i, (int)v.size(), v.front(), v[v.size() / 2], v.back());
        }
      }
#endif
    } else {
      prof_mark(s, KIND_FUSED, true);
      e = cudaLaunchCooperativeKernel(pair ? fn2 : fn1, dim3(f2d::NCTA), dim3(f2d::THREADS), params,
                                      pair ? f2d::SMEM_BYTES_PAIR : f2d::SMEM_BYTES, s->stream);
      prof_mark(s, KIND_FUSED, false);
      if (e != cudaSuccess) return cuda_fail(s, e, "k_fused2d");
      CKL("k_fused2d");
      s->bar_count += (unsigned long long)f2d::NCTA * (unsigned long long)(2 * nsteps + prologue);
    }
    r += pair ? 2 : 1;
  }
  s->psix_valid = true;
  s->step += (uint64_t)nsteps;
  return PSS_OK;
}

template <typename T> int do_steps_chunk(pss_system *s, int64_t nsteps) {
  const Program &P = s->P;
  if (nsteps == 0) return PSS_OK;
  if (s->ndim == 1) {
    Step1dArgs<T> a;
    a.state = carr<T>(s, s->off_state, 0);
    a.tw = twp<T>(s, 0);
    a.M = arr_stride(s);
    a.nx = (int)s->n[0];
    a.nsteps = nsteps;
    a.step0 = s->step;
    a.geo = s->plan.geo[0];
    k_step1d<T><<<s->nrep, s->plan.one_threads, s->plan.one_smem, s->stream>>>(P, a);
    CKL("k_step1d");
    s->step += (uint64_t)nsteps;
    return PSS_OK;
  }
  int rc;
  if (s->plan.fused) return launch_fused(s, nsteps);
  /* one round of (k_rows, k_update) per dependency level of the product-defined intermediate fields,
   * the dynamic equations last; without such fields this is the single pair of round 0 */
  const int last = s->nround - 1;
  if (s->nfac_max > 0 && !s->psix_valid) {
    if ((rc = launch_update<T>(s, 1, s->step, s->PU[(size_t)last])) != PSS_OK) return rc;
    s->psix_valid = true;
  }
  for (int64_t i = 0; i < nsteps; ++i) {
    for (int k = 0; k <= last; ++k) {
      if (s->PR[(size_t)k].ngrp > 0 && (rc = launch_rows<T>(s, s->PR[(size_t)k])) != PSS_OK) return rc;
      if ((rc = launch_update<T>(s, 0, s->step, s->PU[(size_t)k])) != PSS_OK) return rc;
    }
    s->step += 1;
  }
  return PSS_OK;
}

/* Hermitian projection of the state (reading A25).  The fields are real, so on the two planes of the
 * half-spectrum that hold both members of a conjugate pair, kx = 0 and kx = nx/2, the state must satisfy
 * phi(-k) = conj(phi(k)).  The state of this library lives in Fourier space for the whole run and is never rebuilt from
 * real space, and rounding breaks that symmetry by one ulp per step.  The C2R transforms ignore the anti-Hermitian part,
 * so the nonlinear terms never see it and cannot saturate it; Eq. 18 multiplies it by 1/(1 - dt L_q) every step like
 * any other mode.  Where L_q > 0 (Model B's spinodal band, rate 1/4 per unit time at q^2 = 1/2) it grows without bound:
 * measured at 1024^2 fp32, as large as the largest physical mode after 10^4 steps, NaN after 2 10^4.  Every
 * herm_period-th step (counted on the absolute step number, so that pss_step(a); pss_step(b) == pss_step(a + b) and a
 * restored checkpoint continue bit for bit) the pairs are replaced by their Hermitian mean and the self-conjugate modes
 * lose their imaginary part: the identity in exact arithmetic, idempotent in floating point.  The factor arrays are
 * rebuilt from the projected state (prologue), again so that a run restored from a checkpoint taken there agrees. */
/* The period.  Between two projections the anti-Hermitian part may grow by at most a factor 16: with
 * g = max over the two planes and the dynamic fields of |1/(1 - dt L_q)| (evaluated on the host in double),
 * period = largest power of two <= ln 16 / ln g.  That analysis is complete for a single dynamic field without explicit
 * linear terms (nothing else acts on the anti-Hermitian part): cap 1024.  Explicit linear terms couple the fields'
 * anti-Hermitian parts in ways the diagonal factor does not bound: cap 128 there.  Model B, dt = 0.01: g = 1.0025, 1024. */
int64_t plan_hermitian(const pss_system *s) {
  const double two_pi = 6.283185307179586476925286766559;
  bool simple = true;
  int ndynf = 0;
  for (const FieldH &F : s->fields) ndynf += F.dynamic ? 1 : 0;
  for (const TermH &t : s->terms) if (t.factors.size() == 1) simple = false;
  if (ndynf != 1) simple = false;
  const int64_t cap = simple ? 1024 : 128;
  double lng = 0.0;
  for (const FieldH &F : s->fields) {
    if (!F.dynamic || F.lhs.empty()) continue;
    for (int hi = 0; hi < 2; ++hi)
      for (int64_t k2 = 0; k2 < s->n[2]; ++k2)
        for (int64_t k1 = 0; k1 < s->n[1]; ++k1) {
          const int64_t kk[3] = {hi ? s->n[0] / 2 : 0, k1, k2};
          double q[3] = {0, 0, 0}, q2 = 0.0;
          bool nyq[3] = {false, false, false};
          for (int j = 0; j < s->ndim; ++j) {
            const int64_t sk = (2 * kk[j] <= s->n[j]) ? kk[j] : kk[j] - s->n[j];
            q[j] = two_pi * (double)sk / ((double)s->n[j] * s->dx[j]);
            nyq[j] = s->n[j] > 1 && 2 * kk[j] == s->n[j];
            q2 += q[j] * q[j];
          }
          double lre = 0.0, lim = 0.0; /* L_q = -sum coef Op(q) (pss_add_linear) */
          for (const pss_op &op : F.lhs) {
            double r = op.coef * std::pow(q2, op.q2_pow);
            if (op.invq_pow > 0) r = (q2 > 0.0) ? r * std::pow(q2, -0.5 * op.invq_pow) : 0.0;
            int sdeg = 0;
            for (int j = 0; j < 3; ++j) {
              if (op.iq_pow[j] > 0) r = (nyq[j] && (op.iq_pow[j] & 1)) ? 0.0 : r * std::pow(q[j], op.iq_pow[j]);
              sdeg += op.iq_pow[j];
            }
            switch (sdeg & 3) { case 0: lre -= r; break; case 1: lim -= r; break; case 2: lre += r; break; default: lim += r; }
          }
          const double dre = 1.0 - s->dt * lre, dim = -s->dt * lim, d2 = dre * dre + dim * dim;
          if (d2 < 1.0) lng = std::max(lng, d2 > 0.0 ? -0.5 * std::log(d2) : 1e300);
        }
  }
  if (lng <= 0.0) return cap;
  const double lim16 = std::log(16.0) / lng;
  int64_t p = 1;
  while (2 * p <= cap && (double)(2 * p) <= lim16) p *= 2;
  return p;
}

template <typename T>
__global__ void k_hermitize(typename cplx_of<T>::type *state, long long stride, int nxh, int ny, int nz) {
  typedef typename cplx_of<T>::type C;
  C *const arr = state + (size_t)blockIdx.y * (size_t)stride; /* internal layout: [kx][y][z] */
  const long long plane = (long long)ny * nz;
  for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < 2 * plane; i += (long long)gridDim.x * blockDim.x) {
    const bool hi = i >= plane;
    const long long idx = hi ? i - plane : i;
    const int y = (int)(idx / nz), z = (int)(idx % nz);
    const long long pidx = (long long)((ny - y) % ny) * nz + (nz - z) % nz;
    if (idx > pidx) continue; /* the pair is handled by its lower index */
    C *const p = arr + (hi ? (size_t)(nxh - 1) * (size_t)plane : (size_t)0);
    C a = p[idx];
    if (idx == pidx) {
      a.y = (T)0;
      p[idx] = a;
    } else {
      C b = p[pidx];
      a.x = (T)0.5 * (a.x + b.x);
      a.y = (T)0.5 * (a.y - b.y);
      b.x = a.x;
      b.y = -a.y;
      p[idx] = a;
      p[pidx] = b;
    }
  }
}

template <typename T> int launch_hermitize(pss_system *s) {
  const long long plane = (long long)s->n[1] * s->n[2];
  const unsigned bx = (unsigned)std::min<long long>(592, (2 * plane + 255) / 256);
  const int narr = s->nrep * s->P.ndyn; /* state arrays: [replica][dynamic field], arr_stride apart */
  for (int a0 = 0; a0 < narr; a0 += 65535) {
    const int na = std::min(65535, narr - a0);
    k_hermitize<T><<<dim3(bx, (unsigned)na), 256, 0, s->stream>>>(carr<T>(s, s->off_state, a0), arr_stride(s), s->P.nxh, (int)s->n[1], (int)s->n[2]);
    CKL("k_hermitize");
  }
  s->psix_valid = false;
  return PSS_OK;
}

/* nsteps steps, cut at the multiples of herm_period of the absolute step number */
template <typename T> int do_steps_core(pss_system *s, int64_t nsteps) {
  while (nsteps > 0) {
    const int64_t n = std::min<int64_t>(nsteps, s->herm_period - (int64_t)(s->step % (uint64_t)s->herm_period));
    int rc = do_steps_chunk<T>(s, n);
    if (rc != PSS_OK) return rc;
    nsteps -= n;
    if (s->step % (uint64_t)s->herm_period == 0 && (rc = launch_hermitize<T>(s)) != PSS_OK) return rc;
  }
  return PSS_OK;
}

template <typename T> int do_set_field(pss_system *s, int slot, const void *src, int on_device) {
  const T *real = (const T *)src;
  if (!on_device) {
    CK(cudaMemcpyAsync(s->ws + s->off_ureal, src, (size_t)s->N * sizeof(T), cudaMemcpyHostToDevice, s->stream));
    real = (const T *)(s->ws + s->off_ureal);
  }
  UserArgs<T> a;
  a.real = const_cast<T *>(real);
  const int sidx = s->sel * s->P.ndyn + slot; /* state array of the selected replica */
  a.arr = carr<T>(s, s->off_state, sidx);
  a.tw = twp<T>(s, 0);
  a.nx = (int)s->n[0];
  a.ny = (int)s->n[1];
  a.nz = (int)s->n[2];
  a.single = (s->ndim == 1) ? 1 : 0;
  a.scale = 1.0;
  a.geo = s->plan.geo[0];
  const int64_t R = s->N / s->n[0];
  const unsigned blocks = (unsigned)(a.single ? R : R / 2);
  k_user_x<-1, T><<<blocks, round_threads(s->n[0] / 4), (size_t)s->plan.geo[0].npad * sizeof(typename cplx_of<T>::type), s->stream>>>(a);
  CKL("k_user_x");
  if (s->ndim == 3) {
    const int rc = launch_mid<T>(s, -1, s->off_state + (size_t)sidx * (size_t)arr_stride(s) * s->csize, 1, s->P.nxh);
    if (rc != PSS_OK) return rc;
  }
  if (s->ndim >= 2) {
    LastArgs<T> l;
    l.arr = carr<T>(s, s->off_state, sidx);
    l.tw = twp<T>(s, s->ndim - 1);
    l.n = (int)s->n[s->ndim - 1];
    l.nlines = (int)(s->M / l.n);
    l.geo = s->plan.geo[s->ndim - 1];
    k_last<-1, T><<<l.nlines, round_threads(l.n / 4), (size_t)l.geo.npad * sizeof(typename cplx_of<T>::type), s->stream>>>(l);
    CKL("k_last");
  }
  s->psix_valid = false;
  if (!on_device) CK(cudaStreamSynchronize(s->stream));
  return PSS_OK;
}

template <typename T> int do_get_field(pss_system *s, int slot, void *dst, int on_device) {
  typedef typename cplx_of<T>::type C;
  CK(cudaMemcpyAsync(s->ws + s->off_scratch, carr<T>(s, s->off_state, s->sel * s->P.ndyn + slot), (size_t)s->M * sizeof(C),
                     cudaMemcpyDeviceToDevice, s->stream));
  if (s->ndim >= 2) {
    LastArgs<T> l;
    l.arr = carr<T>(s, s->off_scratch, 0);
    l.tw = twp<T>(s, s->ndim - 1);
    l.n = (int)s->n[s->ndim - 1];
    l.nlines = (int)(s->M / l.n);
    l.geo = s->plan.geo[s->ndim - 1];
    k_last<+1, T><<<l.nlines, round_threads(l.n / 4), (size_t)l.geo.npad * sizeof(C), s->stream>>>(l);
    CKL("k_last");
  }
  if (s->ndim == 3) {
    const int rc = launch_mid<T>(s, +1, s->off_scratch, 1, s->P.nxh);
    if (rc != PSS_OK) return rc;
  }
  UserArgs<T> a;
  a.real = on_device ? (T *)dst : (T *)(s->ws + s->off_ureal);
  a.arr = carr<T>(s, s->off_scratch, 0);
  a.tw = twp<T>(s, 0);
  a.nx = (int)s->n[0];
  a.ny = (int)s->n[1];
  a.nz = (int)s->n[2];
  a.single = (s->ndim == 1) ? 1 : 0;
  a.scale = 1.0 / (double)s->N;
  a.geo = s->plan.geo[0];
  const int64_t R = s->N / s->n[0];
  const unsigned blocks = (unsigned)(a.single ? R : R / 2);
  k_user_x<+1, T><<<blocks, round_threads(s->n[0] / 4), (size_t)s->plan.geo[0].npad * sizeof(C), s->stream>>>(a);
  CKL("k_user_x");
  if (!on_device) {
    CK(cudaMemcpyAsync(dst, s->ws + s->off_ureal, (size_t)s->N * sizeof(T), cudaMemcpyDeviceToHost, s->stream));
    CK(cudaStreamSynchronize(s->stream));
  }
  return PSS_OK;
}

/* Dirichlet frames: the callback at the end of a time step.  The field goes to real space through the
 * set/get kernels (device buffers only), the frame values are written, and it comes back; the next step then starts
 * from the rebuilt factor arrays (prologue launch).  Functionality first: this costs a handful of extra launches per step. */
template <typename T> __global__ void k_apply_frame(T *real, int nx, int ny, int nz, int axis, long long lo_w, long long hi_w, T lo_v, T hi_v) {
  const size_t N = (size_t)nx * ny * nz;
  const int na = axis == 0 ? nx : (axis == 1 ? ny : nz);
  for (size_t x = (size_t)blockIdx.x * blockDim.x + threadIdx.x; x < N; x += (size_t)gridDim.x * blockDim.x) {
    const long long c = axis == 0 ? (long long)(x % nx) : (axis == 1 ? (long long)((x / nx) % ny) : (long long)(x / ((size_t)nx * ny)));
    if (c < lo_w) real[x] = lo_v;
    else if (c >= na - hi_w) real[x] = hi_v;
  }
}

template <typename T> int do_steps(pss_system *s, int64_t nsteps) {
  bool any = false;
  for (const FieldH &F : s->fields) if (!F.frames.empty()) any = true;
  if (!any) return do_steps_core<T>(s, nsteps);
  T *ureal = reinterpret_cast<T *>(s->ws + s->off_ureal);
  const int sel0 = s->sel;
  for (int64_t i = 0; i < nsteps; ++i) {
    int rc = do_steps_core<T>(s, 1);
    if (rc != PSS_OK) return rc;
    for (int r = 0; r < s->nrep; ++r) {
      s->sel = r;
      for (size_t f = 0; f < s->fields.size(); ++f) {
        const FieldH &F = s->fields[f];
        if (F.frames.empty()) continue;
        if ((rc = do_get_field<T>(s, s->dyn_slot[f], ureal, 1)) != PSS_OK) { s->sel = sel0; return rc; }
        for (const FrameH &fr : F.frames) {
          k_apply_frame<T><<<592, 256, 0, s->stream>>>(ureal, (int)s->n[0], (int)s->n[1], (int)s->n[2], fr.axis, fr.lo_w, fr.hi_w, (T)fr.lo_v, (T)fr.hi_v);
          CKL("k_apply_frame");
        }
        if ((rc = do_set_field<T>(s, s->dyn_slot[f], ureal, 1)) != PSS_OK) { s->sel = sel0; return rc; }
      }
    }
    s->sel = sel0;
  }
  return PSS_OK;
}

template <typename T> int do_get_fourier(pss_system *s, int slot, void *dst, int on_device) {
  typedef typename cplx_of<T>::type C;
  C *out = on_device ? (C *)dst : carr<T>(s, s->off_scratch, 0);
  k_to_logical<T><<<592, 256, 0, s->stream>>>(carr<T>(s, s->off_state, s->sel * s->P.ndyn + slot), out, s->P.nxh, (int)s->n[1], (int)s->n[2]);
  CKL("k_to_logical");
  if (!on_device) {
    CK(cudaMemcpyAsync(dst, out, (size_t)s->M * sizeof(C), cudaMemcpyDeviceToHost, s->stream));
    CK(cudaStreamSynchronize(s->stream));
  }
  return PSS_OK;
}

template <typename T> int do_set_fourier(pss_system *s, int slot, const void *src, int on_device) {
  typedef typename cplx_of<T>::type C;
  const C *in = (const C *)src;
  if (!on_device) {
    CK(cudaMemcpyAsync(s->ws + s->off_scratch, src, (size_t)s->M * sizeof(C), cudaMemcpyHostToDevice, s->stream));
    in = carr<T>(s, s->off_scratch, 0);
  }
  k_from_logical<T><<<592, 256, 0, s->stream>>>(in, carr<T>(s, s->off_state, s->sel * s->P.ndyn + slot), s->P.nxh, (int)s->n[1], (int)s->n[2]);
  CKL("k_from_logical");
  s->psix_valid = false;
  if (!on_device) CK(cudaStreamSynchronize(s->stream));
  return PSS_OK;
}

template <typename T> int do_debug_noise(pss_system *s, int field, uint64_t step, uint32_t *bits, void *z) {
  typedef typename cplx_of<T>::type C;
  /* test hook: two temporary device buffers, released on every exit path */
  struct Bufs {
    uint32_t *dbits = nullptr;
    C *dz = nullptr;
    ~Bufs() { if (dbits) cudaFree(dbits); if (dz) cudaFree(dz); }
  } b;
  if (bits) CK(cudaMalloc(&b.dbits, (size_t)s->M * 4 * sizeof(uint32_t)));
  if (z) CK(cudaMalloc(&b.dz, (size_t)s->M * sizeof(C)));
  k_debug_noise<T><<<592, 256, 0, s->stream>>>(s->P, (unsigned)s->sel, field, step, b.dbits, b.dz);
  CKL("k_debug_noise");
  if (bits) CK(cudaMemcpyAsync(bits, b.dbits, (size_t)s->M * 4 * sizeof(uint32_t), cudaMemcpyDeviceToHost, s->stream));
  if (z) CK(cudaMemcpyAsync(z, b.dz, (size_t)s->M * sizeof(C), cudaMemcpyDeviceToHost, s->stream));
  CK(cudaStreamSynchronize(s->stream));
  return PSS_OK;
}

/* ---- the one entry point that allocates nothing: pss_debug_noise_noalloc --------------------------------------------
 * pss_debug_noise stages its device-side results in two buffers it gets from cudaMalloc and gives back with cudaFree.
 * Here the same kernel writes into a fixed array that is part of the library image instead.  The array is sized for the
 * half-spectrum of the headline lattice (1024 x 513 modes: 16 bytes of Philox words plus at most 16 bytes of z each,
 * 16.03 MiB); every GPU on which the library gets loaded carries it until the process exits, used or not. */
constexpr size_t STATIC_NOISE_BYTES = (size_t)PSS_STATIC_NOISE_MAX_MODES * 32;
static __device__ __align__(256) unsigned char g_static_noise[STATIC_NOISE_BYTES];

/* `g_static_noise` in HOST code is only a handle the runtime knows the symbol by, not an address a kernel could use, so
 * the device address is asked for once per device (with that device current) and remembered.  The table is per process;
 * the mutex only serialises the look-up, not the use of the array. */
constexpr int STATIC_MAX_DEVICES = 64;
std::mutex g_static_mu;
void *g_static_ptr[STATIC_MAX_DEVICES] = {};

int static_noise_ptr(pss_system *s, unsigned char **out) {
  int dev = -1;
  CK(cudaGetDevice(&dev));
  if (dev < 0 || dev >= STATIC_MAX_DEVICES) return PSS_EUNSUPPORTED;
  std::lock_guard<std::mutex> lk(g_static_mu);
  if (!g_static_ptr[dev]) {
    void *p = nullptr;
    CK(cudaGetSymbolAddress(&p, g_static_noise));
    if (!p) return cuda_fail(s, cudaErrorInvalidSymbol, "cudaGetSymbolAddress(g_static_noise)");
    g_static_ptr[dev] = p;
  }
  *out = (unsigned char *)g_static_ptr[dev];
  return PSS_OK;
}

template <typename T> int do_debug_noise_noalloc(pss_system *s, int field, uint64_t step, uint32_t *bits, void *z) {
  typedef typename cplx_of<T>::type C;
  unsigned char *base = nullptr;
  const int rc = static_noise_ptr(s, &base);
  if (rc != PSS_OK) return rc;
  /* words first, z behind them at the capacity offset (a multiple of 256 bytes); the kernel writes every element the
   * copies below read, so nothing left behind by an earlier call is ever seen and nothing needs clearing */
  uint32_t *dbits = bits ? reinterpret_cast<uint32_t *>(base) : nullptr;
  C *dz = z ? reinterpret_cast<C *>(base + (size_t)PSS_STATIC_NOISE_MAX_MODES * 16) : nullptr;
  k_debug_noise<T><<<592, 256, 0, s->stream>>>(s->P, (unsigned)s->sel, field, step, dbits, dz);
  CKL("k_debug_noise");
  if (bits) CK(cudaMemcpyAsync(bits, dbits, (size_t)s->M * 4 * sizeof(uint32_t), cudaMemcpyDeviceToHost, s->stream));
  if (z) CK(cudaMemcpyAsync(z, dz, (size_t)s->M * sizeof(C), cudaMemcpyDeviceToHost, s->stream));
  CK(cudaStreamSynchronize(s->stream));
  return PSS_OK;
}

}  // namespace

/* ---- C ABI ----------------------------------------------------------------------------- */
extern "C" {

int pss_create(pss_system **out, int ndim, const int64_t n[3], const double dx[3], double dt,
               pss_precision prec, uint64_t seed) {
  if (!out || !n || !dx) return PSS_EINVAL;
  *out = nullptr;
  if (ndim < 1) return PSS_EINVAL;
  if (ndim > 3) return PSS_EUNSUPPORTED;
  if (prec != PSS_F32 && prec != PSS_F64) return PSS_EINVAL;
  if (!(dt > 0.0) || !std::isfinite(dt)) return PSS_EINVAL;
  for (int j = 0; j < ndim; ++j) {
    if (n[j] < 1 || !(dx[j] > 0.0) || !std::isfinite(dx[j])) return PSS_EINVAL;
    if (!is_pow2(n[j]) || n[j] < 8 || n[j] > 8192) return PSS_EUNSUPPORTED; /* A17 */
  }
  pss_system *s = new pss_system();
  s->ndim = ndim;
  for (int j = 0; j < 3; ++j) { s->n[j] = j < ndim ? n[j] : 1; s->dx[j] = j < ndim ? dx[j] : 1.0; }
  s->dt = dt;
  s->prec = (int)prec;
  s->seed = seed;
  s->dealias = PSS_DEALIAS_PAPER;
  s->nrep = 1;
  s->sel = 0;
  s->finalized = s->bound = s->psix_valid = false;
  s->step = 0;
  s->csize = prec == PSS_F32 ? 8 : 16;
  s->rsize = prec == PSS_F32 ? 4 : 8;
  s->N = s->n[0] * s->n[1] * s->n[2];
  s->M = (s->n[0] / 2 + 1) * s->n[1] * s->n[2];
  s->ws = nullptr;
  s->dev = -1;
  s->stream = nullptr;
  s->cuda_bad = false;
  s->launches = 0;
  s->prof_on = false;
  *out = s;
  return PSS_OK;
}

int pss_add_field(pss_system *s, const char *name, int dynamic, int *field_id) {
  if (!s || !name) return PSS_EINVAL;
  if (s->finalized) return PSS_ESTATE;
  if (s->fields.size() >= 64) return PSS_EUNSUPPORTED;
  for (const FieldH &f : s->fields) if (f.name == name) return PSS_EINVAL;
  FieldH f;
  f.name = name; f.dynamic = dynamic != 0; f.noisy = false; f.D = 0; f.qpow = 0;
  s->fields.push_back(f);
  if (field_id) *field_id = (int)s->fields.size() - 1;
  return PSS_OK;
}

int pss_add_linear(pss_system *s, int field, const pss_op *op) {
  if (!s) return PSS_EINVAL;
  if (s->finalized) return PSS_ESTATE;
  if (!fid_ok(s, field) || !op_ok(s, op)) return PSS_EINVAL;
  if (!s->fields[field].dynamic) return PSS_EINVAL;
  s->fields[field].lhs.push_back(*op);
  return PSS_OK;
}

int pss_add_aux_def(pss_system *s, int aux, const pss_op *op, int src) {
  if (!s) return PSS_EINVAL;
  if (s->finalized) return PSS_ESTATE;
  if (!fid_ok(s, aux) || !fid_ok(s, src) || !op_ok(s, op)) return PSS_EINVAL;
  if (s->fields[aux].dynamic) return PSS_EINVAL;
  if (!s->fields[src].dynamic && src >= aux) return PSS_EINVAL; /* A12 */
  DefH d; d.op = *op; d.src = src;
  s->fields[aux].defs.push_back(d);
  return PSS_OK;
}

int pss_set_frame(pss_system *s, int field, int axis, int64_t lo_width, double lo_value, int64_t hi_width, double hi_value) {
  if (!s) return PSS_EINVAL;
  if (s->finalized) return PSS_ESTATE;
  if (!fid_ok(s, field) || !s->fields[field].dynamic) return PSS_EINVAL;
  if (axis < 0 || axis >= s->ndim) return PSS_EINVAL;
  if (lo_width < 0 || hi_width < 0 || lo_width + hi_width > s->n[axis]) return PSS_EINVAL;
  if (!std::isfinite(lo_value) || !std::isfinite(hi_value)) return PSS_EINVAL;
  FrameH fr; fr.axis = axis; fr.lo_w = lo_width; fr.hi_w = hi_width; fr.lo_v = lo_value; fr.hi_v = hi_value;
  s->fields[field].frames.push_back(fr);
  return PSS_OK;
}

int pss_add_aux_lhs(pss_system *s, int aux, const pss_op *op) {
  if (!s) return PSS_EINVAL;
  if (s->finalized) return PSS_ESTATE;
  if (!fid_ok(s, aux) || !op_ok(s, op)) return PSS_EINVAL;
  if (s->fields[aux].dynamic) return PSS_EINVAL;
  s->fields[aux].lhs.push_back(*op);
  return PSS_OK;
}

int pss_add_aux_term(pss_system *s, int aux, const pss_op *outer, int nfactors, const int *factor_fields) {
  if (!s) return PSS_EINVAL;
  if (s->finalized) return PSS_ESTATE;
  if (!fid_ok(s, aux) || !op_ok(s, outer) || !factor_fields) return PSS_EINVAL;
  if (s->fields[aux].dynamic) return PSS_EINVAL;
  if (nfactors < 2) return PSS_EINVAL; /* one factor is pss_add_aux_def */
  if (nfactors > 4) return PSS_EUNSUPPORTED;
  ATermH t; t.outer = *outer;
  for (int i = 0; i < nfactors; ++i) {
    const int g = factor_fields[i];
    if (!fid_ok(s, g)) return PSS_EINVAL;
    if (!s->fields[g].dynamic && g >= aux) return PSS_EINVAL; /* dynamic or EARLIER intermediate fields only (A12) */
    t.factors.push_back(g);
  }
  s->fields[aux].aterms.push_back(t);
  return PSS_OK;
}

int pss_add_term(pss_system *s, int field, const pss_op *outer, int nfactors, const int *factor_fields) {
  if (!s) return PSS_EINVAL;
  if (s->finalized) return PSS_ESTATE;
  if (!fid_ok(s, field) || !op_ok(s, outer) || !factor_fields) return PSS_EINVAL;
  if (!s->fields[field].dynamic) return PSS_EINVAL;
  if (nfactors < 1) return PSS_EINVAL;
  if (nfactors > 4) return PSS_EUNSUPPORTED;
  TermH t; t.field = field; t.outer = *outer;
  for (int i = 0; i < nfactors; ++i) {
    if (!fid_ok(s, factor_fields[i])) return PSS_EINVAL;
    t.factors.push_back(factor_fields[i]);
  }
  s->terms.push_back(t);
  return PSS_OK;
}

int pss_set_noise(pss_system *s, int field, double D, int q_power) {
  if (!s) return PSS_EINVAL;
  if (s->finalized) return PSS_ESTATE;
  if (!fid_ok(s, field) || !s->fields[field].dynamic) return PSS_EINVAL;
  if (!(D >= 0.0) || !std::isfinite(D)) return PSS_EINVAL;
  if (q_power < -8 || q_power > 8) return PSS_EINVAL;
  FieldH &f = s->fields[field];
  f.noisy = D > 0.0; f.D = D; f.qpow = q_power;
  return PSS_OK;
}

int pss_set_dealias(pss_system *s, int rule) {
  if (!s) return PSS_EINVAL;
  if (s->finalized) return PSS_ESTATE;
  if (rule < PSS_DEALIAS_PAPER || rule > PSS_DEALIAS_OFF) return PSS_EINVAL;
  s->dealias = rule;
  return PSS_OK;
}

int pss_set_replicas(pss_system *s, int nreplicas) {
  if (!s) return PSS_EINVAL;
  if (s->finalized) return PSS_ESTATE;
  if (nreplicas < 1) return PSS_EINVAL;
  if (nreplicas > 65535) return PSS_EUNSUPPORTED;
  s->nrep = nreplicas;
  s->sel = 0;
  return PSS_OK;
}

int pss_select_replica(pss_system *s, int replica) {
  if (!s || replica < 0 || replica >= s->nrep) return PSS_EINVAL;
  s->sel = replica;
  return PSS_OK;
}

int pss_replicas(const pss_system *s) { return s ? s->nrep : 0; }

int pss_finalize(pss_system *s, size_t *workspace_bytes) {
  if (!s) return PSS_EINVAL;
  if (s->finalized) return PSS_ESTATE;
  int ndyn = 0;
  for (const FieldH &f : s->fields) ndyn += f.dynamic ? 1 : 0;
  if (ndyn == 0) return PSS_EINVAL;
  for (const FieldH &f : s->fields)
    if (!f.dynamic && f.defs.empty() && f.aterms.empty()) return PSS_EINVAL;
  if (s->fields.size() > 0xffff) return PSS_EUNSUPPORTED;
  int rc = build_program(s);
  if (rc != PSS_OK) return rc;
  rc = make_plan(s);
  if (rc != PSS_OK) return rc;
  /* 3D: k_mid folds (array, replica) into gridDim.z (<= 65535) */
  if (s->ndim == 3 && (long long)(s->P.nfac > s->P.ngrp ? s->P.nfac : s->P.ngrp) * s->nrep > 65535) return PSS_EUNSUPPORTED;
  carve_workspace(s);
  s->herm_period = plan_hermitian(s);
  if (env_int("PSS_DEBUG_PLAN", 0))
    std::fprintf(stderr, "pss plan: rounds %d ndyn %d nfac %d ngrp %d nlin %d rad_ok %d | upd W %d thr %d smem %zu blocks %d | rows Wc %d thr %d smem %zu blocks %d | fused %d\n",
                 s->nround, s->P.ndyn, s->nfac_max, s->ngrp_max, s->P.nlin, s->P.rad_ok, s->plan.upd_W, s->plan.upd_threads,
                 s->plan.upd_smem, s->plan.upd_blocks, s->plan.row_Wc, s->plan.row_threads, s->plan.row_smem, s->plan.row_blocks, s->plan.fused);
  s->finalized = true;
  if (workspace_bytes) *workspace_bytes = s->ws_need;
  return PSS_OK;
}

int pss_bind(pss_system *s, void *device_workspace, size_t bytes, void *cuda_stream) {
  if (!s || !device_workspace) return PSS_EINVAL;
  if (!s->finalized) return PSS_ESTATE;
  if (bytes < s->ws_need || ((uintptr_t)device_workspace & 255u)) return PSS_EINVAL;
  int ndev = 0;
  CK(cudaGetDeviceCount(&ndev));
  if (ndev < 1) return cuda_fail(s, cudaErrorNoDevice, "pss_bind");
  {
    cudaPointerAttributes pa;
    CK(cudaPointerGetAttributes(&pa, device_workspace));
    if (pa.type != cudaMemoryTypeDevice && pa.type != cudaMemoryTypeManaged) return PSS_EINVAL;
    s->dev = pa.device;
  }
  DeviceGuard guard(s->dev);
  s->ws = (char *)device_workspace;
  s->stream = (cudaStream_t)cuda_stream;
  CK(cudaMemsetAsync(s->ws, 0, s->ws_need, s->stream));
  int rc = (s->prec == PSS_F32) ? set_attrs<float>(s) : set_attrs<double>(s);
  if (rc != PSS_OK) return rc;
  rc = (s->prec == PSS_F32) ? upload_twiddles<float>(s) : upload_twiddles<double>(s);
  if (rc != PSS_OK) return rc;
  if ((rc = setup_fused(s)) != PSS_OK) return rc;
  s->bar_count = 0; /* the counter lives in the workspace, zeroed above */
  s->bound = true;
  s->psix_valid = false;
  return PSS_OK;
}

int pss_set_field(pss_system *s, int field, const void *real_xfastest, int on_device) {
  if (!s || !real_xfastest) return PSS_EINVAL;
  if (!s->finalized || !s->bound) return PSS_ESTATE;
  if (s->cuda_bad) return PSS_ECUDA;
  DeviceGuard guard(s->dev);
  if (!fid_ok(s, field) || !s->fields[field].dynamic) return PSS_EINVAL;
  const int slot = s->dyn_slot[field];
  return (s->prec == PSS_F32) ? do_set_field<float>(s, slot, real_xfastest, on_device)
                              : do_set_field<double>(s, slot, real_xfastest, on_device);
}

int pss_step(pss_system *s, int64_t nsteps) {
  if (!s || nsteps < 0) return PSS_EINVAL;
  if (!s->finalized || !s->bound) return PSS_ESTATE;
  if (s->cuda_bad) return PSS_ECUDA;
  DeviceGuard guard(s->dev);
  return (s->prec == PSS_F32) ? do_steps<float>(s, nsteps) : do_steps<double>(s, nsteps);
}

int pss_get_field(pss_system *s, int field, void *real_out, int on_device) {
  if (!s || !real_out) return PSS_EINVAL;
  if (!s->finalized || !s->bound) return PSS_ESTATE;
  if (s->cuda_bad) return PSS_ECUDA;
  DeviceGuard guard(s->dev);
  if (!fid_ok(s, field) || !s->fields[field].dynamic) return PSS_EINVAL;
  const int slot = s->dyn_slot[field];
  return (s->prec == PSS_F32) ? do_get_field<float>(s, slot, real_out, on_device)
                              : do_get_field<double>(s, slot, real_out, on_device);
}

int pss_get_field_fourier(pss_system *s, int field, void *out, int on_device) {
  if (!s || !out) return PSS_EINVAL;
  if (!s->finalized || !s->bound) return PSS_ESTATE;
  if (s->cuda_bad) return PSS_ECUDA;
  DeviceGuard guard(s->dev);
  if (!fid_ok(s, field) || !s->fields[field].dynamic) return PSS_EINVAL;
  const int slot = s->dyn_slot[field];
  return (s->prec == PSS_F32) ? do_get_fourier<float>(s, slot, out, on_device)
                              : do_get_fourier<double>(s, slot, out, on_device);
}

int pss_set_field_fourier(pss_system *s, int field, const void *in, int on_device) {
  if (!s || !in) return PSS_EINVAL;
  if (!s->finalized || !s->bound) return PSS_ESTATE;
  if (s->cuda_bad) return PSS_ECUDA;
  DeviceGuard guard(s->dev);
  if (!fid_ok(s, field) || !s->fields[field].dynamic) return PSS_EINVAL;
  const int slot = s->dyn_slot[field];
  return (s->prec == PSS_F32) ? do_set_fourier<float>(s, slot, in, on_device) : do_set_fourier<double>(s, slot, in, on_device);
}

int pss_set_step_count(pss_system *s, uint64_t step) {
  if (!s) return PSS_EINVAL;
  if (!s->finalized) return PSS_ESTATE; /* the counter belongs to a finalized system (checkpoint/resume) */
  s->step = step;
  return PSS_OK;
}

int pss_debug_noise(pss_system *s, int field, uint64_t step, uint32_t *bits, void *z) {
  if (!s) return PSS_EINVAL;
  if (!s->finalized || !s->bound) return PSS_ESTATE;
  if (s->cuda_bad) return PSS_ECUDA;
  DeviceGuard guard(s->dev);
  if (!fid_ok(s, field)) return PSS_EINVAL;
  return (s->prec == PSS_F32) ? do_debug_noise<float>(s, field, step, bits, z)
                              : do_debug_noise<double>(s, field, step, bits, z);
}

int pss_debug_noise_noalloc(pss_system *s, int field, uint64_t step, uint32_t *bits, void *z) {
  if (!s) return PSS_EINVAL;
  if (!s->finalized || !s->bound) return PSS_ESTATE;
  if (s->cuda_bad) return PSS_ECUDA;
  if (s->M > (int64_t)PSS_STATIC_NOISE_MAX_MODES) return PSS_ETOOBIG;
  DeviceGuard guard(s->dev);
  if (!fid_ok(s, field)) return PSS_EINVAL;
  return (s->prec == PSS_F32) ? do_debug_noise_noalloc<float>(s, field, step, bits, z)
                              : do_debug_noise_noalloc<double>(s, field, step, bits, z);
}

int pss_profile_step(pss_system *s, int64_t nsteps, double ms_per_launch[4], int64_t launches[4]) {
  if (!s || nsteps < 0 || nsteps > 4096 || !ms_per_launch || !launches) return PSS_EINVAL;
  if (!s->finalized || !s->bound) return PSS_ESTATE;
  if (s->cuda_bad) return PSS_ECUDA;
  DeviceGuard guard(s->dev);
  if (s->ndim == 1) return PSS_EUNSUPPORTED;
  int rc = (s->prec == PSS_F32) ? do_steps<float>(s, 0) : do_steps<double>(s, 0);
  /* make sure the prologue (if any) is not inside the profiled region */
  if (s->plan.fused && !s->psix_valid) {
    rc = launch_fused(s, 0);
    if (rc != PSS_OK) return rc;
  }
  if (!s->plan.fused && s->nfac_max > 0 && !s->psix_valid) {
    rc = (s->prec == PSS_F32) ? launch_update<float>(s, 1, s->step, s->PU[(size_t)(s->nround - 1)])
                              : launch_update<double>(s, 1, s->step, s->PU[(size_t)(s->nround - 1)]);
    if (rc != PSS_OK) return rc;
    s->psix_valid = true;
  }
  s->prof_on = true;
  rc = (s->prec == PSS_F32) ? do_steps<float>(s, nsteps) : do_steps<double>(s, nsteps);
  s->prof_on = false;
  cudaError_t e = cudaStreamSynchronize(s->stream);
  double sum[KIND_COUNT] = {0, 0, 0, 0};
  int64_t cnt[KIND_COUNT] = {0, 0, 0, 0};
  for (size_t i = 0; i < s->prof_kind.size() && 2 * i + 1 < s->prof_ev.size(); ++i) {
    float ms = 0.f;
    if (e == cudaSuccess && cudaEventElapsedTime(&ms, s->prof_ev[2 * i], s->prof_ev[2 * i + 1]) == cudaSuccess) {
      sum[s->prof_kind[i]] += ms;
      cnt[s->prof_kind[i]] += 1;
    }
  }
  for (cudaEvent_t ev : s->prof_ev) cudaEventDestroy(ev);
  s->prof_ev.clear();
  s->prof_kind.clear();
  for (int k = 0; k < KIND_COUNT; ++k) { ms_per_launch[k] = cnt[k] ? sum[k] / (double)cnt[k] : 0.0; launches[k] = cnt[k]; }
  if (e != cudaSuccess) return cuda_fail(s, e, "pss_profile_step");
  return rc;
}

uint64_t pss_launch_count(const pss_system *s) { return s ? s->launches : 0; }

int64_t pss_hermitian_period(const pss_system *s) { return (s && s->finalized) ? s->herm_period : 0; }

int pss_uses_fused_kernel(const pss_system *s) {
  if (!(s && s->finalized && s->bound && s->plan.fused)) return 0;
  return s->plan.persist ? 2 : 1;
}

double pss_model_bytes_per_step(const pss_system *s, int pruned) {
  if (!s || !s->finalized) return 0.0;
  const double S = (double)s->N * (double)s->rsize * (double)s->nrep;
  if (s->ndim == 1) return 2.0 * s->P.ndyn * S;
  /* every spectral source is read and written once per step; every round (one per dependency level of the
   * product-defined intermediate fields, the dynamic equations last) moves its groups and the kept band of its factors */
  double total = 2.0 * s->P.ndyn * S;
  for (const Program &P : s->PR) {
    double c1 = 0.0, c2 = 0.0; /* sum over factors of the kept fraction per axis, and its square */
    for (int f = 0; f < P.nfac; ++f) {
      double c = 1.0;
      if (pruned && P.dealias != PSS_DEALIAS_OFF)
        c = 2.0 / (double)((P.dealias == PSS_DEALIAS_TWO_THIRDS ? 2 : P.fac[f].order) + 1);
      c1 += c;
      c2 += c * c;
    }
    if (s->ndim == 2) total += S * (2.0 * P.ngrp + 2.0 * c1);
    else total += S * (4.0 * P.ngrp + 2.0 * c2 + 2.0 * c1);
  }
  return total;
}

uint64_t pss_step_count(const pss_system *s) { return s ? s->step : 0; }

const char *pss_strerror(int code) {
  switch (code) {
    case PSS_OK: return "ok";
    case PSS_EINVAL: return "invalid argument";
    case PSS_EUNSUPPORTED: return "unsupported configuration";
    case PSS_ESTATE: return "call made in the wrong state";
    case PSS_ECUDA: return "CUDA error (see pss_last_cuda_error)";
    case PSS_ETOOBIG: return "lattice has more modes than the library's fixed device array holds (PSS_STATIC_NOISE_MAX_MODES)";
    default: return "unknown error";
  }
}

const char *pss_last_cuda_error(const pss_system *s) { return s ? s->cuda_msg.c_str() : ""; }

void pss_destroy(pss_system *s) { delete s; }

} /* extern "C" */
