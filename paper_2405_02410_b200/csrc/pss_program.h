/*
 * pss_program.h — the frozen term list of one field system, as plain data handed to the kernels
 * by value (a __grid_constant__ kernel parameter, < 4 KB).
 *
 * It restates PAPER.md:82-90 (Eq. 10-11): dynamic fields phi_i with an implicit operator L_i,
 * intermediate fields psi_k that are operators applied to fields, and rhs terms
 * M_ij prod_k psi_k^{n_k}.  Intermediate fields that are linear in the dynamic fields (all of
 * BASELINE's workloads) are flattened on the host into sums of operator monomials acting directly on
 * dynamic fields, so that the kernels evaluate them pointwise per mode from registers.
 */
#ifndef PSS_PROGRAM_H
#define PSS_PROGRAM_H
#include <stdint.h>

#define PSS_P_MAX_DYN 6 /* spectral sources: dynamic fields + product-defined intermediate fields */
#define PSS_P_MAX_DEN 2
#define PSS_P_MAX_FAC 12
#define PSS_P_MAX_GRP 8
#define PSS_P_MAX_TERM 32
#define PSS_P_MAX_LIN 96

/* coef (q^2)^m |q|^-p prod_j (i q_j)^a[j] / den(q) acting on spectral source `src`.
 * den: 0 = none, i > 0 = denominator i - 1 of Program::den (an intermediate field with its own lhs).
 * zflags bit j (j<3): the monomial is 0 at the Nyquist index of axis j (reading A9, applied link by
 * link before flattening); bit 3: it is 0 at q = 0 (reading A10). */
struct DOp {
  double coef;
  int8_t m, p;
  int8_t a[3];
  uint8_t zflags;
  int8_t src;
  int8_t den;
};

/* one product term of a group: coef * prod_{i<nf} factor[f[i]](x) */
struct DTerm {
  double coef;
  int8_t nf;
  int8_t f[4];
  int8_t pad_[3];
};

/* a field that enters products of order >= 2: its de-aliased copy is transformed */
struct DFactor {
  int16_t lin_beg, lin_end; /* psi_q = sum_{e in [beg,end)} lin[e](q) * phi_{src_e}(q) */
  int16_t order;            /* highest order n of a product it appears in           */
  int16_t pad_;
};

/* all product terms with the same target field and the same outer operator are summed in real
 * space before the forward transform (the transform is linear) */
struct DGroup {
  DOp outer; /* coef = 1, src = target dynamic slot */
  int16_t term_beg, term_end;
  int16_t target;
  int16_t pad_;
};

/* denominator polynomial of an intermediate field's lhs: den(q) = sum_{e in [beg,end)} lin[e](q), real-valued monomials;
 * 1/den is 0 where den vanishes (reading A10) */
struct DDen { int16_t beg, end; };

/* one spectral source (a state array): a dynamic field, or an intermediate field defined by products, which is
 * re-evaluated every step in its own round of the two step kernels */
enum { PSS_SLOT_STEP = 0, PSS_SLOT_ASSIGN = 1, PSS_SLOT_KEEP = 2 };
struct DDyn {
  int16_t kind;             /* this launch: STEP = Eq. 18; ASSIGN = (sum of its groups and linear terms) / den; KEEP = untouched */
  int16_t den;              /* ASSIGN: 0 = none, i > 0 = Program::den[i - 1]                           */
  int16_t lhs_beg, lhs_end; /* L_q = - sum lin[e](q)                  (dt phi + lhs = rhs, A3) */
  int16_t lin_beg, lin_end; /* explicit linear terms sum lin[e](q) phi_src(q)   (A8)          */
  double noise_c;           /* 2 D dt N / dV                           (A1)                   */
  int16_t noise_qpow;       /* a in D~ = D |q|^a                       (A13)                  */
  int16_t noisy;
  int32_t field_id;         /* user field id: enters the Philox counter                       */
};

struct Program {
  int32_t ndim;
  int32_t n[3];
  int32_t nxh;
  int32_t dealias;
  double qs[3]; /* 2 pi / (n_j dx_j) */
  double dt;
  double invN;
  uint32_t seed_lo, seed_hi;
  int32_t ndyn, nfac, ngrp, nterm, nlin;
  int32_t any_invq; /* some monomial uses the 1/q keyword: the kernels then evaluate 1/|q| once per mode */
  int32_t nden;
  DDen den[PSS_P_MAX_DEN];
  DDyn dyn[PSS_P_MAX_DYN];
  DFactor fac[PSS_P_MAX_FAC];
  DGroup grp[PSS_P_MAX_GRP];
  DTerm term[PSS_P_MAX_TERM];
  DOp lin[PSS_P_MAX_LIN];
  /* "radial" fast path (set by the host when it applies): one dynamic field, at most one product group, no
   * explicit linear terms, noise power even and >= 0, and
   *   L(q) = rad_L(q^2), outer(q) = rad_O(q^2)                     polynomials in q^2 (Horner, ascending, degree <= 4)
   *   factor f (q) = rad_F[f](q^2) * prod_j (i q_j)^rad_a[f][j]     a polynomial in q^2 times ONE derivative monomial
   *                                                                  (zero at the Nyquist index of every odd axis, A9)
   *   noise amp = sqrt(noise_c (q^2)^rad_nhp).
   * Model B and diffusion have rad_a = 0; KPZ has the factors i q_x h and i q_y h. */
  int32_t rad_ok; /* 0 no, 1 all rad_a zero, 2 some factor has a derivative monomial */
  int32_t rad_nhp;
  double rad_L[5], rad_O[5];
  double rad_F[PSS_P_MAX_FAC][5];
  int8_t rad_a[PSS_P_MAX_FAC][4]; /* [3] = zflags & 7 of the monomial */
};

/* radix schedule of one in-shared-memory FFT of length n = prod R[i] */
struct Geo {
  int32_t n;
  int32_t nr;
  int32_t lg[4]; /* log2 of the radices, first DIF pass first */
  /* shared-memory padding against bank conflicts: slot p lives at row geo_pad(p) = p + sum_i (p >> sh[i]), one pad
   * row per digit boundary of the slot index (unused entries are 31), so that every digit of the slot index maps to
   * an ODD row stride: the stride-1 legs of the last pass and the digit-reversed accesses of the pointwise stages
   * both spread over the banks.  npad = geo_pad(n-1) + 1 rows are allocated. */
  int32_t sh[3];
  int32_t npad;
  /* digit fields of the reversal: digit q of frequency f sits at bits [fs[q], fs[q]+lg[q]) and moves to slot bits
   * starting at ps[q]; fm[q] is its mask (0 for unused passes) */
  int32_t fs[4], ps[4], fm[4];
  /* per-pass twiddle tables behind the n-entry table tw[j] = exp(-2 pi i j / n): pass q (sub-length L, radix R) finds
   * w_L^(m i) at tw[twoff[q] + (m - 1) * (L / R) + i], m = 1..R-1, i < L/R — consecutive butterflies read consecutive
   * entries (two cache lines per warp load instead of up to 32) */
  int32_t twoff[4];
};

#endif
