/*
 * opss.h — C ABI of the CPU ORACLE for the semi-implicit pseudo-spectral SPDE step.
 *
 * TEST INFRASTRUCTURE ONLY.  This is the slow, plain, obviously-correct CPU restatement of
 * the method of cuPSS (arXiv 2405.02410), written from PAPER.md alone.  Only tests/,
 * __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may load it.
 * It shares no code, header, table or helper with the CUDA product under
 * paper_2405_02410_b200/ and include/pss.h; the two never import each other.
 *
 * The entry points mirror include/pss.h one to one (prefix opss_ instead of pss_) so that a
 * single test driver can feed both sides the same term list.  Every pointer is a HOST pointer.
 *
 * What it computes (citations are PAPER.md line numbers):
 *   d phi = F[phi] dt + sqrt(2D) dW                     (Eq. 1,  PAPER.md:13)
 *   field system  dt phi_i = L_i phi_i + sum_j N_ij + noise (Eq. 10-11)
 *   pseudo-spectral products with de-aliased factor copies (Eq. 6-9, 15)
 *   the six-step time-step list and Eq. 18
 *
 * Pins: see tests/test_oracle_*.py ("-m 'not gpu'").  The nematic workload (config 4) has no
 * equations in the paper: beyond the invariants P12 of DESIGN.md it is "parity unpinned".
 */
#ifndef OPSS_H
#define OPSS_H
#include <stddef.h>
#include <stdint.h>
#ifdef __cplusplus
extern "C" {
#endif

typedef struct opss_system opss_system;

enum { OPSS_F32 = 0, OPSS_F64 = 1 };
enum { OPSS_DEALIAS_PAPER = 0, OPSS_DEALIAS_TWO_THIRDS = 1, OPSS_DEALIAS_OFF = 2 };
enum { OPSS_OK = 0, OPSS_EINVAL = -1, OPSS_EUNSUPPORTED = -2, OPSS_ESTATE = -3 };

/* one operator monomial  coef * (q^2)^q2_pow * (1/|q|)^invq_pow * prod_j (i q_j)^iq_pow[j]
 * (keywords q^2n, 1/q, iqx/iqy/iqz of PAPER.md:186-190) */
typedef struct {
  double coef;
  int q2_pow;
  int invq_pow;
  int iq_pow[3];
} opss_op;

int opss_create(opss_system **out, int ndim, const int64_t n[3], const double dx[3], double dt,
                int prec, uint64_t seed);
int opss_add_field(opss_system *, const char *name, int dynamic, int *field_id);
int opss_add_linear(opss_system *, int field, const opss_op *op);
int opss_add_aux_def(opss_system *, int aux, const opss_op *op, int src);
/* Dirichlet frame (Fig. 2): at the end of every time step the field is set, in real space, to
 * lo_value where x_axis < lo_width and to hi_value where x_axis >= n_axis - hi_width.  Dynamic fields, before finalize. */
int opss_set_frame(opss_system *, int field, int axis, int64_t lo_width, double lo_value, int64_t hi_width, double hi_value);
/* intermediate field with its own lhs: (sum of the ops added here)(q) * psi_q = rhs_q; psi_q = 0 where
 * the sum vanishes.  None added = the bare field. */
int opss_add_aux_lhs(opss_system *, int aux, const opss_op *op);
/* rhs term of an intermediate field that is a product of >= 2 fields: psi_q += outer(q) F[prod](q);
 * factors: dynamic fields or intermediate fields created earlier. */
int opss_add_aux_term(opss_system *, int aux, const opss_op *outer, int nfactors, const int *factor_fields);
int opss_add_term(opss_system *, int field, const opss_op *outer, int nfactors,
                  const int *factor_fields);
int opss_set_noise(opss_system *, int field, double D, int q_power);
int opss_set_dealias(opss_system *, int rule);
int opss_finalize(opss_system *, size_t *workspace_bytes);
int opss_set_field(opss_system *, int field, const void *real_xfastest);
int opss_set_threads(opss_system *, int nthreads); /* OpenMP threads over independent lines; 0 = all */
int opss_step(opss_system *, int64_t nsteps);
int opss_get_field(opss_system *, int field, void *real_out);
/* half-spectrum, kx = 0..Nx/2 fastest, then ky, then kz; complex of the system precision */
int opss_get_field_fourier(opss_system *, int field, void *halfspectrum_out);
/* always complex double, regardless of precision (for pins that need the unrounded state) */
int opss_get_field_fourier_f64(opss_system *, int field, double *halfspectrum_out);
/* noise test hook: bits = 4 words per logical mode m; z = unit Hermitian Gaussian field,
 * complex double per mode.  Either pointer may be NULL. */
int opss_debug_noise(opss_system *, int field, uint64_t step, uint32_t *bits4_per_mode,
                     double *z_halfspectrum);
uint64_t opss_step_count(const opss_system *);
const char *opss_strerror(int code);
void opss_destroy(opss_system *);

/* ---- hooks that expose the oracle's own building blocks so the pins can reach them ---- */
/* complex DFT of `howmany` contiguous lines of length n (interleaved re,im doubles), in place.
 * sign = -1 forward (unnormalised), +1 inverse (unnormalised, caller divides). */
int opss_debug_fft_lines(double *data, int64_t n, int64_t howmany, int sign);
/* full R2C / C2R of the oracle (C2R carries 1/N); n[] padded with 1 beyond ndim */
int opss_debug_r2c(const double *real_in, double *half_out, int ndim, const int64_t n[3]);
int opss_debug_c2r(const double *half_in, double *real_out, int ndim, const int64_t n[3]);
/* value of one operator monomial at integer mode k (out = re, im) */
int opss_debug_op(const opss_system *, const opss_op *op, const int64_t k[3], double out[2]);
/* de-alias keep mask (1 keep / 0 zero) of field `field` over the half-spectrum; returns 1 (and writes nothing)
 * if the field is not a factor of any product */
int opss_debug_mask(opss_system *, int field, uint8_t *mask_halfspectrum);
/* one Philox4x32-10 block */
void opss_debug_philox(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]);

#ifdef __cplusplus
}
#endif
#endif
