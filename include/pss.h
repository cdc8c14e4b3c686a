/*
 * pss.h — C ABI of the B200-native semi-implicit pseudo-spectral SPDE stepper.
 *
 * The library implements ONE thing: the per-timestep hot path of cuPSS (arXiv 2405.02410),
 *     d phi = F[phi] dt + sqrt(2D) dW                                   (Eq. 1,  PAPER.md:13)
 * on periodic 1D/2D/3D lattices, for a system of fields (Eq. 10-11)
 *     dt phi_i = L_i phi_i + sum_j M_ij prod_k psi_k^{n_k} + noise,
 * advanced with the semi-implicit update (Eq. 18)
 *     phi_q <- (phi_q + dt N_q + nu_q) / (1 - dt L_q)
 * following the six-step list of PAPER.md:128-135.  Every step of the path runs in hand-written
 * sm_100a CUDA kernels; there is no CPU fallback: a call made without a usable CUDA device returns
 * PSS_ECUDA.
 *
 * Conventions:
 *   - axis 0 is x (fastest in user memory), then y, then z.  n[j], dx[j] for j >= ndim are ignored.
 *   - q_j = 2 pi s(k_j) / (n_j dx_j), s(k) = k for k <= n/2 else k - n
 *   - forward DFT unnormalised, inverse carries 1/N, N = prod n_j.
 *   - user real data: element type = precision of the system, x fastest.
 *   - half-spectrum (pss_get_field_fourier, pss_debug_noise): kx = 0..n0/2 fastest, then ky, then kz;
 *     logical mode index m = (kz*n1 + ky)*(n0/2+1) + kx.  The library's internal layout differs.
 *
 * Ownership: the caller owns every buffer it passes and must keep the bound workspace alive until
 * pss_destroy (or the next pss_bind).  The library owns the opaque handle and small host tables.
 * Handles are not thread-safe.  No exceptions cross this boundary; there is no global state apart from the fixed device
 * array behind pss_debug_noise_noalloc (described there).
 *
 * Errors: every int-returning call gives 0 on success or a negative code:
 *   PSS_EINVAL        bad id / negative power / NULL / aux used before defined / implicit term on aux
 *   PSS_EUNSUPPORTED  n_j not a power of two, n_j < 8, n_j > 8192 (2D/3D axes must fit one CTA's
 *                     shared memory; 1D n <= 8192), more than 3 dims, product of > 4 factors,
 *                     table capacities exceeded (see PSS_MAX_*)
 *   PSS_ESTATE        add_* after finalize; bind/step/get before finalize/bind
 *   PSS_ECUDA         a CUDA call failed (sticky for the handle; text via pss_last_cuda_error)
 *   PSS_ETOOBIG       pss_debug_noise_noalloc only: the lattice has more than PSS_STATIC_NOISE_MAX_MODES modes
 */
#ifndef PSS_H
#define PSS_H
#include <stddef.h>
#include <stdint.h>
#ifdef __cplusplus
extern "C" {
#endif

typedef struct pss_system pss_system;

typedef enum { PSS_F32 = 0, PSS_F64 = 1 } pss_precision;
enum { PSS_DEALIAS_PAPER = 0, PSS_DEALIAS_TWO_THIRDS = 1, PSS_DEALIAS_OFF = 2 };
enum { PSS_OK = 0, PSS_EINVAL = -1, PSS_EUNSUPPORTED = -2, PSS_ESTATE = -3, PSS_ECUDA = -4, PSS_ETOOBIG = -5 };

/* capacities of the device-side term program */
enum {
  PSS_MAX_DYNAMIC = 4,   /* dynamic fields                                         */
  PSS_MAX_FACTORS = 12,  /* distinct fields that appear in products of order >= 2  */
  PSS_MAX_GROUPS = 8,    /* distinct (target field, outer operator) pairs          */
  PSS_MAX_TERMS = 32,    /* product terms                                          */
  PSS_MAX_LINOPS = 96    /* flattened operator monomials                           */
};

/* One operator monomial in Fourier space (keywords of PAPER.md:186-190):
 *   coef * (q^2)^q2_pow * (1/|q|)^invq_pow * (i q_x)^iq_pow[0] (i q_y)^iq_pow[1] (i q_z)^iq_pow[2]
 * (1/|q|)^p := 0 at q = 0; a monomial with an odd iq_pow[j] is 0 at the Nyquist index k_j = n_j/2. */
typedef struct {
  double coef;
  int q2_pow;
  int invq_pow;
  int iq_pow[3];
} pss_op;

/* PAPER.md:141 (i): "evolver system(gpu, Nx, Ny, dx, dy, dt, output)".  n, dx: host arrays of 3. */
int pss_create(pss_system **out, int ndim, const int64_t n[3], const double dx[3], double dt,
               pss_precision prec, uint64_t seed);
/* createField(name, dynamic).  *field_id receives the id (creation order). */
int pss_add_field(pss_system *, const char *name, int dynamic, int *field_id);
/* lhs term of "dt phi + lhs = rhs": L_q -= coef*Op(q).  Dynamic fields only. */
int pss_add_linear(pss_system *, int field, const pss_op *op);
/* intermediate field definition psi_q += coef*Op(q)*src_q; src is a dynamic
 * field or an EARLIER aux field. */
int pss_add_aux_def(pss_system *, int aux, const pss_op *op, int src);
/* Dirichlet frame (section V and Fig. 2: "a buffer zone of infinite stiffness in the boundaries"): at the
 * end of every time step the field is set, in real space, to lo_value where x_axis < lo_width and to hi_value where
 * x_axis >= n_axis - hi_width (widths in lattice sites, 0 = none; several frames of one field are applied in the order
 * given).  This is the built-in form of the paper's callback; an arbitrary callback is a caller kernel between
 * pss_get_field(device) and pss_set_field(device).  Dynamic fields, before pss_finalize. */
int pss_set_frame(pss_system *, int field, int axis, int64_t lo_width, double lo_value, int64_t hi_width, double hi_value);
/* Intermediate field with its own lhs ("psi + psi*q^2 = -q^2*phi"): den(q) psi_q = rhs_q with
 * den(q) = sum of the operators added here; psi_q = 0 where den(q) = 0 (reading A10).  None added = the bare field.
 * The CUDA path takes real-valued lhs operators (even total derivative order) and at most two such fields
 * (PSS_EUNSUPPORTED at pss_finalize otherwise). */
int pss_add_aux_lhs(pss_system *, int aux, const pss_op *op);
/* rhs term of an intermediate field that is a PRODUCT of 2..4 fields: psi_q += outer(q) F[prod](q).
 * factor_fields: host array of dynamic fields or intermediate fields created earlier.  Such a field is re-evaluated
 * every step in its own round of the two step kernels (one round per dependency level) before the fields that use it;
 * 2D/3D single systems (PSS_EUNSUPPORTED for 1D or ensembles). */
int pss_add_aux_term(pss_system *, int aux, const pss_op *outer, int nfactors, const int *factor_fields);
/* rhs term (Eq. 15): N_q += outer(q) * F[ prod_k factor_k(x) ].  nfactors == 1 is an
 * explicit linear term evaluated in Fourier space (no transform, no mask).  factor_fields: host array. */
int pss_add_term(pss_system *, int field, const pss_op *outer, int nfactors, const int *factor_fields);
/* addNoise(field, "D*q^a"): <|nu_q|^2> = 2 D |q|^a dt N / dV. */
int pss_set_noise(pss_system *, int field, double D, int q_power);
/* de-aliasing rule: PAPER = cutoff 2/(n+1) per factor field, n its highest order. */
int pss_set_dealias(pss_system *, int rule);
/* Ensemble (stochastic studies need many realisations): the system holds
 * `nreplicas` independent realisations of the same field system and pss_step advances all of them in the same
 * launches (grid dimension y).  Replica r is, bit for bit, the system created with seed + r.  Call before
 * pss_finalize; 1 <= nreplicas <= 65535, and in 3D additionally max(#factor fields, #product groups) * nreplicas
 * <= 65535 (pss_finalize returns PSS_EUNSUPPORTED otherwise).  The persistent 1024^2 kernel (p2d::k_persist2d) runs one launch per replica. */
int pss_set_replicas(pss_system *, int nreplicas);
/* which replica pss_set_field / pss_get_field / pss_get_field_fourier / pss_debug_noise address (default 0) */
int pss_select_replica(pss_system *, int replica);
int pss_replicas(const pss_system *);
/* validate, freeze the term list, plan the kernels; *workspace_bytes = device bytes pss_bind needs. */
int pss_finalize(pss_system *, size_t *workspace_bytes);
/* device_workspace: DEVICE pointer, 256-byte aligned, >= workspace_bytes, zero-initialised by this
 * call.  cuda_stream: a cudaStream_t of the workspace's device (NULL = default stream); all later work is issued on
 * it.  The device that owns the workspace is recorded here; every later entry point makes it current for the
 * duration of the call and restores the caller's current device, so the caller need not cudaSetDevice. */
int pss_bind(pss_system *, void *device_workspace, size_t bytes, void *cuda_stream);
/* R2C of user real data (x fastest) into the state.  on_device: 1 = DEVICE pointer, 0 = HOST pointer
 * (copied with cudaMemcpyAsync on the bound stream, then the stream is synchronised). */
int pss_set_field(pss_system *, int field, const void *real_xfastest, int on_device);
/* nsteps time steps, asynchronous on the bound stream.
 * pss_step(a); pss_step(b) is bit-identical to pss_step(a+b). */
int pss_step(pss_system *, int64_t nsteps);
/* C2R of the (unmasked) state, including 1/N.  Host destination => stream synchronised on return. */
int pss_get_field(pss_system *, int field, void *real_out, int on_device);
/* the state in the logical half-spectrum layout, complex of the system precision. */
int pss_get_field_fourier(pss_system *, int field, void *halfspectrum_out, int on_device);
/* Checkpoint / resume.  The whole state of a run is the half-spectra of the dynamic fields (pss_get_field_fourier)
 * plus the step counter, which feeds the noise key.  Restoring both into a freshly built system of the same field
 * system and seed continues the run bit for bit (the noise is counter-based: SURVEY.md section 5).
 * halfspectrum_in: logical layout of pss_get_field_fourier, complex of the system precision. */
int pss_set_field_fourier(pss_system *, int field, const void *halfspectrum_in, int on_device);
/* PSS_ESTATE before pss_finalize. */
int pss_set_step_count(pss_system *, uint64_t step);
/* test hook for the noise stream (HOST pointers, either may be NULL): the 4 Philox4x32-10 words per
 * logical mode m, and the unit Hermitian Gaussian z (complex of the system precision) the step uses. */
int pss_debug_noise(pss_system *, int field, uint64_t step, uint32_t *bits4_per_mode, void *z_halfspectrum);
/* pss_debug_noise without any allocation.  Same arguments, same kernel, same values (bit for bit); the only difference
 * is where the kernel's results wait on the device before they are copied to `bits4_per_mode` / `z_halfspectrum`.
 *
 * Why it exists.  pss_debug_noise is the one call of this library that asks the CUDA runtime for device memory
 * (cudaMalloc, released with cudaFree before it returns).  A program built around this library often cannot afford
 * that, or is not allowed to:
 *   - the usual host is a PyTorch (or RMM, or other pooling) process whose caching allocator already holds nearly
 *     all of the GPU's memory; a raw cudaMalloc then fails with "out of memory" although the pool has plenty free;
 *   - cudaFree waits for ALL work on the device, so checking the noise stream from a monitoring thread stalls every
 *     other stream of a running simulation or training job;
 *   - while any thread of the process is capturing a CUDA graph in the default (global) capture mode, cudaMalloc is
 *     an illegal call: it fails and breaks that thread's capture.
 * Such callers use this entry point: it calls no cudaMalloc, cudaFree or any library routine that allocates.
 *
 * How.  The staging area is a fixed array compiled into the library, PSS_STATIC_NOISE_MAX_MODES * 32 bytes
 * (16.03 MiB: room for the 1024 x 513 half-spectrum of the headline lattice in either precision).  The CUDA runtime
 * places it on every GPU on which the library is loaded and keeps it there until the process exits, whether or not
 * this call is ever made.  A system with more modes (n0/2+1)*n1*n2 than that gets PSS_ETOOBIG and nothing is launched.
 *
 * First call on a device: it looks up the array's device address (cudaGetSymbolAddress) and keeps it for later
 * calls.  Make that first call at set-up time, before any stream capture begins.
 *
 * Sharing: there is ONE array per GPU for the whole process.  Every call overwrites what the previous one left there
 * (each call writes all it later reads, so stale contents never reach the caller and nothing needs clearing).  A call
 * returns only after its results are in host memory, but two calls that are in flight at the same time on one GPU —
 * from two threads, through two handles or streams — write the same bytes and corrupt each other: serialise them.
 * HOST pointers, either may be NULL, as for pss_debug_noise. */
enum { PSS_STATIC_NOISE_MAX_MODES = 1024 * 513 };
int pss_debug_noise_noalloc(pss_system *, int field, uint64_t step, uint32_t *bits4_per_mode, void *z_halfspectrum);
/* measurement hook: nsteps (<= 4096) steps exactly as pss_step, with one CUDA-event pair around every
 * kernel launch on the bound stream; synchronises.  Returns the mean device time per launch in ms and
 * the launch count of each kernel family: [0] k_rows, [1] k_update, [2] k_mid (3D only), [3] the persistent 1024^2 fp32
 * kernel (ONE launch runs all nsteps steps; which one: pss_uses_fused_kernel).  Not for 1D. */
int pss_profile_step(pss_system *, int64_t nsteps, double ms_per_launch[4], int64_t launches[4]);
/* 0: this (finalized and bound) system steps with the two generic kernels; 1: with the persistent kernel of
 * pss_fused2d.cuh (f2d::k_fused2d / k_fused2d_pair); 2: with its second generation, pss_persist2d.cuh (p2d::k_persist2d). */
int pss_uses_fused_kernel(const pss_system *);
/* number of kernels this handle has launched so far (for bench.py's gpu_launches claim). */
uint64_t pss_launch_count(const pss_system *);
/* The state is kept in Fourier space for the whole run.  On the planes kx = 0 and kx = n0/2 the half-spectrum stores both
 * members of each conjugate pair, and only their Hermitian combination belongs to the real field; the
 * rest is rounding residue that Eq. 18 would amplify wherever L_q > 0.  pss_step therefore replaces those pairs by their
 * Hermitian mean after every step whose number (pss_step_count) is a multiple of the period returned here (a power of
 * two <= 1024 chosen at pss_finalize from the largest 1/|1 - dt L_q|; 0 before pss_finalize).  The schedule depends on
 * the step number only, so splitting a run into several pss_step calls, or restoring a checkpoint, changes nothing. */
int64_t pss_hermitian_period(const pss_system *);
/* algorithmic bytes one step of this system must move: pruned != 0 gives B_alg,
 * pruned == 0 gives B_model. */
double pss_model_bytes_per_step(const pss_system *, int pruned);
uint64_t pss_step_count(const pss_system *);
const char *pss_strerror(int code);
const char *pss_last_cuda_error(const pss_system *);
void pss_destroy(pss_system *);

#ifdef __cplusplus
}
#endif
#endif
