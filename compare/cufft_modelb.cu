/*
 * cufft_modelb.cu — TIMING COMPARISON ONLY, not part of the product (libpss.so never links or loads this).
 *
 * The 2D Model B step written the way the paper describes its own GPU path: one library call
 * or one pointwise kernel per arrow of the six-step list, cuFFT for every transform, cuRAND for the noise
 * ("generate a Gaussian white noise field and apply its variance").  north_star asks for this
 * build to be timed beside the hand-written path as a baseline.  It shares no code with csrc/ and its result is
 * not compared with anything (different noise stream, standard cuFFT half-spectrum layout [ny][nx/2+1]).
 *
 * Per step: mask copy -> C2R -> cube -> R2C -> curandGenerateNormal -> R2C of the white field -> Eq. 18 update.
 */
#include <cuda_runtime.h>
#include <cufft.h>
#include <curand.h>
#include <curand_kernel.h>
#include <math.h>
#include <stdint.h>

namespace {

struct Par {
  int nx, ny, nxh;
  float qsx, qsy, dt, a, b, k, namp2, invN;
};

__device__ __forceinline__ int sidx(int k, int n) { return (k <= n / 2) ? k : k - n; }

/* psi_hat = phi_hat where 4|s(k)| < n on both axes (cubic term: cutoff 2/(n+1)), else 0 */
__global__ void k_mask(Par p, const float2 *phi, float2 *psi) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= p.nxh * p.ny) return;
  const int kx = i % p.nxh, ky = i / p.nxh;
  const bool keep = 4 * kx < p.nx && 4 * abs(sidx(ky, p.ny)) < p.ny;
  psi[i] = keep ? phi[i] : make_float2(0.f, 0.f);
}
__global__ void k_cube(Par p, float *r) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= p.nx * p.ny) return;
  const float v = r[i] * p.invN;
  r[i] = v * v * v;
}
/* Eq. 18 with N_q = -b q^2 (phi^3)_q, L_q = -(a q^2 + k q^4), noise sqrt(2 D q^2 dt / dV) eta_q */
__global__ void k_upd(Par p, float2 *phi, const float2 *cube, const float2 *eta) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= p.nxh * p.ny) return;
  const int kx = i % p.nxh, ky = i / p.nxh;
  const float qx = p.qsx * kx, qy = p.qsy * sidx(ky, p.ny);
  const float q2 = qx * qx + qy * qy;
  const float amp = sqrtf(p.namp2 * q2);
  const float2 c = cube[i], e = eta[i], f = phi[i];
  const float inv = 1.f / (1.f + p.dt * (p.a * q2 + p.k * q2 * q2));
  phi[i] = make_float2((f.x - p.dt * p.b * q2 * c.x + amp * e.x) * inv, (f.y - p.dt * p.b * q2 * c.y + amp * e.y) * inv);
}

}  // namespace

extern "C" int cmp_cufft_modelb(int nx, int ny, double dx, double dt, double a, double b, double k, double D,
                                int nsteps, int warmup, double *us_per_step) {
  Par p;
  p.nx = nx; p.ny = ny; p.nxh = nx / 2 + 1;
  p.qsx = (float)(2.0 * M_PI / (nx * dx)); p.qsy = (float)(2.0 * M_PI / (ny * dx));
  p.dt = (float)dt; p.a = (float)a; p.b = (float)b; p.k = (float)k;
  p.namp2 = (float)(2.0 * D * dt / (dx * dx));  /* eta_q = FFT of unit white noise: <|eta_q|^2> = N */
  p.invN = (float)(1.0 / ((double)nx * ny));
  const size_t M = (size_t)p.nxh * ny, N = (size_t)nx * ny;
  float2 *phi = nullptr, *psi = nullptr, *eta = nullptr;
  float *real = nullptr, *white = nullptr;
  cufftHandle c2r = 0, r2c = 0;
  curandGenerator_t gen = nullptr;
  cudaEvent_t e0 = nullptr, e1 = nullptr;
  int rc = -1;
  do {
    if (cudaMalloc(&phi, M * sizeof(float2)) || cudaMalloc(&psi, M * sizeof(float2)) || cudaMalloc(&eta, M * sizeof(float2)) ||
        cudaMalloc(&real, N * sizeof(float)) || cudaMalloc(&white, N * sizeof(float))) break;
    if (cudaMemset(phi, 0, M * sizeof(float2))) break;
    if (cufftPlan2d(&c2r, ny, nx, CUFFT_C2R) != CUFFT_SUCCESS || cufftPlan2d(&r2c, ny, nx, CUFFT_R2C) != CUFFT_SUCCESS) break;
    if (curandCreateGenerator(&gen, CURAND_RNG_PSEUDO_PHILOX4_32_10) != CURAND_STATUS_SUCCESS) break;
    curandSetPseudoRandomGeneratorSeed(gen, 2405024102ULL);
    cudaEventCreate(&e0); cudaEventCreate(&e1);
    const int T = 256, gm = (int)((M + T - 1) / T), gn = (int)((N + T - 1) / T);
    bool ok = true;
    for (int s = 0; s < warmup + nsteps && ok; ++s) {
      if (s == warmup) cudaEventRecord(e0, 0);
      k_mask<<<gm, T>>>(p, phi, psi);
      ok = ok && cufftExecC2R(c2r, psi, real) == CUFFT_SUCCESS;
      k_cube<<<gn, T>>>(p, real);
      ok = ok && cufftExecR2C(r2c, real, psi) == CUFFT_SUCCESS;
      ok = ok && curandGenerateNormal(gen, white, N, 0.f, 1.f) == CURAND_STATUS_SUCCESS;
      ok = ok && cufftExecR2C(r2c, white, eta) == CUFFT_SUCCESS;
      k_upd<<<gm, T>>>(p, phi, psi, eta);
    }
    cudaEventRecord(e1, 0);
    if (cudaEventSynchronize(e1) != cudaSuccess || !ok || cudaGetLastError() != cudaSuccess) break;
    float ms = 0.f;
    cudaEventElapsedTime(&ms, e0, e1);
    *us_per_step = 1e3 * (double)ms / (double)nsteps;
    rc = 0;
  } while (0);
  if (e0) cudaEventDestroy(e0);
  if (e1) cudaEventDestroy(e1);
  if (gen) curandDestroyGenerator(gen);
  if (c2r) cufftDestroy(c2r);
  if (r2c) cufftDestroy(r2c);
  cudaFree(phi); cudaFree(psi); cudaFree(eta); cudaFree(real); cudaFree(white);
  return rc;
}

/* Pin P8: the Philox4x32-10 block of cuRAND's DEVICE API for (seed, subsequence, offset): with
 * curand_init(seed, subsequence, offset) the key is the seed, (c2, c3) = subsequence and (c0, c1) = offset / 4, so
 * the block (c0, c1, c2, c3) is subsequence = c2 | c3 << 32, offset = 4 (c0 | c1 << 32) followed by one curand4().
 * Test infrastructure for tests/ only (an independent implementation to compare the oracle's and the product's
 * Philox against); the product never calls it. */
namespace {
__global__ void k_curand_block(unsigned long long seed, unsigned long long subsequence, unsigned long long offset, unsigned int *out) {
  curandStatePhilox4_32_10_t st;
  curand_init(seed, subsequence, offset, &st);
  const uint4 r = curand4(&st);
  out[0] = r.x; out[1] = r.y; out[2] = r.z; out[3] = r.w;
}
}  // namespace

extern "C" int cmp_curand_philox_block(unsigned long long seed, unsigned long long subsequence, unsigned long long offset,
                                       unsigned int out4[4]) {
  unsigned int *d = nullptr;
  if (cudaMalloc(&d, 4 * sizeof(unsigned int)) != cudaSuccess) return -1;
  k_curand_block<<<1, 1>>>(seed, subsequence, offset, d);
  const cudaError_t e = cudaMemcpy(out4, d, 4 * sizeof(unsigned int), cudaMemcpyDeviceToHost);
  cudaFree(d);
  return e == cudaSuccess ? 0 : -1;
}
