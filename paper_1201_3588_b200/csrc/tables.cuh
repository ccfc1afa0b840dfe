// tables.cuh -- set-up kernels (row a0 of SURVEY.md 8(a)) and the batch-end temperature update
// (row a9).  Tables are built in fp64 on the device and stored as fp32 (R33).
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

namespace mcrt {

// CODATA 2018, cgs
#define MCRT_H_PLANCK 6.62607015e-27
#define MCRT_C_LIGHT 2.99792458e10
#define MCRT_K_BOLTZ 1.380649e-16

__device__ __forceinline__ double planck_nu(double nu, double T) {
  double x = MCRT_H_PLANCK * nu / (MCRT_K_BOLTZ * T);
  if (x > 700.0) return 0.0;
  return (2.0 * MCRT_H_PLANCK * nu * nu * nu / (MCRT_C_LIGHT * MCRT_C_LIGHT)) / expm1(x);
}

__global__ void k_sanitize(const float* __restrict__ in, float* __restrict__ out, long long n) {
  long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) { float v = in[i]; out[i] = (v > 0.f) ? v : 0.f; }
}

// O1 + O2 (R4, R13): frequency grid and mass-weighted mixing of the species, fp64.
__global__ void k_mix_opacity(int nb, int ns, const double* __restrict__ edges_um,
                              const double* __restrict__ weight, const float* __restrict__ kabs,
                              const float* __restrict__ ksca, const float* __restrict__ g,
                              double root_size, double* __restrict__ nu, double* __restrict__ dnu,
                              double* __restrict__ kabs_mix, float4* __restrict__ opac) {
  int j = blockIdx.x * blockDim.x + threadIdx.x;
  if (j >= nb) return;
  double l0 = edges_um[j] * 1e-4, l1 = edges_um[j + 1] * 1e-4;
  nu[j] = MCRT_C_LIGHT / sqrt(l0 * l1);
  dnu[j] = MCRT_C_LIGHT / l0 - MCRT_C_LIGHT / l1;
  double ka = 0, ks = 0, gs = 0;
  for (int s = 0; s < ns; ++s) {
    double a = (double)kabs[(size_t)s * nb + j], b = (double)ksca[(size_t)s * nb + j];
    ka += weight[s] * a;
    ks += weight[s] * b;
    gs += weight[s] * b * (double)g[(size_t)s * nb + j];
  }
  double ke = ka + ks;
  kabs_mix[j] = ka;
  opac[j] = make_float4((float)(ke * root_size), ke > 0 ? (float)(ks / ke) : 0.f,
                        ks > 0 ? (float)(gs / ks) : 0.f, (float)ka);
}

// O2 (R5, R11): one block per temperature row.  The running sum over bins is taken serially in
// bin order (the definition of the CDF); Planck terms are evaluated in parallel.
__global__ void k_build_emission_rows(int nb, int nT, double Tmin, double Tmax,
                                      const double* __restrict__ nu, const double* __restrict__ dnu,
                                      const double* __restrict__ kabs_mix, float* __restrict__ lnQ,
                                      float* __restrict__ cdf) {
  extern __shared__ double s_term[];
  int k = blockIdx.x;
  double T = Tmin * pow(Tmax / Tmin, (double)k / (double)(nT - 1));
  for (int j = threadIdx.x; j < nb; j += blockDim.x)
    s_term[j] = kabs_mix[j] * planck_nu(nu[j], T) * dnu[j];
  __syncthreads();
  if (threadIdx.x == 0) {
    double acc = 0;
    for (int j = 0; j < nb; ++j) { acc += s_term[j]; s_term[j] = acc; }
    lnQ[k] = acc > 0 ? (float)log(acc) : -1e30f;
    s_term[nb] = acc;
  }
  __syncthreads();
  double Q = s_term[nb];
  for (int j = threadIdx.x; j < nb; j += blockDim.x)
    cdf[(size_t)k * nb + j] = (j == nb - 1 || !(Q > 0)) ? 1.f : (float)(s_term[j] / Q);
}

// Source spectra: blackbody truncated to the band, same midpoint rule (R5, R6).  Kept in fp64: the
// emission bin is searched once per package with the fp64 uniform, so emitted-per-bin is exact.
__global__ void k_build_source_cdf(int nb, const double* __restrict__ Tbb, const double* __restrict__ nu,
                                   const double* __restrict__ dnu, double* __restrict__ csrc) {
  extern __shared__ double s_term[];
  int s = blockIdx.x;
  double T = Tbb[s];
  for (int j = threadIdx.x; j < nb; j += blockDim.x) s_term[j] = planck_nu(nu[j], T) * dnu[j];
  __syncthreads();
  if (threadIdx.x == 0) {
    double acc = 0;
    for (int j = 0; j < nb; ++j) { acc += s_term[j]; s_term[j] = acc; }
    s_term[nb] = acc;
  }
  __syncthreads();
  double tot = s_term[nb];
  for (int j = threadIdx.x; j < nb; j += blockDim.x)
    csrc[(size_t)s * nb + j] = (j == nb - 1 || !(tot > 0)) ? 1.0 : s_term[j] / tot;
}

// a9 / O7 (R9 reading B, R10, R12): per-leaf radiative-equilibrium temperature from the cumulative
// tally.  ln q = ln(cum) + ln_coef - ln(rho) (+ 3 ln S for subcubes); ln_coef = ln(L_tot /
// (N_cum 4 pi V_root)) is computed on the host in fp64.  Q^-1 by bracketing the ln Q table (in
// shared memory) and linear interpolation in (ln Q, ln T); the result is stored as the table row
// coordinate t = (ln T - ln T_min)/dlnT in [0, nT-1], which is what re-emission needs.
__global__ void k_update_temperature(const float* __restrict__ rho, const unsigned long long* __restrict__ tally,
                                     float* __restrict__ trow, const float* __restrict__ lnQ, int nT,
                                     long long slots, long long n3, float ln_coef, float ln_sub3) {
  extern __shared__ float s_lnQ[];
  for (int i = threadIdx.x; i < nT; i += blockDim.x) s_lnQ[i] = lnQ[i];
  __syncthreads();
  long long stride = (long long)gridDim.x * blockDim.x;
  for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < slots; i += stride) {
    unsigned long long c = tally[i];
    float r = rho[i];
    float t = 0.f;
    if (c > 0 && r > 0.f) {                                   // refined-root markers have r < 0
      float lq = logf((float)c) + ln_coef - logf(r) + (i >= n3 ? ln_sub3 : 0.f);
      if (lq >= s_lnQ[nT - 1]) t = (float)(nT - 1);
      else if (lq > s_lnQ[0]) {
        int lo = 0, hi = nT - 1;                              // lnQ[lo] <= lq < lnQ[hi]
        while (hi - lo > 1) { int mid = (lo + hi) >> 1; if (s_lnQ[mid] <= lq) lo = mid; else hi = mid; }
        t = (float)lo + (lq - s_lnQ[lo]) / (s_lnQ[lo + 1] - s_lnQ[lo]);
      }
    }
    trow[i] = t;
  }
}

__global__ void k_trow_to_T(const float* __restrict__ trow, float* __restrict__ T, long long slots,
                            float lnTmin, float dlnT) {
  long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i < slots) T[i] = expf(lnTmin + dlnT * trow[i]);
}

}  // namespace mcrt
