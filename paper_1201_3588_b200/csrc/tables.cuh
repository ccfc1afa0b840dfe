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

// Bracket guide of the emission rows: the re-emission bin is "the first j with C[j] >= u" (R11), found by bisection
// of a 128...200-entry row -- 7-8 dependent loads from the L2 per absorption.  For u in [k/G, (k+1)/G) that bin lies
// in [g_k, g_{k+1}], g_k = first j with C[j] >= k/G (C is non-decreasing and ends in 1): the pair is stored as one
// word, lo | hi << 16, so ONE load narrows the search to the few bins of that slice.  Built from the fp32 rows with
// the search's own comparison; k/G is exact in fp32, so the bin found is the bisection's, bit for bit.
constexpr int kCdfGuide = 32;
__global__ void k_build_cdf_guide(const float* __restrict__ cdf, int nb, int nT, uint32_t* __restrict__ guide) {
  const int row = blockIdx.x, k = threadIdx.x;
  if (row >= nT || k >= kCdfGuide) return;
  const float* c = cdf + (size_t)row * nb;
  uint32_t g[2];
  for (int e = 0; e < 2; ++e) {
    const float u = (float)(k + e) * (1.f / (float)kCdfGuide);
    int lo = 0, hi = nb - 1;
    while (lo < hi) {
      const int mid = (lo + hi) >> 1;
      if (c[mid] >= u) hi = mid; else lo = mid + 1;
    }
    g[e] = (uint32_t)lo;
  }
  guide[(size_t)row * kCdfGuide + k] = g[0] | (g[1] << 16);
}

// Source spectra: blackbody truncated to the band, same midpoint rule (R5, R6).  Kept in fp64: the
// emission bin is settled once per package with the fp64 uniform, so emitted-per-bin is exact; the
// fp32 copy serves the search loop that emission shares with re-emission.
__global__ void k_build_source_cdf(int nb, const double* __restrict__ Tbb, const double* __restrict__ nu,
                                   const double* __restrict__ dnu, double* __restrict__ csrc,
                                   float* __restrict__ csrc32) {
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
  {
    const double v = (j == nb - 1 || !(tot > 0)) ? 1.0 : s_term[j] / tot;
    csrc[(size_t)s * nb + j] = v;
    csrc32[(size_t)s * nb + j] = (float)v;
  }
}

// a9 / O7 (R9 reading B, R10, R12): per-leaf radiative-equilibrium temperature from the cumulative
// tally.  ln q = ln(cum) + ln_coef - ln(rho) (+ 3 ln S for subcubes); ln_coef = ln(L_tot /
// (N_cum 4 pi V_root)) is computed on the host in fp64.  Q^-1 by bracketing the ln Q table (in
// shared memory) and linear interpolation in (ln Q, ln T); the result is stored as the table row
// coordinate t = (ln T - ln T_min)/dlnT in [0, nT-1], which is what re-emission needs.
//
// The bracket lnQ[lo] <= lq < lnQ[lo+1] is found through a GUIDE table instead of a binary search
// (ten dependent, bank-conflicting shared-memory reads per leaf made the kernel run at 29 % of the
// copy bandwidth): the range [lnQ[0], lnQ[nT-1]] is cut into kGuide equal buckets, guide[b] = the
// largest row k whose lnQ[k] falls into a bucket below b, so lnQ[guide[b]] <= lq for every lq of
// bucket b, and a walk of (mostly 0 or 1) rows from there ends on the same bracket the binary
// search finds.  With ~2.5 buckets per row the kernel is a plain stream.
constexpr int kGuide = 2048;
__device__ __forceinline__ int q_bucket(float x, float lq0, float inv_w) {
  return min(kGuide - 1, max(0, (int)((x - lq0) * inv_w)));
}
__global__ void k_build_guide(const float* __restrict__ lnQ, int nT, int* __restrict__ guide) {
  const int b = blockIdx.x * blockDim.x + threadIdx.x;
  if (b >= kGuide) return;
  const float lq0 = lnQ[0], inv_w = (float)kGuide / (lnQ[nT - 1] - lnQ[0]);
  int lo = 0, hi = nT;                                       // rows [0, lo] are known to lie below bucket b (row 0 by definition)
  while (hi - lo > 1) { int mid = (lo + hi) >> 1; if (q_bucket(lnQ[mid], lq0, inv_w) < b) lo = mid; else hi = mid; }
  guide[b] = lo;
}

__device__ __forceinline__ float row_of_lnq(float lq, const float* s_lnQ, const int* s_guide, int nT, float lq0,
                                            float inv_w, bool use_guide) {
  if (lq >= s_lnQ[nT - 1]) return (float)(nT - 1);
  if (!(lq > s_lnQ[0])) return 0.f;
  int lo;
  if (use_guide) {
    lo = s_guide[q_bucket(lq, lq0, inv_w)];
    while (s_lnQ[lo + 1] <= lq) ++lo;                         // lq < lnQ[nT-1]: stops at the latest at nT-2
  } else {                                                    // degenerate table (rows with Q = 0): plain bisection
    int hi = nT - 1;
    lo = 0;
    while (hi - lo > 1) { int mid = (lo + hi) >> 1; if (s_lnQ[mid] <= lq) lo = mid; else hi = mid; }
  }
  return (float)lo + __fdividef(lq - s_lnQ[lo], s_lnQ[lo + 1] - s_lnQ[lo]);
}

// ln of the density of every storage slot, once per grid (-inf for empty leaves and for the markers of refined
// cubes): the update kernel then takes one logarithm per leaf instead of two
__global__ void k_ln_density(const float* __restrict__ rho, float* __restrict__ lnrho, long long slots) {
  const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= slots) return;
  const float r = rho[i];
  lnrho[i] = r > 0.f ? logf(r) : -INFINITY;
}

// O7 for one leaf: table row coordinate of its temperature from its cumulative count c and ln(density) lnr.
// ln c through the special-function unit (__logf: absolute error < 1e-6 on ln q, i.e. < 3e-7 relative on T).
__device__ __forceinline__ float trow_of_leaf(unsigned long long c, float lnr, bool is_sub, float ln_coef, float ln_sub3,
                                              const float* lnQ, const int* guide, int nT, float lq0, float inv_w,
                                              bool use_guide) {
  if (c == 0 || !(lnr > -1e30f)) return 0.f;                  // nothing absorbed; empty leaf or refined-cube marker
  const float lq = __logf((float)c) + ln_coef - lnr + (is_sub ? ln_sub3 : 0.f);
  return row_of_lnq(lq, lnQ, guide, nT, lq0, inv_w, use_guide);
}

// ADD: first add the batch's absorbed-package counts `delta` (u32, the sum over all ranks of a
// packet-sharded run) to the cumulative tally, then update (one pass over the leaves).
template <bool ADD>
__global__ void __launch_bounds__(256) k_update_temperature(const float* __restrict__ lnrho,
                                     unsigned long long* __restrict__ tally, const uint32_t* __restrict__ delta,
                                     float* __restrict__ trow, const float* __restrict__ lnQ,
                                     const int* __restrict__ guide, int nT, long long slots, long long n3,
                                     float ln_coef, float ln_sub3) {
  extern __shared__ float s_lnQ[];                            // [nT] + int[kGuide]
  int* s_guide = reinterpret_cast<int*>(s_lnQ + nT);
  for (int i = threadIdx.x; i < nT; i += blockDim.x) s_lnQ[i] = lnQ[i];
  for (int i = threadIdx.x; i < kGuide; i += blockDim.x) s_guide[i] = guide[i];
  __syncthreads();
  const float lq0 = s_lnQ[0], inv_w = (float)kGuide / (s_lnQ[nT - 1] - s_lnQ[0]);
  const bool use_guide = lq0 > -1e29f && s_lnQ[nT - 1] > lq0;
  auto one = [&](unsigned long long c, float r, long long i) -> float {
    return trow_of_leaf(c, r, i >= n3, ln_coef, ln_sub3, s_lnQ, s_guide, nT, lq0, inv_w, use_guide);
  };
  const long long stride = 2ll * gridDim.x * blockDim.x;
  for (long long i = 2ll * ((long long)blockIdx.x * blockDim.x + threadIdx.x); i < slots; i += stride) {
    if (i + 1 < slots) {                                      // two leaves per turn: 16-byte tally, 8-byte rho / trow accesses
      ulonglong2 c = *reinterpret_cast<const ulonglong2*>(tally + i);
      const float2 r = *reinterpret_cast<const float2*>(lnrho + i);
      if (ADD) {
        const uint2 d = *reinterpret_cast<const uint2*>(delta + i);
        c.x += d.x; c.y += d.y;
        *reinterpret_cast<ulonglong2*>(tally + i) = c;
      }
      *reinterpret_cast<float2*>(trow + i) = make_float2(one(c.x, r.x, i), one(c.y, r.y, i + 1));
    } else {
      unsigned long long c = tally[i];
      if (ADD) { c += delta[i]; tally[i] = c; }
      trow[i] = one(c, lnrho[i], i);
    }
  }
}

__global__ void k_trow_to_T(const float* __restrict__ trow, float* __restrict__ T, long long slots,
                            float lnTmin, float dlnT) {
  long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i < slots) T[i] = expf(lnTmin + dlnT * trow[i]);
}

}  // namespace mcrt
