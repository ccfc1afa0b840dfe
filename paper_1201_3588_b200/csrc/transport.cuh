// transport.cuh -- pieces shared by the sm_100a transport kernels (rows a1..a8 of
// SURVEY.md 8(a)): kernel parameters, the counter-based random numbers
// (R18, R19), direction draws (R15), the inverse-CDF search, the observer tally (R34) and the
// pre-pass that hands the packages of a batch out grouped by where they start.  The transport
// kernel itself (single-level AND two-level grids) is k_transport_u in transport_u.cuh.
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

namespace mcrt {

// Bounds checks of our own (compute-sanitizer is not available on the GPU pool): a library built
// with -DMCRT_CHECKS counts every storage-slot index outside [0, store slots) before it is used;
// tests/test_gpu_checks.py builds that variant and requires the count to stay 0.
#ifdef MCRT_CHECKS
__device__ unsigned long long g_mcrt_violations = 0ull;
__device__ long long g_mcrt_nstore = 0;
#define MCRT_CHECK_SLOT(s)                                                                     \
  do {                                                                                         \
    if ((unsigned long long)(long long)(s) >= (unsigned long long)g_mcrt_nstore)               \
      atomicAdd(&g_mcrt_violations, 1ull);                                                     \
  } while (0)
#else
#define MCRT_CHECK_SLOT(s) do { } while (0)
#endif

constexpr uint32_t kTagEmit = 0, kTagFlight = 1, kTagReemit = 2, kTagPah = 4;
constexpr uint32_t kMaxFlights = 10000000u;          // R20
constexpr unsigned kFull = 0xffffffffu;

enum : int { CNT_EMITTED = 0, CNT_ESCAPED, CNT_LOST, CNT_ABS, CNT_SCA, CNT_FLIGHTS, CNT_CROSS, CNT_N };

struct SrcDev {
  int type;          // 0 point, 1 external field
  int fine[3];       // point source: floor of the position in finest-level units
  float frac[3];     // ... and its fractional part in [0,1)
  double lcdf;       // cumulative luminosity fraction (fp64: the source pick is exact, see draw_emit)
};

// Direction-resolved tallies of escaping packages (reading R34;
// the paper's product is an image and flux profiles).  Off when n_mu = n_pix = 0.
struct ObserverDev {
  int n_mu, n_pix, bin_lo, bin_hi;
  float o[3], e1[3], e2[3];                    // unit vector towards the observer; image axes
  float cos_alpha, half_width;                 // acceptance cone; image half width in root-cube edges
  unsigned long long* sed_mu;                  // [n_mu][3][nb]
  unsigned long long* image;                   // [n_pix][n_pix], row = e2, column = e1
};

struct TransportParams {
  const float* __restrict__ rho;               // [slots] density / refined-cube marker
  unsigned long long* __restrict__ tally;      // [slots] cumulative absorbed-package counts
  uint32_t* __restrict__ tally32;              // NULL, or [slots] this batch's counts only (packet-sharded runs:
                                               // the ranks all-reduce this array, not the cumulative one)
  const float* __restrict__ trow;              // [slots] temperature as table row coordinate
  const float4* __restrict__ opac;             // [nb] (kappa_ext*root_size, albedo, g, kappa_abs)
  const float* __restrict__ cdf;               // [nT][nb] emission inverse-CDF rows
  const uint32_t* __restrict__ cdf_guide;      // [nT][kCdfGuide] bracket of the search in a row (tables.cuh), or NULL
  const float* __restrict__ csrc;              // [nsrc][nb] source spectrum CDFs, fp32 copy: searched in the same
                                               // instruction stream as the re-emission rows ...
  const double* __restrict__ csrc64;           // ... and the fp64 table that settles the bin exactly
  const SrcDev* __restrict__ src;              // [nsrc]
  // transiently heated PAH (row f2, pah.cuh); pah_q = NULL: no PAH declared
  const float* __restrict__ pah_q;             // [nb] share of an absorption taken by the PAH (R36)
  uint32_t* __restrict__ pah_cnt;              // [slots][nb] packages absorbed by the PAH, per leaf and bin
  const float* __restrict__ pah_cdf;           // [slots][nb] emission CDF of each leaf's PAH (frozen in a batch)
  unsigned long long* next;                    // work-queue head (packet offset within the batch)
  unsigned long long* next_reset;              // the head the NEXT launch will use: set to 0 by this one (two heads
                                               // alternate, so no launch needs a memset of its own in front of it)
  const uint32_t* __restrict__ perm;           // NULL, or the batch's package numbers grouped by source
  unsigned long long* sed;                     // [3][nb]
  unsigned long long* emit_bin;                // [nb]
  unsigned long long* counters;                // [CNT_N]
  unsigned long long seed, first, count;
  int N, S, nb, nT, nsrc, n3;
  ObserverDev obs;
};

// O9 / R34: an escaping package at position (x,y,z) (root-cube edges from the box corner) with
// direction d.  Inclination bin from mu = d_z; image pixel from the impact vector
// b = r - (r.d) d, r relative to the box centre, projected on (e1, e2).
__device__ __forceinline__ void tally_observer(const TransportParams& P, float x, float y, float z, float d0,
                                               float d1, float d2, int bin, int comp) {
  const ObserverDev& O = P.obs;
  if (O.n_mu > 0) {
    int m = (int)floorf((d2 + 1.f) * 0.5f * (float)O.n_mu);
    m = min(O.n_mu - 1, max(0, m));
    atomicAdd(O.sed_mu + ((size_t)m * 3 + comp) * P.nb + bin, 1ull);
  }
  if (O.n_pix > 0 && bin >= O.bin_lo && bin <= O.bin_hi) {
    if (d0 * O.o[0] + d1 * O.o[1] + d2 * O.o[2] >= O.cos_alpha) {
      const float h = 0.5f * (float)P.N;
      const float r0 = x - h, r1 = y - h, r2 = z - h;
      const float rd = r0 * d0 + r1 * d1 + r2 * d2;
      const float b0 = r0 - rd * d0, b1 = r1 - rd * d1, b2 = r2 - rd * d2;
      const float X = b0 * O.e1[0] + b1 * O.e1[1] + b2 * O.e1[2];
      const float Y = b0 * O.e2[0] + b1 * O.e2[1] + b2 * O.e2[2];
      const float fx = (X + O.half_width) / (2.f * O.half_width) * (float)O.n_pix;
      const float fy = (Y + O.half_width) / (2.f * O.half_width) * (float)O.n_pix;
      if (fx >= 0.f && fx < (float)O.n_pix && fy >= 0.f && fy < (float)O.n_pix)
        atomicAdd(O.image + (size_t)floorf(fy) * O.n_pix + (size_t)floorf(fx), 1ull);
    }
  }
}

// ---- Philox4x32-10 (Salmon et al. 2011), counter = (pid_lo, pid_hi, k, tag), key = seed (R18) ----
__device__ __forceinline__ void philox4x32_10(uint32_t k0, uint32_t k1, uint32_t c0, uint32_t c1,
                                              uint32_t c2, uint32_t c3, uint32_t out[4]) {
#pragma unroll
  for (int r = 0; r < 10; ++r) {
    uint32_t hi0 = __umulhi(0xD2511F53u, c0), lo0 = 0xD2511F53u * c0;
    uint32_t hi1 = __umulhi(0xCD9E8D57u, c2), lo1 = 0xCD9E8D57u * c2;
    uint32_t n0 = hi1 ^ c1 ^ k0, n2 = hi0 ^ c3 ^ k1;
    c0 = n0; c1 = lo1; c2 = n2; c3 = lo0;
    k0 += 0x9E3779B9u; k1 += 0xBB67AE85u;
  }
  out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

// R19: 23-bit uniform ((x >> 9) + 0.5) * 2^-23.  n + 0.5 with n < 2^23 needs 24 significant bits,
// so the value is exact in fp32 and lies strictly inside (0,1): never 0, never 1 (a 24-bit
// variant rounds n = 2^24 - 1 up to 1.0).  tau* = -ln u is therefore > 0 and <= 16.6.
__device__ __forceinline__ float u01(uint32_t x) {
  return ((float)(x >> 9) + 0.5f) * 1.1920928955078125e-7f;
}
// The emission decisions (which source, which frequency bin: once per package) are taken in fp64
// with the oracle's uniform (x + 0.5) * 2^-32 against fp64 tables, so that the number of packages
// emitted per source and per bin equals the oracle's exactly.
__device__ __forceinline__ double u01d(uint32_t x) {
  return ((double)x + 0.5) * 2.3283064365386962890625e-10;
}

// the four random words of (seed, package id, k, tag) (R18)
__device__ __forceinline__ void draw4w(unsigned long long seed, unsigned long long pid, uint32_t k,
                                       uint32_t tag, uint32_t x[4]) {
  philox4x32_10((uint32_t)seed, (uint32_t)(seed >> 32), (uint32_t)pid, (uint32_t)(pid >> 32), k, tag, x);
}
__device__ __forceinline__ void draw4(unsigned long long seed, unsigned long long pid, uint32_t k,
                                      uint32_t tag, float u[4]) {
  uint32_t x[4];
  draw4w(seed, pid, k, tag, x);
  u[0] = u01(x[0]); u[1] = u01(x[1]); u[2] = u01(x[2]); u[3] = u01(x[3]);
}

// first j with cdf[j] >= u, known to lie in [lo, hi] (the whole row, or the bracket a guide table gives)
template <typename T>
__device__ __forceinline__ int search_cdf_range(const T* __restrict__ cdf, int lo, int hi, T u) {
  while (lo < hi) {
    int mid = (lo + hi) >> 1;
    if (__ldg(cdf + mid) >= u) hi = mid; else lo = mid + 1;
  }
  return lo;
}

// first j with cdf[j] >= u
template <typename T>
__device__ __forceinline__ int search_cdf(const T* __restrict__ cdf, int n, T u) {
  int lo = 0, hi = n - 1;
  while (lo < hi) {
    int mid = (lo + hi) >> 1;
    if (__ldg(cdf + mid) >= u) hi = mid; else lo = mid + 1;
  }
  return lo;
}

// sin and cos of 2 pi u, u in (0,1), from the special-function unit (MUFU.SIN / MUFU.COS after one range step to
// [-pi, pi]: absolute error < 5e-7, against ~40 instructions of sincospif).  The direction built from them is
// renormalised where it is rotated (rotate_dir) and is a unit vector to 1e-6 where it is not (isotropic_dir) -- the
// size of the fp32 rounding the walk itself carries (R33); the oracle keeps the exact fp64 functions.
__device__ __forceinline__ void sincos_2pi(float u, float* sn, float* cs) {
  const float x = 6.283185307179586f * (u - 0.5f);            // in (-pi, pi): sin(2 pi u) = -sin x, cos(2 pi u) = -cos x
  *sn = -__sinf(x);
  *cs = -__cosf(x);
}

__device__ __forceinline__ void isotropic_dir(float u2, float u3, float& a, float& b, float& c) {
  float mu = 2.f * u2 - 1.f;
  float s = sqrtf(fmaxf(0.f, 1.f - mu * mu));
  float sn, cs;
  sincos_2pi(u3, &sn, &cs);
  a = s * cs; b = s * sn; c = mu;
}

__device__ __forceinline__ float hg_cos(float g, float u) {     // R15
  if (fabsf(g) < 1e-3f) return 2.f * u - 1.f;
  float t = __fdividef(1.f - g * g, 1.f - g + 2.f * g * u);
  float c = __fdividef(1.f + g * g - t * t, 2.f * g);
  return fminf(1.f, fmaxf(-1.f, c));
}

__device__ __forceinline__ void rotate_dir(float d0, float d1, float d2, float ct, float u3,
                                           float& a, float& b, float& c) {
  float st = sqrtf(fmaxf(0.f, 1.f - ct * ct));
  float sp, cp;
  sincos_2pi(u3, &sp, &cp);
  float q2 = d0 * d0 + d1 * d1;                 // = 1 - d2^2, without the cancellation
  if (q2 > 1e-12f) {
    float iq = rsqrtf(q2), q = q2 * iq;
    a = st * (d0 * d2 * cp - d1 * sp) * iq + d0 * ct;
    b = st * (d1 * d2 * cp + d0 * sp) * iq + d1 * ct;
    c = -st * cp * q + d2 * ct;
  } else {
    a = st * cp; b = st * sp; c = (d2 >= 0.f ? ct : -ct);
  }
  float inv = rsqrtf(a * a + b * b + c * c);
  a *= inv; b *= inv; c *= inv;
}

// ---- a8, several sources: hand the packages out GROUPED BY SOURCE ----------------------------
// Packages of one source cross the same neighbourhood, so when the packages in flight share a
// source the L2 serves far more of their density gathers (profiles/r01_summary.md: 512^3 cube,
// one source at a time 1.5-1.8e11 crossings/s against 1.17e11 with the eleven sources mixed);
// packages that also start in the same direction share their whole first flight.
// The source of package i is the first decision of its emission (O4: u0 of its EMIT block), so a
// pre-pass can group the batch's package numbers by source: count, exclusive scan, scatter.  The
// order inside a group is arbitrary; integer tallies make the results independent of it.
#ifndef MCRT_MAX_GROUPS
#define MCRT_MAX_GROUPS 8192
#endif
constexpr int kMaxOrderedSources = MCRT_MAX_GROUPS;   // groups of the hand-out (sources x start-direction bins)

// group key of a package: its source, refined by where it starts to fly: sub = 2 m^2 bins, m x 2m in (mu, phi)
// of the emission direction for a point source (m = 4 ... 64), face x 2 x 2 tiles for the external field.  The
// finer the bins the closer together the packages of a warp fly AND the more alike their flights are, so that they
// stop together: c2 / c3 per launch with 32 bins 3.45 / 7.10 ms, 128: 3.13 / 6.57, 512: 3.02 / 6.28, 2048: 2.93 / 6.08.
__device__ __forceinline__ int group_of(const TransportParams& P, unsigned long long pid, int sub) {
  uint32_t x[4];
  philox4x32_10((uint32_t)P.seed, (uint32_t)(P.seed >> 32), (uint32_t)pid, (uint32_t)(pid >> 32), 0u, kTagEmit, x);
  const double u0 = u01d(x[0]);
  int s = 0;
  while (s < P.nsrc - 1 && P.src[s].lcdf < u0) ++s;
  if (sub == 1) return s;
  int b;
  if (P.src[s].type == 0) {
    const int m = sub >= 8192 ? 64 : sub >= 2048 ? 32 : sub >= 512 ? 16 : sub >= 128 ? 8 : 4;
    b = min(m - 1, (int)((float)m * u01(x[2]))) * (2 * m) + min(2 * m - 1, (int)((float)(2 * m) * u01(x[3])));
  } else {
    philox4x32_10((uint32_t)P.seed, (uint32_t)(P.seed >> 32), (uint32_t)pid, (uint32_t)(pid >> 32), 1u, kTagEmit, x);
    b = min(5, (int)(6.f * u01(x[0]))) * 4 + (u01(x[1]) >= 0.5f ? 1 : 0) + (u01(x[2]) >= 0.5f ? 2 : 0);
  }
  return s * sub + b;
}

// counts[g] += packages of group g (cursor == NULL: the group of every package is also kept in keys[], so that
// the second pass need not repeat its Philox block), or perm[cursor[g]++] = package number
__global__ void k_group_by_source(const TransportParams P, const int sub, unsigned int* __restrict__ counts,
                                  unsigned int* __restrict__ cursor, uint32_t* __restrict__ perm,
                                  uint16_t* __restrict__ keys) {
  extern __shared__ unsigned int s_cnt[];                    // [2 * ngroups]: block histogram, block bases
  const int ng = P.nsrc * sub;
  for (int i = threadIdx.x; i < 2 * ng; i += blockDim.x) s_cnt[i] = 0;
  __syncthreads();
  const unsigned long long per_block = (P.count + gridDim.x - 1) / gridDim.x;
  const unsigned long long lo = per_block * blockIdx.x, hi = min(P.count, lo + per_block);
  if (!cursor) {
    for (unsigned long long i = lo + threadIdx.x; i < hi; i += blockDim.x) {
      const int g = group_of(P, P.first + i, sub);
      keys[i] = (uint16_t)g;
      atomicAdd(&s_cnt[g], 1u);
    }
    __syncthreads();
    for (int i = threadIdx.x; i < ng; i += blockDim.x)
      if (s_cnt[i]) atomicAdd(&counts[i], s_cnt[i]);
    return;
  }
  for (unsigned long long i = lo + threadIdx.x; i < hi; i += blockDim.x) atomicAdd(&s_cnt[keys[i]], 1u);
  __syncthreads();
  for (int i = threadIdx.x; i < ng; i += blockDim.x) {       // reserve this block's range in every group
    s_cnt[ng + i] = s_cnt[i] ? atomicAdd(&cursor[i], s_cnt[i]) : 0u;
    s_cnt[i] = 0;
  }
  __syncthreads();
  for (unsigned long long i = lo + threadIdx.x; i < hi; i += blockDim.x) {
    const int g = keys[i];
    perm[s_cnt[ng + g] + atomicAdd(&s_cnt[g], 1u)] = (uint32_t)i;
  }
}

// cursor[s] = sum of counts[0..s): one block of 1024 threads, each summing a run of consecutive entries
__global__ void k_scan_sources(const unsigned int* __restrict__ counts, unsigned int* __restrict__ cursor, int n) {
  __shared__ unsigned int s_part[1024];
  const int per = (n + 1023) / 1024;
  const int lo = min(n, (int)threadIdx.x * per), hi = min(n, lo + per);
  unsigned int acc = 0;
  for (int i = lo; i < hi; ++i) acc += counts[i];
  s_part[threadIdx.x] = acc;
  __syncthreads();
  for (int o = 1; o < 1024; o <<= 1) {                       // inclusive scan of the partial sums
    const unsigned int v = threadIdx.x >= (unsigned)o ? s_part[threadIdx.x - o] : 0u;
    __syncthreads();
    s_part[threadIdx.x] += v;
    __syncthreads();
  }
  unsigned int run = s_part[threadIdx.x] - acc;              // exclusive
  for (int i = lo; i < hi; ++i) { cursor[i] = run; run += counts[i]; }
}

}  // namespace mcrt
