// transport.cuh -- sm_100a transport kernel: one photon package per thread, persistent threads
// with lane refill (rows a1..a8 of SURVEY.md 8(a)).
//
// A package lives entirely in registers.  It is never located from a floating-point position:
// its state is the integer index of the leaf it is in and, per axis, the remaining path length
// t_a to the face through which it would leave that leaf.  One crossing is
//   tmin = min(t_x,t_y,t_z);  dtau = rho_leaf * kappa_ext * tmin;  interaction if dtau >= tau_rem;
//   else tau_rem -= dtau;  t -= tmin;  the axis whose t became exactly 0 is the exit axis
//   (ties -> lowest axis, R21);  t_axis = (leaf edge)/|d_axis|;  step the integer index.
// The density array doubles as the two-level cell index: a root cube that is refined holds, in
// place of its (unused) density, a value with the sign bit set and the refined-cube number k in
// the low 31 bits, so every crossing costs one 4-byte gather.
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

constexpr uint32_t kTagEmit = 0, kTagFlight = 1, kTagReemit = 2;
constexpr uint32_t kMaxFlights = 10000000u;          // R20
constexpr int kWalkChunk = 32;                       // crossings per outer iteration
constexpr unsigned kFull = 0xffffffffu;

enum : int { ST_FETCH = 0, ST_FLIGHT = 1, ST_WALK = 2, ST_INTERACT = 3, ST_ESCAPE = 4, ST_DONE = 5 };
enum : int { CNT_EMITTED = 0, CNT_ESCAPED, CNT_LOST, CNT_ABS, CNT_SCA, CNT_FLIGHTS, CNT_CROSS, CNT_N };

struct SrcDev {
  int type;          // 0 point, 1 external field
  int fine[3];       // point source: floor of the position in finest-level units
  float frac[3];     // ... and its fractional part in [0,1)
  float lcdf;        // cumulative luminosity fraction
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
  const float* __restrict__ trow;              // [slots] temperature as table row coordinate
  const float4* __restrict__ opac;             // [nb] (kappa_ext*root_size, albedo, g, kappa_abs)
  const float* __restrict__ cdf;               // [nT][nb] emission inverse-CDF rows
  const float* __restrict__ csrc;              // [nsrc][nb] source spectrum CDFs
  const SrcDev* __restrict__ src;              // [nsrc]
  unsigned long long* next;                    // work-queue head (packet offset within the batch)
  const uint32_t* __restrict__ perm;           // NULL, or the batch's package numbers grouped by source
  const int* __restrict__ axtab;               // NULL (x-fastest root), or [3][N] axis terms of the root slot (bricked)
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

// R19: 24-bit uniform strictly inside (0,1), exact in fp32.
__device__ __forceinline__ float u01(uint32_t x) {
  return ((float)(x >> 8) + 0.5f) * 5.9604644775390625e-8f;
}

__device__ __forceinline__ void draw4(unsigned long long seed, unsigned long long pid, uint32_t k,
                                      uint32_t tag, float u[4]) {
  uint32_t x[4];
  philox4x32_10((uint32_t)seed, (uint32_t)(seed >> 32), (uint32_t)pid, (uint32_t)(pid >> 32), k, tag, x);
  u[0] = u01(x[0]); u[1] = u01(x[1]); u[2] = u01(x[2]); u[3] = u01(x[3]);
}

// first j with cdf[j] >= u
__device__ __forceinline__ int search_cdf(const float* __restrict__ cdf, int n, float u) {
  int lo = 0, hi = n - 1;
  while (lo < hi) {
    int mid = (lo + hi) >> 1;
    if (__ldg(cdf + mid) >= u) hi = mid; else lo = mid + 1;
  }
  return lo;
}

struct Packet {
  float d0, d1, d2;        // direction
  float t0, t1, t2;        // remaining path length (root units) to the exit face of the leaf, per axis
  float td0, td1, td2;     // 1/|d_a|: path length per root-cube edge
  int ix, iy, iz;          // root cube
  int sub;                 // packed sub-cell index (4 bits per axis) when lvl = 1
  int kref;                // refined-cube number when lvl = 1
  int lvl;                 // 0 = in an unrefined root cube, 1 = in a subcube
  int slot;                // leaf slot
  int bin, comp;
  uint32_t k;              // flight number
  unsigned long long pid;
  float tau_rem, u1, u2, u3;
};

__device__ __forceinline__ void set_dir(Packet& p, float a, float b, float c) {
  // R21: a component too small to ever be the exit axis is nudged to 1e-12 (keeps its sign)
  if (fabsf(a) < 1e-12f) a = copysignf(1e-12f, a);
  if (fabsf(b) < 1e-12f) b = copysignf(1e-12f, b);
  if (fabsf(c) < 1e-12f) c = copysignf(1e-12f, c);
  p.d0 = a; p.d1 = b; p.d2 = c;
  p.td0 = __frcp_rn(fabsf(a)); p.td1 = __frcp_rn(fabsf(b)); p.td2 = __frcp_rn(fabsf(c));
}

// t's from the leaf-local position u in [0,1]^3 (h = leaf edge in root units)
__device__ __forceinline__ void set_t_from_local(Packet& p, float ux, float uy, float uz, float h) {
  p.t0 = (p.d0 > 0.f ? 1.f - ux : ux) * h * p.td0;
  p.t1 = (p.d1 > 0.f ? 1.f - uy : uy) * h * p.td1;
  p.t2 = (p.d2 > 0.f ? 1.f - uz : uz) * h * p.td2;
}

// leaf-local position from the t's (inverse of the above), clamped to the leaf
__device__ __forceinline__ void local_from_t(const Packet& p, float h, float& ux, float& uy, float& uz) {
  float ih = 1.f / h;
  float w0 = fminf(1.f, p.t0 * fabsf(p.d0) * ih), w1 = fminf(1.f, p.t1 * fabsf(p.d1) * ih),
        w2 = fminf(1.f, p.t2 * fabsf(p.d2) * ih);
  ux = p.d0 > 0.f ? 1.f - w0 : w0;
  uy = p.d1 > 0.f ? 1.f - w1 : w1;
  uz = p.d2 > 0.f ? 1.f - w2 : w2;
}

__device__ __forceinline__ void isotropic_dir(float u2, float u3, float& a, float& b, float& c) {
  float mu = 2.f * u2 - 1.f;
  float s = sqrtf(fmaxf(0.f, 1.f - mu * mu));
  float sn, cs;
  sincospif(2.f * u3, &sn, &cs);
  a = s * cs; b = s * sn; c = mu;
}

__device__ __forceinline__ float hg_cos(float g, float u) {     // R15
  if (fabsf(g) < 1e-3f) return 2.f * u - 1.f;
  float t = (1.f - g * g) / (1.f - g + 2.f * g * u);
  float c = (1.f + g * g - t * t) / (2.f * g);
  return fminf(1.f, fmaxf(-1.f, c));
}

__device__ __forceinline__ void rotate_dir(float d0, float d1, float d2, float ct, float u3,
                                           float& a, float& b, float& c) {
  float st = sqrtf(fmaxf(0.f, 1.f - ct * ct));
  float sp, cp;
  sincospif(2.f * u3, &sp, &cp);
  float q2 = d0 * d0 + d1 * d1;                 // = 1 - d2^2, without the cancellation
  if (q2 > 1e-12f) {
    float q = sqrtf(q2), iq = 1.f / q;
    a = st * (d0 * d2 * cp - d1 * sp) * iq + d0 * ct;
    b = st * (d1 * d2 * cp + d0 * sp) * iq + d1 * ct;
    c = -st * cp * q + d2 * ct;
  } else {
    a = st * cp; b = st * sp; c = (d2 >= 0.f ? ct : -ct);
  }
  float inv = rsqrtf(a * a + b * b + c * c);
  a *= inv; b *= inv; c *= inv;
}

__device__ __forceinline__ int sub_lin(int sub, int S) {
  return (sub & 15) + S * (((sub >> 4) & 15) + S * ((sub >> 8) & 15));
}

// storage slot of root cube (ix,iy,iz): x-fastest, or the sum of three axis terms (bricked root,
// tables in shared memory)
__device__ __forceinline__ int root_lin(const TransportParams& P, const int* s_ax, int ix, int iy, int iz) {
  if (s_ax) return s_ax[ix] + s_ax[P.N + iy] + s_ax[2 * P.N + iz];
  return ix + P.N * (iy + P.N * iz);
}

// Put a packet whose root cube (ix,iy,iz) and root-local position are known into its leaf.
template <bool TL>
__device__ __forceinline__ void place_in_root(const TransportParams& P, const int* s_ax, Packet& p, float ux, float uy,
                                              float uz) {
  int lin = root_lin(P, s_ax, p.ix, p.iy, p.iz);
  p.lvl = 0; p.slot = lin;
  if (TL) {
    MCRT_CHECK_SLOT(lin);
    int bits = __float_as_int(__ldg(P.rho + lin));
    if (bits < 0) {
      const int S = P.S;
      const float fS = (float)S;
      float vx = ux * fS, vy = uy * fS, vz = uz * fS;
      int sx = min(S - 1, (int)vx), sy = min(S - 1, (int)vy), sz = min(S - 1, (int)vz);
      // R7: direction-aware on a sub-face
      if (p.d0 < 0.f && vx == (float)sx && sx > 0) --sx;
      if (p.d1 < 0.f && vy == (float)sy && sy > 0) --sy;
      if (p.d2 < 0.f && vz == (float)sz && sz > 0) --sz;
      p.lvl = 1; p.kref = bits & 0x7fffffff; p.sub = sx | (sy << 4) | (sz << 8);
      p.slot = P.n3 + p.kref * (S * S * S) + sub_lin(p.sub, S);
      set_t_from_local(p, vx - (float)sx, vy - (float)sy, vz - (float)sz, 1.f / fS);
      return;
    }
  }
  set_t_from_local(p, ux, uy, uz, 1.f);
}

// O4: emission of packet pid.
template <bool TL>
__device__ __forceinline__ void emit_packet(const TransportParams& P, const int* s_ax, Packet& p, const float4* s_opac) {
  float u[4];
  draw4(P.seed, p.pid, 0, kTagEmit, u);
  int s = 0;
  while (s < P.nsrc - 1 && P.src[s].lcdf < u[0]) ++s;
  p.bin = search_cdf(P.csrc + (size_t)s * P.nb, P.nb, u[1]);
  p.comp = 0; p.k = 0;
  const SrcDev& sd = P.src[s];
  const int Sf = TL ? P.S : 1;
  if (sd.type == 0) {
    float a, b, c;
    isotropic_dir(u[2], u[3], a, b, c);
    set_dir(p, a, b, c);
    int f0 = sd.fine[0], f1 = sd.fine[1], f2 = sd.fine[2];
    float r0 = sd.frac[0], r1 = sd.frac[1], r2 = sd.frac[2];
    if (p.d0 < 0.f && r0 == 0.f) { --f0; r0 = 1.f; }        // R7: ceil(x) - 1 for d < 0
    if (p.d1 < 0.f && r1 == 0.f) { --f1; r1 = 1.f; }
    if (p.d2 < 0.f && r2 == 0.f) { --f2; r2 = 1.f; }
    p.ix = f0 / Sf; p.iy = f1 / Sf; p.iz = f2 / Sf;
    int sx = f0 - p.ix * Sf, sy = f1 - p.iy * Sf, sz = f2 - p.iz * Sf;
    int lin = root_lin(P, s_ax, p.ix, p.iy, p.iz);
    p.lvl = 0; p.slot = lin;
    bool refined = false;
    if (TL) {
      MCRT_CHECK_SLOT(lin);
    int bits = __float_as_int(__ldg(P.rho + lin));
      if (bits < 0) {
        refined = true;
        p.lvl = 1; p.kref = bits & 0x7fffffff; p.sub = sx | (sy << 4) | (sz << 8);
        p.slot = P.n3 + p.kref * (Sf * Sf * Sf) + sub_lin(p.sub, Sf);
        set_t_from_local(p, r0, r1, r2, 1.f / (float)Sf);
      }
    }
    if (!refined) {
      float is = 1.f / (float)Sf;
      set_t_from_local(p, ((float)sx + r0) * is, ((float)sy + r1) * is, ((float)sz + r2) * is, 1.f);
    }
  } else {                                                  // R25 external isotropic field
    float v[4];
    draw4(P.seed, p.pid, 1, kTagEmit, v);
    int f = min(5, (int)(6.f * v[0]));
    int ax = f >> 1, side = f & 1;
    float mu = sqrtf(u[2]);
    float st = sqrtf(fmaxf(0.f, 1.f - mu * mu));
    float sn, cs;
    sincospif(2.f * u[3], &sn, &cs);
    float dn = side == 0 ? mu : -mu, e1 = st * cs, e2 = st * sn;     // normal, axis+1, axis+2
    float fN = (float)P.N;
    float x1 = v[1] * fN, x2 = v[2] * fN;
    int i1 = min(P.N - 1, (int)x1), i2 = min(P.N - 1, (int)x2);
    float l1 = x1 - (float)i1, l2 = x2 - (float)i2;
    if (e1 < 0.f && l1 == 0.f && i1 > 0) { --i1; l1 = 1.f; }
    if (e2 < 0.f && l2 == 0.f && i2 > 0) { --i2; l2 = 1.f; }
    int in = side == 0 ? 0 : P.N - 1;
    float ln = side == 0 ? 0.f : 1.f;
    float ux, uy, uz;
    if (ax == 0)      { set_dir(p, dn, e1, e2); p.ix = in; p.iy = i1; p.iz = i2; ux = ln; uy = l1; uz = l2; }
    else if (ax == 1) { set_dir(p, e2, dn, e1); p.iy = in; p.iz = i1; p.ix = i2; uy = ln; uz = l1; ux = l2; }
    else              { set_dir(p, e1, e2, dn); p.iz = in; p.ix = i1; p.iy = i2; uz = ln; ux = l1; uy = l2; }
    place_in_root<TL>(P, s_ax, p, ux, uy, uz);
  }
}

// One crossing of the cell walk (O5).  Returns false when the packet stops walking
// (interaction or escape; state says which).
template <bool TL>
__device__ __forceinline__ bool walk_step(const TransportParams& P, const int* s_ax, Packet& p, float kx, int& state,
                                          uint32_t& crossings) {
  MCRT_CHECK_SLOT(p.slot);
  float rho = __ldg(P.rho + p.slot);
  float tmin = fminf(p.t0, fminf(p.t1, p.t2));
  float alpha = rho * kx;
  float dtau = alpha * tmin;
  if (dtau >= p.tau_rem && alpha > 0.f) {                    // interaction inside this leaf
    float dl = fminf(tmin, p.tau_rem / alpha);
    p.t0 -= dl; p.t1 -= dl; p.t2 -= dl;
    state = ST_INTERACT;
    return false;
  }
  p.tau_rem -= dtau;
  p.t0 -= tmin; p.t1 -= tmin; p.t2 -= tmin;
  ++crossings;
  const bool a0 = p.t0 <= 0.f;                               // exactly 0 for the argmin; ties -> lowest axis
  const bool a1 = !a0 && p.t1 <= 0.f;
  const bool a2 = !a0 && !a1;
  const float dsel = a0 ? p.d0 : (a1 ? p.d1 : p.d2);
  const int step = dsel > 0.f ? 1 : -1;
  if (TL && p.lvl) {
    const int S = P.S;
    const float hs = 1.f / (float)S;
    const int sh = a0 ? 0 : (a1 ? 4 : 8);
    int f = ((p.sub >> sh) & 15) + step;
    if ((unsigned)f < (unsigned)S) {                         // next subcube of the same root cube
      p.sub = (p.sub & ~(15 << sh)) | (f << sh);
      if (a0) p.t0 = p.td0 * hs; else if (a1) p.t1 = p.td1 * hs; else p.t2 = p.td2 * hs;
      p.slot = P.n3 + p.kref * (S * S * S) + sub_lin(p.sub, S);
      return true;
    }
    // leaving the refined root cube through axis `a`
    if (a0) p.ix += step; else if (a1) p.iy += step; else p.iz += step;
    int coord = a0 ? p.ix : (a1 ? p.iy : p.iz);
    if ((unsigned)coord >= (unsigned)P.N) { state = ST_ESCAPE; return false; }
    int lin = root_lin(P, s_ax, p.ix, p.iy, p.iz);
    MCRT_CHECK_SLOT(lin);
    int bits = __float_as_int(__ldg(P.rho + lin));
    if (bits < 0) {                                          // refined -> refined: sub faces line up
      int nf = step > 0 ? 0 : S - 1;
      p.sub = (p.sub & ~(15 << sh)) | (nf << sh);
      p.kref = bits & 0x7fffffff;
      if (a0) p.t0 = p.td0 * hs; else if (a1) p.t1 = p.td1 * hs; else p.t2 = p.td2 * hs;
      p.slot = P.n3 + p.kref * (S * S * S) + sub_lin(p.sub, S);
      return true;
    }
    // refined -> unrefined: extend the other axes' t to the root faces
    int sx = p.sub & 15, sy = (p.sub >> 4) & 15, sz = (p.sub >> 8) & 15;
    float r0 = (float)(p.d0 > 0.f ? S - 1 - sx : sx), r1 = (float)(p.d1 > 0.f ? S - 1 - sy : sy),
          r2 = (float)(p.d2 > 0.f ? S - 1 - sz : sz);
    p.t0 = a0 ? p.td0 : p.t0 + r0 * p.td0 * hs;
    p.t1 = a1 ? p.td1 : p.t1 + r1 * p.td1 * hs;
    p.t2 = a2 ? p.td2 : p.t2 + r2 * p.td2 * hs;
    p.lvl = 0; p.slot = lin;
    return true;
  }
  // root level
  p.ix += a0 ? step : 0; p.iy += a1 ? step : 0; p.iz += a2 ? step : 0;
  p.t0 = a0 ? p.td0 : p.t0; p.t1 = a1 ? p.td1 : p.t1; p.t2 = a2 ? p.td2 : p.t2;
  int coord = a0 ? p.ix : (a1 ? p.iy : p.iz);
  if ((unsigned)coord >= (unsigned)P.N) { state = ST_ESCAPE; return false; }
  int lin = root_lin(P, s_ax, p.ix, p.iy, p.iz);
  p.slot = lin;
  if (TL) {
    MCRT_CHECK_SLOT(lin);
    int bits = __float_as_int(__ldg(P.rho + lin));
    if (bits < 0) {                                          // unrefined -> refined: descend
      const int S = P.S;
      const float fS = (float)S, hs = 1.f / fS;
      // distance (root units) to the root exit face along each other axis -> subcube index
      float w0 = fminf(p.t0 * fabsf(p.d0), 1.f), w1 = fminf(p.t1 * fabsf(p.d1), 1.f),
            w2 = fminf(p.t2 * fabsf(p.d2), 1.f);
      int m0 = min(S - 1, (int)(w0 * fS)), m1 = min(S - 1, (int)(w1 * fS)), m2 = min(S - 1, (int)(w2 * fS));
      int sx = p.d0 > 0.f ? S - 1 - m0 : m0, sy = p.d1 > 0.f ? S - 1 - m1 : m1,
          sz = p.d2 > 0.f ? S - 1 - m2 : m2;
      int en = step > 0 ? 0 : S - 1;
      if (a0) sx = en; else if (a1) sy = en; else sz = en;
      p.t0 = a0 ? p.td0 * hs : fmaxf(0.f, p.t0 - (float)m0 * p.td0 * hs);
      p.t1 = a1 ? p.td1 * hs : fmaxf(0.f, p.t1 - (float)m1 * p.td1 * hs);
      p.t2 = a2 ? p.td2 * hs : fmaxf(0.f, p.t2 - (float)m2 * p.td2 * hs);
      p.lvl = 1; p.kref = bits & 0x7fffffff; p.sub = sx | (sy << 4) | (sz << 8);
      p.slot = P.n3 + p.kref * (S * S * S) + sub_lin(p.sub, S);
    }
  }
  return true;
}

template <bool TL>
// compiled for 5 resident blocks per SM (48 registers): c2 6.53 -> 6.41 ms, c3 15.9 -> 14.7 ms per
// 2^22-package launch against the 64-register build (profiles/r01_summary.md)
__global__ void __launch_bounds__(256, 5) k_transport(const TransportParams P) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  float4* s_opac = reinterpret_cast<float4*>(smem_raw);                    // [nb]
  uint32_t* s_sed = reinterpret_cast<uint32_t*>(s_opac + P.nb);             // [3*nb]
  uint32_t* s_emit = s_sed + 3 * P.nb;                                      // [nb]
  int* s_ax = P.axtab ? reinterpret_cast<int*>(s_emit + P.nb) : nullptr;    // [3*N] (bricked root only)
  if (s_ax) for (int i = threadIdx.x; i < 3 * P.N; i += blockDim.x) s_ax[i] = P.axtab[i];
  for (int i = threadIdx.x; i < P.nb; i += blockDim.x) { s_opac[i] = P.opac[i]; s_emit[i] = 0; }
  for (int i = threadIdx.x; i < 3 * P.nb; i += blockDim.x) s_sed[i] = 0;
  __syncthreads();

  const unsigned lane = threadIdx.x & 31;
  const unsigned lt_mask = (1u << lane) - 1u;
  uint32_t cnt[CNT_N];
#pragma unroll
  for (int i = 0; i < CNT_N; ++i) cnt[i] = 0;

  Packet p;
  p.pid = 0; p.k = 0; p.bin = 0; p.comp = 0; p.slot = 0; p.lvl = 0; p.sub = 0; p.kref = 0;
  p.ix = p.iy = p.iz = 0;
  p.d0 = p.d1 = p.d2 = 1.f; p.t0 = p.t1 = p.t2 = 0.f; p.td0 = p.td1 = p.td2 = 1.f;
  p.tau_rem = 0.f; p.u1 = p.u2 = p.u3 = 0.f;
  float kx = 0.f;
  int state = ST_FETCH;

  for (;;) {
    // ---- a8: refill finished lanes from the work queue (one atomic per warp per refill) ----
    unsigned need = __ballot_sync(kFull, state == ST_FETCH);
    if (need) {
      unsigned long long base = 0;
      if (lane == 0) base = atomicAdd(P.next, (unsigned long long)__popc(need));
      base = __shfl_sync(kFull, base, 0);
      if (state == ST_FETCH) {
        unsigned long long my = base + (unsigned long long)__popc(need & lt_mask);
        if (my < P.count) {
          p.pid = P.first + (P.perm ? (unsigned long long)__ldg(P.perm + my) : my);
          emit_packet<TL>(P, s_ax, p, s_opac);              // a1
          kx = s_opac[p.bin].x;
          ++cnt[CNT_EMITTED];
          atomicAdd(&s_emit[p.bin], 1u);
          state = ST_FLIGHT;
        } else {
          state = ST_DONE;
        }
      }
    }
    if (__all_sync(kFull, state == ST_DONE)) break;

    // ---- a2: free-flight optical depth ----
    if (state == ST_FLIGHT) {
      if (p.k >= kMaxFlights) {                              // R20
        ++cnt[CNT_LOST];
        state = ST_FETCH;
      } else {
        float u[4];
        draw4(P.seed, p.pid, p.k, kTagFlight, u);
        p.tau_rem = -logf(u[0]);
        p.u1 = u[1]; p.u2 = u[2]; p.u3 = u[3];
        ++cnt[CNT_FLIGHTS];
        state = ST_WALK;
      }
    }

    // ---- a3: cell walk, up to kWalkChunk crossings ----
    if (state == ST_WALK) {
#pragma unroll 1
      for (int it = 0; it < kWalkChunk; ++it)
        if (!walk_step<TL>(P, s_ax, p, kx, state, cnt[CNT_CROSS])) break;
    }

    // ---- a4..a6: interaction ----
    if (state == ST_INTERACT) {
      const float4 op = s_opac[p.bin];
      const float h = (TL && p.lvl) ? 1.f / (float)P.S : 1.f;
      float ux, uy, uz;
      local_from_t(p, h, ux, uy, uz);
      float a, b, c;
      if (p.u1 < op.y) {                                     // scatter (R16)
        ++cnt[CNT_SCA];
        float ct = hg_cos(op.z, p.u2);
        rotate_dir(p.d0, p.d1, p.d2, ct, p.u3, a, b, c);
        if (p.comp == 0) p.comp = 1;
      } else {                                               // absorb + re-emit (Eqn 11.67)
        ++cnt[CNT_ABS];
        // a6: warp-aggregated integer tally: one atomic per distinct leaf per warp
        MCRT_CHECK_SLOT(p.slot);
        unsigned peers = __match_any_sync(__activemask(), p.slot);
        if ((int)lane == __ffs(peers) - 1)
          atomicAdd(P.tally + p.slot, (unsigned long long)__popc(peers));
        float tr = __ldg(P.trow + p.slot);                   // T frozen = T before absorption
        float r[4];
        draw4(P.seed, p.pid, p.k, kTagReemit, r);
        int k0 = min(P.nT - 1, (int)tr);
        float w = tr - (float)k0;
        int row = (r[1] < w && k0 + 1 < P.nT) ? k0 + 1 : k0;  // R11 stochastic row choice
        p.bin = search_cdf(P.cdf + (size_t)row * P.nb, P.nb, r[0]);
        kx = s_opac[p.bin].x;
        isotropic_dir(r[2], r[3], a, b, c);
        p.comp = 2;
      }
      set_dir(p, a, b, c);
      set_t_from_local(p, ux, uy, uz, h);
      ++p.k;
      state = ST_FLIGHT;
    }

    // ---- a7: escape -> SED ----
    if (state == ST_ESCAPE) {
      if (P.obs.n_mu | P.obs.n_pix) {                        // exit point from the position-free state
        const float h = (TL && p.lvl) ? 1.f / (float)P.S : 1.f;
        float ux, uy, uz;
        local_from_t(p, h, ux, uy, uz);
        const int sx = (TL && p.lvl) ? (p.sub & 15) : 0, sy = (TL && p.lvl) ? ((p.sub >> 4) & 15) : 0,
                  sz = (TL && p.lvl) ? ((p.sub >> 8) & 15) : 0;
        const float fN = (float)P.N;
        const float x = (unsigned)p.ix >= (unsigned)P.N ? (p.ix < 0 ? 0.f : fN) : (float)p.ix + ((float)sx + ux) * h;
        const float y = (unsigned)p.iy >= (unsigned)P.N ? (p.iy < 0 ? 0.f : fN) : (float)p.iy + ((float)sy + uy) * h;
        const float z = (unsigned)p.iz >= (unsigned)P.N ? (p.iz < 0 ? 0.f : fN) : (float)p.iz + ((float)sz + uz) * h;
        tally_observer(P, x, y, z, p.d0, p.d1, p.d2, p.bin, p.comp);
      }
      atomicAdd(&s_sed[p.comp * P.nb + p.bin], 1u);
      ++cnt[CNT_ESCAPED];
      state = ST_FETCH;
    }
  }

  // ---- flush block-private tallies ----
#pragma unroll
  for (int i = 0; i < CNT_N; ++i) {
    unsigned long long v = cnt[i];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(kFull, v, o);
    if (lane == 0 && v) atomicAdd(P.counters + i, v);
  }
  __syncthreads();
  for (int i = threadIdx.x; i < 3 * P.nb; i += blockDim.x)
    if (s_sed[i]) atomicAdd(P.sed + i, (unsigned long long)s_sed[i]);
  for (int i = threadIdx.x; i < P.nb; i += blockDim.x)
    if (s_emit[i]) atomicAdd(P.emit_bin + i, (unsigned long long)s_emit[i]);
}


// ---- a8, several sources: hand the packages out GROUPED BY SOURCE ----------------------------
// Packages of one source cross the same neighbourhood, so when the packages in flight share a
// source the L2 serves far more of their density gathers (profiles/r01_summary.md: 512^3 cube,
// one source at a time 1.5-1.8e11 crossings/s against 1.17e11 with the eleven sources mixed);
// packages that also start in the same direction share their whole first flight.
// The source of package i is the first decision of its emission (O4: u0 of its EMIT block), so a
// pre-pass can group the batch's package numbers by source: count, exclusive scan, scatter.  The
// order inside a group is arbitrary; integer tallies make the results independent of it.
constexpr int kMaxOrderedSources = 2048;

// group key of a package: its source, refined by where it starts to fly: sub = 128 (32) bins, 8 x 16
// (4 x 8) in (mu, phi) of the emission direction for a point source, face x 2 x 2 tiles for the
// external field
__device__ __forceinline__ int group_of(const TransportParams& P, unsigned long long pid, int sub) {
  uint32_t x[4];
  philox4x32_10((uint32_t)P.seed, (uint32_t)(P.seed >> 32), (uint32_t)pid, (uint32_t)(pid >> 32), 0u, kTagEmit, x);
  const float u0 = u01(x[0]);
  int s = 0;
  while (s < P.nsrc - 1 && P.src[s].lcdf < u0) ++s;
  if (sub == 1) return s;
  int b;
  if (P.src[s].type == 0) {
    b = sub == 32 ? min(3, (int)(4.f * u01(x[2]))) * 8 + min(7, (int)(8.f * u01(x[3])))
                  : min(7, (int)(8.f * u01(x[2]))) * 16 + min(15, (int)(16.f * u01(x[3])));
  } else {
    philox4x32_10((uint32_t)P.seed, (uint32_t)(P.seed >> 32), (uint32_t)pid, (uint32_t)(pid >> 32), 1u, kTagEmit, x);
    b = min(5, (int)(6.f * u01(x[0]))) * 4 + (u01(x[1]) >= 0.5f ? 1 : 0) + (u01(x[2]) >= 0.5f ? 2 : 0);
  }
  return s * sub + b;
}

// counts[g] += packages of group g (cursor == NULL), or perm[cursor[g]++] = package number
__global__ void k_group_by_source(const TransportParams P, const int sub, unsigned int* __restrict__ counts,
                                  unsigned int* __restrict__ cursor, uint32_t* __restrict__ perm) {
  extern __shared__ unsigned int s_cnt[];                    // [2 * ngroups]: block histogram, block bases
  const int ng = P.nsrc * sub;
  for (int i = threadIdx.x; i < 2 * ng; i += blockDim.x) s_cnt[i] = 0;
  __syncthreads();
  const unsigned long long per_block = (P.count + gridDim.x - 1) / gridDim.x;
  const unsigned long long lo = per_block * blockIdx.x, hi = min(P.count, lo + per_block);
  for (unsigned long long i = lo + threadIdx.x; i < hi; i += blockDim.x)
    atomicAdd(&s_cnt[group_of(P, P.first + i, sub)], 1u);
  __syncthreads();
  if (!cursor) {
    for (int i = threadIdx.x; i < ng; i += blockDim.x)
      if (s_cnt[i]) atomicAdd(&counts[i], s_cnt[i]);
    return;
  }
  for (int i = threadIdx.x; i < ng; i += blockDim.x) {       // reserve this block's range in every group
    s_cnt[ng + i] = s_cnt[i] ? atomicAdd(&cursor[i], s_cnt[i]) : 0u;
    s_cnt[i] = 0;
  }
  __syncthreads();
  for (unsigned long long i = lo + threadIdx.x; i < hi; i += blockDim.x) {
    const int g = group_of(P, P.first + i, sub);
    perm[s_cnt[ng + g] + atomicAdd(&s_cnt[g], 1u)] = (uint32_t)i;
  }
}

// cursor[s] = sum of counts[0..s) (one block; nsrc <= kMaxOrderedSources)
__global__ void k_scan_sources(const unsigned int* __restrict__ counts, unsigned int* __restrict__ cursor, int nsrc) {
  if (threadIdx.x == 0) {
    unsigned int acc = 0;
    for (int s = 0; s < nsrc; ++s) { cursor[s] = acc; acc += counts[s]; }
  }
}

}  // namespace mcrt
