// pah.cuh -- transiently heated PAH (row f2 of SURVEY.md 8(f); "extended to the
// treatment of transiently heated PAHs", L45 Fig. 3, L49; readings R35..R40).
//
// One PAH kind per context, declared by mcrt_set_pah as a share kappa_PAH,j of the mix's absorption.
// In the transport kernel an absorbed package is taken by the PAH with probability
// q_j = kappa_PAH,j / kappa_abs,j (R36); it is then booked on the per-leaf, per-bin PAH tally and
// re-emitted from the leaf's PAH emission spectrum instead of kappa_nu B_nu(T_leaf).  At the end of a
// batch k_pah_update turns every leaf's absorbed spectrum into photon absorption rates of one molecule
// (R40), solves the stationary temperature distribution P(T) (R38: thermal-continuous cooling, photon
// jumps shared linearly between the two bracketing enthalpy states) and stores the emission CDF
// sum_k P_k C_j B_j(T_k) dnu_j (R39).  All of it in fp64: P(T) spans hundreds of orders of magnitude.
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

#include "tables.cuh"

namespace mcrt {

#define MCRT_M_CARBON 1.99264687992e-23     // g, 12 atomic mass units (CODATA 2018)
#define MCRT_PI 3.14159265358979323846

struct PahDev {
  int nC, K, nb;
  double fP, theta;
  const double* __restrict__ E;       // [nb] photon energy h nu_j
  const double* __restrict__ U;       // [K] enthalpy of state k
  const double* __restrict__ Lam;     // [K] cooling power of one molecule in state k
  const double* __restrict__ W;       // [K][nb] C_j dnu_j B_j(T_k)
  const float* __restrict__ W32;      // the same rounded to fp32 (emission sums of the fast kernel: 6e-8 relative)
  const int* __restrict__ J;          // [K][K] JT[i][f] = number of bins with E_j >= U_f - U_i (f > i)
};

// R37: synthetic enthalpy law, U(T) = 3 N k Theta (x - atan x), x = T / Theta
__device__ __forceinline__ double pah_enthalpy(int nC, double theta, double T) {
  const double x = T / theta;
  return 3.0 * nC * MCRT_K_BOLTZ * theta * (x - atan(x));
}

// kappa left for the grains in equilibrium, the PAH share q_j, cross-section per molecule, photon energies
__global__ void k_pah_split(int nb, const double* __restrict__ kabs_all, const float* __restrict__ kabs_pah,
                            const double* __restrict__ nu, int nC, double fP, double* __restrict__ kabs_eq,
                            float* __restrict__ q, double* __restrict__ Cmol, double* __restrict__ E) {
  int j = blockIdx.x * blockDim.x + threadIdx.x;
  if (j >= nb) return;
  double kp = fmin((double)kabs_pah[j], kabs_all[j]);
  if (!(kp > 0)) kp = 0;
  kabs_eq[j] = kabs_all[j] - kp;
  q[j] = kabs_all[j] > 0 ? (float)(kp / kabs_all[j]) : 0.f;
  Cmol[j] = kp * nC * MCRT_M_CARBON / fP;
  E[j] = MCRT_H_PLANCK * nu[j];
}

// one block per state k: T_k, U_k, W[k][.], Lambda_k (serial sum in bin order, as the oracle's)
__global__ void k_pah_states(int nb, int K, double T_lo, double T_hi, int nC, double theta,
                             const double* __restrict__ nu, const double* __restrict__ dnu,
                             const double* __restrict__ Cmol, double* __restrict__ Tk, double* __restrict__ U,
                             double* __restrict__ Lam, double* __restrict__ W, float* __restrict__ W32) {
  const int k = blockIdx.x;
  const double T = T_lo * pow(T_hi / T_lo, (double)k / (double)(K - 1));
  for (int j = threadIdx.x; j < nb; j += blockDim.x) {
    const double w = Cmol[j] * planck_nu(nu[j], T) * dnu[j];
    W[(size_t)k * nb + j] = w;
    W32[(size_t)k * nb + j] = (float)w;
  }
  __syncthreads();
  if (threadIdx.x == 0) {
    double acc = 0;
    for (int j = 0; j < nb; ++j) acc += W[(size_t)k * nb + j];
    Tk[k] = T; U[k] = pah_enthalpy(nC, theta, T); Lam[k] = 4.0 * MCRT_PI * acc;
  }
}

// JT[i][f] = #{ j : E_j >= U_f - U_i } (E descends with j, so this is an upper bound by bisection); stored with f
// running fastest: the update kernel reads one column i for 32 consecutive states f at a time
__global__ void k_pah_thresholds(int nb, int K, const double* __restrict__ E, const double* __restrict__ U,
                                 int* __restrict__ J) {
  const int idx = blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= K * K) return;
  const int f = idx / K, i = idx % K;
  const double e = U[f] - U[i];
  int lo = 0, hi = nb;                                       // bins [0, lo) have E_j >= e
  while (lo < hi) { int mid = (lo + hi) >> 1; if (E[mid] >= e) lo = mid + 1; else hi = mid; }
  J[(size_t)i * K + f] = lo;
}

// emission CDF of a molecule sitting in state 0 (what every leaf starts with; R10's analogue)
__global__ void k_pah_cold_row(int nb, const double* __restrict__ W, float* __restrict__ row) {
  if (threadIdx.x || blockIdx.x) return;
  double tot = 0;
  for (int j = 0; j < nb; ++j) tot += W[j];
  double acc = 0;
  for (int j = 0; j < nb; ++j) { acc += W[j]; row[j] = (j == nb - 1 || !(tot > 0)) ? 1.f : (float)(acc / tot); }
}
__global__ void k_pah_fill_rows(const float* __restrict__ row, float* __restrict__ cdf, long long slots, int nb) {
  long long e = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (e < slots * nb) cdf[e] = row[e % nb];
}

__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}

// a9 for the PAH: one warp per leaf.  Shared memory per warp: cum[nb] = running sums over the bins of the photon
// rates and of rate x energy (double2), X[K] (doubles).
//
// The recursion X_f = sum_{i<f} B(f,i) X_i / A_f is a forward substitution.  It runs COLUMN by column, 32 states f
// (one per lane) at a time: each lane owns the partial sum of its own f and adds B(f,i) X_i as soon as X_i is final
// -- all 32 lanes work on the columns of earlier blocks, and inside a block X_i is handed on by one shuffle.  No warp
// reduction and no barrier per state (the row-by-row form needed both 127 times per leaf).  B(f,i) takes the rate
// sums at two thresholds, E >= U_f - U_i and E >= U_{f-1} - U_i; the second is the first of the lane below, so it
// arrives by shuffle as well, and the threshold table is stored transposed (JT[i][f]: consecutive lanes, one line).
// only_slot >= 0: just that leaf, and its P(T) is also written to P_out[K] (read-out for inspection).
// leaves per fetch from the work queue (measured on the 64^3 sphere, 128 states, sixth batch: 1 -> 2.15 ms, 2 -> 2.20,
// 4 -> 2.30, 32 -> 3.50) and resident blocks per SM the kernel is compiled for (8 -> 2.60 ms, 10 -> 2.30, 12 -> 2.34 at 4 leaves)
constexpr int kPahChunk = 1;
constexpr int kPahMinBlocks = 10;
__device__ __host__ __forceinline__ int pah_warp_doubles(int nb, int K) { return 2 * (nb + 1) + K + (K & 1); }

__global__ void __launch_bounds__(128, kPahMinBlocks) k_pah_update(const PahDev D, const float* __restrict__ rho,
                                                   const uint32_t* __restrict__ cnt, float* __restrict__ cdf,
                                                   long long slots, long long n3, double coef /* L_tot / N_cum */,
                                                   double v_root, double inv_s3, long long only_slot,
                                                   double* __restrict__ P_out, unsigned long long* __restrict__ next_leaf) {
  extern __shared__ double2 s_pah2[];
  double* s_pah = reinterpret_cast<double*>(s_pah2);
  const int nb = D.nb, K = D.K;
  const unsigned full = 0xffffffffu;
  const int lane = threadIdx.x & 31, wib = threadIdx.x >> 5, wpb = blockDim.x >> 5;
  double2* cum = reinterpret_cast<double2*>(s_pah + (size_t)wib * pah_warp_doubles(nb, K));   // cum[n] = (sum R, sum R E) over the
  double* X = reinterpret_cast<double*>(cum + nb + 1);                                        // first n bins; cum[0] = 0
  double* em = reinterpret_cast<double*>(cum);               // later: emission per bin (the rate sums are no longer needed)
  // The leaves are handed out from a work queue: their cost differs by orders of magnitude (a leaf that absorbed
  // nothing costs one look, the others the whole solve), and the active ones cluster in space.
  (void)wpb;
  long long chunk = 0, s = only_slot >= 0 ? only_slot : 0;
  int left = only_slot >= 0 ? 1 : 0;
  for (;; ++s) {
    if (left == 0) {
      if (only_slot >= 0) break;
      if (lane == 0) chunk = (long long)atomicAdd(next_leaf, (unsigned long long)kPahChunk);
      chunk = __shfl_sync(0xffffffffu, chunk, 0);
      if (chunk >= slots) break;
      s = chunk;
      left = (int)min((long long)kPahChunk, slots - chunk);
    }
    --left;
    const float r = rho[s];
    if (!(r > 0.f)) continue;                                // empty leaf or refined-cube marker
    const uint32_t* c = cnt + (size_t)s * nb;
    // R40: rates of one molecule, and their running sums over the bins (E descends with j)
    const double n_mol = D.fP * (double)r * v_root * (s >= n3 ? inv_s3 : 1.0) / (D.nC * MCRT_M_CARBON);
    double carryN = 0, carryM = 0;
    bool any = false;
    for (int j0 = 0; j0 < nb; j0 += 32) {
      const int j = j0 + lane;
      const uint32_t cj = j < nb ? c[j] : 0u;
      any = any || cj;
      double Rj = j < nb ? (double)cj * coef / (D.E[j] * n_mol) : 0.0;
      double Mj = j < nb ? Rj * D.E[j] : 0.0;
#pragma unroll
      for (int o = 1; o < 32; o <<= 1) {                     // inclusive warp scan
        const double a = __shfl_up_sync(full, Rj, o), b = __shfl_up_sync(full, Mj, o);
        if (lane >= o) { Rj += a; Mj += b; }
      }
      if (j < nb) cum[j + 1] = make_double2(carryN + Rj, carryM + Mj);
      carryN += __shfl_sync(full, Rj, 31);
      carryM += __shfl_sync(full, Mj, 31);
    }
    if (!__any_sync(full, any)) continue;                    // nothing absorbed: the cold row stays
    if (lane == 0) cum[0] = make_double2(0.0, 0.0);
    __syncwarp();
    // R38: X_0 = 1, X_f = sum_{i<f} B(f,i) X_i / A(f-1,f),
    // B(f,i) = N(E >= a+b) + [M(a <= E < a+b) - a N(a <= E < a+b)] / b,  a = U_{f-1} - U_i, b = U_f - U_{f-1}
    // (JT[i][i] = nb: the threshold of the lane below f = i + 1 is "every bin", as it must be for a = 0)
    for (int fb = 0; fb < K; fb += 32) {
      const int f = fb + lane;
      const bool valid = f >= 1 && f < K;
      const double Uf1 = valid ? D.U[f - 1] : 0.0;
      const double bf = valid ? D.U[f] - Uf1 : 1.0;
      const double inv_b = 1.0 / bf;
      const double inv_A = valid ? bf / D.Lam[f] : 1.0;      // A(f-1,f) = Lambda_f / b
      double part = f == 0 ? 1.0 : 0.0;                      // (X_0 = 1)
      const int* JTf = D.J + min(f, K - 1);                  // this lane's entry of column i: JTf[i * K]
      // columns of earlier blocks: every lane adds its B(f,i) X_i
      for (int i = 0; i < fb; ++i) {
        const double xi = X[i];
        if (xi == 0.0) continue;                             // (the same for all lanes)
        const double2 hi = cum[__ldg(JTf + (size_t)i * K)];  // bins with E >= a + b: they land at or above f
        double loN = __shfl_up_sync(full, hi.x, 1), loM = __shfl_up_sync(full, hi.y, 1);   // threshold a: the lane below
        if (lane == 0) {                                     // ... which belongs to the block before
          const double2 lo = cum[__ldg(JTf + (size_t)i * K - 1)];
          loN = lo.x; loM = lo.y;
        }
        const double a = Uf1 - __ldg(D.U + i);
        const double B = fma(fma(-a, loN - hi.x, loM - hi.y), inv_b, hi.x);
        if (valid) part = fma(B, xi, part);
      }
      // the block's own columns: X_i becomes final, is handed on, and the lanes above it add their share
      const int i_end = min(fb + 32, K);
      for (int i = fb; i < i_end; ++i) {
        double xi = __shfl_sync(full, part * inv_A, i - fb);
        if (xi > 1e200) {                                    // rescale (the normalisation comes last)
          __syncwarp();
          for (int k = lane; k < i; k += 32) X[k] *= 1e-200;
          part *= 1e-200;
          xi *= 1e-200;
        }
        if (lane == i - fb) X[i] = xi;
        if (xi == 0.0) continue;
        const double2 hi = cum[f >= i && f < K ? __ldg(JTf + (size_t)i * K) : 0];
        const double loN = __shfl_up_sync(full, hi.x, 1), loM = __shfl_up_sync(full, hi.y, 1);
        const double a = Uf1 - __ldg(D.U + i);
        const double B = fma(fma(-a, loN - hi.x, loM - hi.y), inv_b, hi.x);
        if (valid && f > i) part = fma(B, xi, part);
      }
      __syncwarp();
    }
    __syncwarp();
    double tot = 0;
    for (int k = lane; k < K; k += 32) tot += X[k];
    tot = warp_sum(tot);
    if (P_out && only_slot >= 0)
      for (int k = lane; k < K; k += 32) P_out[k] = X[k] / tot;
    __syncwarp();
    // R39: emission CDF.  P_k replaces X_k; the emission per bin goes where the rate sums were.
    for (int k = lane; k < K; k += 32) X[k] /= tot;
    __syncwarp();
    float* row = cdf + (size_t)s * nb;
    double etot = 0;
    for (int j0 = 4 * lane; j0 < nb; j0 += 128) {            // W rounded to fp32 (L1-resident), four bins per lane and turn
      double e0 = 0, e1 = 0, e2 = 0, e3 = 0;
      if (j0 + 3 < nb && (nb & 3) == 0) {
        for (int k = 0; k < K; ++k) {
          const double pk = X[k];
          const float4 w = __ldg(reinterpret_cast<const float4*>(D.W32 + (size_t)k * nb + j0));
          e0 += pk * (double)w.x; e1 += pk * (double)w.y; e2 += pk * (double)w.z; e3 += pk * (double)w.w;
        }
        em[j0] = e0; em[j0 + 1] = e1; em[j0 + 2] = e2; em[j0 + 3] = e3;
        etot += (e0 + e1) + (e2 + e3);
      } else {
        for (int j = j0; j < min(nb, j0 + 4); ++j) {
          double e = 0;
          for (int k = 0; k < K; ++k) e += X[k] * (double)__ldg(D.W32 + (size_t)k * nb + j);
          em[j] = e;
          etot += e;
        }
      }
    }
    etot = warp_sum(etot);
    __syncwarp();
    double carry = 0;
    for (int j0 = 0; j0 < nb; j0 += 32) {
      const int j = j0 + lane;
      double e = j < nb ? em[j] : 0.0;
#pragma unroll
      for (int o = 1; o < 32; o <<= 1) {
        const double a = __shfl_up_sync(full, e, o);
        if (lane >= o) e += a;
      }
      if (j < nb) row[j] = (j == nb - 1 || !(etot > 0)) ? 1.f : (float)((carry + e) / etot);
      carry += __shfl_sync(full, e, 31);
    }
    __syncwarp();
  }
}

// per-leaf rows (PAH tallies, emission CDFs): storage order -> the caller's slot order
template <typename T>
__global__ void k_rows_store_to_ext(const T* __restrict__ store, T* __restrict__ ext, LayoutU lay, long long n3, int nb) {
  long long e = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (e >= n3 * nb) return;
  const long long cell = e / nb;
  const int j = (int)(e % nb);
  int ix = (int)(cell % lay.N), iy = (int)((cell / lay.N) % lay.N), iz = (int)(cell / ((long long)lay.N * lay.N));
  ext[e] = store[(size_t)slot_of(lay, ix, iy, iz) * nb + j];
}

// packet-sharded batches: the PAH counts of one batch (summed over ranks) join the cumulative ones
__global__ void k_add_u32(uint32_t* __restrict__ acc, const uint32_t* __restrict__ delta, long long n) {
  const long long stride = (long long)gridDim.x * blockDim.x;
  for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += stride) {
    const uint32_t d = delta[i];
    if (d) acc[i] += d;
  }
}

}  // namespace mcrt
