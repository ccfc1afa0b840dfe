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
  const int* __restrict__ J;          // [K][K] J[f][i] = number of bins with E_j >= U_f - U_i (f > i)
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

// J[f][i] = #{ j : E_j >= U_f - U_i } (E descends with j, so this is an upper bound by bisection)
__global__ void k_pah_thresholds(int nb, int K, const double* __restrict__ E, const double* __restrict__ U,
                                 int* __restrict__ J) {
  const int idx = blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= K * K) return;
  const int f = idx / K, i = idx % K;
  const double e = U[f] - U[i];
  int lo = 0, hi = nb;                                       // bins [0, lo) have E_j >= e
  while (lo < hi) { int mid = (lo + hi) >> 1; if (E[mid] >= e) lo = mid + 1; else hi = mid; }
  J[idx] = lo;
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

// a9 for the PAH: one warp per leaf.  Shared memory per warp: cumN[nb], cumM[nb], X[K] (doubles).
// only_slot >= 0: just that leaf, and its P(T) is also written to P_out[K] (read-out for inspection).
__global__ void __launch_bounds__(128) k_pah_update(const PahDev D, const float* __restrict__ rho,
                                                   const uint32_t* __restrict__ cnt, float* __restrict__ cdf,
                                                   long long slots, long long n3, double coef /* L_tot / N_cum */,
                                                   double v_root, double inv_s3, long long only_slot,
                                                   double* __restrict__ P_out) {
  extern __shared__ double s_pah[];
  const int nb = D.nb, K = D.K;
  const int lane = threadIdx.x & 31, wib = threadIdx.x >> 5, wpb = blockDim.x >> 5;
  double* cumN = s_pah + (size_t)wib * (2 * nb + K);
  double* cumM = cumN + nb;
  double* X = cumM + nb;
  const long long first = only_slot >= 0 ? only_slot : (long long)blockIdx.x * wpb + wib;
  const long long step = only_slot >= 0 ? slots : (long long)gridDim.x * wpb;
  for (long long s = first; s < slots; s += step) {
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
        const double a = __shfl_up_sync(0xffffffffu, Rj, o), b = __shfl_up_sync(0xffffffffu, Mj, o);
        if (lane >= o) { Rj += a; Mj += b; }
      }
      if (j < nb) { cumN[j] = carryN + Rj; cumM[j] = carryM + Mj; }
      carryN += __shfl_sync(0xffffffffu, Rj, 31);
      carryM += __shfl_sync(0xffffffffu, Mj, 31);
    }
    if (!__any_sync(0xffffffffu, any)) continue;             // nothing absorbed: the cold row stays
    __syncwarp();
    // R38: X_0 = 1, X_f = sum_{i<f} B(f,i) X_i / A(f-1,f)
    for (int k = lane; k < K; k += 32) X[k] = k == 0 ? 1.0 : 0.0;
    __syncwarp();
    for (int f = 1; f < K; ++f) {
      const double Uf1 = D.U[f - 1], b = D.U[f] - Uf1;
      const int* Jf = D.J + (size_t)f * K;
      const int* Jf1 = D.J + (size_t)(f - 1) * K;
      double part = 0;
      for (int i = lane; i < f; i += 32) {
        const double xi = X[i];
        if (xi == 0.0) continue;
        const double a = Uf1 - D.U[i];
        const int nhi = Jf[i];                               // bins with E >= a + b: they land at or above f
        const int nlo = i == f - 1 ? nb : Jf1[i];            // bins with E >= a (a = 0 for i = f-1: all)
        const double Nhi = nhi ? cumN[nhi - 1] : 0.0, Mhi = nhi ? cumM[nhi - 1] : 0.0;
        const double Nlo = nlo ? cumN[nlo - 1] : 0.0, Mlo = nlo ? cumM[nlo - 1] : 0.0;
        part += (Nhi + ((Mlo - Mhi) - a * (Nlo - Nhi)) / b) * xi;
      }
      const double xf = warp_sum(part) / (D.Lam[f] / b);
      if (lane == 0) X[f] = xf;
      __syncwarp();
      if (xf > 1e200) {                                      // rescale (the normalisation comes last)
        for (int k = lane; k <= f; k += 32) X[k] *= 1e-200;
        __syncwarp();
      }
    }
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
        cumN[j0] = e0; cumN[j0 + 1] = e1; cumN[j0 + 2] = e2; cumN[j0 + 3] = e3;
        etot += (e0 + e1) + (e2 + e3);
      } else {
        for (int j = j0; j < min(nb, j0 + 4); ++j) {
          double e = 0;
          for (int k = 0; k < K; ++k) e += X[k] * (double)__ldg(D.W32 + (size_t)k * nb + j);
          cumN[j] = e;
          etot += e;
        }
      }
    }
    etot = warp_sum(etot);
    __syncwarp();
    double carry = 0;
    for (int j0 = 0; j0 < nb; j0 += 32) {
      const int j = j0 + lane;
      double e = j < nb ? cumN[j] : 0.0;
#pragma unroll
      for (int o = 1; o < 32; o <<= 1) {
        const double a = __shfl_up_sync(0xffffffffu, e, o);
        if (lane >= o) e += a;
      }
      if (j < nb) row[j] = (j == nb - 1 || !(etot > 0)) ? 1.f : (float)((carry + e) / etot);
      carry += __shfl_sync(0xffffffffu, e, 31);
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
