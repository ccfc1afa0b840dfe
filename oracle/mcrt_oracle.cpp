// oracle/mcrt_oracle.cpp -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
//
// Plain, slow, serial-in-spirit fp64 CPU implementation of the hot path of
// Siebenmorgen, Heymann & Kruegel, "PAH in vectorized three dimensional Monte Carlo dust
// radiative transfer models", following the paper's section 2 step by step:
//
//   PAPER.md L23     cubes / subcubes (cells); packages of constant energy eps and different
//                    frequencies; per cell an interaction with the probability given by the
//                    extinction optical depth along the path in the cell; scattering changes the
//                    direction by the phase function; absorption raises the cell's energy by eps
//                    and a package of the same energy is re-emitted isotropically from the spot
//                    at a new frequency (see the paper for the wording);
//   PAPER.md L25-27  nu_new from the cell temperature BEFORE the absorption, no Bjorkman & Wood
//                    correction (Eqn 11.67 instead of 11.65 of Kruegel 2006): dP/dnu ~ kappa_nu B_nu(T).
//
// Where the paper is silent the readings R1..R33 of SURVEY.md 8(c) / DESIGN.md section 3 are
// taken; each function below names the step (O0..O8) and reading it implements.
//
// Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference leg may
// load this file.  It shares no code, header, table or constant generator with the CUDA
// path under paper_1201_3588_b200/csrc/.
//
// Pins (tests/test_oracle_pins.py): Philox vs the cuRAND host library; isotropy and HG
// moments; Planck sum vs sigma T^4/pi; Q(T) vs the Gamma*zeta closed form; CDF sampling vs
// its definition; temperature-inversion identity; integer packet accounting; pure-scattering
// bin-by-bin conservation; Beer-Lambert escape vs brute-force chords; optically thin
// T ~ r^(-2/(4+beta)); per-flight agreement with an "intersect every box" walker (a second,
// independent algorithm, also re-implemented in numpy in the tests); split invariance on a
// two-level grid; external-field mean chord 2a/3; tests/test_oracle_pins2.py: source pick
// proportional to L_s (and its boundary case), sub-cell mass through the temperature identity
// of an all-refined grid over two batches, albedo and g indexed per bin.  O9 (direction-resolved tallies,
// tests/test_oracle_observer.py): sum identity, isotropy in mu, cone fraction, hand-computed
// projection geometry, symmetry.  O10 (serial Bjorkman-Wood scheme, tests/test_oracle_bw.py):
// telescoping of the corrected emission to the Planck spectrum at the final temperature.
// O11..O13 (transiently heated PAH, PAPER.md L23/L45/L49; DESIGN.md readings
// R35..R40; tests/test_oracle_pah.py): the temperature distribution P(T) is pinned by its two
// physical limits (strong heating -> a narrow peak at the equilibrium temperature; rare hard
// photons -> the cooling-curve distribution C(T)/Lambda(T)), by the balance of mean heating and
// mean cooling, and by the exact split of absorptions between PAH and equilibrium grains; the photon rates per
// molecule that feed it (pah_rates, R40) by the energy identity with a molecule count formed in the test from
// the inputs (root leaves and sub-cells), joined to the solver through heating = cooling.
// The WHOLE interaction loop (flights, scattering, absorption + re-emission, cubes and subcubes) at any optical
// depth is pinned by two situations in which the mathematics fixes its answer (tests/test_oracle_invariants.py):
// mean-chord invariance (a body in a uniform isotropic field: the expected absorbed count of every leaf, the
// scatterings and absorptions per package in closed form, for grey kappa, anisotropic scattering, refined cubes)
// and the black-body enclosure (dust at T0 in a black-body field of T0: escaped = emitted bin by bin, leaf tallies
// from the Planck mean, the temperature update returns T0, for non-grey kappa / albedo / g).  No function of this
// file is left unpinned.  What has no independent reference are the VALUES of the five benchmark configurations
// (no closed form; the paper's benchmark tables, are not available): there GPU <-> oracle
// agreement is the check, by functions that are each pinned.
//
// The per-packet loop may run under OpenMP (packets are independent within a batch: T is
// frozen, every packet has its own Philox stream, tallies are integers), which changes no
// result.

#include <algorithm>
#include <cmath>
#include <cstdint>
#include <cstdio>
#include <cstring>
#include <vector>
#ifdef _OPENMP
#include <omp.h>
#endif

namespace {

// ---- O0 constants (cgs, CODATA 2018) --------------------------------------------------
const double H_PLANCK = 6.62607015e-27;
const double C_LIGHT = 2.99792458e10;
const double K_BOLTZ = 1.380649e-16;
const double PI = 3.14159265358979323846;

const uint32_t TAG_EMIT = 0, TAG_FLIGHT = 1, TAG_REEMIT = 2, TAG_PAH = 4;
const double M_CARBON = 1.99264687992e-23;   // g, 12 amu (CODATA 2018 atomic mass constant x 12)
const uint32_t K_MAX_FLIGHTS = 10000000u;   // R20
const int COMP_DIRECT = 0, COMP_SCATTERED = 1, COMP_THERMAL = 2;

// ---- O3 Philox4x32-10 (Salmon et al. 2011) -------------------------------------------
void philox4x32_10(const uint32_t key_in[2], const uint32_t ctr_in[4], uint32_t out[4]) {
  const uint32_t M0 = 0xD2511F53u, M1 = 0xCD9E8D57u, W0 = 0x9E3779B9u, W1 = 0xBB67AE85u;
  uint32_t c0 = ctr_in[0], c1 = ctr_in[1], c2 = ctr_in[2], c3 = ctr_in[3];
  uint32_t k0 = key_in[0], k1 = key_in[1];
  for (int r = 0; r < 10; ++r) {
    if (r > 0) { k0 += W0; k1 += W1; }
    uint64_t p0 = (uint64_t)M0 * c0, p1 = (uint64_t)M1 * c2;
    uint32_t hi0 = (uint32_t)(p0 >> 32), lo0 = (uint32_t)p0;
    uint32_t hi1 = (uint32_t)(p1 >> 32), lo1 = (uint32_t)p1;
    uint32_t n0 = hi1 ^ c1 ^ k0, n1 = lo1, n2 = hi0 ^ c3 ^ k1, n3 = lo0;
    c0 = n0; c1 = n1; c2 = n2; c3 = n3;
  }
  out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

// R18/R19: block of four uniforms in (0,1) for (seed, packet id, k, tag).
void draw4(uint64_t seed, uint64_t pid, uint32_t k, uint32_t tag, double u[4]) {
  uint32_t key[2] = {(uint32_t)seed, (uint32_t)(seed >> 32)};
  uint32_t ctr[4] = {(uint32_t)pid, (uint32_t)(pid >> 32), k, tag};
  uint32_t x[4];
  philox4x32_10(key, ctr, x);
  for (int i = 0; i < 4; ++i) u[i] = ((double)x[i] + 0.5) * (1.0 / 4294967296.0);
}

// ---- O2 Planck -------------------------------------------------------------------------
double planck_nu(double nu, double T) {
  double x = H_PLANCK * nu / (K_BOLTZ * T);
  double e = std::expm1(x);
  if (!(e < 1e300)) return 0.0;
  return (2.0 * H_PLANCK * nu * nu * nu / (C_LIGHT * C_LIGHT)) / e;
}

// ---- O6 direction draws ----------------------------------------------------------------
void isotropic_dir(double u2, double u3, double d[3]) {
  double mu = 2.0 * u2 - 1.0, phi = 2.0 * PI * u3;
  double s = std::sqrt(std::max(0.0, 1.0 - mu * mu));
  d[0] = s * std::cos(phi); d[1] = s * std::sin(phi); d[2] = mu;
}

double hg_cos(double g, double u) {   // R15
  if (std::fabs(g) < 1e-3) return 2.0 * u - 1.0;
  double t = (1.0 - g * g) / (1.0 - g + 2.0 * g * u);
  double c = (1.0 + g * g - t * t) / (2.0 * g);
  return std::min(1.0, std::max(-1.0, c));
}

void rotate_dir(const double d[3], double ct, double phi, double out[3]) {
  double st = std::sqrt(std::max(0.0, 1.0 - ct * ct));
  double cp = std::cos(phi), sp = std::sin(phi);
  if (std::fabs(d[2]) < 1.0 - 1e-10) {
    double q = std::sqrt(1.0 - d[2] * d[2]);
    out[0] = st * (d[0] * d[2] * cp - d[1] * sp) / q + d[0] * ct;
    out[1] = st * (d[1] * d[2] * cp + d[0] * sp) / q + d[1] * ct;
    out[2] = -st * cp * q + d[2] * ct;
  } else {
    out[0] = st * cp; out[1] = st * sp; out[2] = (d[2] >= 0 ? 1.0 : -1.0) * ct;
  }
  double n = std::sqrt(out[0] * out[0] + out[1] * out[1] + out[2] * out[2]);
  out[0] /= n; out[1] /= n; out[2] /= n;
}

struct Source { int type; double pos[3]; double L; double Tbb; };

struct Counters { uint64_t emitted, escaped, lost, absorptions, scatterings, flights, crossings; };

struct Ctx {
  // grid (O1 of the build: D1, D2; layout R22). Positions are in root-cube units.
  int N = 0, S = 1;
  double origin[3] = {0, 0, 0}, root_size = 1;
  std::vector<int32_t> refidx;          // [N^3]: k-th refined cube, or -1
  int64_t n_ref = 0, slots = 0;
  std::vector<double> rho;              // [slots] g cm^-3
  // opacity tables (O1, O2)
  int nb = 0;
  std::vector<double> nu, dnu, kabs, ksca, kext, alb, g;
  int nT = 0; double Tmin = 1, Tmax = 1e4, dlnT = 0;
  std::vector<double> Q, C;             // Q[nT], C[nT*nb]
  // sources
  std::vector<Source> src; std::vector<double> Lcdf, Csrc; double Ltot = 0;
  // state
  std::vector<uint64_t> cum; std::vector<double> T; uint64_t Ncum = 0;
  std::vector<uint64_t> sed, emitted_per_bin; Counters cnt{};
  int walker = 0;                       // 0 = cell walk (O5), 1 = brute force (tests)
  // O10: the ORIGINAL serial scheme the paper departs from:
  // immediate temperature update at every absorption + Bjorkman & Wood (2001) corrected re-emission
  bool bw_mode = false; uint64_t bw_ntotal = 0;
  // O9 observer (reading R34): escape-direction binning
  int n_mu = 0; std::vector<uint64_t> sed_mu;               // [n_mu][3][nb]
  int n_pix = 0; double obs[3] = {0, 0, 1}, e1[3] = {1, 0, 0}, e2[3] = {0, 1, 0};
  double cos_alpha = 1, half_width = 1; int img_lo = 0, img_hi = -1;
  std::vector<uint64_t> image;                              // [n_pix][n_pix], row = e2, column = e1
  // O11..O13 (f2): transiently heated PAH, one kind per context
  bool pah = false;
  int nC = 0, KP = 0;                   // carbon atoms per molecule; temperature bins of P(T)
  double fP = 0, thetaP = 0;            // mass fraction of the dust in PAH; Debye-like temperature of the enthalpy law
  std::vector<double> kabs_all;         // [nb] absorption of the whole mix (kabs then holds the equilibrium grains only)
  std::vector<double> kP, qP, CP, EP;   // [nb] PAH absorption per g of mix; kP / kabs_all; per molecule; photon energy
  std::vector<double> TP, UP, LamP;     // [KP] temperature grid, enthalpy U(T_k), cooling power of one molecule
  std::vector<double> WP;               // [KP][nb] C_j dnu_j B_j(T_k): emission of one molecule at T_k into bin j
  std::vector<uint64_t> cumP;           // [slots][nb] PAH absorptions per leaf and bin, cumulative
  std::vector<double> EcdfP;            // [slots][nb] emission CDF of the PAH of each leaf (frozen within a batch)
  uint64_t pah_absorptions = 0;
  bool have_opacity = false, have_source = false;
};

inline int64_t root_lin(const Ctx& c, const int i[3]) {
  return (int64_t)i[0] + (int64_t)c.N * ((int64_t)i[1] + (int64_t)c.N * i[2]);
}
inline int64_t leaf_slot(const Ctx& c, const int ir[3], const int is[3], bool refined) {
  int64_t r = root_lin(c, ir);
  if (!refined) return r;
  int64_t k = c.refidx[r];
  return (int64_t)c.N * c.N * c.N + k * (int64_t)(c.S * c.S * c.S) +
         (is[0] + c.S * (is[1] + c.S * is[2]));
}

struct Packet {
  double x[3], d[3];
  int bin, comp;
  int ir[3], is[3];
  bool refined;
};

// R7: direction-aware location of the start cell, per axis in finest-level units.
bool locate(const Ctx& c, Packet& p) {
  for (int a = 0; a < 3; ++a) {
    double xf = p.x[a] * c.S;
    long f = (p.d[a] >= 0) ? (long)std::floor(xf) : (long)std::ceil(xf) - 1;
    if (f < 0 || f >= (long)c.N * c.S) return false;
    p.ir[a] = (int)(f / c.S);
    p.is[a] = (int)(f % c.S);
  }
  p.refined = c.refidx[root_lin(c, p.ir)] >= 0;
  if (!p.refined) p.is[0] = p.is[1] = p.is[2] = 0;
  return true;
}

// ---- O9 (R34): direction-resolved tallies of an escaping package.
//  * inclination: mu = d_z, n_mu bins uniform in mu over [-1, 1]: SED_mu[m][comp][bin] += 1;
//  * image: packages of bins img_lo..img_hi leaving within the cone d.obs >= cos(alpha) are
//    binned by their impact vector b = r - (r.d) d (r = position relative to the box centre; b
//    does not depend on where along the last flight it is taken) projected on the image axes
//    e1, e2 (both normal to obs), n_pix x n_pix pixels over [-half_width, half_width]^2.
void tally_observer(Ctx& c, const Packet& p) {
  if (c.n_mu > 0) {
    int m = (int)std::floor((p.d[2] + 1.0) * 0.5 * c.n_mu);
    m = std::min(c.n_mu - 1, std::max(0, m));
#pragma omp atomic
    c.sed_mu[((size_t)m * 3 + p.comp) * c.nb + p.bin] += 1;
  }
  if (c.n_pix > 0 && p.bin >= c.img_lo && p.bin <= c.img_hi) {
    double dot = p.d[0] * c.obs[0] + p.d[1] * c.obs[1] + p.d[2] * c.obs[2];
    if (dot >= c.cos_alpha) {
      double r[3], rd = 0;
      for (int a = 0; a < 3; ++a) { r[a] = p.x[a] - 0.5 * c.N; rd += r[a] * p.d[a]; }
      double X = 0, Y = 0;
      for (int a = 0; a < 3; ++a) { double b = r[a] - rd * p.d[a]; X += b * c.e1[a]; Y += b * c.e2[a]; }
      double fx = (X + c.half_width) / (2.0 * c.half_width) * c.n_pix;
      double fy = (Y + c.half_width) / (2.0 * c.half_width) * c.n_pix;
      if (fx >= 0 && fx < c.n_pix && fy >= 0 && fy < c.n_pix) {
#pragma omp atomic
        c.image[(size_t)std::floor(fy) * c.n_pix + (size_t)std::floor(fx)] += 1;
      }
    }
  }
}

// ---- O5: one flight by the cell walk.  Returns 1 = interaction in leaf *slot at p.x,
//      0 = escaped.  crossings is incremented once per leaf left through a face (R27).
int walk_cells(const Ctx& c, Packet& p, double tau_star, int64_t* slot, uint64_t* crossings) {
  const double hs = 1.0 / c.S;
  double tau_acc = 0.0;
  const double kx = c.kext[p.bin] * c.root_size;   // optical depth per (g cm^-3) per root unit
  for (;;) {
    double lo[3], hi[3];
    for (int a = 0; a < 3; ++a) {
      if (p.refined) { lo[a] = p.ir[a] + p.is[a] * hs; hi[a] = lo[a] + hs; }
      else { lo[a] = p.ir[a]; hi[a] = p.ir[a] + 1.0; }
    }
    double ell = 1e300; int ax = -1;
    for (int a = 0; a < 3; ++a) {
      if (std::fabs(p.d[a]) < 1e-30) continue;     // R21
      double t = ((p.d[a] > 0 ? hi[a] : lo[a]) - p.x[a]) / p.d[a];
      if (t < 0) t = 0;
      if (t < ell) { ell = t; ax = a; }            // strict <: ties -> lowest axis
    }
    int64_t s = leaf_slot(c, p.ir, p.is, p.refined);
    double alpha = c.rho[s] * kx;
    if (alpha > 0 && tau_acc + alpha * ell >= tau_star) {
      double dl = (tau_star - tau_acc) / alpha;
      for (int a = 0; a < 3; ++a) p.x[a] += p.d[a] * dl;
      *slot = s;
      return 1;
    }
    tau_acc += alpha * ell;
    for (int a = 0; a < 3; ++a) p.x[a] += p.d[a] * ell;
    p.x[ax] = (p.d[ax] > 0) ? hi[ax] : lo[ax];
    ++*crossings;
    int step = p.d[ax] > 0 ? 1 : -1;
    bool leave_root = true;
    if (p.refined) {
      int ns = p.is[ax] + step;
      if (ns >= 0 && ns < c.S) { p.is[ax] = ns; leave_root = false; }
    }
    if (leave_root) {
      p.ir[ax] += step;
      if (p.ir[ax] < 0 || p.ir[ax] >= c.N) return 0;          // escape by integer index
      p.refined = c.refidx[root_lin(c, p.ir)] >= 0;
      if (p.refined) {
        for (int b = 0; b < 3; ++b) {
          if (b == ax) { p.is[b] = step > 0 ? 0 : c.S - 1; continue; }
          int v = (int)std::floor((p.x[b] - p.ir[b]) / hs);
          p.is[b] = std::min(c.S - 1, std::max(0, v));
        }
      } else { p.is[0] = p.is[1] = p.is[2] = 0; }
    }
  }
}

// ---- second, independent walker for the pins: intersect EVERY leaf box with the ray by the
//      slab method, sort by entry distance, accumulate optical depth.  O(leaves) per flight.
int walk_bruteforce(const Ctx& c, Packet& p, double tau_star, int64_t* slot,
                    uint64_t* crossings) {
  struct Seg { double t0, t1; int64_t slot; int ir[3], is[3]; bool refined; };
  std::vector<Seg> segs;
  const double hs = 1.0 / c.S;
  const double kx = c.kext[p.bin] * c.root_size;
  auto clip = [&](const double lo[3], const double hi[3], double& t0, double& t1) {
    t0 = 0.0; t1 = 1e300;
    for (int a = 0; a < 3; ++a) {
      if (std::fabs(p.d[a]) < 1e-30) {
        if (p.x[a] < lo[a] || p.x[a] > hi[a]) return false;
        continue;
      }
      double ta = (lo[a] - p.x[a]) / p.d[a], tb = (hi[a] - p.x[a]) / p.d[a];
      if (ta > tb) std::swap(ta, tb);
      t0 = std::max(t0, ta); t1 = std::min(t1, tb);
    }
    return t1 > t0;
  };
  for (int z = 0; z < c.N; ++z) for (int y = 0; y < c.N; ++y) for (int x = 0; x < c.N; ++x) {
    int ir[3] = {x, y, z};
    bool ref = c.refidx[root_lin(c, ir)] >= 0;
    int n = ref ? c.S : 1;
    for (int sz = 0; sz < n; ++sz) for (int sy = 0; sy < n; ++sy) for (int sx = 0; sx < n; ++sx) {
      int is[3] = {sx, sy, sz};
      double lo[3], hi[3];
      for (int a = 0; a < 3; ++a) {
        lo[a] = ref ? ir[a] + is[a] * hs : ir[a];
        hi[a] = lo[a] + (ref ? hs : 1.0);
      }
      double t0, t1;
      if (!clip(lo, hi, t0, t1)) continue;
      Seg s; s.t0 = t0; s.t1 = t1; s.slot = leaf_slot(c, ir, is, ref); s.refined = ref;
      for (int a = 0; a < 3; ++a) { s.ir[a] = ir[a]; s.is[a] = is[a]; }
      segs.push_back(s);
    }
  }
  std::sort(segs.begin(), segs.end(), [](const Seg& a, const Seg& b) { return a.t0 < b.t0; });
  double tau_acc = 0.0;
  for (const Seg& s : segs) {
    double alpha = c.rho[s.slot] * kx, ell = s.t1 - s.t0;
    if (alpha > 0 && tau_acc + alpha * ell >= tau_star) {
      double t = s.t0 + (tau_star - tau_acc) / alpha;
      for (int a = 0; a < 3; ++a) { p.x[a] += p.d[a] * t; p.ir[a] = s.ir[a]; p.is[a] = s.is[a]; }
      p.refined = s.refined;
      *slot = s.slot;
      return 1;
    }
    tau_acc += alpha * ell;
    ++*crossings;
  }
  return 0;
}

// first j with cdf[j] >= u (R19: zero-probability bins are never selected)
int search_cdf(const double* cdf, int n, double u) {
  int lo = 0, hi = n - 1;
  while (lo < hi) { int mid = (lo + hi) / 2; if (cdf[mid] >= u) hi = mid; else lo = mid + 1; }
  return lo;
}

// O6 / R11: emission bin at temperature T from the table rows, stochastic row choice.
int sample_emission_bin(const Ctx& c, double T, double u0, double u1) {
  double t = (std::log(T) - std::log(c.Tmin)) / c.dlnT;
  t = std::min((double)(c.nT - 1), std::max(0.0, t));
  int k0 = (int)std::floor(t);
  double w = t - k0;
  int row = (u1 < w && k0 + 1 < c.nT) ? k0 + 1 : k0;
  return search_cdf(&c.C[(size_t)row * c.nb], c.nb, u0);
}

double leaf_mass(const Ctx& c, int64_t slot);

// O10: Bjorkman & Wood (2001) temperature-corrected re-emission.  The cell went from T_old to
// T_new by absorbing this package; the new package's frequency is drawn from
// dP/dnu ~ kappa_nu [B_nu(T_new) - B_nu(T_old)], so that the sum of everything the cell has
// emitted so far telescopes to kappa_nu B_nu(T_new).  CDF over the bins by the midpoint rule R5.
int sample_bw_bin(const Ctx& c, double T_old, double T_new, double u) {
  std::vector<double> cdf(c.nb);
  double acc = 0;
  for (int j = 0; j < c.nb; ++j) {
    double w = c.kabs[j] * (planck_nu(c.nu[j], T_new) - planck_nu(c.nu[j], T_old)) * c.dnu[j];
    acc += w > 0 ? w : 0.0;
    cdf[j] = acc;
  }
  if (!(acc > 0)) return sample_emission_bin(c, T_new, u, 0.0);     // T did not move: Eqn 11.67 at T_new
  for (int j = 0; j < c.nb; ++j) cdf[j] /= acc;
  cdf[c.nb - 1] = 1.0;
  return search_cdf(cdf.data(), c.nb, u);
}

// O7 / R12: invert Q(T) = q by bracketing + log-log interpolation; clamp.
double temperature_from_q(const Ctx& c, double q) {
  if (!(q > c.Q[0])) return c.Tmin;
  if (q >= c.Q[c.nT - 1]) return c.Tmax;
  int lo = 0, hi = c.nT - 1;                 // Q[lo] <= q < Q[hi]
  while (hi - lo > 1) { int mid = (lo + hi) / 2; if (c.Q[mid] <= q) lo = mid; else hi = mid; }
  double f = (std::log(q) - std::log(c.Q[lo])) / (std::log(c.Q[lo + 1]) - std::log(c.Q[lo]));
  double lnT = std::log(c.Tmin) + c.dlnT * (lo + f);
  return std::min(c.Tmax, std::max(c.Tmin, std::exp(lnT)));
}

// O4: emission of packet pid.  Returns false if the source lies outside the grid.
bool emit(const Ctx& c, uint64_t seed, uint64_t pid, Packet& p) {
  double u[4];
  draw4(seed, pid, 0, TAG_EMIT, u);
  int s = 0;
  while (s < (int)c.src.size() - 1 && c.Lcdf[s] < u[0]) ++s;      // s = min{s: Lcdf_s >= u0}
  p.bin = search_cdf(&c.Csrc[(size_t)s * c.nb], c.nb, u[1]);
  p.comp = COMP_DIRECT;
  if (c.src[s].type == 0) {
    isotropic_dir(u[2], u[3], p.d);
    for (int a = 0; a < 3; ++a) p.x[a] = c.src[s].pos[a];
  } else {                                                         // R25 external field
    double v[4];
    draw4(seed, pid, 1, TAG_EMIT, v);
    int f = std::min(5, (int)std::floor(6.0 * v[0]));
    int ax = f / 2, side = f % 2, b1 = (ax + 1) % 3, b2 = (ax + 2) % 3;
    double mu = std::sqrt(u[2]), phi = 2.0 * PI * u[3];
    double st = std::sqrt(std::max(0.0, 1.0 - mu * mu));
    p.d[ax] = side == 0 ? mu : -mu;
    p.d[b1] = st * std::cos(phi);
    p.d[b2] = st * std::sin(phi);
    p.x[ax] = side == 0 ? 0.0 : (double)c.N;
    p.x[b1] = v[1] * c.N;
    p.x[b2] = v[2] * c.N;
  }
  return locate(c, p);
}

struct Event { int32_t type; int32_t bin; int64_t slot; double x[3]; };  // for traces

// O4..O6: full life of one packet with temperatures frozen.  Tallies are integer atomics.
void run_packet(Ctx& c, uint64_t seed, uint64_t pid, std::vector<uint64_t>& batch,
                Event* trace, int trace_cap, int* trace_n) {
  Packet p;
  Counters loc{};
  auto rec = [&](int type, int64_t slot) {
    if (trace && *trace_n < trace_cap) {
      Event& e = trace[(*trace_n)++];
      e.type = type; e.bin = p.bin; e.slot = slot;
      for (int a = 0; a < 3; ++a) e.x[a] = p.x[a];
    }
  };
  bool ok = emit(c, seed, pid, p);
  loc.emitted = 1;
#pragma omp atomic
  c.emitted_per_bin[p.bin] += 1;
  rec(0, -1);
  if (!ok) { loc.lost = 1; }
  uint32_t k = 0;
  while (ok) {
    if (k >= K_MAX_FLIGHTS) { loc.lost = 1; break; }            // R20
    double u[4];
    draw4(seed, pid, k, TAG_FLIGHT, u);
    double tau_star = -std::log(u[0]);                           // R17
    loc.flights++;
    int64_t slot = -1;
    int hit = (c.walker == 0) ? walk_cells(c, p, tau_star, &slot, &loc.crossings)
                              : walk_bruteforce(c, p, tau_star, &slot, &loc.crossings);
    if (!hit) {                                                  // escape -> SED (R24)
      loc.escaped = 1;
#pragma omp atomic
      c.sed[(size_t)p.comp * c.nb + p.bin] += 1;
      tally_observer(c, p);
      rec(3, -1);
      break;
    }
    if (u[1] < c.alb[p.bin]) {                                   // scatter (R16)
      loc.scatterings++;
      double ct = hg_cos(c.g[p.bin], u[2]);
      double nd[3];
      rotate_dir(p.d, ct, 2.0 * PI * u[3], nd);
      p.d[0] = nd[0]; p.d[1] = nd[1]; p.d[2] = nd[2];
      if (p.comp == COMP_DIRECT) p.comp = COMP_SCATTERED;
      rec(1, slot);
    } else {                                                     // absorb + re-emit
      loc.absorptions++;
      double r[4];
      draw4(seed, pid, k, TAG_REEMIT, r);
      bool by_pah = false;
      double v[4] = {0, 0, 0, 0};
      if (c.pah) {                                               // O11 (R36): which grain absorbed the package
        draw4(seed, pid, k, TAG_PAH, v);
        by_pah = v[0] < c.qP[p.bin];
      }
      if (by_pah) {
#pragma omp atomic
        c.cumP[(size_t)slot * c.nb + p.bin] += 1;
#pragma omp atomic
        c.pah_absorptions += 1;
        p.bin = search_cdf(&c.EcdfP[(size_t)slot * c.nb], c.nb, v[1]);   // from the leaf's P(T), frozen in the batch
      } else {
#pragma omp atomic
      batch[slot] += 1;
      if (c.bw_mode) {                                             // O10: serial only
        double T_old = c.T[slot];
        c.cum[slot] += 1;
        double q = (double)c.cum[slot] * c.Ltot / ((double)c.bw_ntotal * 4.0 * PI * leaf_mass(c, slot));
        double T_new = temperature_from_q(c, q);
        c.T[slot] = T_new;
        p.bin = sample_bw_bin(c, T_old, T_new, r[0]);
      } else
      p.bin = sample_emission_bin(c, c.T[slot], r[0], r[1]);     // T frozen = T before absorption
      }
      isotropic_dir(r[2], r[3], p.d);
      p.comp = COMP_THERMAL;
      rec(2, slot);
    }
    ++k;
  }
#pragma omp atomic
  c.cnt.emitted += loc.emitted;
#pragma omp atomic
  c.cnt.escaped += loc.escaped;
#pragma omp atomic
  c.cnt.lost += loc.lost;
#pragma omp atomic
  c.cnt.absorptions += loc.absorptions;
#pragma omp atomic
  c.cnt.scatterings += loc.scatterings;
#pragma omp atomic
  c.cnt.flights += loc.flights;
#pragma omp atomic
  c.cnt.crossings += loc.crossings;
}

double leaf_mass(const Ctx& c, int64_t slot) {
  double V = c.root_size * c.root_size * c.root_size;
  if (slot >= (int64_t)c.N * c.N * c.N) V /= (double)(c.S * c.S * c.S);
  return c.rho[slot] * V;
}

// O7: merge the batch tally and update every leaf temperature (R9 reading B, R10, R12).
void merge_tally(Ctx& c, const std::vector<uint64_t>& batch, uint64_t n_packets) {
  for (int64_t i = 0; i < c.slots; ++i) c.cum[i] += batch[i];
  c.Ncum += n_packets;
}
// temperatures from absorbed-package counts `cum` after n_cum emitted packages
void update_temperatures(Ctx& c, const uint64_t* cum, uint64_t n_cum) {
  for (int64_t i = 0; i < c.slots; ++i) {
    double m = leaf_mass(c, i);
    if (m > 0 && cum[i] > 0) {
      double q = (double)cum[i] * c.Ltot / ((double)n_cum * 4.0 * PI * m);
      c.T[i] = temperature_from_q(c, q);
    } else {
      c.T[i] = c.Tmin;
    }
  }
}
void pah_update(Ctx& c, const uint64_t* counts, uint64_t n_cum);
void batch_end(Ctx& c, const std::vector<uint64_t>& batch, uint64_t n_packets) {
  merge_tally(c, batch, n_packets);
  update_temperatures(c, c.cum.data(), c.Ncum);
  if (c.pah) pah_update(c, c.cumP.data(), c.Ncum);
}

// O2: Q(T_k) and the emission CDF rows C_k[j] from c.kabs (midpoint rule R5, R11)
void build_emission_tables(Ctx& c) {
  const int nT = c.nT, n_bins = c.nb;
  c.Q.assign(nT, 0); c.C.assign((size_t)nT * n_bins, 0);
  for (int k = 0; k < nT; ++k) {
    double T = c.Tmin * std::pow(c.Tmax / c.Tmin, (double)k / (nT - 1));
    double acc = 0;
    for (int j = 0; j < n_bins; ++j) {
      acc += c.kabs[j] * planck_nu(c.nu[j], T) * c.dnu[j];
      c.C[(size_t)k * n_bins + j] = acc;
    }
    c.Q[k] = acc;
    for (int j = 0; j < n_bins; ++j)
      c.C[(size_t)k * n_bins + j] = acc > 0 ? c.C[(size_t)k * n_bins + j] / acc : 1.0;
    c.C[(size_t)k * n_bins + n_bins - 1] = 1.0;
  }
}

// ---- O11 (R37): synthetic enthalpy law of a PAH with N carbon atoms.  Heat capacity
// C(T) = 3 N k x^2/(1+x^2), x = T/Theta (quadratic at low T as for graphitic sheets, 3Nk at high T);
// enthalpy U(T) = integral_0^T C = 3 N k Theta (x - atan x).
double pah_heat_capacity(const Ctx& c, double T) {
  double x = T / c.thetaP;
  return 3.0 * c.nC * K_BOLTZ * x * x / (1.0 + x * x);
}
double pah_enthalpy(const Ctx& c, double T) {
  double x = T / c.thetaP;
  return 3.0 * c.nC * K_BOLTZ * c.thetaP * (x - std::atan(x));
}

// ---- O12 (R38): stationary temperature distribution of one PAH molecule that absorbs photons of
// bin j at the rate R[j] (1/s).  States k = 0..K-1 with enthalpies U_k = U(T_k).
//  * heating: a photon of energy E takes state i to the enthalpy U* = U_i + E, shared between the two
//    states that bracket U* in proportion to the distance (mean enthalpy conserved); beyond the last
//    state everything lands in it.  The rate from i into states >= f is therefore
//        B(f,i) = sum_j R_j clamp((U_i + E_j - U_{f-1}) / (U_f - U_{f-1}), 0, 1)        (f > i);
//    photons too soft to reach the next state act as continuous heating (the same formula).
//  * cooling: only to the next lower state, A(f-1,f) = Lambda(T_f) / (U_f - U_{f-1})
//    ("thermal continuous" cooling of Guhathakurta & Draine 1989, as in Kruegel's treatment).
//  * stationarity in that case is the recursion X_0 = 1, X_f = sum_{i<f} B(f,i) X_i / A(f-1,f),
//    P = X / sum X (all terms positive; X is rescaled when it grows large).
void pah_temperature_distribution(const Ctx& c, const double* R, double* P) {
  const int K = c.KP, nb = c.nb;
  std::vector<double> X(K, 0.0);
  X[0] = 1.0;
  for (int f = 1; f < K; ++f) {
    const double dU = c.UP[f] - c.UP[f - 1];
    double sum = 0;
    for (int i = 0; i < f; ++i) {
      if (X[i] == 0) continue;
      double B = 0;
      for (int j = 0; j < nb; ++j) {
        if (R[j] == 0) continue;
        double w = (c.UP[i] + c.EP[j] - c.UP[f - 1]) / dU;
        B += R[j] * std::min(1.0, std::max(0.0, w));
      }
      sum += B * X[i];
    }
    X[f] = sum / (c.LamP[f] / dU);
    if (X[f] > 1e200) for (int i = 0; i <= f; ++i) X[i] *= 1e-200;
  }
  double tot = 0;
  for (int k = 0; k < K; ++k) tot += X[k];
  for (int k = 0; k < K; ++k) P[k] = X[k] / tot;
}

// photon absorption rates (1/s) of one PAH molecule of leaf `slot` from cumulative counts (R40):
// counts_j * (L_tot / N_cum) / (h nu_j) / (number of molecules in the leaf)
bool pah_rates(const Ctx& c, int64_t slot, const uint64_t* counts, uint64_t n_cum, double* R) {
  double m = leaf_mass(c, slot);
  bool any = false;
  for (int j = 0; j < c.nb; ++j) { R[j] = 0; any = any || counts[j] > 0; }
  if (!(m > 0) || !any || n_cum == 0) return false;
  double n_mol = c.fP * m / (c.nC * M_CARBON);
  for (int j = 0; j < c.nb; ++j)
    R[j] = (double)counts[j] * c.Ltot / ((double)n_cum * c.EP[j] * n_mol);
  return true;
}

// ---- O13 (R39): emission CDF of the PAH of a leaf from P(T): E_j = sum_k P_k C_j dnu_j B_j(T_k)
void pah_emission_cdf(const Ctx& c, const double* P, double* cdf) {
  const int K = c.KP, nb = c.nb;
  double acc = 0;
  for (int j = 0; j < nb; ++j) {
    double e = 0;
    for (int k = 0; k < K; ++k) e += P[k] * c.WP[(size_t)k * nb + j];
    acc += e;
    cdf[j] = acc;
  }
  for (int j = 0; j < nb; ++j) cdf[j] = acc > 0 ? cdf[j] / acc : 1.0;
  cdf[nb - 1] = 1.0;
}

// batch end for the PAH: P(T) and emission CDF of every leaf from counts after n_cum packages
void pah_update(Ctx& c, const uint64_t* counts, uint64_t n_cum) {
  const int nb = c.nb, K = c.KP;
#pragma omp parallel
  {
    std::vector<double> R(nb), P(K);
#pragma omp for schedule(dynamic, 64)
    for (int64_t i = 0; i < c.slots; ++i) {
      if (!pah_rates(c, i, counts + (size_t)i * nb, n_cum, R.data())) continue;   // cold row stays
      pah_temperature_distribution(c, R.data(), P.data());
      pah_emission_cdf(c, P.data(), &c.EcdfP[(size_t)i * nb]);
    }
  }
}

}  // namespace

// =======================================================================================
// C interface for ctypes (tests, smoke, cpu_baseline only)
// =======================================================================================
extern "C" {

void* orc_create(int n_root, int sub, const double* origin, double root_size,
                 const uint8_t* refine, const float* rho_root, const float* rho_sub) {
  if (n_root < 1 || root_size <= 0) return nullptr;
  Ctx* c = new Ctx;
  c->N = n_root; c->S = sub > 1 ? sub : 1; c->root_size = root_size;
  for (int a = 0; a < 3; ++a) c->origin[a] = origin[a];
  int64_t n3 = (int64_t)n_root * n_root * n_root;
  c->refidx.assign(n3, -1);
  int64_t k = 0;
  if (refine && c->S > 1)
    for (int64_t i = 0; i < n3; ++i) if (refine[i]) c->refidx[i] = (int32_t)k++;
  c->n_ref = k;
  if (k == 0) c->S = 1;
  int64_t s3 = (int64_t)c->S * c->S * c->S;
  c->slots = n3 + k * s3;
  c->rho.assign(c->slots, 0.0);
  for (int64_t i = 0; i < n3; ++i) c->rho[i] = c->refidx[i] >= 0 ? 0.0 : (double)rho_root[i];
  for (int64_t i = 0; i < k * s3; ++i) c->rho[n3 + i] = (double)rho_sub[i];
  c->cum.assign(c->slots, 0);
  c->T.assign(c->slots, 1.0);
  return c;
}

void orc_destroy(void* h) { delete (Ctx*)h; }
int64_t orc_leaf_slots(void* h) { return ((Ctx*)h)->slots; }
void orc_set_walker(void* h, int w) { ((Ctx*)h)->walker = w; }

// O1 + O2 (R4, R5, R6, R11, R13, R33): tables in fp64 from the fp32 input opacities.
int orc_set_opacity(void* h, int n_bins, const double* lambda_edges_um, int n_species,
                    const double* weight, const float* kabs, const float* ksca, const float* g,
                    double Tmin, double Tmax, int nT) {
  Ctx& c = *(Ctx*)h;
  if (n_bins < 1 || n_species < 1) return -1;
  if (nT <= 0) { Tmin = 1.0; Tmax = 1.0e4; nT = 801; }
  c.nb = n_bins; c.nT = nT; c.Tmin = Tmin; c.Tmax = Tmax;
  c.dlnT = (std::log(Tmax) - std::log(Tmin)) / (nT - 1);
  c.nu.resize(n_bins); c.dnu.resize(n_bins);
  for (int j = 0; j < n_bins; ++j) {
    double l0 = lambda_edges_um[j] * 1e-4, l1 = lambda_edges_um[j + 1] * 1e-4;   // cm
    c.nu[j] = C_LIGHT / std::sqrt(l0 * l1);
    c.dnu[j] = C_LIGHT / l0 - C_LIGHT / l1;
  }
  c.kabs.assign(n_bins, 0); c.ksca.assign(n_bins, 0); c.kext.assign(n_bins, 0);
  c.alb.assign(n_bins, 0); c.g.assign(n_bins, 0);
  for (int j = 0; j < n_bins; ++j) {
    double gs = 0;
    for (int s = 0; s < n_species; ++s) {
      c.kabs[j] += weight[s] * (double)kabs[(size_t)s * n_bins + j];
      c.ksca[j] += weight[s] * (double)ksca[(size_t)s * n_bins + j];
      gs += weight[s] * (double)ksca[(size_t)s * n_bins + j] * (double)g[(size_t)s * n_bins + j];
    }
    c.kext[j] = c.kabs[j] + c.ksca[j];
    c.alb[j] = c.kext[j] > 0 ? c.ksca[j] / c.kext[j] : 0.0;
    c.g[j] = c.ksca[j] > 0 ? gs / c.ksca[j] : 0.0;
  }
  build_emission_tables(c);
  c.sed.assign((size_t)3 * n_bins, 0);
  c.emitted_per_bin.assign(n_bins, 0);
  c.have_opacity = true;
  return 0;
}

// O2 (sources): spectrum CDF by the same midpoint rule, luminosity CDF.  pos in cm.
int orc_set_source(void* h, int n_src, const int* type, const double* pos, const double* L,
                   const double* Tbb) {
  Ctx& c = *(Ctx*)h;
  if (!c.have_opacity || n_src < 1) return -2;
  c.src.resize(n_src); c.Lcdf.resize(n_src); c.Csrc.assign((size_t)n_src * c.nb, 0);
  c.Ltot = 0;
  for (int s = 0; s < n_src; ++s) c.Ltot += L[s];
  double acc = 0;
  for (int s = 0; s < n_src; ++s) {
    c.src[s].type = type[s]; c.src[s].L = L[s]; c.src[s].Tbb = Tbb[s];
    for (int a = 0; a < 3; ++a) c.src[s].pos[a] = (pos[3 * s + a] - c.origin[a]) / c.root_size;
    acc += L[s]; c.Lcdf[s] = acc / c.Ltot;
    double sum = 0;
    for (int j = 0; j < c.nb; ++j) {
      sum += planck_nu(c.nu[j], Tbb[s]) * c.dnu[j];
      c.Csrc[(size_t)s * c.nb + j] = sum;
    }
    for (int j = 0; j < c.nb; ++j) c.Csrc[(size_t)s * c.nb + j] /= sum;
    c.Csrc[(size_t)s * c.nb + c.nb - 1] = 1.0;
  }
  c.Lcdf[n_src - 1] = 1.0;
  c.have_source = true;
  return 0;
}

// O4..O7 for packets [first, first+n): transport with T frozen, then batch end.
int orc_run_batch(void* h, uint64_t seed, uint64_t first, uint64_t n, int n_threads) {
  Ctx& c = *(Ctx*)h;
  if (!c.have_source) return -2;
  std::vector<uint64_t> batch(c.slots, 0);
#ifdef _OPENMP
  if (n_threads > 0) omp_set_num_threads(n_threads);
#endif
#pragma omp parallel for schedule(dynamic, 64)
  for (int64_t i = 0; i < (int64_t)n; ++i)
    run_packet(c, seed, first + (uint64_t)i, batch, nullptr, 0, nullptr);
  batch_end(c, batch, n);
  return 0;
}

// The two halves of a batch, for packet-sharded runs: transport of this
// rank's packets with T frozen and NO temperature update ...
int orc_transport_batch(void* h, uint64_t seed, uint64_t first, uint64_t n, int n_threads) {
  Ctx& c = *(Ctx*)h;
  if (!c.have_source) return -2;
  std::vector<uint64_t> batch(c.slots, 0);
#ifdef _OPENMP
  if (n_threads > 0) omp_set_num_threads(n_threads);
#endif
#pragma omp parallel for schedule(dynamic, 64)
  for (int64_t i = 0; i < (int64_t)n; ++i)
    run_packet(c, seed, first + (uint64_t)i, batch, nullptr, 0, nullptr);
  merge_tally(c, batch, n);
  return 0;
}
// ... and O7's temperature step on counts summed over all ranks (n_cum = packages emitted by
// all ranks so far).  Same arithmetic as batch_end; this rank's own cum/Ncum are not touched.
int orc_update_temperature(void* h, const uint64_t* tally_sum, uint64_t n_cum) {
  Ctx& c = *(Ctx*)h;
  if (!c.have_source || !tally_sum || n_cum == 0) return -2;
  update_temperatures(c, tally_sum, n_cum);
  return 0;
}

// O11: declare the PAH (one kind per context).  kabs_pah[nb] = absorption of the PAH per gram of the dust MIX
// (it must be part of the mix given to orc_set_opacity: clipped to the mix's kappa_abs).  The equilibrium
// tables Q(T), C_k are rebuilt from what is left for the grains in equilibrium.  Temperature grid of P(T):
// K log-spaced values T_lo..T_hi.
void pah_cold_rows(Ctx& c) {
  std::vector<double> P(c.KP, 0.0), row(c.nb);
  P[0] = 1.0;
  pah_emission_cdf(c, P.data(), row.data());
  c.EcdfP.assign((size_t)c.slots * c.nb, 0.0);
  for (int64_t i = 0; i < c.slots; ++i) std::copy(row.begin(), row.end(), c.EcdfP.begin() + (size_t)i * c.nb);
}
int orc_set_pah(void* h, int n_C, double mass_fraction, double theta_K, const float* kabs_pah, double T_lo,
                double T_hi, int K) {
  Ctx& c = *(Ctx*)h;
  if (!c.have_opacity || n_C < 1 || !(mass_fraction > 0) || !(theta_K > 0) || K < 4 || !(T_lo > 0) || !(T_hi > T_lo))
    return -1;
  const int nb = c.nb;
  if (c.kabs_all.empty()) c.kabs_all = c.kabs;
  c.pah = true; c.nC = n_C; c.fP = mass_fraction; c.thetaP = theta_K; c.KP = K;
  c.kP.assign(nb, 0); c.qP.assign(nb, 0); c.CP.assign(nb, 0); c.EP.assign(nb, 0);
  for (int j = 0; j < nb; ++j) {
    c.kP[j] = std::min((double)kabs_pah[j], c.kabs_all[j]);
    if (!(c.kP[j] > 0)) c.kP[j] = 0;
    c.kabs[j] = c.kabs_all[j] - c.kP[j];                       // grains in equilibrium
    c.qP[j] = c.kabs_all[j] > 0 ? c.kP[j] / c.kabs_all[j] : 0.0;
    c.CP[j] = c.kP[j] * n_C * M_CARBON / mass_fraction;        // cm^2 per molecule
    c.EP[j] = H_PLANCK * c.nu[j];
  }
  build_emission_tables(c);
  c.TP.resize(K); c.UP.resize(K); c.LamP.resize(K); c.WP.assign((size_t)K * nb, 0);
  for (int k = 0; k < K; ++k) {
    c.TP[k] = T_lo * std::pow(T_hi / T_lo, (double)k / (K - 1));
    c.UP[k] = pah_enthalpy(c, c.TP[k]);
    double lam = 0;
    for (int j = 0; j < nb; ++j) {
      double w = c.CP[j] * planck_nu(c.nu[j], c.TP[k]) * c.dnu[j];
      c.WP[(size_t)k * nb + j] = w;
      lam += w;
    }
    c.LamP[k] = 4.0 * PI * lam;
  }
  c.cumP.assign((size_t)c.slots * nb, 0);
  c.pah_absorptions = 0;
  pah_cold_rows(c);
  return 0;
}
void orc_get_pah_grid(void* h, double* T, double* U, double* Lam, double* Cmol, double* q) {
  Ctx& c = *(Ctx*)h;
  for (int k = 0; k < c.KP; ++k) { T[k] = c.TP[k]; U[k] = c.UP[k]; Lam[k] = c.LamP[k]; }
  for (int j = 0; j < c.nb; ++j) { Cmol[j] = c.CP[j]; q[j] = c.qP[j]; }
}
// O12 / O13 as component entry points (pins), and for the tallies of another implementation (parity)
void orc_pah_solve(void* h, const double* R, double* P, double* cdf) {
  Ctx& c = *(Ctx*)h;
  pah_temperature_distribution(c, R, P);
  if (cdf) pah_emission_cdf(c, P, cdf);
}
int orc_pah_rates(void* h, int64_t slot, const uint64_t* counts, uint64_t n_cum, double* R) {
  return pah_rates(*(Ctx*)h, slot, counts, n_cum, R) ? 1 : 0;
}
void orc_pah_update(void* h, const uint64_t* counts, uint64_t n_cum) {
  Ctx& c = *(Ctx*)h;
  pah_cold_rows(c);
  pah_update(c, counts, n_cum);
}
double orc_pah_enthalpy(void* h, double T) { return pah_enthalpy(*(Ctx*)h, T); }
double orc_pah_heat_capacity(void* h, double T) { return pah_heat_capacity(*(Ctx*)h, T); }
void orc_get_pah_absorbed(void* h, uint64_t* out, uint64_t* total) {
  Ctx& c = *(Ctx*)h;
  std::memcpy(out, c.cumP.data(), sizeof(uint64_t) * c.cumP.size());
  if (total) *total = c.pah_absorptions;
}
void orc_get_pah_cdf(void* h, double* out) {
  Ctx& c = *(Ctx*)h;
  std::memcpy(out, c.EcdfP.data(), sizeof(double) * c.EcdfP.size());
}

// O9: observer set-up.  dir need not be normalised; half_width in cm; n_mu = 0 / n_pix = 0 switch
// the respective tally off.  Image axes: e1 = z x obs normalised (within 2.6 degrees of the pole: the
// part of x normal to obs), e2 = obs x e1.
int orc_set_observer(void* h, int n_mu, int n_pix, const double* dir, double half_angle_deg,
                     double half_width_cm, int bin_lo, int bin_hi) {
  Ctx& c = *(Ctx*)h;
  if (!c.have_opacity || n_mu < 0 || n_pix < 0) return -2;
  c.n_mu = n_mu; c.sed_mu.assign((size_t)n_mu * 3 * c.nb, 0);
  c.n_pix = n_pix; c.image.assign((size_t)n_pix * n_pix, 0);
  if (n_pix > 0) {
    double n = std::sqrt(dir[0] * dir[0] + dir[1] * dir[1] + dir[2] * dir[2]);
    if (!(n > 0) || !(half_width_cm > 0)) return -1;
    for (int a = 0; a < 3; ++a) c.obs[a] = dir[a] / n;
    if (std::fabs(c.obs[2]) < 0.999) {
      double q = std::sqrt(c.obs[0] * c.obs[0] + c.obs[1] * c.obs[1]);
      c.e1[0] = -c.obs[1] / q; c.e1[1] = c.obs[0] / q; c.e1[2] = 0;          // z x obs, normalised
    } else {
      // near the pole z x obs is ill-conditioned: e1 = the part of x normal to obs, normalised
      // (x itself for obs exactly along z, as R34 says), so that (e1, e2, obs) stays orthonormal
      double v[3] = {1.0 - c.obs[0] * c.obs[0], -c.obs[0] * c.obs[1], -c.obs[0] * c.obs[2]};
      double q = std::sqrt(v[0] * v[0] + v[1] * v[1] + v[2] * v[2]);
      for (int a = 0; a < 3; ++a) c.e1[a] = v[a] / q;
    }
    c.e2[0] = c.obs[1] * c.e1[2] - c.obs[2] * c.e1[1];
    c.e2[1] = c.obs[2] * c.e1[0] - c.obs[0] * c.e1[2];
    c.e2[2] = c.obs[0] * c.e1[1] - c.obs[1] * c.e1[0];
    c.cos_alpha = std::cos(half_angle_deg * PI / 180.0);
    c.half_width = half_width_cm / c.root_size;
    c.img_lo = bin_lo; c.img_hi = bin_hi;
  }
  return 0;
}
void orc_get_observer_axes(void* h, double* obs, double* e1, double* e2) {
  Ctx& c = *(Ctx*)h;
  for (int a = 0; a < 3; ++a) { obs[a] = c.obs[a]; e1[a] = c.e1[a]; e2[a] = c.e2[a]; }
}
void orc_get_sed_mu(void* h, uint64_t* out) {
  Ctx& c = *(Ctx*)h;
  for (size_t i = 0; i < c.sed_mu.size(); ++i) out[i] = c.sed_mu[i];
}
void orc_get_image(void* h, uint64_t* out) {
  Ctx& c = *(Ctx*)h;
  for (size_t i = 0; i < c.image.size(); ++i) out[i] = c.image[i];
}

// O10: packages [first, first+n) of a job of n_total packages by the original serial scheme:
// epsilon = L_tot / n_total fixed for the whole job (R9 reading A), every absorption raises the
// cell's temperature at once, re-emission by sample_bw_bin.  Strictly serial (each absorption
// changes T for the next package); cum[] holds the running counts, Ncum the packages run so far.
int orc_run_bw(void* h, uint64_t seed, uint64_t first, uint64_t n, uint64_t n_total) {
  Ctx& c = *(Ctx*)h;
  if (!c.have_source || n_total == 0) return -2;
  c.bw_mode = true; c.bw_ntotal = n_total;
  std::vector<uint64_t> unused(c.slots, 0);
  for (uint64_t i = 0; i < n; ++i) run_packet(c, seed, first + i, unused, nullptr, 0, nullptr);
  c.bw_mode = false;
  c.Ncum += n;
  return 0;
}

int orc_max_threads() {
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}

// Event trace of a single packet against the current (frozen) temperatures; tallies ARE
// updated in a scratch copy only (the context is left untouched except counters/SED).
int orc_trace_packet(void* h, uint64_t seed, uint64_t pid, int cap, int32_t* type,
                     int32_t* bin, int64_t* slot, double* xyz) {
  Ctx& c = *(Ctx*)h;
  std::vector<uint64_t> batch(c.slots, 0);
  std::vector<Event> ev(cap);
  int n = 0;
  Counters save = c.cnt;
  std::vector<uint64_t> sed = c.sed, epb = c.emitted_per_bin;
  run_packet(c, seed, pid, batch, ev.data(), cap, &n);
  c.cnt = save; c.sed = sed; c.emitted_per_bin = epb;
  for (int i = 0; i < n; ++i) {
    type[i] = ev[i].type; bin[i] = ev[i].bin; slot[i] = ev[i].slot;
    for (int a = 0; a < 3; ++a) xyz[3 * i + a] = ev[i].x[a];
  }
  return n;
}

// getters (O8)
void orc_get_cell_energy(void* h, uint64_t* n_abs, double* eps) {
  Ctx& c = *(Ctx*)h;
  std::memcpy(n_abs, c.cum.data(), sizeof(uint64_t) * c.slots);
  *eps = c.Ncum ? c.Ltot / (double)c.Ncum : 0.0;
}
void orc_get_cell_temperature(void* h, double* T) {
  Ctx& c = *(Ctx*)h; std::memcpy(T, c.T.data(), sizeof(double) * c.slots);
}
void orc_set_cell_temperature(void* h, const double* T) {      // tests: fixed-T emission pins
  Ctx& c = *(Ctx*)h; std::memcpy(c.T.data(), T, sizeof(double) * c.slots);
}
void orc_get_sed(void* h, uint64_t* out) {
  Ctx& c = *(Ctx*)h; std::memcpy(out, c.sed.data(), sizeof(uint64_t) * 3 * c.nb);
}
void orc_get_counters(void* h, uint64_t* out7, uint64_t* emitted_per_bin) {
  Ctx& c = *(Ctx*)h;
  out7[0] = c.cnt.emitted; out7[1] = c.cnt.escaped; out7[2] = c.cnt.lost;
  out7[3] = c.cnt.absorptions; out7[4] = c.cnt.scatterings; out7[5] = c.cnt.flights;
  out7[6] = c.cnt.crossings;
  if (emitted_per_bin) std::memcpy(emitted_per_bin, c.emitted_per_bin.data(), 8 * c.nb);
}
void orc_reset_tallies(void* h, int what) {
  Ctx& c = *(Ctx*)h;
  if (what & 1) { std::fill(c.sed.begin(), c.sed.end(), 0);
                  std::fill(c.emitted_per_bin.begin(), c.emitted_per_bin.end(), 0); c.cnt = Counters{};
                  std::fill(c.sed_mu.begin(), c.sed_mu.end(), 0); std::fill(c.image.begin(), c.image.end(), 0); }
  if (what & 2) { std::fill(c.cum.begin(), c.cum.end(), 0); std::fill(c.T.begin(), c.T.end(), c.Tmin);
                  c.Ncum = 0;
                  if (c.pah) { std::fill(c.cumP.begin(), c.cumP.end(), 0); c.pah_absorptions = 0; pah_cold_rows(c); } }
}
void orc_get_tables(void* h, double* nu, double* dnu, double* kabs, double* kext, double* alb,
                    double* g, double* Q, double* C) {
  Ctx& c = *(Ctx*)h;
  auto cp = [](double* d, const std::vector<double>& v) { if (d) std::memcpy(d, v.data(), 8 * v.size()); };
  cp(nu, c.nu); cp(dnu, c.dnu); cp(kabs, c.kabs); cp(kext, c.kext); cp(alb, c.alb); cp(g, c.g);
  cp(Q, c.Q); cp(C, c.C);
}
void orc_get_source_cdf(void* h, double* Csrc, double* Lcdf) {
  Ctx& c = *(Ctx*)h;
  std::memcpy(Csrc, c.Csrc.data(), 8 * c.Csrc.size());
  std::memcpy(Lcdf, c.Lcdf.data(), 8 * c.Lcdf.size());
}

// ---- component entry points for the pins ------------------------------------------------
void orc_philox(const uint32_t* key2, const uint32_t* ctr4, uint32_t* out4) {
  philox4x32_10(key2, ctr4, out4);
}
void orc_draw4(uint64_t seed, uint64_t pid, uint32_t k, uint32_t tag, double* u4) {
  draw4(seed, pid, k, tag, u4);
}
void orc_isotropic(double u2, double u3, double* d) { isotropic_dir(u2, u3, d); }
double orc_hg_cos(double g, double u) { return hg_cos(g, u); }
void orc_rotate(const double* d, double ct, double phi, double* out) { rotate_dir(d, ct, phi, out); }
double orc_planck(double nu, double T) { return planck_nu(nu, T); }
int orc_sample_emission_bin(void* h, double T, double u0, double u1) {
  return sample_emission_bin(*(Ctx*)h, T, u0, u1);
}
double orc_temperature_from_q(void* h, double q) { return temperature_from_q(*(Ctx*)h, q); }
double orc_leaf_mass(void* h, int64_t slot) { return leaf_mass(*(Ctx*)h, slot); }

// One emission (O4): position (root units), direction, bin, start leaf slot.
int orc_emit(void* h, uint64_t seed, uint64_t pid, double* x, double* d, int* bin, int64_t* slot) {
  Ctx& c = *(Ctx*)h;
  Packet p;
  bool ok = emit(c, seed, pid, p);
  for (int a = 0; a < 3; ++a) { x[a] = p.x[a]; d[a] = p.d[a]; }
  *bin = p.bin;
  *slot = ok ? leaf_slot(c, p.ir, p.is, p.refined) : -1;
  return ok ? 0 : -1;
}

// One flight (O5) from x (root units) along d in frequency bin `bin` with optical depth
// tau_star, using walker w.  Returns 1 = interaction (slot, x_out), 0 = escaped, -1 = outside.
int orc_walk(void* h, int w, const double* x, const double* d, int bin, double tau_star,
             int64_t* slot, double* x_out, uint64_t* crossings) {
  Ctx& c = *(Ctx*)h;
  Packet p;
  for (int a = 0; a < 3; ++a) { p.x[a] = x[a]; p.d[a] = d[a]; }
  p.bin = bin; p.comp = 0;
  if (!locate(c, p)) return -1;
  *crossings = 0; *slot = -1;
  int r = w == 0 ? walk_cells(c, p, tau_star, slot, crossings)
                 : walk_bruteforce(c, p, tau_star, slot, crossings);
  for (int a = 0; a < 3; ++a) x_out[a] = p.x[a];
  return r;
}

}  // extern "C"
