"""Seeded synthetic input generators for the five BASELINE.json configs (C0..C4).

This module only *describes inputs*: grids, densities, opacity tables, sources, packet
counts.  It holds none of the method's arithmetic (no Planck function, no CDFs, no random
walk, no Philox) and is the ONLY code shared by the CUDA path and the oracle.  Everything
the method itself computes from these inputs is done independently on each side.

The paper measures on published benchmarks (Ivezic 1997 spheres, Pascucci 2004 disks,
PAPER.md L27) and real dust data, none of which is available; the
inputs below take their shapes and stand in for them (recipe: DESIGN.md section 4,
SURVEY.md section 8(d)).

Units: cgs.  Wavelengths in micron.  Opacities cm^2 g^-1 (scale arbitrary: only rho*kappa
enters the transport).
"""
from __future__ import annotations

from dataclasses import dataclass, field
from typing import List, Optional

import numpy as np

AU = 1.495978707e13      # cm
LSUN = 3.828e33          # erg s^-1

SRC_POINT = 0            # isotropic point source
SRC_EXTERNAL = 1         # external isotropic field entering through the six box faces


@dataclass
class Source:
    type: int
    pos: tuple            # cm (ignored for SRC_EXTERNAL)
    L: float              # erg/s inside the wavelength band
    T_bb: float           # K


@dataclass
class Workload:
    name: str
    n_root: int
    sub: int                              # 0 = no refinement, else subcubes per edge (4)
    origin: tuple                         # cm, low corner of the box
    root_size: float                      # cm
    refine: Optional[np.ndarray]          # uint8 [N^3] x-fastest, or None
    rho_root: np.ndarray                  # float32 [N^3] x-fastest
    rho_sub: Optional[np.ndarray]         # float32 [n_ref * S^3]
    lambda_edges_um: np.ndarray           # float64 [n_bins+1] ascending
    weight: np.ndarray                    # float64 [n_species], sum 1
    kabs: np.ndarray                      # float32 [n_species, n_bins]
    ksca: np.ndarray                      # float32 [n_species, n_bins]
    g: np.ndarray                         # float32 [n_species, n_bins]
    sources: List[Source]
    n_packets: int
    batch: int
    seed: int = 1
    meta: dict = field(default_factory=dict)

    @property
    def n_bins(self) -> int:
        return len(self.lambda_edges_um) - 1

    @property
    def n_ref(self) -> int:
        return 0 if self.refine is None else int(self.refine.sum())

    @property
    def leaf_slots(self) -> int:
        s = self.sub if self.sub > 1 else 0
        return self.n_root ** 3 + self.n_ref * s ** 3

    def batches(self, n_packets: Optional[int] = None, batch: Optional[int] = None):
        """Yield (first_packet_id, count) for the config's batch partition."""
        n = self.n_packets if n_packets is None else n_packets
        b = self.batch if batch is None else batch
        first = 0
        while first < n:
            c = min(b, n - first)
            yield first, c
            first += c


# ---------------------------------------------------------------------------------------
# helper shapes: pl, G, Lz
# ---------------------------------------------------------------------------------------
def lambda_edges(n_bins: int, lam_min: float, lam_max: float) -> np.ndarray:
    j = np.arange(n_bins + 1, dtype=np.float64)
    e = lam_min * (lam_max / lam_min) ** (j / n_bins)
    e[0], e[-1] = lam_min, lam_max
    return e


def lambda_centres(edges: np.ndarray) -> np.ndarray:
    return np.sqrt(edges[:-1] * edges[1:])


def pl(lam, lam_c, beta):
    return np.minimum(1.0, (lam_c / lam) ** beta)


def gauss(x, x0, sig):
    return np.exp(-((x - x0) ** 2) / (2.0 * sig * sig))


def lorentz(x, x0, gamma):
    hw2 = (0.5 * gamma) ** 2
    return hw2 / ((x - x0) ** 2 + hw2)


def v_bin(edges: np.ndarray) -> int:
    """Index of the bin that contains 0.55 micron (reading R2)."""
    return int(np.searchsorted(edges, 0.55, side="right") - 1)


def kext_mixed(weight, kabs, ksca) -> np.ndarray:
    """Mass-weighted extinction, used only to scale the input density to a target tau_V."""
    w = np.asarray(weight, dtype=np.float64)[:, None]
    return (w * (kabs.astype(np.float64) + ksca.astype(np.float64))).sum(axis=0)


def _grey_single_species(edges, albedo, gval):
    lam = lambda_centres(edges)
    kabs = pl(lam, 1.0, 1.5)                       # reading R1
    if albedo >= 1.0:                              # pure scattering: no absorption at all
        ksca = kabs.copy()
        kabs = np.zeros_like(kabs)
    else:
        ksca = kabs * albedo / (1.0 - albedo)
    g = np.full_like(lam, gval)
    return (np.array([1.0]), kabs[None].astype(np.float32), ksca[None].astype(np.float32),
            g[None].astype(np.float32))


# ---------------------------------------------------------------------------------------
# C0 / C1: uniform sphere, central star
# ---------------------------------------------------------------------------------------
def sphere(n_root=16, tau_v=1.0, n_bins=64, lam_min=0.1, lam_max=1000.0, albedo=0.5,
           gval=0.0, n_packets=100_000, batch=10_000, seed=1, name="C0",
           T_star=5800.0) -> Workload:
    """Uniform dust sphere of radius 80 AU (= n_root/2 cells) in a 160 AU box (R8)."""
    box = 160.0 * AU
    h = box / n_root
    R_cells = n_root / 2.0
    edges = lambda_edges(n_bins, lam_min, lam_max)
    w, kabs, ksca, g = _grey_single_species(edges, albedo, gval)
    kv = kext_mixed(w, kabs, ksca)[v_bin(edges)]
    rho0 = tau_v / (kv * R_cells * h)
    c = np.arange(n_root, dtype=np.float64) + 0.5 - R_cells
    r2 = c[None, None, :] ** 2 + c[None, :, None] ** 2 + c[:, None, None] ** 2   # [z,y,x]
    rho = np.where(r2 < R_cells * R_cells, rho0, 0.0).astype(np.float32).ravel()
    ctr = (0.5 * box,) * 3
    return Workload(name=name, n_root=n_root, sub=0, origin=(0.0, 0.0, 0.0), root_size=h,
                    refine=None, rho_root=rho, rho_sub=None, lambda_edges_um=edges,
                    weight=w, kabs=kabs, ksca=ksca, g=g,
                    sources=[Source(SRC_POINT, ctr, LSUN, T_star)],
                    n_packets=n_packets, batch=batch, seed=seed,
                    meta=dict(tau_v=tau_v, rho0=rho0, R_cm=R_cells * h, albedo=albedo,
                              g=gval))


def c0(**kw) -> Workload:
    return sphere(**kw)


def c1(tau_v=1.0, n_root=64, n_packets=10_000_000, batch=1 << 20, **kw) -> Workload:
    return sphere(n_root=n_root, tau_v=tau_v, n_bins=128, lam_min=0.05, lam_max=1000.0,
                  albedo=0.5, gval=0.6, n_packets=n_packets, batch=batch,
                  name=f"C1_tau{tau_v:g}", **kw)


# ---------------------------------------------------------------------------------------
# C2 / C3: flared disk, five synthetic species, two-level grid
# ---------------------------------------------------------------------------------------
def disk_species(edges):
    lam = lambda_centres(edges)
    x = 1.0 / lam
    uv = pl(lam, 0.1, 2.0) + 1.5 * lorentz(x, 4.6, 1.0)
    bands = 3.3 * (20.0 / 3.3) ** (np.arange(17) / 16.0)
    kabs, ksca, g = [], [], []
    # silicate (10 micron bump on silicate only, R31)
    kabs.append(pl(lam, 0.3, 2.0) + 0.004 * gauss(lam, 9.7, 1.5))
    ksca.append(pl(lam, 0.3, 2.0) * pl(lam, 1.0, 2.0))
    g.append(0.6 * pl(lam, 1.0, 1.0))
    # amorphous carbon
    ka = 1.5 * pl(lam, 0.5, 1.2)
    kabs.append(ka)
    ksca.append(ka * pl(lam, 1.0, 2.8))
    g.append(0.5 * pl(lam, 1.0, 1.0))
    # graphite, 2175 A Lorentzian
    kabs.append(2.0 * uv)
    ksca.append(np.zeros_like(lam))
    g.append(np.zeros_like(lam))
    # PAH with 30 and 200 C atoms: 17 synthetic Lorentzian bands + graphite-like hard UV
    for lam_cut, a_n in ((0.4, 0.01), (0.8, 0.02)):
        b = sum(lorentz(lam, lk, 0.03 * lk) for lk in bands)
        kabs.append(2.0 * uv / (1.0 + (lam / lam_cut) ** 4) + a_n * b)
        ksca.append(np.zeros_like(lam))
        g.append(np.zeros_like(lam))
    w = np.array([31.0, 150.0, 50.0, 15.0, 15.0])
    w = w / w.sum()
    f32 = lambda a: np.asarray(a, dtype=np.float32)
    return w, f32(kabs), f32(ksca), f32(g)


def _disk_rho(x, y, z, planet):
    """Density / rho0 at positions in units of r0 (arrays broadcast)."""
    r = np.sqrt(x * x + y * y)
    rs = np.maximum(r, 1e-30)
    hh = 0.05 * rs ** 1.125
    rho = (1.0 / rs) * np.exp(-(z * z) / (2.0 * hh * hh))
    rho = np.where((r >= 1.0) & (r <= 20.0), rho, 0.0)
    if planet:
        f_gap = 1.0 - 0.99 * gauss(r, 10.0, 1.0)
        psi = np.arctan2(y, x) - np.log(rs / 10.0) / np.tan(np.deg2rad(15.0))
        psi = (psi + np.pi) % (2.0 * np.pi) - np.pi
        rho = rho * f_gap * (1.0 + gauss(psi, 0.0, 0.3))
    return rho


def disk(n_root=128, planet=False, n_packets=100_000_000, batch=1 << 22, seed=1,
         tau_v=100.0, name=None, refine_on=True) -> Workload:
    r0 = AU
    S = 4
    half = 20.0
    h = 2.0 * half / n_root                        # root cube edge in r0
    edges = lambda_edges(200, 0.05, 1000.0)
    w, kabs, ksca, g = disk_species(edges)
    kv = kext_mixed(w, kabs, ksca)[v_bin(edges)]
    rho0 = tau_v / (kv * r0 * np.log(20.0))
    c = -half + (np.arange(n_root, dtype=np.float64) + 0.5) * h
    X, Y, Z = c[None, None, :], c[None, :, None], c[:, None, None]
    rho_root = _disk_rho(X, Y, Z, planet) * rho0
    rsph2 = X * X + Y * Y + Z * Z
    refine = rsph2 < 25.0
    if planet:
        rc = np.sqrt(X * X + Y * Y)
        hh = 0.05 * np.maximum(rc, 1e-30) ** 1.125
        refine = refine | ((np.abs(rc - 10.0) <= 1.0) & (np.abs(Z) <= 2.0 * hh))
    refine = np.broadcast_to(refine, (n_root,) * 3)
    if not refine_on:
        refine = np.zeros((n_root,) * 3, dtype=bool)
    refine_flat = np.ascontiguousarray(refine).ravel()
    ridx = np.flatnonzero(refine_flat)
    rho_sub = None
    if len(ridx):
        iz, iy, ix = np.unravel_index(ridx, (n_root,) * 3)
        o = (np.arange(S, dtype=np.float64) + 0.5) * (h / S)
        # in-block order x fastest: index = sx + S*(sy + S*sz)
        sx = o[None, None, None, :]
        sy = o[None, None, :, None]
        sz = o[None, :, None, None]
        x0 = (-half + ix * h)[:, None, None, None]
        y0 = (-half + iy * h)[:, None, None, None]
        z0 = (-half + iz * h)[:, None, None, None]
        rho_sub = (_disk_rho(x0 + sx, y0 + sy, z0 + sz, planet) * rho0)
        rho_sub = rho_sub.astype(np.float32).reshape(-1)
    rho_root = np.where(refine, 0.0, rho_root).astype(np.float32).ravel()
    return Workload(name=name or ("C3" if planet else "C2"), n_root=n_root, sub=S,
                    origin=(-half * r0,) * 3, root_size=h * r0,
                    refine=refine_flat.astype(np.uint8), rho_root=rho_root, rho_sub=rho_sub,
                    lambda_edges_um=edges, weight=w, kabs=kabs, ksca=ksca, g=g,
                    sources=[Source(SRC_POINT, (0.0, 0.0, 0.0), LSUN, 4000.0)],
                    n_packets=n_packets, batch=batch, seed=seed,
                    meta=dict(tau_v=tau_v, rho0=rho0, r0=r0))


def c2(**kw) -> Workload:
    return disk(n_root=kw.pop("n_root", 128), planet=False, **kw)


def c3(**kw) -> Workload:
    return disk(n_root=kw.pop("n_root", 256), planet=True, **kw)


# ---------------------------------------------------------------------------------------
# C4: clumpy cube, 10 interior point sources + external isotropic field
# ---------------------------------------------------------------------------------------
def lognormal_field(n: int, corr_cells: float, sigma_ln: float, seed: int) -> np.ndarray:
    """Periodic lognormal field, mean 1: white noise smoothed by a Gaussian of std
    corr_cells (FFT), standardised, exponentiated."""
    import scipy.fft as sfft
    rng = np.random.default_rng(seed)
    wn = rng.standard_normal((n, n, n), dtype=np.float32)
    k = np.fft.fftfreq(n).astype(np.float32) * (2.0 * np.pi)
    kr = np.fft.rfftfreq(n).astype(np.float32) * (2.0 * np.pi)
    s2 = np.float32(0.5 * corr_cells * corr_cells)
    f = sfft.rfftn(wn, workers=-1)
    del wn
    f *= np.exp(-s2 * k * k)[:, None, None]
    f *= np.exp(-s2 * k * k)[None, :, None]
    f *= np.exp(-s2 * kr * kr)[None, None, :]
    gfield = sfft.irfftn(f, s=(n, n, n), workers=-1)
    del f
    gfield -= gfield.mean(dtype=np.float64)
    gfield /= np.sqrt((gfield.astype(np.float64) ** 2).mean())
    rho = np.exp(sigma_ln * gfield - 0.5 * sigma_ln * sigma_ln)
    rho /= rho.mean(dtype=np.float64)
    return rho.astype(np.float32)


def c4(n_root=512, n_packets=1_000_000_000, batch=1 << 24, seed=1, tau_v=10.0,
       corr_cells=8.0) -> Workload:
    """BASELINE.json configs[4]: clumpy cube, ten interior stars + an external field.  Deviation from
    SURVEY.md 8(d), which proposed drawing the field and the star positions from Philox SETUP blocks:
    they come from numpy's default_rng(seed) / default_rng(seed + 1000) -- an input generator shared by
    both sides needs no tie to the method's own generator, and neither side redraws them."""
    h = 1.0 * AU
    edges = lambda_edges(128, 0.05, 1000.0)
    w, kabs, ksca, g = _grey_single_species(edges, 0.6, 0.5)
    kv = kext_mixed(w, kabs, ksca)[v_bin(edges)]
    rho_mean = tau_v / (kv * n_root * h)
    rho = lognormal_field(n_root, corr_cells, 1.0, seed) * np.float32(rho_mean)
    rng = np.random.default_rng(seed + 1000)
    pos = (0.1 + 0.8 * rng.random((10, 3))) * (n_root * h)
    srcs = [Source(SRC_POINT, tuple(p), LSUN, 5800.0) for p in pos]
    srcs.append(Source(SRC_EXTERNAL, (0.0, 0.0, 0.0), LSUN, 1.0e4))
    return Workload(name="C4", n_root=n_root, sub=0, origin=(0.0, 0.0, 0.0), root_size=h,
                    refine=None, rho_root=rho.ravel(), rho_sub=None, lambda_edges_um=edges,
                    weight=w, kabs=kabs, ksca=ksca, g=g, sources=srcs,
                    n_packets=n_packets, batch=batch, seed=seed,
                    meta=dict(tau_v=tau_v, rho_mean=rho_mean))


# ---------------------------------------------------------------------------------------
# tiny random grids for brute-force pins (tests only; no config of the paper)
# ---------------------------------------------------------------------------------------
def tiny_random(n_root=2, sub=0, n_refined=0, seed=0, tau_cell=0.7, albedo=0.5, gval=0.3,
                n_bins=16, n_packets=20000, batch=5000, external=False,
                off_centre=True) -> Workload:
    rng = np.random.default_rng(seed)
    h = 10.0 * AU
    edges = lambda_edges(n_bins, 0.1, 1000.0)
    w, kabs, ksca, g = _grey_single_species(edges, albedo, gval)
    kv = kext_mixed(w, kabs, ksca)[v_bin(edges)]
    n3 = n_root ** 3
    rho_root = (rng.random(n3) * 2.0 * tau_cell / (kv * h)).astype(np.float32)
    if n3 > 2:
        rho_root[rng.integers(n3)] = 0.0                       # one empty cell
    refine, rho_sub = None, None
    if sub > 1 and n_refined > 0:
        refine = np.zeros(n3, dtype=np.uint8)
        refine[rng.choice(n3, size=n_refined, replace=False)] = 1
        rho_sub = (rng.random(n_refined * sub ** 3) * 2.0 * tau_cell * sub / (kv * h))
        rho_sub = rho_sub.astype(np.float32)
        rho_root[refine == 1] = 0.0
    if off_centre:
        p = tuple((0.15 + 0.7 * rng.random(3)) * n_root * h)
    else:
        p = (0.5 * n_root * h,) * 3
    srcs = [Source(SRC_POINT, p, LSUN, 5800.0)]
    if external:
        srcs.append(Source(SRC_EXTERNAL, (0.0, 0.0, 0.0), 0.5 * LSUN, 8000.0))
    return Workload(name=f"tiny{n_root}_{sub}_{n_refined}", n_root=n_root,
                    sub=sub if (sub > 1 and n_refined > 0) else 0, origin=(0.0, 0.0, 0.0),
                    root_size=h, refine=refine, rho_root=rho_root, rho_sub=rho_sub,
                    lambda_edges_um=edges, weight=w, kabs=kabs, ksca=ksca, g=g, sources=srcs,
                    n_packets=n_packets, batch=batch, seed=seed + 1)


# ---------------------------------------------------------------------------------------
# transiently heated PAH: input description only
# ---------------------------------------------------------------------------------------
@dataclass
class Pah:
    n_C: int                 # carbon atoms per molecule
    mass_fraction: float     # of the dust mass
    kabs: np.ndarray         # float32 [n_bins] absorption of the PAH per gram of the dust MIX (part of the mix's kappa_abs)
    theta_K: float = 500.0   # temperature scale of the synthetic enthalpy law (R37)
    T_lo: float = 5.0
    T_hi: float = 1.0e4
    n_Tp: int = 128


def pah_share(wl: Workload, n_C=100, mass_fraction=0.05, uv_share=0.4, band_share=0.2) -> Pah:
    """A synthetic PAH living inside the workload's dust mix: it takes `uv_share` of the mix's
    absorption below 0.4 micron, falling off towards the visible, plus `band_share` in 17
    Lorentzian bands between 3.3 and 20 micron (the shape of BASELINE.json configs[2]; the real
    cross-sections and band table are not available)."""
    lam = lambda_centres(wl.lambda_edges_um)
    kmix = (np.asarray(wl.weight, np.float64)[:, None] * wl.kabs.astype(np.float64)).sum(axis=0)
    bands = 3.3 * (20.0 / 3.3) ** (np.arange(17) / 16.0)
    share = uv_share / (1.0 + (lam / 0.4) ** 4) + band_share * np.clip(
        sum(lorentz(lam, lk, 0.03 * lk) for lk in bands), 0.0, 1.0)
    return Pah(n_C=n_C, mass_fraction=mass_fraction,
               kabs=(np.clip(share, 0.0, 1.0) * kmix).astype(np.float32))
