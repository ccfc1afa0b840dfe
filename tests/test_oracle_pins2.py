"""More pins of the fp64 oracle (CPU only, -m "not gpu"): the parts round 1 left to GPU<->oracle
agreement ("Oracle pins that are still absent"; SURVEY.md 8(c) pins table).

  * O4 / R26  source pick proportional to L_s, including the boundary case Lcdf[s] == u;
  * O7        mass of a sub-cell = rho_sub V / S^3, through a two-batch run of an all-refined grid
              whose temperatures obey 4 pi m_i Q(T_i) = cum_i L / N_cum with m_i formed here;
  * O6 / R15, R16  albedo and g indexed PER BIN: a two-valued albedo and g over the bins, and the
              scattering fraction / mean scattering cosine measured per bin from packet traces.
"""
import math

import numpy as np
import pytest

from paper_1201_3588_b200 import workloads as W


# =========================================================================================
# O4 / R26: source selection
# =========================================================================================
def _three_source_workload(L):
    wl = W.tiny_random(n_root=4, seed=21, external=True)
    h = wl.root_size
    wl.sources = [W.Source(W.SRC_POINT, (0.7 * h, 1.3 * h, 2.2 * h), L[0], 5800.0),
                  W.Source(W.SRC_POINT, (3.1 * h, 2.6 * h, 0.4 * h), L[1], 4000.0),
                  W.Source(W.SRC_EXTERNAL, (0.0, 0.0, 0.0), L[2], 1.0e4)]
    return wl


def _source_of_start(wl, x):
    """Which source a package started from, from its start position only (root-cube units)."""
    for s, src in enumerate(wl.sources):
        if src.type == W.SRC_POINT and np.allclose(x, np.array(src.pos) / wl.root_size, atol=1e-12):
            return s
    on_face = np.any((np.abs(x) < 1e-12) | (np.abs(x - wl.n_root) < 1e-12))
    assert on_face, x
    return 2


def test_source_pick_proportional_to_luminosity(oracle_mod):
    """Two point sources with L ratio 3:1 plus an external field: the number of packages from
    each source is within 4 sigma of L_s / sum L, and package by package the source is
    min{s : Lambda_s >= u0} with Lambda formed HERE from the luminosities and u0 = first word
    of the package's EMIT block (O4)."""
    O = oracle_mod
    L = np.array([3.0, 1.0, 2.0]) * W.LSUN
    wl = _three_source_workload(L)
    o = O.Oracle(wl)
    n = 30000
    lam = np.cumsum(L) / L.sum()
    got = np.zeros(3)
    for p in range(n):
        x, d, b, slot = o.emit(9, p)
        s = _source_of_start(wl, x)
        got[s] += 1
        u0 = O.draw4(9, p, 0, 0)[0]
        assert s == int(np.searchsorted(lam, u0, side="left")), p
    frac = L / L.sum()
    sig = np.sqrt(n * frac * (1 - frac))
    assert np.all(np.abs(got - n * frac) < 4 * sig), (got, n * frac)
    # the spectra follow the sources too: mean emitted wavelength bin ordered as 1e4 K < 5800 K < 4000 K
    t = o.tables()
    assert np.allclose(t["Lcdf"], lam, rtol=1e-15)


def test_source_pick_boundary_case(oracle_mod):
    """Lcdf[0] == u0 exactly must pick source 0 ("first s with Lambda_s >= u").  L_0 = v,
    L_1 = 1 - v with v = the u0 of a chosen package (v >= 0.5, so that 1 - v and v + (1 - v) = 1
    are exact in fp64 and Lambda_0 = v bit for bit)."""
    O = oracle_mod
    pid, v = next((p, O.draw4(5, p, 0, 0)[0]) for p in range(1000) if O.draw4(5, p, 0, 0)[0] >= 0.5)
    assert v + (1.0 - v) == 1.0
    wl = _three_source_workload([v, 1.0 - v, 1.0])
    wl.sources = wl.sources[:2]
    o = O.Oracle(wl)
    assert o.tables()["Lcdf"][0] == v
    x, *_ = o.emit(5, pid)
    assert _source_of_start(wl, x) == 0
    # a package whose u0 is the next representable number above v goes to source 1
    wl.sources[0].L = math.nextafter(v, 0.0)
    wl.sources[1].L = 1.0 - wl.sources[0].L
    o = O.Oracle(wl)
    assert o.tables()["Lcdf"][0] < v
    x, *_ = o.emit(5, pid)
    assert _source_of_start(wl, x) == 1


# =========================================================================================
# O7: sub-cell mass and the temperature identity on an all-refined grid with T feedback
# =========================================================================================
def test_subcell_mass_and_temperature_identity_two_batches(oracle_mod):
    O = oracle_mod
    wl = W.tiny_random(n_root=2, sub=4, n_refined=8, seed=31, albedo=0.3, tau_cell=1.5,
                       n_packets=60000, batch=30000)
    assert wl.n_ref == 8 and wl.leaf_slots == 8 + 8 * 64
    o = O.Oracle(wl).run()                       # two batches: T of batch 1 feeds re-emission of batch 2
    t = o.tables()
    n, eps = o.cell_energy()
    T = o.cell_temperature()
    V = wl.root_size ** 3
    # (a) the mass of a sub-cell, formed here from the inputs
    for slot in (8, 8 + 17, 8 + 511):
        assert o.leaf_mass(slot) == pytest.approx(float(wl.rho_sub[slot - 8]) * V / 64.0, rel=1e-13)
    assert o.leaf_mass(3) == 0.0                  # the slot of a refined cube holds no dust (R22)
    # (b) identity per sub-cell with Q from its definition and m formed here
    m = wl.rho_sub.astype(np.float64) * V / 64.0
    idx = np.flatnonzero((n[8:] > 0) & (m > 0))
    assert len(idx) > 300
    nu, dnu, ka = t["nu"], t["dnu"], t["kabs"]
    lhs_sum, n_unclamped = 0.0, 0
    for i in idx:
        Ti = T[8 + i]
        if not (1.0 < Ti < 1.0e4):
            continue
        Q = sum(k * O.planck(v, Ti) * dv for k, v, dv in zip(ka, nu, dnu))
        lhs = 4 * math.pi * m[i] * Q
        assert lhs == pytest.approx(n[8 + i] * eps, rel=3e-5), i
        lhs_sum += lhs
        n_unclamped += 1
    assert n_unclamped > 300
    # (c) summed over the cells: the absorbed power (SURVEY pins table, "Temperature inversion")
    sel = np.array([1.0 < T[8 + i] < 1.0e4 for i in idx])
    assert lhs_sum == pytest.approx(float(n[8:][idx][sel].sum()) * eps, rel=1e-5)
    assert eps == pytest.approx(sum(s.L for s in wl.sources) / 60000, rel=1e-14)
    assert n[:8].sum() == 0


def test_split_invariance_with_temperature_feedback(oracle_mod):
    """Refining every cube of a UNIFORM-density grid: with two batches the temperatures feed
    back into re-emission.  Root-aggregated absorbed counts must agree statistically and the
    temperature of the aggregated cube (from sum of counts and sum of masses) must agree with
    the unrefined grid's -- a sub-cell mass off by S^3 would move T by 64^(1/(4+beta))."""
    O = oracle_mod
    base = W.tiny_random(n_root=2, seed=12, albedo=0.2, n_packets=40000, batch=20000)
    base.rho_root[:] = base.rho_root.max()
    a = O.Oracle(base).run()
    fine = W.tiny_random(n_root=2, seed=12, albedo=0.2, n_packets=40000, batch=20000)
    fine.sub = 4
    fine.refine = np.ones(8, dtype=np.uint8)
    fine.rho_sub = np.repeat(base.rho_root, 64).astype(np.float32)
    fine.rho_root = np.zeros(8, dtype=np.float32)
    b = O.Oracle(fine).run()
    na, eps = a.cell_energy()
    nb_ = b.cell_energy()[0][8:].reshape(8, 64).sum(axis=1)
    assert np.all(np.abs(na[:8].astype(float) - nb_) < 4 * np.sqrt(na[:8] + nb_) + 5)
    V = base.root_size ** 3
    for r in range(8):
        q = float(nb_[r]) * eps / (4 * math.pi * float(base.rho_root[r]) * V)
        assert b.temperature_from_q(q) == pytest.approx(a.cell_temperature()[r], rel=0.02)
    # (the thermal SEDs legitimately differ: sub-cells near the source are hotter than their cube's mean)


# =========================================================================================
# O6: albedo and g are per-bin quantities
# =========================================================================================
def test_albedo_and_g_indexed_per_bin(oracle_mod):
    """Even bins: albedo 0.25, g = 0.1; odd bins: albedo 0.8, g = 0.7.  From packet traces, per
    bin: scatterings / interactions = that bin's albedo and <cos theta> of the scatterings =
    that bin's g (4 sigma).  An implementation that indexed albedo or g with anything but the
    package's current bin (a constant, the emission bin, the re-emitted bin) fails."""
    O = oracle_mod
    wl = W.sphere(n_root=8, tau_v=4.0, n_bins=16, n_packets=6000, batch=6000)
    nb = wl.n_bins
    alb = np.where(np.arange(nb) % 2 == 0, 0.25, 0.8)
    gg = np.where(np.arange(nb) % 2 == 0, 0.1, 0.7)
    kabs = np.ones(nb)
    wl.kabs = kabs[None].astype(np.float32)
    wl.ksca = (kabs * alb / (1 - alb))[None].astype(np.float32)
    wl.g = gg[None].astype(np.float32)
    wl.rho_root = (wl.rho_root > 0).astype(np.float32) * np.float32(
        4.0 / ((1.0 + 4.0) * 4 * wl.root_size))           # tau ~ 4 in the odd bins, ~1 in the even ones
    o = O.Oracle(wl)
    o.set_cell_temperature(300.0)                          # re-emission spread over several bins
    t = o.tables()
    assert np.allclose(t["alb"], alb, rtol=1e-6) and np.allclose(t["g"], gg, rtol=1e-6)
    n_sca, n_abs = np.zeros(nb), np.zeros(nb)
    cs_sum, cs_sq = np.zeros(nb), np.zeros(nb)
    for p in range(wl.n_packets):
        ty, bn, sl, xyz = o.trace_packet(wl.seed, p, cap=4096)
        assert ty[-1] == 3
        for i in range(1, len(ty) - 1):
            b = bn[i - 1]                                  # bin the package flew in when it interacted
            if ty[i] == 1:
                n_sca[b] += 1
                d_in = xyz[i] - xyz[i - 1]
                d_out = xyz[i + 1] - xyz[i]
                c = float(d_in @ d_out / (np.linalg.norm(d_in) * np.linalg.norm(d_out)))
                cs_sum[b] += c
                cs_sq[b] += c * c
            elif ty[i] == 2:
                n_abs[b] += 1
    tot = n_sca + n_abs
    used = tot > 400
    assert used[::2].any() and used[1::2].any() and used.sum() >= 6
    frac = n_sca[used] / tot[used]
    sig = np.sqrt(alb[used] * (1 - alb[used]) / tot[used])
    assert np.all(np.abs(frac - alb[used]) < 4 * sig), (frac, alb[used])
    mean_c = cs_sum[used] / n_sca[used]
    var_c = cs_sq[used] / n_sca[used] - mean_c ** 2
    assert np.all(np.abs(mean_c - gg[used]) < 4 * np.sqrt(var_c / n_sca[used]) + 1e-3), (mean_c, gg[used])
