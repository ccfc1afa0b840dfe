"""Pins of the oracle's transiently heated PAH (O11..O13; "extended
to the treatment of transiently heated PAHs", L45 Fig. 3, L49).  The paper gives no formula and the
book it cites is not available: the method is the reading R35..R40 of DESIGN.md, and what fixes it
here are the limits the physics prescribes, not values of the paper.  CPU only."""
import math

import numpy as np
import pytest

from paper_1201_3588_b200 import workloads as W

H, CL, KB = 6.62607015e-27, 2.99792458e10, 1.380649e-16
M_C = 1.99264687992e-23


def _planck(nu, T):
    x = H * nu / (KB * T)
    with np.errstate(over="ignore"):
        return np.where(x < 700, 2 * H * nu ** 3 / CL ** 2 / np.expm1(np.minimum(x, 700)), 0.0)


def _setup(O, n_C=100, n_Tp=128, T_hi=1.0e4, **kw):
    wl = W.c0(n_packets=20000, batch=10000)
    pah = W.pah_share(wl, n_C=n_C, **kw)
    pah.n_Tp, pah.T_hi = n_Tp, T_hi
    o = O.Oracle(wl)
    o.set_pah(pah.n_C, pah.mass_fraction, pah.kabs, pah.theta_K, pah.T_lo, pah.T_hi, pah.n_Tp)
    return wl, pah, o


def _cooling_power(o, pah, T):
    """Lambda(T) = 4 pi sum_j C_j B_j(T) dnu_j of one molecule, formed here from the inputs."""
    t = o.tables()
    kmix_share = pah.kabs.astype(np.float64)
    Cmol = kmix_share * pah.n_C * M_C / pah.mass_fraction
    return 4 * math.pi * float((Cmol * _planck(t["nu"], T) * t["dnu"]).sum())


def test_enthalpy_law(oracle_mod):
    """R37: U(T) = integral of C(T); C -> 3 N k at high T and ~ T^2 at low T."""
    wl, pah, o = _setup(oracle_mod)
    for T in (20.0, 300.0, 2500.0):
        xs = np.linspace(0.0, T, 20001)
        C = np.array([o.pah_heat_capacity(x) for x in xs[::50]])
        U_num = np.trapezoid(C, xs[::50])
        assert o.pah_enthalpy(T) == pytest.approx(U_num, rel=2e-5)
    assert o.pah_heat_capacity(1e6) == pytest.approx(3 * 100 * KB, rel=1e-6)
    assert o.pah_heat_capacity(10.0) / o.pah_heat_capacity(5.0) == pytest.approx(4.0, rel=1e-3)
    g = o.pah_grid()
    assert np.allclose(g["U"], [o.pah_enthalpy(T) for T in g["T"]], rtol=1e-14)
    assert np.allclose(g["Lam"], [_cooling_power(o, pah, T) for T in g["T"]], rtol=1e-6)
    assert np.allclose(g["q"], np.minimum(1.0, pah.kabs / np.maximum(o.tables()["kext"] * (1 - o.tables()["alb"]), 1e-300)),
                       rtol=1e-6)


def test_mean_heating_equals_mean_cooling(oracle_mod):
    """Stationarity of the linear-sharing scheme: sum_{k>=1} P_k Lambda(T_k) = sum_j R_j h nu_j exactly
    (as long as no photon carries the molecule beyond the last state), for any rates."""
    wl, pah, o = _setup(oracle_mod, n_Tp=96, T_hi=2.0e4)
    g = o.pah_grid()
    E = H * o.tables()["nu"]
    rng = np.random.default_rng(2)
    for scale in (1e-9, 1e-4, 1e1, 1e2):
        R = rng.random(o.nb) * scale * (g["Cmol"] > 0)
        P, cdf = o.pah_solve(R)
        assert P.min() >= 0 and P.sum() == pytest.approx(1.0, abs=1e-12) and P[-1] < 1e-10
        assert float((P[1:] * g["Lam"][1:]).sum()) == pytest.approx(float((R * E).sum()), rel=1e-9)
        assert np.all(np.diff(cdf) >= -1e-15) and cdf[-1] == 1.0


def test_strong_heating_limit_is_the_equilibrium_temperature(oracle_mod):
    """A very large grain (10^5 C atoms) bathed in soft photons (E << U): P(T) collapses onto the
    temperature at which the heating power equals the cooling power Lambda(T_eq)."""
    wl, pah, o = _setup(oracle_mod, n_C=100_000, n_Tp=400, T_hi=3000.0)
    t = o.tables()
    E = H * t["nu"]
    lam = CL / t["nu"] * 1e4
    soft = (lam > 8.0) & (lam < 12.0) & (pah.kabs > 0)               # ~0.1 eV photons
    assert soft.any()
    T_eq = 250.0
    power = _cooling_power(o, pah, T_eq)
    R = np.zeros(o.nb)
    R[soft] = power / (E[soft].sum())                                  # sum_j R_j E_j = Lambda(T_eq)
    assert E[soft].max() < 1e-3 * o.pah_enthalpy(T_eq)
    P, _ = o.pah_solve(R)
    g = o.pah_grid()
    mean_T = float((P * g["T"]).sum())
    std_T = math.sqrt(float((P * (g["T"] - mean_T) ** 2).sum()))
    assert mean_T == pytest.approx(T_eq, rel=0.01)
    assert std_T / mean_T < 0.08                  # a few bins of the T grid wide (numerical diffusion of the scheme) ...
    assert P[np.abs(g["T"] / T_eq - 1) > 0.3].sum() < 1e-6      # ... and nothing far from T_eq
    # refining the grid narrows the peak towards the delta function of the limit
    wl2, pah2, o2 = _setup(oracle_mod, n_C=100_000, n_Tp=1600, T_hi=3000.0)
    P2, _ = o2.pah_solve(R)
    g2 = o2.pah_grid()
    m2 = float((P2 * g2["T"]).sum())
    s2 = math.sqrt(float((P2 * (g2["T"] - m2) ** 2).sum()))
    assert m2 == pytest.approx(T_eq, rel=0.003) and s2 < 0.6 * std_T


def test_single_photon_limit_is_the_cooling_curve(oracle_mod):
    """Rare hard photons (the molecule cools completely between two of them): starting from the ground
    state one photon of energy E lifts it to U(T_peak) = U_0 + E, from where it slides down through
    every state, spending the time (U_k - U_{k-1}) / Lambda(T_k) in state k.  Hence
    P_k = R (U_k - U_{k-1}) / Lambda_k below the peak, O(R^2) above it, the weights of the two states
    that bracket the peak share as the scheme prescribes, and sum_{k>0} P_k = R t_cool."""
    wl, pah, o = _setup(oracle_mod, n_Tp=160)
    g = o.pah_grid()
    t = o.tables()
    E = H * t["nu"]
    j = int(np.argmax((pah.kabs > 0) * E))                              # the hardest photon the PAH absorbs (~12 eV)
    rate = 1e-24                                                        # far below 1 / t_cool (~1e-13 per s down to 5 K)
    R = np.zeros(o.nb); R[j] = rate
    P, _ = o.pah_solve(R)
    U, Lam = g["U"], np.array([_cooling_power(o, pah, T) for T in g["T"]])
    Ustar = U[0] + E[j]
    f = int(np.searchsorted(U, Ustar, side="right") - 1)                # U_f <= U* < U_{f+1}
    assert 10 < f < len(U) - 2
    dwell = np.zeros_like(U); dwell[1:] = np.diff(U) / Lam[1:]
    w = (Ustar - U[f]) / (U[f + 1] - U[f])
    assert np.allclose(P[1:f + 1], rate * dwell[1:f + 1], rtol=1e-9)
    assert P[f + 1] == pytest.approx(rate * w * dwell[f + 1], rel=1e-9)
    assert P[f + 2:].max() < 1e-12 * P[f]                                # only reachable with a second photon: O(rate^2)
    assert 1.0 - P[0] == pytest.approx(rate * (dwell[1:f + 1].sum() + w * dwell[f + 1]), rel=1e-3)
    # harder photons reach higher temperatures ("P(T) depends strongly on the hardness")
    peaks = []
    for jj in np.flatnonzero(pah.kabs > 0)[::6]:
        Rj = np.zeros(o.nb); Rj[jj] = rate
        Pj, _ = o.pah_solve(Rj)
        peaks.append((E[jj], g["T"][np.flatnonzero(Pj > 0).max()]))
    peaks.sort()
    assert all(a[1] <= b[1] for a, b in zip(peaks, peaks[1:])) and peaks[-1][1] > 3 * peaks[0][1]


def test_emission_spectrum_from_PT(oracle_mod):
    """R39: the emission CDF of a molecule = cumulative sum over bins of C_j dnu_j sum_k P_k B_j(T_k)."""
    wl, pah, o = _setup(oracle_mod)
    g, t = o.pah_grid(), o.tables()
    rng = np.random.default_rng(5)
    R = rng.random(o.nb) * 1e-3 * (g["Cmol"] > 0)
    P, cdf = o.pah_solve(R)
    e = np.array([(P * g["Cmol"][j] * t["dnu"][j] * _planck(t["nu"][j], g["T"])).sum() for j in range(o.nb)])
    ref = np.cumsum(e) / e.sum()
    assert np.allclose(cdf[:-1], ref[:-1], rtol=1e-9, atol=1e-15) and cdf[-1] == 1.0
    # the emission of a hot PAH peaks in its bands, far bluer than the thermal emission of the cool grains
    lam = CL / t["nu"] * 1e4
    med = lam[np.searchsorted(cdf, 0.5)]
    assert 3.0 < med < 25.0


def test_absorptions_split_between_pah_and_equilibrium_grains(oracle_mod):
    """R36: a package absorbed in bin j is taken by the PAH with probability q_j = kappa_PAH,j / kappa_abs,j.
    With q in {0, 1/2, 1} over the bins: bins with q = 1 book every absorption on the PAH tally, bins
    with q = 0 none, the others half of them (binomial, 4 sigma); tallies add up to the counter."""
    O = oracle_mod
    wl = W.sphere(n_root=8, tau_v=3.0, albedo=0.3, n_bins=24, n_packets=40000, batch=20000)
    nb = wl.n_bins
    q = np.array([0.0, 0.5, 1.0])[np.arange(nb) % 3]
    o = O.Oracle(wl)
    kmix = o.tables()["kabs"].copy()
    o.set_pah(60, 0.1, (q * kmix).astype(np.float32), n_Tp=48)
    assert np.allclose(o.pah_grid()["q"], q, atol=1e-6)
    assert np.allclose(o.tables()["kabs"], (1 - q) * kmix, rtol=1e-6, atol=1e-30)   # what is left for equilibrium
    absorbed_in = np.zeros(nb)
    for p in range(4000):                                               # traces: the bin a package had when absorbed
        ty, bn, sl, xyz = o.trace_packet(wl.seed, p, cap=8192)
        for i in range(1, len(ty)):
            if ty[i] == 2:
                absorbed_in[bn[i - 1]] += 1
    o2 = O.Oracle(wl)
    o2.set_pah(60, 0.1, (q * kmix).astype(np.float32), n_Tp=48)
    o2.run_batch(wl.seed, 0, 4000)                                      # the same packages, first batch
    cumP, total = o2.pah_absorbed()
    per_bin = cumP.sum(axis=0).astype(float)
    n_eq, _ = o2.cell_energy()
    c = o2.counters()
    assert total == cumP.sum() and int(n_eq.sum()) + total == c["absorptions"]
    assert c["emitted"] == c["escaped"] == 4000
    assert np.array_equal(per_bin[q == 1.0], absorbed_in[q == 1.0])
    assert per_bin[q == 0.0].sum() == 0
    half = q == 0.5
    n = absorbed_in[half]
    assert n.sum() > 500
    assert np.all(np.abs(per_bin[half] - 0.5 * n) <= 4 * np.sqrt(0.25 * n) + 1)


def test_pah_run_heats_up_and_emits_in_the_bands(oracle_mod):
    """A whole run with PAH: the second batch re-emits from the P(T) of the first; the PAH packages reach
    the 3-6 micron bands, where the equilibrium grains of this sphere hardly emit."""
    O = oracle_mod
    wl = W.c0(n_packets=30000, batch=10000)
    pah = W.pah_share(wl, n_C=60, mass_fraction=0.05, uv_share=0.5, band_share=0.3)
    o = O.Oracle(wl)
    o.set_pah(pah.n_C, pah.mass_fraction, pah.kabs, n_Tp=64)
    o.run()
    base = O.Oracle(wl).run()
    lam = W.lambda_centres(wl.lambda_edges_um)
    mid = (lam > 3.0) & (lam < 6.0)                 # bluewards of what the ~100-300 K grains of this sphere emit
    assert o.sed()[2][mid].sum() > 2 * base.sed()[2][mid].sum() > 100
    cdf = o.pah_cdf()
    cumP, total = o.pah_absorbed()
    hot = np.flatnonzero(cumP.sum(axis=1) > 3)
    assert total > 1000 and len(hot) > 5
    assert np.all(cdf[hot, -1] == 1.0) and np.all(np.diff(cdf[hot], axis=1) >= -1e-15)
    # cells that absorbed nothing keep the cold row
    cold = np.flatnonzero(cumP.sum(axis=1) == 0)
    assert np.array_equal(cdf[cold[0]], cdf[cold[-1]])
    c = o.counters()
    assert c["emitted"] == c["escaped"] == 30000 and c["lost"] == 0
    # deterministic function of the tallies: recomputing from the counts reproduces the rows
    o.pah_update(cumP, 30000)
    assert np.array_equal(o.pah_cdf(), cdf)


def test_photon_rates_per_molecule_from_the_leaf_tallies(oracle_mod):
    """R40 (`pah_rates`, the input of O12): the absorption rate of ONE molecule in bin j is the leaf's
    absorbed PAH power in that bin, counts_j L_tot / N_cum, divided by the photon energy h nu_j and by
    the number of molecules in the leaf.  The molecule count is formed HERE from the inputs --
    mass fraction x rho x V / (N_C x 12 u), V = root_size^3 for a cube and (root_size / S)^3 for a
    subcube -- so a missing N_C, a missing mass fraction or a wrong sub-cell volume fails:
      sum_j R_j h nu_j n_mol = sum_j counts_j L_tot / N_cum            (energy, to 1e-12)
      sum_k P_k Lambda(T_k) n_mol = the same power                     (joins R to the pinned solver)
    on root leaves and sub-cells of a two-level grid after a real PAH run (the PAH sits
    in a heating bath fixed by the radiation field; the bath here is the leaf's own tally)."""
    O = oracle_mod
    wl = W.c2(n_root=8, n_packets=120_000, batch=40_000)
    assert wl.sub == 4 and wl.refine is not None and wl.refine.sum() > 0
    pah = W.pah_share(wl, n_C=60, mass_fraction=0.05, uv_share=0.5, band_share=0.3)
    o = O.Oracle(wl)
    o.set_pah(pah.n_C, pah.mass_fraction, pah.kabs, n_Tp=96, T_hi=2.0e4)
    o.run()
    counts, total = o.pah_absorbed()
    assert total > 500                                                  # (a 4000 K star: few hard photons)
    n3, S = wl.n_root ** 3, wl.sub
    edges_cm = np.asarray(wl.lambda_edges_um, np.float64) * 1e-4
    E = H * CL / np.sqrt(edges_cm[:-1] * edges_cm[1:])                  # h nu_j at the bin centres (R4)
    L_tot = sum(s.L for s in wl.sources)
    n_cum = wl.n_packets
    g = o.pah_grid()
    per_leaf = counts.sum(axis=1)
    hot = np.flatnonzero(per_leaf > 0)
    roots, subs = hot[hot < n3], hot[hot >= n3]
    assert len(roots) > 3 and len(subs) > 3                             # both kinds of leaf
    picked = list(roots[np.argsort(per_leaf[roots])[-4:]]) + list(subs[np.argsort(per_leaf[subs])[-6:]]) + [int(subs[0])]
    for slot in picked:
        if slot < n3:
            rho, V = float(wl.rho_root[slot]), wl.root_size ** 3
        else:
            rho, V = float(wl.rho_sub[slot - n3]), (wl.root_size / S) ** 3
        assert rho > 0
        n_mol = pah.mass_fraction * rho * V / (pah.n_C * M_C)
        R = o.pah_rates(slot, counts[slot], n_cum)
        power = float(counts[slot].astype(np.float64).sum()) * L_tot / n_cum
        assert float((R * E).sum()) * n_mol == pytest.approx(power, rel=1e-12)
        assert np.allclose(R * E * n_mol, counts[slot].astype(np.float64) * L_tot / n_cum, rtol=1e-12, atol=0.0)
        P, _ = o.pah_solve(R)
        assert P[-1] < 1e-12
        assert float((P[1:] * g["Lam"][1:]).sum()) * n_mol == pytest.approx(power, rel=1e-8)
    # twice the packages behind the same counts: every package carries half the energy
    R1, R2 = o.pah_rates(picked[0], counts[picked[0]], n_cum), o.pah_rates(picked[0], counts[picked[0]], 2 * n_cum)
    assert np.allclose(R2, 0.5 * R1, rtol=1e-15)
    # a leaf without dust, or without absorptions, has no rates
    empty = np.flatnonzero(np.concatenate([wl.rho_root, wl.rho_sub]) == 0)
    empty = [e for e in empty if e >= n3 or not wl.refine[e]]
    if empty:
        assert o.pah_rates(int(empty[0]), np.ones(o.nb, np.uint64), n_cum) is None
    assert o.pah_rates(int(picked[0]), np.zeros(o.nb, np.uint64), n_cum) is None
