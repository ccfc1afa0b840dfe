"""-m gpu: the configurations at their OWN size and length (VERDICT r02 row g; SURVEY.md 8(d) "Parity
twins": "the oracle runs C0 and C1 (tau_V <= 10) at full size").

configs[1] at tau_V = 0.1, 1, 10: all 10^7 packages in BASELINE.json's partition (9 batches of 2^20 and a
last one of 562 816) on both sides -- the temperatures feed back nine times -- compared by the rules of
tests/parity.py.  At this length cells with >= 10^3 absorptions exist (the central cells of the sphere), so
north_star's per-cell rules bite: absorbed energy within 3 sigma + 0.5 % and temperature within 1 % on those
cells, radial shells, SED per component within 2 % or 3 sigma, emitted-per-bin and accounting bit-exact, and
the GPU's temperature on EVERY leaf slot against the oracle's O7 applied to the GPU's tally."""
import numpy as np
import pytest

import parity as PR
from paper_1201_3588_b200 import workloads as W

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def M():
    import torch
    assert torch.cuda.is_available(), "-m gpu tests need a CUDA device"
    from paper_1201_3588_b200 import build, mcrt
    build.build_library()
    mcrt.lib()
    return mcrt


@pytest.mark.parametrize("tau_v,min_hot_cells", [(0.1, 4), (1.0, 100), (10.0, 1000)])
def test_c1_full_size(M, oracle_mod, tau_v, min_hot_cells):
    wl = W.c1(tau_v=tau_v)
    parts = list(wl.batches())
    assert wl.n_packets == 10_000_000 and len(parts) == 10 and parts[-1] == (9 << 20, 562_816)
    ctx = M.run_workload(wl)
    orc = oracle_mod.Oracle(wl).run()
    cg, co = ctx.get_counters(), orc.counters()
    PR.check_accounting(cg, co)
    assert cg["emitted"] == cg["escaped"] == 10_000_000 and cg["lost"] == 0
    ng, eps_g = ctx.get_cell_energy()
    no, eps_o = orc.cell_energy()
    sg, so = ctx.get_sed(), orc.sed()
    PR.check_self_consistency(cg, ng, sg)
    assert eps_g == pytest.approx(eps_o, rel=1e-12)
    n_cells, n_groups = PR.check_cell_energy(ng, no, min_count=1000, groups=PR.radial_shells(64, 16))
    assert n_cells >= min_hot_cells and n_groups >= 12, (n_cells, n_groups)
    Tg = ctx.get_cell_temperature()
    n_T = PR.check_temperature(Tg, orc.cell_temperature(), ng, no, min_count=1000)     # 1 % per cell
    assert n_T >= min_hot_cells, n_T
    PR.check_sed(sg, so)
    for k in ("absorptions", "scatterings", "crossings"):
        assert PR.counts_close(cg[k], co[k], 0.005), (k, cg[k], co[k])
    n_slots, n_hot = PR.check_temperature_of_tally(Tg, orc, ng, cg["emitted"])
    assert n_slots == len(ng) and n_hot > 100_000


def _temperature_identity(ctx, wl, n_abs, n_cum, sample=40000):
    """O7 on sampled leaf slots (cubes and subcubes) that are neither empty nor clamped:
    4 pi rho V Q(T) N_cum = n_abs L_tot, Q from the library's ln Q table interpolated in ln T as the
    update kernel does; density and volume per slot formed here from the inputs (layout R22)."""
    T = ctx.get_cell_temperature().astype(np.float64)
    _, lnQ, _ = ctx.get_tables()
    lnQ = lnQ.astype(np.float64)
    nT = len(lnQ)
    n3 = wl.n_root ** 3
    rho = np.asarray(wl.rho_root, dtype=np.float64).ravel()
    vol = np.full(n3, wl.root_size ** 3)
    if wl.n_ref:
        rho = np.concatenate([rho, np.asarray(wl.rho_sub, dtype=np.float64).ravel()])
        vol = np.concatenate([vol, np.full(wl.n_ref * wl.sub ** 3, (wl.root_size / wl.sub) ** 3)])
        rho[np.flatnonzero(np.asarray(wl.refine).ravel())] = 0.0           # the slot of a refined cube is unused
    assert len(rho) == len(n_abs) == len(T)
    idx = np.flatnonzero((n_abs > 0) & (rho > 0))
    idx = np.random.default_rng(3).choice(idx, size=min(sample, len(idx)), replace=False)
    t = np.log(T[idx]) / (np.log(1.0e4) / (nT - 1))                    # row coordinate on the default T grid
    ok = (t > 0.5) & (t < nT - 1.5)
    idx, t = idx[ok], t[ok]
    k = np.floor(t).astype(int)
    lnq_T = lnQ[k] + (t - k) * (lnQ[k + 1] - lnQ[k])
    Ltot = sum(s.L for s in wl.sources)
    lnq = np.log(n_abs[idx].astype(np.float64)) + np.log(Ltot / (n_cum * 4 * np.pi)) - np.log(rho[idx] * vol[idx])
    assert len(idx) > 1000
    if wl.n_ref:
        assert (idx >= n3).sum() > 100                                  # sub-cells among them
    assert np.abs(lnq_T - lnq).max() < 2e-3, np.abs(lnq_T - lnq).max()


def _groups(wl, name):
    if name == "c1_tau100":
        return [PR.radial_shells(64, 16)]
    if name == "c4":
        return [PR.super_blocks(512, 8), PR.super_blocks(512, 32)]
    return [PR.root_of_slot(wl), PR.blocks_of_slot(wl, 4), PR.blocks_of_slot(wl, 8)]


@pytest.mark.parametrize("name,maker,n_batches,last,sample", [
    ("c1_tau100", lambda: W.c1(tau_v=100.0), 10, (9 << 20, 562_816), 562_816),
    ("c2", W.c2, 24, (23 << 22, 3_531_008), 3_531_008),
    ("c3", W.c3, 24, (23 << 22, 3_531_008), 3_531_008),
    ("c4", W.c4, 60, (59 << 24, 10_144_256), 1 << 21)])
def test_full_length_run(M, oracle_mod, name, maker, n_batches, last, sample):
    """One run of the configuration from its first package to its last in BASELINE.json's batch
    partition (ragged last batch included), in the launch configuration bench.py times.

    Against the oracle AT THE END of the run, where the temperatures have been fed back n_batches - 1
    times: the GPU's cumulative tally after the last-but-one batch is handed to the oracle's
    temperature step (O7), then both sides transport the same packages of the last batch with those
    temperatures frozen, and the batch's INCREMENTS are compared by north_star's rules -- emitted per
    bin bit-exact, leaf / shell / super-block absorptions within 3 sigma + 0.5 %, SED per component
    within 2 % or 3 sigma, event totals.  (A short twin run is no yardstick for the end state: its first
    batch re-emits at the start temperature, which is 1/4 of a 4-batch twin but 1/24 of the run -- the
    SEDs differ by 80 %, measured.)  On C4 the oracle takes the first 2^21 packages of the last batch and
    the GPU runs that batch in two pieces.  Then the invariants of the whole run: every package
    accounted for exactly, none lost, tallies consistent, and the temperature identity (O7) on
    sampled leaves."""
    wl = maker()
    parts = list(wl.batches())
    assert len(parts) == n_batches and parts[-1] == last and sum(c for _, c in parts) == wl.n_packets
    ctx = M.from_workload(wl)
    for first, cnt in parts[:-1]:
        ctx.run_batch(wl.seed, first, cnt)
    n_prev, _ = ctx.get_cell_energy()
    sed_prev, c_prev = ctx.get_sed(), ctx.get_counters()
    first, cnt = parts[-1]
    assert c_prev["emitted"] == c_prev["escaped"] == first and c_prev["lost"] == 0
    ns = min(cnt, sample)
    ctx.run_batch(wl.seed, first, ns)
    n_now, _ = ctx.get_cell_energy()
    sed_now, c_now = ctx.get_sed(), ctx.get_counters()
    orc = oracle_mod.Oracle(wl)
    orc.update_temperature(n_prev, first)                      # the temperatures the GPU's last batch sees
    orc.run_batch(wl.seed, first, ns)
    co = orc.counters()
    no, _ = orc.cell_energy()
    dn = (n_now - n_prev).astype(np.int64)
    assert np.array_equal((c_now["emitted_per_bin"] - c_prev["emitted_per_bin"]).astype(np.int64),
                          co["emitted_per_bin"].astype(np.int64))
    assert c_now["emitted"] - c_prev["emitted"] == co["emitted"] == co["escaped"] == ns
    n_cells = n_groups = 0
    for g in _groups(wl, name):
        n_cells, k = PR.check_cell_energy(dn, no, min_count=1000, groups=g)
        n_groups += k
    assert n_groups > 10, (n_cells, n_groups)
    PR.check_sed((sed_now - sed_prev).astype(np.int64), orc.sed())
    for k in ("absorptions", "scatterings", "crossings"):
        assert PR.counts_close(c_now[k] - c_prev[k], co[k], 0.005), (k, c_now[k] - c_prev[k], co[k])
    del orc
    if ns < cnt:
        ctx.run_batch(wl.seed, first + ns, cnt - ns)
    c = ctx.get_counters()
    n_abs, eps = ctx.get_cell_energy()
    sed = ctx.get_sed()
    assert c["emitted"] == c["escaped"] == wl.n_packets and c["lost"] == 0
    assert int(c["emitted_per_bin"].sum()) == wl.n_packets
    PR.check_self_consistency(c, n_abs, sed)
    _temperature_identity(ctx, wl, n_abs, wl.n_packets)
