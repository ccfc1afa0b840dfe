"""-m gpu: transiently heated PAH (row f2; mcrt_set_pah and friends) of the CUDA path against the
oracle's O11..O13 on the same seeded inputs.  The split of absorptions is decided in fp32 on the GPU
and in fp64 by the oracle, so tallies are compared under the usual statistical rules; P(T) and the
emission CDF are deterministic functions of the tallies and are compared by handing the GPU's own
tallies to the oracle's solver."""
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


def _both(M, O, wl, pah, layout=0, n_packets=None, batch=None):
    ctx = M.from_workload(wl, layout=layout)
    ctx.set_pah(pah.n_C, pah.mass_fraction, pah.kabs, pah.theta_K, pah.T_lo, pah.T_hi, pah.n_Tp)
    orc = O.Oracle(wl)
    orc.set_pah(pah.n_C, pah.mass_fraction, pah.kabs, pah.theta_K, pah.T_lo, pah.T_hi, pah.n_Tp)
    for first, cnt in wl.batches(n_packets, batch):
        ctx.run_batch(wl.seed, first, cnt)
        orc.run_batch(wl.seed, first, cnt)
    return ctx, orc


def _check(ctx, orc, wl, groups=None, min_count=300, min_total=1000):
    cg, co = ctx.get_counters(), orc.counters()
    PR.check_accounting(cg, co)
    ng, _ = ctx.get_cell_energy()
    no, _ = orc.cell_energy()
    pg = ctx.get_pah_absorbed().astype(np.int64)
    po, total_o = orc.pah_absorbed()
    po = po.astype(np.int64)
    # exact identities on the GPU side: every absorption is booked on exactly one of the two tallies
    assert int(ng.sum()) + int(pg.sum()) == cg["absorptions"]
    assert int(no.sum()) + int(po.sum()) == co["absorptions"] and total_o == po.sum()
    sg, so = ctx.get_sed(), orc.sed()
    assert int(sg.sum()) == cg["escaped"]
    PR.check_sed(sg, so)
    PR.check_cell_energy(ng, no, min_count=min_count, groups=groups)
    # PAH tallies: per bin (summed over leaves), per leaf (summed over bins), and in total
    assert PR.counts_close(pg.sum(axis=0), po.sum(axis=0), 0.02).all()
    PR.check_cell_energy(pg.sum(axis=1), po.sum(axis=1), min_count=min_count, groups=groups)
    assert PR.counts_close(pg.sum(), po.sum(), 0.005) and pg.sum() > min_total
    for k in ("absorptions", "scatterings", "crossings"):
        assert PR.counts_close(cg[k], co[k], 0.005), (k, cg[k], co[k])
    # P(T) and the emission CDF are functions of (tallies, N_cum, rho): the oracle's solver on the GPU's tallies
    cdf_g = ctx.get_pah_emission_cdf().astype(np.float64)
    orc.pah_update(pg.astype(np.uint64), cg["emitted"])
    cdf_o = orc.pah_cdf()
    assert np.abs(cdf_g - cdf_o).max() < 3e-6
    hot = np.flatnonzero(pg.sum(axis=1) > 0)
    assert len(hot) > 20
    for slot in hot[:: max(1, len(hot) // 6)]:
        T, P = ctx.get_pah_temperature_distribution(int(slot))
        R = orc.pah_rates(int(slot), pg[slot].astype(np.uint64), cg["emitted"])
        Po, _ = orc.pah_solve(R)
        assert np.allclose(T, orc.pah_grid()["T"], rtol=1e-12)
        assert np.abs(P - Po).max() < 1e-9 and abs(P.sum() - 1) < 1e-12
    PR.check_temperature_of_tally(ctx.get_cell_temperature(), orc, ng, cg["emitted"])
    return cg


def test_pah_tables_match_oracle(M, oracle_mod):
    """set_pah rebuilds Q(T) and the emission rows from what is left for the grains in equilibrium."""
    wl = W.c0()
    pah = W.pah_share(wl)
    ctx = M.from_workload(wl)
    before = ctx.get_tables()
    ctx.set_pah(pah.n_C, pah.mass_fraction, pah.kabs)
    orc = oracle_mod.Oracle(wl)
    orc.set_pah(pah.n_C, pah.mass_fraction, pah.kabs)
    opac, lnQ, cdf = ctx.get_tables()
    t = orc.tables()
    assert np.array_equal(opac[:, :3], before[0][:, :3])                # extinction, albedo, g: the whole mix
    ok = t["Q"] > 1e-280
    np.testing.assert_allclose(lnQ[ok], np.log(t["Q"][ok]), rtol=2e-7, atol=2e-6)
    np.testing.assert_allclose(cdf, t["C"], rtol=0, atol=1.2e-7)
    assert np.abs(lnQ - before[1]).max() > 0.01                         # ... and they did change
    T, P = ctx.get_pah_temperature_distribution(100)                     # nothing absorbed yet: ground state
    assert P[0] == 1.0 and P[1:].sum() == 0.0 and T[0] == pytest.approx(5.0)


def test_pah_sphere_against_oracle(M, oracle_mod):
    wl = W.c0(n_packets=400_000, batch=100_000)
    pah = W.pah_share(wl, n_C=60, mass_fraction=0.05, uv_share=0.5, band_share=0.3)
    pah.n_Tp = 96
    ctx, orc = _both(M, oracle_mod, wl, pah)
    _check(ctx, orc, wl, groups=PR.radial_shells(16, 8))


@pytest.mark.parametrize("layout", [1, 2, 3])
def test_pah_layouts_and_macro_cubes(M, oracle_mod, layout):
    """x-fastest, Morton bricks, macro cubes: the per-leaf PAH rows come back in the caller's slot order."""
    wl = W.sphere(n_root=24, tau_v=2.0, gval=0.3, n_bins=48, n_packets=300_000, batch=100_000)
    pah = W.pah_share(wl, n_C=100, mass_fraction=0.04)
    pah.n_Tp = 64
    ctx, orc = _both(M, oracle_mod, wl, pah, layout=layout)
    _check(ctx, orc, wl, groups=PR.radial_shells(24, 6))


def test_pah_two_level_disk(M, oracle_mod):
    """The disk recipe on a 32^3 + 4^3 grid: sub-cell volumes enter the number of molecules per leaf."""
    wl = W.c2(n_root=32, n_packets=600_000, batch=200_000)
    mix = (np.asarray(wl.weight)[:, None] * wl.kabs.astype(np.float64)).sum(axis=0)
    kp = (np.asarray(wl.weight)[3:, None] * wl.kabs[3:].astype(np.float64)).sum(axis=0)   # the two PAH species of the mix
    pah = W.Pah(n_C=100, mass_fraction=float(np.asarray(wl.weight)[3:].sum()), kabs=np.minimum(kp, mix).astype(np.float32),
                n_Tp=64)
    ctx, orc = _both(M, oracle_mod, wl, pah)
    cg = _check(ctx, orc, wl, groups=PR.blocks_of_slot(wl, 4), min_count=200, min_total=500)
    pg = ctx.get_pah_absorbed()
    assert pg[wl.n_root ** 3:].sum() > 0.5 * pg.sum()                    # mostly in subcubes


def test_pah_reset_and_states(M):
    wl = W.c0(n_packets=40_000, batch=20_000)
    pah = W.pah_share(wl)
    ctx = M.from_workload(wl)
    with pytest.raises(M.McrtError):
        ctx.n_Tp = 8
        ctx.get_pah_absorbed()                                           # ESTATE: no PAH declared
    with pytest.raises(M.McrtError):
        ctx.set_pah(0, 0.1, pah.kabs)                                    # EINVAL
    ctx.set_pah(pah.n_C, pah.mass_fraction, pah.kabs, n_Tp=32)
    cold = ctx.get_pah_emission_cdf().copy()
    assert np.all(cold == cold[0]) and cold[0, -1] == 1.0
    for f, c in wl.batches():
        ctx.run_batch(wl.seed, f, c)
    first = (ctx.get_pah_absorbed().copy(), ctx.get_sed().copy(), ctx.get_pah_emission_cdf().copy())
    assert first[0].sum() > 500 and not np.array_equal(first[2], cold)
    ctx.reset_tallies(3)
    assert ctx.get_pah_absorbed().sum() == 0 and np.array_equal(ctx.get_pah_emission_cdf(), cold)
    for f, c in wl.batches():
        ctx.run_batch(wl.seed, f, c)
    assert np.array_equal(ctx.get_pah_absorbed(), first[0]) and np.array_equal(ctx.get_sed(), first[1])
    assert np.array_equal(ctx.get_pah_emission_cdf(), first[2])          # bit-reproducible
    ctx.set_opacity(wl.lambda_edges_um, wl.weight, wl.kabs, wl.ksca, wl.g)   # a new opacity set drops the PAH
    with pytest.raises(M.McrtError):
        ctx.get_pah_absorbed()


@pytest.mark.parametrize("maker,layout", [
    (lambda: W.sphere(n_root=16, tau_v=2.0, gval=0.3, n_bins=32, n_packets=120_000, batch=40_000), 1),
    (lambda: W.sphere(n_root=16, tau_v=2.0, gval=0.3, n_bins=32, n_packets=120_000, batch=40_000), 3),
    (lambda: W.c2(n_root=24, n_packets=150_000, batch=50_000), 0)])
def test_pah_two_emulated_ranks_equal_one(M, maker, layout):
    """Packet-sharded batches with a PAH: the per-batch delta array carries the PAH's
    absorbed spectrum of every leaf behind the equilibrium counts; two contexts playing two ranks end up with
    the tallies, temperatures, P(T) and emission CDFs of the single-context run, bit for bit."""
    from paper_1201_3588_b200.sharding import rank_range
    wl = maker()
    if wl.n_ref:
        mix = (np.asarray(wl.weight)[:, None] * wl.kabs.astype(np.float64)).sum(axis=0)
        kp = (np.asarray(wl.weight)[3:, None] * wl.kabs[3:].astype(np.float64)).sum(axis=0)
        pah = W.Pah(n_C=100, mass_fraction=float(np.asarray(wl.weight)[3:].sum()),
                    kabs=np.minimum(kp, mix).astype(np.float32), n_Tp=32)
    else:
        pah = W.pah_share(wl, n_C=100, mass_fraction=0.04)
        pah.n_Tp = 32

    def make():
        ctx = M.from_workload(wl, layout=layout)
        ctx.set_pah(pah.n_C, pah.mass_fraction, pah.kabs, n_Tp=pah.n_Tp)
        return ctx

    one = make()
    for f, c in wl.batches():
        one.run_batch(wl.seed, f, c)
    ranks = [make(), make()]
    words = int(M.lib().mcrt_delta_words(ranks[0].h))
    assert words == int(M.lib().mcrt_store_slots(ranks[0].h)) * (1 + wl.n_bins)
    done = 0
    for first, cnt in wl.batches():
        deltas = []
        for r, ctx in enumerate(ranks):
            f, c = rank_range(first, cnt, 2, r)
            d = ctx.transport_batch_delta(wl.seed, f, c)
            assert d.numel() == words
            deltas.append(d)
        total = deltas[0] + deltas[1]
        done += cnt
        for ctx in ranks:
            ctx.accumulate_update(total, done)
    assert one.get_pah_absorbed().sum() > 100
    for ctx in ranks:
        assert np.array_equal(ctx.get_cell_energy()[0], one.get_cell_energy()[0])
        assert np.array_equal(ctx.get_cell_temperature(), one.get_cell_temperature())
        assert np.array_equal(ctx.get_pah_absorbed(), one.get_pah_absorbed())
        assert np.array_equal(ctx.get_pah_emission_cdf(), one.get_pah_emission_cdf())
    assert np.array_equal(ranks[0].get_sed() + ranks[1].get_sed(), one.get_sed())
    ca, cb, c1 = ranks[0].get_counters(), ranks[1].get_counters(), one.get_counters()
    for k in c1:
        assert np.array_equal(ca[k] + cb[k], c1[k]), k
