"""-m gpu: the CUDA path (through the C-ABI, include/mcrt.h) against the fp64 oracle on the same
seeded inputs.  Tolerances: BASELINE.json north_star (tests/parity.py)."""
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


def _run_both(M, O, wl, n_packets=None, batch=None, threads=0):
    ctx = M.run_workload(wl, n_packets, batch)
    orc = O.Oracle(wl).run(n_packets, batch, threads=threads)
    return ctx, orc


def _compare(ctx, orc, groups=None, min_count=1000, expect_cells=True, expect_T_cells=0):
    """GPU run against the oracle's run of the same packages.  `groups`: one array or a list of
    arrays of aggregation indices per leaf slot.  Last of all the GPU's temperatures are checked on
    every leaf slot against the oracle's temperature step applied to the GPU's own tally (this
    overwrites the oracle's temperatures: _compare is the last use of `orc`)."""
    cg, co = ctx.get_counters(), orc.counters()
    PR.check_accounting(cg, co)
    ng, eps_g = ctx.get_cell_energy()
    no, eps_o = orc.cell_energy()
    sg, so = ctx.get_sed(), orc.sed()
    PR.check_self_consistency(cg, ng, sg)
    assert eps_g == pytest.approx(eps_o, rel=1e-12)
    if groups is None or isinstance(groups, np.ndarray):
        groups = [groups]
    n_cells = n_groups = 0
    for g in groups:
        n_cells, k = PR.check_cell_energy(ng, no, min_count=min_count, groups=g)
        n_groups += k
    if expect_cells:
        assert n_cells + n_groups > 0
    Tg = ctx.get_cell_temperature()
    n_T = PR.check_temperature(Tg, orc.cell_temperature(), ng, no, min_count=min_count)
    assert n_T >= expect_T_cells, (n_T, expect_T_cells)
    PR.check_sed(sg, so)
    n_slots, n_hot = PR.check_temperature_of_tally(Tg, orc, ng, cg["emitted"])
    assert n_slots == len(ng) and 0.99 * (ng > 0).sum() <= n_hot <= (ng > 0).sum()
    # event totals are sums of ~1e5+ events: 3 sigma + 0.5 %
    for k in ("absorptions", "scatterings", "crossings"):
        assert PR.counts_close(cg[k], co[k], 0.005), (k, cg[k], co[k])
    return cg, co


# ---- generator ------------------------------------------------------------------------------
def test_philox_device_matches_oracle(M, oracle_mod):
    rng = np.random.default_rng(7)
    key = rng.integers(0, 2 ** 32, size=2, dtype=np.uint64).astype(np.uint32)
    ctr = rng.integers(0, 2 ** 32, size=(20000, 4), dtype=np.uint64).astype(np.uint32)
    ctr[0] = 0
    ctr[1] = 0xFFFFFFFF
    out = M.philox_blocks(key, ctr)
    for i in list(range(64)) + list(range(0, 20000, 97)):
        assert np.array_equal(out[i], oracle_mod.philox(key, ctr[i])), i


def test_device_uniforms_stay_inside_the_unit_interval(M):
    """R19: the fp32 uniform of a flight is ((w >> 9) + 0.5) 2^-23, exact in fp32 and
    strictly inside (0,1) for every word -- in particular 0xFFFFFFFF, which a 24-bit variant
    rounds to 1.0 -- so tau* = -ln u > 0; the fp64 uniform of the emission decisions is the
    oracle's (w + 0.5) 2^-32."""
    rng = np.random.default_rng(3)
    w = np.concatenate([np.array([0, 1, 511, 512, 0x7FFFFFFF, 0x80000000, 0xFFFFFE00, 0xFFFFFFFF],
                                 dtype=np.uint64), rng.integers(0, 2 ** 32, size=5000, dtype=np.uint64)])
    u, ud, tau = M.uniforms(w.astype(np.uint32))
    assert u.dtype == np.float32 and 0.0 < u.min() and u.max() < 1.0
    assert np.array_equal(u.astype(np.float64), ((w >> 9).astype(np.float64) + 0.5) * 2.0 ** -23)
    assert np.array_equal(ud, (w.astype(np.float64) + 0.5) * 2.0 ** -32)
    assert tau.min() > 0.0 and np.isfinite(tau).all() and tau.max() < 16.7
    assert u[7] == np.float32(1.0) - np.float32(2.0 ** -24)


# ---- tables (row a0) ------------------------------------------------------------------------
@pytest.mark.parametrize("maker", [W.c0, lambda: W.c2(n_root=8, n_packets=10, batch=10)])
def test_tables_match_oracle(M, oracle_mod, maker):
    wl = maker()
    ctx = M.from_workload(wl)
    orc = oracle_mod.Oracle(wl)
    opac, lnQ, cdf = ctx.get_tables()
    t = orc.tables()
    np.testing.assert_allclose(opac[:, 0], t["kext"] * wl.root_size, rtol=2e-7)
    np.testing.assert_allclose(opac[:, 1], t["alb"], rtol=2e-7, atol=1e-30)
    np.testing.assert_allclose(opac[:, 2], t["g"], rtol=2e-7, atol=1e-30)
    ok = t["Q"] > 1e-280
    np.testing.assert_allclose(lnQ[ok], np.log(t["Q"][ok]), rtol=2e-7, atol=2e-6)
    np.testing.assert_allclose(cdf, t["C"], rtol=0, atol=1.2e-7)


# ---- C0 at full size ------------------------------------------------------------------------
def test_c0_full(M, oracle_mod):
    wl = W.c0()
    ctx, orc = _run_both(M, oracle_mod, wl)
    cg, co = _compare(ctx, orc, groups=PR.radial_shells(16, 8))
    assert cg["emitted"] == 100_000


def test_c0_bit_reproducible_and_launch_shape_invariant(M):
    wl = W.c0()
    a = M.run_workload(wl)
    for shape in ((64, 2), (256, 4), (256, 5), (128, 12)):    # 64- and 48-register builds of the kernel
        b = M.from_workload(wl)
        b.set_launch(*shape)
        for first, cnt in wl.batches():
            b.run_batch(wl.seed, first, cnt)
        assert np.array_equal(a.get_cell_energy()[0], b.get_cell_energy()[0])
        assert np.array_equal(a.get_sed(), b.get_sed())
        assert np.array_equal(a.get_cell_temperature(), b.get_cell_temperature())
        ca, cb = a.get_counters(), b.get_counters()
        for k in ca:
            assert np.array_equal(ca[k], cb[k]), k


def test_pure_scattering_exact(M, oracle_mod):
    """albedo 1: no tally, frequency never changes -> SED total per bin == emitted per bin
    exactly, and batch-partition independent bit-exactly (R29)."""
    wl = W.sphere(n_root=16, albedo=1.0, gval=0.4, n_packets=200_000, batch=50_000)
    ctx = M.run_workload(wl)
    c = ctx.get_counters()
    sed = ctx.get_sed()
    assert np.array_equal(sed.sum(0), c["emitted_per_bin"])
    assert int(ctx.get_cell_energy()[0].sum()) == 0 and c["absorptions"] == 0
    assert c["escaped"] == 200_000 and c["lost"] == 0
    other = M.run_workload(wl, batch=200_000)
    assert np.array_equal(other.get_sed(), sed)
    co = other.get_counters()
    assert co["crossings"] == c["crossings"] and co["scatterings"] == c["scatterings"]
    orc = oracle_mod.Oracle(wl).run()
    PR.check_accounting(c, orc.counters())
    PR.check_sed(sed, orc.sed())


def test_beer_lambert_direct_fraction(M):
    """Pure absorber, central source: direct/emitted per bin = exp(-tau_j) within the voxel
    staircase (closed form, BASELINE.json check 2) -- pins the GPU walk without the oracle."""
    wl = W.sphere(n_root=32, albedo=0.0, tau_v=1.0, n_packets=2_000_000, batch=2_000_000)
    ctx = M.run_workload(wl)
    c = ctx.get_counters()
    sed = ctx.get_sed()
    kext = (wl.kabs[0] + wl.ksca[0]).astype(np.float64)
    tau = kext * wl.meta["rho0"] * wl.meta["R_cm"]
    em = c["emitted_per_bin"].astype(np.float64)
    sel = em > 20000
    frac = sed[0][sel] / em[sel]
    # staircase: chord through filled voxels differs from R by O(1 cell) = 1/16 of R
    lo, hi = np.exp(-tau[sel] * (1 + 1.5 / 16)), np.exp(-tau[sel] * (1 - 1.5 / 16))
    sig = 3 * np.sqrt(frac * (1 - frac) / em[sel])
    assert np.all(frac <= hi + sig) and np.all(frac >= lo - sig)


# ---- C1 twins: 64^3, HG g = 0.6, several tiles of batches and a ragged tail ------------------
@pytest.mark.parametrize("tau_v,n_packets", [(0.1, 1_000_000), (1.0, 1_000_000),
                                             (10.0, 400_000), (100.0, 30_000)])
def test_c1_twin(M, oracle_mod, tau_v, n_packets):
    wl = W.c1(tau_v=tau_v, n_packets=n_packets, batch=n_packets // 10 + 7)
    ctx, orc = _run_both(M, oracle_mod, wl)
    _compare(ctx, orc, groups=PR.radial_shells(64, 16))


# ---- two-level grids ------------------------------------------------------------------------
@pytest.mark.parametrize("n_root,sub,n_ref,ext", [(2, 4, 1, False), (2, 4, 8, True),
                                                  (3, 4, 5, False), (4, 2, 9, True),
                                                  (3, 0, 0, True), (3, 3, 11, True),
                                                  (2, 8, 3, False), (5, 5, 40, True)])
def test_tiny_grids(M, oracle_mod, n_root, sub, n_ref, ext):
    wl = W.tiny_random(n_root=n_root, sub=sub, n_refined=n_ref, seed=11 + n_ref,
                       external=ext, n_packets=400_000, batch=100_000)
    ctx, orc = _run_both(M, oracle_mod, wl)
    _compare(ctx, orc)


def test_c2_twin_small_disk(M, oracle_mod):
    """Disk twin: 32^3 root grid of the C2 recipe (refined inside r < 5 r0), tau_V = 100."""
    wl = W.c2(n_root=32, n_packets=1_000_000, batch=100_000)
    assert wl.n_ref > 0
    ctx, orc = _run_both(M, oracle_mod, wl)
    _compare(ctx, orc, groups=[PR.root_of_slot(wl), PR.blocks_of_slot(wl, 4)])


def test_c3_twin_small_disk(M, oracle_mod):
    wl = W.c3(n_root=32, n_packets=1_000_000, batch=100_000)
    assert wl.n_ref > 0
    ctx, orc = _run_both(M, oracle_mod, wl)
    _compare(ctx, orc, groups=[PR.root_of_slot(wl), PR.blocks_of_slot(wl, 4)])


@pytest.mark.parametrize("maker,n_ref", [(W.c2, 17_256), (W.c3, 224_872)])
def test_disk_configs_full_grid_against_oracle(M, oracle_mod, maker, n_ref):
    """configs[2] / configs[3] on their OWN grids (128^3 + 17 256 x 4^3, 256^3 + 224 872 x 4^3 leaf
    slots, the two-level walk at full size): 2^22 packages in four batches of 2^20 on both sides
    (temperatures feed back three times), compared per leaf, per root cube (sub-cells folded
    back into their cube), per 4^3 and 8^3 super-block of cubes, SED, counters, and the
    temperature of every leaf slot."""
    wl = maker()
    assert wl.n_ref == n_ref and wl.sub == 4
    n, batch = 1 << 22, 1 << 20
    ctx, orc = _run_both(M, oracle_mod, wl, n, batch)
    cg, co = _compare(ctx, orc, groups=[PR.root_of_slot(wl), PR.blocks_of_slot(wl, 4),
                                        PR.blocks_of_slot(wl, 8)])
    assert cg["emitted"] == n and cg["absorptions"] > 100_000
    n_abs, _ = ctx.get_cell_energy()
    n3 = wl.n_root ** 3
    assert n_abs[n3:].sum() > 0.5 * n_abs.sum()               # most absorptions happen in subcubes
    assert n_abs[:n3][np.asarray(wl.refine).ravel() > 0].sum() == 0


def test_c4_twin_small_cube(M, oracle_mod):
    """Clumpy cube twin: 64^3 of the C4 recipe, 10 point sources + external field."""
    wl = W.c4(n_root=64, n_packets=300_000, batch=30_000, corr_cells=4.0)
    ctx, orc = _run_both(M, oracle_mod, wl)
    _compare(ctx, orc, groups=PR.super_blocks(64, 8))


# ---- edge cases -----------------------------------------------------------------------------
def test_empty_batch_and_single_packet(M, oracle_mod):
    wl = W.c0()
    ctx = M.from_workload(wl)
    ctx.run_batch(1, 0, 0)
    assert ctx.get_counters()["emitted"] == 0
    assert np.all(ctx.get_cell_temperature() == np.float32(1.0))
    ctx.run_batch(1, 5, 1)
    c = ctx.get_counters()
    assert c["emitted"] == 1 and c["escaped"] == 1
    orc = oracle_mod.Oracle(wl)
    orc.run_batch(1, 5, 1)
    assert np.array_equal(ctx.get_sed(), orc.sed())


def test_empty_grid_all_escape_direct(M):
    wl = W.c0()
    wl.rho_root = np.zeros_like(wl.rho_root)
    ctx = M.run_workload(wl, 50_000, 50_000)
    c = ctx.get_counters()
    sed = ctx.get_sed()
    assert c["escaped"] == 50_000 and c["flights"] == 50_000
    assert sed[1:].sum() == 0 and np.array_equal(sed[0], c["emitted_per_bin"])
    # centre vertex of a 16^3 grid: every packet leaves 8 cells per axis-ish; at least 8 crossings
    assert c["crossings"] >= 8 * 50_000


def test_packet_ids_beyond_32_bits(M, oracle_mod):
    wl = W.c0()
    first = (1 << 40) + 12345
    ctx = M.from_workload(wl)
    ctx.run_batch(3, first, 20_000)
    orc = oracle_mod.Oracle(wl)
    orc.run_batch(3, first, 20_000)
    PR.check_accounting(ctx.get_counters(), orc.counters())
    PR.check_sed(ctx.get_sed(), orc.sed())


def test_device_inputs_and_outputs(M):
    import torch
    wl = W.c0()
    a = M.run_workload(wl, 20_000, 10_000)
    b = M.run_workload(wl, 20_000, 10_000, device_inputs=True)
    n_dev, eps = b.get_cell_energy(device=True)
    assert n_dev.is_cuda and np.array_equal(n_dev.cpu().numpy().astype(np.uint64),
                                            a.get_cell_energy()[0])
    assert np.array_equal(b.get_cell_temperature(device=True).cpu().numpy(),
                          a.get_cell_temperature())
    assert np.array_equal(b.get_sed(device=True).cpu().numpy().astype(np.uint64), a.get_sed())
    s = torch.cuda.Stream()
    with torch.cuda.stream(s):
        c = M.run_workload(wl, 20_000, 10_000)
    assert np.array_equal(c.get_sed(), a.get_sed())


def test_error_paths(M):
    ctx = M.Context()
    wl = W.c0()
    with pytest.raises(M.McrtError):
        ctx.grid_create(0, 0, wl.origin, wl.root_size, None, wl.rho_root, None)
    with pytest.raises(M.McrtError):          # beyond the largest grid (N^3 must stay below 2^31 slots)
        ctx.grid_create(1291, 0, wl.origin, wl.root_size, None, wl.rho_root, None)
    with pytest.raises(M.McrtError):          # unknown storage layout
        ctx.grid_create(wl.n_root, 0, wl.origin, wl.root_size, None, wl.rho_root, None, layout=7)
    ctx.grid_create(wl.n_root, 0, wl.origin, wl.root_size, None, wl.rho_root, None)
    with pytest.raises(M.McrtError):          # ESTATE: opacity not set
        ctx.set_source(wl.sources)
    with pytest.raises(M.McrtError):          # ESTATE
        ctx.run_batch(1, 0, 10)
    ctx.set_opacity(wl.lambda_edges_um, wl.weight, wl.kabs, wl.ksca, wl.g)
    with pytest.raises(M.McrtError):          # source outside the box
        ctx.set_source([W.Source(W.SRC_POINT, (-1.0, 0.0, 0.0), W.LSUN, 5800.0)])
    with pytest.raises(M.McrtError):
        ctx.set_opacity(wl.lambda_edges_um[::-1], wl.weight, wl.kabs, wl.ksca, wl.g)


def test_reset_tallies(M):
    wl = W.c0()
    ctx = M.run_workload(wl, 20_000, 10_000)
    first = ctx.get_sed().copy()
    ctx.reset_tallies(3)
    assert ctx.get_sed().sum() == 0 and ctx.get_cell_energy()[0].sum() == 0
    for f, c in wl.batches(20_000, 10_000):
        ctx.run_batch(wl.seed, f, c)
    assert np.array_equal(ctx.get_sed(), first)


# ---- storage layouts of single-level grids (never visible in the getters, R22) ----------------
def _run_layout(M, wl, layout, quorum=0, n_packets=None, batch=None):
    ctx = M.from_workload(wl, layout=layout)
    if quorum:
        ctx.set_walk_quorum(quorum)
    for first, cnt in wl.batches(n_packets, batch):
        ctx.run_batch(wl.seed, first, cnt)
    return ctx


def _assert_identical(a, b):
    assert np.array_equal(a.get_cell_energy()[0], b.get_cell_energy()[0])
    assert np.array_equal(a.get_sed(), b.get_sed())
    assert np.array_equal(a.get_cell_temperature(), b.get_cell_temperature())
    ca, cb = a.get_counters(), b.get_counters()
    for k in ca:
        assert np.array_equal(ca[k], cb[k]), k


@pytest.mark.parametrize("maker", [
    lambda: W.c0(),
    lambda: W.tiny_random(n_root=3, seed=4, external=True, n_packets=40_000, batch=10_000),
    lambda: W.tiny_random(n_root=13, seed=5, external=True, tau_cell=0.2, n_packets=60_000,
                          batch=20_000),
    lambda: W.c4(n_root=24, n_packets=60_000, batch=20_000, corr_cells=3.0)])
def test_bricked_layout_bit_identical_to_x_fastest(M, maker):
    """Same walk, same Philox slots, integer tallies: the storage order (x-fastest vs 8^3 Morton
    bricks, with padding when N is not a multiple of 8) must not change a single count."""
    wl = maker()
    a = _run_layout(M, wl, 1)
    b = _run_layout(M, wl, 2)
    _assert_identical(a, b)
    assert a.get_counters()["emitted"] == wl.n_packets


def test_walk_quorum_does_not_change_results(M):
    wl = W.c4(n_root=24, n_packets=60_000, batch=20_000, corr_cells=3.0)
    a = _run_layout(M, wl, 0, quorum=1)
    b = _run_layout(M, wl, 0, quorum=32)
    c = _run_layout(M, wl, 2, quorum=8)
    _assert_identical(a, b)
    _assert_identical(a, c)


@pytest.mark.parametrize("maker,layout", [
    (lambda: W.c0(), 0),                                                    # density staged in shared memory
    (lambda: W.c1(tau_v=10.0, n_packets=300_000, batch=100_000), 0),       # plain single-level walk
    (lambda: W.c1(tau_v=10.0, n_packets=300_000, batch=100_000), 3),       # macro cubes
    (lambda: W.c2(n_root=32, n_packets=300_000, batch=100_000), 0),        # cubes and subcubes
    (lambda: W.c4(n_root=24, n_packets=90_000, batch=30_000, corr_cells=3.0), 2),
    (lambda: W.tiny_random(n_root=3, sub=8, n_refined=5, seed=11, external=True, n_packets=40_000, batch=10_000), 0)])
def test_end_of_batch_modes_do_not_change_results(M, maker, layout):
    """mcrt_set_tail_mode: how a warp schedules its last packages once the work queue is empty, and whether the
    temperature update runs at the end of the transport launch (grid-wide barrier) or in a launch of its own, is
    scheduling only -- tallies, SED, temperatures and every counter stay bit-identical."""
    wl = maker()
    runs = []
    for mode in (0, 1, 2, 3, -1):
        ctx = M.from_workload(wl, layout=layout)
        ctx.set_tail_mode(mode)
        for first, cnt in wl.batches():
            ctx.run_batch(wl.seed, first, cnt)
        runs.append(ctx)
    for r in runs[1:]:
        _assert_identical(runs[0], r)
    c = runs[1].get_counters()
    assert c["emitted"] == c["escaped"] == wl.n_packets and c["lost"] == 0


@pytest.mark.parametrize("layout", [1, 2])
def test_split_batch_halves_equal_run_batch(M, layout):
    """transport_batch + update_temperature(sum in slot order) == run_batch (multi-GPU path,
    DESIGN.md section 12), for both storage layouts."""
    wl = W.tiny_random(n_root=13, seed=6, tau_cell=0.3, n_packets=40_000, batch=10_000)
    a = _run_layout(M, wl, layout)
    b = M.from_workload(wl, layout=layout)
    done = 0
    for first, cnt in wl.batches():
        b.transport_batch(wl.seed, first, cnt)
        tally, _ = b.get_cell_energy(device=True)
        done += cnt
        b.update_temperature(tally, done)
    _assert_identical(a, b)


def test_gather_calibration_orders_by_footprint(M):
    """The gather-roofline calibration returns a finite rate that falls as the footprint leaves
    the caches (16 KB: L1; 64 MB: L2; 1 GB: HBM)."""
    g = [M.gather_calibrate(fb, 1 << 28)[0] for fb in (16 << 10, 64 << 20, 1 << 30)]
    assert all(np.isfinite(v) and v > 1e9 for v in g), g
    assert g[0] > g[1] > g[2], g
    with pytest.raises(M.McrtError):
        M.gather_calibrate(0, 10)


# ---- BASELINE.json's full sizes, in the launch configuration bench.py times -------------------
def _temperature_identity(M, ctx, wl, n_cum, sample=20000):
    """4 pi m Q(T) N_cum / (cum L_tot) = 1 on sampled cells that are neither empty nor clamped
    (O7; Q from the library's own ln Q table, interpolated as the update kernel does)."""
    n_abs, eps = ctx.get_cell_energy()
    T = ctx.get_cell_temperature().astype(np.float64)
    _, lnQ, _ = ctx.get_tables()
    lnQ = lnQ.astype(np.float64)
    nT = len(lnQ)
    rho = np.asarray(wl.rho_root, dtype=np.float64).ravel()
    idx = np.flatnonzero((n_abs > 0) & (rho > 0))
    rng = np.random.default_rng(3)
    idx = rng.choice(idx, size=min(sample, len(idx)), replace=False)
    t = np.log(T[idx]) / (np.log(1.0e4) / (nT - 1))          # row coordinate on the default T grid
    ok = (t > 0.5) & (t < nT - 1.5)
    idx, t = idx[ok], t[ok]
    k = np.floor(t).astype(int)
    lnq_T = lnQ[k] + (t - k) * (lnQ[k + 1] - lnQ[k])
    Ltot = sum(s.L for s in wl.sources)
    lnq = np.log(n_abs[idx].astype(np.float64)) + np.log(Ltot / (n_cum * 4 * np.pi * wl.root_size ** 3)) \
        - np.log(rho[idx])
    assert len(idx) > 100
    assert np.abs(lnq_T - lnq).max() < 2e-3, np.abs(lnq_T - lnq).max()
    assert eps == pytest.approx(Ltot / n_cum, rel=1e-12)


def test_c1_full_batch_against_oracle(M, oracle_mod):
    """One full 2^20-package batch of configs[1] (tau_V = 1) in bench.py's launch configuration:
    the oracle runs the same batch; then a second batch for the temperature identity."""
    wl = W.c1(tau_v=1.0)
    n = wl.batch
    assert n == 1 << 20
    ctx = M.from_workload(wl)
    ctx.run_batch(wl.seed, 0, n)
    orc = oracle_mod.Oracle(wl)
    orc.run_batch(wl.seed, 0, n)
    cg, co = _compare(ctx, orc, groups=PR.radial_shells(64, 32))
    assert cg["emitted"] == n
    ctx.run_batch(wl.seed, n, n)
    _temperature_identity(M, ctx, wl, 2 * n)


def test_c4_full_grid_against_oracle(M, oracle_mod):
    """configs[4]'s full 512^3 clumpy cube (bricked storage, 11 sources): 2^21 packages on both
    sides compared by 8^3 super-blocks; then invariants on a second, 2^22-package batch."""
    wl = W.c4()
    assert wl.n_root == 512
    n = 1 << 21
    ctx = M.from_workload(wl)
    ctx.run_batch(wl.seed, 0, n)
    orc = oracle_mod.Oracle(wl)
    orc.run_batch(wl.seed, 0, n)
    _compare(ctx, orc, groups=PR.super_blocks(512, 8), expect_cells=True)
    del orc
    m = 1 << 22
    ctx.run_batch(wl.seed, n, m)
    c = ctx.get_counters()
    n_abs, _ = ctx.get_cell_energy()
    sed = ctx.get_sed()
    assert c["emitted"] == c["escaped"] == n + m and c["lost"] == 0
    PR.check_self_consistency(c, n_abs, sed)
    _temperature_identity(M, ctx, wl, n + m)


@pytest.mark.parametrize("layout", [1, 2])
def test_source_grouped_handout_does_not_change_results(M, layout):
    """Several sources: handing the packages of a batch out grouped by source (mcrt_set_source_order)
    only changes which lane carries which package; every count must be identical.  Batches of
    2^17 packages so that the pre-pass really runs (it skips batches below 65536)."""
    wl = W.c4(n_root=24, n_packets=3 << 17, batch=1 << 17, corr_cells=3.0)
    assert len(wl.sources) == 11
    runs, launches = [], []
    for mode in (0, 1, 2):                                      # off / by source / by source and direction
        ctx = M.from_workload(wl, layout=layout)
        ctx.set_source_order(mode)
        for first, cnt in wl.batches():
            ctx.run_batch(wl.seed, first, cnt)
        runs.append(ctx)
        launches.append(ctx.kernel_launches())                  # before any getter launches a conversion
    _assert_identical(runs[0], runs[1])
    _assert_identical(runs[0], runs[2])
    assert runs[1].get_counters()["emitted"] == wl.n_packets
    assert launches[1] == launches[2] == launches[0] + 3 * 3    # three pre-pass kernels per batch


@pytest.mark.parametrize("maker", [W.c2, W.c3])
def test_disk_configs_full_size_invariants(M, maker):
    """configs[2] / configs[3] at their full grids (128^3 + 17 256 x 4^3, 256^3 + 224 872 x 4^3), one
    full 2^22-package batch in bench.py's launch configuration (grouped hand-out on): exact
    integer accounting and consistency of every tally; refined root slots stay untouched."""
    wl = maker()
    n = wl.batch
    assert n == 1 << 22 and wl.n_ref > 0
    ctx = M.from_workload(wl)
    ctx.run_batch(wl.seed, 0, n)
    c = ctx.get_counters()
    n_abs, eps = ctx.get_cell_energy()
    sed = ctx.get_sed()
    assert c["emitted"] == c["escaped"] == n and c["lost"] == 0
    PR.check_self_consistency(c, n_abs, sed)
    assert int(c["emitted_per_bin"].sum()) == n
    refined = np.flatnonzero(np.asarray(wl.refine).ravel())
    assert n_abs[refined].sum() == 0                            # the slot of a refined cube is unused (R22)
    T = ctx.get_cell_temperature()
    assert np.all(T[refined] == np.float32(1.0)) and np.isfinite(T).all() and T.min() >= 1.0
    assert (T[n_abs > 0] > 1.0).all()


def test_grouped_handout_two_level_grid(M):
    """The grouped hand-out on the two-level kernel (one star, direction groups only)."""
    wl = W.c2(n_root=32, n_packets=3 << 17, batch=1 << 17)
    runs = []
    for mode in (0, 2):
        ctx = M.from_workload(wl)
        ctx.set_source_order(mode)
        for first, cnt in wl.batches():
            ctx.run_batch(wl.seed, first, cnt)
        runs.append(ctx)
    _assert_identical(runs[0], runs[1])
    assert runs[1].get_counters()["emitted"] == wl.n_packets


@pytest.mark.parametrize("maker", [
    lambda: W.tiny_random(n_root=2, sub=4, n_refined=8, seed=2, external=True, n_packets=40_000, batch=10_000),
    lambda: W.tiny_random(n_root=3, sub=2, n_refined=5, seed=9, external=True, n_packets=40_000, batch=10_000),
    lambda: W.c2(n_root=20, n_packets=60_000, batch=20_000),
    lambda: W.c3(n_root=32, n_packets=60_000, batch=20_000)])
def test_two_level_bricked_root_bit_identical_to_x_fastest(M, maker):
    """Two-level grids: the root array in bricks (padding when N is not a multiple of 8) must not
    change a single count, in the getters' slot order (root cells AND sub-cells), nor through the
    split batch halves with a tally handed back in slot order."""
    wl = maker()
    assert wl.n_ref > 0
    a = _run_layout(M, wl, 1)
    b = _run_layout(M, wl, 2)
    _assert_identical(a, b)
    assert a.get_counters()["emitted"] == wl.n_packets
    c = M.from_workload(wl, layout=2)
    done = 0
    for first, cnt in wl.batches():
        c.transport_batch(wl.seed, first, cnt)
        tally, _ = c.get_cell_energy(device=True)
        done += cnt
        c.update_temperature(tally, done)
    _assert_identical(a, c)


# ---- packet-sharded batches on the real kernels, and the combined read-out ------
@pytest.mark.parametrize("maker,layout", [
    (lambda: W.tiny_random(n_root=13, seed=6, tau_cell=0.3, n_packets=40_000, batch=10_000), 1),
    (lambda: W.tiny_random(n_root=13, seed=6, tau_cell=0.3, n_packets=40_000, batch=10_000), 2),
    (lambda: W.c3(n_root=32, n_packets=60_000, batch=20_000), 0),
    (lambda: W.c3(n_root=32, n_packets=60_000, batch=20_000), 2)])
def test_two_emulated_ranks_equal_one(M, maker, layout):
    """Two contexts play two ranks on one GPU: each transports its contiguous half of every batch
    into its own per-batch uint32 delta array (storage order), the arrays are summed (what the
    NCCL all-reduce does), and both add the sum and update T with the global package count.
    Tallies and temperatures of BOTH equal the single-context run bit for bit; SEDs and counters
    add up to it."""
    from paper_1201_3588_b200.sharding import rank_range
    wl = maker()
    one = _run_layout(M, wl, layout)
    ranks = [M.from_workload(wl, layout=layout) for _ in range(2)]
    done = 0
    for first, cnt in wl.batches():
        deltas = []
        for r, ctx in enumerate(ranks):
            f, c = rank_range(first, cnt, 2, r)
            deltas.append(ctx.transport_batch_delta(wl.seed, f, c))
        total = deltas[0] + deltas[1]
        done += cnt
        for ctx in ranks:
            ctx.accumulate_update(total, done)
    for ctx in ranks:
        assert np.array_equal(ctx.get_cell_energy()[0], one.get_cell_energy()[0])
        assert np.array_equal(ctx.get_cell_temperature(), one.get_cell_temperature())
        assert ctx.get_cell_energy()[1] == one.get_cell_energy()[1]       # eps = L / packages of ALL ranks
    assert np.array_equal(ranks[0].get_sed() + ranks[1].get_sed(), one.get_sed())
    ca, cb, c1 = ranks[0].get_counters(), ranks[1].get_counters(), one.get_counters()
    for k in c1:
        assert np.array_equal(ca[k] + cb[k], c1[k]), k


@pytest.mark.parametrize("maker", [W.c0, lambda: W.c2(n_root=20, n_packets=60_000, batch=20_000),
                                   lambda: W.c4(n_root=24, n_packets=60_000, batch=20_000, corr_cells=3.0)])
def test_combined_and_overlapped_read_out(M, maker):
    """mcrt_get_results = the four getters in one call; mcrt_results_begin / _wait deliver the state
    of the batch they were queued behind even though the next batch is already running."""
    import torch
    wl = maker()
    batches = list(wl.batches())
    ref = M.from_workload(wl, layout=2 if wl.n_root == 24 else 0)
    ctx = M.from_workload(wl, layout=2 if wl.n_root == 24 else 0)
    pin = lambda shape, dt: torch.empty(shape, dtype=dt).pin_memory().numpy()
    mk = lambda: dict(n_abs=pin((ctx.slots,), torch.int64).view(np.uint64), T=pin((ctx.slots,), torch.float32),
                      sed=pin((3, wl.n_bins), torch.int64).view(np.uint64),
                      emitted_per_bin=pin((wl.n_bins,), torch.int64).view(np.uint64))
    bufs = [mk(), mk()]
    handles, snaps = [], []
    for i, (first, cnt) in enumerate(batches):
        ref.run_batch(wl.seed, first, cnt)
        snaps.append((ref.get_cell_energy()[0].copy(), ref.get_cell_temperature().copy(), ref.get_sed().copy(),
                      ref.get_counters()))
        ctx.run_batch(wl.seed, first, cnt)
        handles.append(ctx.results_begin(bufs[i % 2]))          # the next batch is issued before this is read
        if i > 0:
            out = ctx.results_wait(handles[i - 1])
            n_abs, T, sed, c = snaps[i - 1]
            assert np.array_equal(out["n_abs"], n_abs) and np.array_equal(out["T"], T)
            assert np.array_equal(out["sed"], sed)
            assert np.array_equal(out["emitted_per_bin"], c["emitted_per_bin"])
            assert all(out["counters"][k] == c[k] for k in out["counters"])
    out = ctx.results_wait(handles[-1])
    assert np.array_equal(out["n_abs"], snaps[-1][0]) and out["eps"] == ref.get_cell_energy()[1]
    # one call, device buffers
    dev = dict(n_abs=torch.empty(ctx.slots, dtype=torch.int64, device="cuda"),
               T=torch.empty(ctx.slots, dtype=torch.float32, device="cuda"),
               sed=torch.empty((3, wl.n_bins), dtype=torch.int64, device="cuda"))
    out = ctx.get_results(dev)
    assert np.array_equal(dev["n_abs"].cpu().numpy().astype(np.uint64), snaps[-1][0])
    assert np.array_equal(dev["T"].cpu().numpy(), snaps[-1][1])
    assert np.array_equal(dev["sed"].cpu().numpy().astype(np.uint64), snaps[-1][2])
    assert out["counters"]["emitted"] == wl.n_packets
    with pytest.raises(M.McrtError):                           # a third ticket while two are in flight
        h1, h2 = ctx.results_begin(bufs[0]), ctx.results_begin(bufs[1])
        ctx.results_begin(bufs[0])
    ctx.results_wait(h1), ctx.results_wait(h2)


def test_set_opacity_with_more_bins_after_a_read_out(M):
    """a read-out ticket's device snapshot of the small tallies is sized by n_bins.
    Re-setting the opacity with MORE bins after mcrt_get_results must not let the next read-out copy
    past the old block (which the caching allocator places beside the library's own tables): the
    context re-used with 4096 bins gives exactly what a fresh context gives, its tables included,
    and mcrt_set_opacity is refused while a ticket is still in flight."""
    small = W.sphere(n_root=16, n_bins=16, n_packets=20_000, batch=20_000)
    big = W.sphere(n_root=16, n_bins=4096, n_packets=20_000, batch=20_000)
    mk = lambda wl, c: dict(sed=np.zeros((3, wl.n_bins), np.uint64), emitted_per_bin=np.zeros(wl.n_bins, np.uint64),
                            n_abs=np.zeros(c.slots, np.uint64), T=np.zeros(c.slots, np.float32))
    ctx = M.run_workload(small)
    ctx.get_results(mk(small, ctx))                            # both tickets now own snapshots sized for 16 bins
    ctx.get_results(mk(small, ctx))
    h = ctx.results_begin(mk(small, ctx))
    with pytest.raises(M.McrtError, match="ticket is in flight"):
        ctx.set_opacity(big.lambda_edges_um, big.weight, big.kabs, big.ksca, big.g)
    ctx.results_wait(h)
    ctx.set_opacity(big.lambda_edges_um, big.weight, big.kabs, big.ksca, big.g)
    ctx.set_source(big.sources)
    ctx.reset_tallies(3)
    fresh = M.from_workload(big)
    tables = [t.copy() for t in ctx.get_tables()]
    for first, cnt in big.batches():
        ctx.run_batch(big.seed, first, cnt)
        fresh.run_batch(big.seed, first, cnt)
    for _ in range(3):                                         # both tickets, and the first one again
        a, b = ctx.get_results(mk(big, ctx)), fresh.get_results(mk(big, fresh))
        for k in ("sed", "emitted_per_bin", "n_abs", "T"):
            assert np.array_equal(a[k], b[k]), k
        assert a["counters"] == b["counters"] and a["counters"]["emitted"] == big.n_packets
        assert a["sed"].sum() == big.n_packets
    for t0, t1, t2 in zip(tables, ctx.get_tables(), fresh.get_tables()):
        assert np.array_equal(t0, t1) and np.array_equal(t1, t2)   # no table was written over
    assert M.release_cached_memory() >= 0


def test_cached_device_memory_is_reused_and_can_be_released(M):
    """the library keeps the device blocks of a destroyed context (up to 1 GB) for the next
    context of the same shape; mcrt_release_cached_memory hands them back to the driver (so that torch,
    NCCL or the caller's own cudaMalloc can have them) and reports the bytes; a context created
    afterwards allocates afresh and gives the same results."""
    import torch
    wl = W.sphere(n_root=128, n_packets=50_000, batch=25_000)     # 2 M cells: blocks of 8-16 MB, well above the driver's 2 MB slabs
    M.release_cached_memory()
    ctx = M.run_workload(wl)
    sed = ctx.get_sed().copy()
    torch.cuda.synchronize()
    free_live = torch.cuda.mem_get_info()[0]
    ctx.destroy()
    assert torch.cuda.mem_get_info()[0] <= free_live + (1 << 20)   # destroyed, but the blocks stay with the library
    again = M.run_workload(wl)                                      # ... and serve the next context of this shape
    assert np.array_equal(again.get_sed(), sed)
    again.destroy()
    released = M.release_cached_memory()
    assert released >= 128 ** 3 * (4 + 4 + 8 + 4)                   # at least density, ln density, tally, temperature rows
    assert torch.cuda.mem_get_info()[0] >= free_live + released // 2
    assert M.release_cached_memory() == 0
    fresh = M.run_workload(wl)
    assert np.array_equal(fresh.get_sed(), sed)


@pytest.mark.parametrize("maker", [lambda: W.c1(tau_v=10.0, n_packets=3 << 17, batch=1 << 17),
                                   lambda: W.c2(n_root=32, n_packets=3 << 17, batch=1 << 17),
                                   lambda: W.sphere(n_root=16, n_bins=4096, tau_v=5.0, n_packets=60_000, batch=20_000),
                                   lambda: W.sphere(n_root=16, n_bins=3, tau_v=5.0, n_packets=60_000, batch=20_000)])
def test_cdf_guide_does_not_change_results(M, maker):
    """The bracket guide of the emission rows (mcrt_set_cdf_guide, tables.cuh k_build_cdf_guide) only shortens
    the bisection that finds the re-emission bin: with and without it every tally is identical, over
    several batches (the temperatures, hence the rows searched, move), with 3, 128, 200 and 4096 bins."""
    wl = maker()
    a = M.from_workload(wl)
    a.set_cdf_guide(False)
    b = M.from_workload(wl)                                     # the default: guide on
    for first, cnt in wl.batches():
        a.run_batch(wl.seed, first, cnt)
        b.run_batch(wl.seed, first, cnt)
    _assert_identical(a, b)
    c = b.get_counters()
    assert c["emitted"] == wl.n_packets and c["absorptions"] > 10_000


def test_automatic_walk_quorum_does_not_change_results(M):
    """quorum 0 = chosen by the kernel from the job's crossings per flight."""
    wl = W.c2(n_root=32, n_packets=3 << 17, batch=1 << 17)
    a = M.from_workload(wl)
    a.set_walk_quorum(16)
    b = M.from_workload(wl)                                     # automatic
    for first, cnt in wl.batches():
        a.run_batch(wl.seed, first, cnt)
        b.run_batch(wl.seed, first, cnt)
    _assert_identical(a, b)


def test_density_staged_in_shared_memory_does_not_change_results(M):
    """Small single-level problems keep their density in shared memory (one cp.async.bulk per
    block): the fp32 array itself up to 40 KB (C0), one bit per cell for a two-valued grid (the
    64^3 sphere of C1).  Every count must equal the global-gather path's; grids that qualify for
    neither (three densities, > 40 KB) stay on global gathers."""
    three = W.c1(n_packets=50_000, batch=25_000)
    three.rho_root = three.rho_root.copy()
    three.rho_root[::7] *= np.float32(0.5)                     # a third distinct density
    for wl, mode in ((W.c0(), 1),
                     (W.tiny_random(n_root=3, seed=4, external=True, n_packets=40_000, batch=10_000), 1),
                     (W.c1(n_packets=300_000, batch=100_000), 2),
                     (W.c1(tau_v=100.0, n_packets=20_000, batch=10_000), 2),
                     (W.sphere(n_root=40, albedo=1.0, gval=0.4, n_packets=100_000, batch=50_000), 2),
                     (three, 0)):
        a = M.from_workload(wl, layout=1)                       # plain x-fastest grid (no macro cubes)
        assert a.density_staging() == (mode if mode == 1 else 0)   # the one-bit form is opt-in (measured slower)
        a.set_density_staging(2)
        assert a.density_staging() == mode, (wl.name, a.density_staging())
        b = M.from_workload(wl, layout=1)
        b.set_density_staging(1)
        assert b.density_staging() == 0
        for first, cnt in wl.batches():
            a.run_batch(wl.seed, first, cnt)
            b.run_batch(wl.seed, first, cnt)
        _assert_identical(a, b)
        assert a.get_counters()["emitted"] == wl.n_packets


# ---- macro cubes: uniform blocks of cells crossed in one step --------------------
def _blocky(n_root, block, seed, external=True, n_packets=300_000, batch=100_000):
    """A single-level grid whose density is constant on block^3 blocks (a few of them empty), point
    source off-centre + external field."""
    wl = W.tiny_random(n_root=n_root, seed=seed, external=external, tau_cell=0.25, n_packets=n_packets, batch=batch)
    rng = np.random.default_rng(seed)
    nb = n_root // block
    coarse = rng.random((nb, nb, nb)) * (rng.random((nb, nb, nb)) > 0.3)
    fine = np.kron(coarse, np.ones((block, block, block)))
    if n_root > 8:                                              # ... and one block with structure inside
        fine[:block, :block, :block] = rng.random((block, block, block))
    wl.rho_root = (fine.ravel() * wl.rho_root.max()).astype(np.float32)
    return wl


@pytest.mark.parametrize("maker,layout", [
    (lambda: W.c1(tau_v=1.0, n_packets=600_000, batch=200_000), 3),      # 4^3 macro cubes
    (lambda: W.c1(tau_v=10.0, n_packets=200_000, batch=50_000), 4),
    (lambda: W.sphere(n_root=32, tau_v=3.0, gval=0.3, n_packets=400_000, batch=100_000), 3),
    (lambda: _blocky(16, 4, 3), 3),
    (lambda: _blocky(24, 8, 5), 4),
    (lambda: _blocky(24, 4, 6, external=False), 3)])
def test_macro_cubes_against_oracle_and_plain_walk(M, oracle_mod, maker, layout):
    """Single-level grids run with macro cubes (uniform cubes of cells crossed in one step, empty space
    skipped, crossings counted from the ends of each flight): full parity rules against the oracle,
    and against the plain cell-by-cell walk of the same kernel the histories coincide except at
    rounding level -- event totals within 1e-3, including the arithmetic crossings count."""
    wl = maker()
    a = _run_layout(M, wl, 1)                                    # plain x-fastest walk
    b = _run_layout(M, wl, layout)
    ca, cb = a.get_counters(), b.get_counters()
    assert cb["emitted"] == cb["escaped"] == wl.n_packets and cb["lost"] == 0
    assert np.array_equal(ca["emitted_per_bin"], cb["emitted_per_bin"])
    for k in ("crossings", "absorptions", "scatterings", "flights"):
        assert abs(ca[k] - cb[k]) <= 1e-3 * ca[k] + 20, (k, ca[k], cb[k])
    na, nb_ = a.get_cell_energy()[0].astype(np.int64), b.get_cell_energy()[0].astype(np.int64)
    assert len(nb_) == wl.n_root ** 3 and np.abs(na - nb_).sum() <= 2e-3 * na.sum() + 50
    orc = oracle_mod.Oracle(wl).run()
    _compare(b, orc, groups=PR.super_blocks(wl.n_root, 4), min_count=300)


def test_macro_cubes_are_a_storage_layout_on_request(M):
    sphere = M.from_workload(W.c1(n_packets=10, batch=10))       # 64^3 sphere, automatic layout: the plain grid
    assert sphere.slots == 64 ** 3 and int(M.lib().mcrt_store_slots(sphere.h)) == 64 ** 3
    macro = M.from_workload(W.c1(n_packets=10, batch=10), layout=3)      # 16^3 macro cubes in front of the cells
    assert macro.slots == 64 ** 3 and int(M.lib().mcrt_store_slots(macro.h)) == 64 ** 3 + 16 ** 3


def test_region_sweeps_with_sharded_batches_and_observer(M):
    """Swept batches under the packet-sharded pair of calls (uint32 per-batch tally) and with the direction-resolved
    tallies switched on: two emulated ranks, swept, against ONE unswept context, bit for bit; the inclination-binned
    SEDs and images add up."""
    from paper_1201_3588_b200.sharding import rank_range
    wl = W.c4(n_root=256, n_packets=3 * (1 << 19), batch=1 << 20)
    obs = dict(n_mu=6, n_pix=16, direction=(0.3, -0.5, 0.81), half_angle_deg=12.0, half_width_cm=128 * wl.root_size)
    one = M.from_workload(wl)
    one.set_region_sweeps(0)
    one.set_observer(**obs)
    for first, cnt in wl.batches():
        one.run_batch(wl.seed, first, cnt)
    ranks = [M.from_workload(wl) for _ in range(2)]
    for ctx, sweeps in zip(ranks, (2, 5)):
        ctx.set_region_sweeps(sweeps, (128, 256, 128))
        ctx.set_observer(**obs)
    done = 0
    for first, cnt in wl.batches():
        deltas = []
        for r, ctx in enumerate(ranks):
            f, c = rank_range(first, cnt, 2, r)
            deltas.append(ctx.transport_batch_delta(wl.seed, f, c))
        done += cnt
        for ctx in ranks:
            ctx.accumulate_update(deltas[0] + deltas[1], done)
    for ctx in ranks:
        assert np.array_equal(ctx.get_cell_energy()[0], one.get_cell_energy()[0])
        assert np.array_equal(ctx.get_cell_temperature(), one.get_cell_temperature())
        assert ctx.get_region_sweep_counts()[0] > 0
    assert np.array_equal(ranks[0].get_sed() + ranks[1].get_sed(), one.get_sed())
    assert np.array_equal(ranks[0].get_sed_mu() + ranks[1].get_sed_mu(), one.get_sed_mu())
    assert np.array_equal(ranks[0].get_image() + ranks[1].get_image(), one.get_image())
    ca, cb, c1 = ranks[0].get_counters(), ranks[1].get_counters(), one.get_counters()
    for k in c1:
        assert np.array_equal(ca[k] + cb[k], c1[k]), k


def test_region_sweeps_do_not_change_results(M):
    """Grids far larger than the L2 are swept region by region (packages that cross a region boundary are
    suspended and continue in the next sweep, restored exactly): every count must equal the unswept run's,
    for any number of sweeps.  256^3 clumpy cube (8 regions of 128^3), 11 sources, batches of 2^20."""
    wl = W.c4(n_root=256, n_packets=(1 << 21) + 12345, batch=1 << 20)
    runs = []
    for sweeps, shape in ((0, (0, 0, 0)), (-1, (0, 0, 0)), (1, (0, 0, 0)), (3, (0, 0, 0)),
                          (2, (256, 128, 64)), (4, (64, 32, 128))):      # region shapes per axis
        ctx = M.from_workload(wl)
        ctx.set_region_sweeps(sweeps, shape)
        for first, cnt in wl.batches():
            ctx.run_batch(wl.seed, first, cnt)                   # the last batch (12345 packages) is never swept
        runs.append(ctx)
    for other in runs[1:]:
        _assert_identical(runs[0], other)
    c = runs[1].get_counters()
    assert c["emitted"] == c["escaped"] == wl.n_packets and c["lost"] == 0
    assert runs[1].kernel_launches() >= runs[0].kernel_launches() + 2 * 6 * 3     # two batches of six sweeps
    # packages suspended at the end of each sweep of the last batch (a forced sweep count applies to batches of any
    # size: here the 12345 left over): fewer every sweep, never more than the batch
    assert runs[0].get_region_sweep_counts().size == 0
    susp = runs[3].get_region_sweep_counts()[:3].astype(np.int64)
    assert 12345 > susp[0] > susp[1] > susp[2] > 0
    with pytest.raises(M.McrtError):
        runs[1].set_region_sweeps(2, (100, 128, 128))            # edges: multiples of 8 that divide n_root
    with pytest.raises(M.McrtError):
        runs[1].set_region_sweeps(2, (256, 256, 256))            # at least two regions
