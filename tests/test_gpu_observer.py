"""-m gpu: direction-resolved tallies (mcrt_set_observer / mcrt_get_sed_mu / mcrt_get_image) of
the CUDA path against the oracle's O9 on the same seeded inputs.  Both kernels (single-level and
two-level grids), both storage layouts.  Bin and pixel decisions are taken in fp32 on the GPU
and fp64 in the oracle, so counts are compared under the SED rule (2 % or 3 sigma) and exact
identities are checked on each side separately."""
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


def _both(M, O, wl, obs, layout=0, n_packets=None, batch=None):
    ctx = M.from_workload(wl, layout=layout)
    ctx.set_observer(**obs)
    orc = O.Oracle(wl)
    orc.set_observer(**obs)
    for first, cnt in wl.batches(n_packets, batch):
        ctx.run_batch(wl.seed, first, cnt)
        orc.run_batch(wl.seed, first, cnt)
    return ctx, orc


def _check(ctx, orc, img_min_total=1000):
    sm_g, sm_o = ctx.get_sed_mu(), orc.sed_mu()
    assert np.array_equal(sm_g.sum(axis=0), ctx.get_sed())      # exact identity on the GPU side
    assert sm_g.sum() == sm_o.sum() == ctx.get_counters()["escaped"]
    ok = PR.counts_close(sm_g.astype(np.int64), sm_o.astype(np.int64), 0.02)
    assert ok.all(), f"{(~ok).sum()} (mu, component, bin) counts outside 2 % or 3 sigma"
    # per inclination bin, summed over frequency: tight
    a, b = sm_g.sum(axis=(1, 2)).astype(np.int64), sm_o.sum(axis=(1, 2)).astype(np.int64)
    assert PR.counts_close(a, b, 0.005).all(), (a, b)
    ig, io = ctx.get_image().astype(np.int64), orc.image().astype(np.int64)
    assert io.sum() >= img_min_total
    assert PR.counts_close(ig.sum(), io.sum(), 0.005)
    ok = PR.counts_close(ig, io, 0.02)
    assert ok.all(), f"{(~ok).sum()} pixels outside 2 % or 3 sigma"
    return ig, io


@pytest.mark.parametrize("layout", [1, 2])
def test_observer_uniform_grid(M, oracle_mod, layout):
    wl = W.c0()
    obs = dict(n_mu=6, n_pix=9, direction=(0.4, -0.3, 0.8), half_angle_deg=25.0,
               half_width_cm=9 * wl.root_size)
    ctx, orc = _both(M, oracle_mod, wl, obs, layout=layout)
    ig, io = _check(ctx, orc)
    assert (io > 0).sum() > 40                                  # a resolved image, not one pixel


def test_observer_clumpy_cube_with_external_field(M, oracle_mod):
    wl = W.c4(n_root=24, n_packets=200_000, batch=50_000, corr_cells=3.0)
    obs = dict(n_mu=4, n_pix=12, direction=(1.0, 0.2, 0.1), half_angle_deg=30.0,
               half_width_cm=14 * wl.root_size, bin_lo=20, bin_hi=100)
    ctx, orc = _both(M, oracle_mod, wl, obs)
    _check(ctx, orc)


@pytest.mark.parametrize("direction", [(0.0, 0.0, 1.0), (0.0, 1.0, 0.15)])
def test_observer_two_level_disk(M, oracle_mod, direction):
    """Flared disk on a two-level grid (k_transport_u<., true>): face-on and nearly edge-on."""
    wl = W.c2(n_root=32, n_packets=300_000, batch=100_000)
    obs = dict(n_mu=8, n_pix=15, direction=direction, half_angle_deg=20.0,   # odd: the star is mid-pixel
               half_width_cm=16 * wl.root_size)
    ctx, orc = _both(M, oracle_mod, wl, obs)
    _check(ctx, orc)


def test_observer_near_the_pole(M, oracle_mod):
    """An observer 2 degrees off the z axis: the image axes are the orthonormal pair of R34's
    near-polar rule on both sides (e1 = x there was not normal to the line of sight)."""
    wl = W.c0()
    obs = dict(n_mu=4, n_pix=9, direction=(0.03, 0.02, 1.0), half_angle_deg=25.0,
               half_width_cm=9 * wl.root_size)
    ctx, orc = _both(M, oracle_mod, wl, obs)
    _check(ctx, orc)


def test_observer_geometry_without_oracle(M):
    """Empty grid, displaced point source: every accepted package lands in the pixel that the
    projection predicts (observer +x: columns = +y, rows = +z), and mu is uniform."""
    wl = W.c0()
    wl.rho_root = np.zeros_like(wl.rho_root)
    c = 8.0 * wl.root_size
    wl.sources = [W.Source(W.SRC_POINT, (c, c + 3 * wl.root_size, c - 2 * wl.root_size), W.LSUN, 5800.0)]
    ctx = M.from_workload(wl)
    ctx.set_observer(n_mu=10, n_pix=11, direction=(1, 0, 0), half_angle_deg=3.0, half_width_cm=5.5 * wl.root_size)
    n = 400_000
    ctx.run_batch(wl.seed, 0, n)
    img = ctx.get_image()
    assert img.sum() > 100 and img[3, 8] == img.sum(), np.argwhere(img > 0)
    per_mu = ctx.get_sed_mu().sum(axis=(1, 2)).astype(np.float64)
    assert per_mu.sum() == n
    assert (((per_mu - n / 10) ** 2) / (n / 10)).sum() < 9 + 5 * np.sqrt(18)


def test_observer_api_states(M):
    wl = W.c0()
    ctx = M.Context()
    ctx.grid_create(wl.n_root, 0, wl.origin, wl.root_size, None, wl.rho_root, None)
    with pytest.raises(M.McrtError):                            # ESTATE: needs n_bins
        ctx.set_observer(n_mu=4)
    ctx.set_opacity(wl.lambda_edges_um, wl.weight, wl.kabs, wl.ksca, wl.g)
    ctx.set_source(wl.sources)
    with pytest.raises(M.McrtError):                            # ESTATE: nothing set
        ctx.n_mu, ctx.n_pix = 4, 4
        ctx.get_sed_mu()
    with pytest.raises(M.McrtError):                            # EINVAL
        ctx.set_observer(n_pix=8, direction=(0, 0, 0), half_width_cm=1.0)
    ctx.set_observer(n_mu=4, n_pix=8, half_angle_deg=40.0, half_width_cm=8 * wl.root_size)
    ctx.run_batch(1, 0, 20_000)
    assert ctx.get_sed_mu().sum() == 20_000 and ctx.get_image().sum() > 0
    ctx.reset_tallies(1)
    assert ctx.get_sed_mu().sum() == 0 and ctx.get_image().sum() == 0
