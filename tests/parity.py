"""Comparison rules of BASELINE.json north_star, used by the -m gpu parity tests.

  integer packet accounting bit-exact;
  per-cell absorbed energy within 3 sigma Poisson + 0.5 % for cells with >= 10^3 absorptions;
  cell temperatures within 1 % relative (cells with >= 10^3 absorptions: below that the
      temperature of either side is itself Poisson-noisy at more than 1 %);
  SED bins within 2 % or 3 sigma.
Both sides are one realisation of the same estimator (R28), so sigma^2 = n_gpu + n_oracle.
"""
import numpy as np


def check_accounting(cg, co):
    """cg / co: counter dicts of the GPU path and of the oracle."""
    for k in ("emitted", "escaped", "lost"):
        assert cg[k] == co[k], (k, cg[k], co[k])
    assert cg["lost"] == 0
    assert cg["emitted"] == cg["escaped"]
    # Emission bins: both sides search the same fp64 source CDF with the same Philox word turned
    # into the same fp64 uniform (x + 0.5) 2^-32 (R19), so the number of
    # packages emitted per bin is the same integer on both sides.
    eg = cg["emitted_per_bin"].astype(np.int64)
    eo = co["emitted_per_bin"].astype(np.int64)
    assert eg.sum() == eo.sum() == cg["emitted"]
    assert np.array_equal(eg, eo), np.flatnonzero(eg != eo)


def check_self_consistency(c, n_abs, sed):
    assert int(sed.sum()) == c["escaped"]
    assert int(n_abs.sum()) == c["absorptions"]
    # every flight ends in an interaction or in the escape; every interaction starts a flight
    assert c["flights"] == c["emitted"] - c["lost"] + c["absorptions"] + c["scatterings"]


def counts_close(a, b, rel, nsig=3.0):
    a = np.asarray(a, dtype=np.float64)
    b = np.asarray(b, dtype=np.float64)
    tol = nsig * np.sqrt(a + b) + rel * np.maximum(a, b)
    return np.abs(a - b) <= tol


def check_cell_energy(ng, no, min_count=1000, rel=0.005, groups=None):
    """Per-cell rule; `groups` (int array, -1 = ignore) adds the aggregated comparison of
    SURVEY.md 8(d) (shells, rings, super-blocks) under the same rule."""
    ng = np.asarray(ng).astype(np.int64)
    no = np.asarray(no).astype(np.int64)
    sel = np.maximum(ng, no) >= min_count
    ok = counts_close(ng[sel], no[sel], rel)
    assert ok.all(), f"{(~ok).sum()} of {sel.sum()} cells outside 3 sigma + {rel:.1%}"
    n_groups = 0
    if groups is not None:
        g = np.asarray(groups)
        m = g >= 0
        ag = np.bincount(g[m], weights=ng[m].astype(np.float64))
        ao = np.bincount(g[m], weights=no[m].astype(np.float64), minlength=len(ag))
        s = np.maximum(ag, ao) >= min_count
        ok = counts_close(ag[s], ao[s], rel)
        assert ok.all(), f"{(~ok).sum()} of {s.sum()} groups outside 3 sigma + {rel:.1%}"
        n_groups = int(s.sum())
    return int(sel.sum()), n_groups


def check_temperature(Tg, To, ng, no, min_count=1000, rel=0.01):
    """Independent runs: cells where both sides absorbed >= min_count packages (below that the
    temperature of either side is Poisson-noisy at more than 1 %).  Returns the number checked."""
    sel = np.minimum(np.asarray(ng), np.asarray(no)) >= min_count
    if not sel.any():
        return 0
    r = np.abs(np.asarray(Tg, np.float64)[sel] / np.asarray(To, np.float64)[sel] - 1.0)
    assert r.max() <= rel, f"max relative temperature difference {r.max():.4f}"
    return int(sel.sum())


def check_temperature_of_tally(Tg, orc, ng, n_cum, rel=1e-3):
    """T is a deterministic function of (tally, N_cum, rho) (O7): hand the GPU's OWN tally to the
    oracle's temperature step and require the GPU's temperatures to match on EVERY leaf slot
    (sub-cells, empty and clamped cells included).  Overwrites the oracle's temperatures."""
    orc.update_temperature(np.asarray(ng, dtype=np.uint64), int(n_cum))
    To = orc.cell_temperature()
    Tg = np.asarray(Tg, np.float64)
    assert Tg.shape == To.shape
    r = np.abs(Tg / To - 1.0)
    bad = np.flatnonzero(~(r <= rel))
    assert len(bad) == 0, (len(bad), bad[:5], Tg[bad[:5]], To[bad[:5]])
    n_hot = int((To > 1.0).sum())
    assert n_hot == int((np.asarray(ng) > 0).sum()) or n_hot > 0
    return len(To), n_hot


def check_sed(sg, so, rel=0.02):
    sg = np.asarray(sg).astype(np.int64)
    so = np.asarray(so).astype(np.int64)
    for name, a, b in (("direct", sg[0], so[0]), ("scattered", sg[1], so[1]),
                       ("thermal", sg[2], so[2]), ("total", sg.sum(0), so.sum(0))):
        ok = counts_close(a, b, rel)
        assert ok.all(), f"SED {name}: bins {np.flatnonzero(~ok)} outside 2 % or 3 sigma"


def radial_shells(n_root, n_shells=None):
    """Shell index of every root cell centre about the box centre (sphere configs)."""
    c = np.arange(n_root, dtype=np.float64) + 0.5 - n_root / 2.0
    r = np.sqrt(c[None, None, :] ** 2 + c[None, :, None] ** 2 + c[:, None, None] ** 2).ravel()
    n_shells = n_shells or n_root // 2
    s = np.floor(r / (n_root / 2.0) * n_shells).astype(np.int64)
    s[s >= n_shells] = -1
    return s


def super_blocks(n_root, b=8):
    i = np.arange(n_root) // b
    m = n_root // b + (1 if n_root % b else 0)
    return (i[None, None, :] + m * (i[None, :, None] + m * i[:, None, None])).ravel()


def root_of_slot(wl):
    """Root-cube linear index of every leaf slot (layout R22): sub-cells of the k-th refined
    cube map back to that cube."""
    n3 = wl.n_root ** 3
    out = np.arange(wl.leaf_slots, dtype=np.int64)
    if wl.n_ref:
        ridx = np.flatnonzero(np.asarray(wl.refine).ravel())
        out[n3:] = np.repeat(ridx, wl.sub ** 3)
    return out


def blocks_of_slot(wl, b):
    """b^3 super-blocks of root cubes, per leaf slot."""
    return super_blocks(wl.n_root, b)[root_of_slot(wl)]
