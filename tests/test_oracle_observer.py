"""Pins of the oracle's direction-resolved tallies (O9, reading R34; the
paper's science product is an image and flux profiles).  No closed form of the
paper exists for them; these are invariants, symmetry and hand-computable geometry."""
import numpy as np
import pytest

from paper_1201_3588_b200 import workloads as W


def _empty(wl):
    wl.rho_root = np.zeros_like(wl.rho_root)
    return wl


def test_sed_mu_sums_to_sed_and_resets(oracle_mod):
    wl = W.c0()
    o = oracle_mod.Oracle(wl)
    o.set_observer(n_mu=7, n_pix=9, direction=(0.3, -0.2, 0.9), half_angle_deg=25.0,
                   half_width_cm=9 * wl.root_size)
    o.run_batch(wl.seed, 0, 30000)
    sm, sed, img = o.sed_mu(), o.sed(), o.image()
    assert np.array_equal(sm.sum(axis=0), sed)                 # every escape lands in one mu bin
    assert 0 < img.sum() <= sed.sum()
    o.reset_tallies(1)
    assert o.sed_mu().sum() == 0 and o.image().sum() == 0


def test_isotropic_source_is_uniform_in_mu_and_fills_the_cone(oracle_mod):
    """Empty grid, central star: escape directions are the emission directions, uniform in
    mu = d_z; the fraction inside a cone of half-angle alpha is (1 - cos alpha)/2; every
    package has impact vector 0, so all of them fall in the central pixel (n_pix odd)."""
    wl = _empty(W.c0())
    n = 400_000
    for direction in ((0, 0, 1), (1, 1, 1), (-2, 0.5, -0.3)):
        o = oracle_mod.Oracle(wl)
        alpha = 17.0
        o.set_observer(n_mu=20, n_pix=11, direction=direction, half_angle_deg=alpha,
                       half_width_cm=5.5 * wl.root_size)
        o.run_batch(wl.seed, 0, n)
        per_mu = o.sed_mu().sum(axis=(1, 2)).astype(np.float64)
        assert per_mu.sum() == n
        chi2 = ((per_mu - n / 20) ** 2 / (n / 20)).sum()
        assert chi2 < 19 + 5 * np.sqrt(2 * 19), chi2
        img = o.image()
        expect = n * (1 - np.cos(np.radians(alpha))) / 2
        assert abs(img.sum() - expect) < 4 * np.sqrt(expect)
        assert img[5, 5] == img.sum()                          # impact vector = 0 -> centre pixel


@pytest.mark.parametrize("obs,shift,pixel", [
    # observer +z: e1 = +x (columns), e2 = obs x e1 = +y (rows)
    ((0, 0, 1), (3.0, 0.0, 0.0), (5, 8)),
    ((0, 0, 1), (0.0, -2.0, 0.0), (3, 5)),
    ((0, 0, 1), (0.0, 0.0, 4.0), (5, 5)),                      # along the line of sight: no shift
    # observer +x: e1 = z x obs = +y (columns), e2 = obs x e1 = +z (rows)
    ((1, 0, 0), (0.0, 3.0, 0.0), (5, 8)),
    ((1, 0, 0), (0.0, 0.0, 2.0), (7, 5)),
    # observer -y: e1 = z x obs = +x, e2 = obs x e1 = (-y) x x = +z
    ((0, -1, 0), (1.0, 0.0, -3.0), (2, 6)),
])
def test_image_axes_and_orientation(oracle_mod, obs, shift, pixel):
    """A point source displaced from the box centre in an empty grid appears in the pixel its
    projection on (e1, e2) predicts (1 pixel = 1 cell here): pins basis, signs and row/column."""
    wl = _empty(W.c0())
    c = 8.0 * wl.root_size
    wl.sources = [W.Source(W.SRC_POINT, tuple(c + s * wl.root_size for s in shift), W.LSUN, 5800.0)]
    o = oracle_mod.Oracle(wl)
    o.set_observer(n_mu=0, n_pix=11, direction=obs, half_angle_deg=3.0, half_width_cm=5.5 * wl.root_size)
    o.run_batch(wl.seed, 0, 300_000)
    img = o.image()
    assert img.sum() > 100
    # within the 3-degree cone the impact vector of the same source moves by at most
    # |shift| * sin(3 deg) < 0.27 cell around the exact projection, which sits mid-pixel
    assert img[pixel] == img.sum(), (np.argwhere(img > 0), pixel)


def test_symmetric_sphere_is_uniform_in_mu(oracle_mod):
    """Uniform sphere, central star, scattering + re-emission: the escaping radiation field is
    isotropic by symmetry, so every (component, mu-bin) count is flat in mu."""
    wl = W.c0()
    o = oracle_mod.Oracle(wl)
    o.set_observer(n_mu=8)
    o.run(200_000, 50_000)
    sm = o.sed_mu().sum(axis=2).astype(np.float64)             # [mu][component]
    for comp in range(3):
        col = sm[:, comp]
        chi2 = ((col - col.mean()) ** 2 / col.mean()).sum()
        assert chi2 < 7 + 5 * np.sqrt(14), (comp, chi2)
    # image of the sphere seen along an axis is invariant under the 90-degree rotation about it
    o2 = oracle_mod.Oracle(wl)
    o2.set_observer(n_pix=9, direction=(0, 0, 1), half_angle_deg=30.0, half_width_cm=9 * wl.root_size)
    o2.run(400_000, 100_000)
    img = o2.image().astype(np.float64)
    rot = np.rot90(img)
    sel = (img + rot) > 200
    z = (img - rot)[sel] / np.sqrt((img + rot)[sel])
    assert np.abs(z).max() < 5.0 and sel.sum() >= 9


@pytest.mark.parametrize("obs", [(0.0, 0.0, 1.0), (0.03, 0.02, 1.0), (-0.04, 0.01, -1.0),
                                 (0.044, 0.0, 0.999), (0.3, -0.2, 0.9), (1.0, 0.0, 0.0)])
def test_image_axes_are_orthonormal(oracle_mod, obs):
    """(e1, e2, obs) is a right-handed orthonormal triad for every observer direction, also within
    2.6 degrees of the pole where z x obs is ill-conditioned (R34; the old rule kept
    e1 = x there, which is not normal to obs)."""
    o = oracle_mod.Oracle(W.c0())
    o.set_observer(n_pix=3, direction=obs, half_width_cm=1.0)
    d, e1, e2 = o.observer_axes()
    want = np.array(obs) / np.linalg.norm(obs)
    assert np.allclose(d, want, atol=1e-15)
    for v in (e1, e2):
        assert abs(np.linalg.norm(v) - 1) < 1e-14
    assert abs(e1 @ d) < 1e-14 and abs(e2 @ d) < 1e-14 and abs(e1 @ e2) < 1e-14
    assert np.allclose(np.cross(d, e1), e2, atol=1e-14)
    if obs == (0.0, 0.0, 1.0):
        assert np.array_equal(e1, [1.0, 0.0, 0.0])
