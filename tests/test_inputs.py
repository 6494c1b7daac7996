"""The seeded input generators follow the frozen recipe and are deterministic."""
import numpy as np
import pytest

from paper_1908_03301_b200 import inputs


def test_deterministic_and_fp32():
    a = inputs.cfg3_percolation_3d(8, 7, 6, seed=2)
    b = inputs.cfg3_percolation_3d(8, 7, 6, seed=2)
    assert a.sha256() == b.sha256()
    assert a.gx.dtype == np.float32 and a.gx.shape == (6, 7, 8) and a.gx.flags.c_contiguous
    assert inputs.cfg3_percolation_3d(8, 7, 6, seed=3).sha256() != a.sha256()


def test_cfg1_range_half_open():
    n = inputs.cfg1_iid_2d(64, 64, seed=0)
    for g in (n.gx, n.gy):
        assert g.min() > 0.01 - 1e-7 and g.max() <= 1.0
    assert n.gz is None and n.nz == 1 and n.directions == (0,)


def test_cfg3_open_fraction_and_range():
    n = inputs.cfg3_percolation_3d(40, 40, 40, seed=2, p=0.30)
    for g in (n.gx, n.gy, n.gz):
        frac = np.mean(g > 0)
        assert abs(frac - 0.30) < 0.01
        assert g[g > 0].min() > 0.1 - 1e-7 and g.max() <= 1.0


def test_fbm_normalisation_spectrum_and_half_shift():
    rng = np.random.Generator(np.random.PCG64(1))
    H = 0.7
    B0, B = inputs.fbm_fields((256, 256), H, rng, bond_axes=(1, 0))
    assert abs(B0.mean()) < 1e-12 and abs(B0.std() - 1.0) < 1e-12
    # radial spectrum slope ~ -(2H + 2) in 2D (eq.(1): S ~ (w^2)^-(H+1))
    F = np.abs(np.fft.fft2(B0)) ** 2
    f = np.fft.fftfreq(256)
    k = np.sqrt(f[:, None] ** 2 + f[None, :] ** 2)
    sel = (k > 0.02) & (k < 0.3) & (F > 0)
    slope = np.polyfit(np.log(k[sel]), np.log(F[sel]), 1)[0]
    assert abs(slope + (2 * H + 2)) < 0.15
    # shifting by half a cell twice = shifting by one cell (band-limited, Nyquist removed)
    Fx = np.fft.fft(B[1], axis=1)
    m = np.rint(np.fft.fftfreq(256) * 256)
    again = np.fft.ifft(Fx * np.exp(1j * np.pi * m / 256)[None, :], axis=1).real
    assert np.max(np.abs(again - np.roll(B0, -1, axis=1))) < 1e-9
    # midpoint values interpolate the neighbours
    mid = 0.5 * (B0 + np.roll(B0, -1, axis=1))
    assert np.corrcoef(mid.ravel(), B[1].ravel())[0, 1] > 0.99


def test_cfg4_cut_fraction_is_pooled_quantile():
    n = inputs.cfg4_fbm_cut_3d(24, 24, 24, seed=3)
    closed = (np.sum(n.gx[:, :, :-1] == 0) + np.sum(n.gy[:, :-1, :] == 0) + np.sum(n.gz[:-1] == 0))
    total = n.gx[:, :, :-1].size + n.gy[:, :-1, :].size + n.gz[:-1].size
    assert abs(closed / total - 0.40) < 2.0 / total + 1e-6
    assert n.prune


def test_cfg5_layers():
    n = inputs.cfg5_stratified_3d(8, 8, 16, seed=4)
    lay = n.meta["layer_node"]
    ratio = n.gx.astype(np.float64) / lay[:, None, None]
    assert ratio.min() > 0.5 - 1e-6 and ratio.max() <= 1.5 + 1e-6
    assert n.directions == (0, 2)


def test_transpose_axes_moves_bonds_with_their_axis():
    n = inputs.iid_diluted(4, 3, 2, seed=1, p=1.0)
    t = inputs.transpose_axes(n, (1, 2, 0))
    # new x bond at new (i',j',k') = old y bond at old (i=k', j=i', k=j')
    assert t.gx[1, 0, 2] == n.gy[0, 2, 1]
    assert (t.nx, t.ny, t.nz) == (3, 2, 4)


def test_anisotropic_fbm_recipe():
    """PAPER.md:33-37 eq.(2): beta_x = beta_y is CFG2's isotropic recipe bit for bit; beta_x / beta_y > 1 gives
    layers parallel to x (the field varies less along x than along y); seeded, so reproducible."""
    a = inputs.cfg2_fbm_2d(64, 48, seed=5)
    b = inputs.aniso_fbm_2d(64, 48, 5, 0.7, 1.0, 1.0)
    assert np.array_equal(a.gx, b.gx) and np.array_equal(a.gy, b.gy)
    c = inputs.aniso_fbm_2d(128, 128, 5, 0.75, 16.0, 1.0)
    B = np.log(c.gx[0].astype(np.float64))
    assert np.var(np.diff(B, axis=1)) < 0.3 * np.var(np.diff(B, axis=0))
    d = inputs.aniso_fbm_2d(128, 128, 5, 0.75, 16.0, 1.0)
    assert c.sha256() == d.sha256() and c.directions == (0, 1)
