"""Seeded synthetic bond networks (inputs only -- none of the solver's arithmetic lives here).

This module is the ONE piece shared by the CPU oracle's tests and the CUDA path's tests / bench:
it turns a seed into the per-bond conductance arrays `gx, gy, gz` of a square / simple-cubic bond
network.  It never assembles an operator, never solves anything, never labels clusters.

Layout ("1D arrays"): every array is float32, C-ordered with shape
`(nz, ny, nx)` (x fastest; `nz == 1` for 2D), *forward-bond convention*:
    gx[k, j, i] = conductance of the bond (i,j,k) -- (i+1,j,k)
    gy[k, j, i] = conductance of the bond (i,j,k) -- (i,j+1,k)
    gz[k, j, i] = conductance of the bond (i,j,k) -- (i,j,k+1)          (None for 2D)
Entries whose forward neighbour lies outside the lattice (i == nx-1 for gx, ...) are NOT bonds; the
generators leave whatever the recipe drew there, on purpose, so that both sides are tested to ignore
them.  The float32 values ARE the problem (SURVEY.md 8(c) reading 14): both sides widen them exactly.

Recipes (SURVEY.md 8(d) "Frozen input recipe"; they stand in for the paper's own synthetic networks,
PAPER.md:27-51 FBM-correlated conductances, PAPER.md:132 random percolation, PAPER.md:140 correlated
deletion of the smallest conductances, PAPER.md:142 stratified media):
    RNG = numpy.random.Generator(numpy.random.PCG64(seed)); draws in the order written, each a full
    `(nz, ny, nx)` array in C order.
"""
from __future__ import annotations

from dataclasses import dataclass, field
import hashlib

import numpy as np
import scipy.fft as sfft


@dataclass
class Network:
    """A bond network: shapes, float32 conductances and a description of how it was made."""
    nx: int
    ny: int
    nz: int
    gx: np.ndarray
    gy: np.ndarray
    gz: np.ndarray | None
    directions: tuple = (0,)          # solve directions the config asks for (0=x, 1=y, 2=z)
    prune: bool = False               # config contains closed (g == 0) bonds
    name: str = ""
    meta: dict = field(default_factory=dict)

    @property
    def n_nodes(self) -> int:
        return self.nx * self.ny * self.nz

    def sha256(self) -> str:
        h = hashlib.sha256()
        for a in (self.gx, self.gy, self.gz):
            if a is not None:
                h.update(np.ascontiguousarray(a).tobytes())
        return h.hexdigest()


def _rng(seed: int) -> np.random.Generator:
    return np.random.Generator(np.random.PCG64(seed))


def _shape(nx: int, ny: int, nz: int) -> tuple:
    return (int(nz), int(ny), int(nx))


def _f32(a) -> np.ndarray:
    return np.ascontiguousarray(a, dtype=np.float32)


# --------------------------------------------------------------------------------------------------
# Fractional-Brownian-motion field by spectral synthesis (eq.(1), generalised to d
# dimensions as S(k) ~ |k|^-(2H+d), SURVEY.md 8(c) readings 12-13).
# --------------------------------------------------------------------------------------------------
def fbm_fields(shape: tuple, H: float, rng: np.random.Generator, bond_axes=(), beta=None) -> tuple:
    """Node-centred FBM field `B0` and, for each axis in `bond_axes`, the same realisation sampled at
    the midpoints of the bonds along that axis (half-cell Fourier shift).

    white noise w -> W = fftn(w) -> W * |k|^-(H + d/2) with k_i = m_i / n_i (cycles per sample), the
    k = 0 mode and every Nyquist plane (even n) zeroed -> inverse FFT.  All fields are normalised with
    the NODE field's mean and standard deviation.  Periodic on the box, no padding.
    `beta` (one positive number per array axis): the anisotropic spectrum of PAPER.md:33-35 eq.(2),
    S ~ (sum_a beta_a k_a^2)^-(H + d/2); None = isotropic, eq.(1).
    Returns (B0, {axis: B_axis}); axes index the array dimensions of `shape` (C order).
    """
    shape = tuple(int(s) for s in shape)
    d = sum(1 for s in shape if s > 1) or 1
    w = rng.standard_normal(shape)
    W = sfft.fftn(w, workers=-1)
    del w
    k2 = np.zeros(shape, dtype=np.float64)
    keep = np.ones(shape, dtype=bool)
    for ax, n in enumerate(shape):
        f = sfft.fftfreq(n)                      # m / n, signed
        sl = [None] * len(shape)
        sl[ax] = slice(None)
        k2 = k2 + (1.0 if beta is None else float(beta[ax])) * (f * f)[tuple(sl)]
        if n % 2 == 0 and n > 1:
            nyq = np.zeros(n, dtype=bool)
            nyq[n // 2] = True
            keep &= ~nyq[tuple(sl)]
    zero = k2 == 0.0
    k2[zero] = 1.0
    amp = k2 ** (-0.5 * (H + 0.5 * d))
    amp[zero] = 0.0
    amp[~keep] = 0.0
    del k2, keep, zero
    W *= amp
    del amp
    B0 = sfft.ifftn(W, workers=-1).real.copy()
    mean, std = float(B0.mean()), float(B0.std())
    out = {}
    for ax in bond_axes:
        n = shape[ax]
        m = np.rint(sfft.fftfreq(n) * n)         # signed integer frequency
        ph = np.exp(1j * np.pi * m / n)
        sl = [None] * len(shape)
        sl[ax] = slice(None)
        Ba = sfft.ifftn(W * ph[tuple(sl)], workers=-1).real
        out[ax] = (Ba - mean) / std
    B0 = (B0 - mean) / std
    return B0, out


# --------------------------------------------------------------------------------------------------
# The five BASELINE.json configs (and their scaled-down siblings: pass smaller n).
# --------------------------------------------------------------------------------------------------
def cfg1_iid_2d(nx: int = 64, ny: int = 64, seed: int = 0) -> Network:
    """CFG1: 2D, iid Uniform(0.01, 1] bonds; g = 1 - 0.99 u, u in [0,1); gx drawn first, then gy."""
    r = _rng(seed)
    shp = _shape(nx, ny, 1)
    gx = 1.0 - 0.99 * r.random(shp)
    gy = 1.0 - 0.99 * r.random(shp)
    return Network(nx, ny, 1, _f32(gx), _f32(gy), None, (0,), False, f"cfg1_iid2d_{nx}x{ny}_s{seed}")


def cfg2_fbm_2d(nx: int = 2048, ny: int = 2048, seed: int = 1, H: float = 0.7,
                sigma: float = 1.0) -> Network:
    """CFG2: 2D isotropic FBM log-conductance, g = exp(sigma * B) sampled at bond midpoints."""
    r = _rng(seed)
    _, B = fbm_fields((ny, nx), H, r, bond_axes=(1, 0))
    gx = np.exp(sigma * B[1]).reshape(_shape(nx, ny, 1))
    gy = np.exp(sigma * B[0]).reshape(_shape(nx, ny, 1))
    return Network(nx, ny, 1, _f32(gx), _f32(gy), None, (0,), False,
                   f"cfg2_fbm2d_{nx}x{ny}_H{H}_s{seed}")


def aniso_fbm_2d(nx: int, ny: int, seed: int, H: float, beta_x: float, beta_y: float = 1.0,
                 sigma: float = 1.0) -> Network:
    """2D FBM log-conductance with the ANISOTROPIC spectrum of PAPER.md:33-37 eq.(2),
    S = b / (beta_x w_x^2 + beta_y w_y^2)^(H+1); g = exp(sigma * B) at bond midpoints as in CFG2.
    beta_x / beta_y > 1 damps the variation along x: layers parallel to x.  Solved along x and y
    for the permeability anisotropy K_x / K_y of Fig.10.  beta_x = beta_y reproduces cfg2_fbm_2d."""
    r = _rng(seed)
    _, B = fbm_fields((ny, nx), H, r, bond_axes=(1, 0), beta=(beta_y, beta_x))
    gx = np.exp(sigma * B[1]).reshape(_shape(nx, ny, 1))
    gy = np.exp(sigma * B[0]).reshape(_shape(nx, ny, 1))
    return Network(nx, ny, 1, _f32(gx), _f32(gy), None, (0, 1), False,
                   f"anisofbm2d_{nx}x{ny}_H{H}_bx{beta_x}_by{beta_y}_s{seed}",
                   {"H": H, "beta_x": beta_x, "beta_y": beta_y, "sigma": sigma})


def cfg3_percolation_3d(nx: int = 256, ny: int = 256, nz: int = 256, seed: int = 2,
                        p: float = 0.30) -> Network:
    """CFG3: uncorrelated bond percolation; per array: u1 (open iff u1 < p), u2, g = open ? 1-0.9 u2 : 0."""
    r = _rng(seed)
    shp = _shape(nx, ny, nz)
    gs = []
    for _ in range(3):
        u1 = r.random(shp)
        u2 = r.random(shp)
        gs.append(_f32(np.where(u1 < p, 1.0 - 0.9 * u2, 0.0)))
    return Network(nx, ny, nz, gs[0], gs[1], gs[2], (0,), True,
                   f"cfg3_perc3d_{nx}x{ny}x{nz}_p{p}_s{seed}")


def cfg4_fbm_cut_3d(nx: int = 512, ny: int = 512, nz: int = 512, seed: int = 3, H: float = 0.3,
                    sigma: float = 1.5, cut: float = 0.40) -> Network:
    """CFG4: 3D FBM log-conductance + correlated percolation: bonds whose FBM value lies below the
    `cut` quantile (pooled over all in-lattice bonds of all directions) are closed."""
    r = _rng(seed)
    _, B = fbm_fields((nz, ny, nx), H, r, bond_axes=(2, 1, 0))
    Bx, By, Bz = B[2], B[1], B[0]
    pooled = np.concatenate([Bx[:, :, :nx - 1].ravel(), By[:, :ny - 1, :].ravel(),
                             Bz[:nz - 1, :, :].ravel()])
    t = float(np.quantile(pooled, cut)) if pooled.size else -np.inf
    del pooled
    gs = [_f32(np.where(b < t, 0.0, np.exp(sigma * b))) for b in (Bx, By, Bz)]
    return Network(nx, ny, nz, gs[0], gs[1], gs[2], (0,), True,
                   f"cfg4_fbmcut3d_{nx}x{ny}x{nz}_H{H}_s{seed}", {"threshold": t})


def cfg5_stratified_3d(nx: int = 512, ny: int = 512, nz: int = 512, seed: int = 4, H: float = 0.8,
                       sigma: float = 1.0) -> Network:
    """CFG5: layers along z from a 1D FBM profile, times iid Uniform(0.5, 1.5] in-layer noise."""
    r = _rng(seed)
    B0, B = fbm_fields((nz,), H, r, bond_axes=(0,))
    Bz = B[0]
    shp = _shape(nx, ny, nz)
    lay0 = np.exp(sigma * B0)[:, None, None]
    layz = np.exp(sigma * Bz)[:, None, None]
    gx = lay0 * (1.5 - r.random(shp))
    gy = lay0 * (1.5 - r.random(shp))
    gz = layz * (1.5 - r.random(shp))
    return Network(nx, ny, nz, _f32(gx), _f32(gy), _f32(gz), (0, 2), False,
                   f"cfg5_strat3d_{nx}x{ny}x{nz}_H{H}_s{seed}",
                   {"layer_node": np.exp(sigma * B0), "layer_bond_z": np.exp(sigma * Bz)})


# --------------------------------------------------------------------------------------------------
# Small structured networks used by pins and edge-case tests.
# --------------------------------------------------------------------------------------------------
def uniform(nx: int, ny: int, nz: int, g: float) -> Network:
    shp = _shape(nx, ny, nz)
    full = np.full(shp, g, dtype=np.float32)
    return Network(nx, ny, nz, full.copy(), full.copy(), full.copy() if nz > 1 else None,
                   (0,), False, f"uniform_{nx}x{ny}x{nz}_g{g}")


def layered_exact(nx: int, ny: int, nz: int, c, e) -> Network:
    """Noise-free stratified medium: gx = gy = c[k] inside layer k, gz = e[k] between layers k, k+1."""
    c = np.asarray(c, dtype=np.float32)
    e = np.asarray(e, dtype=np.float32)
    shp = _shape(nx, ny, nz)
    gx = np.broadcast_to(c[:, None, None], shp)
    gz = np.broadcast_to(e[:, None, None], shp)
    return Network(nx, ny, nz, _f32(gx), _f32(gx), _f32(gz), (0, 2), False,
                   f"layered_{nx}x{ny}x{nz}")


def iid_diluted(nx: int, ny: int, nz: int, seed: int, p: float, lo: float = 0.1,
                hi: float = 1.0) -> Network:
    """Random diluted network of any shape (2D when nz == 1): open with probability p, g in (lo, hi]."""
    r = _rng(seed)
    shp = _shape(nx, ny, nz)
    gs = []
    for _ in range(3 if nz > 1 else 2):
        u1 = r.random(shp)
        u2 = r.random(shp)
        gs.append(_f32(np.where(u1 < p, hi - (hi - lo) * u2, 0.0)))
    return Network(nx, ny, nz, gs[0], gs[1], gs[2] if nz > 1 else None, (0,), p < 1.0,
                   f"iid_{nx}x{ny}x{nz}_p{p}_s{seed}")


def transpose_axes(net: Network, perm: tuple) -> Network:
    """Relabel the lattice axes: new axis a is old axis perm[a] (0=x, 1=y, 2=z).  Data only."""
    old = {0: net.gx, 1: net.gy, 2: net.gz if net.gz is not None
           else np.zeros_like(net.gx)}
    dims = (net.nx, net.ny, net.nz)
    # array dims are (z, y, x) = lattice axes (2, 1, 0)
    arr_perm = tuple(2 - perm[2 - ad] for ad in range(3))
    new = [_f32(np.transpose(old[perm[a]], arr_perm)) for a in range(3)]
    nnx, nny, nnz = (dims[perm[0]], dims[perm[1]], dims[perm[2]])
    return Network(nnx, nny, nnz, new[0], new[1], new[2] if nnz > 1 else None,
                   net.directions, net.prune, net.name + f"_perm{perm}")
