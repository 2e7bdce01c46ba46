"""Seeded synthetic inputs for the five BASELINE.json configs (recipe: DESIGN.md §4).

This module serves BOTH the CUDA path (tests, bench.py) and the CPU oracle's tests.  It holds none of
the method's arithmetic: no forward model, no loss, no gradient.  It only draws seeded random numbers and
builds the *inputs* the paper's problem statement names: object slices O_i, probe
modes P_k, scan positions X_j — plus (a) Poisson sampling of a mean pattern that the CALLER supplies
(the tests pass the oracle's forward intensity) and (b) a closed-form stand-in pattern recipe for
full-size runs where no CPU forward is affordable.

The paper's experimental datasets (PrScO3, BaTiO3, Si) are not available; these inputs
stand in for them with the shapes the paper states (128x128 patterns, 64x64 / 80x80 scans, 20 slices,
300 kV, 25 mrad, ~10 nm defocus, perovskite ~3.9 A lattice).
"""
from __future__ import annotations

from dataclasses import dataclass, field, replace
from typing import List, Optional, Tuple

import numpy as np

LOSS_AMPLITUDE, LOSS_POISSON, LOSS_GAUSSIAN = 0, 1, 2


@dataclass
class Config:
    name: str
    n: int                      # N pattern / probe side
    scan: Tuple[int, int]       # raster (ny, nx)
    step_px: float              # raster step in px
    jitter_px: float            # uniform +-jitter per axis in px
    pixel_size: float           # Angstrom / px
    wavelength: float           # Angstrom
    obj_n: int                  # object side in px
    n_modes: int
    n_slices: int
    dz: float                   # slice thickness (Angstrom)
    tilt_mrad: Tuple[float, float] = (0.0, 0.0)   # (tilt_x, tilt_y)
    bandlimit: float = 0.0
    loss: int = LOSS_AMPLITUDE
    loss_c: float = 0.0
    eps: float = 0.5
    dose: float = 1e5           # electrons per pattern
    probe_kind: str = "stem"    # "stem" (aperture+defocus, Angstrom units) or "cfg1" (pixel units)
    object_kind: str = "perovskite"  # or "cfg1"
    pos_error_px: float = 0.0   # cfg 5: sigma of true-minus-nominal offsets
    seed: int = 0

    @property
    def n_pos(self) -> int:
        return self.scan[0] * self.scan[1]


def config(idx: int, **over) -> Config:
    """BASELINE.json configs 1..5.  Keyword overrides make reduced test cases."""
    lam = 0.0197
    base = {
        1: Config("cfg1_spoa_64", 64, (16, 16), 4.0, 0.5, 1.0, 1.0, 128, 1, 1, 0.0, loss=LOSS_AMPLITUDE, eps=0.5,
                  dose=1e4, probe_kind="cfg1", object_kind="cfg1", seed=1000),
        2: Config("cfg2_mixed_128", 128, (32, 32), 4.0, 0.25, 0.1, lam, 420, 4, 1, 0.0, loss=LOSS_AMPLITUDE, eps=0.5,
                  dose=1e5, seed=2000),
        3: Config("cfg3_multislice_128", 128, (64, 64), 4.0, 0.25, 0.1, lam, 420, 8, 20, 10.0, tilt_mrad=(0.8, 0.6),
                  loss=LOSS_POISSON, eps=0.8, dose=1e5, seed=3000),
        4: Config("cfg4_large_256", 256, (128, 128), 6.4, 0.25, 0.05, lam, 1100, 10, 30, 10.0, tilt_mrad=(0.8, 0.6),
                  loss=LOSS_POISSON, eps=0.8, dose=5e4, seed=4000),
        5: Config("cfg5_lsqml_128", 128, (64, 64), 4.0, 0.25, 0.1, lam, 420, 8, 20, 10.0, tilt_mrad=(0.8, 0.6),
                  loss=LOSS_POISSON, eps=0.8, dose=1e5, pos_error_px=0.3, seed=5000),
    }[idx]
    return replace(base, **over)


def _rng(cfg: Config, stream: int) -> np.random.Generator:
    # seed = 1000*config + stream; streams: 1 scan jitter, 2 object, 3 Poisson, 4 true-position offsets, 5 batch permutation
    return np.random.Generator(np.random.PCG64(cfg.seed + stream))


# ----------------------------------------------------------------------------------------------------
# scan positions X_j: probe-centre coordinates in Angstrom, object pixel (0,0) at 0
# ----------------------------------------------------------------------------------------------------
def positions(cfg: Config) -> np.ndarray:
    """Nominal positions [J][2] (y, x) float32 in Angstrom: centred raster + seeded uniform jitter."""
    ny, nx = cfg.scan
    yy = (np.arange(ny) - (ny - 1) / 2.0) * cfg.step_px + cfg.obj_n / 2.0
    xx = (np.arange(nx) - (nx - 1) / 2.0) * cfg.step_px + cfg.obj_n / 2.0
    Y, X = np.meshgrid(yy, xx, indexing="ij")
    p = np.stack([Y.ravel(), X.ravel()], axis=1)
    p = p + _rng(cfg, 1).uniform(-cfg.jitter_px, cfg.jitter_px, size=p.shape)
    return (p * cfg.pixel_size).astype(np.float32)


def true_positions(cfg: Config) -> np.ndarray:
    """cfg 5: nominal + N(0, pos_error_px) per axis (the positions the data are generated at)."""
    p = positions(cfg).astype(np.float64)
    if cfg.pos_error_px > 0:
        p = p + _rng(cfg, 4).normal(0.0, cfg.pos_error_px, size=p.shape) * cfg.pixel_size
    return p.astype(np.float32)


def batches(cfg: Config, batch: int, compact: bool = False) -> List[np.ndarray]:
    """Mini-batches (PAPER.md:55 'groups'): seeded permutation (sparse grouping) or raster blocks (compact)."""
    J = cfg.n_pos
    order = np.arange(J) if compact else _rng(cfg, 5).permutation(J)
    return [order[i:i + batch].astype(np.int32) for i in range(0, J, batch)]


# ----------------------------------------------------------------------------------------------------
# probe modes P_k: [M][N][N] complex64, real space, centred at (N/2, N/2)
# ----------------------------------------------------------------------------------------------------
def _signed_index(n: int) -> np.ndarray:
    i = np.arange(n)
    return np.where(i < n // 2, i, i - n)


def aperture_radius_px(cfg: Config) -> float:
    if cfg.probe_kind == "cfg1":
        return 12.0
    return 0.025 / cfg.wavelength * cfg.n * cfg.pixel_size   # 25 mrad semi-angle in Fourier pixels


def probe(cfg: Config) -> np.ndarray:
    N, M = cfg.n, cfg.n_modes
    s = _signed_index(N).astype(np.float64)
    KY, KX = np.meshgrid(s, s, indexing="ij")
    k2 = KY ** 2 + KX ** 2
    if cfg.probe_kind == "cfg1":
        Pt = (k2 <= 12.0 ** 2) * np.exp(1j * 0.02 * k2)                      # aperture radius 12 px, defocus 0.02 k^2 rad
    else:
        kap2 = k2 / (N * cfg.pixel_size) ** 2                                  # (cycles/Angstrom)^2
        kmax = 0.025 / cfg.wavelength
        Pt = (kap2 <= kmax ** 2) * np.exp(-1j * np.pi * cfg.wavelength * 100.0 * kap2)   # 100 A defocus (reading R22)
    base = np.fft.fftshift(np.fft.ifft2(Pt))                                   # centred at (N/2, N/2)
    if cfg.probe_kind == "cfg1":
        modes = [base]
        weights = [1.0]
    else:
        r = (np.arange(N) - N // 2) * cfg.pixel_size / 1.25                    # s = 1.25 Angstrom
        Yr, Xr = np.meshgrid(r, r, indexing="ij")
        he = [lambda t: np.ones_like(t), lambda t: t, lambda t: t * t - 1.0, lambda t: t ** 3 - 3.0 * t]
        order = [(0, 0), (1, 0), (0, 1), (1, 1), (2, 0), (0, 2), (2, 1), (1, 2), (2, 2), (3, 0), (0, 3), (3, 1)]
        modes = []
        for (m, n) in order[:M]:
            v = base * he[m](Xr) * he[n](Yr)
            for u in modes:                                                   # Gram-Schmidt in this order
                v = v - u * (np.vdot(u, v) / np.vdot(u, u))
            modes.append(v)
        w = np.array([0.7, 0.15, 0.1, 0.05] + [0.05 / 2 ** (i + 1) for i in range(max(0, M - 4))])[:M]
        weights = list(w / w.sum())
    out = np.empty((M, N, N), np.complex64)
    for k in range(M):
        v = modes[k]
        out[k] = (v * np.sqrt(weights[k] * cfg.dose / np.sum(np.abs(v) ** 2))).astype(np.complex64)
    return out


# ----------------------------------------------------------------------------------------------------
# object slices O_i: [S][No][No] complex64, O = exp(-0.05 phi) exp(i phi)
# ----------------------------------------------------------------------------------------------------
def _add_gaussians(phi: np.ndarray, cy, cx, peak, sigma: float):
    n = phi.shape[0]
    h = int(np.ceil(5 * sigma))
    for y0, x0, a in zip(cy, cx, peak):
        iy, ix = int(round(y0)), int(round(x0))
        ys = np.arange(max(0, iy - h), min(n, iy + h + 1)); xs = np.arange(max(0, ix - h), min(n, ix + h + 1))
        if ys.size == 0 or xs.size == 0:
            continue
        gy = np.exp(-0.5 * ((ys - y0) / sigma) ** 2); gx = np.exp(-0.5 * ((xs - x0) / sigma) ** 2)
        phi[np.ix_(ys, xs)] += a * np.outer(gy, gx)


def object_phase(cfg: Config) -> np.ndarray:
    """True projected phase per slice, [S][No][No] float64 (radians)."""
    n, S = cfg.obj_n, cfg.n_slices
    rng = _rng(cfg, 2)
    phi = np.zeros((S, n, n))
    if cfg.object_kind == "cfg1":
        c = 6.0 * np.arange(21) + 3.0
        CY, CX = np.meshgrid(c, c, indexing="ij")
        for i in range(S):
            _add_gaussians(phi[i], CY.ravel(), CX.ravel(), np.full(CY.size, 0.5), 1.5)
        return phi
    a = 3.9 / cfg.pixel_size
    sig = 0.3 / cfg.pixel_size
    ncell = int(np.ceil(n / a)) + 1
    motif = [(0.0, 0.0, 1.0), (0.5, 0.5, 0.7), (0.5, 0.0, 0.3), (0.0, 0.5, 0.3)]     # A, B, O, O
    for i in range(S):
        cy, cx, pk = [], [], []
        for (fy, fx, amp) in motif:
            gy, gx = np.meshgrid((np.arange(ncell) + fy) * a, (np.arange(ncell) + fx) * a, indexing="ij")
            cy.append(gy.ravel()); cx.append(gx.ravel()); pk.append(np.full(gy.size, amp))
        cy = np.concatenate(cy); cx = np.concatenate(cx); pk = np.concatenate(pk)
        if S > 1:                                                                 # per-slice seeded atom columns
            pk = pk * rng.uniform(0.8, 1.2, size=pk.shape)
            cy = cy + rng.normal(0.0, 0.05 / cfg.pixel_size, size=cy.shape)
            cx = cx + rng.normal(0.0, 0.05 / cfg.pixel_size, size=cx.shape)
        _add_gaussians(phi[i], cy, cx, pk, sig)
    return phi


def object_from_phase(phi: np.ndarray, scale: float = 1.0) -> np.ndarray:
    """O = exp((i - 0.05) * scale * phi); scale=1 true object, 0 vacuum start (a), 0.8 start (b)."""
    return np.exp((1j - 0.05) * scale * phi).astype(np.complex64)


# ----------------------------------------------------------------------------------------------------
# measured patterns I_exp: [J][N][N] float32, zero frequency at [0][0]
# ----------------------------------------------------------------------------------------------------
def poisson_patterns(cfg: Config, mean: np.ndarray) -> np.ndarray:
    """Seeded Poisson draw around a caller-supplied mean (the tests pass the ORACLE's forward intensity)."""
    return _rng(cfg, 3).poisson(np.maximum(mean, 0.0)).astype(np.float32)


def standin_patterns(cfg: Config, rows: Optional[np.ndarray] = None) -> np.ndarray:
    """Closed-form stand-in patterns for full-size runs (no forward model involved).

    mean_j[q] = dose * (0.9 * disk(q)/area + 0.1 * gauss_tail(q)) * (1 + 0.3 cos(2 pi (u_j . q)/N + phi_j)),
    disk = bright-field disk of the probe-forming aperture; then a seeded Poisson draw per pixel.  Row j
    depends only on (seed, j), so any subset of rows can be regenerated independently.
    """
    N = cfg.n
    s = _signed_index(N).astype(np.float64)
    QY, QX = np.meshgrid(s, s, indexing="ij")
    r = aperture_radius_px(cfg)
    disk = ((QY ** 2 + QX ** 2) <= r * r).astype(np.float64)
    tail = np.exp(-0.5 * (QY ** 2 + QX ** 2) / (2.0 * r) ** 2)
    base = cfg.dose * (0.9 * disk / disk.sum() + 0.1 * tail / tail.sum())
    rows = np.arange(cfg.n_pos) if rows is None else np.asarray(rows)
    out = np.empty((rows.size, N, N), np.float32)
    for o, j in enumerate(rows):
        g = np.random.Generator(np.random.PCG64([cfg.seed + 3, int(j)]))
        u = g.uniform(-3.0, 3.0, size=2); ph = g.uniform(0, 2 * np.pi)
        mean = base * (1.0 + 0.3 * np.cos(2 * np.pi * (u[0] * QY + u[1] * QX) / N + ph))
        out[o] = g.poisson(mean)
    return out
