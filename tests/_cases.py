"""Shared set-up of the parity cases: seeded inputs (paper_2505_14372_b200.synth) -> the two Problem structs.

Holds no arithmetic of the method.  `make_case` builds object / probe / positions from a synth.Config and asks
the ORACLE for the noiseless pattern at the true state (then draws seeded Poisson counts), as DESIGN.md §4
states; nothing here ever comes from the CUDA path.
"""
from __future__ import annotations

from dataclasses import dataclass
from typing import Optional

import numpy as np

from oracle import oracle as orc
from paper_2505_14372_b200 import synth


def problem_kwargs(cfg: synth.Config, **over):
    kw = dict(n=cfg.n, n_modes=cfg.n_modes, n_slices=cfg.n_slices, obj_ny=cfg.obj_n, obj_nx=cfg.obj_n,
              pixel_size=cfg.pixel_size, wavelength=cfg.wavelength,
              slice_thickness=[cfg.dz] * cfg.n_slices, tilt_x_mrad=cfg.tilt_mrad[0], tilt_y_mrad=cfg.tilt_mrad[1],
              bandlimit=cfg.bandlimit, loss=cfg.loss, loss_c=cfg.loss_c, eps=cfg.eps)
    kw.update(over)
    return kw


def oracle_problem(cfg: synth.Config, **over) -> orc.Problem:
    return orc.Problem(**problem_kwargs(cfg, **over))


def gpu_problem(cfg: synth.Config, **over):
    from paper_2505_14372_b200 import ptycho
    return ptycho.Problem(**problem_kwargs(cfg, **over))


@dataclass
class Case:
    cfg: synth.Config
    obj_true: np.ndarray        # [S][No][No] complex64
    obj_start: np.ndarray       # [S][No][No] complex64
    probe: np.ndarray           # [M][N][N] complex64
    positions: np.ndarray       # [J][2] float32 nominal (start) positions
    positions_true: np.ndarray  # [J][2] float32
    intensity: np.ndarray       # [J][N][N] float32


def make_case(cfg: synth.Config, start_scale: float = 0.0, noise: bool = True, rows: Optional[np.ndarray] = None) -> Case:
    """start_scale: 0 -> vacuum start O = 1 (state (a)), 0.8 -> state (b) of SURVEY §8(d)."""
    phi = synth.object_phase(cfg)
    obj_true = synth.object_from_phase(phi, 1.0)
    obj_start = synth.object_from_phase(phi, start_scale)
    pr = synth.probe(cfg)
    pos = synth.positions(cfg)
    pos_true = synth.true_positions(cfg)
    if rows is not None:
        pos, pos_true = pos[rows], pos_true[rows]
    mean = orc.forward_loss(oracle_problem(cfg), obj_true, pr, pos_true)["intensity"]
    inten = synth.poisson_patterns(cfg, mean) if noise else mean.astype(np.float32)
    return Case(cfg, obj_true, obj_start, pr, pos, pos_true, inten)


def rel_l2(a, b) -> float:
    a = np.asarray(a); b = np.asarray(b)
    d = np.linalg.norm((a.astype(np.complex128) - b.astype(np.complex128)).ravel())
    return float(d / max(np.linalg.norm(b.astype(np.complex128).ravel()), 1e-300))
