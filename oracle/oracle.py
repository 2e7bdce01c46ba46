"""ctypes loader for the CPU oracle (oracle/ptycho_oracle.cpp) — TEST INFRASTRUCTURE, NOT THE PRODUCT.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference leg may import
this module.  It imports nothing from paper_2505_14372_b200 and the CUDA path imports nothing
from here.  All arithmetic is in the C++ file; this file only marshals numpy arrays.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from dataclasses import dataclass, field
from typing import Optional, Sequence

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "ptycho_oracle.cpp")
_LIB = os.path.join(_HERE, "libptycho_oracle.so")


def build(force: bool = False) -> str:
    """Compile the oracle with g++ (fp64, OpenMP over positions, no fast-math, no FMA contraction)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        cmd = ["g++", "-O2", "-std=c++17", "-fopenmp", "-ffp-contract=off", "-fPIC", "-shared", _SRC, "-o", _LIB]
        subprocess.run(cmd, check=True)
    return _LIB


class _Problem(C.Structure):
    _fields_ = [
        ("n", C.c_int32), ("n_modes", C.c_int32), ("n_slices", C.c_int32),
        ("obj_ny", C.c_int32), ("obj_nx", C.c_int32),
        ("n_pos_total", C.c_int32), ("n_batch", C.c_int32),
        ("pixel_size", C.c_float), ("wavelength", C.c_float),
        ("slice_thickness", C.POINTER(C.c_float)),
        ("tilt_x_mrad", C.c_float), ("tilt_y_mrad", C.c_float), ("bandlimit", C.c_float),
        ("loss", C.c_int32), ("loss_c", C.c_float), ("eps", C.c_float),
        ("lsqml_delta_o", C.c_float), ("lsqml_delta_p", C.c_float), ("shift_mode", C.c_int32),
        ("lsqml_chi_scale", C.c_float),
    ]


LOSS_AMPLITUDE, LOSS_POISSON, LOSS_GAUSSIAN = 0, 1, 2
SHIFT_FOURIER_PROBE, SHIFT_BILINEAR_OBJECT = 0, 1

_lib = None


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(build())
        _lib.orc_num_threads.restype = C.c_int32
    return _lib


def _p(a, ty):
    return None if a is None else a.ctypes.data_as(C.POINTER(ty))


@dataclass
class Problem:
    """Paper-side problem statement; the same float32 scalars the GPU gets."""
    n: int
    n_modes: int
    n_slices: int
    obj_ny: int
    obj_nx: int
    pixel_size: float = 1.0
    wavelength: float = 1.0
    slice_thickness: Sequence[float] = field(default_factory=lambda: [0.0])
    tilt_x_mrad: float = 0.0
    tilt_y_mrad: float = 0.0
    bandlimit: float = 0.0
    loss: int = LOSS_AMPLITUDE
    loss_c: float = 0.0
    eps: float = 0.5
    lsqml_delta_o: float = 1.0
    lsqml_delta_p: float = 0.0
    shift_mode: int = 0
    lsqml_chi_scale: float = 1.0    # chi = -lsqml_chi_scale gPhi: 1 steepest descent (R20), 2 modulus-constraint update (R31)

    def _c(self, n_pos_total: int, n_batch: int):
        dz = np.ascontiguousarray(np.asarray(self.slice_thickness, dtype=np.float32))
        if dz.size < self.n_slices:
            dz = np.concatenate([dz, np.zeros(self.n_slices - dz.size, np.float32)])
        s = _Problem(self.n, self.n_modes, self.n_slices, self.obj_ny, self.obj_nx, n_pos_total, n_batch,
                     self.pixel_size, self.wavelength, _p(dz, C.c_float), self.tilt_x_mrad, self.tilt_y_mrad,
                     self.bandlimit, self.loss, self.loss_c, self.eps, self.lsqml_delta_o, self.lsqml_delta_p,
                     self.shift_mode, self.lsqml_chi_scale)
        s._keep = dz
        return s


def _c64(a):
    return np.ascontiguousarray(a, dtype=np.complex64)


def _f32(a):
    return np.ascontiguousarray(a, dtype=np.float32)


def _batch(batch_idx, n_pos_total):
    if batch_idx is None:
        return None, n_pos_total
    b = np.ascontiguousarray(batch_idx, dtype=np.int32)
    return b, b.size


# ---- primitives exported for the pins ---------------------------------------------------------
def dft2_naive(a, sign=-1):
    a = np.ascontiguousarray(a, dtype=np.complex128); n = a.shape[0]; out = np.empty_like(a)
    lib().orc_dft2_naive(n, _p(a, C.c_double), _p(out, C.c_double), sign); return out


def dft2_bruteforce(a, sign=-1):
    a = np.ascontiguousarray(a, dtype=np.complex128); n = a.shape[0]; out = np.empty_like(a)
    lib().orc_dft2_bruteforce(n, _p(a, C.c_double), _p(out, C.c_double), sign); return out


def fft2(a, sign=-1):
    a = np.ascontiguousarray(a, dtype=np.complex128); n = a.shape[0]; out = np.empty_like(a)
    lib().orc_fft2(n, _p(a, C.c_double), _p(out, C.c_double), sign); return out


def position_split(X, px, n):
    r0 = C.c_int32(); d = C.c_float()
    lib().orc_position_split(C.c_float(X), C.c_float(px), n, C.byref(r0), C.byref(d))
    return r0.value, d.value


def position_split_floor(X, px, n):
    i0 = C.c_int32(); f = C.c_float()
    lib().orc_position_split_floor(C.c_float(X), C.c_float(px), n, C.byref(i0), C.byref(f))
    return i0.value, f.value


def bilinear(n, obj, i0y, i0x, fy, fx, patch=None):
    """patch = bilinear gather of obj (complex128 [ony][onx]) at corner (i0 + f); with `patch` given: the adjoint,
    obj += scatter(patch) in place (returns obj)."""
    obj = np.ascontiguousarray(obj, dtype=np.complex128); ony, onx = obj.shape
    if patch is None:
        out = np.empty((n, n), np.complex128)
        lib().orc_bilinear(n, ony, onx, _p(obj, C.c_double), i0y, i0x, C.c_double(fy), C.c_double(fx), _p(out, C.c_double), 0)
        return out
    patch = np.ascontiguousarray(patch, dtype=np.complex128)
    lib().orc_bilinear(n, ony, onx, _p(obj, C.c_double), i0y, i0x, C.c_double(fy), C.c_double(fx), _p(patch, C.c_double), 1)
    return obj


def propagator(n, px, lam, dz, tx=0.0, ty=0.0, bandlimit=0.0):
    out = np.empty((n, n), np.complex128)
    lib().orc_propagator(n, C.c_double(px), C.c_double(lam), C.c_double(dz), C.c_double(tx), C.c_double(ty),
                         C.c_double(bandlimit), _p(out, C.c_double)); return out


def shift(a, dy, dx, adjoint=False):
    a = np.ascontiguousarray(a, dtype=np.complex128); out = np.empty_like(a)
    lib().orc_shift(a.shape[0], _p(a, C.c_double), C.c_double(dy), C.c_double(dx), _p(out, C.c_double), int(adjoint)); return out


def propagate(a, px, lam, dz, tx=0.0, ty=0.0, bandlimit=0.0, adjoint=False):
    a = np.ascontiguousarray(a, dtype=np.complex128); out = np.empty_like(a)
    lib().orc_propagate(a.shape[0], _p(a, C.c_double), C.c_double(px), C.c_double(lam), C.c_double(dz), C.c_double(tx),
                        C.c_double(ty), C.c_double(bandlimit), _p(out, C.c_double), int(adjoint)); return out


def gather(obj, r0y, r0x, n):
    obj = np.ascontiguousarray(obj, dtype=np.complex128); out = np.empty((n, n), np.complex128)
    lib().orc_gather(n, obj.shape[0], obj.shape[1], _p(obj, C.c_double), r0y, r0x, _p(out, C.c_double)); return out


def scatter_add(obj, r0y, r0x, patch):
    assert obj.dtype == np.complex128 and obj.flags.c_contiguous
    patch = np.ascontiguousarray(patch, dtype=np.complex128)
    lib().orc_scatter_add(patch.shape[0], obj.shape[0], obj.shape[1], _p(obj, C.c_double), r0y, r0x, _p(patch, C.c_double))


def loss_pixel(kind, I, Iexp, c, eps):
    l = C.c_double(); w = C.c_double()
    lib().orc_loss_pixel(kind, C.c_double(I), C.c_double(Iexp), C.c_double(c), C.c_double(eps), C.byref(l), C.byref(w))
    return l.value, w.value


# ---- the model ---------------------------------------------------------------------------------
def forward_loss(pb: Problem, obj, probe, positions, intensity=None, batch_idx=None, want_intensity=True):
    """O0..O6. Returns dict(loss, loss_per_pos, intensity). intensity=None -> losses are zero."""
    obj = _c64(obj); probe = _c64(probe); positions = _f32(positions)
    npos = positions.shape[0]; b, J = _batch(batch_idx, npos)
    inten = None if intensity is None else _f32(intensity)
    cp = pb._c(npos, J)
    loss = C.c_double(0.0); lpp = np.zeros(J, np.float64)
    mi = np.zeros((J, pb.n, pb.n), np.float64) if want_intensity else None
    rc = lib().orc_forward_loss(C.byref(cp), _p(obj, C.c_float), _p(probe, C.c_float), _p(positions, C.c_float),
                                _p(inten, C.c_float), _p(b, C.c_int32), C.byref(loss), _p(lpp, C.c_double), _p(mi, C.c_double))
    if rc != 0:
        raise ValueError("oracle: window out of bounds")
    return dict(loss=loss.value, loss_per_pos=lpp, intensity=mi)


def epie(pb: Problem, obj, probe, positions, intensity, batch_idx=None):
    """Multislice ePIE update directions. Returns dict(loss, loss_per_pos, dir_object, dir_probe)."""
    obj = _c64(obj); probe = _c64(probe); positions = _f32(positions); inten = _f32(intensity)
    npos = positions.shape[0]; b, J = _batch(batch_idx, npos)
    cp = pb._c(npos, J)
    dO = np.zeros((pb.n_slices, pb.obj_ny, pb.obj_nx), np.complex128)
    dP = np.zeros((pb.n_modes, pb.n, pb.n), np.complex128)
    loss = C.c_double(); lpp = np.zeros(J, np.float64)
    rc = lib().orc_epie(C.byref(cp), _p(obj, C.c_float), _p(probe, C.c_float), _p(positions, C.c_float), _p(inten, C.c_float),
                        _p(b, C.c_int32), _p(dO, C.c_double), _p(dP, C.c_double), C.byref(loss), _p(lpp, C.c_double))
    if rc != 0:
        raise RuntimeError(f"orc_epie failed: {rc}")
    return dict(loss=loss.value, loss_per_pos=lpp, dir_object=dO, dir_probe=dP)


def gradient(pb: Problem, obj, probe, positions, intensity, batch_idx=None, want_illum=False):
    """O0..O12. Returns dict(loss, loss_per_pos, grad_object, grad_probe, grad_pos, illum)."""
    obj = _c64(obj); probe = _c64(probe); positions = _f32(positions); inten = _f32(intensity)
    npos = positions.shape[0]; b, J = _batch(batch_idx, npos)
    cp = pb._c(npos, J)
    gO = np.zeros((pb.n_slices, pb.obj_ny, pb.obj_nx), np.complex128)
    gP = np.zeros((pb.n_modes, pb.n, pb.n), np.complex128)
    gX = np.zeros((J, 2), np.float64)
    il = np.zeros((pb.n_slices, pb.obj_ny, pb.obj_nx), np.float64) if want_illum else None
    loss = C.c_double(0.0); lpp = np.zeros(J, np.float64)
    rc = lib().orc_gradient(C.byref(cp), _p(obj, C.c_float), _p(probe, C.c_float), _p(positions, C.c_float),
                            _p(inten, C.c_float), _p(b, C.c_int32), _p(gO, C.c_double), _p(gP, C.c_double),
                            _p(gX, C.c_double), _p(il, C.c_double), C.byref(loss), _p(lpp, C.c_double))
    if rc != 0:
        raise ValueError("oracle: window out of bounds")
    return dict(loss=loss.value, loss_per_pos=lpp, grad_object=gO, grad_probe=gP, grad_pos=gX, illum=il)


def step_terms(pb: Problem, obj, probe, positions, intensity, grad_object, grad_probe, illum_prev, batch_idx=None, probe_precond=None):
    """O13/O14. Returns [J][2S+6] float64."""
    obj = _c64(obj); probe = _c64(probe); positions = _f32(positions); inten = _f32(intensity)
    npos = positions.shape[0]; b, J = _batch(batch_idx, npos)
    cp = pb._c(npos, J)
    gO = np.ascontiguousarray(grad_object, np.complex128); gP = np.ascontiguousarray(grad_probe, np.complex128)
    ip = np.ascontiguousarray(illum_prev, np.float64)
    pc = None if probe_precond is None else np.ascontiguousarray(probe_precond, np.float64)
    out = np.zeros((J, 2 * pb.n_slices + 6), np.float64)
    rc = lib().orc_step_terms(C.byref(cp), _p(obj, C.c_float), _p(probe, C.c_float), _p(positions, C.c_float),
                              _p(inten, C.c_float), _p(b, C.c_int32), _p(gO, C.c_double), _p(gP, C.c_double),
                              _p(ip, C.c_double), _p(pc, C.c_double), _p(out, C.c_double))
    if rc == -2:
        raise ValueError("oracle: the modulus-constraint wavefront update (PAPER.md:173) is defined for the amplitude loss only")
    if rc != 0:
        raise ValueError("oracle: window out of bounds")
    return out


def apply_update(pb: Problem, mode, obj, probe, positions, grad_object=None, grad_probe=None, grad_pos=None,
                 illum_prev=None, step_terms_=None, batch_idx=None, lr_obj=0.0, lr_probe=0.0, lr_pos=0.0,
                 beta_obj=1.0, beta_probe=1.0, gamma=0.0, probe_precond=None):
    """O15/H15. Returns updated (object, probe, positions) as complex128/float64 copies."""
    o = np.array(obj, dtype=np.complex128, order="C"); pr = np.array(probe, dtype=np.complex128, order="C")
    x = np.array(positions, dtype=np.float64, order="C")
    npos = x.shape[0]; b, J = _batch(batch_idx, npos)
    cp = pb._c(npos, J)
    f = lambda a, t: None if a is None else np.ascontiguousarray(a, t)
    gO = f(grad_object, np.complex128); gP = f(grad_probe, np.complex128); gX = f(grad_pos, np.float64)
    ip = f(illum_prev, np.float64); st = f(step_terms_, np.float64); pc = f(probe_precond, np.float64)
    lib().orc_apply_update(C.byref(cp), int(mode), _p(o, C.c_double), _p(pr, C.c_double), _p(x, C.c_double),
                           _p(gO, C.c_double), _p(gP, C.c_double), _p(gX, C.c_double), _p(ip, C.c_double),
                           _p(st, C.c_double), _p(b, C.c_int32), C.c_double(lr_obj), C.c_double(lr_probe),
                           C.c_double(lr_pos), C.c_double(beta_obj), C.c_double(beta_probe), C.c_double(gamma), _p(pc, C.c_double))
    return o, pr, x


def object_transparency(pb: Problem, obj, positions, batch_idx=None):
    """sum_j prod_i |O_i|^2 in the probe/cutout view, [N][N] (reading R25)."""
    obj = _c64(obj); positions = _f32(positions)
    npos = positions.shape[0]; b, J = _batch(batch_idx, npos)
    cp = pb._c(npos, J)
    out = np.zeros((pb.n, pb.n), np.float64)
    rc = lib().orc_object_transparency(C.byref(cp), _p(obj, C.c_float), _p(positions, C.c_float), _p(b, C.c_int32), _p(out, C.c_double))
    if rc != 0:
        raise ValueError("oracle: window out of bounds")
    return out


def weighted_illum(pb: Problem, obj, probe, positions, step_terms_, gamma, batch_idx=None):
    """W_i = sum_j alpha_{O,i,j} sum_k |Psi_{i,k,j}|^2 scattered, alpha = numO/(denO+gamma) per position."""
    obj = _c64(obj); probe = _c64(probe); positions = _f32(positions)
    npos = positions.shape[0]; b, J = _batch(batch_idx, npos)
    cp = pb._c(npos, J)
    st = np.ascontiguousarray(step_terms_, np.float64)
    out = np.zeros((pb.n_slices, pb.obj_ny, pb.obj_nx), np.float64)
    rc = lib().orc_weighted_illum(C.byref(cp), _p(obj, C.c_float), _p(probe, C.c_float), _p(positions, C.c_float),
                                  _p(b, C.c_int32), _p(st, C.c_double), C.c_double(gamma), _p(out, C.c_double))
    if rc != 0:
        raise ValueError(f"oracle: weighted_illum failed ({rc})")
    return out


def lsqml_weighted_object(pb: Problem, obj, grad_object, illum_prev, illum_batch, willum, beta_obj=1.0):
    """O_i += beta_O dOhat_i W_i / I_i (PAPER.md:225 as printed). Returns the updated object (complex128 copy)."""
    o = np.array(obj, dtype=np.complex128, order="C")
    f = lambda a, t: np.ascontiguousarray(a, t)
    gO = f(grad_object, np.complex128); ip = f(illum_prev, np.float64); ib = f(illum_batch, np.float64); wi = f(willum, np.float64)
    cp = pb._c(1, 1)
    lib().orc_lsqml_weighted_object(C.byref(cp), _p(o, C.c_double), _p(gO, C.c_double), _p(ip, C.c_double), _p(ib, C.c_double),
                                    _p(wi, C.c_double), C.c_double(beta_obj))
    return o


REG_L2, REG_L1, REG_TIKHONOV, REG_TV, REG_LAYER_TIKHONOV, REG_LAYER_TV, REG_L1_PHASE, REG_L1_FOURIER = range(8)
CON_AMPLITUDE_CLAMP, CON_SUPPORT_MASK, CON_LAYER_BLUR, CON_LOWPASS, CON_SUPPORT_MASK_FOURIER, CON_PHASE_DERAMP = range(6)


def cost_regularizer(kind, weight, field_, ref=1.0, eps=0.0, grad=None):
    """Cost regulariser R (reading R26) of a [S][ny][nx] complex field; returns (R, grad + dR/dconj(field))."""
    z = np.ascontiguousarray(field_, np.complex128); S, ny, nx = z.shape
    g = np.zeros_like(z) if grad is None else np.array(grad, dtype=np.complex128, order="C")
    f = lib().orc_cost_regularizer; f.restype = C.c_double
    R = f(int(kind), C.c_double(weight), C.c_double(ref), C.c_double(eps), S, ny, nx, _p(z, C.c_double), _p(g, C.c_double))
    return float(R), g


def apply_constraint(kind, field_, a=0.0, b=0.0, mask=None):
    """Constraint regulariser (reading R27) on a [S][ny][nx] complex field; returns the new field."""
    z = np.array(field_, dtype=np.complex128, order="C"); S, ny, nx = z.shape
    mk = None if mask is None else np.ascontiguousarray(mask, np.float64)
    rc = lib().orc_apply_constraint(int(kind), C.c_double(a), C.c_double(b), _p(mk, C.c_double), S, ny, nx, _p(z, C.c_double))
    if rc != 0:
        raise ValueError(f"oracle: apply_constraint failed ({rc})")
    return z


def adam_update(z, g, m, v, lr, b1=0.9, b2=0.999, eps=1e-8, t=1):
    """One Adam step (reading R28). Complex z: complex m, real v = EMA of |g|^2. Returns new (z, m, v) copies."""
    cplx = np.iscomplexobj(z)
    ty = np.complex128 if cplx else np.float64
    z2 = np.array(z, dtype=ty, order="C"); m2 = np.array(m, dtype=ty, order="C"); v2 = np.array(v, dtype=np.float64, order="C")
    g2 = np.ascontiguousarray(g, ty)
    lib().orc_adam_update(int(cplx), _p(z2, C.c_double), _p(g2, C.c_double), _p(m2, C.c_double), _p(v2, C.c_double),
                          C.c_int64(z2.size), C.c_double(lr), C.c_double(b1), C.c_double(b2), C.c_double(eps), int(t))
    return z2, m2, v2


def num_threads() -> int:
    return int(lib().orc_num_threads())
