"""Thin binding over the C-ABI library (include/ptycho.h): argument marshalling only.

Every numerical step runs in the CUDA kernels of csrc/ptycho_kernels.cu.  PyTorch supplies device memory and
the stream.  There is no CPU fallback: if the library is missing or no CUDA device is present, calls raise.
Names and arguments follow include/ptycho.h (ptycho_forward_loss, ptycho_gradient, ptycho_apply_update).
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from dataclasses import dataclass, field
from typing import Optional, Sequence

_HERE = os.path.dirname(os.path.abspath(__file__))
_CSRC = os.path.join(_HERE, "csrc")
LIB_PATH = os.path.join(_HERE, "libptycho_b200.so")

LOSS_AMPLITUDE, LOSS_POISSON, LOSS_GAUSSIAN = 0, 1, 2
SHIFT_FOURIER_PROBE, SHIFT_BILINEAR_OBJECT = 0, 1
WANT_POS_GRAD, WANT_ILLUM, WANT_STEP_SIZES, ACCUMULATE, EPIE, WANT_WEIGHTED_ILLUM, NO_MODE_PAIRS, LSQML_MODULUS_CHI, STASH_FP16, NO_SINGLE_SLICE_FUSION = 1, 2, 4, 16, 32, 64, 128, 256, 512, 1024
UPDATE_SGD, UPDATE_LSQML, UPDATE_EPIE, UPDATE_LSQML_WEIGHTED = 0, 1, 2, 3
OK = 0
EXPORTS = ["ptycho_workspace_bytes", "ptycho_workspace_min_bytes", "ptycho_positions_in_flight", "ptycho_forward_loss", "ptycho_gradient",
           "ptycho_apply_update", "ptycho_object_transparency", "ptycho_workspace_host_bytes", "ptycho_gradient_host", "ptycho_status",
           "ptycho_launch_count", "ptycho_strerror", "ptycho_profile_enable", "ptycho_profile_num_kernels",
           "ptycho_profile_kernel_name", "ptycho_profile_read", "ptycho_profile_fp32_peak", "ptycho_regularizer_workspace_bytes", "ptycho_cost_regularizer",
           "ptycho_apply_constraint", "ptycho_apply_constraint_static", "ptycho_adam_update", "ptycho_adam_update_real"]


def build(force: bool = False, verbose: bool = False) -> str:
    """nvcc -gencode arch=compute_100a,code=sm_100a -lineinfo ... -> in-tree libptycho_b200.so"""
    srcs = [os.path.join(_CSRC, f) for f in ("ptycho_kernels.cu", "fft_core.cuh", "regularizers.cuh")] + [os.path.join(_HERE, "..", "include", "ptycho.h")]
    if not force and os.path.exists(LIB_PATH) and all(os.path.getmtime(LIB_PATH) >= os.path.getmtime(s) for s in srcs):
        return LIB_PATH
    # four build units compiled side by side (csrc/ptycho_kernels.cu, PTK_ONLY_GEO): the C ABI and one per FFT geometry
    base = ["nvcc", "-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-std=c++17", "-lineinfo", "-Xcompiler", "-fPIC"]
    if verbose:
        base.append("-Xptxas=-v")
    bdir = os.path.join(_HERE, "build")
    os.makedirs(bdir, exist_ok=True)
    units = [(g, os.path.join(bdir, f"ptycho_geo{g}.o")) for g in (0, 64, 128, 256)]
    procs = [subprocess.Popen(base + [f"-DPTK_ONLY_GEO={g}", "-c", "-o", o, os.path.join(_CSRC, "ptycho_kernels.cu")]) for g, o in units]
    if any(pr.wait() != 0 for pr in procs):
        raise RuntimeError("nvcc failed")
    subprocess.run(["nvcc", "-shared", "-o", LIB_PATH] + [o for _, o in units], check=True)
    return LIB_PATH


class PtProblem(C.Structure):
    _fields_ = [
        ("n", C.c_int32), ("n_modes", C.c_int32), ("n_slices", C.c_int32), ("obj_ny", C.c_int32), ("obj_nx", C.c_int32),
        ("n_pos_total", C.c_int32), ("n_batch", C.c_int32), ("pixel_size", C.c_float), ("wavelength", C.c_float),
        ("slice_thickness", C.POINTER(C.c_float)), ("tilt_x_mrad", C.c_float), ("tilt_y_mrad", C.c_float),
        ("bandlimit", C.c_float), ("loss", C.c_int32), ("loss_c", C.c_float), ("eps", C.c_float),
        ("shift_mode", C.c_int32), ("flags", C.c_int32), ("lsqml_delta_o", C.c_float), ("lsqml_delta_p", C.c_float),
        ("lsqml_gamma", C.c_float), ("lsqml_probe_precond_d", C.c_void_p),
    ]


class PtUpdate(C.Structure):
    _fields_ = [("mode", C.c_int32), ("lr_obj", C.c_float), ("lr_probe", C.c_float), ("lr_pos", C.c_float),
                ("beta_obj", C.c_float), ("beta_probe", C.c_float), ("gamma", C.c_float), ("illum_batch_d", C.c_void_p)]


_lib = None


def lib():
    """Load the CUDA library; raise loudly if it is not there (no fallback of any kind)."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise RuntimeError(f"{LIB_PATH} is missing: run `python -c 'import __graft_entry__ as g; g.build()'`")
        l = C.CDLL(LIB_PATH)
        l.ptycho_workspace_bytes.restype = C.c_size_t
        l.ptycho_workspace_min_bytes.restype = C.c_size_t
        l.ptycho_workspace_host_bytes.restype = C.c_size_t
        l.ptycho_launch_count.restype = C.c_int64
        l.ptycho_strerror.restype = C.c_char_p
        l.ptycho_profile_kernel_name.restype = C.c_char_p
        for f in ("ptycho_forward_loss", "ptycho_gradient", "ptycho_apply_update", "ptycho_gradient_host", "ptycho_status",
                  "ptycho_object_transparency"):
            getattr(l, f).restype = C.c_int32
        _lib = l
    return _lib


class PtychoError(RuntimeError):
    def __init__(self, code):
        self.code = code
        super().__init__(f"ptycho error {code}: {lib().ptycho_strerror(code).decode()}")


@dataclass
class Problem:
    """pt_problem (include/ptycho.h); n_pos_total / n_batch are filled per call from the tensors."""
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
    shift_mode: int = SHIFT_FOURIER_PROBE
    lsqml_delta_o: float = 1.0
    lsqml_delta_p: float = 0.0
    lsqml_gamma: float = 0.0
    lsqml_probe_precond: object = None      # CUDA float32 [N][N] tensor or None (include/ptycho.h)

    def c_struct(self, n_pos_total: int, n_batch: int, flags: int = 0) -> PtProblem:
        dz = list(self.slice_thickness) + [0.0] * max(0, self.n_slices - len(self.slice_thickness))
        arr = (C.c_float * self.n_slices)(*dz[: self.n_slices])
        s = PtProblem(self.n, self.n_modes, self.n_slices, self.obj_ny, self.obj_nx, n_pos_total, n_batch,
                      self.pixel_size, self.wavelength, C.cast(arr, C.POINTER(C.c_float)), self.tilt_x_mrad,
                      self.tilt_y_mrad, self.bandlimit, self.loss, self.loss_c, self.eps, self.shift_mode, flags,
                      self.lsqml_delta_o, self.lsqml_delta_p, self.lsqml_gamma,
                      None if self.lsqml_probe_precond is None else _precond_ptr(self.lsqml_probe_precond))
        s._keep = arr
        return s


def _precond_ptr(t):
    import torch
    if not (isinstance(t, torch.Tensor) and t.is_cuda and t.dtype == torch.float32 and t.is_contiguous()):
        raise TypeError("lsqml_probe_precond: expected a contiguous CUDA float32 tensor")
    return t.data_ptr()


def _ptr(t):
    return C.c_void_p(0) if t is None else C.c_void_p(t.data_ptr())


def _stream():
    import torch
    return C.c_void_p(torch.cuda.current_stream().cuda_stream)


def _check(rc):
    if rc != OK:
        raise PtychoError(rc)


def _dev(t, dtype, name):
    import torch
    if t is None:
        return None
    if not (isinstance(t, torch.Tensor) and t.is_cuda and t.dtype == dtype and t.is_contiguous()):
        raise TypeError(f"{name}: expected a contiguous CUDA tensor of dtype {dtype}")
    return t


def workspace_bytes(pb: Problem, n_pos_total: int, n_batch: int, flags: int = 0, minimum: bool = False, host: bool = False) -> int:
    cs = pb.c_struct(n_pos_total, n_batch, flags)
    f = lib().ptycho_workspace_host_bytes if host else (lib().ptycho_workspace_min_bytes if minimum else lib().ptycho_workspace_bytes)
    n = int(f(C.byref(cs)))
    if n == 0:
        raise PtychoError(-2)
    return n


def positions_in_flight(pb: Problem, n_pos_total: int, n_batch: int, flags: int = 0, workspace_bytes_: Optional[int] = None) -> int:
    """ptycho_positions_in_flight: chunk size for a workspace of the given (default: recommended) size."""
    cs = pb.c_struct(n_pos_total, n_batch, flags)
    n = workspace_bytes(pb, n_pos_total, n_batch, flags) if workspace_bytes_ is None else workspace_bytes_
    f = lib().ptycho_positions_in_flight
    f.restype = C.c_int32
    return int(f(C.byref(cs), C.c_size_t(n)))


def make_workspace(pb: Problem, n_pos_total: int, n_batch: int, flags: int = 0, max_bytes: Optional[int] = None, host: bool = False):
    """Allocate (with torch) a workspace tensor for the given problem; the first 256 bytes are zeroed (status word)."""
    import torch
    n = workspace_bytes(pb, n_pos_total, n_batch, flags, host=host)
    if max_bytes is not None and n > max_bytes:
        n = max(max_bytes, workspace_bytes(pb, n_pos_total, n_batch, flags, minimum=True))
    ws = torch.empty(n, dtype=torch.uint8, device="cuda")
    ws[:256].zero_()
    return ws


def forward_loss(pb: Problem, obj, probe, positions, intensity=None, batch_idx=None, *, workspace, loss=None,
                 loss_per_pos=None, model_intensity=None, flags: int = 0):
    """ptycho_forward_loss. All tensors are CUDA; outputs are written in place (pass the ones you want)."""
    import torch
    obj = _dev(obj, torch.complex64, "obj"); probe = _dev(probe, torch.complex64, "probe")
    positions = _dev(positions, torch.float32, "positions"); intensity = _dev(intensity, torch.float32, "intensity")
    batch_idx = _dev(batch_idx, torch.int32, "batch_idx")
    npos = positions.shape[0]; J = npos if batch_idx is None else batch_idx.numel()
    cs = pb.c_struct(npos, J, flags)
    _check(lib().ptycho_forward_loss(C.byref(cs), _ptr(obj), _ptr(probe), _ptr(positions), _ptr(intensity), _ptr(batch_idx),
                                     _ptr(_dev(loss, torch.float64, "loss")), _ptr(_dev(loss_per_pos, torch.float32, "loss_per_pos")),
                                     _ptr(_dev(model_intensity, torch.float32, "model_intensity")), _ptr(workspace),
                                     C.c_size_t(workspace.numel()), _stream()))


def gradient(pb: Problem, obj, probe, positions, intensity, batch_idx=None, *, workspace, grad_object, grad_probe,
             grad_pos=None, illum=None, illum_prev=None, step_terms=None, loss=None, loss_per_pos=None, flags: int = 0):
    """ptycho_gradient. flags |= WANT_* is derived from which outputs are given."""
    import torch
    obj = _dev(obj, torch.complex64, "obj"); probe = _dev(probe, torch.complex64, "probe")
    positions = _dev(positions, torch.float32, "positions"); intensity = _dev(intensity, torch.float32, "intensity")
    batch_idx = _dev(batch_idx, torch.int32, "batch_idx")
    npos = positions.shape[0]; J = npos if batch_idx is None else batch_idx.numel()
    if grad_pos is not None: flags |= WANT_POS_GRAD
    if illum is not None: flags |= WANT_ILLUM
    if step_terms is not None: flags |= WANT_STEP_SIZES
    cs = pb.c_struct(npos, J, flags)
    _check(lib().ptycho_gradient(C.byref(cs), _ptr(obj), _ptr(probe), _ptr(positions), _ptr(intensity), _ptr(batch_idx),
                                 _ptr(_dev(grad_object, torch.complex64, "grad_object")), _ptr(_dev(grad_probe, torch.complex64, "grad_probe")),
                                 _ptr(_dev(grad_pos, torch.float32, "grad_pos")), _ptr(_dev(illum, torch.float32, "illum")),
                                 _ptr(_dev(illum_prev, torch.float32, "illum_prev")), _ptr(_dev(step_terms, torch.float32, "step_terms")),
                                 _ptr(_dev(loss, torch.float64, "loss")), _ptr(_dev(loss_per_pos, torch.float32, "loss_per_pos")),
                                 _ptr(workspace), C.c_size_t(workspace.numel()), _stream()))


def apply_update(pb: Problem, obj=None, probe=None, positions=None, *, grad_object=None, grad_probe=None, grad_pos=None,
                 illum_prev=None, step_terms=None, batch_idx=None, n_batch: Optional[int] = None, mode=UPDATE_SGD,
                 lr_obj=0.0, lr_probe=0.0, lr_pos=0.0, beta_obj=1.0, beta_probe=1.0, gamma=0.0, workspace=None, illum_batch=None, flags: int = 0):
    """ptycho_apply_update (in place). illum_batch: the [2][S][ny][nx] (I, W) planes of WANT_WEIGHTED_ILLUM (UPDATE_LSQML_WEIGHTED)."""
    import torch
    npos = positions.shape[0] if positions is not None else (n_batch or 1)
    J = batch_idx.numel() if batch_idx is not None else (n_batch if n_batch is not None else npos)
    cs = pb.c_struct(max(npos, J), J, flags)
    ib = _dev(illum_batch, torch.float32, "illum_batch")
    u = PtUpdate(mode, lr_obj, lr_probe, lr_pos, beta_obj, beta_probe, gamma, None if ib is None else ib.data_ptr())
    _check(lib().ptycho_apply_update(C.byref(cs), _ptr(_dev(obj, torch.complex64, "obj")), _ptr(_dev(probe, torch.complex64, "probe")),
                                     _ptr(_dev(positions, torch.float32, "positions")), _ptr(_dev(grad_object, torch.complex64, "grad_object")),
                                     _ptr(_dev(grad_probe, torch.complex64, "grad_probe")), _ptr(_dev(grad_pos, torch.float32, "grad_pos")),
                                     _ptr(_dev(illum_prev, torch.float32, "illum_prev")), _ptr(_dev(step_terms, torch.float32, "step_terms")),
                                     _ptr(_dev(batch_idx, torch.int32, "batch_idx")), C.byref(u), _ptr(workspace),
                                     C.c_size_t(0 if workspace is None else workspace.numel()), _stream()))


def object_transparency(pb: Problem, obj, positions, batch_idx=None, *, out, workspace, flags: int = 0):
    """ptycho_object_transparency: out [N][N] float32 <- sum_j prod_i |O_i|^2 in the probe view."""
    import torch
    obj = _dev(obj, torch.complex64, "obj"); positions = _dev(positions, torch.float32, "positions")
    batch_idx = _dev(batch_idx, torch.int32, "batch_idx")
    npos = positions.shape[0]; J = npos if batch_idx is None else batch_idx.numel()
    cs = pb.c_struct(npos, J, flags)
    _check(lib().ptycho_object_transparency(C.byref(cs), _ptr(obj), _ptr(positions), _ptr(batch_idx), _ptr(_dev(out, torch.float32, "out")),
                                            _ptr(workspace), C.c_size_t(workspace.numel()), _stream()))


def gradient_host(pb: Problem, obj_h, probe_h, positions_h, intensity_h, batch_idx_h=None, *, workspace, grad_object_h,
                  grad_probe_h, grad_pos_h=None, loss_h=None, loss_per_pos_h=None):
    """ptycho_gradient_host: HOST (pinned) tensors in and out, copies inside the call, synchronises."""
    npos = positions_h.shape[0]; J = npos if batch_idx_h is None else batch_idx_h.numel()
    cs = pb.c_struct(npos, J, 0)
    for t in (obj_h, probe_h, positions_h, intensity_h, grad_object_h, grad_probe_h):
        if t.is_cuda or not t.is_contiguous():
            raise TypeError("gradient_host expects contiguous host tensors")
    _check(lib().ptycho_gradient_host(C.byref(cs), _ptr(obj_h), _ptr(probe_h), _ptr(positions_h), _ptr(intensity_h),
                                      _ptr(batch_idx_h), _ptr(grad_object_h), _ptr(grad_probe_h), _ptr(grad_pos_h), _ptr(loss_h),
                                      _ptr(loss_per_pos_h), _ptr(workspace), C.c_size_t(workspace.numel()), _stream()))


def status(workspace) -> int:
    """ptycho_status: synchronise and return (then clear) the deferred device status."""
    return int(lib().ptycho_status(_ptr(workspace), _stream()))


def launch_count() -> int:
    return int(lib().ptycho_launch_count())


def profile_enable(on: bool = True) -> None:
    _check(lib().ptycho_profile_enable(1 if on else 0))


def profile_read() -> dict:
    """ptycho_profile_read: {kernel name: (summed device ms, launches)} since profile_enable / the last read."""
    n = int(lib().ptycho_profile_num_kernels())
    ms = (C.c_float * n)(); cnt = (C.c_int64 * n)()
    _check(lib().ptycho_profile_read(ms, cnt))
    return {lib().ptycho_profile_kernel_name(i).decode(): (float(ms[i]), int(cnt[i])) for i in range(n) if cnt[i]}


def profile_fp32_peak(workspace) -> float:
    """ptycho_profile_fp32_peak: measured FP32 FMA throughput of the current device, TFLOP/s."""
    v = C.c_double(0.0)
    f = lib().ptycho_profile_fp32_peak
    f.restype = C.c_int32
    _check(f(C.byref(v), _ptr(workspace), _stream()))
    return float(v.value)


# ---- cost / constraint regularisers and Adam (include/ptycho.h) -----------------------------------
REG_L2, REG_L1, REG_TIKHONOV, REG_TV, REG_LAYER_TIKHONOV, REG_LAYER_TV, REG_L1_PHASE, REG_L1_FOURIER = range(8)
CON_AMPLITUDE_CLAMP, CON_SUPPORT_MASK, CON_LAYER_BLUR, CON_LOWPASS, CON_SUPPORT_MASK_FOURIER, CON_PHASE_DERAMP = range(6)


def _field3(t, name):
    import torch
    t = _dev(t, torch.complex64, name)
    if t.dim() != 3:
        raise TypeError(f"{name}: expected a [n_slices][ny][nx] tensor")
    return t


def regularizer_workspace_bytes() -> int:
    f = lib().ptycho_regularizer_workspace_bytes
    f.restype = C.c_size_t
    return int(f())


def cost_regularizer(kind: int, weight: float, field_, *, grad=None, cost=None, ref: float = 1.0, eps: float = 0.0, workspace):
    """ptycho_cost_regularizer: grad += weight dR/dconj(field), cost[0] += R (both optional, in place)."""
    import torch
    z = _field3(field_, "field")
    S, ny, nx = z.shape
    f = lib().ptycho_cost_regularizer
    f.restype = C.c_int32
    _check(f(int(kind), C.c_float(weight), C.c_float(ref), C.c_float(eps), S, ny, nx, _ptr(z), _ptr(_dev(grad, torch.complex64, "grad")),
             _ptr(_dev(cost, torch.float64, "cost")), _ptr(workspace), C.c_size_t(workspace.numel()), _stream()))


def apply_constraint(kind: int, field_, *, a: float = 0.0, b: float = 0.0, mask=None, workspace=None):
    """ptycho_apply_constraint (in place)."""
    import torch
    z = _field3(field_, "field")
    S, ny, nx = z.shape
    f = lib().ptycho_apply_constraint
    f.restype = C.c_int32
    _check(f(int(kind), C.c_float(a), C.c_float(b), _ptr(_dev(mask, torch.float32, "mask")), S, ny, nx, _ptr(z), _ptr(workspace),
             C.c_size_t(0 if workspace is None else workspace.numel()), _stream()))


STATIC_SCRATCH_BYTES = 16 << 20                                       # PT_STATIC_SCRATCH_BYTES
ERR_UNSUPPORTED, ERR_STATIC_LIMIT = -8, -9


def apply_constraint_static(kind: int, field_, *, a: float = 0.0):
    """ptycho_apply_constraint_static (in place): layer blur / low pass / phase deramp with the library's own static device
    scratch; allocates nothing, fields beyond STATIC_SCRATCH_BYTES of scratch raise PtychoError(ERR_STATIC_LIMIT)."""
    z = _field3(field_, "field")
    S, ny, nx = z.shape
    f = lib().ptycho_apply_constraint_static
    f.restype = C.c_int32
    _check(f(int(kind), C.c_float(a), S, ny, nx, _ptr(z), _stream()))


def adam_update(z, g, m, v, *, lr: float, beta1: float = 0.9, beta2: float = 0.999, eps: float = 1e-8, step: int = 1):
    """ptycho_adam_update (complex64 z, g, m; float32 v) or ptycho_adam_update_real (all float32); in place."""
    import torch
    cplx = z.dtype == torch.complex64
    ty = torch.complex64 if cplx else torch.float32
    z = _dev(z, ty, "z"); g = _dev(g, ty, "g"); m = _dev(m, ty, "m"); v = _dev(v, torch.float32, "v")
    if not (g.numel() == z.numel() == m.numel() == v.numel()):
        raise TypeError("adam_update: z, g, m, v must have the same number of elements")
    f = lib().ptycho_adam_update if cplx else lib().ptycho_adam_update_real
    f.restype = C.c_int32
    _check(f(_ptr(z), _ptr(g), _ptr(m), _ptr(v), C.c_size_t(z.numel()), C.c_float(lr), C.c_float(beta1), C.c_float(beta2),
             C.c_float(eps), int(step), _stream()))
