"""CPU-side checks of the product: the C-ABI library builds, loads and exports every symbol include/ptycho.h
declares; host-side argument validation and workspace sizing (no kernel is launched, no GPU needed); the index
maps / exchange slots / in-register DFTs of the register-resident FFT, emulated thread by thread on the host by
tests/host_harness (a test harness around the device header, not a product path) against numpy.fft.
"""
import ctypes as C
import os
import re
import subprocess

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_2505_14372_b200 import ptycho
    ptycho.build()
    return ptycho.lib()


def declared_functions():
    src = open(os.path.join(ROOT, "include", "ptycho.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(ptycho_[a-z_0-9]+)\s*\(", src)))


def test_library_exports_every_declared_symbol(lib):
    names = declared_functions()
    assert {"ptycho_forward_loss", "ptycho_gradient", "ptycho_apply_update"} <= set(names)
    for n in names:
        assert hasattr(lib, n), n
    from paper_2505_14372_b200 import ptycho
    assert sorted(ptycho.EXPORTS) == names


def test_struct_layout_matches_header(lib):
    # pt_problem as the binding marshals it must have the header's field order; sizes on LP64
    from paper_2505_14372_b200 import ptycho
    hdr = open(os.path.join(ROOT, "include", "ptycho.h")).read()
    body = hdr[:hdr.index("} pt_problem;")]
    body = body[body.rindex("typedef struct {") + len("typedef struct {"):]
    body = re.sub(r"/\*.*?\*/", "", body, flags=re.S)
    fields = []
    for decl in body.split(";"):
        decl = decl.strip()
        if not decl:
            continue
        names = decl.replace("*", " ").split()
        first = [n for n in names if n not in ("const", "int32_t", "float")]
        fields += [f.strip(",") for f in first]
    assert fields == [f[0] for f in ptycho.PtProblem._fields_]
    assert C.sizeof(ptycho.PtProblem) == 104
    # pt_update: seven 4-byte scalars, then the device pointer of PT_UPDATE_LSQML_WEIGHTED (8-byte aligned)
    ub = hdr[:hdr.index("} pt_update;")]
    ub = re.sub(r"/\*.*?\*/", "", ub[ub.rindex("typedef struct {") + len("typedef struct {"):], flags=re.S)
    unames = [n.strip(",") for d in ub.split(";") for n in d.replace("*", " ").split() if n not in ("const", "int32_t", "float")]
    assert unames == [f[0] for f in ptycho.PtUpdate._fields_]
    assert C.sizeof(ptycho.PtUpdate) == 40 and ptycho.PtUpdate.illum_batch_d.offset == 32


def test_validation_and_workspace_sizes(lib):
    import dataclasses
    from paper_2505_14372_b200 import ptycho
    pb = ptycho.Problem(n=128, n_modes=8, n_slices=20, obj_ny=420, obj_nx=420, pixel_size=0.1, wavelength=0.0197,
                        slice_thickness=[10.0] * 20, loss=ptycho.LOSS_POISSON, eps=0.8)
    lo = ptycho.workspace_bytes(pb, 4096, 64, minimum=True)
    hi = ptycho.workspace_bytes(pb, 4096, 64)
    assert 0 < lo < hi
    # per-position scratch is dominated by the stash (M fields per slice) + the staged patch gradients (M/2 per slice: the
    # backward pass sums pairs of modes on chip): 1.5 * M * S * N^2 * 8 bytes
    per_pos = (hi - lo) / 63
    assert 1.5 * 8 * 20 * 128 * 128 * 8 <= per_pos <= 1.1 * 1.5 * 8 * 20 * 128 * 128 * 8
    odd = dataclasses.replace(pb, n_modes=7)                       # odd mode count: one mode per CTA, M planes staged
    per_pos_odd = (ptycho.workspace_bytes(odd, 4096, 64) - ptycho.workspace_bytes(odd, 4096, 64, minimum=True)) / 63
    assert 2 * 7 * 20 * 128 * 128 * 8 <= per_pos_odd <= 1.1 * 2 * 7 * 20 * 128 * 128 * 8
    big = ptycho.workspace_bytes(pb, 4096, 4096)
    assert big <= (49 << 30) + (1 << 20)                          # chunked: capped recommendation
    for bad in (dict(n=100), dict(n_modes=0), dict(obj_ny=100)):
        with pytest.raises(ptycho.PtychoError):
            ptycho.workspace_bytes(dataclasses.replace(pb, **bad), 64, 64)
    # argument errors are reported before anything touches the device
    cs = pb.c_struct(64, 64, 0)
    rc = lib.ptycho_forward_loss(C.byref(cs), None, None, None, None, None, None, None, None, None, C.c_size_t(0), None)
    assert rc == -1 and lib.ptycho_strerror(rc).decode() == "null pointer"
    cs = dataclasses.replace(pb, eps=0.0).c_struct(64, 64, 0)
    assert lib.ptycho_gradient(C.byref(cs), *([None] * 15), C.c_size_t(0), None) == -3
    cs = dataclasses.replace(pb, shift_mode=7).c_struct(64, 64, 0)
    assert lib.ptycho_gradient(C.byref(cs), *([None] * 15), C.c_size_t(0), None) == -3


def test_binding_refuses_cpu_tensors(lib):
    import torch
    from paper_2505_14372_b200 import ptycho
    pb = ptycho.Problem(n=64, n_modes=1, n_slices=1, obj_ny=128, obj_nx=128)
    z = torch.zeros((1, 128, 128), dtype=torch.complex64)
    with pytest.raises(TypeError):
        ptycho.forward_loss(pb, z, z, torch.zeros((4, 2)), None, workspace=torch.zeros(1 << 20, dtype=torch.uint8))


@pytest.mark.parametrize("n", [64, 128])
def test_register_fft_layout_on_host(tmp_path, n):
    exe = tmp_path / "harness"
    src = os.path.join(ROOT, "tests", "host_harness", "fft_layout_harness.cu")
    subprocess.run(["nvcc", "-O1", "-std=c++17", "-Wno-deprecated-gpu-targets", "-o", str(exe), src], check=True)
    rng = np.random.default_rng(n)
    a = (rng.standard_normal((n, n)) + 1j * rng.standard_normal((n, n))).astype(np.complex64)
    fin, ffwd, frt = tmp_path / "in.bin", tmp_path / "fwd.bin", tmp_path / "rt.bin"
    a.tofile(fin)
    rc = subprocess.run([str(exe), str(n), str(fin), str(ffwd), str(frt)], capture_output=True, text=True)
    assert rc.returncode == 0, rc.stdout
    fwd = np.fromfile(ffwd, np.complex64).reshape(n, n)
    rt = np.fromfile(frt, np.complex64).reshape(n, n)
    ref = np.fft.fft2(a.astype(np.complex128))
    assert np.linalg.norm(fwd - ref) / np.linalg.norm(ref) < 5e-7
    assert np.linalg.norm(rt / (n * n) - a) / np.linalg.norm(a) < 1e-6
