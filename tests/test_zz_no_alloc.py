"""ptycho_apply_constraint_static (include/ptycho.h): the blur / low-pass / deramp constraints with their scratch in the
library's own static device array, for callers that cannot allocate device memory.  Checked against the existing
ptycho_apply_constraint (caller-owned workspace) on two calls in a row that share the array — the second on a smaller field,
so the array still holds the first call's values wherever the second does not write — plus the size limit and that the call
leaves the device's free memory where it was.  This file sorts last on purpose (the suite runs with pytest -x)."""
import numpy as np
import pytest


pytestmark = pytest.mark.gpu

TOL = 1e-6          # the bar tests/test_gpu_parity.py::test_constraints uses for these kernels (relative L2)


def _field(shape, seed):
    """object-like transmission function: unit-ish amplitude, smooth phase plus noise, and an affine ramp for the deramp"""
    rng = np.random.default_rng(seed)
    S, ny, nx = shape
    yy, xx = np.meshgrid(np.arange(ny), np.arange(nx), indexing="ij")
    ph = 0.4 * np.sin(2 * np.pi * yy / 37.0)[None] * np.cos(2 * np.pi * xx / 23.0)[None] + 0.1 * rng.standard_normal(shape)
    ph = ph + (0.013 * yy - 0.021 * xx)[None] + 0.3 * np.arange(S)[:, None, None]
    amp = 1.0 + 0.05 * rng.standard_normal(shape)
    return (amp * np.exp(1j * ph)).astype(np.complex64)


def _both(kind, z, a):
    """(existing path with a torch-owned workspace, static-scratch entry point) on copies of the same field"""
    import torch
    from paper_2505_14372_b200 import ptycho
    ws = torch.empty(max(z.size * 8, 256 + z.shape[0] * 2080), dtype=torch.uint8, device="cuda")
    ref = torch.from_numpy(z).cuda()
    ptycho.apply_constraint(kind, ref, a=a, workspace=ws)
    got = torch.from_numpy(z).cuda()
    torch.cuda.synchronize()
    free0 = torch.cuda.mem_get_info()[0]
    ptycho.apply_constraint_static(kind, got, a=a)
    torch.cuda.synchronize()
    free1 = torch.cuda.mem_get_info()[0]
    return ref.cpu().numpy(), got.cpu().numpy(), free0, free1


def test_static_scratch_constraints_match_workspace_path_twice_in_a_row():
    import torch
    from paper_2505_14372_b200 import ptycho
    from tests._cases import rel_l2
    assert torch.cuda.is_available(), "needs the GPU"
    big, small = _field((5, 301, 333), 11), _field((3, 150, 97), 12)      # ragged sizes, several blocks; 4.0 MB then 0.35 MB of scratch
    calls = 0
    for kind, a in ((ptycho.CON_LOWPASS, 1.3), (ptycho.CON_LAYER_BLUR, 0.9), (ptycho.CON_PHASE_DERAMP, 0.0)):
        for n_call, z in enumerate((big, small, big)):                     # back to back on the shared array, stale contents in between
            ref, got, free0, free1 = _both(kind, z, a)
            assert np.isfinite(got.view(np.float32)).all()
            assert rel_l2(got, ref) <= TOL, (kind, n_call, rel_l2(got, ref))
            assert np.abs(got - ref).max() <= TOL * np.abs(ref).max()
            assert rel_l2(got, z) > 1e-3                                   # the constraint did something
            if calls > 0:                                                  # the first call may load the module's kernels lazily
                assert free1 == free0, "device free memory changed across the call"
            calls += 1


def test_static_scratch_limit_and_kinds():
    import torch
    from paper_2505_14372_b200 import ptycho
    n_max = ptycho.STATIC_SCRATCH_BYTES // 8
    too_big = torch.ones((1, 1449, 1449), dtype=torch.complex64, device="cuda")        # 2 099 601 > 2 097 152 complex pixels
    assert too_big.numel() > n_max
    with pytest.raises(ptycho.PtychoError) as e:
        ptycho.apply_constraint_static(ptycho.CON_LOWPASS, too_big, a=1.0)
    assert e.value.code == ptycho.ERR_STATIC_LIMIT and "static" in str(e.value)
    assert bool((too_big == 1).all())                                      # rejected before any launch
    at_limit = torch.ones((8, 512, 512), dtype=torch.complex64, device="cuda")         # exactly the limit: accepted
    assert at_limit.numel() == n_max
    ptycho.apply_constraint_static(ptycho.CON_LOWPASS, at_limit, a=1.0)
    torch.cuda.synchronize()
    assert torch.allclose(at_limit, torch.ones_like(at_limit), atol=1e-6)  # a normalised blur keeps a constant field
    many = torch.ones((9000, 2, 2), dtype=torch.complex64, device="cuda")  # deramp scratch grows with the slice count
    with pytest.raises(ptycho.PtychoError) as e:
        ptycho.apply_constraint_static(ptycho.CON_PHASE_DERAMP, many)
    assert e.value.code == ptycho.ERR_STATIC_LIMIT
    for kind in (ptycho.CON_AMPLITUDE_CLAMP, ptycho.CON_SUPPORT_MASK, ptycho.CON_SUPPORT_MASK_FOURIER):
        with pytest.raises(ptycho.PtychoError) as e:
            ptycho.apply_constraint_static(kind, too_big[:, :64, :64].contiguous(), a=1.0)
        assert e.value.code == ptycho.ERR_UNSUPPORTED
    with pytest.raises(ptycho.PtychoError):
        ptycho.apply_constraint_static(ptycho.CON_LOWPASS, at_limit, a=9.0)            # sigma beyond the 65-tap table
