"""Pins for the CPU oracle (oracle/ptycho_oracle.cpp) against what the paper and the mathematics fix.

None of these call the CUDA path.  Each test names the passage (PAPER.md line / DESIGN.md reading) it pins.
The paper prints no numeric worked example, so the pins are closed forms, invariants,
library routines on special cases (numpy.fft), brute force on tiny inputs, central finite differences and
an autograd (torch, complex128) re-derivation of the adjoint.
"""
import numpy as np
import pytest

from oracle import oracle as orc

RNG = np.random.default_rng(12345)


def crandn(*shape):
    return RNG.standard_normal(shape) + 1j * RNG.standard_normal(shape)


# ------------------------------------------------------------------------------------------------
# FFT (O0, O2, O3, O5)  — definitions block of DESIGN.md §2
# ------------------------------------------------------------------------------------------------
def test_dft_bruteforce_8x8():
    a = crandn(8, 8)
    ref = orc.dft2_bruteforce(a, -1)           # direct O(N^4) double sum
    assert np.abs(orc.fft2(a, -1) - ref).max() < 1e-12
    assert np.abs(orc.dft2_naive(a, -1) - ref).max() < 1e-12
    # sign convention: forward kernel exp(-2 pi i q r / N) == numpy.fft.fft2
    assert np.abs(ref - np.fft.fft2(a)).max() < 1e-12
    assert np.abs(orc.dft2_bruteforce(a, +1) - np.fft.ifft2(a) * 64).max() < 1e-12


def test_fft_inverse_parseval_delta():
    for n in (8, 64):
        a = crandn(n, n)
        A = orc.fft2(a, -1)
        assert np.abs(orc.fft2(A, +1) / n ** 2 - a).max() < 1e-12            # Finv F = id
        assert abs(np.sum(np.abs(A) ** 2) - n ** 2 * np.sum(np.abs(a) ** 2)) < 1e-9 * n ** 2 * np.sum(np.abs(a) ** 2)
        d = np.zeros((n, n), complex); d[0, 0] = 1.0
        assert np.abs(orc.fft2(d, -1) - 1.0).max() < 1e-13                   # delta <-> constant
        d = np.zeros((n, n), complex); d[3, 5] = 1.0                         # shifted delta <-> plane wave
        qy, qx = np.meshgrid(np.arange(n), np.arange(n), indexing="ij")
        assert np.abs(orc.fft2(d, -1) - np.exp(-2j * np.pi * (3 * qy + 5 * qx) / n)).max() < 1e-12


def test_recursive_fft_vs_naive_dft_64_and_128():
    for n in (64, 128):
        a = crandn(n, n)
        assert np.abs(orc.fft2(a, -1) - orc.dft2_naive(a, -1)).max() < 1e-9
        assert np.abs(orc.fft2(a, -1) - np.fft.fft2(a)).max() < 1e-9


# ------------------------------------------------------------------------------------------------
# position split (O1, reading R2)
# ------------------------------------------------------------------------------------------------
def test_position_split():
    # p = X/px, c = p - N/2, r0 = floor(c + 1/2), delta = c - r0 in [-1/2, 1/2)
    assert orc.position_split(40.0, 1.0, 64) == (8, 0.0)
    r0, d = orc.position_split(40.25, 1.0, 64); assert r0 == 8 and abs(d - 0.25) < 1e-7
    r0, d = orc.position_split(40.5, 1.0, 64); assert r0 == 9 and abs(d + 0.5) < 1e-7     # round half up
    r0, d = orc.position_split(40.75, 1.0, 64); assert r0 == 9 and abs(d + 0.25) < 1e-7
    r0, d = orc.position_split(4.06, 0.1, 64); assert r0 == 9 and abs(d - (-0.4)) < 1e-5
    for X in RNG.uniform(10, 40, 200):
        r0, d = orc.position_split(float(np.float32(X)), 0.1, 128)
        assert -0.5 <= d < 0.5
        assert abs((r0 + d) - (np.float32(X) / np.float32(0.1) - 64)) < 1e-4


# ------------------------------------------------------------------------------------------------
# sub-pixel shift (O1, O2; PAPER.md:115 P_k(r - X_j))
# ------------------------------------------------------------------------------------------------
def test_shift_integer_is_roll_and_inverse():
    a = crandn(16, 16)
    # delta = +1 moves content to the next higher index: out[r] = in[r - delta]
    assert np.abs(orc.shift(a, 1.0, 0.0) - np.roll(a, 1, axis=0)).max() < 1e-12
    assert np.abs(orc.shift(a, 0.0, -3.0) - np.roll(a, -3, axis=1)).max() < 1e-12
    b = orc.shift(orc.shift(a, 0.3, -0.2), -0.3, 0.2)
    assert np.abs(b - a).max() < 1e-12
    s = orc.shift(a, 0.37, 0.11)
    assert abs(np.sum(np.abs(s) ** 2) - np.sum(np.abs(a) ** 2)) < 1e-10
    # band-limited signal: shift equals evaluating the trigonometric interpolant
    n = 16; y, x = np.meshgrid(np.arange(n), np.arange(n), indexing="ij")
    f = lambda yy, xx: np.exp(2j * np.pi * (2 * yy - 3 * xx) / n) + 0.5 * np.exp(2j * np.pi * (-5 * yy + 1 * xx) / n)
    assert np.abs(orc.shift(f(y, x), 0.3, -0.45) - f(y - 0.3, x + 0.45)).max() < 1e-12


# ------------------------------------------------------------------------------------------------
# propagator (O3, O4; readings R7, R8, R9)
# ------------------------------------------------------------------------------------------------
def test_propagator_identity_composition_unit_modulus():
    a = crandn(16, 16)
    assert np.abs(orc.propagate(a, 0.1, 0.0197, 0.0, 0.8, 0.6) - a).max() < 1e-12         # dz = 0 -> identity
    H1 = orc.propagator(16, 0.1, 0.0197, 7.0, 0.8, 0.6)
    H2 = orc.propagator(16, 0.1, 0.0197, 5.0, 0.8, 0.6)
    H3 = orc.propagator(16, 0.1, 0.0197, 12.0, 0.8, 0.6)
    assert np.abs(H1 * H2 - H3).max() < 1e-12                                             # H(a)H(b) = H(a+b)
    assert np.abs(np.abs(H1) - 1.0).max() < 1e-14                                         # |H| = 1 without mask
    b = orc.propagate(a, 0.1, 0.0197, 9.0, 0.8, 0.6)
    assert abs(np.sum(np.abs(b) ** 2) - np.sum(np.abs(a) ** 2)) < 1e-10


def test_propagator_tilt_integer_shift_sign():
    # R8: exp(+2 pi i dz (kx tan tx + ky tan ty)); with dz*tan(theta)/px = +m px the field moves by -m px.
    n, px = 16, 0.1
    a = crandn(n, n)
    dz = 100.0
    tx_mrad = np.arctan(2 * px / dz) * 1e3         # dz tan(tx) = +2 px
    ty_mrad = np.arctan(-3 * px / dz) * 1e3        # dz tan(ty) = -3 px
    # lambda = 0 removes the Fresnel term, leaving the pure tilt
    out = orc.propagate(a, px, 0.0, dz, tx_mrad, ty_mrad)
    assert np.abs(out - np.roll(np.roll(a, -2, axis=1), +3, axis=0)).max() < 1e-10


def test_propagator_gaussian_closed_form():
    # Fresnel sign/units (R7): H = exp(-i pi lambda dz k^2), k in cycles/Angstrom.  A Gaussian
    # exp(-r^2/(2 s^2)) propagates to (s^2/s'^2) exp(-r^2/(2 s'^2)) with s'^2 = s^2 + i lambda dz/(2 pi).
    n, px, lam, dz, s = 128, 0.1, 0.0197, 40.0, 0.5
    r = (np.arange(n) - n // 2) * px
    Y, X = np.meshgrid(r, r, indexing="ij")
    g = np.exp(-(X ** 2 + Y ** 2) / (2 * s ** 2))
    s2 = s ** 2 + 1j * lam * dz / (2 * np.pi)
    ref = (s ** 2 / s2) * np.exp(-(X ** 2 + Y ** 2) / (2 * s2))
    out = orc.propagate(g, px, lam, dz)
    assert np.abs(out - ref).max() < 1e-8


def test_bandlimit_mask():
    n = 32
    H = orc.propagator(n, 0.1, 0.0197, 10.0, 0.0, 0.0, 2.0 / 3.0)
    s = np.where(np.arange(n) < n // 2, np.arange(n), np.arange(n) - n)
    QY, QX = np.meshgrid(s, s, indexing="ij")
    inside = (QY ** 2 + QX ** 2) <= (0.5 * (2.0 / 3.0) * n) ** 2
    assert np.all(np.abs(np.abs(H) - inside) < 1e-14)
    assert 0 < inside.sum() < n * n


# ------------------------------------------------------------------------------------------------
# whole forward (O1..O5; readings R5, R6, R10)
# ------------------------------------------------------------------------------------------------
def small_problem(n=8, M=2, S=3, on=20, J=3, loss=orc.LOSS_POISSON, eps=0.3, bandlimit=0.0, c=0.0, tilt=(30.0, -20.0)):
    pb = orc.Problem(n=n, n_modes=M, n_slices=S, obj_ny=on, obj_nx=on + 2, pixel_size=0.2, wavelength=0.05,
                     slice_thickness=[3.0 + 0.5 * i for i in range(S)], tilt_x_mrad=tilt[0], tilt_y_mrad=tilt[1],
                     bandlimit=bandlimit, loss=loss, loss_c=c, eps=eps)
    obj = (np.exp(0.3 * crandn(S, on, on + 2))).astype(np.complex64)
    probe = crandn(M, n, n).astype(np.complex64)
    pos_px = RNG.uniform(n / 2 + 1.0, on - n / 2 - 1.0, size=(J, 2))
    pos = (pos_px * 0.2).astype(np.float32)
    return pb, obj, probe, pos


def test_forward_vacuum_invariant():
    # O == 1: every pattern equals sum_k |F(P_k)|^2 / N^2, for any S, dz, tilt, positions
    pb, obj, probe, pos = small_problem(n=16, M=3, S=4, on=40, J=5)
    obj[:] = 1.0
    out = orc.forward_loss(pb, obj, probe, pos)
    ref = sum(np.abs(np.fft.fft2(probe[k].astype(complex))) ** 2 for k in range(3)) / 16 ** 2
    for j in range(5):
        assert np.abs(out["intensity"][j] - ref).max() < 1e-10 * ref.max()


def test_forward_spoa_single_slice_matches_numpy():
    # S = 1 reduces to |F(P_shift . O_patch)|^2 / N^2 (SPOA; BASELINE.json config 1)
    n, on = 16, 40
    pb, obj, probe, pos = small_problem(n=n, M=2, S=1, on=on, J=4)
    out = orc.forward_loss(pb, obj, probe, pos)
    s = np.where(np.arange(n) < n // 2, np.arange(n), np.arange(n) - n) / n
    for j in range(4):
        c = pos[j].astype(np.float64) / 0.2 - n / 2          # exact here: compare r0/delta to the fp32 split
        r0 = np.floor(c + 0.5).astype(int); d = c - r0
        r0y, dy = orc.position_split(float(pos[j, 0]), 0.2, n); r0x, dx = orc.position_split(float(pos[j, 1]), 0.2, n)
        assert (r0y, r0x) == (r0[0], r0[1]) and abs(dy - d[0]) < 1e-5 and abs(dx - d[1]) < 1e-5
        R = np.exp(-2j * np.pi * (s[:, None] * dy + s[None, :] * dx))
        I = np.zeros((n, n))
        for k in range(2):
            Ps = np.fft.ifft2(R * np.fft.fft2(probe[k].astype(complex)))
            patch = obj[0, r0y:r0y + n, r0x:r0x + n].astype(complex)
            I += np.abs(np.fft.fft2(Ps * patch)) ** 2 / n ** 2
        assert np.abs(out["intensity"][j] - I).max() < 1e-10 * I.max()
        # electron count (Parseval, reading R5)
        assert abs(out["intensity"][j].sum() - sum(np.sum(np.abs(np.fft.ifft2(R * np.fft.fft2(probe[k].astype(complex))) * patch) ** 2) for k in range(2))) < 1e-9 * I.sum()


def test_forward_phase_ramp_object_shifts_pattern():
    # integer-linear phase ramp exp(2 pi i a.r/N) at S = 1 circularly shifts the pattern by a
    n, on = 16, 40
    pb, obj, probe, pos = small_problem(n=n, M=1, S=1, on=on, J=2)
    y, x = np.meshgrid(np.arange(on), np.arange(on + 2), indexing="ij")
    obj0 = np.ones_like(obj)
    obj1 = np.exp(2j * np.pi * (3 * y - 2 * x) / n)[None].astype(np.complex64)
    I0 = orc.forward_loss(pb, obj0, probe, pos)["intensity"]
    I1 = orc.forward_loss(pb, obj1, probe, pos)["intensity"]
    for j in range(2):
        assert np.abs(I1[j] - np.roll(np.roll(I0[j], 3, axis=0), -2, axis=1)).max() < 1e-5 * I0[j].max()


def test_forward_translation_covariance_and_scaling_ambiguity():
    pb, obj, probe, pos = small_problem(n=8, M=2, S=3, on=24, J=3)
    pos = np.clip(pos, (8 / 2 + 1) * 0.2, (24 - 8 / 2 - 4) * 0.2).astype(np.float32)
    I0 = orc.forward_loss(pb, obj, probe, pos)["intensity"]
    obj_s = np.roll(np.roll(obj, 2, axis=1), 1, axis=2)
    pos_s = (pos.astype(np.float64) + np.array([2, 1]) * 0.2).astype(np.float32)
    I1 = orc.forward_loss(pb, obj_s, probe, pos_s)["intensity"]
    assert np.abs(I1 - I0).max() < 2e-4 * I0.max()      # fp32 positions: delta differs by ~1e-6 px
    # P -> aP, O_0 -> O_0 / a leaves I unchanged
    obj2 = obj.copy(); obj2[0] /= 2.0
    I2 = orc.forward_loss(pb, obj2, (probe * 2.0).astype(np.complex64), pos)["intensity"]
    assert np.abs(I2 - I0).max() < 1e-6 * I0.max()


# ------------------------------------------------------------------------------------------------
# loss (O6; readings R11, R12)
# ------------------------------------------------------------------------------------------------
def test_loss_closed_forms():
    # amplitude loss exactly as printed: hand-computed 2x2 example
    I = [4.0, 9.0, 1.0, 0.0]; Ie = [1.0, 16.0, 1.0, 2.0]
    tot = sum(orc.loss_pixel(orc.LOSS_AMPLITUDE, a, b, 0.0, 1e-12)[0] for a, b in zip(I, Ie))
    assert abs(tot - (0.5 + 0.5 + 0.0 + 1.0)) < 1e-12
    # Anscombe c = 3/8
    l, w = orc.loss_pixel(orc.LOSS_AMPLITUDE, 4.0 - 0.375, 9.0 - 0.375, 0.375, 1e-12)
    assert abs(l - 0.5) < 1e-12 and abs(w - 0.5 * (1 - 3.0 / 2.0)) < 1e-11
    # zero loss and weight at I = Iexp
    for kind in (0, 1):
        l, w = orc.loss_pixel(kind, 7.3, 7.3, 0.0, 1e-14)
        assert abs(l) < 1e-12 and abs(w) < 1e-12
    # Poisson: l = I where Iexp = 0; w = 1 - Iexp/(I + eps)
    l, w = orc.loss_pixel(1, 2.5, 0.0, 0.0, 0.8); assert abs(l - 2.5) < 1e-14 and abs(w - 1.0) < 1e-14
    l, w = orc.loss_pixel(1, 2.0, 3.0, 0.0, 0.5)
    assert abs(l - (2.0 - 3.0 * (np.log(2.5) - np.log(3.5) + 1.0))) < 1e-14 and abs(w - (1 - 3.0 / 2.5)) < 1e-14
    # Stirling form vs exact Poisson NLL: difference is 0.5 log(2 pi Iexp) + O(1/Iexp)
    from math import lgamma
    Ie, I = 400.0, 380.0
    exact = I - Ie * np.log(I) + lgamma(Ie + 1)
    l, _ = orc.loss_pixel(1, I, Ie, 0.0, 0.0)
    assert abs((exact - l) - 0.5 * np.log(2 * np.pi * Ie)) < 1e-3
    # w is the derivative of l (both losses), convexity in I
    for kind, eps in ((0, 1e-12), (1, 0.8)):
        for I0 in (0.7, 3.0, 50.0):
            h = 1e-6
            lp, _ = orc.loss_pixel(kind, I0 + h, 5.0, 0.0, eps); lm, _ = orc.loss_pixel(kind, I0 - h, 5.0, 0.0, eps)
            l0, w0 = orc.loss_pixel(kind, I0, 5.0, 0.0, eps)
            assert abs((lp - lm) / (2 * h) - w0) < 1e-6
            lp, _ = orc.loss_pixel(kind, I0 + 0.25, 5.0, 0.0, eps); lm, _ = orc.loss_pixel(kind, I0 - 0.25, 5.0, 0.0, eps)
            assert lp + lm - 2 * l0 > 0
    # Gaussian (constant dropped): (I - Iexp)^2 / (2 sigma^2), sigma in the c slot; hand values, and the
    # printed likelihood: -log P = l + log(sigma sqrt(2 pi)) per pixel
    l, w = orc.loss_pixel(orc.LOSS_GAUSSIAN, 7.0, 4.0, 1.5, 0.3)
    assert abs(l - 9.0 / (2 * 2.25)) < 1e-14 and abs(w - 3.0 / 2.25) < 1e-14
    sig = 1.5
    nll = -np.log(np.exp(-(7.0 - 4.0) ** 2 / (2 * sig ** 2)) / (sig * np.sqrt(2 * np.pi)))
    assert abs(nll - (l + np.log(sig * np.sqrt(2 * np.pi)))) < 1e-12
    assert orc.loss_pixel(orc.LOSS_GAUSSIAN, 5.0, 5.0, 2.0, 0.3) == (0.0, 0.0)


# ------------------------------------------------------------------------------------------------
# linear adjoint pieces (O7..O11): <A x, y> = <x, A^H y>
# ------------------------------------------------------------------------------------------------
def test_adjoint_dot_products():
    n = 16
    x, y = crandn(n, n), crandn(n, n)
    assert abs(np.vdot(y, orc.shift(x, 0.3, -0.2)) - np.vdot(orc.shift(y, 0.3, -0.2, adjoint=True), x)) < 1e-11
    args = (0.1, 0.0197, 12.0, 0.8, 0.6, 2.0 / 3.0)
    assert abs(np.vdot(y, orc.propagate(x, *args)) - np.vdot(orc.propagate(y, *args, adjoint=True), x)) < 1e-11
    obj = crandn(30, 33); patch = crandn(n, n)
    acc = np.zeros((30, 33), np.complex128); orc.scatter_add(acc, 5, 9, patch)
    assert abs(np.vdot(patch, orc.gather(obj, 5, 9, n)) - np.vdot(acc, obj)) < 1e-11


def test_scatter_add_coverage_map():
    # all-ones patch gradients on an integer raster -> coverage = outer product of 1-D overlap counts
    n, on = 8, 24
    acc = np.zeros((on, on), np.complex128)
    starts = [0, 4, 8, 12, 16]
    for r0y in starts:
        for r0x in starts:
            orc.scatter_add(acc, r0y, r0x, np.ones((n, n)))
    c1 = np.zeros(on); [c1.__setitem__(slice(s, s + n), c1[s:s + n] + 1) for s in starts]
    assert np.abs(acc - np.outer(c1, c1)).max() == 0


# ------------------------------------------------------------------------------------------------
# full gradient: central finite differences (O7..O11; PAPER.md:181-185 Wirtinger convention, reading R15)
# ------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("loss,eps,bandlimit", [(orc.LOSS_POISSON, 0.3, 0.0), (orc.LOSS_POISSON, 0.3, 2.0 / 3.0),
                                                (orc.LOSS_AMPLITUDE, 1e-12, 0.0), (orc.LOSS_GAUSSIAN, 0.3, 0.0)])
def test_gradient_finite_differences(loss, eps, bandlimit):
    pb, obj, probe, pos = small_problem(loss=loss, eps=eps, bandlimit=bandlimit, c=2.0 if loss == orc.LOSS_GAUSSIAN else 0.0)
    obj_t = (obj * np.exp(0.2 * crandn(*obj.shape))).astype(np.complex64)
    Iexp = orc.forward_loss(pb, obj_t, probe, pos)["intensity"].astype(np.float32) + 0.05
    g = orc.gradient(pb, obj, probe, pos, Iexp)
    L0 = orc.forward_loss(pb, obj, probe, pos, Iexp)["loss"]
    assert abs(L0 - g["loss"]) < 1e-12 * abs(L0)

    # perturbations must be exactly representable in the float32 inputs: use h = 2^-k and work on copies
    def L(o, p):
        return orc.forward_loss(pb, o, p, pos, Iexp, want_intensity=False)["loss"]

    h = 2.0 ** -9
    for which in ("obj", "probe"):
        base = obj if which == "obj" else probe
        D = crandn(*base.shape).astype(np.complex64)
        # keep everything on the fp32 grid: z +- h*D evaluated in fp64 then cast would round; instead
        # compute in complex128 and feed the oracle complex64 casts of both, measuring the actual step
        zp = (base.astype(np.complex128) + h * D).astype(np.complex64)
        zm = (base.astype(np.complex128) - h * D).astype(np.complex64)
        Dact = (zp.astype(np.complex128) - zm.astype(np.complex128)) / 2.0
        if which == "obj":
            fd = (L(zp, probe) - L(zm, probe)) / 2.0
            lin = 2.0 * np.real(np.vdot(g["grad_object"], Dact))
        else:
            fd = (L(obj, zp) - L(obj, zm)) / 2.0
            lin = 2.0 * np.real(np.vdot(g["grad_probe"], Dact))
        assert abs(fd - lin) < 2e-4 * abs(lin) + 1e-9, (which, fd, lin)


def test_position_gradient_finite_differences():
    pb, obj, probe, pos = small_problem(J=4)
    Iexp = orc.forward_loss(pb, (obj * 1.1).astype(np.complex64), probe, pos)["intensity"].astype(np.float32) + 0.05
    # keep delta away from +-1/2 so r0 does not flip
    for j in range(4):
        for a in range(2):
            r0, d = orc.position_split(float(pos[j, a]), 0.2, 8)
            if abs(d) > 0.3:
                pos[j, a] = np.float32((r0 + 8 / 2 + 0.1 * np.sign(d)) * 0.2)
    g = orc.gradient(pb, obj, probe, pos, Iexp)
    h = 2e-3 * 0.2
    for j in range(4):
        for a in range(2):
            pp = pos.copy(); pm = pos.copy()
            pp[j, a] += np.float32(h); pm[j, a] -= np.float32(h)
            step = float(pp[j, a]) - float(pm[j, a])
            fd = (orc.forward_loss(pb, obj, probe, pp, Iexp)["loss"] - orc.forward_loss(pb, obj, probe, pm, Iexp)["loss"]) / step
            assert abs(fd - g["grad_pos"][j, a]) < 2e-3 * abs(fd) + 1e-6, (j, a, fd, g["grad_pos"][j, a])


def test_zero_gradient_at_truth_noiseless():
    # noiseless data, eps -> 0: loss and all gradients vanish at the true state (both losses)
    for loss in (orc.LOSS_POISSON, orc.LOSS_AMPLITUDE):
        pb, obj, probe, pos = small_problem(loss=loss, eps=1e-20)
        Iexp = orc.forward_loss(pb, obj, probe, pos)["intensity"]
        # fp32 storage of Iexp limits this to ~1e-7 relative
        g = orc.gradient(pb, obj, probe, pos, Iexp.astype(np.float32))
        scale = np.abs(obj).max() * np.abs(probe).max() ** 2
        assert abs(g["loss"]) < 1e-9 * Iexp.sum()
        assert np.abs(g["grad_object"]).max() < 1e-5 * scale
        assert np.abs(g["grad_probe"]).max() < 1e-5 * scale
        assert np.abs(g["grad_pos"]).max() < 1e-4 * Iexp.sum()


# ------------------------------------------------------------------------------------------------
# autograd re-derivation (torch, complex128): guards against a derivation error shared by the
# hand-written adjoints (SURVEY.md §8(c) "optional independent check")
# ------------------------------------------------------------------------------------------------
def _torch_model(pb, obj, probe, pos, Iexp, retain=False):
    import torch
    n, M, S = pb.n, pb.n_modes, pb.n_slices
    dt = torch.complex128
    O = torch.tensor(obj.astype(np.complex128), requires_grad=True)
    P = torch.tensor(probe.astype(np.complex128), requires_grad=True)
    s = torch.tensor(np.where(np.arange(n) < n // 2, np.arange(n), np.arange(n) - n) / n)
    px = float(np.float32(pb.pixel_size)); lam = float(np.float32(pb.wavelength))
    tx = np.tan(float(np.float32(pb.tilt_x_mrad)) * 1e-3); ty = np.tan(float(np.float32(pb.tilt_y_mrad)) * 1e-3)
    ky = (s / px)[:, None]; kx = (s / px)[None, :]
    deltas = []; L = 0.0; inter = []
    for j in range(pos.shape[0]):
        r0y, dy = orc.position_split(float(pos[j, 0]), pb.pixel_size, n)
        r0x, dx = orc.position_split(float(pos[j, 1]), pb.pixel_size, n)
        d = torch.tensor([dy, dx], dtype=torch.float64, requires_grad=True); deltas.append(d)
        R = torch.exp(-2j * np.pi * (s[:, None] * d[0] + s[None, :] * d[1]))
        I = torch.zeros((n, n), dtype=torch.float64)
        for k in range(M):
            psi = torch.fft.ifft2(R * torch.fft.fft2(P[k]))
            for i in range(S):
                phi = psi * O[i, r0y:r0y + n, r0x:r0x + n]
                if retain:
                    phi.retain_grad(); inter.append((j, i, k, psi, phi))
                if i < S - 1:
                    dz = float(np.float32(pb.slice_thickness[i]))
                    H = torch.exp(-1j * np.pi * lam * dz * (kx ** 2 + ky ** 2) + 2j * np.pi * dz * (kx * tx + ky * ty))
                    if pb.bandlimit > 0:
                        si = torch.tensor(np.where(np.arange(n) < n // 2, np.arange(n), np.arange(n) - n))
                        H = H * ((si[:, None] ** 2 + si[None, :] ** 2) <= (0.5 * float(np.float32(pb.bandlimit)) * n) ** 2)
                    psi = torch.fft.ifft2(H * torch.fft.fft2(phi))
            I = I + torch.abs(torch.fft.fft2(phi) / n) ** 2
        Ie = torch.tensor(Iexp[j].astype(np.float64)); eps = float(np.float32(pb.eps)); c = float(np.float32(pb.loss_c))
        if pb.loss == orc.LOSS_POISSON:
            L = L + torch.sum(I - Ie * (torch.log(I + eps) - torch.log(Ie + eps) + 1.0))
        else:
            L = L + torch.sum(0.5 * (torch.sqrt(I + c) - torch.sqrt(Ie + c)) ** 2)
    L.backward()
    gd = np.array([d.grad.numpy() for d in deltas])
    return L.item(), O.grad.numpy() / 2.0, P.grad.numpy() / 2.0, gd, inter     # torch returns 2 dL/dconj(z) (R15)


@pytest.mark.parametrize("loss,eps,S,bandlimit", [(orc.LOSS_POISSON, 0.8, 3, 0.0), (orc.LOSS_POISSON, 0.8, 2, 2.0 / 3.0),
                                                  (orc.LOSS_AMPLITUDE, 1e-12, 1, 0.0), (orc.LOSS_AMPLITUDE, 1e-12, 3, 0.0)])
def test_gradient_vs_torch_autograd(loss, eps, S, bandlimit):
    pb, obj, probe, pos = small_problem(n=16, M=2, S=S, on=36, J=4, loss=loss, eps=eps, bandlimit=bandlimit)
    Iexp = orc.forward_loss(pb, (obj * 1.05).astype(np.complex64), probe, pos)["intensity"].astype(np.float32) + 0.1
    g = orc.gradient(pb, obj, probe, pos, Iexp)
    L, gO, gP, gd, _ = _torch_model(pb, obj, probe, pos, Iexp)
    rel = lambda a, b: np.linalg.norm(a - b) / np.linalg.norm(b)
    assert abs(g["loss"] - L) < 1e-10 * abs(L)
    assert rel(g["grad_object"], gO) < 1e-9
    assert rel(g["grad_probe"], gP) < 1e-9
    assert rel(g["grad_pos"], gd / float(np.float32(pb.pixel_size))) < 1e-8


def test_single_slice_epie_relation():
    # in single slice, gO|patch = -conj(P_shift) chi and gP-contribution = -conj(O) chi,
    # chi = -N Finv(w psi~)  — i.e. ePIE's Delta O ~ P* chi is the negative Wirtinger gradient.
    n, on = 16, 36
    pb, obj, probe, pos = small_problem(n=n, M=1, S=1, on=on, J=1, loss=orc.LOSS_POISSON, eps=0.8)
    Iexp = orc.forward_loss(pb, (obj * 1.05).astype(np.complex64), probe, pos)["intensity"].astype(np.float32) + 0.1
    g = orc.gradient(pb, obj, probe, pos, Iexp)
    r0y, dy = orc.position_split(float(pos[0, 0]), pb.pixel_size, n); r0x, dx = orc.position_split(float(pos[0, 1]), pb.pixel_size, n)
    Ps = orc.shift(probe[0].astype(complex), dy, dx)
    patch = obj[0, r0y:r0y + n, r0x:r0x + n].astype(complex)
    psit = np.fft.fft2(Ps * patch) / n
    I = np.abs(psit) ** 2
    w = 1 - Iexp[0] / (I + float(np.float32(0.8)))
    chi = -n * np.fft.ifft2(w * psit)
    assert np.abs(g["grad_object"][0, r0y:r0y + n, r0x:r0x + n] - (-np.conj(Ps) * chi)).max() < 1e-9 * np.abs(chi).max() * np.abs(Ps).max()
    gP_ref = orc.shift(-np.conj(patch) * chi, dy, dx, adjoint=True)
    assert np.abs(g["grad_probe"][0] - gP_ref).max() < 1e-9 * np.abs(gP_ref).max()


# ------------------------------------------------------------------------------------------------
# LSQML-style terms (O12..O15; readings R18..R21)
# ------------------------------------------------------------------------------------------------
def test_lsqml_terms_vs_torch_intermediates():
    pb, obj, probe, pos = small_problem(n=16, M=2, S=3, on=36, J=3, loss=orc.LOSS_POISSON, eps=0.8)
    pb.lsqml_delta_o = 0.7; pb.lsqml_delta_p = 0.2
    Iexp = orc.forward_loss(pb, (obj * 1.05).astype(np.complex64), probe, pos)["intensity"].astype(np.float32) + 0.1
    g = orc.gradient(pb, obj, probe, pos, Iexp, want_illum=True)
    illum_prev = g["illum"] * 1.3 + 0.1
    st = orc.step_terms(pb, obj, probe, pos, Iexp, g["grad_object"], g["grad_probe"], illum_prev)
    # numX = -1/2 dL/d delta  (O14)
    px = float(np.float32(pb.pixel_size)); S = 3
    assert np.abs(st[:, 2 * S + 2] + 0.5 * g["grad_pos"][:, 0] * px).max() < 1e-9 * np.abs(g["grad_pos"]).max()
    assert np.abs(st[:, 2 * S + 4] + 0.5 * g["grad_pos"][:, 1] * px).max() < 1e-9 * np.abs(g["grad_pos"]).max()
    # illumination map (O12) and object terms against autograd intermediates chi = -gPhi
    _, _, _, _, inter = _torch_model(pb, obj, probe, pos, Iexp, retain=True)
    n = 16
    dOhat = -g["grad_object"] / (illum_prev + float(np.float32(0.7)))
    num = np.zeros((3, S)); den = np.zeros((3, S)); il = np.zeros_like(g["illum"])
    for (j, i, k, psi, phi) in inter:
        r0y, _ = orc.position_split(float(pos[j, 0]), pb.pixel_size, n); r0x, _ = orc.position_split(float(pos[j, 1]), pb.pixel_size, n)
        chi = -(phi.grad.numpy() / 2.0); Psi = psi.detach().numpy()
        u = dOhat[i, r0y:r0y + n, r0x:r0x + n] * Psi
        num[j, i] += np.sum(np.real(chi * np.conj(u))); den[j, i] += np.sum(np.abs(u) ** 2)
        il[i, r0y:r0y + n, r0x:r0x + n] += np.abs(Psi) ** 2
    assert np.abs(il - g["illum"]).max() < 1e-10 * il.max()
    assert np.abs(st[:, 0:2 * S:2] - num).max() < 1e-9 * np.abs(num).max()
    assert np.abs(st[:, 1:2 * S:2] - den).max() < 1e-9 * np.abs(den).max()


@pytest.mark.parametrize("S", [1, 2])
def test_lsqml_probe_and_position_terms_numpy_restatement(S):
    # O14 probe / position terms written out in numpy (PAPER.md:221 applied to the probe and to the shift, readings R19, R21):
    #   v_k = shift_j(dPhat_k) T_0,  s_{a,k} = Finv(-2 pi i f_a R P~_k) T_0,  chi_{0,k} = -gPhi_{0,k}
    #   numP = sum_k Re<chi, v>, denP = sum_k |v|^2, numX_a = sum_k Re<chi, s_a>, denX_a = sum_k |s_a|^2
    # S = 1: chi_0 is the numpy one-liner -N Finv(w psi~), so num and den are both pinned; S = 2: the denominators only
    # (they must use the FIRST slice's patch and sum over both modes).
    n, on, M, J = 16, 40, 2, 3
    pb, obj, probe, pos = small_problem(n=n, M=M, S=S, on=on, J=J, loss=orc.LOSS_POISSON, eps=0.8)
    pb.lsqml_delta_o = 0.7; pb.lsqml_delta_p = 0.2
    Iexp = orc.forward_loss(pb, (obj * 1.05).astype(np.complex64), probe, pos)["intensity"].astype(np.float32) + 0.1
    g = orc.gradient(pb, obj, probe, pos, Iexp, want_illum=True)
    st = orc.step_terms(pb, obj, probe, pos, Iexp, g["grad_object"], g["grad_probe"], g["illum"] + 0.5)
    f = np.where(np.arange(n) < n // 2, np.arange(n), np.arange(n) - n) / n
    dPhat = -g["grad_probe"] / (1.0 + float(np.float32(0.2)))
    Pt = np.fft.fft2(probe.astype(complex))
    for j in range(J):
        r0y, dy = orc.position_split(float(pos[j, 0]), pb.pixel_size, n); r0x, dx = orc.position_split(float(pos[j, 1]), pb.pixel_size, n)
        R = np.exp(-2j * np.pi * (f[:, None] * dy + f[None, :] * dx))
        T0 = obj[0, r0y:r0y + n, r0x:r0x + n].astype(complex)
        numP = denP = 0.0; numX = np.zeros(2); denX = np.zeros(2)
        if S == 1:
            psit = np.stack([np.fft.fft2(np.fft.ifft2(R * Pt[k]) * T0) / n for k in range(M)])
            w = 1 - Iexp[j] / ((np.abs(psit) ** 2).sum(0) + float(np.float32(0.8)))
        for k in range(M):
            v = np.fft.ifft2(R * np.fft.fft2(dPhat[k])) * T0
            sa = [np.fft.ifft2(-2j * np.pi * fa * R * Pt[k]) * T0 for fa in (f[:, None] + 0 * f[None, :], f[None, :] + 0 * f[:, None])]
            denP += np.sum(np.abs(v) ** 2)
            for a in range(2):
                denX[a] += np.sum(np.abs(sa[a]) ** 2)
            if S == 1:
                chi = -n * np.fft.ifft2(w * psit[k])
                numP += np.sum(np.real(chi * np.conj(v)))
                for a in range(2):
                    numX[a] += np.sum(np.real(chi * np.conj(sa[a])))
        assert abs(st[j, 2 * S + 1] - denP) < 1e-10 * denP
        assert abs(st[j, 2 * S + 3] - denX[0]) < 1e-10 * denX[0] and abs(st[j, 2 * S + 5] - denX[1]) < 1e-10 * denX[1]
        if S == 1:
            assert abs(st[j, 2 * S] - numP) < 1e-9 * abs(numP)
            assert abs(st[j, 2 * S + 2] - numX[0]) < 1e-9 * abs(numX[0]) and abs(st[j, 2 * S + 4] - numX[1]) < 1e-9 * abs(numX[1])


def test_lsqml_alpha_closed_form_single_position():
    # single position, single slice, one mode, illum_prev = this position's |Psi|^2, delta_O -> 0, gamma = 0:
    # dOhat|patch = conj(Psi) chi / |Psi|^2, so dOhat Psi = chi and alpha_O = sum|chi|^2 / sum|chi|^2 = 1,
    # i.e. the step that zeroes the linearised exit-wave residual.
    n, on = 16, 36
    pb, obj, probe, pos = small_problem(n=n, M=1, S=1, on=on, J=1, loss=orc.LOSS_POISSON, eps=0.8)
    pb.lsqml_delta_o = 1e-30
    Iexp = orc.forward_loss(pb, (obj * 1.05).astype(np.complex64), probe, pos)["intensity"].astype(np.float32) + 0.1
    g = orc.gradient(pb, obj, probe, pos, Iexp, want_illum=True)
    illum_prev = np.where(g["illum"] > 0, g["illum"], 1.0)
    st = orc.step_terms(pb, obj, probe, pos, Iexp, g["grad_object"], g["grad_probe"], illum_prev)
    assert abs(st[0, 0] / st[0, 1] - 1.0) < 1e-9
    # and the update moves the object by exactly beta * alpha * dOhat
    o2, p2, x2 = orc.apply_update(pb, 1, obj, probe, pos, g["grad_object"], None, None, illum_prev, st, beta_obj=0.5)
    assert np.abs((o2 - obj) - 0.5 * (-g["grad_object"] / (illum_prev + 1e-30))).max() < 1e-9


def test_lsqml_position_step_recovers_offset():
    # reading R21 (parity unpinned against the paper): the least-squares shift num/(den+gamma) walks a
    # known sub-pixel offset back monotonically on a noiseless single-position toy with a strong object.
    # (chi from an intensity-only loss sees only the amplitude part of the residual, so the contraction
    # per step is ~0.8, not a one-step Newton solve.)
    n, on = 16, 40
    pb, obj, probe, pos = small_problem(n=n, M=1, S=1, on=on, J=1, loss=orc.LOSS_AMPLITUDE, eps=1e-6)
    s = np.where(np.arange(n) < n // 2, np.arange(n), np.arange(n) - n)
    Pt = (s[:, None] ** 2 + s[None, :] ** 2 <= 16) * np.exp(1j * 0.25 * (s[:, None] ** 2 + s[None, :] ** 2))
    probe = (np.fft.fftshift(np.fft.ifft2(Pt))[None] * 30).astype(np.complex64)
    yy, xx = np.meshgrid(np.arange(on), np.arange(on + 2), indexing="ij")
    ph = 1.5 * (np.sin(2 * np.pi * yy / 9.0) + np.cos(2 * np.pi * xx / 7.0) + np.sin(2 * np.pi * (yy + xx) / 5.0))
    obj = np.exp(1j * ph)[None].astype(np.complex64)
    true = np.array([[(20.0 + 0.12) * 0.2, (21.0 - 0.08) * 0.2]], np.float32)
    Iexp = orc.forward_loss(pb, obj, probe, true)["intensity"].astype(np.float32)
    x = np.array([[20.0 * 0.2, 21.0 * 0.2]], np.float32)
    errs = [np.abs(x - true).max()]
    for _ in range(8):
        g = orc.gradient(pb, obj, probe, x, Iexp, want_illum=True)
        st = orc.step_terms(pb, obj, probe, x, Iexp, g["grad_object"], g["grad_probe"], g["illum"] + 1.0)
        _, _, x2 = orc.apply_update(pb, 1, obj, probe, x, None, None, None, g["illum"] + 1.0, st)
        x = x2.astype(np.float32); errs.append(np.abs(x - true).max())
    assert all(b < a for a, b in zip(errs, errs[1:]))
    assert errs[-1] < 0.3 * errs[0]


def test_lsqml_weighted_update_per_position_alpha():
    # PAPER.md:225 as printed (reading R24): O_i += beta sum_j alpha_{i,j} dOhat_i sum_k|Psi_{i,k,j}|^2 / sum_{j,k}|Psi_{i,k,j}|^2
    pb, obj, probe, pos = small_problem(n=16, M=2, S=3, on=36, J=4, loss=orc.LOSS_POISSON, eps=0.8)
    pb.lsqml_delta_o = 0.7
    Iexp = orc.forward_loss(pb, (obj * 1.05).astype(np.complex64), probe, pos)["intensity"].astype(np.float32) + 0.1
    g = orc.gradient(pb, obj, probe, pos, Iexp, want_illum=True)
    illum_prev = g["illum"] * 1.3 + 0.1
    st = orc.step_terms(pb, obj, probe, pos, Iexp, g["grad_object"], g["grad_probe"], illum_prev)
    gamma, S, J = 0.3, 3, 4
    W = orc.weighted_illum(pb, obj, probe, pos, st, gamma)
    # (a) linearity route: W = sum_j alpha_{i,j} illum_j with illum_j the (already pinned, O12) map of the one-position batch {j}
    alpha = st[:, 0:2 * S:2] / (st[:, 1:2 * S:2] + gamma)                       # PAPER.md:221 per position
    ref = np.zeros_like(W)
    for j in range(J):
        ilj = orc.gradient(pb, obj, probe, pos, Iexp, batch_idx=[j], want_illum=True)["illum"]
        ref += alpha[j][:, None, None] * ilj
    assert np.abs(W - ref).max() < 1e-12 * np.abs(ref).max()
    # (b) equal step sizes for every position collapse :225 to the per-group form O_i += beta alpha_i dOhat_i (reading R18)
    st_eq = st.copy(); a_i = np.array([0.4, -0.2, 1.1])
    st_eq[:, 0:2 * S:2] = a_i[None, :] * (st[:, 1:2 * S:2] + gamma)
    W_eq = orc.weighted_illum(pb, obj, probe, pos, st_eq, gamma)
    cov = g["illum"] > 0
    assert np.abs(W_eq - a_i[:, None, None] * g["illum"]).max() < 1e-12 * np.abs(g["illum"]).max()
    o_w = orc.lsqml_weighted_object(pb, obj, g["grad_object"], illum_prev, g["illum"], W_eq, beta_obj=0.5)
    dOhat = -g["grad_object"] / (illum_prev + float(np.float32(0.7)))
    o_g = obj.astype(np.complex128) + 0.5 * a_i[:, None, None] * dOhat
    assert np.abs(o_w - o_g)[cov].max() < 1e-12
    assert np.abs(o_w - obj.astype(np.complex128))[~cov].max() == 0.0          # uncovered pixels are left alone
    # (c) the printed formula, written out pixel by pixel on one slice (brute force)
    o_w = orc.lsqml_weighted_object(pb, obj, g["grad_object"], illum_prev, g["illum"], W, beta_obj=0.8)
    i = 1
    ys, xs = np.nonzero(g["illum"][i] > 0)
    for (y, x) in [(ys[0], xs[0]), (ys[len(ys) // 2], xs[len(ys) // 2]), (ys[-1], xs[-1])]:
        expect = obj[i, y, x].astype(np.complex128) + 0.8 * dOhat[i, y, x] * ref[i, y, x] / g["illum"][i, y, x]
        assert abs(o_w[i, y, x] - expect) < 1e-12


def test_lsqml_probe_preconditioner_object_transparency():
    # PAPER.md:227 (reading R25): sum_j prod_i |O_i|^2 recorded in the probe/cutout view
    n, on, S, J = 16, 36, 3, 4
    pb, obj, probe, pos = small_problem(n=n, M=2, S=S, on=on, J=J, loss=orc.LOSS_POISSON, eps=0.8)
    ot = orc.object_transparency(pb, obj, pos)
    # (a) numpy restatement through the (separately pinned) position split
    ref = np.zeros((n, n))
    for j in range(J):
        r0y, _ = orc.position_split(float(pos[j, 0]), pb.pixel_size, n); r0x, _ = orc.position_split(float(pos[j, 1]), pb.pixel_size, n)
        ref += np.prod(np.abs(obj[:, r0y:r0y + n, r0x:r0x + n].astype(np.complex128)) ** 2, axis=0)
    assert np.abs(ot - ref).max() < 1e-12 * ref.max()
    # (b) vacuum object: every window is fully transparent, the map is the number of positions
    assert np.abs(orc.object_transparency(pb, np.ones_like(obj), pos) - J).max() == 0.0
    assert np.abs(orc.object_transparency(pb, np.ones_like(obj), pos, batch_idx=[2, 0]) - 2).max() == 0.0
    # (c) closed form of the probe step (the probe analogue of test_lsqml_alpha_closed_form_single_position): one position,
    # one slice, one mode, preconditioner = this position's |T|^2, delta_P -> 0, delta = 0 (no sub-pixel shift): dPhat T = chi on
    # the support, so alpha_P = 1 — the step that zeroes the linearised exit-wave residual
    pb1, obj1, probe1, pos1 = small_problem(n=n, M=1, S=1, on=on, J=1, loss=orc.LOSS_POISSON, eps=0.8)
    pos1 = (np.round(pos1 / pb1.pixel_size) * pb1.pixel_size).astype(np.float32)              # integer pixel position
    assert orc.position_split(float(pos1[0, 0]), pb1.pixel_size, n)[1] == 0.0
    pb1.lsqml_delta_p = 1e-30
    Iexp = orc.forward_loss(pb1, (obj1 * 1.05).astype(np.complex64), probe1, pos1)["intensity"].astype(np.float32) + 0.1
    g = orc.gradient(pb1, obj1, probe1, pos1, Iexp, want_illum=True)
    pc = orc.object_transparency(pb1, obj1, pos1)
    st = orc.step_terms(pb1, obj1, probe1, pos1, Iexp, g["grad_object"], g["grad_probe"], g["illum"] + 1.0, probe_precond=pc)
    assert abs(st[0, 2] / st[0, 3] - 1.0) < 1e-9
    # the update divides by the same map; without it the divisor is the constant 1 (reading R19)
    _, p2, _ = orc.apply_update(pb1, 1, obj1, probe1, pos1, None, g["grad_probe"], None, g["illum"] + 1.0, st, beta_probe=0.5, probe_precond=pc)
    assert np.abs((p2 - probe1) - 0.5 * (st[0, 2] / st[0, 3]) * (-g["grad_probe"] / (pc + 1e-30))).max() < 1e-9
    st1 = orc.step_terms(pb1, obj1, probe1, pos1, Iexp, g["grad_object"], g["grad_probe"], g["illum"] + 1.0)
    st_ones = orc.step_terms(pb1, obj1, probe1, pos1, Iexp, g["grad_object"], g["grad_probe"], g["illum"] + 1.0, probe_precond=np.ones((n, n)))
    assert np.array_equal(st1, st_ones)


def test_sgd_update():
    pb, obj, probe, pos = small_problem()
    gO = crandn(*obj.shape); gP = crandn(*probe.shape); gX = RNG.standard_normal(pos.shape)
    o, p, x = orc.apply_update(pb, 0, obj, probe, pos, gO, gP, gX, lr_obj=0.1, lr_probe=0.2, lr_pos=0.3)
    assert np.abs(o - (obj - 0.1 * gO)).max() < 1e-12 and np.abs(p - (probe - 0.2 * gP)).max() < 1e-12
    assert np.abs(x - (pos - 0.3 * gX)).max() < 1e-12


# ------------------------------------------------------------------------------------------------
# bilinear object sampling (SURVEY.md §8(c) R1 secondary mode, "sampled"; shift_mode = 1)
# ------------------------------------------------------------------------------------------------
def test_bilinear_split_and_gather_closed_forms():
    # floor split: c = X/px - N/2 = i0 + f, f in [0,1)
    for X, px, n, want in [(2.0, 0.2, 8, (6, 0.0)), (2.05, 0.2, 8, (6, 0.25)), (0.79, 0.2, 8, (-1, 0.95))]:
        i0, f = orc.position_split_floor(X, px, n)
        assert i0 == want[0] and abs(f - want[1]) < 1e-5
    # a bilinear interpolant reproduces any function a + b y + c x + d x y exactly
    on, n = 14, 6
    yy, xx = np.meshgrid(np.arange(on), np.arange(on), indexing="ij")
    obj = (0.3 + 0.7j) + (0.2 - 0.1j) * yy + (-0.4 + 0.5j) * xx + 0.05j * xx * yy
    i0y, i0x, fy, fx = 3, 5, 0.37, 0.81
    T = orc.bilinear(n, obj, i0y, i0x, fy, fx)
    ys, xs = np.meshgrid(i0y + fy + np.arange(n), i0x + fx + np.arange(n), indexing="ij")
    assert np.abs(T - ((0.3 + 0.7j) + (0.2 - 0.1j) * ys + (-0.4 + 0.5j) * xs + 0.05j * xs * ys)).max() < 1e-12
    # f = 0: the plain integer window
    assert np.abs(orc.bilinear(n, obj, i0y, i0x, 0.0, 0.0) - obj[i0y:i0y + n, i0x:i0x + n]).max() == 0
    # adjoint pair (dot-product test) and weight sum: scattering ones deposits n*n in total
    a = crandn(on, on); y = crandn(n, n)
    lhs = np.vdot(orc.bilinear(n, a, i0y, i0x, fy, fx), y)
    rhs = np.vdot(a, orc.bilinear(n, np.zeros((on, on), complex), i0y, i0x, fy, fx, patch=y))
    assert abs(lhs - rhs) < 1e-12 * abs(lhs)
    acc = orc.bilinear(n, np.zeros((on, on), complex), i0y, i0x, fy, fx, patch=np.ones((n, n), complex))
    assert abs(acc.sum() - n * n) < 1e-12


def _bilinear_problem(**kw):
    pb, obj, probe, pos = small_problem(**kw)
    pb.shift_mode = orc.SHIFT_BILINEAR_OBJECT
    return pb, obj, probe, pos


def test_bilinear_forward_special_cases():
    n, on = 8, 20
    pb, obj, probe, pos = _bilinear_problem(n=n, M=2, S=3, on=on, J=4)
    # (1) integer corners: identical to the Fourier-shift mode, whose shift is then zero too
    pos_int = (np.array([[5, 6], [4, 9], [7, 5], [9, 9]]) * 0.2).astype(np.float32)
    pf = orc.Problem(**{**pb.__dict__, "shift_mode": orc.SHIFT_FOURIER_PROBE})
    a = orc.forward_loss(pb, obj, probe, pos_int)["intensity"]; b = orc.forward_loss(pf, obj, probe, pos_int)["intensity"]
    assert np.abs(a - b).max() < 1e-12 * np.abs(b).max()
    # (2) an object that is constant in the plane: the pattern does not depend on the position at all
    flat = np.ones_like(obj) * np.exp(0.3j * np.arange(3))[:, None, None].astype(np.complex64)
    out = orc.forward_loss(pb, flat, probe, pos)["intensity"]
    assert np.abs(out - out[0]).max() < 1e-10 * np.abs(out).max()
    # (3) S = 1: |F(P . T)|^2 / N^2 with T the bilinear patch and the probe NOT shifted
    pb1, obj1, probe1, pos1 = _bilinear_problem(n=n, M=1, S=1, on=on, J=2)
    out = orc.forward_loss(pb1, obj1, probe1, pos1)["intensity"]
    for j in range(2):
        (i0y, fy), (i0x, fx) = orc.position_split_floor(float(pos1[j, 0]), 0.2, n), orc.position_split_floor(float(pos1[j, 1]), 0.2, n)
        T = orc.bilinear(n, obj1[0].astype(complex), i0y, i0x, fy, fx)
        ref = np.abs(np.fft.fft2(probe1[0].astype(complex) * T)) ** 2 / n ** 2
        assert np.abs(out[j] - ref).max() < 1e-10 * ref.max()


def test_bilinear_gradient_finite_differences():
    pb, obj, probe, pos = _bilinear_problem(J=4)
    obj_t = (obj * np.exp(0.2 * crandn(*obj.shape))).astype(np.complex64)
    Iexp = orc.forward_loss(pb, obj_t, probe, pos)["intensity"].astype(np.float32) + 0.05
    # keep the fractions away from 0 and 1 so the integer corner does not flip under the position steps
    for j in range(4):
        for a in range(2):
            i0, f = orc.position_split_floor(float(pos[j, a]), 0.2, 8)
            if f < 0.2 or f > 0.8:
                pos[j, a] = np.float32((i0 + 4 + 0.5) * 0.2)
    g = orc.gradient(pb, obj, probe, pos, Iexp, want_illum=True)

    def L(o, p, x=pos):
        return orc.forward_loss(pb, o, p, x, Iexp, want_intensity=False)["loss"]

    assert abs(L(obj, probe) - g["loss"]) < 1e-12 * abs(g["loss"])
    h = 2.0 ** -9
    for which in ("obj", "probe"):
        base = obj if which == "obj" else probe
        D = crandn(*base.shape).astype(np.complex64)
        zp = (base.astype(np.complex128) + h * D).astype(np.complex64); zm = (base.astype(np.complex128) - h * D).astype(np.complex64)
        Dact = (zp.astype(np.complex128) - zm.astype(np.complex128)) / 2.0
        fd = (L(zp, probe) - L(zm, probe)) / 2.0 if which == "obj" else (L(obj, zp) - L(obj, zm)) / 2.0
        gw = g["grad_object" if which == "obj" else "grad_probe"]
        lin = 2.0 * np.real(np.vdot(gw, Dact))
        # the O(h^2) truncation error scales with |g||D|, not with the (possibly cancelling) directional derivative
        assert abs(fd - lin) < 2e-4 * abs(lin) + 1e-4 * np.linalg.norm(gw) * np.linalg.norm(Dact), (which, fd, lin)
    hx = 2e-3 * 0.2
    for j in range(4):
        for a in range(2):
            pp = pos.copy(); pm = pos.copy(); pp[j, a] += np.float32(hx); pm[j, a] -= np.float32(hx)
            fd = (L(obj, probe, pp) - L(obj, probe, pm)) / (float(pp[j, a]) - float(pm[j, a]))
            assert abs(fd - g["grad_pos"][j, a]) < 2e-3 * abs(fd) + 1e-6, (j, a, fd, g["grad_pos"][j, a])
    # illumination map: the weights of a position sum to one, so the total equals the total entering intensity
    pf = orc.Problem(**{**pb.__dict__, "shift_mode": orc.SHIFT_FOURIER_PROBE})
    assert g["illum"].min() >= 0
    # slice 0: sum_r |Psi_0|^2 = sum |P|^2 per position (unshifted probe), 4 positions
    assert abs(g["illum"][0].sum() - 4 * (np.abs(probe.astype(complex)) ** 2).sum()) < 1e-9 * g["illum"][0].sum()


def test_bilinear_step_terms():
    # readings R1 / R30: LSQML step-size terms with the patches sampled bilinearly.
    n, on, M, S, J = 8, 20, 2, 3, 4
    pb, obj, probe, pos = _bilinear_problem(n=n, M=M, S=S, on=on, J=J)
    pb.lsqml_delta_o = 0.7; pb.lsqml_delta_p = 0.2
    obj_t = (obj * np.exp(0.2 * crandn(*obj.shape))).astype(np.complex64)
    Iexp = orc.forward_loss(pb, obj_t, probe, pos)["intensity"].astype(np.float32) + 0.05
    g = orc.gradient(pb, obj, probe, pos, Iexp, want_illum=True)
    illum_prev = g["illum"] * 1.3 + 0.1
    st = orc.step_terms(pb, obj, probe, pos, Iexp, g["grad_object"], g["grad_probe"], illum_prev)
    px = float(np.float32(pb.pixel_size))
    # (1) numX_a = -1/2 dL/df_a (f in px; grad_pos is per Angstrom and is itself pinned by finite differences above)
    assert np.abs(st[:, 2 * S + 2] + 0.5 * g["grad_pos"][:, 0] * px).max() < 1e-9 * np.abs(g["grad_pos"] * px).max()
    assert np.abs(st[:, 2 * S + 4] + 0.5 * g["grad_pos"][:, 1] * px).max() < 1e-9 * np.abs(g["grad_pos"] * px).max()
    # (2) denominators restated in numpy from the illumination of ONE position: sum_k |Psi_{i,k}|^2 in the probe view is the
    # oracle's own illumination map of that position sampled back... instead use S = 1, where Psi_0 = P_k (unshifted probe):
    pb1, obj1, probe1, pos1 = _bilinear_problem(n=n, M=M, S=1, on=on, J=2)
    pb1.lsqml_delta_o = 0.7; pb1.lsqml_delta_p = 0.2
    I1 = orc.forward_loss(pb1, (obj1 * 1.05).astype(np.complex64), probe1, pos1)["intensity"].astype(np.float32) + 0.1
    g1 = orc.gradient(pb1, obj1, probe1, pos1, I1, want_illum=True)
    ip1 = g1["illum"] + 0.5
    st1 = orc.step_terms(pb1, obj1, probe1, pos1, I1, g1["grad_object"], g1["grad_probe"], ip1)
    dOhat = -g1["grad_object"] / (ip1 + float(np.float32(0.7)))
    dPhat = -g1["grad_probe"] / (1.0 + float(np.float32(0.2)))
    P2 = (np.abs(probe1.astype(complex)) ** 2).sum(0)
    for j in range(2):
        (i0y, fy), (i0x, fx) = orc.position_split_floor(float(pos1[j, 0]), 0.2, n), orc.position_split_floor(float(pos1[j, 1]), 0.2, n)
        T = orc.bilinear(n, obj1[0].astype(complex), i0y, i0x, fy, fx)
        dT = orc.bilinear(n, dOhat[0], i0y, i0x, fy, fx)                       # dOhat sampled like the patch
        psit = np.stack([np.fft.fft2(probe1[k].astype(complex) * T) / n for k in range(M)])
        w = 1 - I1[j] / ((np.abs(psit) ** 2).sum(0) + float(np.float32(pb1.eps)))
        chi = np.stack([-n * np.fft.ifft2(w * psit[k]) for k in range(M)])
        num = sum(np.sum(np.real(chi[k] * np.conj(dT * probe1[k]))) for k in range(M))
        assert abs(st1[j, 0] - num) < 1e-9 * abs(num) and abs(st1[j, 1] - np.sum(np.abs(dT) ** 2 * P2)) < 1e-10 * st1[j, 1]
        numP = sum(np.sum(np.real(chi[k] * np.conj(dPhat[k] * T))) for k in range(M))
        denP = sum(np.sum(np.abs(dPhat[k] * T) ** 2) for k in range(M))
        assert abs(st1[j, 2] - numP) < 1e-9 * abs(numP) and abs(st1[j, 3] - denP) < 1e-10 * denP
        # dT/df by central differences of the sampler itself (bilinear sampling is bilinear in f: exact)
        h = 1e-3
        dTy = (orc.bilinear(n, obj1[0].astype(complex), i0y, i0x, fy + h, fx) - orc.bilinear(n, obj1[0].astype(complex), i0y, i0x, fy - h, fx)) / (2 * h)
        dTx = (orc.bilinear(n, obj1[0].astype(complex), i0y, i0x, fy, fx + h) - orc.bilinear(n, obj1[0].astype(complex), i0y, i0x, fy, fx - h)) / (2 * h)
        for a, d in enumerate((dTy, dTx)):
            den = np.sum(np.abs(d) ** 2 * P2)
            numx = sum(np.sum(np.real(chi[k] * np.conj(probe1[k] * d))) for k in range(M))
            assert abs(st1[j, 5 + 2 * a] - den) < 1e-8 * den and abs(st1[j, 4 + 2 * a] - numx) < 1e-8 * abs(numx) + 1e-12
    # (3) integer corners: object and probe terms equal those of the Fourier-shift mode (both reduce to the integer window and the
    # unshifted probe)
    pos_int = (np.array([[5, 6], [4, 9], [7, 5], [9, 9]]) * 0.2).astype(np.float32)
    pf = orc.Problem(**{**pb.__dict__, "shift_mode": orc.SHIFT_FOURIER_PROBE})
    gb = orc.gradient(pb, obj, probe, pos_int, Iexp, want_illum=True)
    sb = orc.step_terms(pb, obj, probe, pos_int, Iexp, gb["grad_object"], gb["grad_probe"], illum_prev)
    sf = orc.step_terms(pf, obj, probe, pos_int, Iexp, gb["grad_object"], gb["grad_probe"], illum_prev)
    assert np.abs(sb[:, :2 * S + 2] - sf[:, :2 * S + 2]).max() < 1e-10 * np.abs(sf[:, :2 * S + 2]).max()


def test_lsqml_modulus_constraint_chi():
    # reading R31: lsqml_chi_scale = 2 makes chi the modulus-constraint wavefront update of PAPER.md:173 (amplitude model).
    # (1) one position, one slice, one mode, illum_prev = this position's |Psi|^2, delta_O -> 0, gamma = 0, eps -> 0, c = 0: the
    #     LSQML object step with beta = 1 turns the exit wave into the modulus-projected one, Finv(sqrt(Iexp) F(psi) / |F(psi)|)
    #     ("the classic modulus constraint"), wherever the probe is non-zero
    n, on = 16, 40
    pb, obj, probe, pos = small_problem(n=n, M=1, S=1, on=on, J=1, loss=orc.LOSS_AMPLITUDE, eps=1e-30)
    pb.lsqml_delta_o = 1e-30; pb.lsqml_chi_scale = 2.0
    pos[:] = (np.array([[21, 18]]) * 0.2).astype(np.float32)                 # integer corner
    Iexp = RNG.uniform(0.5, 3.0, size=(1, n, n)).astype(np.float32)
    g = orc.gradient(pb, obj, probe, pos, Iexp, want_illum=True)
    illum_prev = np.where(g["illum"] > 0, g["illum"], 1.0)
    st = orc.step_terms(pb, obj, probe, pos, Iexp, g["grad_object"], g["grad_probe"], illum_prev)
    assert abs(st[0, 0] / st[0, 1] - 1.0) < 1e-9                             # alpha_O = 1
    o2, _, _ = orc.apply_update(pb, 1, obj, probe, pos, g["grad_object"], None, None, illum_prev, st, beta_obj=1.0)
    r0y, r0x = 21 - n // 2, 18 - n // 2
    f = np.where(np.arange(n) < n // 2, np.arange(n), np.arange(n) - n) / n
    (_, dy), (_, dx) = orc.position_split(float(pos[0, 0]), 0.2, n), orc.position_split(float(pos[0, 1]), 0.2, n)
    P = np.fft.ifft2(np.exp(-2j * np.pi * (f[:, None] * dy + f[None, :] * dx)) * np.fft.fft2(probe[0].astype(complex)))
    psi = P * obj[0, r0y:r0y + n, r0x:r0x + n].astype(complex)
    Fp = np.fft.fft2(psi)
    psi_c = np.fft.ifft2(np.sqrt(Iexp[0].astype(float)) * n * Fp / np.abs(Fp))
    assert np.abs(P * o2[0, r0y:r0y + n, r0x:r0x + n] - psi_c).max() < 1e-8 * np.abs(psi_c).max()
    # (2) against chi_scale = 1 on a multislice, two-mode case: object / probe terms x4, position numerators x2, position
    #     denominators unchanged; the update direction doubles
    pb2, obj2, probe2, pos2 = small_problem(n=8, M=2, S=3, on=20, J=3, loss=orc.LOSS_AMPLITUDE, eps=0.5)
    pb2.lsqml_delta_o = 0.7; pb2.lsqml_delta_p = 0.2
    I2 = orc.forward_loss(pb2, (obj2 * 1.05).astype(np.complex64), probe2, pos2)["intensity"].astype(np.float32) + 0.1
    g2 = orc.gradient(pb2, obj2, probe2, pos2, I2, want_illum=True)
    ip = g2["illum"] + 0.5
    s1 = orc.step_terms(pb2, obj2, probe2, pos2, I2, g2["grad_object"], g2["grad_probe"], ip)
    import dataclasses
    pbm = dataclasses.replace(pb2, lsqml_chi_scale=2.0)
    s2 = orc.step_terms(pbm, obj2, probe2, pos2, I2, g2["grad_object"], g2["grad_probe"], ip)
    S = 3
    scale = np.array([4.0] * (2 * S + 2) + [2.0, 1.0, 2.0, 1.0])
    assert np.abs(s2 - s1 * scale).max() < 1e-12 * np.abs(s2).max()
    a1 = orc.apply_update(pb2, 1, obj2, probe2, pos2, g2["grad_object"], g2["grad_probe"], None, ip, s1, beta_obj=0.5, beta_probe=0.5)
    a2 = orc.apply_update(pbm, 1, obj2, probe2, pos2, g2["grad_object"], g2["grad_probe"], None, ip, s2, beta_obj=0.5, beta_probe=0.5)
    assert np.abs((a2[0] - obj2) - 2 * (a1[0] - obj2)).max() < 1e-9 * np.abs(a1[0] - obj2).max()
    assert np.abs((a2[1] - probe2) - 2 * (a1[1] - probe2)).max() < 1e-9 * np.abs(a1[1] - probe2).max()
    assert np.abs((a2[2] - pos2) - 2 * (a1[2] - pos2)).max() < 1e-9 * np.abs(a1[2] - pos2).max()
    # (3) the paper gives the modulus-constraint update for the amplitude model only
    with pytest.raises(ValueError):
        orc.step_terms(dataclasses.replace(pbm, loss=orc.LOSS_POISSON), obj2, probe2, pos2, I2, g2["grad_object"], g2["grad_probe"], ip)


# ------------------------------------------------------------------------------------------------
# change detector: stored oracle outputs of a tiny seeded case (tests/golden/, written by make_golden.py from oracle/ only)
# ------------------------------------------------------------------------------------------------
def test_golden_oracle_tiny_case():
    import importlib.util
    import os
    here = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")
    spec = importlib.util.spec_from_file_location("make_golden", os.path.join(here, "make_golden.py"))
    mg = importlib.util.module_from_spec(spec); spec.loader.exec_module(mg)
    want = {}
    for line in open(os.path.join(here, "oracle_tiny_case.txt")):
        if line.startswith("#"):
            continue
        mode, key, val = line.split()
        want[(mode, key)] = float(val)
    assert len(want) == 16
    for mode, name in ((0, "fourier_probe"), (1, "bilinear_object")):
        for k, v in mg.checksums(mode):
            assert abs(float(v) - want[(name, k)]) <= 1e-10 * max(abs(want[(name, k)]), 1e-3), (name, k, v, want[(name, k)])


# ------------------------------------------------------------------------------------------------
# multislice ePIE directions (reading R23)
# ------------------------------------------------------------------------------------------------
def test_epie_single_slice_is_classic_epie():
    # S = 1, one mode, one position, eps -> 0, c = 0: the textbook ePIE step ("classic modulus constraint"):
    # psi_c = Finv( sqrt(Iexp) F(psi) / |F(psi)| ),  dO|patch = conj(P) / max|P|^2 (psi_c - psi),  dP = conj(O) / max|O|^2 (psi_c - psi)
    n, on = 16, 40
    pb, obj, probe, pos = small_problem(n=n, M=1, S=1, on=on, J=1, loss=orc.LOSS_AMPLITUDE, eps=1e-30)
    pos[:] = (np.array([[13, 17]]) * 0.2).astype(np.float32)                 # integer corner: no sub-pixel shift
    Iexp = (RNG.uniform(0.5, 3.0, size=(1, n, n))).astype(np.float32)
    e = orc.epie(pb, obj, probe, pos, Iexp)
    (r0y, dy), (r0x, dx) = orc.position_split(float(pos[0, 0]), 0.2, n), orc.position_split(float(pos[0, 1]), 0.2, n)
    assert (r0y, r0x) == (13 - n // 2, 17 - n // 2) and abs(dy) < 1e-5 and abs(dx) < 1e-5   # float32 X/px: a ~1e-6 px remainder
    f = np.where(np.arange(n) < n // 2, np.arange(n), np.arange(n) - n) / n
    ramp = np.exp(-2j * np.pi * (f[:, None] * dy + f[None, :] * dx))
    O = obj[0, r0y:r0y + n, r0x:r0x + n].astype(complex)
    P = np.fft.ifft2(ramp * np.fft.fft2(probe[0].astype(complex)))           # the probe as placed
    psi = P * O
    Fp = np.fft.fft2(psi)
    psi_c = np.fft.ifft2(np.sqrt(Iexp[0].astype(float)) * n * Fp / np.abs(Fp))   # |F psi|^2 / N^2 = I: amplitude sqrt(Iexp) N
    dpsi = psi_c - psi
    ref_dO = np.conj(P) / np.max(np.abs(P) ** 2) * dpsi
    ref_dP = np.conj(O) / np.max(np.abs(O) ** 2) * dpsi
    got = e["dir_object"][0, r0y:r0y + n, r0x:r0x + n]
    assert np.abs(got - ref_dO).max() < 1e-9 * np.abs(ref_dO).max()
    ref_dP = np.fft.ifft2(np.conj(ramp) * np.fft.fft2(ref_dP))               # back to the un-shifted probe frame
    assert np.abs(e["dir_probe"][0] - ref_dP).max() < 1e-9 * np.abs(ref_dP).max()
    outside = e["dir_object"].copy(); outside[0, r0y:r0y + n, r0x:r0x + n] = 0
    assert np.abs(outside).max() == 0


def test_epie_multislice_invariants():
    pb, obj, probe, pos = small_problem(n=8, M=2, S=3, on=20, J=3, loss=orc.LOSS_AMPLITUDE, eps=1e-30)
    # (1) noiseless data at the true state: both directions vanish
    Itrue = orc.forward_loss(pb, obj, probe, pos)["intensity"].astype(np.float64)
    # float32 storage of the data limits how exactly the modulus constraint is met: compare with the probe's own scale
    e0 = orc.epie(pb, obj, probe, pos, Itrue.astype(np.float32))
    assert np.abs(e0["dir_object"]).max() < 1e-6 and np.abs(e0["dir_probe"]).max() < 1e-6 * np.abs(probe).max()
    # (2) intensity-scaling covariance: P -> a P, Iexp -> a^2 Iexp leaves dO unchanged and scales dP by a
    Iexp = (Itrue * RNG.uniform(0.5, 1.5, size=Itrue.shape)).astype(np.float32)
    e1 = orc.epie(pb, obj, probe, pos, Iexp)
    e2 = orc.epie(pb, obj, (2.0 * probe).astype(np.complex64), pos, (4.0 * Iexp).astype(np.float32))
    assert np.abs(e2["dir_object"] - e1["dir_object"]).max() < 1e-6 * np.abs(e1["dir_object"]).max()
    assert np.abs(e2["dir_probe"] - 2.0 * e1["dir_probe"]).max() < 1e-6 * np.abs(e1["dir_probe"]).max()
    # (3) a small step along the directions lowers the amplitude loss (ePIE as gradient descent with a
    # variable step), and the loss it reports is the amplitude loss of the forward model
    L0 = orc.forward_loss(pb, obj, probe, pos, Iexp)["loss"]
    assert abs(e1["loss"] - L0) < 1e-12 * L0
    beta = 0.05
    L1 = orc.forward_loss(pb, (obj + beta * e1["dir_object"]).astype(np.complex64), (probe + beta * e1["dir_probe"]).astype(np.complex64), pos, Iexp)["loss"]
    assert L1 < L0
    # (4) relation to the gradient chain for a single slice and mode ("single-slice ePIE can be considered a
    # gradient descent method"): with eps -> 0, chi = -2 gPhi, hence dO = -2 gO / max|P_shift|^2 for ONE position
    pb1, obj1, probe1, pos1 = small_problem(n=8, M=1, S=1, on=20, J=1, loss=orc.LOSS_AMPLITUDE, eps=1e-30)
    I1 = (orc.forward_loss(pb1, obj1, probe1, pos1)["intensity"] * RNG.uniform(0.5, 1.5, size=(1, 8, 8))).astype(np.float32)
    g = orc.gradient(pb1, obj1, probe1, pos1, I1); e = orc.epie(pb1, obj1, probe1, pos1, I1)
    r0y, dy = orc.position_split(float(pos1[0, 0]), 0.2, 8); r0x, dx = orc.position_split(float(pos1[0, 1]), 0.2, 8)
    Ps = orc.shift(probe1[0].astype(complex), dy, dx)
    assert np.abs(e["dir_object"] + 2.0 * g["grad_object"] / np.max(np.abs(Ps) ** 2)).max() < 1e-9 * np.abs(e["dir_object"]).max()


def test_epie_dead_mode_contributes_nothing():
    # reading R23b: an identically zero probe mode (max|Psi|^2 = 0 in PAPER.md:203) adds nothing — the directions are finite
    # and equal those of the problem without that mode
    pb, obj, probe, pos = small_problem(n=8, M=2, S=2, on=20, J=3, loss=orc.LOSS_AMPLITUDE, eps=0.5)
    Iexp = (orc.forward_loss(pb, obj, probe, pos)["intensity"] * RNG.uniform(0.5, 1.5, size=(3, 8, 8))).astype(np.float32)
    dead = probe.copy(); dead[1] = 0
    e2 = orc.epie(pb, obj, dead, pos, Iexp)
    import dataclasses
    e1 = orc.epie(dataclasses.replace(pb, n_modes=1), obj, dead[:1], pos, Iexp)
    assert np.isfinite(e2["dir_object"]).all() and np.isfinite(e2["dir_probe"]).all()
    assert np.array_equal(e2["dir_object"], e1["dir_object"]) and np.array_equal(e2["dir_probe"][0], e1["dir_probe"][0])
    assert not e2["dir_probe"][1].any()


# ------------------------------------------------------------------------------------------------
# cost regularisers (R26), constraint regularisers (R27), Adam
# (R28)
# ------------------------------------------------------------------------------------------------
def test_cost_regularizers_closed_forms_and_finite_differences():
    S, ny, nx = 3, 5, 6
    z = 1.0 + 0.3 * crandn(S, ny, nx)
    # closed forms
    R, g = orc.cost_regularizer(orc.REG_L2, 0.7, z, ref=1.0)
    assert abs(R - 0.7 * np.sum(np.abs(z - 1) ** 2)) < 1e-12 and np.abs(g - 0.7 * (z - 1)).max() < 1e-14
    assert orc.cost_regularizer(orc.REG_L2, 0.7, np.ones_like(z))[0] == 0.0               # vacuum costs nothing
    y, x = np.meshgrid(np.arange(ny), np.arange(nx), indexing="ij")
    ramp = np.broadcast_to(2.0 * x + 3.0j * y, (S, ny, nx))
    assert abs(orc.cost_regularizer(orc.REG_TIKHONOV, 0.5, ramp)[0] - 0.5 * S * (4.0 * ny * (nx - 1) + 9.0 * (ny - 1) * nx)) < 1e-10
    step = np.ones((S, ny, nx), complex); step[:, :, 3:] = 1.0 + 0.4j                     # one edge of height 0.4 per row
    assert abs(orc.cost_regularizer(orc.REG_TV, 2.0, step, eps=0.0)[0] - 2.0 * S * ny * 0.4) < 1e-12
    layers = np.stack([np.full((ny, nx), v) for v in (1.0, 1.5, 1.5 + 2j)])
    assert abs(orc.cost_regularizer(orc.REG_LAYER_TIKHONOV, 1.0, layers)[0] - ny * nx * (0.25 + 4.0)) < 1e-12
    assert abs(orc.cost_regularizer(orc.REG_LAYER_TV, 1.0, layers, eps=0.0)[0] - ny * nx * (0.5 + 2.0)) < 1e-12
    assert abs(orc.cost_regularizer(orc.REG_L1, 3.0, layers, ref=1.0, eps=0.0)[0] - 3.0 * ny * nx * (0.0 + 0.5 + abs(0.5 + 2j))) < 1e-12
    # L1 on the phase (R26b): for z = r exp(i phi), R = w sum |phi| whatever r; the gradient is tangential (no radial part: scaling
    # a pixel does not change its phase) with modulus w / (2 r); the vacuum and a zero pixel cost nothing
    r = 0.5 + RNG.uniform(size=(S, ny, nx)); phi = RNG.uniform(-1.0, 1.0, size=(S, ny, nx))
    zp = r * np.exp(1j * phi)
    Rph, gph = orc.cost_regularizer(orc.REG_L1_PHASE, 1.7, zp, eps=0.0)
    assert abs(Rph - 1.7 * np.sum(np.abs(phi))) < 1e-11
    assert np.abs(np.real(np.conj(zp) * gph)).max() < 1e-13                                # tangential
    assert np.abs(np.abs(gph) - 1.7 / (2 * r)).max() < 1e-12
    assert np.abs(np.angle(gph * np.conj(1j * zp * np.sign(phi)))).max() < 1e-12          # along +i z for phi > 0: descent lowers |phi|
    Rv, gv = orc.cost_regularizer(orc.REG_L1_PHASE, 1.7, np.ones_like(zp), eps=0.0)
    assert Rv == 0.0 and np.abs(gv).max() == 0.0
    z0 = zp.copy(); z0[1, 2, 3] = 0.0
    assert np.isfinite(orc.cost_regularizer(orc.REG_L1_PHASE, 1.7, z0, eps=0.1)[1]).all()
    assert abs(orc.cost_regularizer(orc.REG_L1_PHASE, 2.0, zp, eps=0.3)[0] - 2.0 * np.sum(np.sqrt(phi ** 2 + 0.09))) < 1e-11
    # L1 on the Fourier amplitudes per slice (R26c), sizes that are no power of two: a constant slice and a plane wave have ONE
    # non-zero coefficient of modulus ny nx |c|; a delta has ny nx coefficients of modulus |c|; in general the amplitudes are
    # numpy's fft2 (a library routine); the gradient of a one-peak spectrum is (w / 2) times the unit-modulus wave itself
    yy, xx = np.meshgrid(np.arange(ny), np.arange(nx), indexing="ij")
    c = 0.8 - 0.6j
    const = np.full((S, ny, nx), c)
    assert abs(orc.cost_regularizer(orc.REG_L1_FOURIER, 1.3, const, eps=0.0)[0] - 1.3 * S * ny * nx * abs(c)) < 1e-9
    wave = c * np.exp(2j * np.pi * (2 * xx / nx + 3 * yy / ny))[None].repeat(S, 0)
    assert abs(orc.cost_regularizer(orc.REG_L1_FOURIER, 1.3, wave, eps=0.0)[0] - 1.3 * S * ny * nx * abs(c)) < 1e-9
    # gradient with a small eps (at eps = 0 the rounding noise of the empty coefficients has an arbitrary phase): F^H of
    # (w/2) Z / sqrt(|Z|^2 + eps^2) at the one peak = (w/2) exp(i arg c) x the unit wave, the other coefficients ~1e-12
    gw = orc.cost_regularizer(orc.REG_L1_FOURIER, 1.3, wave, eps=1e-3)[1]
    assert np.abs(gw - 0.65 * wave / abs(c)).max() < 1e-8
    delta = np.zeros((S, ny, nx), complex); delta[:, 2, 4] = c
    assert abs(orc.cost_regularizer(orc.REG_L1_FOURIER, 1.3, delta, eps=0.0)[0] - 1.3 * S * ny * nx * abs(c)) < 1e-9
    Rg = orc.cost_regularizer(orc.REG_L1_FOURIER, 0.7, z, eps=0.25)[0]
    assert abs(Rg - 0.7 * np.sum(np.sqrt(np.abs(np.fft.fft2(z, axes=(1, 2))) ** 2 + 0.0625))) < 1e-9 * Rg
    # Wirtinger gradient against central finite differences: dR = 2 Re sum conj(g) dz, for every kind; grad is ADDED into
    for kind in range(8):
        d = crandn(S, ny, nx); h = 1e-6; g0 = crandn(S, ny, nx)
        R, g = orc.cost_regularizer(kind, 0.9, z, ref=1.0, eps=0.05, grad=g0)
        Rp = orc.cost_regularizer(kind, 0.9, z + h * d, ref=1.0, eps=0.05)[0]
        Rm = orc.cost_regularizer(kind, 0.9, z - h * d, ref=1.0, eps=0.05)[0]
        assert abs((Rp - Rm) / (2 * h) - 2 * np.real(np.sum(np.conj(g - g0) * d))) < 1e-6 * max(1.0, abs(R)), kind


def test_constraints_clamp_mask_blur():
    S, ny, nx = 6, 9, 10
    z = crandn(S, ny, nx)
    c = orc.apply_constraint(orc.CON_AMPLITUDE_CLAMP, z, 0.5, 1.2)
    assert np.abs(c).min() >= 0.5 - 1e-12 and np.abs(c).max() <= 1.2 + 1e-12
    assert np.abs(np.angle(c * np.conj(z))).max() < 1e-12                                  # phase kept
    inside = (np.abs(z) >= 0.5) & (np.abs(z) <= 1.2)
    assert np.array_equal(c[inside], z[inside]) and inside.any() and (~inside).any()
    mask = (RNG.uniform(size=(ny, nx)) > 0.4).astype(float)
    assert np.array_equal(orc.apply_constraint(orc.CON_SUPPORT_MASK, z, mask=mask), z * mask[None])
    # Gaussian blurs: constants are preserved up to the edges (no wrap-around, renormalised taps)
    k = 2.0 - 1.5j
    for kind, sig in ((orc.CON_LAYER_BLUR, 0.8), (orc.CON_LOWPASS, 1.1)):
        assert np.abs(orc.apply_constraint(kind, np.full((S, ny, nx), k), sig) - k).max() < 1e-14
    # interior delta response = normalised Gaussian taps; nothing leaks from the top layer to the bottom one
    sig = 0.8; R = int(np.ceil(4 * sig)); w = np.exp(-np.arange(-R, R + 1) ** 2 / (2 * sig ** 2))
    S2 = 2 * R + 3; d = np.zeros((S2, 2, 2), complex); d[R + 1] = 1.0
    out = orc.apply_constraint(orc.CON_LAYER_BLUR, d, sig)
    # row p of the blur matrix is w_{q-p} / (sum of the taps of p that fall inside): the column of the centre pixel
    col = np.array([w[(R + 1 - p) + R] / sum(w[t + R] for t in range(-R, R + 1) if 0 <= p + t < S2) if abs(R + 1 - p) <= R else 0.0 for p in range(S2)])
    assert np.abs(out[:, 0, 0] - col).max() < 1e-14
    top = np.zeros((12, 1, 1), complex); top[0] = 1.0
    assert np.abs(orc.apply_constraint(orc.CON_LAYER_BLUR, top, sig)[-1]).max() == 0.0     # periodic filtering would leak here
    # in-plane low pass is separable: delta -> outer product of the two 1-D responses; layers do not mix
    d2 = np.zeros((2, 15, 15), complex); d2[0, 7, 7] = 1.0
    o2 = orc.apply_constraint(orc.CON_LOWPASS, d2, 1.1)
    R2 = int(np.ceil(4 * 1.1)); w2 = np.exp(-np.arange(-R2, R2 + 1) ** 2 / (2 * 1.1 ** 2))
    def col1(n, c):
        return np.array([w2[(c - p) + R2] / sum(w2[t + R2] for t in range(-R2, R2 + 1) if 0 <= p + t < n) if abs(c - p) <= R2 else 0.0 for p in range(n)])
    assert np.abs(o2[0] - np.outer(col1(15, 7), col1(15, 7))).max() < 1e-14 and np.abs(o2[1]).max() == 0.0


def test_adam_closed_forms():
    z = crandn(4, 5); g = crandn(4, 5)
    # first step, eps -> 0: bias correction makes m^ = g, v^ = |g|^2, so the step is -lr g/|g| whatever beta1, beta2
    z1, m1, v1 = orc.adam_update(z, g, np.zeros_like(z), np.zeros(z.shape), lr=0.01, b1=0.9, b2=0.999, eps=0.0, t=1)
    assert np.abs((z1 - z) + 0.01 * g / np.abs(g)).max() < 1e-13
    assert np.abs(m1 - 0.1 * g).max() < 1e-15 and np.abs(v1 - 0.001 * np.abs(g) ** 2).max() < 1e-15
    # constant gradient: every later step is the same -lr g/|g|
    zc, mc, vc = z1, m1, v1
    for t in range(2, 6):
        zc, mc, vc = orc.adam_update(zc, g, mc, vc, lr=0.01, eps=0.0, t=t)
    assert np.abs((zc - z) + 5 * 0.01 * g / np.abs(g)).max() < 1e-12
    # sign flip of the gradient at step 2: m^ = (0.09 - 0.1) g / 0.19, v^ = |g|^2
    z2, _, _ = orc.adam_update(z1, -g, m1, v1, lr=0.01, eps=0.0, t=2)
    assert np.abs((z2 - z1) - 0.01 * (0.01 / 0.19) * g / np.abs(g)).max() < 1e-13
    # real variables (positions): per-component form
    x = RNG.standard_normal(7); gx = RNG.standard_normal(7)
    x1, _, _ = orc.adam_update(x, gx, np.zeros(7), np.zeros(7), lr=0.1, eps=0.0, t=1)
    assert np.abs((x1 - x) + 0.1 * np.sign(gx)).max() < 1e-13
    # eps enters as sqrt(v^) + eps
    x1e, _, _ = orc.adam_update(x, gx, np.zeros(7), np.zeros(7), lr=0.1, eps=0.5, t=1)
    assert np.abs((x1e - x) + 0.1 * gx / (np.abs(gx) + 0.5)).max() < 1e-13


def test_constraints_fourier_support_and_phase_deramp():
    # reciprocal-space probe support: z <- Finv(mask F z), against numpy.fft; all-ones = identity; 0/1 mask idempotent
    n = 16
    z = crandn(2, n, n)
    s = np.where(np.arange(n) < n // 2, np.arange(n), np.arange(n) - n)
    mask = ((s[:, None] ** 2 + s[None, :] ** 2) <= 25).astype(float)
    out = orc.apply_constraint(orc.CON_SUPPORT_MASK_FOURIER, z, mask=mask)
    assert np.abs(out - np.fft.ifft2(np.fft.fft2(z) * mask[None])).max() < 1e-12
    assert np.abs(orc.apply_constraint(orc.CON_SUPPORT_MASK_FOURIER, z, mask=np.ones((n, n))) - z).max() < 1e-13
    assert np.abs(orc.apply_constraint(orc.CON_SUPPORT_MASK_FOURIER, out, mask=mask) - out).max() < 1e-13
    # phase deramp (reading R29): a pure ramp becomes a positive real constant; an object without a ramp is
    # unchanged; the result does not depend on a ramp put on top (the ambiguity of PAPER.md:125 is removed)
    ny, nx = 12, 15
    y, x = np.meshgrid(np.arange(ny), np.arange(nx), indexing="ij")
    ramp = np.exp(1j * (0.7 + 0.21 * y - 0.13 * x))
    flat = orc.apply_constraint(orc.CON_PHASE_DERAMP, (2.5 * ramp)[None])
    assert np.abs(flat - 2.5).max() < 1e-12
    amp = 1.0 + 0.3 * RNG.uniform(size=(1, ny, nx))                            # real positive object: nothing to remove
    assert np.abs(orc.apply_constraint(orc.CON_PHASE_DERAMP, amp.astype(complex)) - amp).max() < 1e-12
    obj = amp * np.exp(1j * 0.2 * np.sin(2 * np.pi * x / nx) * np.cos(2 * np.pi * y / ny))[None]
    d0 = orc.apply_constraint(orc.CON_PHASE_DERAMP, obj)
    d1 = orc.apply_constraint(orc.CON_PHASE_DERAMP, obj * ramp[None])
    assert np.abs(d0 - d1).max() < 1e-12
    assert np.abs(np.abs(d0) - np.abs(obj)).max() < 1e-13                      # a pure phase factor
    # slices are treated one by one
    two = np.concatenate([obj * ramp[None], obj * np.conj(ramp)[None]])
    d2 = orc.apply_constraint(orc.CON_PHASE_DERAMP, two)
    assert np.abs(d2[0] - d0[0]).max() < 1e-12 and np.abs(d2[1] - d0[0]).max() < 1e-12
