"""Writes tests/golden/oracle_tiny_case.txt: loss and gradient checksums of the ORACLE on a tiny seeded problem.

The paper prints no numeric worked example for this path ("parity unpinned" for absolute
values), so there is no paper value to store.  This fixture is a change detector for the oracle itself: its numbers
come from oracle/ only (never from the CUDA path) and tests/test_oracle_pins.py::test_golden_oracle_tiny_case
recomputes them.  A commit that changes the oracle's arithmetic must regenerate this file and name, in its message,
the passage of the paper or the DESIGN.md reading that justifies the change.

    python tests/golden/make_golden.py
"""
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)
from oracle import oracle as orc  # noqa: E402


def tiny_case(shift_mode):
    """N=8, 2 modes, 3 slices, 3 overlapping windows, tilt, Poisson loss; inputs from a fixed
    linear-congruential sequence so that the file does not depend on numpy's generators."""
    state = [12345]

    def u():
        state[0] = (1103515245 * state[0] + 12345) % (1 << 31)
        return state[0] / float(1 << 31)

    n, M, S, on = 8, 2, 3, 20
    obj = np.array([np.exp(0.3 * (u() - 0.5) + 1j * 0.8 * (u() - 0.5)) for _ in range(S * on * on)]).reshape(S, on, on).astype(np.complex64)
    probe = np.array([(u() - 0.5) + 1j * (u() - 0.5) for _ in range(M * n * n)]).reshape(M, n, n).astype(np.complex64)
    pos = (np.array([[5.3, 6.1], [6.9, 7.4], [8.2, 5.6]]) * 0.2).astype(np.float32)
    inten = np.array([3.0 * u() for _ in range(3 * n * n)]).reshape(3, n, n).astype(np.float32)
    pb = orc.Problem(n=n, n_modes=M, n_slices=S, obj_ny=on, obj_nx=on, pixel_size=0.2, wavelength=0.05,
                     slice_thickness=[3.0, 3.5, 4.0], tilt_x_mrad=30.0, tilt_y_mrad=-20.0, bandlimit=0.0,
                     loss=orc.LOSS_POISSON, loss_c=0.0, eps=0.3, shift_mode=shift_mode)
    return pb, obj, probe, pos, inten


def checksums(shift_mode):
    pb, obj, probe, pos, inten = tiny_case(shift_mode)
    g = orc.gradient(pb, obj, probe, pos, inten)
    wo = np.cos(np.arange(g["grad_object"].size)).reshape(g["grad_object"].shape)       # fixed weights: index-sensitive sums
    wp = np.cos(np.arange(g["grad_probe"].size)).reshape(g["grad_probe"].shape)
    return [("loss", g["loss"]), ("loss_pos0", g["loss_per_pos"][0]),
            ("gO_wsum_re", float(np.sum(wo * g["grad_object"].real))), ("gO_wsum_im", float(np.sum(wo * g["grad_object"].imag))),
            ("gP_wsum_re", float(np.sum(wp * g["grad_probe"].real))), ("gP_wsum_im", float(np.sum(wp * g["grad_probe"].imag))),
            ("gX_00", g["grad_pos"][0, 0]), ("gX_21", g["grad_pos"][2, 1])]


if __name__ == "__main__":
    out = os.path.join(os.path.dirname(os.path.abspath(__file__)), "oracle_tiny_case.txt")
    with open(out, "w") as f:
        f.write("# written by tests/golden/make_golden.py from oracle/ only; see that file's docstring\n")
        for mode, name in ((0, "fourier_probe"), (1, "bilinear_object")):
            for k, v in checksums(mode):
                f.write(f"{name} {k} {float(v):.15e}\n")
    print(open(out).read())
