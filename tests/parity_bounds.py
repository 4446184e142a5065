"""The parity bar, in one place (DESIGN.md section 6 derives the numbers).

  TOL_SMALL / TOL_LARGE   north_star's tolerance: relative L2 error <= 2e-5 for n <= 20, <= 1e-4 up to n = 33.
  REG_L2                  regression bound near the measured level (1.3e-7 ... 4e-7 on a B200): a change that
                          costs an order of magnitude of accuracy fails although it would still meet north_star.
  MAXABS_FRAC             element bound: max |gpu - ref| <= MAXABS_FRAC * max |ref|.  A relative-L2 bound alone lets a
                          few wrong amplitudes through at large n (one amplitude of a 2^30 Gaussian state carries
                          2^-30 of the energy); a mis-addressed or dropped amplitude is off by about its own
                          modulus, i.e. >= 1e-1 * max |ref| for the inputs used here, four orders above this bound,
                          while rounding stays below 1e-6 * max |ref|.
"""
from __future__ import annotations

import math

TOL_SMALL = 2e-5
TOL_LARGE = 1e-4
REG_L2 = 2e-6
MAXABS_FRAC = 1e-5


def tol_for(n: int) -> float:
    return TOL_SMALL if n <= 20 else TOL_LARGE


def assert_parity_numpy(got, ref, n: int, what=""):
    """got, ref: numpy complex arrays (ref in double)."""
    import numpy as np

    d = got.astype(np.complex128) - ref
    rel = float(np.linalg.norm(d) / np.linalg.norm(ref))
    mx = float(np.max(np.abs(d)))
    rmax = float(np.max(np.abs(ref)))
    assert rel <= tol_for(n), (what, "north_star tolerance", rel)
    assert rel <= REG_L2, (what, "regression bound", rel)
    assert mx <= MAXABS_FRAC * rmax, (what, "element bound", mx, rmax)
    return rel, mx / rmax


class ChunkedParity:
    """Accumulates |d|^2, |ref|^2, max |d|, max |ref| over chunks that live on the GPU (torch, float64)."""

    def __init__(self):
        self.num = 0.0
        self.den = 0.0
        self.mx = 0.0
        self.rmax = 0.0

    def add(self, got, ref):
        import torch

        d = got.to(torch.complex128) - ref
        self.num += float((d.real * d.real + d.imag * d.imag).sum().item())
        self.den += float((ref.real * ref.real + ref.imag * ref.imag).sum().item())
        self.mx = max(self.mx, float(d.abs().max().item()))
        self.rmax = max(self.rmax, float(ref.abs().max().item()))

    def check(self, n: int, what=""):
        rel = math.sqrt(self.num / self.den)
        assert rel <= tol_for(n), (what, "north_star tolerance", rel)
        assert rel <= REG_L2, (what, "regression bound", rel)
        assert self.mx <= MAXABS_FRAC * self.rmax, (what, "element bound", self.mx, self.rmax)
        return rel, self.mx / self.rmax
