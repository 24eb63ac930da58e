"""FP64 oracle of the time -> frequency transform of the input section.

TEST INFRASTRUCTURE ONLY.  PAPER.md:51 and Alg. 1 (:58): the zero-offset section is Fourier
transformed along the TIME axis only, trace by trace, giving the f-x section that the
depth loop consumes.  With the sign convention of reading R4 (data = sum_w P(w) e^{+iwt}, i.e.
P0(w,x) carries e^{-iwt(x)}), the transform is the plain definition, written out:

    P0[j][x] = sum_{n=0}^{nt-1} d[n][x] * exp(-2*pi*i * bins[j] * n / nt)        (no scaling)

for the selected DFT bins only (omega_j = 2*pi*bins[j]/(nt*dt)).  The exponent is reduced with
exact integer arithmetic ((bins[j]*n) mod nt) before the call to exp; the sum over n is a FP64
matrix product (a library primitive used as one step, no blocking or reordering of our own).
"""
from __future__ import annotations

import numpy as np


def section_to_fx(section: np.ndarray, bins: np.ndarray, chunk: int = 64) -> np.ndarray:
    """section: real [nt][nx] (time-major); bins: int [nw] in [0, nt/2].  Returns complex128 [nw][nx]."""
    d = np.asarray(section, dtype=np.float64)
    nt, nx = d.shape
    bins = np.asarray(bins, dtype=np.int64)
    if bins.ndim != 1 or (bins < 0).any() or (bins > nt // 2).any():
        raise ValueError("bins must be a 1-D array of DFT bins in [0, nt/2]")
    n = np.arange(nt, dtype=np.int64)
    out = np.empty((bins.size, nx), dtype=np.complex128)
    for j0 in range(0, bins.size, chunk):
        m = (bins[j0:j0 + chunk, None] * n[None, :]) % nt          # exact
        E = np.exp(-2j * np.pi * m.astype(np.float64) / nt)
        out[j0:j0 + chunk] = E @ d
    return out
