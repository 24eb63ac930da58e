"""FP64 CPU oracle of the extrapolator-table design -- TEST INFRASTRUCTURE ONLY.

The paper designs its filters offline and gives no recipe ("short length filters ... vs
large length filters", :83 "Designing filters itself is optimization problem ... we design the filters
in advance and store it on the disk", refs :179-180).  SURVEY.md 8(c) fixes one, D1-D4, described as
mathematics; this file is that description written out step by step with numpy's FFT on the FULL
periodic N-point grid, taps k = -L..L held at FFT positions k mod N -- no half-grid folding, no cosine
matrices.  It is the checker of the device design `pdm_design_table` (tests/test_gpu_design.py) and is
itself pinned by tests/test_design_oracle_pins.py:
  G-P1  its two steps (taps -> response, response -> truncated symmetric taps) against pure-Python
        direct sums of the DFT definition on a tiny grid,
  G-P2  per-tap agreement with the structurally different half-grid cosine statement of the same recipe
        in pdm_inputs/filters.py (<= 1e-12 of the row maximum, before rounding),
  G-P3  the designed response against the analytic one-way phase shift exp(i sqrt(u^2 - (r kappa)^2))
        on the passband, within the D4 figures, on kappa points that are not design-grid points,
  G-P4  |H| <= 1 + 1e-6 after rounding, bitwise symmetry, and one more D2 sweep moves no tap by more
        than the stated residual.
Nothing here is imported by the product package or by pdm_inputs; it shares no code with either.

Conventions (R3/R4, pdm.h): u_j = j*du; H(kappa) = sum_k W_k exp(-i k kappa); target
    D(kappa) = exp(+i sqrt(u^2 - (r kappa)^2))   for |r kappa| <= u   (propagating)
             = exp(  - sqrt((r kappa)^2 - u^2))  otherwise             (evanescent),   r = dz/dx;
table[j][L+k] = W_k(u_j).
"""
from __future__ import annotations

import numpy as np

N_GRID = 2048                 # D1
N_ITER = 200                  # D2 ("~150-300 times")
PASSBAND_ANGLE_DEG = 55.0     # D2
KAPPA_CAP = 0.8 * np.pi       # D2
STOP_CAP = 0.9995             # D2
N_CHECK = 16384               # D3 (">= 16384 kappa-points")
ROUND_MARGIN = 4e-7           # D3: head-room so that the ROUNDED taps still satisfy |H| <= 1 + 1e-6 (pdm.h)


def grid_kappa(n_grid: int = N_GRID) -> np.ndarray:
    """D1: the periodic grid kappa_m = 2 pi m / N at FFT positions (m >= N/2 stands for m - N)."""
    return 2.0 * np.pi * np.fft.fftfreq(n_grid)


def target(u: float, kappa: np.ndarray, r: float) -> np.ndarray:
    """D1 / R4: exact one-way phase-shift response D(kappa; u, r) for one table entry."""
    arg = u * u - (r * kappa) ** 2
    out = np.empty(kappa.shape, dtype=np.complex128)
    prop = arg >= 0.0
    out[prop] = np.exp(1j * np.sqrt(arg[prop]))
    out[~prop] = np.exp(-np.sqrt(-arg[~prop]))
    return out


def passband_edge(u: float, r: float, angle_deg: float = PASSBAND_ANGLE_DEG, kappa_cap: float = KAPPA_CAP) -> float:
    """D2: |kappa| <= min((u/r) sin(angle), kappa_cap)."""
    return min((u / r) * np.sin(np.deg2rad(angle_deg)), kappa_cap)


def response_to_taps(H: np.ndarray, L: int) -> np.ndarray:
    """D2 "inverse DFT; keep taps |k| <= L only; average h_k and h_-k".  H: [N] at FFT positions.
    Returns h: [N] at FFT positions (h[k] = W_k, h[N-k] = W_-k), zero for L < k < N-L."""
    n = H.shape[0]
    h = np.fft.ifft(H)
    h[L + 1:n - L] = 0.0
    for k in range(1, L + 1):
        mean = 0.5 * (h[k] + h[n - k])
        h[k] = mean
        h[n - k] = mean
    return h


def taps_to_response(h: np.ndarray) -> np.ndarray:
    """D2 "DFT": H_m = sum_k h_k exp(-2 pi i k m / N)."""
    return np.fft.fft(h)


def project(H: np.ndarray, D: np.ndarray, in_pass: np.ndarray, stop_cap: float = STOP_CAP) -> np.ndarray:
    """D2: inside the passband reset H <- D; outside it, where |H| > stop_cap, rescale to stop_cap."""
    out = H.copy()
    mag = np.abs(H)
    over = (~in_pass) & (mag > stop_cap)
    out[over] = H[over] * (stop_cap / mag[over])
    out[in_pass] = D[in_pass]
    return out


def design_row_taps(u: float, L: int, r: float = 1.0, n_iter: int = N_ITER, n_grid: int = N_GRID,
                    angle_deg: float = PASSBAND_ANGLE_DEG, kappa_cap: float = KAPPA_CAP,
                    stop_cap: float = STOP_CAP) -> np.ndarray:
    """D1 + D2 for one entry: complex128 taps W_-L..W_L (before D3).  "start H = D; repeat { inverse
    DFT, truncate, symmetrise; DFT; project }; finish on the truncation step"."""
    kappa = grid_kappa(n_grid)
    D = target(u, kappa, r)
    in_pass = np.abs(kappa) <= passband_edge(u, r, angle_deg, kappa_cap)
    H = D
    for _ in range(n_iter):
        h = response_to_taps(H, L)
        H = project(taps_to_response(h), D, in_pass, stop_cap)
    h = response_to_taps(H, L)                                   # finish on the truncation step
    return np.concatenate([h[n_grid - L:], h[:L + 1]]) if L > 0 else h[:1].copy()


def response(taps: np.ndarray, kappa: np.ndarray) -> np.ndarray:
    """H(kappa) = sum_{k=-L..L} W_k exp(-i k kappa) for taps W_-L..W_L, by the definition."""
    L = (taps.shape[-1] - 1) // 2
    k = np.arange(-L, L + 1, dtype=np.float64)
    return np.asarray(taps, dtype=np.complex128) @ np.exp(-1j * k[:, None] * np.asarray(kappa, dtype=np.float64)[None, :])


def normalise(taps: np.ndarray, n_check: int = N_CHECK) -> np.ndarray:
    """D3: evaluate |H| on n_check points of [0, pi] (H is even); divide all taps by
    max(1, max|H|) * (1 + ROUND_MARGIN)."""
    kappa = np.pi * np.arange(n_check, dtype=np.float64) / (n_check - 1)
    peak = np.abs(response(taps, kappa)).max()
    return taps / (max(peak, 1.0) * (1.0 + ROUND_MARGIN))


def design_table_taps(ntab: int, ntaps: int, du: float, r: float = 1.0, **opts) -> np.ndarray:
    """D1-D3 for every entry, complex128 [ntab, ntaps], before the rounding to complex64."""
    if ntaps < 1 or ntaps % 2 != 1:
        raise ValueError("ntaps must be odd")
    L = (ntaps - 1) // 2
    n_check = opts.pop("n_check", N_CHECK)
    out = np.empty((ntab, ntaps), dtype=np.complex128)
    for j in range(ntab):
        out[j] = normalise(design_row_taps(j * float(du), L, r, **opts), n_check)
    return out


def design_table(ntab: int, ntaps: int, du: float, r: float = 1.0, **opts) -> np.ndarray:
    """D1-D3 + the cast: complex64 [ntab, ntaps] in the layout pdm_create reads, W_-k == W_k bitwise
    (the symmetrised FP64 pairs are equal before rounding; the mirror below makes it explicit)."""
    t = design_table_taps(ntab, ntaps, du, r, **opts).astype(np.complex64)
    L = (ntaps - 1) // 2
    for k in range(1, L + 1):
        t[:, L - k] = t[:, L + k]
    return np.ascontiguousarray(t)
