"""Extrapolator-table design for the harness (setup, not hot path).

The paper designs its FIR extrapolators offline ("we design the filters in advance and
store it on the disk") and treats the design as an optimisation problem
(refs [20][21] :179-180) without giving a recipe.  The table is therefore an
INPUT to both the oracle and the CUDA path; parity never depends on its quality.  This
module holds the recipe SURVEY.md §8(c) D1-D4 proposes (a projections-onto-convex-sets
style iteration, the family of ref [21]) written from its mathematical description.

Nothing in here is imported by `oracle/` or by the CUDA package's compute path; it only
produces arrays that are handed, byte-identical, to both.

Conventions (readings R3/R4):
  * entry j of the table belongs to the normalised wavenumber  u_j = j * du,
    u = omega * dz / v  (dimensionless, radians of vertical phase per depth step);
  * the target response on the periodic grid kappa = k_x * dx in [-pi, pi) is
        D(kappa) = exp(+i * sqrt(u^2 - (r kappa)^2))      |r kappa| <= u   (propagating)
                 = exp(   - sqrt((r kappa)^2 - u^2))      otherwise         (evanescent)
    with r = dz / dx;
  * table[j, L + k] = W_k(u_j), k = -L..L, and W_k == W_{-k} bit for bit.
"""
from __future__ import annotations

import numpy as np

PASSBAND_ANGLE_DEG = 55.0      # D2: passband |kappa| <= (u/r) sin(55 deg)
KAPPA_CAP = 0.8 * np.pi        # D2: anti-alias cap of the passband
STOP_CAP = 0.9995              # D2: |H| ceiling outside the passband during iteration
NGRID = 2048                   # D1: periodic kappa grid of the iteration
NCHECK = 16384                 # D3: kappa points of the stability check (0..pi, H is even)


def target_response(u: np.ndarray, kappa: np.ndarray, r: float) -> np.ndarray:
    """D1: exact one-way phase-shift response D(kappa; u, r); shape [len(u), len(kappa)]."""
    u = np.asarray(u, dtype=np.float64)[:, None]
    rk2 = (r * np.asarray(kappa, dtype=np.float64)[None, :]) ** 2
    arg = u * u - rk2
    prop = arg >= 0.0
    root = np.sqrt(np.abs(arg))
    return np.where(prop, np.exp(1j * root), np.exp(-root))


def response_on_grid(half_taps: np.ndarray, ncheck: int = NCHECK) -> np.ndarray:
    """H_j(kappa) = W_0 + 2 sum_{k>=1} W_k cos(k kappa) on kappa = pi*m/(ncheck-1), m=0..ncheck-1.

    `half_taps` is [ntab, L+1] (k = 0..L) of a symmetric filter; the response of a symmetric
    filter is even in kappa, so [0, pi] covers the whole period.
    """
    half = np.asarray(half_taps, dtype=np.complex128)
    Lp1 = half.shape[1]
    kappa = np.pi * np.arange(ncheck, dtype=np.float64) / (ncheck - 1)
    cosm = np.cos(np.arange(Lp1, dtype=np.float64)[:, None] * kappa[None, :])
    cosm[1:] *= 2.0
    return half @ cosm


def design_half_taps(ntab: int, ntaps: int, du: float, r: float = 1.0,
                     n_iter: int = 200) -> np.ndarray:
    """D1-D3 in FP64: complex128 [ntab, L+1] half taps W_0..W_L, normalised, before the cast."""
    if ntaps % 2 != 1 or ntaps < 1:
        raise ValueError("ntaps must be odd")
    L = (ntaps - 1) // 2
    if 2 * L + 1 > NGRID:
        raise ValueError("filter longer than the design grid")
    u = np.arange(ntab, dtype=np.float64) * float(du)
    # D and every iterate are even in kappa (symmetric taps), so the periodic NGRID-point
    # DFT pair reduces to cosine sums over the half grid kappa_m = 2 pi m / NGRID, m = 0..NGRID/2:
    #   H_m = W_0 + 2 sum_{k=1..L} W_k cos(k kappa_m)
    #   W_k = (1/NGRID) [ H_0 + (-1)^k H_{NGRID/2} + 2 sum_{m=1}^{NGRID/2-1} H_m cos(k kappa_m) ]
    # The second line IS "inverse DFT, keep |k| <= L, average W_k and W_-k".
    M = NGRID // 2
    kappa = 2.0 * np.pi * np.arange(M + 1, dtype=np.float64) / NGRID
    D = target_response(u, kappa, r)
    pass_edge = np.minimum((u / r) * np.sin(np.deg2rad(PASSBAND_ANGLE_DEG)), KAPPA_CAP)
    passband = kappa[None, :] <= pass_edge[:, None]
    kk = np.arange(L + 1, dtype=np.float64)
    fwd = np.cos(kk[:, None] * kappa[None, :])            # [L+1, M+1]
    fwd[1:] *= 2.0
    inv = np.cos(kappa[:, None] * kk[None, :]) * 2.0      # [M+1, L+1]
    inv[0, :] = 1.0
    inv[M, :] = np.cos(np.pi * kk)
    inv /= NGRID

    half = D @ inv                                         # truncate (+ symmetrise)
    for _ in range(n_iter):
        H = half @ fwd
        mag = np.abs(H)
        scale = np.where((~passband) & (mag > STOP_CAP), STOP_CAP / np.maximum(mag, 1e-300), 1.0)
        H = np.where(passband, D, H * scale)
        half = H @ inv                                     # finish on the truncation step

    # D3: normalise so that max |H| <= 1, then round to complex64 and re-check
    mag_max = np.abs(response_on_grid(half)).max(axis=1)
    return half / (np.maximum(mag_max, 1.0) * (1.0 + 4e-7))[:, None]


def design_table(ntab: int, ntaps: int, du: float, r: float = 1.0,
                 n_iter: int = 200) -> np.ndarray:
    """Design the full table: complex64 [ntab, ntaps], exactly symmetric, |H| <= 1 (D1-D4)."""
    L = (ntaps - 1) // 2
    half32 = design_half_taps(ntab, ntaps, du, r, n_iter).astype(np.complex64)
    table = np.empty((ntab, ntaps), dtype=np.complex64)
    table[:, L] = half32[:, 0]
    for k in range(1, L + 1):
        table[:, L + k] = half32[:, k]
        table[:, L - k] = half32[:, k]
    return np.ascontiguousarray(table)


def mcclellan_table(table1d: np.ndarray) -> np.ndarray:
    """2-D extrapolators for the 3-D variant ("requires 2-D filters as extrapolators"; ref :177)
    from a symmetric 1-D table by the McClellan transformation: with the 1-D response written as
        H(kappa) = W_0 + 2 sum_n W_n cos(n kappa) = sum_n a_n T_n(cos kappa),  a_0 = W_0, a_n = 2 W_n,
    cos kappa is replaced by the 9-point approximation of cos sqrt(kx^2 + ky^2),
        M(kx, ky) = -1 + (1 + cos kx)(1 + cos ky) / 2
    (3 x 3 kernel: centre -1/2, edge neighbours 1/4, corners 1/8), and the Chebyshev recurrence
    T_n = 2 M T_{n-1} - T_{n-2} is run on 2-D kernels (convolutions).  Exact along the axes (M(kx, 0) =
    cos kx), circularly symmetric to O(k^4) elsewhere.  Returns complex64 [ntab, ntaps, ntaps], symmetric in
    kx and in ky bit for bit, |H2(kx, ky)| = |H(arccos M)| <= max|H| (stability carries over).
    Input generator only: both the oracle and the CUDA path receive the table as an array."""
    t = np.asarray(table1d)
    ntab, ntaps = t.shape
    L = (ntaps - 1) // 2
    a = t[:, L:].astype(np.complex128).copy()
    a[:, 1:] *= 2.0
    m = np.array([[0.125, 0.25, 0.125], [0.25, -0.5, 0.25], [0.125, 0.25, 0.125]])

    def conv_m(k):                                   # k: [2L+1, 2L+1] kernel centred at (L, L); support grows by 1
        out = np.zeros_like(k)
        for dy in (-1, 0, 1):
            for dx in (-1, 0, 1):
                w = m[dy + 1, dx + 1]
                ys = slice(max(0, dy), ntaps + min(0, dy)); yd = slice(max(0, -dy), ntaps + min(0, -dy))
                xs = slice(max(0, dx), ntaps + min(0, dx)); xd = slice(max(0, -dx), ntaps + min(0, -dx))
                out[ys, xs] += w * k[yd, xd]
        return out

    cheb = [np.zeros((ntaps, ntaps)), None]
    cheb[0][L, L] = 1.0
    kernels = [cheb[0]]
    if L >= 1:
        kernels.append(conv_m(cheb[0]))
    for n in range(2, L + 1):
        kernels.append(2.0 * conv_m(kernels[n - 1]) - kernels[n - 2])
    basis = np.stack(kernels)                        # [L+1, ntaps, ntaps], real
    out = np.tensordot(a, basis, axes=(1, 0)).astype(np.complex64)
    q = out[:, L:, L:]                               # enforce the double mirror symmetry bit for bit
    out = np.concatenate([np.concatenate([q[:, :0:-1, :0:-1], q[:, :0:-1, :]], 2),
                          np.concatenate([q[:, :, :0:-1], q], 2)], 1)
    return np.ascontiguousarray(out)


def delta_table(ntab: int, ntaps: int) -> np.ndarray:
    """Identity extrapolator (W_0 = 1, every other tap 0) for every entry: pin P1 input."""
    t = np.zeros((ntab, ntaps), dtype=np.complex64)
    t[:, (ntaps - 1) // 2] = 1.0
    return t


def random_symmetric_table(rng: np.random.Generator, ntab: int, ntaps: int,
                           scale: float = 0.2) -> np.ndarray:
    """Random exactly-symmetric complex64 table (test input; no physical meaning)."""
    L = (ntaps - 1) // 2
    half = (rng.standard_normal((ntab, L + 1)) + 1j * rng.standard_normal((ntab, L + 1)))
    half = (scale * half).astype(np.complex64)
    t = np.empty((ntab, ntaps), dtype=np.complex64)
    t[:, L] = half[:, 0]
    for k in range(1, L + 1):
        t[:, L + k] = half[:, k]
        t[:, L - k] = half[:, k]
    return t
