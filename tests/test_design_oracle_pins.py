"""Pins G-P1..G-P4 of oracle/design_oracle.py (the FP64 statement of the table design D1-D4, SURVEY.md
8(c), refs :179-180) -- all CPU, none touches the CUDA path.

Why these: the design is an iteration with no closed-form answer, so the oracle follows the recipe step
by step and is pinned (a) step by step against the DFT DEFINITION written as pure-Python sums on a tiny
grid (G-P1), (b) as a whole against a structurally different statement of the same recipe (half-grid
cosine sums, pdm_inputs/filters.py) to 1e-12 (G-P2), (c) against what the filter is FOR -- the analytic
one-way phase shift on the passband, which no line of the recipe code is shared with (G-P3), and (d) by
the invariants D3 promises (G-P4).  A dropped factor, a wrong sign of the phase, a mis-indexed or
mis-scaled tap, a wrong passband edge or a missing symmetrisation fails at least one of them; e.g. the
"outermost tap 3 % low in every truncation" mutant fails G-P1 and G-P2 in whichever file it sits.
"""
import cmath
import math

import numpy as np
import pytest

from oracle import design_oracle as do
from pdm_inputs import filters


# ---------------------------------------------------------------- G-P1 the two steps vs the DFT definition
@pytest.mark.parametrize("n,L", [(16, 2), (12, 5), (8, 0), (10, 4)])
def test_GP1_steps_match_direct_sums_of_the_definition(n, L):
    rng = np.random.default_rng(n * 31 + L)
    H = rng.standard_normal(n) + 1j * rng.standard_normal(n)          # NOT even: symmetrisation has work to do
    # inverse DFT by the definition, h_k = (1/N) sum_m H_m e^{+2 pi i k m / N}, k = -L..L
    raw = {k: sum(H[m] * cmath.exp(2j * math.pi * k * m / n) for m in range(n)) / n for k in range(-L, L + 1)}
    want = np.zeros(n, dtype=np.complex128)
    for k in range(-L, L + 1):
        want[k % n] = 0.5 * (raw[k] + raw[-k])                        # average h_k and h_-k
    got = do.response_to_taps(H.copy(), L)
    assert np.abs(got - want).max() <= 1e-15 * n
    assert np.count_nonzero(got) <= 2 * L + 1
    # DFT by the definition, H_m = sum_k h_k e^{-2 pi i k m / N}, taps at positions k mod N
    back = np.array([sum(want[k % n] * cmath.exp(-2j * math.pi * k * m / n) for k in range(-L, L + 1))
                     for m in range(n)])
    assert np.abs(do.taps_to_response(want) - back).max() <= 1e-14 * n
    # and `response` (used by D3 and by G-P3) is the same sum at arbitrary kappa
    taps = np.array([want[k % n] for k in range(-L, L + 1)])
    kap = rng.uniform(-math.pi, math.pi, 7)
    direct = np.array([sum(taps[L + k] * cmath.exp(-1j * k * x) for k in range(-L, L + 1)) for x in kap])
    assert np.abs(do.response(taps, kap) - direct).max() <= 1e-14 * n


def test_GP1_grid_target_and_projection():
    n = 32
    kap = do.grid_kappa(n)
    assert kap[0] == 0.0 and np.isclose(kap[1], 2 * math.pi / n) and np.isclose(kap[n - 1], -2 * math.pi / n)
    assert np.isclose(abs(kap[n // 2]), math.pi)
    u, r = 1.3, 0.7
    D = do.target(u, kap, r)
    for m in range(n):                                                # R4, branch by branch, scalar arithmetic
        a = u * u - (r * kap[m]) ** 2
        want = cmath.exp(1j * math.sqrt(a)) if a >= 0 else math.exp(-math.sqrt(-a))
        assert abs(D[m] - want) <= 1e-15
    assert np.all(np.abs(D) <= 1.0 + 1e-15) and D[0] == cmath.exp(1j * u)
    assert D[1].imag > 0                                              # +i: downward continuation (R4)
    edge = do.passband_edge(u, r)
    assert np.isclose(edge, (u / r) * math.sin(math.radians(55.0)))
    assert do.passband_edge(50.0, 1.0) == 0.8 * math.pi               # the anti-alias cap
    in_pass = np.abs(kap) <= edge
    H = 1.5 * np.exp(1j * np.linspace(0, 3, n))
    P = do.project(H, D, in_pass)
    assert np.array_equal(P[in_pass], D[in_pass])
    assert np.allclose(np.abs(P[~in_pass]), 0.9995) and np.allclose(np.angle(P[~in_pass]), np.angle(H[~in_pass]))
    small = 0.5 * H
    assert np.array_equal(do.project(small, D, in_pass)[~in_pass], small[~in_pass])


# ---------------------------------------------------------------- G-P2 two statements of the recipe agree
@pytest.mark.parametrize("ntab,ntaps,du,r", [(24, 25, 4.2 / 23, 1.0), (16, 15, 3.2 / 15, 1.0), (9, 9, 3.0 / 8, 0.5),
                                             (6, 51, 4.0 / 5, 1.0), (4, 1, 0.4, 1.0)])
def test_GP2_full_grid_fft_statement_equals_half_grid_cosine_statement(ntab, ntaps, du, r):
    L = (ntaps - 1) // 2
    a = do.design_table_taps(ntab, ntaps, du, r)
    b = filters.design_half_taps(ntab, ntaps, du, r)
    scale = np.abs(b).max(axis=1, keepdims=True)
    assert (np.abs(a[:, L:] - b) / scale).max() <= 1e-12
    assert np.array_equal(a[:, :L][:, ::-1], a[:, L + 1:])            # symmetric already in FP64
    t = do.design_table(ntab, ntaps, du, r)
    f = filters.design_table(ntab, ntaps, du, r)
    assert t.dtype == np.complex64 and t.shape == (ntab, ntaps)
    assert (np.abs(t.astype(np.complex128) - f) / scale).max() <= 2.0 ** -23


# ---------------------------------------------------------------- G-P3 what the filter is for
@pytest.mark.parametrize("ntaps,ntab,umax,bound_all,bound_mid", [
    (25, 48, 4.2, 3.5e-2, 2.0e-2),        # D4: <= 2.5e-2 at L = 12 and tiny u before D3's g <= 1.006; 1e-3..8e-3 typical
    (51, 32, 4.2, 1.2e-2, 7.0e-3),        # D4: 3e-4..3e-3 for L = 25
    (15, 32, 3.3, 4.8e-2, 4.8e-2),
])
def test_GP3_passband_response_is_the_one_way_phase_shift(ntaps, ntab, umax, bound_all, bound_mid):
    """max over the passband of |H_j(kappa) - exp(+i sqrt(u_j^2 - kappa^2))| per row, on random kappa that
    are not design-grid points.  (A conjugated table misses by ~2 sin(u); a passband edge of 65 degrees or
    a dropped D2 projection by several times the bound.)"""
    rng = np.random.default_rng(ntaps)
    du = umax / (ntab - 1)
    taps = do.design_table_taps(ntab, ntaps, du, 1.0)
    for j in range(1, ntab):
        u = j * du
        edge = do.passband_edge(u, 1.0)
        kap = rng.uniform(-edge, edge, 400)
        exact = np.exp(1j * np.sqrt(u * u - kap * kap))
        err = np.abs(do.response(taps[j], kap) - exact).max()
        assert err <= (bound_mid if u >= 0.6 else bound_all), (j, u, err)
        assert np.abs(do.response(np.conj(taps[j]), kap) - exact).max() > 10 * err or u < 0.3


# ---------------------------------------------------------------- G-P4 what D3 promises
def test_GP4_stability_symmetry_and_residual():
    ntab, ntaps, du = 20, 25, 4.2 / 19
    L = (ntaps - 1) // 2
    t = do.design_table(ntab, ntaps, du, 1.0)
    assert np.array_equal(t[:, :L][:, ::-1].view(np.uint64), t[:, L + 1:].view(np.uint64))
    kap = np.pi * np.arange(16384) / 16383
    assert np.abs(do.response(t.astype(np.complex128), kap)).max() <= 1.0 + 1e-6          # pin P6's statement
    for j in (1, 7, 19):                                              # D2 has (nearly) settled after 200 sweeps
        a = do.design_row_taps(j * du, L, 1.0, n_iter=200)
        b = do.design_row_taps(j * du, L, 1.0, n_iter=201)
        assert np.abs(a - b).max() <= 2e-5, j
    # the stop band is capped: outside the passband |H| <= 1 on the design grid after D3
    for j in (3, 12):
        u = j * du
        g = do.grid_kappa()
        out = np.abs(g) > do.passband_edge(u, 1.0)
        assert np.abs(do.response(t[j].astype(np.complex128), g[out])).max() <= 1.0 + 1e-6
