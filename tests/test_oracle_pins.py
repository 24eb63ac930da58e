"""Pins P1-P12 of the FP64 oracle -- all CPU, none uses the CUDA path.

The paper prints no worked example, wavefield value or image value (checked: PAPER.md has
two timing tables only), so the oracle is pinned by closed forms, invariants, a textbook
special case (exact f-k phase shift) and an independently written brute force.
Each test names the part of the oracle it pins and the mistake it would catch.
"""
import numpy as np
import pytest

import oracle
import pdm_inputs
from pdm_inputs import filters


def _cfg(nx, nz, omega, v, table, du, P0, dz=10.0):
    omega = np.asarray(omega, np.float32)
    return dict(nx=nx, nz=nz, nw=omega.size, dz=dz, dx=10.0, du=float(du), omega=omega,
                velocity=np.ascontiguousarray(np.broadcast_to(np.asarray(v, np.float32), (nz, nx))),
                table=np.ascontiguousarray(table, np.complex64), ntab=table.shape[0],
                ntaps=table.shape[1], P0=np.ascontiguousarray(P0, np.complex64))


# ---------------------------------------------------------------- P1 delta table = identity
def test_P1_delta_table_is_identity():
    """W_0 = 1, all other taps 0  =>  image[z][x] = sum_w Re P0(w,x) for every z.
    Catches: wrong centre-tap index, dropped/duplicated w in the imaging sum, row layout."""
    c = pdm_inputs.tiny_random_problem(3, nx=37, nz=6, nw=5, L=4, ntab=11)
    c["table"] = filters.delta_table(11, 9)
    img = oracle.migrate(c)
    expect = c["P0"].real.astype(np.float64).sum(axis=0)
    assert img.shape == (6, 37)
    for z in range(6):
        np.testing.assert_allclose(img[z], expect, rtol=1e-15, atol=1e-15)


# ---------------------------------------------------------------- P2 brute force
@pytest.mark.parametrize("seed,nx,nz,nw,L,ntab,sym", [
    (11, 9, 3, 2, 2, 7, True), (12, 5, 4, 3, 3, 5, True),      # filter longer than the line
    (13, 16, 2, 1, 1, 4, False), (14, 1, 3, 2, 2, 6, False),   # asymmetric rows; nx = 1
    (15, 12, 5, 2, 0, 9, True)])                                # single tap
def test_P2_brute_force(seed, nx, nz, nw, L, ntab, sym):
    """Independent literal loop of Eq. (1) (oracle/brute.py).  Asymmetric tables expose a
    flipped x-k orientation (R11); short lines expose the zero-edge rule (R5)."""
    c = pdm_inputs.tiny_random_problem(seed, nx=nx, nz=nz, nw=nw, L=L, ntab=ntab, symmetric=sym)
    np.testing.assert_allclose(oracle.migrate(c), oracle.brute_force_migrate(c),
                               rtol=1e-13, atol=1e-13)


# ---------------------------------------------------------------- P3 spectral identity
def test_P3_spectral_identity():
    """Constant v, data padded by >= nz*L zeros: n steps == IDFT( H(kappa)^n DFT(P0) ),
    H(kappa) = sum_k W_k exp(-i k kappa).  Pins the whole recursion O4-O9 (a step that reads
    the wrong buffer, skips a swap or mis-orients the taps breaks it)."""
    rng = np.random.default_rng(5)
    L, nz, ntab, core = 3, 12, 9, 40
    pad = nz * L
    nx = core + 2 * pad
    table = (0.3 * (rng.standard_normal((ntab, 2 * L + 1)) +
                    1j * rng.standard_normal((ntab, 2 * L + 1)))).astype(np.complex64)  # asymmetric
    omega = np.array([40.0, 95.0], np.float32)
    v, dz = 2000.0, 10.0
    du = float(omega.max()) * dz / v / (ntab - 1)
    P0 = np.zeros((2, nx), np.complex64)
    P0[:, pad:pad + core] = (rng.standard_normal((2, core)) + 1j * rng.standard_normal((2, core)))
    c = _cfg(nx, nz, omega, v, table, du, P0, dz)
    _, field = oracle.migrate_field(c)
    for iw in range(2):
        j = int(np.rint(np.float32(omega[iw]) * np.float32(dz / (np.float64(np.float32(v)) * du))))
        h = np.zeros(nx, np.complex128)
        for k in range(-L, L + 1):
            h[k % nx] = table[j, L + k]                    # circular placement of W_k at lag k
        expect = np.fft.ifft(np.fft.fft(h) ** nz * np.fft.fft(P0[iw].astype(np.complex128)))
        np.testing.assert_allclose(field[iw], expect, rtol=0, atol=1e-12 * np.abs(expect).max())


# ---------------------------------------------------------------- P4 exact phase shift
@pytest.mark.parametrize("nsteps", [1, 32])
def test_P4_phase_shift_constant_velocity(config0, nsteps):
    """Constant velocity: the designed table must reproduce the exact f-k phase shift
    exp(+i n sqrt(u_j^2 - kappa^2)) on its passband within n * eps_design,
    with the QUANTISED u_j = idx*du.  Pins sign convention R4 (a conjugated table gives O(1)
    error), the table<->u mapping R3 and the design D1-D3."""
    c0 = config0
    L = (c0["ntaps"] - 1) // 2
    nx = 256 + 2 * nsteps * L
    pad = nsteps * L
    iw = [20, 60, 91]
    omega = c0["omega"][iw]
    v = float(c0["velocity"][0, 0])
    kappa = 2 * np.pi * np.fft.fftfreq(nx)
    rng = np.random.default_rng(9)
    P0 = np.zeros((3, nx), np.complex64)
    errs, bounds = [], []
    specs = []
    for i, w in enumerate(omega):
        j = oracle.table_index(w, v, c0["dz"], c0["du"], c0["ntab"])
        uj = j * c0["du"]
        edge = 0.8 * min(uj * np.sin(np.deg2rad(55.0)), 0.8 * np.pi)   # well inside the passband
        spec = (rng.standard_normal(nx) + 1j * rng.standard_normal(nx)) * (np.abs(kappa) <= edge)
        x = np.fft.ifft(spec)
        win = np.zeros(nx); win[pad:nx - pad] = np.hanning(nx - 2 * pad)
        x = x * win                                         # compact support (slightly widens the spectrum)
        P0[i] = x
        specs.append((j, uj))
    c = _cfg(nx, nsteps, omega, v, c0["table"], c0["du"], P0, c0["dz"])
    _, field = oracle.migrate_field(c)
    for i, (j, uj) in enumerate(specs):
        S = np.fft.fft(P0[i].astype(np.complex128))
        arg = uj * uj - kappa ** 2
        Dk = np.where(arg >= 0, np.exp(1j * np.sqrt(np.abs(arg))), np.exp(-np.sqrt(np.abs(arg))))
        exact = np.fft.ifft(Dk ** nsteps * S)
        # design error of row j measured independently on the energetic part of the spectrum
        h = np.zeros(nx, np.complex128)
        for k in range(-L, L + 1):
            h[k % nx] = c0["table"][j, L + k]
        Hk = np.fft.fft(h)
        wgt = np.abs(S) / np.abs(S).max()
        eps = np.max(np.abs(Hk - Dk) * (wgt > 1e-3))
        rel = np.linalg.norm(field[i] - exact) / np.linalg.norm(exact)
        errs.append(rel); bounds.append(nsteps * eps + 1e-3)
        assert rel <= nsteps * eps + 1e-3, (i, rel, eps)
        assert eps < 0.05
    # the test must have teeth: a conjugated (wrong-sign) operator is far outside the bound
    cc = dict(c); cc["table"] = np.conj(c0["table"])
    _, wrong = oracle.migrate_field(cc)
    j, uj = specs[-1]
    arg = uj * uj - kappa ** 2
    Dk = np.where(arg >= 0, np.exp(1j * np.sqrt(np.abs(arg))), np.exp(-np.sqrt(np.abs(arg))))
    exact = np.fft.ifft(Dk ** nsteps * np.fft.fft(P0[-1].astype(np.complex128)))
    assert np.linalg.norm(wrong[-1] - exact) / np.linalg.norm(exact) > 10 * bounds[-1]


# ---------------------------------------------------------------- P5 diffractor focusing
def test_P5_point_diffractor_focuses(config0):
    """One diffractor at (x0, z0), exploding-reflector data with half velocity (R2): the image
    peak must sit at column round(x0/dx) +-1 and row round(z0/dz)-1 +-1 (R6: row iz is depth
    (iz+1) dz).  Pins R2, R4, R6 and the rad/s unit of omega."""
    from pdm_inputs.configs import diffractor_section, ricker_spectrum
    c = dict(config0)
    x = np.arange(c["nx"]) * c["dx"]
    for x0, z0 in [(640.0, 640.0), (410.0, 900.0)]:
        P0 = diffractor_section(c["omega"], ricker_spectrum(c["omega"], 20.0), x,
                                [x0], [z0], [2000.0], [1.0])
        c["P0"] = P0.astype(np.complex64)
        img = oracle.migrate(c)
        iz, ix = np.unravel_index(np.argmax(np.abs(img)), img.shape)
        assert abs(ix - round(x0 / c["dx"])) <= 1, (ix, x0)
        assert abs(iz - (round(z0 / c["dz"]) - 1)) <= 1, (iz, z0)
        # focusing, not just a maximum somewhere: the peak dominates the far field of the image
        far = np.abs(img).copy()
        far[max(0, iz - 8):iz + 9, max(0, ix - 8):ix + 9] = 0
        assert far.max() < 0.5 * np.abs(img[iz, ix])
    # conjugated data (wrong sign convention) must NOT focus there
    c["P0"] = np.conj(c["P0"])
    bad = oracle.migrate(c)
    assert np.abs(bad[iz, ix]) < 0.5 * np.abs(img[iz, ix])


# ---------------------------------------------------------------- P6 table stability
@pytest.mark.parametrize("ntaps", [15, 25])
def test_P6_designed_table_is_stable_and_symmetric(ntaps):
    """|H_j(kappa)| <= 1 + 1e-6 for every row after rounding to complex64; exact symmetry."""
    t = pdm_inputs.configs.cached_table(256, ntaps, 3.2 / 255, 1.0)
    L = (ntaps - 1) // 2
    assert np.array_equal(t[:, :L][:, ::-1].view(np.uint64), t[:, L + 1:].view(np.uint64))
    H = filters.response_on_grid(t[:, L:], 16384)
    assert np.abs(H).max() <= 1.0 + 1e-6
    # and the direct DFT of the full row agrees with the cosine form used above
    row = t[100].astype(np.complex128)
    kap = np.pi * np.arange(16384) / 16383
    direct = sum(row[L + k] * np.exp(-1j * k * kap) for k in range(-L, L + 1))
    np.testing.assert_allclose(direct, H[100], atol=1e-12)


# ---------------------------------------------------------------- P7 superposition
def test_P7_superposition_real_linear():
    c = pdm_inputs.random_problem(21, nx=96, nz=20, nw=6, ntaps=9, ntab=64, model="field")
    rng = np.random.default_rng(2)
    A = c["P0"]
    B = (rng.standard_normal(A.shape) + 1j * rng.standard_normal(A.shape)).astype(np.complex64)
    a, b = 0.75, -1.5                    # exactly representable: a*A + b*B rounds like the inputs
    cA, cB, cS = dict(c), dict(c), dict(c)
    cB["P0"] = B
    S = (a * A.astype(np.complex128) + b * B.astype(np.complex128))
    cS["P0"] = S.astype(np.complex64)
    resid = S - cS["P0"].astype(np.complex128)            # rounding of the combined input
    lhs = oracle.migrate(cS)
    rhs = a * oracle.migrate(cA) + b * oracle.migrate(cB)
    tol = 1e-13 * np.abs(rhs).max() + 4 * np.abs(resid).max() * c["nw"]
    np.testing.assert_allclose(lhs, rhs, rtol=0, atol=tol)
    # imaging takes Re: complex scaling must NOT commute (guards against imaging |P| or P)
    cI = dict(c); cI["P0"] = (1j * A).astype(np.complex64)
    assert np.abs(oracle.migrate(cI) - oracle.migrate(cA)).max() > 1e-3 * np.abs(rhs).max()


# ---------------------------------------------------------------- P8 omega additivity / permutation
def test_P8_omega_additivity_and_permutation():
    c = pdm_inputs.random_problem(22, nx=80, nz=16, nw=7, ntaps=7, ntab=64, model="layers")
    full = oracle.migrate(c)
    s1 = oracle.migrate(c, omega_index=[0, 2, 3])
    s2 = oracle.migrate(c, omega_index=[1, 4, 5, 6])
    np.testing.assert_allclose(s1 + s2, full, rtol=0, atol=1e-13 * np.abs(full).max())
    perm = np.array([3, 0, 6, 1, 5, 2, 4])
    cp = dict(c); cp["omega"] = c["omega"][perm]; cp["P0"] = c["P0"][perm]
    np.testing.assert_allclose(oracle.migrate(cp), full, rtol=0, atol=1e-13 * np.abs(full).max())


# ---------------------------------------------------------------- P9 mirror
def test_P9_mirror_symmetry():
    c = pdm_inputs.random_problem(23, nx=75, nz=14, nw=4, ntaps=11, ntab=64, model="white")
    img = oracle.migrate(c)
    cm = dict(c)
    cm["P0"] = np.ascontiguousarray(c["P0"][:, ::-1])
    cm["velocity"] = np.ascontiguousarray(c["velocity"][:, ::-1])
    np.testing.assert_allclose(oracle.migrate(cm)[:, ::-1], img, rtol=0,
                               atol=1e-13 * np.abs(img).max())


# ---------------------------------------------------------------- P10 energy non-growth
def test_P10_energy_does_not_grow(config0):
    c = dict(config0)
    rng = np.random.default_rng(4)
    c["P0"] = (rng.standard_normal(c["P0"].shape) + 1j * rng.standard_normal(c["P0"].shape)
               ).astype(np.complex64)
    prev = np.linalg.norm(c["P0"].astype(np.complex128), axis=1)
    for nz in (1, 2, 5, 20):
        cz = dict(c); cz["nz"] = nz; cz["velocity"] = c["velocity"][:nz]
        _, f = oracle.migrate_field(cz)
        e = np.linalg.norm(f, axis=1)
        assert np.all(e <= prev * (1 + 1e-6) ** nz)
        prev_e = e
    assert np.all(prev_e < prev)          # white input has evanescent energy: it must decay


# ---------------------------------------------------------------- P11 shift invariance
def test_P11_shift_invariance_in_vz():
    L, nz, core, s = 4, 10, 30, 7
    pad = nz * L + s
    nx = core + 2 * pad
    c = pdm_inputs.random_problem(24, nx=nx, nz=nz, nw=3, ntaps=2 * L + 1, ntab=64, model="layers")
    P0 = np.zeros_like(c["P0"]); P0[:, pad:pad + core] = c["P0"][:, pad:pad + core]
    c["P0"] = P0
    img = oracle.migrate(c)
    cs = dict(c); cs["P0"] = np.roll(P0, s, axis=1)
    np.testing.assert_allclose(oracle.migrate(cs), np.roll(img, s, axis=1), rtol=0,
                               atol=1e-12 * np.abs(img).max())


# ---------------------------------------------------------------- P12 index rule
def _index_rule_inputs():
    """16 frequencies, each with its own velocity row: 300 random velocities plus velocities
    SEARCHED (numpy only) so that the two plausible wrong rules -- FP64 product, q formed in
    float arithmetic -- give a different table row than R3 on them."""
    rng = np.random.default_rng(7)
    dz, du, ntab = 10.0, 0.00307, 1024
    lines = []
    for w in rng.uniform(10, 400, 16).astype(np.float32):
        v = rng.uniform(700, 2600, 1_000_000).astype(np.float32)
        q32 = (np.float64(dz) / (v.astype(np.float64) * du)).astype(np.float32)   # R3: one rounding
        expect = np.clip(np.rint(w * q32), 0, ntab - 1).astype(np.int64)           # float32 product, half-even
        alt_dp = np.clip(np.rint(np.float64(w) * q32.astype(np.float64)), 0, ntab - 1).astype(np.int64)
        qf = np.float32(dz) / (v * np.float32(du))                                  # q in float arithmetic
        alt_fq = np.clip(np.rint(w * qf), 0, ntab - 1).astype(np.int64)
        hard = np.flatnonzero((alt_dp != expect) | (alt_fq != expect))
        keep = np.concatenate([np.arange(300), hard])
        lines.append((w, v[keep], expect[keep], alt_dp[keep], alt_fq[keep]))
    n_dp = sum(int((l[3] != l[2]).sum()) for l in lines)
    n_fq = sum(int((l[4] != l[2]).sum()) for l in lines)
    return (dz, du, ntab), lines, n_dp, n_fq


def test_P12a_index_rule_matches_float32_definition():
    """idx = clamp(rint_half_even(fl32(w32 * fl32(dz/(v*du))))) -- compared with numpy float32 on
    random pairs AND on pairs where an FP64 product or a float-formed q gives another row."""
    (dz, du, ntab), lines, n_dp, n_fq = _index_rule_inputs()
    for w, v, expect, _, _ in lines:
        got = np.array([oracle.table_index(w, v[i], dz, du, ntab) for i in range(v.size)])
        assert np.array_equal(got, expect)
    # exact ties round to even, and both clamps are active
    assert oracle.table_index(2.5, 1.0, 1.0, 1.0, 1024) == 2
    assert oracle.table_index(3.5, 1.0, 1.0, 1.0, 1024) == 4
    assert oracle.table_index(5000.0, 1.0, 1.0, 1.0, 1024) == 1023
    assert oracle.table_index(0.2, 1.0, 1.0, 1.0, 1024) == 0
    # the rule is a real choice (R3): both wrong variants differ on this set, so a slip to either
    # cannot pass the equality above
    assert n_dp > 50 and n_fq > 50, (n_dp, n_fq)


def test_P12b_index_rule_through_the_migrate_loop():
    """The rule as pdm_oracle_migrate's OWN loop applies it (not a twin function): nz = 1, P0 = 1,
    a table whose centre tap of row j is the real number j and every other tap 0  =>
    image[0][x] = sum_w idx(w, v[0][x]).  One frequency per call makes every pixel one (w, v)
    pair.  Catches: FP64 product in the loop, q rounded twice / formed in float, truncation
    instead of round-half-even, missing clamps, q row mis-indexing."""
    (dz, du, ntab), lines, n_dp, n_fq = _index_rule_inputs()
    assert n_dp > 50 and n_fq > 50, (n_dp, n_fq)                 # the set has teeth
    ntaps = 5
    table = np.zeros((ntab, ntaps), np.complex64)
    table[:, ntaps // 2] = np.arange(ntab, dtype=np.float32)     # row j -> the number j
    for w, v, expect, _, _ in lines:
        nx = v.size
        c = _cfg(nx, 1, [w], v[None, :], table, du, np.ones((1, nx), np.complex64), dz)
        np.testing.assert_array_equal(oracle.migrate(c)[0], expect.astype(np.float64))
    # both clamps through the loop: u far beyond the table and u -> 0
    c = _cfg(2, 1, [400.0], np.array([[1.0, 1e9]], np.float32), table, du, np.ones((1, 2), np.complex64), dz)
    np.testing.assert_array_equal(oracle.migrate(c)[0], [ntab - 1, 0])
    # several frequencies and depth rows in ONE call (w loop, q row of step z): rows z >= 1 see the
    # field after z+1 applications of the centre taps, so use nz = 1 per row check via the velocity row
    nx, nw = 257, 6
    ws = np.array([l[0] for l in lines[:nw]], np.float32)
    vv = lines[0][1][:nx]
    c = _cfg(nx, 1, ws, vv[None, :], table, du, np.ones((nw, nx), np.complex64), dz)
    q32 = (np.float64(dz) / (vv.astype(np.float64) * du)).astype(np.float32)
    want = sum(np.clip(np.rint(wi * q32), 0, ntab - 1) for wi in ws)
    np.testing.assert_array_equal(oracle.migrate(c)[0], want.astype(np.float64))


# ---------------------------------------------------------------- regression fixture
def test_golden_tiny_image_regression():
    """tests/golden/tiny_image.txt (written by make_golden.py from the oracle alone)."""
    import os
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", "tiny_image.txt")
    rows = [[float.fromhex(t) for t in ln.split()] for ln in open(path) if not ln.startswith("#")]
    c = pdm_inputs.tiny_random_problem(101, nx=12, nz=4, nw=3, L=2, ntab=8)
    np.testing.assert_allclose(oracle.migrate(c), np.array(rows), rtol=1e-14, atol=1e-15)
    np.testing.assert_allclose(oracle.brute_force_migrate(c), np.array(rows), rtol=1e-13, atol=1e-14)
