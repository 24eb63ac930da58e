"""Pins of the oracle's prestack (shot-profile) variant, pdm_oracle_migrate_shot (reading R17 of
DESIGN.md; PAPER.md:151 names the extension, gives no equations).  CPU only.

  S-P1  delta table: image[z][x] = sum_w Re(conj(S0) R0) for every z            (closed form)
  S-P2  brute force on tiny grids: an independent literal loop in Python complex128
  S-P3  spectral identity in constant velocity, ASYMMETRIC table: R(n) = IDFT(H^n DFT R0),
        S(n) = IDFT(G^n DFT S0), G(kappa) = sum_k conj(W_k) e^{-ik kappa}; the image row follows
  S-P4  invariants: a global phase on both inputs cancels; real bilinearity; shots add up
  S-P5  a point source and a point diffractor: the image focuses at the diffractor; the
        poststack special case (S0 = 1, laterally invariant) equals pdm_oracle_migrate
"""
import numpy as np
import pytest

import oracle
import pdm_inputs
from pdm_inputs import filters


def _cfg(nx, nz, omega, v, table, du, dz=10.0):
    omega = np.asarray(omega, np.float32)
    return dict(nx=nx, nz=nz, nw=omega.size, dz=dz, dx=10.0, du=float(du), omega=omega,
                velocity=np.ascontiguousarray(np.broadcast_to(np.asarray(v, np.float32), (nz, nx))),
                table=np.ascontiguousarray(table, np.complex64), ntab=table.shape[0], ntaps=table.shape[1])


def _rand_c(rng, shape):
    return (rng.standard_normal(shape) + 1j * rng.standard_normal(shape)).astype(np.complex64)


def test_SP1_delta_table_closed_form():
    rng = np.random.default_rng(1)
    nx, nz, nw, L, ntab = 23, 5, 4, 3, 6
    table = filters.delta_table(ntab, 2 * L + 1)
    omega = np.linspace(20, 80, nw)
    v = rng.uniform(1500, 4000, (nz, nx))
    c = _cfg(nx, nz, omega, v, table, float(omega.max()) * 10.0 / 1500.0 / (ntab - 1))
    S0, R0 = _rand_c(rng, (nw, nx)), _rand_c(rng, (nw, nx))
    img = oracle.migrate_shot(c, S0, R0)
    want = np.sum(np.real(np.conj(S0.astype(np.complex128)) * R0.astype(np.complex128)), axis=0)
    np.testing.assert_allclose(img, np.broadcast_to(want, (nz, nx)), rtol=0, atol=1e-13 * np.abs(want).max())


def _brute_shot(c, S0, R0):
    nx, nz, nw = c["nx"], c["nz"], c["nw"]
    tab = c["table"].astype(np.complex128)
    L = (tab.shape[1] - 1) // 2
    img = np.zeros((nz, nx))
    for iw in range(nw):
        S = [complex(a) for a in S0[iw]]
        R = [complex(a) for a in R0[iw]]
        for z in range(nz):
            Sn, Rn = [0j] * nx, [0j] * nx
            for x in range(nx):
                q = np.float32(c["dz"] / (np.float64(c["velocity"][z, x]) * c["du"]))
                j = int(np.clip(np.rint(np.float32(c["omega"][iw]) * q), 0, tab.shape[0] - 1))
                for k in range(-L, L + 1):
                    if 0 <= x - k < nx:
                        Rn[x] += tab[j, L + k] * R[x - k]
                        Sn[x] += np.conj(tab[j, L + k]) * S[x - k]
            S, R = Sn, Rn
            for x in range(nx):
                img[z, x] += (np.conj(S[x]) * R[x]).real
    return img


@pytest.mark.parametrize("seed,nx,nz,nw,L,ntab", [(1, 9, 3, 2, 2, 7), (2, 5, 4, 3, 3, 5), (3, 17, 2, 1, 1, 9)])
def test_SP2_brute_force(seed, nx, nz, nw, L, ntab):
    rng = np.random.default_rng(seed)
    table = (0.25 * _rand_c(rng, (ntab, 2 * L + 1))).astype(np.complex64)          # asymmetric
    omega = np.linspace(30, 90, nw)
    v = rng.uniform(1500, 4000, (nz, nx))
    c = _cfg(nx, nz, omega, v, table, float(omega.max()) * 10.0 / 1500.0 / (ntab - 1))
    S0, R0 = _rand_c(rng, (nw, nx)), _rand_c(rng, (nw, nx))
    img = oracle.migrate_shot(c, S0, R0)
    np.testing.assert_allclose(img, _brute_shot(c, S0, R0), rtol=0, atol=1e-13 * np.abs(img).max())


def test_SP3_spectral_identity_both_fields():
    rng = np.random.default_rng(5)
    L, nz, ntab, core = 3, 10, 9, 36
    pad = nz * L
    nx = core + 2 * pad
    table = (0.3 * _rand_c(rng, (ntab, 2 * L + 1))).astype(np.complex64)           # asymmetric
    omega = np.array([40.0, 95.0], np.float32)
    v, dz = 2000.0, 10.0
    du = float(omega.max()) * dz / v / (ntab - 1)
    S0 = np.zeros((2, nx), np.complex64); R0 = np.zeros((2, nx), np.complex64)
    S0[:, pad:pad + core] = _rand_c(rng, (2, core)); R0[:, pad:pad + core] = _rand_c(rng, (2, core))
    for n in (1, nz):
        c = _cfg(nx, n, omega, v, table, du, dz)
        img = oracle.migrate_shot(c, S0, R0)
        want = np.zeros(nx)
        for iw in range(2):
            j = int(np.rint(np.float32(omega[iw]) * np.float32(dz / (np.float64(np.float32(v)) * du))))
            h = np.zeros(nx, np.complex128); g = np.zeros(nx, np.complex128)
            for k in range(-L, L + 1):
                h[k % nx] = table[j, L + k]
                g[k % nx] = np.conj(table[j, L + k])
            Rn = np.fft.ifft(np.fft.fft(h) ** n * np.fft.fft(R0[iw].astype(np.complex128)))
            Sn = np.fft.ifft(np.fft.fft(g) ** n * np.fft.fft(S0[iw].astype(np.complex128)))
            want += np.real(np.conj(Sn) * Rn)
        np.testing.assert_allclose(img[n - 1], want, rtol=0, atol=1e-12 * np.abs(want).max())


def test_SP4_phase_invariance_bilinearity_and_shot_sum():
    rng = np.random.default_rng(8)
    c = pdm_inputs.random_problem(3, 60, 9, 5, 11, ntab=40, model="field")
    S0, R0 = _rand_c(rng, (5, 60)), _rand_c(rng, (5, 60))
    S1, R1 = _rand_c(rng, (5, 60)), _rand_c(rng, (5, 60))
    base = oracle.migrate_shot(c, S0, R0)
    ph = np.complex64(np.exp(0.7j))
    scale = np.abs(base).max()
    np.testing.assert_allclose(oracle.migrate_shot(c, S0 * ph, R0 * ph), base, rtol=0, atol=2e-6 * scale)
    np.testing.assert_allclose(oracle.migrate_shot(c, 2 * S0, -4 * R0), -8 * base, rtol=0, atol=1e-12 * scale)
    # linear in R for a fixed S
    lin = oracle.migrate_shot(c, S0, (R0 + R1).astype(np.complex64))
    np.testing.assert_allclose(lin, base + oracle.migrate_shot(c, S0, R1), rtol=0, atol=2e-6 * scale)
    # two shots accumulated into one image
    acc = oracle.migrate_shot(c, S0, R0)
    oracle.migrate_shot(c, S1, R1, image=acc)
    np.testing.assert_allclose(acc, base + oracle.migrate_shot(c, S1, R1), rtol=0, atol=1e-12 * scale)
    # a conjugated source is NOT the same image (the conjugate operator on S matters)
    assert np.abs(oracle.migrate_shot(c, np.conj(S0), R0) - base).max() > 1e-3 * scale


def test_SP5_point_source_and_diffractor_focus(config0):
    """One shot: point source at the surface, one diffractor at (x0, z0) in constant velocity; one-way
    times, so the true velocity is passed (config0's table was designed for v_in = 1000 m/s).  The
    cross-correlation image must peak at the diffractor: column +-1, row z0/dz - 1 +-1."""
    from pdm_inputs.configs import ricker_spectrum
    c = dict(config0)
    v = float(c["velocity"][0, 0])                         # migration velocity of the plan
    nx, dx, dz = c["nx"], c["dx"], c["dz"]
    x = np.arange(nx) * dx
    w = c["omega"].astype(np.float64)
    spec = ricker_spectrum(c["omega"], 20.0)
    for xs, x0, z0 in [(640.0, 600.0, 400.0), (300.0, 800.0, 700.0)]:
        S0 = np.zeros((w.size, nx), np.complex128)
        S0[:, int(round(xs / dx))] = spec
        t = (np.sqrt(z0 ** 2 + (x0 - xs) ** 2) + np.sqrt(z0 ** 2 + (x - x0) ** 2)) / v
        R0 = spec[:, None] * np.exp(-1j * w[:, None] * t[None, :])
        img = oracle.migrate_shot(c, S0.astype(np.complex64), R0.astype(np.complex64))
        deep = np.abs(img).copy()
        deep[:15] = 0                                      # the source's own near field
        iz, ix = np.unravel_index(np.argmax(deep), deep.shape)
        assert abs(ix - round(x0 / dx)) <= 1 and abs(iz - (round(z0 / dz) - 1)) <= 1, (ix, iz, x0, z0)
        far = deep.copy()
        far[max(0, iz - 8):iz + 9, max(0, ix - 8):ix + 9] = 0
        assert far.max() < 0.5 * deep[iz, ix]              # focusing, not just a maximum somewhere
        # conjugated data (wrong sign convention) must NOT focus there
        bad = oracle.migrate_shot(c, S0.astype(np.complex64), np.conj(R0).astype(np.complex64))
        assert np.abs(bad[iz, ix]) < 0.5 * deep[iz, ix]


def test_SP5b_poststack_special_case():
    """Laterally invariant v(z), symmetric table, S0 = 1 on a long line: away from the edges the
    source field stays a constant c_w(z) = prod_z conj(H_j(0)) per frequency, so the shot image equals
    sum_w Re(conj(c_w(z)) R(z)) -- assembled here from pdm_oracle_migrate's own wavefields."""
    rng = np.random.default_rng(12)
    nx, nz, nw, L, ntab = 200, 6, 3, 2, 12
    table = filters.random_symmetric_table(rng, ntab, 2 * L + 1, scale=0.4)
    omega = np.linspace(30, 90, nw).astype(np.float32)
    vz = rng.uniform(1500, 4000, nz)[:, None]
    du = float(omega.max()) * 10.0 / 1500.0 / (ntab - 1)
    c = _cfg(nx, nz, omega, vz, table, du)
    R0 = _rand_c(rng, (nw, nx))
    img = oracle.migrate_shot(c, np.ones((nw, nx), np.complex64), R0)
    want = np.zeros((nz, nx))
    for n in range(1, nz + 1):
        cn = dict(c, nz=n, velocity=c["velocity"][:n], P0=R0)
        _, field = oracle.migrate_field(cn)
        for iw in range(nw):
            cw = 1.0 + 0j
            for z in range(n):
                j = oracle.table_index(omega[iw], c["velocity"][z, 0], 10.0, du, ntab)
                cw *= np.conj(table[j].astype(np.complex128).sum())
            want[n - 1] += np.real(np.conj(cw) * field[iw])
    mid = slice(nz * L + 1, nx - nz * L - 1)
    np.testing.assert_allclose(img[:, mid], want[:, mid], rtol=0, atol=1e-12 * np.abs(want).max())
