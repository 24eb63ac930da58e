"""Pins of the oracle's 3-D variant pdm_oracle_migrate3d (reading R18 of DESIGN.md; PAPER.md:41, :47:
"requires 2-D filters as extrapolators").  CPU only.

  T-P1  delta table: image[z][y][x] = sum_w Re P0 for every z                        (closed form)
  T-P2  brute force on tiny grids: an independent literal loop in Python complex128
  T-P3  2-D spectral identity, constant velocity, ASYMMETRIC table: n steps == IFFT2(H^n FFT2(P0))
  T-P4  separable table W[ky][kx] = a[ky] b[kx], constant velocity: the 3-D step is the pinned 1-D
        oracle applied along x with b and along y with a (pdm_oracle_migrate's own wavefields)
  T-P5  transposition: swapping the roles of x and y (inputs, velocity and table) transposes the image
  T-P6  physics: with 2-D extrapolators made from the designed 1-D rows by the McClellan transformation
        (pdm_inputs/filters.py::mcclellan_table, ref :177), the zero-offset record of a point
        diffractor in constant velocity focuses at (x0, y0, z0) +- 1 cell, and conjugated data does not
"""
import numpy as np
import pytest

import oracle


def _rand_c(rng, shape, scale=1.0):
    return (scale * (rng.standard_normal(shape) + 1j * rng.standard_normal(shape))).astype(np.complex64)


def _cfg3(nx, ny, nz, omega, v, table, du, P0, dz=10.0):
    omega = np.asarray(omega, np.float32)
    return dict(nx=nx, ny=ny, nz=nz, nw=omega.size, dz=dz, dx=10.0, dy=10.0, du=float(du), omega=omega,
                velocity=np.ascontiguousarray(np.broadcast_to(np.asarray(v, np.float32), (nz, ny, nx))),
                table=np.ascontiguousarray(table, np.complex64), ntab=table.shape[0], ntaps=table.shape[1],
                P0=np.ascontiguousarray(P0, np.complex64))


def test_TP1_delta_table_is_identity():
    rng = np.random.default_rng(1)
    nx, ny, nz, nw, L, ntab = 11, 7, 4, 3, 2, 5
    table = np.zeros((ntab, 2 * L + 1, 2 * L + 1), np.complex64)
    table[:, L, L] = 1
    omega = np.linspace(20, 80, nw)
    v = rng.uniform(1500, 4000, (nz, ny, nx))
    P0 = _rand_c(rng, (nw, ny, nx))
    c = _cfg3(nx, ny, nz, omega, v, table, float(omega.max()) * 10.0 / 1500.0 / (ntab - 1), P0)
    img = oracle.migrate3d(c)
    want = P0.astype(np.complex128).real.sum(axis=0)
    np.testing.assert_allclose(img, np.broadcast_to(want, (nz, ny, nx)), rtol=0, atol=1e-14 * np.abs(want).max())


def _brute3d(c):
    nx, ny, nz, nw = c["nx"], c["ny"], c["nz"], c["nw"]
    tab = c["table"].astype(np.complex128)
    L = (tab.shape[1] - 1) // 2
    img = np.zeros((nz, ny, nx))
    for iw in range(nw):
        P = c["P0"][iw].astype(np.complex128)
        for z in range(nz):
            Pn = np.zeros_like(P)
            for y in range(ny):
                for x in range(nx):
                    q = np.float32(c["dz"] / (np.float64(c["velocity"][z, y, x]) * c["du"]))
                    j = int(np.clip(np.rint(np.float32(c["omega"][iw]) * q), 0, tab.shape[0] - 1))
                    s = 0j
                    for ky in range(-L, L + 1):
                        for kx in range(-L, L + 1):
                            if 0 <= y - ky < ny and 0 <= x - kx < nx:
                                s += tab[j, L + ky, L + kx] * P[y - ky, x - kx]
                    Pn[y, x] = s
            P = Pn
            img[z] += P.real
    return img


@pytest.mark.parametrize("seed,nx,ny,nz,nw,L,ntab", [(1, 6, 5, 3, 2, 1, 7), (2, 4, 7, 2, 2, 2, 5), (3, 9, 3, 2, 1, 1, 9)])
def test_TP2_brute_force(seed, nx, ny, nz, nw, L, ntab):
    rng = np.random.default_rng(seed)
    table = _rand_c(rng, (ntab, 2 * L + 1, 2 * L + 1), 0.15)                       # fully asymmetric
    omega = np.linspace(30, 90, nw)
    v = rng.uniform(1500, 4000, (nz, ny, nx))
    c = _cfg3(nx, ny, nz, omega, v, table, float(omega.max()) * 10.0 / 1500.0 / (ntab - 1), _rand_c(rng, (nw, ny, nx)))
    img = oracle.migrate3d(c)
    np.testing.assert_allclose(img, _brute3d(c), rtol=0, atol=1e-13 * np.abs(img).max())


def test_TP3_spectral_identity_2d():
    rng = np.random.default_rng(5)
    L, nz, ntab, core = 2, 6, 9, 10
    pad = nz * L
    n = core + 2 * pad
    table = _rand_c(rng, (ntab, 2 * L + 1, 2 * L + 1), 0.12)                        # asymmetric in both axes
    omega = np.array([40.0, 95.0], np.float32)
    v, dz = 2000.0, 10.0
    du = float(omega.max()) * dz / v / (ntab - 1)
    P0 = np.zeros((2, n, n), np.complex64)
    P0[:, pad:pad + core, pad:pad + core] = _rand_c(rng, (2, core, core))
    c = _cfg3(n, n, nz, omega, v, table, du, P0, dz)
    img, field = oracle.migrate3d(c, want_field=True)
    for iw in range(2):
        j = int(np.rint(np.float32(omega[iw]) * np.float32(dz / (np.float64(np.float32(v)) * du))))
        h = np.zeros((n, n), np.complex128)
        for ky in range(-L, L + 1):
            for kx in range(-L, L + 1):
                h[ky % n, kx % n] = table[j, L + ky, L + kx]                         # W at lag (ky, kx)
        expect = np.fft.ifft2(np.fft.fft2(h) ** nz * np.fft.fft2(P0[iw].astype(np.complex128)))
        np.testing.assert_allclose(field[iw], expect, rtol=0, atol=1e-12 * np.abs(expect).max())


def test_TP4_separable_table_reduces_to_the_1d_oracle():
    rng = np.random.default_rng(9)
    L, nz, ntab, nx, ny = 2, 3, 6, 14, 11
    a = _rand_c(rng, (ntab, 2 * L + 1), 0.3)
    b = _rand_c(rng, (ntab, 2 * L + 1), 0.3)
    table = (a[:, :, None].astype(np.complex128) * b[:, None, :].astype(np.complex128)).astype(np.complex64)
    # use the ROUNDED product as the truth on both sides: factor it back exactly is impossible, so the
    # 1-D passes are run with a and b and compared at the rounding level of the complex64 product
    omega = np.array([50.0], np.float32)
    v, dz = 2500.0, 10.0
    du = float(omega.max()) * dz / v / (ntab - 1)
    P0 = _rand_c(rng, (1, ny, nx))
    c = _cfg3(nx, ny, 1, omega, v, table, du, P0, dz)
    _, field = oracle.migrate3d(c, want_field=True)
    # one step: first along x (every y row is a "frequency line" of the 1-D oracle), then along y
    line = dict(nx=nx, nz=1, nw=ny, dz=dz, du=du, omega=np.full(ny, omega[0], np.float32),
                velocity=np.full((1, nx), v, np.float32), table=b, P0=P0[0])
    _, fx = oracle.migrate_field(line)                                              # [ny, nx]
    col = dict(nx=ny, nz=1, nw=nx, dz=dz, du=du, omega=np.full(nx, omega[0], np.float32),
               velocity=np.full((1, ny), v, np.float32), table=a,
               P0=np.ascontiguousarray(fx.T).astype(np.complex64))
    _, fy = oracle.migrate_field(col)                                               # [nx, ny]
    np.testing.assert_allclose(field[0], fy.T, rtol=0, atol=3e-7 * np.abs(fy).max())


def test_TP5_transposition():
    rng = np.random.default_rng(11)
    nx, ny, nz, nw, L, ntab = 9, 6, 3, 2, 2, 8
    table = _rand_c(rng, (ntab, 2 * L + 1, 2 * L + 1), 0.1)
    omega = np.linspace(30, 90, nw)
    v = rng.uniform(1500, 4000, (nz, ny, nx))
    du = float(omega.max()) * 10.0 / 1500.0 / (ntab - 1)
    P0 = _rand_c(rng, (nw, ny, nx))
    img = oracle.migrate3d(_cfg3(nx, ny, nz, omega, v, table, du, P0))
    imgT = oracle.migrate3d(_cfg3(ny, nx, nz, omega, v.transpose(0, 2, 1), table.transpose(0, 2, 1), du,
                                  P0.transpose(0, 2, 1)))
    np.testing.assert_allclose(imgT, img.transpose(0, 2, 1), rtol=0, atol=1e-13 * np.abs(img).max())


def test_TP6_point_diffractor_focuses_in_3d():
    """Pins what T-P1..T-P5 cannot (they are self-consistent under any sign or axis convention): the sign
    of the phase (R4), the half velocity (R2), row <-> depth (R6) and the (ky, kx) <-> (y, x) table
    orientation of R18, through pdm_oracle_migrate3d with a physically meaningful table."""
    from pdm_inputs import filters
    from pdm_inputs.configs import dft_bin_omegas, ricker_spectrum, diffractor_volume
    nx, ny, nz, dx, dz, v = 56, 48, 40, 10.0, 10.0, 2000.0
    omega = dft_bin_omegas(256, 4e-3, 8.0, 45.0)
    v_in = 0.5 * v
    ntab, ntaps = 64, 15
    du = float(omega.max()) * dz / v_in / (ntab - 1)
    table = filters.mcclellan_table(filters.design_table(ntab, ntaps, du, dz / dx))
    L = (ntaps - 1) // 2
    assert np.array_equal(table[:, ::-1, :].view(np.uint64), table.view(np.uint64))      # symmetric in ky
    assert np.array_equal(table[:, :, ::-1].view(np.uint64), table.view(np.uint64))      # and in kx
    # along the kx axis the 2-D response IS the 1-D response (M(kx, 0) = cos kx)
    row1 = filters.design_table(ntab, ntaps, du, dz / dx)[40].astype(np.complex128)
    kap = np.linspace(0.0, 2.0, 9)
    k = np.arange(-L, L + 1)
    h1 = (row1[None, :] * np.exp(-1j * kap[:, None] * k[None, :])).sum(1)
    h2 = (table[40].astype(np.complex128).sum(0)[None, :] * np.exp(-1j * kap[:, None] * k[None, :])).sum(1)
    assert np.abs(h1 - h2).max() < 1e-5
    x, y = np.arange(nx) * dx, np.arange(ny) * dx
    x0, y0, z0 = 310.0, 200.0, 250.0                      # deliberately not symmetric in x and y
    P0 = diffractor_volume(omega, ricker_spectrum(omega, 22.0), x, y, x0, y0, z0, v)
    cfg = _cfg3(nx, ny, nz, omega, v_in, table, du, P0, dz=dz)
    img = oracle.migrate3d(cfg)
    iz, iy, ix = np.unravel_index(np.argmax(np.abs(img)), img.shape)
    assert abs(ix - round(x0 / dx)) <= 1 and abs(iy - round(y0 / dx)) <= 1, (ix, iy)
    assert abs(iz - (round(z0 / dz) - 1)) <= 1, iz
    far = np.abs(img).copy()
    far[max(0, iz - 6):iz + 7, max(0, iy - 6):iy + 7, max(0, ix - 6):ix + 7] = 0
    assert far.max() < 0.5 * np.abs(img[iz, iy, ix])
    bad = oracle.migrate3d(dict(cfg, P0=np.conj(cfg["P0"])))                           # wrong sign convention
    assert np.abs(bad[iz, iy, ix]) < 0.5 * np.abs(img[iz, iy, ix])
    worse = oracle.migrate3d(dict(cfg, table=np.conj(table)))                          # conjugated operator
    assert np.abs(worse[iz, iy, ix]) < 0.5 * np.abs(img[iz, iy, ix])
