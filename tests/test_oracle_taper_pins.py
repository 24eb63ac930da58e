"""Pins of the oracle's absorbing edge-taper variant (reading R5b of DESIGN.md: the paper is silent on
the lateral boundary; SURVEY 8(f) N2 lists the taper as an optional variant of R5).  CPU only.

  E-P1  ntaper = 0 is plain R5, bit for bit
  E-P2  delta table: image[z][x] = t(x)^(z+1) * sum_w Re P0(w,x), t written out here independently
  E-P3  brute force on tiny grids (independent Python loop, taper applied after every step)
  E-P4  the taper only removes energy: per-frequency field norms never exceed the untapered ones'
        bound, and samples further than nz*L + ntaper from both edges are unchanged
"""
import numpy as np
import pytest

import oracle
import pdm_inputs
from pdm_inputs import filters


def _taper(nx, n):
    x = np.arange(nx)
    d = np.minimum(x, nx - 1 - x)
    t = np.ones(nx)
    m = d < n
    t[m] = np.sin(0.5 * np.pi * (d[m] + 1) / (n + 1)) ** 2
    return t


def test_EP1_zero_width_is_plain_R5():
    c = pdm_inputs.random_problem(3, 77, 9, 4, 11, ntab=30, model="field")
    assert np.array_equal(oracle.migrate(c), oracle.migrate(c, ntaper=0))


def test_EP2_delta_table_closed_form():
    rng = np.random.default_rng(2)
    nx, nz, nw, n = 41, 6, 3, 7
    c = pdm_inputs.random_problem(4, nx, nz, nw, 5, ntab=12, model="white")
    c = dict(c, table=filters.delta_table(12, 5))
    img = oracle.migrate(c, ntaper=n)
    base = c["P0"].astype(np.complex128).real.sum(axis=0)
    t = _taper(nx, n)
    want = np.stack([base * t ** (z + 1) for z in range(nz)])
    np.testing.assert_allclose(img, want, rtol=0, atol=1e-13 * np.abs(base).max())
    assert t[0] < 0.1 and t[n] == 1.0 and np.all(np.diff(t[:n + 1]) > 0) and np.array_equal(t, t[::-1])


@pytest.mark.parametrize("seed,nx,nz,nw,L,ntab,n", [(1, 9, 3, 2, 2, 7, 3), (2, 6, 4, 2, 1, 5, 10), (3, 17, 2, 1, 3, 9, 1)])
def test_EP3_brute_force(seed, nx, nz, nw, L, ntab, n):
    c = pdm_inputs.tiny_random_problem(seed, nx=nx, nz=nz, nw=nw, L=L, ntab=ntab, symmetric=False)
    tab = c["table"].astype(np.complex128)
    t = _taper(nx, n)
    img = np.zeros((nz, nx))
    for iw in range(nw):
        P = c["P0"][iw].astype(np.complex128)
        for z in range(nz):
            Pn = np.zeros(nx, np.complex128)
            for x in range(nx):
                q = np.float32(c["dz"] / (np.float64(c["velocity"][z, x]) * c["du"]))
                j = int(np.clip(np.rint(np.float32(c["omega"][iw]) * q), 0, ntab - 1))
                for k in range(-L, L + 1):
                    if 0 <= x - k < nx:
                        Pn[x] += tab[j, L + k] * P[x - k]
            P = Pn * t
            img[z] += P.real
    got = oracle.migrate(c, ntaper=n)
    np.testing.assert_allclose(got, img, rtol=0, atol=1e-13 * max(np.abs(img).max(), 1e-300))


def test_EP4_interior_unchanged_and_edges_absorb():
    c = pdm_inputs.random_problem(9, 300, 8, 3, 7, ntab=40, model="layers")
    n, L, nz = 20, 3, 8
    img0, f0 = oracle.migrate_field(c)
    img1, f1 = oracle.migrate_field(c, ntaper=n)
    reach = nz * L + n
    np.testing.assert_array_equal(img1[:, reach:-reach], img0[:, reach:-reach])
    # the field inside the taper zone is damped; stable random tables (sum |W| < 1) make that strict at the wall
    assert np.abs(f1[:, 0]).max() < np.abs(f0[:, 0]).max() * 0.2
    assert np.linalg.norm(f1) <= np.linalg.norm(f0) * (1 + 1e-12)
