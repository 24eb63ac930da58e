"""Pins of the oracle's interpolated-table variant pdm_oracle_migrate_interp (reading R3c;
SURVEY.md 8(f) N3 "optional linear interpolation between rows"; PAPER.md:65 Alg. 1 "Look-up Table", :83
"the required filter bank is accessed" -- the paper only says the filter is looked up).  CPU only.

  I-P1  wherever u = w*dz/v lands exactly on a table row the blend weight is 0: on such inputs the variant
        equals the nearest-row oracle BIT FOR BIT (and the plain entry point is unchanged by the new code)
  I-P2  brute force on tiny grids: an independent pure-Python loop (bracketing rows, weight, Eq. (1))
  I-P3  a table that is LINEAR in the row number, W_k(j) = A_k + j B_k, is reproduced exactly by linear
        interpolation: the result equals Eq. (1) with the continuous operator A_k + (u/du) B_k, which the
        test evaluates directly from u -- no rows, no weights
  I-P4  continuity: moving one velocity sample across a rounding boundary of the nearest-row rule changes
        the nearest-row image by a jump and the interpolated image by O(perturbation)
  I-P5  the last row clamps: u beyond the table uses row ntab-1 alone
"""
import numpy as np
import pytest

import oracle
import pdm_inputs


def _exact_row_problem(seed, nx=40, nz=6, nw=3, L=3, ntab=33):
    """omega, v and du chosen so that fl32(w * q32) is an integer for every (w, x, z): du = dz/(v0*64),
    v = v0 / m with m a power of two, w = 4, 8, 12 ... -> u/du = w * 64 * m / ... exactly representable."""
    rng = np.random.default_rng(seed)
    cfg = pdm_inputs.tiny_random_problem(seed, nx=nx, nz=nz, nw=nw, L=L, ntab=ntab, symmetric=False)
    dz, v0 = 8.0, 2048.0
    cfg = dict(cfg, dz=dz, du=dz / (v0 * 2.0))                       # q32 = 2 * v0 / v
    m = rng.choice([1.0, 2.0, 4.0], size=(nz, nx))
    cfg["velocity"] = (v0 / m).astype(np.float32)                    # q32 = 2 m  in {2, 4, 8}
    cfg["omega"] = np.arange(1, nw + 1, dtype=np.float32)            # u/du = w * q in {2 .. 8 nw} < ntab
    return cfg


def test_IP1_equals_nearest_row_when_u_hits_the_rows_exactly(config0):
    cfg = _exact_row_problem(3)
    q = cfg["dz"] / (cfg["velocity"].astype(np.float64) * cfg["du"])
    u = cfg["omega"][:, None, None].astype(np.float64) * q[None]
    assert np.array_equal(u, np.rint(u)) and u.max() <= cfg["ntab"] - 1
    assert np.array_equal(oracle.migrate(cfg, interp=True), oracle.migrate(cfg))
    # ... and on a generic problem the two differ (the variant is not a no-op)
    gen = pdm_inputs.random_problem(4, 64, 5, 3, 7, ntab=32, model="field")
    a, b = oracle.migrate(gen, interp=True), oracle.migrate(gen)
    assert np.abs(a - b).max() > 1e-3 * np.abs(b).max()


def _brute_interp(cfg, op=None):
    """Independent literal loop.  op(u_over_du, k) -> complex tap; default: blend of the bracketing rows."""
    nx, nz, nw = cfg["nx"], cfg["nz"], cfg["nw"]
    table = cfg["table"]
    ntab, ntaps = table.shape
    half = (ntaps - 1) // 2
    image = np.zeros((nz, nx))
    for iw in range(nw):
        w32 = np.float32(cfg["omega"][iw])
        prev = [complex(c) for c in cfg["P0"][iw]]
        for iz in range(nz):
            nxt = []
            for i in range(nx):
                q32 = np.float32(np.float64(cfg["dz"]) / (np.float64(cfg["velocity"][iz, i]) * np.float64(cfg["du"])))
                u = float(np.float32(w32 * q32))                     # the float product of R3, then plain arithmetic
                total = 0j
                for n in range(-half, half + 1):
                    if not 0 <= i - n < nx:
                        continue
                    if op is not None:
                        tap = op(u, n)
                    elif u >= ntab - 1:
                        tap = complex(table[ntab - 1, half + n])
                    else:
                        lo = int(u // 1)
                        frac = u - lo
                        tap = (1.0 - frac) * complex(table[lo, half + n]) + frac * complex(table[lo + 1, half + n])
                    total += tap * prev[i - n]
                nxt.append(total)
            prev = nxt
            image[iz] += [p.real for p in prev]
    return image


@pytest.mark.parametrize("seed,nx,nz,nw,L,ntab", [(1, 9, 3, 2, 2, 7), (2, 13, 4, 3, 1, 5), (3, 6, 2, 2, 4, 9)])
def test_IP2_brute_force(seed, nx, nz, nw, L, ntab):
    cfg = pdm_inputs.tiny_random_problem(seed, nx=nx, nz=nz, nw=nw, L=L, ntab=ntab, symmetric=False)
    got = oracle.migrate(cfg, interp=True)
    want = _brute_interp(cfg)
    assert np.abs(got - want).max() <= 1e-13 * max(1.0, np.abs(want).max())


def test_IP3_table_linear_in_the_row_number_is_reproduced_exactly():
    cfg = dict(pdm_inputs.tiny_random_problem(5, nx=11, nz=3, nw=2, L=2, ntab=17, symmetric=False))
    rng = np.random.default_rng(7)
    ntaps = cfg["table"].shape[1]
    # A, B dyadic so that A + j B is exact in complex64 for every row
    A = (rng.integers(-8, 9, ntaps) + 1j * rng.integers(-8, 9, ntaps)) / 64.0
    B = (rng.integers(-4, 5, ntaps) + 1j * rng.integers(-4, 5, ntaps)) / 1024.0
    j = np.arange(17)[:, None]
    cfg["table"] = (A[None, :] + j * B[None, :]).astype(np.complex64)
    half = (ntaps - 1) // 2
    got = oracle.migrate(cfg, interp=True)
    want = _brute_interp(cfg, op=lambda u, n: A[half + n] + min(u, 16.0) * B[half + n])
    assert np.abs(got - want).max() <= 1e-13 * max(1.0, np.abs(want).max())
    assert np.abs(oracle.migrate(cfg) - want).max() > 1e-6           # nearest-row does not reproduce it


def test_IP4_continuous_in_the_velocity_where_nearest_row_jumps():
    cfg = dict(pdm_inputs.tiny_random_problem(9, nx=15, nz=1, nw=1, L=2, ntab=33, symmetric=False))
    dz, du, w = 10.0, 0.01, np.float32(40.0)
    cfg.update(dz=dz, du=du, omega=np.array([w], np.float32))
    # u/du = w*dz/(v*du): v chosen so that u/du sits at j + 0.5 -/+ eps for the middle sample
    def vel(target):
        v = np.full((1, 15), w * dz / (du * 12.25), dtype=np.float64)
        v[0, 7] = w * dz / (du * target)
        return v.astype(np.float32)
    lo, hi = dict(cfg, velocity=vel(20.5 - 2e-3)), dict(cfg, velocity=vel(20.5 + 2e-3))
    assert oracle.table_index(w, lo["velocity"][0, 7], dz, du, 33) == 20
    assert oracle.table_index(w, hi["velocity"][0, 7], dz, du, 33) == 21
    jump = np.abs(oracle.migrate(hi) - oracle.migrate(lo)).max()
    smooth = np.abs(oracle.migrate(hi, interp=True) - oracle.migrate(lo, interp=True)).max()
    assert jump > 1e-3 and smooth < 1e-2 * jump, (jump, smooth)


def test_IP5_beyond_the_table_the_last_row_is_used_alone():
    cfg = dict(pdm_inputs.tiny_random_problem(11, nx=10, nz=2, nw=2, L=1, ntab=5, symmetric=False))
    cfg.update(dz=10.0, du=0.01, omega=np.array([50.0, 60.0], np.float32),
               velocity=np.full((2, 10), 1000.0, np.float32))        # u/du = 50, 60 >> 4
    last = dict(cfg, table=np.repeat(cfg["table"][-1:], 5, axis=0))
    assert np.array_equal(oracle.migrate(cfg, interp=True), oracle.migrate(last))
