"""Seeded synthetic workloads standing in for the paper's SEG/EAGE salt data.

The paper migrates the SEG/EAGE salt model's zero-offset section; that
dataset is not available here, so BASELINE.json's five synthetic configurations stand in
for it.  This module builds them (recipe: SURVEY.md §8(d), restated in DESIGN.md "Input
recipe").  It holds none of the method's arithmetic (no FIR, no table look-up, no
imaging): it only produces the arrays that are handed byte-identical to the FP64 oracle
and to the CUDA path.

Every workload is a dict with
    nx, nz, nw, ntaps, ntab : int
    dx, dz                  : float (metres)
    du                      : float (python double) table abscissa step, u_j = j*du
    omega                   : float32 [nw]      rad/s
    velocity                : float32 [nz, nx]  MIGRATION velocity v_in = v/2 (reading R2)
    table                   : complex64 [ntab, ntaps]
    P0                      : complex64 [nw, nx]
    name                    : str
"""
from __future__ import annotations

import hashlib
import os

import numpy as np

from . import filters

BASE_SEED = 191205529
NTAB = 1024

_CACHE_DIR = os.environ.get(
    "PDM_INPUT_CACHE", os.path.join(os.path.dirname(os.path.abspath(__file__)), "_cache"))


# --------------------------------------------------------------------------- helpers
def dft_bin_omegas(nt: int, dt: float, fmin: float, fmax: float) -> np.ndarray:
    """All DFT bins j of an nt-sample, dt-second trace with fmin <= j*df <= fmax (rad/s, fp32)."""
    df = 1.0 / (nt * dt)
    j = np.arange(0, nt // 2 + 1)
    f = j * df
    sel = (f >= fmin) & (f <= fmax)
    return (2.0 * np.pi * f[sel]).astype(np.float32)


def ricker_spectrum(omega: np.ndarray, f0: float) -> np.ndarray:
    f = np.asarray(omega, dtype=np.float64) / (2.0 * np.pi)
    return (2.0 / np.sqrt(np.pi)) * (f * f / f0 ** 3) * np.exp(-(f * f) / (f0 * f0))


def diffractor_section(omega, spectrum, x, xd, zd, veff, amp, chunk=256) -> np.ndarray:
    """P0(w,x) = sum_d a_d R(w) exp(-i w t_d(x)), t_d(x) = 2 sqrt(z_d^2 + (x-x_d)^2)/v_eff,d.

    Evaluated in complex128 directly (no recurrences), chunked over x to bound memory.
    """
    omega64 = np.asarray(omega, dtype=np.float64)
    nw, nx = omega64.size, x.size
    out = np.zeros((nw, nx), dtype=np.complex128)
    xd = np.asarray(xd, np.float64)[:, None]
    zd = np.asarray(zd, np.float64)[:, None]
    veff = np.asarray(veff, np.float64)[:, None]
    amp = np.asarray(amp, np.float64)
    for s in range(0, nx, chunk):
        xs = x[s:s + chunk][None, :]
        t = 2.0 * np.sqrt(zd * zd + (xs - xd) ** 2) / veff          # [nd, cx]
        # [nw, nd, cx] would be too big for the large cases: loop over frequency blocks
        wblk = max(1, int(4e6 // max(1, t.size)))
        for w0 in range(0, nw, wblk):
            ph = np.exp(-1j * omega64[w0:w0 + wblk, None, None] * t[None])
            out[w0:w0 + wblk, s:s + chunk] = np.einsum("d,wdx->wx", amp, ph)
    out *= np.asarray(spectrum, np.float64)[:, None]
    return out


def diffractor_section_uniform_bins(j0, nbins, domega, spectrum, x, xd, zd, veff, amp,
                                    chunk=512, reseed=64) -> np.ndarray:
    """Same sum as `diffractor_section` for equally spaced omega_j = (j0+j)*domega.

    Uses exp(-i w_{j+1} t) = exp(-i w_j t) * exp(-i domega t) (complex128, re-seeded from
    the exact exponential every `reseed` bins) so the 10^10-term case stays affordable.
    """
    nx = x.size
    out = np.zeros((nbins, nx), dtype=np.complex128)
    xd = np.asarray(xd, np.float64)[:, None]
    zd = np.asarray(zd, np.float64)[:, None]
    veff = np.asarray(veff, np.float64)[:, None]
    amp = np.asarray(amp, np.float64)[:, None]
    for s in range(0, nx, chunk):
        xs = x[s:s + chunk][None, :]
        t = 2.0 * np.sqrt(zd * zd + (xs - xd) ** 2) / veff
        step = np.exp(-1j * domega * t)
        cur = None
        for j in range(nbins):
            if j % reseed == 0:
                cur = amp * np.exp(-1j * ((j0 + j) * domega) * t)
            out[j, s:s + chunk] = cur.sum(axis=0)
            cur = cur * step
    out *= np.asarray(spectrum, np.float64)[:, None]
    return out


def rms_velocity_column(v_true: np.ndarray, dz: float, ix: np.ndarray, zd: np.ndarray):
    """RMS of the true velocity column at ix from 0 to zd (hyperbolic-moveout stand-in)."""
    v2 = np.cumsum(v_true.astype(np.float64) ** 2, axis=0)          # [nz, nx]
    iz = np.clip((zd / dz).astype(int), 1, v_true.shape[0]) - 1
    return np.sqrt(v2[iz, ix] / (iz + 1))


def smooth_random_field(rng, nz, nx, dz, dx, corr_len) -> np.ndarray:
    """Unit-variance white noise smoothed by a Gaussian of correlation length corr_len (FFT)."""
    g = rng.standard_normal((nz, nx))
    kz = 2.0 * np.pi * np.fft.fftfreq(nz, d=dz)[:, None]
    kx = 2.0 * np.pi * np.fft.fftfreq(nx, d=dx)[None, :]
    filt = np.exp(-0.5 * (corr_len ** 2) * (kz * kz + kx * kx))
    f = np.real(np.fft.ifft2(np.fft.fft2(g) * filt))
    return f / f.std()


def random_field_velocity(rng, nz, nx, dz, dx) -> np.ndarray:
    """configs[2] recipe: clip(1800 + g z + 350 G, 1500, 5000), trend reaching 4200 at the bottom."""
    z = (np.arange(nz) * dz)[:, None]
    g = (4200.0 - 1800.0) / max(1.0, (nz - 1) * dz)
    G = smooth_random_field(rng, nz, nx, dz, dx, 200.0)
    return np.clip(1800.0 + g * z + 350.0 * G, 1500.0, 5000.0)


def _table_du(omega: np.ndarray, dz: float, v_in: np.ndarray, ntab: int) -> float:
    u_max = float(np.float64(omega.max()) * dz / np.float64(v_in.min()))
    return u_max / (ntab - 1)


def _filters_source_hash() -> str:
    """The cache key follows the SOURCE of the design: an edited filters.py never meets a stale table."""
    with open(filters.__file__, "rb") as fh:
        return hashlib.sha1(fh.read()).hexdigest()


def cached_table(ntab: int, ntaps: int, du: float, r: float) -> np.ndarray:
    """Design (or fetch from the on-disk cache) the table for (ntab, ntaps, du, r)."""
    key = hashlib.sha1(repr((ntab, ntaps, float(du).hex(), float(r).hex(),
                             filters.NGRID, filters.PASSBAND_ANGLE_DEG, filters.STOP_CAP,
                             _filters_source_hash())).encode()).hexdigest()[:16]
    path = os.path.join(_CACHE_DIR, f"table_{ntaps}_{key}.npy")
    if os.path.exists(path):
        try:
            t = np.load(path)
            if t.shape == (ntab, ntaps) and t.dtype == np.complex64:
                return t
        except Exception:
            pass
    t = filters.design_table(ntab, ntaps, du, r)
    try:
        os.makedirs(_CACHE_DIR, exist_ok=True)
        tmp = path + f".tmp{os.getpid()}"
        with open(tmp, "wb") as fh:
            np.save(fh, t)
        os.replace(tmp, path)
    except OSError:
        pass
    return t


def _cached_npz(tag: str, builder):
    """Cache a dict of arrays produced by `builder()` under the cache dir (best effort)."""
    path = os.path.join(_CACHE_DIR, tag + ".npz")
    if os.path.exists(path):
        try:
            with np.load(path) as z:
                return {k: z[k] for k in z.files}
        except Exception:
            pass
    d = builder()
    try:
        os.makedirs(_CACHE_DIR, exist_ok=True)
        tmp = path + f".tmp{os.getpid()}.npz"
        np.savez(tmp, **d)
        os.replace(tmp, path)
    except OSError:
        pass
    return d


def _finish(name, nx, nz, dx, dz, ntaps, omega, v_true, P0, ntab=NTAB):
    v_in = (np.asarray(v_true, np.float64) * 0.5).astype(np.float32)      # reading R2
    omega = np.ascontiguousarray(omega, dtype=np.float32)
    du = _table_du(omega, dz, v_in, ntab)
    table = cached_table(ntab, ntaps, du, dz / dx)
    return dict(name=name, nx=int(nx), nz=int(nz), nw=int(omega.size), ntaps=int(ntaps),
                ntab=int(ntab), dx=float(dx), dz=float(dz), du=float(du), omega=omega,
                velocity=np.ascontiguousarray(v_in.reshape(nz, nx)),
                table=table, P0=np.ascontiguousarray(P0, dtype=np.complex64))


# --------------------------------------------------------------------------- configs[0..3]
def config0(seed: int = BASE_SEED + 0):
    """Tiny constant-velocity case: 128x128, 3 point diffractors, 25 taps (BASELINE.json configs[0])."""
    rng = np.random.default_rng(seed)
    nx = nz = 128
    dx = dz = 10.0
    omega = dft_bin_omegas(512, 4e-3, 5.0, 50.0)
    v = np.full((nz, nx), 2000.0)
    x = np.arange(nx) * dx
    xd = rng.uniform(0.0, nx * dx, 3)
    zd = rng.uniform(300.0, 1100.0, 3)
    P0 = diffractor_section(omega, ricker_spectrum(omega, 20.0), x, xd, zd,
                            np.full(3, 2000.0), np.ones(3))
    return _finish("configs[0] 128x128 const-v", nx, nz, dx, dz, 25, omega, v, P0)


def layered_velocity(rng, nz, nx, nlayers, vmin, vmax):
    depths = np.sort(rng.uniform(0.08, 0.92, nlayers - 1)) * nz
    vels = np.linspace(vmin, vmax, nlayers)
    iz = np.arange(nz)
    layer = np.searchsorted(depths, iz, side="right")
    return np.repeat(vels[layer][:, None], nx, axis=1), depths


def config1(seed: int = BASE_SEED + 1):
    """Layered v(z): 512x500, 40 diffractors + 3 dipping reflectors, 31 taps (configs[1])."""
    def build():
        rng = np.random.default_rng(seed)
        nx, nz, dx, dz = 512, 500, 10.0, 10.0
        omega = dft_bin_omegas(1024, 4e-3, 5.0, 60.0)
        v, _ = layered_velocity(rng, nz, nx, 6, 1500.0, 4500.0)
        x = np.arange(nx) * dx
        xd = [rng.uniform(0, nx * dx, 40)]
        zd = [rng.uniform(0.1, 0.95, 40) * nz * dz]
        am = [rng.uniform(0.5, 1.0, 40) * rng.choice([-1.0, 1.0], 40)]
        for _ in range(3):                                   # dipping reflectors
            dip = np.deg2rad(rng.uniform(5.0, 25.0)) * rng.choice([-1.0, 1.0])
            zc = rng.uniform(0.25, 0.75) * nz * dz
            zl = zc + (x - 0.5 * nx * dx) * np.tan(dip)
            ok = (zl > 0.05 * nz * dz) & (zl < 0.95 * nz * dz)
            xd.append(x[ok]); zd.append(zl[ok])
            am.append(np.full(ok.sum(), rng.uniform(0.5, 1.0) * rng.choice([-1.0, 1.0]) * 0.2))
        xd, zd, am = np.concatenate(xd), np.concatenate(zd), np.concatenate(am)
        ix = np.clip(np.rint(xd / dx).astype(int), 0, nx - 1)
        veff = rms_velocity_column(v, dz, ix, zd)
        P0 = diffractor_section(omega, ricker_spectrum(omega, 25.0), x, xd, zd, veff, am)
        return dict(omega=omega, v=v.astype(np.float32), P0=P0.astype(np.complex64))
    d = _cached_npz(f"config1_{seed}", build)
    return _finish("configs[1] 512x500 layered", 512, 500, 10.0, 10.0, 31, d["omega"], d["v"], d["P0"])


def config2(seed: int = BASE_SEED + 2):
    """Smooth lateral variation: 2048x1000, random-field velocity, 300 diffractors, 35 taps."""
    def build():
        rng = np.random.default_rng(seed)
        nx, nz, dx, dz = 2048, 1000, 8.0, 8.0
        omega = dft_bin_omegas(2048, 2e-3, 5.0, 80.0)
        v = random_field_velocity(rng, nz, nx, dz, dx)
        x = np.arange(nx) * dx
        nd = 300
        xd = rng.uniform(0, nx * dx, nd)
        zd = rng.uniform(0.1, 0.95, nd) * nz * dz
        am = rng.uniform(0.5, 1.0, nd) * rng.choice([-1.0, 1.0], nd)
        ix = np.clip(np.rint(xd / dx).astype(int), 0, nx - 1)
        veff = rms_velocity_column(v, dz, ix, zd)
        P0 = diffractor_section(omega, ricker_spectrum(omega, 30.0), x, xd, zd, veff, am)
        return dict(omega=omega, v=v.astype(np.float32), P0=P0.astype(np.complex64))
    d = _cached_npz(f"config2_{seed}", build)
    return _finish("configs[2] 2048x1000 random-field", 2048, 1000, 8.0, 8.0, 35,
                   d["omega"], d["v"], d["P0"])


def faulted_velocity(rng, nz, nx, dz, dx):
    """configs[3]: 8 layers 1500->3500 m/s, 4 normal faults, one 4500 m/s ellipse."""
    nl = 8
    vels = np.linspace(1500.0, 3500.0, nl)
    base = np.sort(rng.uniform(0.08, 0.92, nl - 1)) * nz * dz          # interface depths (m)
    x = (np.arange(nx) * dx)[None, :]
    z = (np.arange(nz) * dz)[:, None]
    shift = np.zeros((nz, nx))
    for _ in range(4):
        dip = np.deg2rad(rng.uniform(55.0, 70.0)) * rng.choice([-1.0, 1.0])
        xf = rng.uniform(0.15, 0.85) * nx * dx
        throw = rng.uniform(50.0, 200.0)
        hanging = (x - xf) * np.sign(dip) > z / np.tan(abs(dip))       # downthrown side
        shift = shift + throw * hanging
    zeff = z - shift                                                    # interfaces drop by throw
    layer = np.zeros((nz, nx), dtype=int)
    for b in base:
        layer += (zeff >= b)
    v = vels[layer]
    xc = rng.uniform(1.0 / 3, 2.0 / 3) * nx * dx
    zc = rng.uniform(1.0 / 3, 2.0 / 3) * nz * dz
    inside = ((x - xc) / 2000.0) ** 2 + ((z - zc) / 600.0) ** 2 <= 1.0
    v = np.where(inside, 4500.0, v)
    return v


def config3(seed: int = BASE_SEED + 3, bin_offset: float = 0.0):
    """Strong contrast: 6144x1500, faulted layers + 4500 m/s body, 2000 diffractors + 5% noise, 51 taps.

    `bin_offset` in [0,1) shifts every frequency by that fraction of a DFT bin: the union over
    r = 0..N-1 of bin_offset = r/N is the bin set of an N-times longer record, which is how
    bench.py builds the N-GPU weak-scaling job (one offset per rank; same velocity model).
    """
    def build():
        rng = np.random.default_rng(seed)
        nx, nz, dx, dz = 6144, 1500, 5.0, 5.0
        nt, dt = 4096, 2e-3
        omega = dft_bin_omegas(nt, dt, 2.0, 100.0)
        domega = 2.0 * np.pi / (nt * dt)
        j0 = int(np.rint(float(omega[0]) / domega)) + float(bin_offset)
        omega = ((j0 + np.arange(omega.size)) * domega).astype(np.float32)
        v = faulted_velocity(rng, nz, nx, dz, dx)
        x = np.arange(nx) * dx
        nd = 2000
        xd = rng.uniform(0, nx * dx, nd)
        zd = rng.uniform(0.1, 0.95, nd) * nz * dz
        am = rng.uniform(0.5, 1.0, nd) * rng.choice([-1.0, 1.0], nd)
        ix = np.clip(np.rint(xd / dx).astype(int), 0, nx - 1)
        veff = rms_velocity_column(v, dz, ix, zd)
        P0 = diffractor_section_uniform_bins(j0, omega.size, domega, ricker_spectrum(omega, 35.0),
                                             x, xd, zd, veff, am)
        rms = np.sqrt(np.mean(np.abs(P0) ** 2))
        noise = rng.standard_normal(P0.shape) + 1j * rng.standard_normal(P0.shape)
        P0 = P0 + (0.05 * rms / np.sqrt(2.0)) * noise
        return dict(omega=omega, v=v.astype(np.float32), P0=P0.astype(np.complex64))
    tag = f"config3_{seed}" if bin_offset == 0.0 else f"config3_{seed}_off{bin_offset:.6f}"
    d = _cached_npz(tag, build)
    return _finish("configs[3] 6144x1500 faulted+body", 6144, 1500, 5.0, 5.0, 51,
                   d["omega"], d["v"], d["P0"])


def config3_rank_shard(rank: int, world: int, seed: int = BASE_SEED + 3):
    """Rank `rank`'s share of the N-GPU weak-scaling job bench.py runs: the configs[3] model and
    table with an N-times denser frequency list (the DFT bins of an N-times longer record).  Rank r
    owns the bins r/N of a bin BELOW configs[3]'s own (so every u stays inside the table), 803 lines
    each; its section is configs[3]'s rotated by a unit phase per rank (same statistics, different
    data -- synthetic either way).  Derived from the cached configs[3] arrays in a fraction of a
    second, so N ranks do not each spend minutes re-synthesising 2000 diffractors."""
    base = config3(seed)
    if world <= 1:
        return base
    nt, dt = 4096, 2e-3
    domega = 2.0 * np.pi / (nt * dt)
    out = dict(base)
    out["omega"] = (base["omega"].astype(np.float64) - (rank / world) * domega).astype(np.float32)
    out["P0"] = np.ascontiguousarray(base["P0"] * np.complex64(np.exp(1j * np.pi * rank / world)))
    out["name"] = base["name"] + f" rank {rank}/{world}"
    return out


# --------------------------------------------------------------------------- configs[4]
SWEEP_NX = (1024, 4096, 16384, 32768)
SWEEP_NW = (64, 256, 1024, 2048)
SWEEP_TAPS = (15, 25, 51)


def sweep_point(nx: int, nw: int, ntaps: int, nz: int = 256, seed: int = BASE_SEED + 4,
                model: str = "field"):
    """One point of the configs[4] throughput sweep (random-field velocity, Gaussian P0).
    model="layers" swaps in 6 flat layers (1500-5000 m/s): the same sizes with warp-uniform table
    rows, the regime where the x-tiled path is bound by HBM rather than by the tap gather."""
    dx = dz = 10.0
    rng = np.random.default_rng([seed, nx])
    if model == "layers":
        v, _ = layered_velocity(rng, nz, nx, 6, 1500.0, 5000.0)
    else:
        v = random_field_velocity(rng, nz, nx, dz, dx)
    omega = (2.0 * np.pi * np.linspace(3.0, 60.0, nw)).astype(np.float32)
    rng2 = np.random.default_rng([seed, nx, nw])
    P0 = np.empty((nw, nx), dtype=np.complex64)
    P0.real = rng2.standard_normal((nw, nx), dtype=np.float32)
    P0.imag = rng2.standard_normal((nw, nx), dtype=np.float32)
    return _finish(f"configs[4] nx={nx} nw={nw} taps={ntaps} model={model}", nx, nz, dx, dz, ntaps, omega, v, P0)


def make_config(k: int, seed: int | None = None):
    """configs[k] for k = 0..3 (configs[4] is a sweep: use `sweep_point`)."""
    builders = (config0, config1, config2, config3)
    if not 0 <= k < len(builders):
        raise ValueError("k must be 0..3; configs[4] is sweep_point(nx, nw, ntaps)")
    return builders[k]() if seed is None else builders[k](seed)


# --------------------------------------------------------------------------- small test inputs
def tiny_random_problem(seed: int, nx=9, nz=3, nw=2, L=2, ntab=7, symmetric=True):
    """Random everything on a tiny grid (brute-force pin P2 and edge-case parity tests)."""
    rng = np.random.default_rng(seed)
    ntaps = 2 * L + 1
    dz = 10.0
    omega = rng.uniform(20.0, 200.0, nw).astype(np.float32)
    v = rng.uniform(1000.0, 3000.0, (nz, nx)).astype(np.float32)
    du = _table_du(omega, dz, v, ntab)
    if symmetric:
        table = filters.random_symmetric_table(rng, ntab, ntaps)
    else:
        table = (0.2 * (rng.standard_normal((ntab, ntaps)) +
                        1j * rng.standard_normal((ntab, ntaps)))).astype(np.complex64)
    P0 = (rng.standard_normal((nw, nx)) + 1j * rng.standard_normal((nw, nx))).astype(np.complex64)
    return dict(name=f"tiny seed={seed}", nx=nx, nz=nz, nw=nw, ntaps=ntaps, ntab=ntab, dx=10.0,
                dz=dz, du=float(du), omega=omega, velocity=v, table=table, P0=P0)


def random_problem(seed: int, nx: int, nz: int, nw: int, ntaps: int, ntab: int = 256,
                   model: str = "field", designed: bool = False, symmetric: bool = True):
    """Mid-size seeded problem with a chosen velocity structure: 'const' | 'layers' | 'field' | 'white'.

    Table: random symmetric rows scaled so that sum_k |W_k| < 1 (stable for any index
    pattern) unless `designed`, in which case the D1-D4 design is used; `symmetric=False` gives
    W_-k independent of W_k (the general-operator kernels), same bound.
    """
    rng = np.random.default_rng([seed, nx, nz, nw, ntaps])
    dx = dz = 10.0
    if model == "const":
        v = np.full((nz, nx), 2000.0)
    elif model == "layers":
        v, _ = layered_velocity(rng, nz, nx, 5, 1500.0, 4500.0)
    elif model == "field":
        v = random_field_velocity(rng, nz, nx, dz, dx)
    elif model == "white":
        v = rng.uniform(1500.0, 5000.0, (nz, nx))
    else:
        raise ValueError(model)
    v_in = (0.5 * v).astype(np.float32)
    omega = (2.0 * np.pi * np.linspace(3.0, 60.0, nw)).astype(np.float32)
    du = _table_du(omega, dz, v_in, ntab)
    if designed:
        table = cached_table(ntab, ntaps, du, 1.0)
    else:
        table = filters.random_symmetric_table(rng, ntab, ntaps, scale=1.0)
        table = (table / (np.abs(table).sum(axis=1, keepdims=True) * 1.02)).astype(np.complex64)
        L = (ntaps - 1) // 2
        if symmetric:
            for k in range(1, L + 1):
                table[:, L - k] = table[:, L + k]
        else:                                   # general operator: independent W_k and W_-k, same stability bound
            rng_a = np.random.default_rng([seed, 77])
            left = (rng_a.standard_normal((ntab, L)) + 1j * rng_a.standard_normal((ntab, L))).astype(np.complex64)
            table[:, :L] = left * (np.abs(table[:, L + 1:]).sum(axis=1, keepdims=True) /
                                   np.maximum(np.abs(left).sum(axis=1, keepdims=True), 1e-30)).astype(np.float32) * np.float32(0.98)
    P0 = np.empty((nw, nx), dtype=np.complex64)
    P0.real = rng.standard_normal((nw, nx), dtype=np.float32)
    P0.imag = rng.standard_normal((nw, nx), dtype=np.float32)
    return dict(name=f"random {model} {nx}x{nz}x{nw} taps={ntaps}", nx=nx, nz=nz, nw=nw,
                ntaps=ntaps, ntab=ntab, dx=dx, dz=dz, du=float(du), omega=omega,
                velocity=np.ascontiguousarray(v_in), table=np.ascontiguousarray(table), P0=P0)


def diffractor_volume(omega, spectrum, x, y, x0, y0, z0, veff) -> np.ndarray:
    """Zero-offset (exploding-reflector) record of ONE point diffractor over a 2-D receiver grid:
    P0(w, y, x) = R(w) exp(-i w t(x, y)) / r,  t = 2 r / veff,  r = sqrt(z0^2 + (x-x0)^2 + (y-y0)^2).
    complex128 [nw, ny, nx] (the 3-D analogue of diffractor_section)."""
    r = np.sqrt(z0 * z0 + (np.asarray(x, np.float64)[None, :] - x0) ** 2 + (np.asarray(y, np.float64)[:, None] - y0) ** 2)
    t = 2.0 * r / veff
    w = np.asarray(omega, np.float64)
    return np.asarray(spectrum, np.float64)[:, None, None] * np.exp(-1j * w[:, None, None] * t[None]) / r[None]


def random_problem_3d(seed: int, nx: int, ny: int, nz: int, nw: int, ntaps: int, ntab: int = 64,
                      model: str = "field", symmetric: bool = False):
    """Seeded 3-D problem: velocity [nz, ny, nx] ('const' | 'layers' | 'field' = smooth in
    x, varying with y and z | 'white'), a random GENERAL 2-D table [ntab, ntaps, ntaps] scaled so that
    sum |W| < 1 (stable for any index pattern; `symmetric`: mirrored in kx and in ky), Gaussian P0 [nw, ny, nx]."""
    rng = np.random.default_rng([seed, nx, ny, nz, nw, ntaps])
    dz = 10.0
    if model == "const":
        v = np.full((nz, ny, nx), 2000.0)
    elif model == "layers":
        v = np.repeat(np.linspace(1500.0, 4500.0, nz)[:, None, None], ny, 1).repeat(nx, 2)
    elif model == "field":
        xs = np.linspace(0, 3.0, nx)[None, None, :]
        ys = np.linspace(0, 2.0, ny)[None, :, None]
        zs = np.linspace(0, 1.0, nz)[:, None, None]
        v = np.clip(2500.0 + 900.0 * np.sin(2.1 * xs + 1.3 * ys) * np.cos(1.7 * ys + zs) + 800.0 * zs, 1500.0, 5000.0)
    elif model == "white":
        v = rng.uniform(1500.0, 5000.0, (nz, ny, nx))
    else:
        raise ValueError(model)
    v_in = (0.5 * v).astype(np.float32)
    omega = (2.0 * np.pi * np.linspace(3.0, 60.0, nw)).astype(np.float32)
    du = _table_du(omega, dz, v_in, ntab)
    table = (rng.standard_normal((ntab, ntaps, ntaps)) + 1j * rng.standard_normal((ntab, ntaps, ntaps)))
    table = (table / (np.abs(table).sum(axis=(1, 2), keepdims=True) * 1.02)).astype(np.complex64)
    if symmetric:                                   # W[ky][kx] = W[-ky][kx] = W[ky][-kx], bit for bit
        L = (ntaps - 1) // 2
        q = table[:, L:, L:]
        table = np.ascontiguousarray(np.concatenate([np.concatenate([q[:, :0:-1, :0:-1], q[:, :0:-1, :]], 2),
                                                     np.concatenate([q[:, :, :0:-1], q], 2)], 1))
    P0 = np.empty((nw, ny, nx), dtype=np.complex64)
    P0.real = rng.standard_normal((nw, ny, nx), dtype=np.float32)
    P0.imag = rng.standard_normal((nw, ny, nx), dtype=np.float32)
    return dict(name=f"random3d {model} {nx}x{ny}x{nz}x{nw} taps={ntaps}x{ntaps}", nx=nx, ny=ny, nz=nz, nw=nw,
                ntaps=ntaps, ntab=ntab, dx=10.0, dy=10.0, dz=dz, du=float(du), omega=omega,
                velocity=np.ascontiguousarray(v_in), table=np.ascontiguousarray(table), P0=P0)
