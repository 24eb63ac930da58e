"""ctypes wrapper around oracle/pdm_oracle.c (plain C, FP64, OpenMP over frequency lines).

TEST INFRASTRUCTURE ONLY (see pdm_oracle.c header).  `build()` compiles the C file with gcc;
it is also called by __graft_entry__.build() -- building the checker is not using it.
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "pdm_oracle.c")
_LIB = os.path.join(_HERE, "libpdm_oracle.so")
_lib = None


def build(force: bool = False) -> str:
    """gcc -O2 -fopenmp -ffp-contract=off pdm_oracle.c -> libpdm_oracle.so (in-tree)."""
    if (not force and os.path.exists(_LIB)
            and os.path.getmtime(_LIB) >= os.path.getmtime(_SRC)):
        return _LIB
    tmp = _LIB + f".tmp{os.getpid()}"
    cmd = ["gcc", "-O2", "-std=c11", "-fopenmp", "-ffp-contract=off", "-fPIC", "-shared",
           "-o", tmp, _SRC, "-lm"]
    subprocess.run(cmd, check=True)
    os.replace(tmp, _LIB)
    return _LIB


def _load():
    global _lib
    if _lib is None:
        lib = ctypes.CDLL(build())
        lib.pdm_oracle_migrate.restype = ctypes.c_int
        lib.pdm_oracle_migrate.argtypes = [
            ctypes.c_int, ctypes.c_int, ctypes.c_int, ctypes.c_double,
            ctypes.c_void_p, ctypes.c_void_p,
            ctypes.c_void_p, ctypes.c_int, ctypes.c_int, ctypes.c_double,
            ctypes.c_void_p, ctypes.c_void_p, ctypes.c_int,
            ctypes.c_void_p, ctypes.c_void_p]
        lib.pdm_oracle_migrate_taper.restype = ctypes.c_int
        lib.pdm_oracle_migrate_taper.argtypes = [
            ctypes.c_int, ctypes.c_int, ctypes.c_int, ctypes.c_double,
            ctypes.c_void_p, ctypes.c_void_p,
            ctypes.c_void_p, ctypes.c_int, ctypes.c_int, ctypes.c_double,
            ctypes.c_void_p, ctypes.c_void_p, ctypes.c_int, ctypes.c_int,
            ctypes.c_void_p, ctypes.c_void_p]
        lib.pdm_oracle_index.restype = ctypes.c_int
        lib.pdm_oracle_index.argtypes = [ctypes.c_float, ctypes.c_float, ctypes.c_double,
                                         ctypes.c_double, ctypes.c_int]
        lib.pdm_oracle_num_threads.restype = ctypes.c_int
        lib.pdm_oracle_migrate3d.restype = ctypes.c_int
        lib.pdm_oracle_migrate3d.argtypes = [
            ctypes.c_int, ctypes.c_int, ctypes.c_int, ctypes.c_int, ctypes.c_double,
            ctypes.c_void_p, ctypes.c_void_p,
            ctypes.c_void_p, ctypes.c_int, ctypes.c_int, ctypes.c_double,
            ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p]
        lib.pdm_oracle_migrate_shot.restype = ctypes.c_int
        lib.pdm_oracle_migrate_shot.argtypes = [
            ctypes.c_int, ctypes.c_int, ctypes.c_int, ctypes.c_double,
            ctypes.c_void_p, ctypes.c_void_p,
            ctypes.c_void_p, ctypes.c_int, ctypes.c_int, ctypes.c_double,
            ctypes.c_void_p, ctypes.c_void_p, ctypes.c_int, ctypes.c_void_p]
        _lib = lib
    return _lib


def num_threads() -> int:
    return int(_load().pdm_oracle_num_threads())


def table_index(omega, velocity, dz: float, du: float, ntab: int) -> int:
    """O1 + O6 for one (omega32, v32) pair."""
    return int(_load().pdm_oracle_index(float(np.float32(omega)), float(np.float32(velocity)),
                                        float(dz), float(du), int(ntab)))


def _run(nx, nz, nw, dz, omega, velocity, table, du, P0, omega_index, want_field, ntaper=0, interp=False):
    lib = _load()
    omega = np.ascontiguousarray(omega, dtype=np.float32)
    velocity = np.ascontiguousarray(velocity, dtype=np.float32)
    table = np.ascontiguousarray(table, dtype=np.complex64)
    P0 = np.ascontiguousarray(P0, dtype=np.complex64)
    assert omega.shape == (nw,) and velocity.shape == (nz, nx) and P0.shape == (nw, nx)
    ntab, ntaps = table.shape
    if omega_index is None:
        sub, nsub, nlines = None, 0, nw
    else:
        sub = np.ascontiguousarray(omega_index, dtype=np.int32)
        nsub = nlines = int(sub.size)
        assert nsub > 0 and sub.min() >= 0 and sub.max() < nw
    image = np.zeros((nz, nx), dtype=np.float64)
    field = np.zeros((nlines, nx), dtype=np.complex128) if want_field else None
    if interp:
        assert not ntaper
        lib.pdm_oracle_migrate_interp.restype = ctypes.c_int
        lib.pdm_oracle_migrate_interp.argtypes = lib.pdm_oracle_migrate.argtypes
        rc = lib.pdm_oracle_migrate_interp(
            nx, nz, nw, float(dz), omega.ctypes.data, velocity.ctypes.data,
            table.ctypes.data, ntab, ntaps, float(du), P0.ctypes.data,
            None if sub is None else sub.ctypes.data, nsub,
            image.ctypes.data, None if field is None else field.ctypes.data)
    elif ntaper:
        rc = lib.pdm_oracle_migrate_taper(
            nx, nz, nw, float(dz), omega.ctypes.data, velocity.ctypes.data,
            table.ctypes.data, ntab, ntaps, float(du), P0.ctypes.data,
            None if sub is None else sub.ctypes.data, nsub, int(ntaper),
            image.ctypes.data, None if field is None else field.ctypes.data)
    else:
        rc = lib.pdm_oracle_migrate(
            nx, nz, nw, float(dz), omega.ctypes.data, velocity.ctypes.data,
            table.ctypes.data, ntab, ntaps, float(du), P0.ctypes.data,
            None if sub is None else sub.ctypes.data, nsub,
            image.ctypes.data, None if field is None else field.ctypes.data)
    if rc != 0:
        raise RuntimeError(f"pdm_oracle_migrate failed with code {rc}")
    return image, field


def migrate(cfg: dict, omega_index=None, ntaper: int = 0, interp: bool = False) -> np.ndarray:
    """image float64 [nz, nx] for a workload dict (pdm_inputs layout); optional omega subset;
    ntaper > 0: the absorbing edge-taper variant of R5 (reading R5b); interp: the operator is the linear
    blend of the two table rows bracketing u (reading R3c) instead of the nearest row."""
    img, _ = _run(cfg["nx"], cfg["nz"], cfg["nw"], cfg["dz"], cfg["omega"], cfg["velocity"],
                  cfg["table"], cfg["du"], cfg["P0"], omega_index, False, ntaper, interp)
    return img


def migrate_field(cfg: dict, omega_index=None, ntaper: int = 0):
    """(image, final wavefield complex128 [nlines, nx]) -- the field after the last depth step."""
    return _run(cfg["nx"], cfg["nz"], cfg["nw"], cfg["dz"], cfg["omega"], cfg["velocity"],
                cfg["table"], cfg["du"], cfg["P0"], omega_index, True, ntaper)


def migrate_shot(cfg: dict, S0, R0, image=None) -> np.ndarray:
    """Prestack shot-profile image float64 [nz, nx] (reading R17): both wavefields marched with the
    looked-up operator (the source with its conjugate), zero-lag cross-correlation imaging.
    `image`: an earlier float64 image to ADD this shot to (returned, modified in place)."""
    lib = _load()
    nx, nz, nw = cfg["nx"], cfg["nz"], cfg["nw"]
    omega = np.ascontiguousarray(cfg["omega"], dtype=np.float32)
    velocity = np.ascontiguousarray(cfg["velocity"], dtype=np.float32)
    table = np.ascontiguousarray(cfg["table"], dtype=np.complex64)
    S0 = np.ascontiguousarray(S0, dtype=np.complex64)
    R0 = np.ascontiguousarray(R0, dtype=np.complex64)
    assert omega.shape == (nw,) and velocity.shape == (nz, nx) and S0.shape == (nw, nx) and R0.shape == (nw, nx)
    acc = image is not None
    if acc:
        assert image.dtype == np.float64 and image.shape == (nz, nx) and image.flags.c_contiguous
    else:
        image = np.zeros((nz, nx), dtype=np.float64)
    ntab, ntaps = table.shape
    rc = lib.pdm_oracle_migrate_shot(nx, nz, nw, float(cfg["dz"]), omega.ctypes.data, velocity.ctypes.data,
                                     table.ctypes.data, ntab, ntaps, float(cfg["du"]),
                                     S0.ctypes.data, R0.ctypes.data, 1 if acc else 0, image.ctypes.data)
    if rc != 0:
        raise RuntimeError(f"pdm_oracle_migrate_shot failed with code {rc}")
    return image


def migrate3d(cfg: dict, want_field: bool = False):
    """3-D variant (reading R18): cfg has nx, ny, nz, nw, dz, du, omega [nw], velocity [nz, ny, nx],
    table [ntab, ntaps, ntaps] (ky slow, kx fast), P0 [nw, ny, nx].  -> image float64 [nz, ny, nx]
    (and the final wavefield complex128 [nw, ny, nx] when want_field)."""
    lib = _load()
    nx, ny, nz, nw = cfg["nx"], cfg["ny"], cfg["nz"], cfg["nw"]
    omega = np.ascontiguousarray(cfg["omega"], dtype=np.float32)
    velocity = np.ascontiguousarray(cfg["velocity"], dtype=np.float32)
    table = np.ascontiguousarray(cfg["table"], dtype=np.complex64)
    P0 = np.ascontiguousarray(cfg["P0"], dtype=np.complex64)
    ntab, ntaps, ntaps2 = table.shape
    assert ntaps == ntaps2 and omega.shape == (nw,) and velocity.shape == (nz, ny, nx) and P0.shape == (nw, ny, nx)
    image = np.zeros((nz, ny, nx), dtype=np.float64)
    field = np.zeros((nw, ny, nx), dtype=np.complex128) if want_field else None
    rc = lib.pdm_oracle_migrate3d(nx, ny, nz, nw, float(cfg["dz"]), omega.ctypes.data, velocity.ctypes.data,
                                  table.ctypes.data, ntab, ntaps, float(cfg["du"]), P0.ctypes.data,
                                  image.ctypes.data, None if field is None else field.ctypes.data)
    if rc != 0:
        raise RuntimeError(f"pdm_oracle_migrate3d failed with code {rc}")
    return (image, field) if want_field else image
