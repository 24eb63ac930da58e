"""ctypes binding of libpdm.so: same names and argument order as include/pdm.h.

Marshalling only.  If the shared library is missing this module raises -- there is no Python,
PyTorch or CPU implementation of the path to fall back to.
"""
from __future__ import annotations

import ctypes
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIB_PATH = os.path.join(_HERE, "libpdm.so")
_lib = None

PDM_OK = 0
PDM_ERR_INVALID_ARG = -1
PDM_ERR_TABLE_RANGE = -2
PDM_ERR_TABLE_ASYMMETRIC = -3
PDM_ERR_UNSUPPORTED = -4
PDM_ERR_NOMEM = -5
PDM_ERR_CUDA = -6
PDM_ERR_TOO_LARGE = -7
PDM_STATIC_MAX_SAMPLES = 1 << 20

PDM_PATH_AUTO, PDM_PATH_SMEM, PDM_PATH_TILED, PDM_PATH_NAIVE, PDM_PATH_CLUSTER, PDM_PATH_PACKED = 0, 1, 2, 3, 4, 5
PDM_TAPS_AUTO, PDM_TAPS_GLOBAL, PDM_TAPS_SLICE, PDM_TAPS_COMPACT = 0 << 4, 1 << 4, 2 << 4, 3 << 4
PDM_FORCE_GENERAL, PDM_NO_BALANCE, PDM_REQUIRE_SYMMETRIC, PDM_PRESTACK = 1 << 6, 1 << 7, 1 << 20, 1 << 21
PDM_THREADS_SHIFT, PDM_CTAS_SHIFT, PDM_TAPER_SHIFT = 8, 16, 22
PDM_TABLE_INTERP = 1 << 30

EXPORTED_SYMBOLS = ("pdm_create", "pdm_migrate", "pdm_migrate_host", "pdm_migrate_shot", "pdm_migrate_static", "pdm_destroy", "pdm_get_info",
                    "pdm_strerror", "pdm_debug_table_index", "pdm_fp32_peak",
                    "pdm_profile_enable", "pdm_profile_read",
                    "pdm_tf_create", "pdm_tf_forward", "pdm_tf_destroy", "pdm_design_table",
                    "pdm3_create", "pdm3_migrate", "pdm3_get_info", "pdm3_destroy")


class PdmInfo(ctypes.Structure):
    _fields_ = [("path", ctypes.c_int), ("taps_mode", ctypes.c_int),
                ("nx", ctypes.c_int), ("nz", ctypes.c_int), ("nw", ctypes.c_int),
                ("ntab", ctypes.c_int), ("ntaps", ctypes.c_int),
                ("grid_ctas", ctypes.c_int), ("threads_per_cta", ctypes.c_int),
                ("ctas_per_sm", ctypes.c_int), ("smem_bytes", ctypes.c_int),
                ("launches_per_migrate", ctypes.c_int), ("sm_count", ctypes.c_int),
                ("last_cuda_error", ctypes.c_int), ("table_symmetric", ctypes.c_int),
                ("samples", ctypes.c_double), ("counted_flops", ctypes.c_double),
                ("executed_lane_ops", ctypes.c_double), ("workspace_bytes", ctypes.c_double)]

    def as_dict(self) -> dict:
        return {name: getattr(self, name) for name, _ in self._fields_}


class PdmDesignOpts(ctypes.Structure):
    _fields_ = [("n_iter", ctypes.c_int), ("n_grid", ctypes.c_int), ("n_check", ctypes.c_int),
                ("passband_angle_deg", ctypes.c_double), ("kappa_cap", ctypes.c_double),
                ("stop_cap", ctypes.c_double)]


class PdmError(RuntimeError):
    def __init__(self, code: int, where: str):
        self.code = int(code)
        super().__init__(f"{where}: {pdm_strerror(code)} ({code})")


def load_library(path: str | None = None):
    """dlopen libpdm.so (built in-tree by paper_1912_05529_b200.build.build_lib). Raises if absent."""
    global _lib
    if _lib is not None and path is None:
        return _lib
    path = path or _LIB_PATH
    if not os.path.exists(path):
        raise RuntimeError(f"{path} is missing: build it with __graft_entry__.build() "
                           "(nvcc, sm_100a). There is no fallback implementation.")
    lib = ctypes.CDLL(path)
    vp, ci, cf, cd, cu = ctypes.c_void_p, ctypes.c_int, ctypes.c_float, ctypes.c_double, ctypes.c_uint
    lib.pdm_create.restype = ci
    lib.pdm_create.argtypes = [ctypes.POINTER(vp), ci, ci, ci, cf, cf, vp, vp, vp, ci, ci, cd, cu]
    lib.pdm_migrate.restype = ci
    lib.pdm_migrate.argtypes = [vp, vp, vp, vp]
    lib.pdm_migrate_shot.restype = ci
    lib.pdm_migrate_shot.argtypes = [vp, vp, vp, vp, ci, vp]
    lib.pdm_migrate_host.restype = ci
    lib.pdm_migrate_host.argtypes = [vp, vp, vp, vp]
    lib.pdm_migrate_static.restype = ci
    lib.pdm_migrate_static.argtypes = [ci, ci, ci, cf, vp, vp, vp, ci, ci, cd, vp, vp, vp]
    lib.pdm_destroy.restype = ci
    lib.pdm_destroy.argtypes = [vp]
    lib.pdm_get_info.restype = ci
    lib.pdm_get_info.argtypes = [vp, ctypes.POINTER(PdmInfo)]
    lib.pdm_strerror.restype = ctypes.c_char_p
    lib.pdm_strerror.argtypes = [ci]
    lib.pdm_debug_table_index.restype = ci
    lib.pdm_debug_table_index.argtypes = [vp, vp, ci, cd, cd, ci, vp]
    lib.pdm_fp32_peak.restype = ci
    lib.pdm_fp32_peak.argtypes = [ci, ci, ci, vp, ctypes.POINTER(cd)]
    lib.pdm_profile_enable.restype = ci
    lib.pdm_profile_enable.argtypes = [vp, ci]
    lib.pdm_profile_read.restype = ci
    lib.pdm_profile_read.argtypes = [vp, ctypes.POINTER(cf), ctypes.POINTER(cf)]
    lib.pdm_tf_create.restype = ci
    lib.pdm_tf_create.argtypes = [ctypes.POINTER(vp), ci, ci, ci, vp]
    lib.pdm_tf_forward.restype = ci
    lib.pdm_tf_forward.argtypes = [vp, vp, vp, vp]
    lib.pdm_tf_destroy.restype = ci
    lib.pdm_tf_destroy.argtypes = [vp]
    lib.pdm3_create.restype = ci
    lib.pdm3_create.argtypes = [ctypes.POINTER(vp), ci, ci, ci, ci, cf, vp, vp, vp, ci, ci, cd, cu]
    lib.pdm3_migrate.restype = ci
    lib.pdm3_migrate.argtypes = [vp, vp, vp, vp]
    lib.pdm3_get_info.restype = ci
    lib.pdm3_get_info.argtypes = [vp, ctypes.POINTER(PdmInfo)]
    lib.pdm3_destroy.restype = ci
    lib.pdm3_destroy.argtypes = [vp]
    lib.pdm_design_table.restype = ci
    lib.pdm_design_table.argtypes = [vp, ci, ci, cd, cd, ctypes.POINTER(PdmDesignOpts), vp]
    _lib = lib
    return lib


_STRERROR_LOCAL = {0: "ok", -1: "invalid argument", -2: "table range", -3: "table asymmetric",
                   -4: "unsupported", -5: "out of memory", -6: "CUDA call failed",
                   -7: "too large for the built-in scratch"}


def pdm_strerror(code: int) -> str:
    try:
        return load_library().pdm_strerror(int(code)).decode()
    except RuntimeError:
        return _STRERROR_LOCAL.get(int(code), "unknown")


# ------------------------------------------------------------------ raw calls (names of pdm.h)
def pdm_create(nx, nz, nw, dx, dz, omega, velocity, table, tab_du, flags=0):
    """-> (status, plan handle or None).  omega/velocity/table are HOST numpy arrays."""
    lib = load_library()
    omega = np.ascontiguousarray(omega, dtype=np.float32)
    velocity = np.ascontiguousarray(velocity, dtype=np.float32)
    table = np.ascontiguousarray(table, dtype=np.complex64)
    if omega.shape != (nw,) or velocity.shape != (nz, nx) or table.ndim != 2:
        return PDM_ERR_INVALID_ARG, None
    ntab, ntaps = table.shape
    handle = ctypes.c_void_p()
    rc = lib.pdm_create(ctypes.byref(handle), int(nx), int(nz), int(nw), float(dx), float(dz),
                        omega.ctypes.data, velocity.ctypes.data, table.ctypes.data,
                        int(ntab), int(ntaps), float(tab_du), int(flags))
    return rc, (handle if rc == PDM_OK else None)


def pdm_migrate(plan, P0_dev_ptr: int, image_dev_ptr: int, cuda_stream: int = 0) -> int:
    return load_library().pdm_migrate(plan, ctypes.c_void_p(P0_dev_ptr), ctypes.c_void_p(image_dev_ptr),
                                      ctypes.c_void_p(cuda_stream))


def pdm_migrate_shot(plan, src_dev_ptr: int, rec_dev_ptr: int, image_dev_ptr: int, accumulate: bool = False,
                     cuda_stream: int = 0) -> int:
    return int(load_library().pdm_migrate_shot(plan, ctypes.c_void_p(src_dev_ptr), ctypes.c_void_p(rec_dev_ptr),
                                               ctypes.c_void_p(image_dev_ptr), 1 if accumulate else 0,
                                               ctypes.c_void_p(cuda_stream)))


def pdm_migrate_host(plan, P0_host_ptr: int, image_host_ptr: int, cuda_stream: int = 0) -> int:
    return load_library().pdm_migrate_host(plan, ctypes.c_void_p(P0_host_ptr),
                                           ctypes.c_void_p(image_host_ptr), ctypes.c_void_p(cuda_stream))


def pdm_migrate_static(nx, nz, nw, dz, omega_dev_ptr: int, velocity_dev_ptr: int, table_dev_ptr: int,
                       ntab, ntaps, tab_du, P0_dev_ptr: int, image_dev_ptr: int, cuda_stream: int = 0) -> int:
    """Raw call of pdm.h's pdm_migrate_static: the migration for callers that may not allocate device
    memory (every pointer is a DEVICE address the caller owns; scratch is the library's built-in 16 MiB
    array, so nx*nw <= PDM_STATIC_MAX_SAMPLES).  Returns the status."""
    vp = ctypes.c_void_p
    return int(load_library().pdm_migrate_static(int(nx), int(nz), int(nw), float(dz), vp(omega_dev_ptr),
                                                 vp(velocity_dev_ptr), vp(table_dev_ptr), int(ntab), int(ntaps),
                                                 float(tab_du), vp(P0_dev_ptr), vp(image_dev_ptr), vp(cuda_stream)))


def migrate_static(omega, velocity, table, dz, tab_du, P0, image, stream=None):
    """pdm_migrate_static on torch CUDA tensors the caller already holds: omega float32 [nw], velocity
    float32 [nz, nx], table complex64 [ntab, ntaps], P0 complex64 [nw, nx] -> image float32 [nz, nx]
    (filled asynchronously, returned).  For code that must not trigger a device allocation: this
    wrapper creates no tensor (hence `image` is required) and the library call allocates nothing.
    All calls on one GPU share one scratch array -- keep them on one stream or order them with events."""
    import torch
    nz, nx = velocity.shape
    nw = omega.shape[0]
    ntab, ntaps = table.shape
    want = ((omega, torch.float32, (nw,)), (velocity, torch.float32, (nz, nx)), (table, torch.complex64, (ntab, ntaps)),
            (P0, torch.complex64, (nw, nx)), (image, torch.float32, (nz, nx)))
    for t, dt, shape in want:
        if not (t.is_cuda and t.dtype == dt and t.is_contiguous() and tuple(t.shape) == shape
                and t.device == P0.device):
            raise ValueError(f"expected a contiguous CUDA {dt} tensor of shape {shape} on {P0.device}")
    st = (stream or torch.cuda.current_stream(P0.device)).cuda_stream
    rc = pdm_migrate_static(nx, nz, nw, dz, omega.data_ptr(), velocity.data_ptr(), table.data_ptr(), ntab, ntaps,
                            tab_du, P0.data_ptr(), image.data_ptr(), st)
    if rc != PDM_OK:
        raise PdmError(rc, "pdm_migrate_static")
    return image


def pdm_destroy(plan) -> int:
    return load_library().pdm_destroy(plan)


def pdm_get_info(plan) -> PdmInfo:
    info = PdmInfo()
    rc = load_library().pdm_get_info(plan, ctypes.byref(info))
    if rc != PDM_OK:
        raise PdmError(rc, "pdm_get_info")
    return info


def pdm_profile_enable(plan, enable: bool = True) -> int:
    return load_library().pdm_profile_enable(plan, int(bool(enable)))


def pdm_profile_read(plan):
    """-> (main_ms, reduce_ms) of the most recent pdm_migrate (synchronises on its last event)."""
    a, b = ctypes.c_float(), ctypes.c_float()
    rc = load_library().pdm_profile_read(plan, ctypes.byref(a), ctypes.byref(b))
    if rc != PDM_OK:
        raise PdmError(rc, "pdm_profile_read")
    return float(a.value), float(b.value)


def pdm_debug_table_index(omega, velocity, dz, tab_du, ntab) -> np.ndarray:
    omega = np.ascontiguousarray(omega, dtype=np.float32)
    velocity = np.ascontiguousarray(velocity, dtype=np.float32)
    out = np.empty(omega.size, dtype=np.int32)
    rc = load_library().pdm_debug_table_index(omega.ctypes.data, velocity.ctypes.data, int(omega.size),
                                              float(dz), float(tab_du), int(ntab), out.ctypes.data)
    if rc != PDM_OK:
        raise PdmError(rc, "pdm_debug_table_index")
    return out


def pdm_fp32_peak(packed: bool = True, iters: int = 20000, repeats: int = 5, cuda_stream: int = 0) -> float:
    val = ctypes.c_double()
    rc = load_library().pdm_fp32_peak(int(bool(packed)), int(iters), int(repeats),
                                      ctypes.c_void_p(cuda_stream), ctypes.byref(val))
    if rc != PDM_OK:
        raise PdmError(rc, "pdm_fp32_peak")
    return float(val.value)


def pdm_tf_create(nt: int, nx: int, nw: int, bins):
    """-> (rc, handle or None).  bins: int32 array [nw] of DFT bins in [0, nt/2] (host)."""
    b = np.ascontiguousarray(bins, dtype=np.int32)
    h = ctypes.c_void_p()
    rc = load_library().pdm_tf_create(ctypes.byref(h), int(nt), int(nx), int(nw),
                                      b.ctypes.data_as(ctypes.c_void_p) if b.size else None)
    return rc, (h if rc == PDM_OK else None)


def pdm_tf_forward(handle, section_ptr: int, P0_ptr: int, cuda_stream: int = 0) -> int:
    return load_library().pdm_tf_forward(handle, ctypes.c_void_p(section_ptr), ctypes.c_void_p(P0_ptr),
                                         ctypes.c_void_p(cuda_stream))


def pdm_tf_destroy(handle) -> int:
    return load_library().pdm_tf_destroy(handle)


def pdm_design_table(ntab: int, ntaps: int, tab_du: float, dz_over_dx: float = 1.0, opts: dict | None = None,
                     cuda_stream: int = 0) -> np.ndarray:
    """-> complex64 [ntab, ntaps] designed on the device (D1-D4); `opts` overrides pdm_design_opts fields."""
    out = np.empty((int(ntab), int(ntaps)), dtype=np.complex64)
    o = None
    if opts is not None:
        o = PdmDesignOpts(200, 2048, 16384, 55.0, 0.8 * np.pi, 0.9995)
        for k, v in opts.items():
            setattr(o, k, v)
    rc = load_library().pdm_design_table(out.ctypes.data, int(ntab), int(ntaps), float(tab_du), float(dz_over_dx),
                                         ctypes.byref(o) if o is not None else None, ctypes.c_void_p(cuda_stream))
    if rc != PDM_OK:
        raise PdmError(rc, "pdm_design_table")
    return out


class SectionTransform:
    """Owns a pdm_tf: time-major section float32 [nt][nx] (cuda) -> P0 complex64 [nw][nx] (cuda)."""

    def __init__(self, nt: int, nx: int, bins):
        self.nt, self.nx = int(nt), int(nx)
        self.bins = np.ascontiguousarray(bins, dtype=np.int32)
        rc, self._h = pdm_tf_create(self.nt, self.nx, self.bins.size, self.bins)
        if rc != PDM_OK:
            raise PdmError(rc, "pdm_tf_create")

    def forward(self, section, out=None, stream=None):
        import torch
        if not (section.is_cuda and section.dtype == torch.float32 and section.is_contiguous()
                and tuple(section.shape) == (self.nt, self.nx)):
            raise ValueError("section must be a contiguous cuda float32 tensor [nt][nx]")
        if out is None:
            out = torch.empty((self.bins.size, self.nx), dtype=torch.complex64, device=section.device)
        elif not (out.is_cuda and out.dtype == torch.complex64 and out.is_contiguous()
                  and tuple(out.shape) == (self.bins.size, self.nx)):
            raise ValueError("out must be a contiguous cuda complex64 tensor [nw][nx]")
        st = (stream or torch.cuda.current_stream(section.device)).cuda_stream
        rc = pdm_tf_forward(self._h, section.data_ptr(), out.data_ptr(), st)
        if rc != PDM_OK:
            raise PdmError(rc, "pdm_tf_forward")
        return out

    def close(self):
        if self._h is not None:
            pdm_tf_destroy(self._h)
            self._h = None

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.close()


# ------------------------------------------------------------------ convenience wrapper
class Plan:
    """Owns a pdm_plan.  `cfg` is a workload dict in the pdm_inputs layout (or pass the fields)."""

    def __init__(self, nx, nz, nw, dx, dz, omega, velocity, table, tab_du, flags=0):
        rc, handle = pdm_create(nx, nz, nw, dx, dz, omega, velocity, table, tab_du, flags)
        if rc != PDM_OK:
            raise PdmError(rc, "pdm_create")
        self._h = handle
        self.nx, self.nz, self.nw = int(nx), int(nz), int(nw)

    @classmethod
    def from_config(cls, cfg: dict, flags: int = 0) -> "Plan":
        return cls(cfg["nx"], cfg["nz"], cfg["nw"], cfg["dx"], cfg["dz"], cfg["omega"],
                   cfg["velocity"], cfg["table"], cfg["du"], flags)

    @property
    def info(self) -> dict:
        return pdm_get_info(self._h).as_dict()

    def migrate(self, P0, image=None, stream=None):
        """P0: torch.complex64 CUDA tensor [nw, nx] -> image torch.float32 CUDA [nz, nx] (async)."""
        import torch
        if not (P0.is_cuda and P0.dtype == torch.complex64 and P0.is_contiguous()
                and tuple(P0.shape) == (self.nw, self.nx)):
            raise ValueError("P0 must be a contiguous CUDA complex64 tensor [nw, nx]")
        if image is None:
            image = torch.empty((self.nz, self.nx), dtype=torch.float32, device=P0.device)
        elif not (image.is_cuda and image.dtype == torch.float32 and image.is_contiguous()
                  and tuple(image.shape) == (self.nz, self.nx)):
            raise ValueError("image must be a contiguous CUDA float32 tensor [nz, nx]")
        st = (stream or torch.cuda.current_stream(P0.device)).cuda_stream
        rc = pdm_migrate(self._h, P0.data_ptr(), image.data_ptr(), st)
        if rc != PDM_OK:
            raise PdmError(rc, "pdm_migrate")
        return image

    def migrate_shot(self, src, rec, image=None, accumulate=False, stream=None):
        """One prestack shot (plan created with PDM_PRESTACK): src, rec torch.complex64 CUDA [nw, nx] ->
        image float32 CUDA [nz, nx], overwritten or (accumulate) added to."""
        import torch
        for t in (src, rec):
            if not (t.is_cuda and t.dtype == torch.complex64 and t.is_contiguous()
                    and tuple(t.shape) == (self.nw, self.nx)):
                raise ValueError("src and rec must be contiguous CUDA complex64 tensors [nw, nx]")
        if image is None:
            if accumulate:
                raise ValueError("accumulate needs an image to add to")
            image = torch.empty((self.nz, self.nx), dtype=torch.float32, device=rec.device)
        elif not (image.is_cuda and image.dtype == torch.float32 and image.is_contiguous()
                  and tuple(image.shape) == (self.nz, self.nx)):
            raise ValueError("image must be a contiguous CUDA float32 tensor [nz, nx]")
        st = (stream or torch.cuda.current_stream(rec.device)).cuda_stream
        rc = pdm_migrate_shot(self._h, src.data_ptr(), rec.data_ptr(), image.data_ptr(), accumulate, st)
        if rc != PDM_OK:
            raise PdmError(rc, "pdm_migrate_shot")
        return image

    def migrate_section(self, transform: "SectionTransform", section, image=None, stream=None):
        """t-x section (cuda float32 [nt][nx]) -> image: pdm_tf_forward then pdm_migrate, both
        enqueued on one stream (marshalling only; P0 is the unscaled transform)."""
        import torch
        st = stream or torch.cuda.current_stream(section.device)
        # the temporary P0 is allocated (and later freed) under `st`, so the caching allocator
        # cannot hand its block to another stream while pdm_migrate is still reading it
        with torch.cuda.stream(st):
            P0 = transform.forward(section, stream=st)
            return self.migrate(P0, image, stream=st)

    def migrate_host(self, P0_host, image_host=None, stream=None):
        """End-to-end call: HOST complex64 [nw, nx] (numpy or pinned torch) -> HOST float32 [nz, nx]."""
        import torch
        if isinstance(P0_host, np.ndarray):
            P0_host = np.ascontiguousarray(P0_host, dtype=np.complex64)
            src_ptr, shape = P0_host.ctypes.data, P0_host.shape
        else:
            if P0_host.is_cuda or P0_host.dtype != torch.complex64 or not P0_host.is_contiguous():
                raise ValueError("P0_host must be a contiguous host complex64 tensor")
            src_ptr, shape = P0_host.data_ptr(), tuple(P0_host.shape)
        if tuple(shape) != (self.nw, self.nx):
            raise ValueError("P0_host must be [nw, nx]")
        if image_host is None:
            image_host = np.empty((self.nz, self.nx), dtype=np.float32)
        if isinstance(image_host, np.ndarray):
            if image_host.dtype != np.float32 or not image_host.flags.c_contiguous:
                raise ValueError("image_host must be contiguous float32")
            dst_ptr = image_host.ctypes.data
        else:
            dst_ptr = image_host.data_ptr()
        st = (stream.cuda_stream if stream is not None
              else torch.cuda.current_stream().cuda_stream)
        rc = pdm_migrate_host(self._h, src_ptr, dst_ptr, st)
        if rc != PDM_OK:
            raise PdmError(rc, "pdm_migrate_host")
        return image_host

    def profile(self, enable: bool = True):
        rc = pdm_profile_enable(self._h, enable)
        if rc != PDM_OK:
            raise PdmError(rc, "pdm_profile_enable")

    def profile_read(self):
        return pdm_profile_read(self._h)

    def close(self):
        if self._h is not None:
            pdm_destroy(self._h)
            self._h = None

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.close()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


# ------------------------------------------------------------------ 3-D variant
def pdm3_create(nx, ny, nz, nw, dz, omega, velocity, table, tab_du, flags=0):
    """-> (status, plan handle or None).  velocity [nz, ny, nx], table [ntab, ntaps, ntaps] HOST arrays."""
    lib = load_library()
    omega = np.ascontiguousarray(omega, dtype=np.float32)
    velocity = np.ascontiguousarray(velocity, dtype=np.float32)
    table = np.ascontiguousarray(table, dtype=np.complex64)
    if omega.shape != (nw,) or velocity.shape != (nz, ny, nx) or table.ndim != 3 or table.shape[1] != table.shape[2]:
        return PDM_ERR_INVALID_ARG, None
    h = ctypes.c_void_p()
    rc = lib.pdm3_create(ctypes.byref(h), int(nx), int(ny), int(nz), int(nw), float(dz), omega.ctypes.data,
                         velocity.ctypes.data, table.ctypes.data, int(table.shape[0]), int(table.shape[1]),
                         float(tab_du), int(flags))
    return int(rc), (h if rc == PDM_OK else None)


class Plan3D:
    """Owns a pdm3_plan (3-D variant: 2-D extrapolators)."""

    def __init__(self, nx, ny, nz, nw, dz, omega, velocity, table, tab_du, flags=0):
        rc, handle = pdm3_create(nx, ny, nz, nw, dz, omega, velocity, table, tab_du, flags)
        if rc != PDM_OK:
            raise PdmError(rc, "pdm3_create")
        self._h = handle
        self.nx, self.ny, self.nz, self.nw = int(nx), int(ny), int(nz), int(nw)

    @classmethod
    def from_config(cls, cfg: dict, flags: int = 0) -> "Plan3D":
        return cls(cfg["nx"], cfg["ny"], cfg["nz"], cfg["nw"], cfg["dz"], cfg["omega"], cfg["velocity"],
                   cfg["table"], cfg["du"], flags)

    @property
    def info(self) -> dict:
        out = PdmInfo()
        rc = load_library().pdm3_get_info(self._h, ctypes.byref(out))
        if rc != PDM_OK:
            raise PdmError(rc, "pdm3_get_info")
        return out.as_dict()

    def migrate(self, P0, image=None, stream=None):
        """P0: torch.complex64 CUDA [nw, ny, nx] -> image torch.float32 CUDA [nz, ny, nx] (async)."""
        import torch
        if not (P0.is_cuda and P0.dtype == torch.complex64 and P0.is_contiguous()
                and tuple(P0.shape) == (self.nw, self.ny, self.nx)):
            raise ValueError("P0 must be a contiguous CUDA complex64 tensor [nw, ny, nx]")
        if image is None:
            image = torch.empty((self.nz, self.ny, self.nx), dtype=torch.float32, device=P0.device)
        elif not (image.is_cuda and image.dtype == torch.float32 and image.is_contiguous()
                  and tuple(image.shape) == (self.nz, self.ny, self.nx)):
            raise ValueError("image must be a contiguous CUDA float32 tensor [nz, ny, nx]")
        st = (stream or torch.cuda.current_stream(P0.device)).cuda_stream
        rc = load_library().pdm3_migrate(self._h, ctypes.c_void_p(P0.data_ptr()), ctypes.c_void_p(image.data_ptr()),
                                         ctypes.c_void_p(st))
        if rc != PDM_OK:
            raise PdmError(rc, "pdm3_migrate")
        return image

    def close(self):
        if getattr(self, "_h", None) is not None:
            load_library().pdm3_destroy(self._h)
            self._h = None

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.close()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass
