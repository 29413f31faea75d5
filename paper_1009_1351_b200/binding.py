"""ctypes binding of libtnlm.so: same names as include/tnlm.h, argument marshalling only."""
import ctypes as C
import os
from dataclasses import dataclass

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIB = None

STATUS = {0: "TNLM_OK", 1: "TNLM_INVALID_ARG", 2: "TNLM_CUDA_ERROR", 3: "TNLM_ALLOC_FAILED", 4: "TNLM_UNSUPPORTED"}

# every symbol include/tnlm.h declares
EXPORTS = ["tnlm_create", "tnlm_destroy", "tnlm_project", "tnlm_backproject", "tnlm_cgls_step",
           "tnlm_regularize_step", "tnlm_reconstruct", "tnlm_regularize_step_host",
           "tnlm_reconstruct_host", "tnlm_last_error", "tnlm_launch_count", "tnlm_version",
           "tnlm_profile_kernels", "tnlm_kernel_times", "tnlm_fbp_init", "tnlm_fma_peak",
           "tnlm_reserve", "tnlm_set_option", "tnlm_device", "tnlm_regularize_step_noalloc"]

# TNLM_NOALLOC_MAX_PIXELS of include/tnlm.h: the most pixels (n_slices * n_phase * ny * nx) regularize_step_noalloc takes
NOALLOC_MAX_PIXELS = 2621440

# tnlm_kernel_kind
KERNEL_KINDS = {0: "sweep", 1: "sweep_store", 2: "apply", 3: "project", 4: "backproject", 5: "transpose",
                6: "cgls_vector", 7: "clip", 8: "fbp"}


class TnlmError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"{STATUS.get(code, code)}: {msg}")
        self.code = code


class _CGeometry(C.Structure):
    _fields_ = [("n_views", C.c_int), ("n_bins", C.c_int), ("sid_mm", C.c_double), ("sdd_mm", C.c_double),
                ("bin_pitch_mm", C.c_double), ("bin_offset", C.c_double), ("pixel_mm", C.c_double),
                ("detector_arc", C.c_int), ("angles_rad", C.POINTER(C.c_double))]


@dataclass
class Geometry:
    """Fan-beam arc-detector geometry of one slice; angles_rad is [n_phase][n_views]."""
    n_views: int
    n_bins: int
    sid_mm: float
    sdd_mm: float
    bin_pitch_mm: float
    angles_rad: np.ndarray
    bin_offset: float = 0.0
    pixel_mm: float = 1.0
    detector_arc: int = 1


def lib_path() -> str:
    """The in-tree library, built by `python -m paper_1009_1351_b200.build`."""
    return os.path.join(_HERE, "libtnlm.so")


def library():
    """Load libtnlm.so (never builds, never falls back)."""
    global _LIB
    if _LIB is None:
        path = lib_path()
        if not os.path.exists(path):
            raise ImportError(f"{path} is missing: run `python -m paper_1009_1351_b200.build` "
                              "(there is no CPU fallback)")
        L = C.CDLL(path)
        P, I, F = C.c_void_p, C.c_int, C.c_float
        L.tnlm_create.argtypes = [C.POINTER(_CGeometry), I, I, I, I, I, F, F, C.POINTER(P)]
        L.tnlm_destroy.argtypes = [P]
        L.tnlm_project.argtypes = [P, P, P, I, P]
        L.tnlm_backproject.argtypes = [P, P, P, I, P]
        L.tnlm_cgls_step.argtypes = [P, P, P, P, I, P, I, P]
        L.tnlm_regularize_step.argtypes = [P, P, I, P, I, P]
        L.tnlm_regularize_step_noalloc.argtypes = [P, P, I, P, I, P]
        L.tnlm_reconstruct.argtypes = [P, P, P, P, I, I, I, P, I, P]
        L.tnlm_regularize_step_host.argtypes = [P, P, I, P, I, P]
        L.tnlm_reconstruct_host.argtypes = [P, P, P, P, I, I, I, P, I, P]
        L.tnlm_last_error.argtypes = [P]
        L.tnlm_last_error.restype = C.c_char_p
        L.tnlm_launch_count.argtypes = [P]
        L.tnlm_launch_count.restype = C.c_longlong
        L.tnlm_version.restype = C.c_char_p
        L.tnlm_profile_kernels.argtypes = [P, I]
        L.tnlm_fbp_init.argtypes = [P, P, P, I, P]
        L.tnlm_fma_peak.argtypes = [C.POINTER(C.c_double), P]
        L.tnlm_kernel_times.argtypes = [P, C.POINTER(C.c_float), C.POINTER(I), I, C.POINTER(I)]
        L.tnlm_reserve.argtypes = [P, I, I, I, I]
        L.tnlm_set_option.argtypes = [P, C.c_char_p, C.c_longlong]
        L.tnlm_device.argtypes = [P]
        _LIB = L
    return _LIB


def version() -> str:
    return library().tnlm_version().decode()


class Handle:
    """Owner of a tnlm_handle*; destroyed with the object."""

    def __init__(self, ptr, nx, ny, n_phase, geometry):
        self.ptr, self.nx, self.ny, self.n_phase, self.geometry = ptr, nx, ny, n_phase, geometry
        self.device = int(library().tnlm_device(ptr))          # the CUDA device the handle lives on
        self.img_per_slice = n_phase * ny * nx
        self.sino_per_slice = n_phase * geometry.n_views * geometry.n_bins if geometry is not None else 0

    def sino_count(self, n_slices):
        """Elements of a sinogram argument for n_slices (None without geometry: the library reports that)."""
        return n_slices * self.sino_per_slice if self.geometry is not None else None

    def close(self):
        if self.ptr:
            library().tnlm_destroy(self.ptr)
            self.ptr = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    @property
    def launch_count(self) -> int:
        return int(library().tnlm_launch_count(self.ptr))

    def check(self, rc):
        if rc != 0:
            raise TnlmError(rc, (library().tnlm_last_error(self.ptr) or b"").decode())


def create(geometry, nx, ny, n_phase, window, patch, h, mu) -> Handle:
    """tnlm_create: geometry may be None (TNLM-only handle)."""
    L = library()
    out = C.c_void_p()
    if geometry is None:
        rc = L.tnlm_create(None, nx, ny, n_phase, window, patch, h, mu, C.byref(out))
    else:
        ang = np.ascontiguousarray(geometry.angles_rad, dtype=np.float64)
        if ang.shape != (n_phase, geometry.n_views):
            raise ValueError(f"angles_rad must be [n_phase][n_views], got {ang.shape}")
        cg = _CGeometry(geometry.n_views, geometry.n_bins, geometry.sid_mm, geometry.sdd_mm,
                        geometry.bin_pitch_mm, geometry.bin_offset, geometry.pixel_mm,
                        geometry.detector_arc, ang.ctypes.data_as(C.POINTER(C.c_double)))
        rc = L.tnlm_create(C.byref(cg), nx, ny, n_phase, window, patch, h, mu, C.byref(out))
    if rc != 0:
        raise TnlmError(rc, (L.tnlm_last_error(None) or b"").decode())
    return Handle(out.value, nx, ny, n_phase, geometry)


# ---- device-pointer calls: torch tensors provide memory and the current stream -----------------
# Every tensor argument is checked here (dtype, contiguity, device of the handle, element count
# for the number of slices the call names): the C side sees raw pointers and cannot.
def _dev(h, t, name, count=None):
    import torch
    if t is None:
        return None
    if not (isinstance(t, torch.Tensor) and t.is_cuda and t.dtype == torch.float32 and t.is_contiguous()):
        raise TypeError(f"{name} must be a contiguous float32 CUDA tensor")
    if t.device.index != h.device:
        raise ValueError(f"{name} is on cuda:{t.device.index}, the handle was created on cuda:{h.device}")
    if count is not None and t.numel() != count:
        raise ValueError(f"{name} has {t.numel()} elements, the call needs {count}")
    return t.data_ptr()


def _stream(stream):
    import torch
    return (stream if stream is not None else torch.cuda.current_stream()).cuda_stream


def _slices(t, per_slice, name):
    n = t.numel()
    if per_slice <= 0 or n == 0 or n % per_slice:
        raise ValueError(f"{name}: size is not a whole number of slices")
    return n // per_slice


def project(h: Handle, img, sino, stream=None):
    S = _slices(img, h.img_per_slice, "img")
    h.check(library().tnlm_project(h.ptr, _dev(h, img, "img"), _dev(h, sino, "sino", h.sino_count(S)), S,
                                   _stream(stream)))
    return sino


def backproject(h: Handle, sino, img, stream=None):
    S = _slices(img, h.img_per_slice, "img")
    h.check(library().tnlm_backproject(h.ptr, _dev(h, sino, "sino", h.sino_count(S)), _dev(h, img, "img"), S,
                                       _stream(stream)))
    return img


def fbp_init(h: Handle, y, f0, stream=None):
    S = _slices(f0, h.img_per_slice, "f0")
    h.check(library().tnlm_fbp_init(h.ptr, _dev(h, y, "y", h.sino_count(S)), _dev(h, f0, "f0"), S, _stream(stream)))
    return f0


def cgls_step(h: Handle, f_in, y, w, m1, g_out, stream=None):
    S = _slices(f_in, h.img_per_slice, "f_in")
    ns = h.sino_count(S)
    h.check(library().tnlm_cgls_step(h.ptr, _dev(h, f_in, "f_in"), _dev(h, y, "y", ns), _dev(h, w, "w", ns), m1,
                                     _dev(h, g_out, "g_out", S * h.img_per_slice), S, _stream(stream)))
    return g_out


def regularize_step(h: Handle, g, m2, f_out, stream=None):
    S = _slices(g, h.img_per_slice, "g")
    h.check(library().tnlm_regularize_step(h.ptr, _dev(h, g, "g"), m2, _dev(h, f_out, "f_out", S * h.img_per_slice), S,
                                           _stream(stream)))
    return f_out


def regularize_step_noalloc(h: Handle, g, m2, f_out, stream=None):
    """tnlm_regularize_step_noalloc: regularize_step for callers that must not allocate device memory.

    Use it when cudaMalloc is off the table: all of HBM already belongs to another allocator (torch's caching
    allocator holding a large batch, say), or other streams are busy and must not be stalled by the device-wide
    synchronisation an allocation implies.  The sweeps ping-pong through a 20 MiB array compiled into the
    library instead of handle-owned buffers, and the weights are recomputed in fp32 in every sweep.  At most
    NOALLOC_MAX_PIXELS pixels per call (larger raises TnlmError, TNLM_UNSUPPORTED); the array is shared by every
    handle and stream of a device, so calls that overlap on the GPU race; make the first call on a device during
    set-up (it looks up the array's address), before any stream capture."""
    S = _slices(g, h.img_per_slice, "g")
    h.check(library().tnlm_regularize_step_noalloc(h.ptr, _dev(h, g, "g"), m2,
                                                   _dev(h, f_out, "f_out", S * h.img_per_slice), S, _stream(stream)))
    return f_out


def reconstruct(h: Handle, y, w, f0, k_outer, m1, m2, f_out, stream=None):
    S = _slices(f_out, h.img_per_slice, "f_out")
    ns = h.sino_count(S)
    h.check(library().tnlm_reconstruct(h.ptr, _dev(h, y, "y", ns), _dev(h, w, "w", ns),
                                       _dev(h, f0, "f0", S * h.img_per_slice), k_outer, m1, m2,
                                       _dev(h, f_out, "f_out"), S, _stream(stream)))
    return f_out


def reserve(h: Handle, n_slices, m1, m2, host_entry_points=False):
    """tnlm_reserve: allocate the workspace now so that later enqueue calls never allocate."""
    h.check(library().tnlm_reserve(h.ptr, n_slices, m1, m2, int(bool(host_entry_points))))


def set_option(h: Handle, name: str, value: int):
    """tnlm_set_option: a tuning option of this handle; the names and ranges are those of include/tnlm.h
    ("Stored weights and tuning knobs"), e.g. "weight_cache_mb" (0 = recompute the weights in fp32 every sweep).
    Unknown names and out-of-range values raise TnlmError (TNLM_INVALID_ARG)."""
    h.check(library().tnlm_set_option(h.ptr, name.encode(), int(value)))


def fma_peak(stream=None) -> float:
    """Measured FP32 FMA peak of the current device, TFLOP/s."""
    out = C.c_double(0.0)
    rc = library().tnlm_fma_peak(C.byref(out), _stream(stream))
    if rc != 0:
        raise TnlmError(rc, (library().tnlm_last_error(None) or b"").decode())
    return float(out.value)


def profile_kernels(h: Handle, enable: bool):
    h.check(library().tnlm_profile_kernels(h.ptr, int(bool(enable))))


def kernel_times(h: Handle, capacity: int = 16384):
    """[(kind name, milliseconds)] of the kernel launches recorded since the last call."""
    ms = (C.c_float * capacity)()
    kind = (C.c_int * capacity)()
    n = C.c_int(0)
    h.check(library().tnlm_kernel_times(h.ptr, ms, kind, capacity, C.byref(n)))
    return [(KERNEL_KINDS.get(kind[i], str(kind[i])), float(ms[i])) for i in range(min(n.value, capacity))]


# ---- host-pointer calls: CPU tensors (pinned or pageable); copies happen inside the library ----
def _host(t, name, count=None):
    import torch
    if t is None:
        return None
    if not (isinstance(t, torch.Tensor) and not t.is_cuda and t.dtype == torch.float32 and t.is_contiguous()):
        raise TypeError(f"{name} must be a contiguous float32 CPU tensor")
    if count is not None and t.numel() != count:
        raise ValueError(f"{name} has {t.numel()} elements, the call needs {count}")
    return t.data_ptr()


def regularize_step_host(h: Handle, g_host, m2, f_out_host, stream=None):
    S = _slices(g_host, h.img_per_slice, "g_host")
    h.check(library().tnlm_regularize_step_host(h.ptr, _host(g_host, "g_host"), m2,
                                                _host(f_out_host, "f_out_host", S * h.img_per_slice), S,
                                                _stream(stream)))
    return f_out_host


def reconstruct_host(h: Handle, y_host, w_host, f0_host, k_outer, m1, m2, f_out_host, stream=None):
    S = _slices(f_out_host, h.img_per_slice, "f_out_host")
    ns = h.sino_count(S)
    h.check(library().tnlm_reconstruct_host(h.ptr, _host(y_host, "y_host", ns), _host(w_host, "w_host", ns),
                                            _host(f0_host, "f0_host", S * h.img_per_slice), k_outer, m1, m2,
                                            _host(f_out_host, "f_out_host"), S, _stream(stream)))
    return f_out_host
