"""Thin ctypes binding over liblinmin.so (include/linmin.h).  Argument marshalling only.

Every step of the path runs in the CUDA kernels of csrc/; this module allocates nothing but the
output tensors (PyTorch is used for device memory and streams) and never falls back to a CPU or
PyTorch implementation: if the library or a CUDA device is missing, calls raise.
Function names mirror the C ABI: unmix, unmix_lib, unmix_host, library_create, library_destroy.
"""
from __future__ import annotations

import ctypes
import os
from typing import Optional

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "liblinmin.so")

OK = 0
ERR_INVALID_ARGUMENT = -1
ERR_UNSUPPORTED_SIZE = -2
ERR_NOT_IMPLEMENTED = -3
ERR_CUDA = -4
ERR_OUT_OF_MEMORY = -5
ERR_LIBRARY_NONFINITE = -6
ERR_COVARIANCE = -7
ERR_STATIC_SCRATCH = -8
STATIC_MAX_R = 64
CONSTRAINT_SUM_TO_ONE, CONSTRAINT_SUM_LOWER_THAN_ONE, CONSTRAINT_POSITIVITY_ONLY = 0, 1, 2
WEIGHTING_NONE, WEIGHTING_SHARED_COVARIANCE, WEIGHTING_SHARED_DIAGONAL = 0, 1, 2
WARN_RANK_DEFICIENT = 1

INFO_CONVERGED = 0x01
INFO_MAX_ITER = 0x02
INFO_NONFINITE_INPUT = 0x04
INFO_CHOL_REGULARISED = 0x08
INFO_FINISH_FALLBACK = 0x10
INFO_BAD_SIGMA = 0x20
INFO_LIBRARY_NONFINITE = 0x40
INFO_COVARIANCE = 0x80

EXPORTS = ["linmin_version", "linmin_strerror", "linmin_library_create", "linmin_library_destroy",
           "linmin_library_last_launches", "linmin_library_enable_timing", "linmin_library_last_timing",
           "linmin_trim_memory",
           "linmin_unmix_lib", "linmin_unmix", "linmin_unmix_host",
           "linmin_additional_spectra", "linmin_detection_thresholds", "linmin_detection_thresholds_ex", "linmin_detection_thresholds_static", "linmin_detect", "linmin_second_pass",
           "linmin_autofit"]


class LinminOpts(ctypes.Structure):
    _fields_ = [("struct_size", ctypes.c_uint32), ("stream", ctypes.c_void_p),
                ("ldY", ctypes.c_int64), ("sigma_pixel_stride", ctypes.c_int64),
                ("constraint", ctypes.c_int32), ("weighting", ctypes.c_int32),
                ("max_iter", ctypes.c_int32), ("gap_tol", ctypes.c_float),
                ("feas_tol", ctypes.c_float), ("info_out", ctypes.c_void_p),
                ("deterministic", ctypes.c_int32), ("reserved", ctypes.c_int32), ("cov", ctypes.c_void_p)]


class LinminError(RuntimeError):
    def __init__(self, code: int, msg: str):
        super().__init__(f"linmin error {code}: {msg}")
        self.code = code


_lib = None


def load() -> ctypes.CDLL:
    """Load liblinmin.so (built in-tree by paper_1402_2518_b200.build).  Fails loudly if missing."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise ImportError(f"{LIB_PATH} is missing: run `python -m paper_1402_2518_b200.build` "
                              "(there is no CPU fallback)")
        lib = ctypes.CDLL(LIB_PATH)
        P, I64, I32 = ctypes.c_void_p, ctypes.c_int64, ctypes.c_int32
        lib.linmin_version.restype = ctypes.c_int
        lib.linmin_strerror.restype = ctypes.c_char_p
        lib.linmin_strerror.argtypes = [ctypes.c_int]
        lib.linmin_library_create.argtypes = [P, I32, I32, ctypes.POINTER(LinminOpts), ctypes.POINTER(P)]
        lib.linmin_library_destroy.argtypes = [P]
        lib.linmin_library_destroy.restype = None
        lib.linmin_library_last_launches.argtypes = [P]
        lib.linmin_library_enable_timing.argtypes = [P, ctypes.c_int]
        lib.linmin_library_last_timing.argtypes = [P, ctypes.POINTER(ctypes.c_float), ctypes.POINTER(ctypes.c_float)]
        lib.linmin_unmix_lib.argtypes = [P, P, P, I64, ctypes.POINTER(LinminOpts), P, P, P]
        lib.linmin_unmix.argtypes = [P, P, P, I64, I32, I32, ctypes.POINTER(LinminOpts), P, P, P]
        lib.linmin_unmix_host.argtypes = [P, P, P, I64, I32, I32, ctypes.POINTER(LinminOpts), P, P, P]
        lib.linmin_additional_spectra.argtypes = [P, I32, I32, P, I32, I32, P]
        lib.linmin_detection_thresholds.argtypes = [P, P, I64, I32, P, P]
        lib.linmin_detection_thresholds_ex.argtypes = [P, P, I64, I32, I32, P, P]
        lib.linmin_detection_thresholds_static.argtypes = [P, P, I64, I32, P, P]
        lib.linmin_detect.argtypes = [P, P, P, P, ctypes.c_float, I64, I32, P, P, P]
        lib.linmin_second_pass.argtypes = [P, P, P, I64, I32, I32, P, ctypes.POINTER(LinminOpts), P, P, P]
        lib.linmin_autofit.argtypes = [P, I32, I32, P, P, P]
        _lib = lib
    return _lib


def strerror(code: int) -> str:
    return load().linmin_strerror(int(code)).decode()


def version() -> int:
    return int(load().linmin_version())


def _check(code: int) -> int:
    if code < 0:
        raise LinminError(code, strerror(code))
    return code


def _torch():
    import torch
    return torch


def _dev_ptr(t, name, dtype=None):
    torch = _torch()
    if t is None:
        return None
    if not t.is_cuda:
        raise ValueError(f"{name} must be a CUDA tensor")
    if not t.is_contiguous():
        raise ValueError(f"{name} must be contiguous")
    if t.dtype != (dtype or torch.float32):
        raise ValueError(f"{name} must be {dtype or torch.float32}")
    return ctypes.c_void_p(t.data_ptr())


def _make_opts(stream=None, ldY=0, sigma_pixel_stride=0, constraint=0, weighting=0, max_iter=0,
               gap_tol=0.0, feas_tol=0.0, info_ptr=None, cov_ptr=None) -> LinminOpts:
    o = LinminOpts()
    o.struct_size = ctypes.sizeof(LinminOpts)
    o.stream = stream
    o.ldY = ldY
    o.sigma_pixel_stride = sigma_pixel_stride
    o.constraint = constraint
    o.weighting = weighting
    o.max_iter = max_iter
    o.gap_tol = gap_tol
    o.feas_tol = feas_tol
    o.info_out = info_ptr
    o.deterministic = 1
    o.cov = cov_ptr
    return o


def _weighting_of(cov, L, cuda, device=None):
    """(weighting code, pointer) of a covariance argument: None, (L,) noise std, or (L, L) covariance matrix."""
    torch = _torch()
    if cov is None:
        return WEIGHTING_NONE, None
    if cov.dim() == 1:
        _check_tensor(cov, "cov", (L,), torch.float32, cuda, device)
        return WEIGHTING_SHARED_DIAGONAL, cov.data_ptr()
    _check_tensor(cov, "cov", (L, L), torch.float32, cuda, device)
    return WEIGHTING_SHARED_COVARIANCE, cov.data_ptr()


def _sigma_stride(sigma, N, L):
    if sigma is None:
        return 0
    if sigma.dim() == 1:
        if sigma.shape[0] != L:
            raise ValueError("shared sigma must have L entries")
        return 0
    if tuple(sigma.shape) != (N, L):
        raise ValueError("per-pixel sigma must be (N, L)")
    return L


class Library:
    """linmin_library handle: once-per-library precompute kept on the device."""

    def __init__(self, A, constraint=0, cov=None):
        torch = _torch()
        if A.dim() != 2:
            raise ValueError("A must be (L, R)")
        self.L, self.R = int(A.shape[0]), int(A.shape[1])
        _check_tensor(A, "A", (self.L, self.R), torch.float32, True)
        self._h = ctypes.c_void_p()
        self.device = A.device
        self.constraint = int(constraint)
        self.weighting, cov_ptr = _weighting_of(cov, self.L, True, A.device)
        with torch.cuda.device(A.device):
            o = _make_opts(stream=torch.cuda.current_stream().cuda_stream, constraint=self.constraint,
                           weighting=self.weighting, cov_ptr=cov_ptr)
            self.status = _check(load().linmin_library_create(_dev_ptr(A, "A"), self.L, self.R,
                                                              ctypes.byref(o), ctypes.byref(self._h)))

    def last_launches(self) -> int:
        return int(load().linmin_library_last_launches(self._h))

    def enable_timing(self, enable: bool = True) -> None:
        _check(load().linmin_library_enable_timing(self._h, int(enable)))

    def last_timing(self):
        """(ipls_ms, finish_ms) of the last unmix_lib call; blocks until its kernels have finished."""
        a, b = ctypes.c_float(), ctypes.c_float()
        _check(load().linmin_library_last_timing(self._h, ctypes.byref(a), ctypes.byref(b)))
        return float(a.value), float(b.value)

    def destroy(self):
        if self._h:
            load().linmin_library_destroy(self._h)
            self._h = ctypes.c_void_p()

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass


def trim_memory() -> None:
    """Return the library's cached staging memory to the driver."""
    _check(load().linmin_trim_memory())


def library_create(A, constraint=0, cov=None) -> Library:
    """constraint: CONSTRAINT_*; cov: None | (L,) per-channel noise std | (L, L) covariance (the renormalised problem)."""
    return Library(A, constraint, cov)


def library_destroy(lib: Library) -> None:
    lib.destroy()


def _check_tensor(t, name, shape, dtype, cuda, device=None):
    """Argument marshalling guard: the C ABI reads and writes exactly shape x dtype through data_ptr()."""
    if t is None:
        return
    if tuple(t.shape) != tuple(shape):
        raise ValueError(f"{name} must have shape {tuple(shape)}, got {tuple(t.shape)}")
    if t.dtype != dtype:
        raise ValueError(f"{name} must be {dtype}, got {t.dtype}")
    if not t.is_contiguous():
        raise ValueError(f"{name} must be contiguous")
    if bool(t.is_cuda) != bool(cuda):
        raise ValueError(f"{name} must be a {'CUDA' if cuda else 'CPU'} tensor")
    if cuda and device is not None and t.device != device:
        raise ValueError(f"{name} must live on {device}")


def _check_outputs(N, R, coeffs, csig, resid, info, cuda, device=None):
    torch = _torch()
    _check_tensor(coeffs, "out['coeffs']", (N, R), torch.float32, cuda, device)
    _check_tensor(csig, "out['coeff_sigma']", (N, R), torch.float32, cuda, device)
    _check_tensor(resid, "out['resid']", (N,), torch.float32, cuda, device)
    _check_tensor(info, "out['info']", (N,), torch.int32, cuda, device)


def _check_sigma(sigma, N, L, cuda, device=None):
    torch = _torch()
    if sigma is None:
        return
    if sigma.dim() == 1:
        _check_tensor(sigma, "sigma", (L,), torch.float32, cuda, device)
    else:
        _check_tensor(sigma, "sigma", (N, L), torch.float32, cuda, device)


def _alloc_outputs(N, R, device, want_sigma, want_resid, want_info, out):
    torch = _torch()
    out = dict(out or {})
    coeffs = out.get("coeffs")
    if coeffs is None:
        coeffs = torch.empty((N, R), dtype=torch.float32, device=device)
    csig = out.get("coeff_sigma")
    if csig is None and want_sigma:
        csig = torch.empty((N, R), dtype=torch.float32, device=device)
    resid = out.get("resid")
    if resid is None and want_resid:
        resid = torch.empty((N,), dtype=torch.float32, device=device)
    info = out.get("info")
    if info is None and want_info:
        info = torch.empty((N,), dtype=torch.int32, device=device)
    _check_outputs(N, R, coeffs, csig, resid, info, True, device)
    return coeffs, csig, resid, info


def unmix_lib(lib: Library, Y, sigma=None, *, want_sigma=True, want_resid=True, want_info=True,
              out: Optional[dict] = None, max_iter=0, gap_tol=0.0, feas_tol=0.0):
    """linmin_unmix_lib.  Y (N, L) CUDA float32 (rows may be strided); returns
    (coeffs, coeff_sigma, resid, info, status); enqueued on the current stream, not synchronised."""
    torch = _torch()
    if Y.dim() != 2 or Y.shape[1] != lib.L:
        raise ValueError("Y must be (N, L)")
    N = int(Y.shape[0])
    ldY = int(Y.stride(0)) if N > 1 else lib.L
    if Y.stride(1) != 1 and N > 0:
        raise ValueError("spectra must be contiguous along channels")
    if not Y.is_cuda or Y.dtype != torch.float32:
        raise ValueError("Y must be a CUDA float32 tensor")
    if Y.device != lib.device:
        raise ValueError(f"Y must live on the library's device {lib.device}")
    _check_sigma(sigma, N, lib.L, True, Y.device)
    coeffs, csig, resid, info = _alloc_outputs(N, lib.R, Y.device, want_sigma, want_resid, want_info, out)
    with torch.cuda.device(Y.device):
        o = _make_opts(stream=torch.cuda.current_stream().cuda_stream, ldY=ldY,
                       sigma_pixel_stride=_sigma_stride(sigma, N, lib.L), constraint=lib.constraint,
                       weighting=lib.weighting, max_iter=max_iter, gap_tol=gap_tol, feas_tol=feas_tol,
                       info_ptr=None if info is None else info.data_ptr())
        yp = ctypes.c_void_p(Y.data_ptr()) if N > 0 else None
        st = _check(load().linmin_unmix_lib(lib._h, yp, _dev_ptr(sigma, "sigma"), N, ctypes.byref(o),
                                            _dev_ptr(coeffs, "coeffs"), _dev_ptr(csig, "coeff_sigma"),
                                            _dev_ptr(resid, "resid")))
    return coeffs, csig, resid, info, st


def unmix(A, Y, sigma=None, *, want_sigma=True, want_resid=True, want_info=True,
          out: Optional[dict] = None, max_iter=0, gap_tol=0.0, feas_tol=0.0, constraint=0, cov=None):
    """linmin_unmix (one-shot: precompute + solve).  All tensors CUDA float32.
    constraint: CONSTRAINT_*; cov: None | (L,) noise std | (L, L) covariance (renormalised problem, eq. 5-6)."""
    torch = _torch()
    if A.dim() != 2:
        raise ValueError("A must be (L, R)")
    L, R = int(A.shape[0]), int(A.shape[1])
    _check_tensor(A, "A", (L, R), torch.float32, True)
    if Y.dim() != 2 or int(Y.shape[1]) != L:
        raise ValueError("Y must be (N, L)")
    N = int(Y.shape[0])
    _check_tensor(Y, "Y", (N, L), torch.float32, True, A.device)
    _check_sigma(sigma, N, L, True, A.device)
    coeffs, csig, resid, info = _alloc_outputs(N, R, A.device, want_sigma, want_resid, want_info, out)
    weighting, cov_ptr = _weighting_of(cov, L, True, A.device)
    with torch.cuda.device(A.device):
        o = _make_opts(stream=torch.cuda.current_stream().cuda_stream, ldY=0,
                       sigma_pixel_stride=_sigma_stride(sigma, N, L), constraint=constraint,
                       weighting=weighting, max_iter=max_iter, gap_tol=gap_tol, feas_tol=feas_tol,
                       info_ptr=None if info is None else info.data_ptr(), cov_ptr=cov_ptr)
        st = _check(load().linmin_unmix(_dev_ptr(A, "A"), _dev_ptr(Y, "Y") if N > 0 else None,
                                        _dev_ptr(sigma, "sigma"), N, L, R, ctypes.byref(o),
                                        _dev_ptr(coeffs, "coeffs"), _dev_ptr(csig, "coeff_sigma"),
                                        _dev_ptr(resid, "resid")))
    return coeffs, csig, resid, info, st


def unmix_host(A, Y, sigma=None, *, want_sigma=True, want_resid=True, want_info=False,
               out: Optional[dict] = None, max_iter=0, gap_tol=0.0, feas_tol=0.0, constraint=0, cov=None):
    """linmin_unmix_host: numpy arrays or CPU tensors (pinned memory gives full copy bandwidth).
    Blocks until the outputs are complete.  Returns (coeffs, coeff_sigma, resid, info, status) as
    CPU tensors (pinned when freshly allocated)."""
    torch = _torch()

    def as_cpu(x, name):
        if x is None:
            return None
        t = torch.as_tensor(x)
        if t.is_cuda or t.dtype != torch.float32 or not t.is_contiguous():
            raise ValueError(f"{name} must be a contiguous CPU float32 array")
        return t

    A, Y, sigma, cov = as_cpu(A, "A"), as_cpu(Y, "Y"), as_cpu(sigma, "sigma"), as_cpu(cov, "cov")
    if A.dim() != 2:
        raise ValueError("A must be (L, R)")
    L, R = int(A.shape[0]), int(A.shape[1])
    if Y.dim() != 2 or int(Y.shape[1]) != L:
        raise ValueError("Y must be (N, L)")
    N = int(Y.shape[0])
    _check_sigma(sigma, N, L, False)
    out = dict(out or {})
    pin = torch.cuda.is_available()

    def host_empty(shape, dtype):
        return torch.empty(shape, dtype=dtype, pin_memory=pin)

    coeffs = out.get("coeffs") if out.get("coeffs") is not None else host_empty((N, R), torch.float32)
    csig = out.get("coeff_sigma")
    if csig is None and want_sigma:
        csig = host_empty((N, R), torch.float32)
    resid = out.get("resid")
    if resid is None and want_resid:
        resid = host_empty((N,), torch.float32)
    info = out.get("info")
    if info is None and want_info:
        info = host_empty((N,), torch.int32)
    _check_outputs(N, R, coeffs, csig, resid, info, False)
    weighting, cov_ptr = _weighting_of(cov, L, False)
    o = _make_opts(ldY=0, sigma_pixel_stride=_sigma_stride(sigma, N, L), max_iter=max_iter, constraint=constraint,
                   weighting=weighting, cov_ptr=cov_ptr,
                   gap_tol=gap_tol, feas_tol=feas_tol, info_ptr=None if info is None else info.data_ptr())

    def hp(t):
        return None if t is None else ctypes.c_void_p(t.data_ptr())

    st = _check(load().linmin_unmix_host(hp(A), hp(Y) if N > 0 else None, hp(sigma), N, L, R,
                                         ctypes.byref(o), hp(coeffs), hp(csig), hp(resid)))
    return coeffs, csig, resid, info, st


# ------------------------------------------------------------------ NEXT rows 3-4: library builder, detection, autofit
def _stream():
    return ctypes.c_void_p(_torch().cuda.current_stream().cuda_stream)


def additional_spectra(L, n_extra, device, wavelength=None, out=None, col0=0):
    """linmin_additional_spectra: (L, n_extra) tensor, or columns col0.. of `out` (L, ld)."""
    torch = _torch()
    if out is None:
        out = torch.empty((L, n_extra), dtype=torch.float32, device=device)
        col0 = 0
    _check_tensor(out, "out", (L, out.shape[1]), torch.float32, True)
    _check_tensor(wavelength, "wavelength", (L,), torch.float32, True, out.device)
    with torch.cuda.device(out.device):
        _check(load().linmin_additional_spectra(_dev_ptr(wavelength, "wavelength"), L, n_extra, _dev_ptr(out, "out"),
                                                int(out.shape[1]), col0, _stream()))
    return out


def build_library(A_ref, n_extra, wavelength=None):
    """The reference spectra (L, R0) followed by the paper's 4 or 12 additional spectra: (L, R0 + n_extra)."""
    torch = _torch()
    L, R0 = int(A_ref.shape[0]), int(A_ref.shape[1])
    out = torch.empty((L, R0 + n_extra), dtype=torch.float32, device=A_ref.device)
    out[:, :R0] = A_ref
    return additional_spectra(L, n_extra, A_ref.device, wavelength, out, R0)


def detection_thresholds(coeffs, present, whole_class=False):
    """linmin_detection_thresholds[_ex] (eq. 8): coeffs (N, R) float32, present (N, R) uint8 / bool -> (R,) float32.
    whole_class: every pixel of a class enters, exact zeros included, instead of the detections only."""
    torch = _torch()
    N, R = int(coeffs.shape[0]), int(coeffs.shape[1])
    present = present.to(torch.uint8)
    _check_tensor(coeffs, "coeffs", (N, R), torch.float32, True)
    _check_tensor(present, "present", (N, R), torch.uint8, True, coeffs.device)
    thr = torch.empty((R,), dtype=torch.float32, device=coeffs.device)
    with torch.cuda.device(coeffs.device):
        _check(load().linmin_detection_thresholds_ex(_dev_ptr(coeffs, "coeffs"), ctypes.c_void_p(present.data_ptr()), N, R,
                                                     int(bool(whole_class)), _dev_ptr(thr, "thr"), _stream()))
    return thr


def detection_thresholds_static(coeffs, present, out):
    """linmin_detection_thresholds_static: eq. 8 thresholds without any device allocation by the library.

    For callers whose GPU memory is all spoken for (an application-owned arena) or who cannot afford an
    allocation's stall: the partial sums live in a fixed 384 KiB array inside liblinmin.so.  Nothing is allocated
    here either: `present` must already be uint8 (or bool, viewed in place) and `out` is the caller's (R,) float32
    tensor, returned filled.  R <= STATIC_MAX_R (64), else LinminError(ERR_STATIC_SCRATCH).  Calls on one device
    share the array: keep them in stream order, and make the first one before any stream capture."""
    torch = _torch()
    N, R = int(coeffs.shape[0]), int(coeffs.shape[1])
    if present.dtype == torch.bool:
        present = present.view(torch.uint8)
    _check_tensor(coeffs, "coeffs", (N, R), torch.float32, True)
    _check_tensor(present, "present", (N, R), torch.uint8, True, coeffs.device)
    _check_tensor(out, "out", (R,), torch.float32, True, coeffs.device)
    with torch.cuda.device(coeffs.device):
        _check(load().linmin_detection_thresholds_static(_dev_ptr(coeffs, "coeffs"), ctypes.c_void_p(present.data_ptr()),
                                                         N, R, _dev_ptr(out, "out"), _stream()))
    return out


def detect(coeffs, coeff_sigma, resid, thresholds, rms_max):
    """linmin_detect: (mask (N, R) uint8, counts (R,) int64)."""
    torch = _torch()
    N, R = int(coeffs.shape[0]), int(coeffs.shape[1])
    _check_tensor(coeffs, "coeffs", (N, R), torch.float32, True)
    _check_tensor(coeff_sigma, "coeff_sigma", (N, R), torch.float32, True, coeffs.device)
    _check_tensor(resid, "resid", (N,), torch.float32, True, coeffs.device)
    _check_tensor(thresholds, "thresholds", (R,), torch.float32, True, coeffs.device)
    mask = torch.empty((N, R), dtype=torch.uint8, device=coeffs.device)
    counts = torch.empty((R,), dtype=torch.int64, device=coeffs.device)
    with torch.cuda.device(coeffs.device):
        _check(load().linmin_detect(_dev_ptr(coeffs, "coeffs"), _dev_ptr(coeff_sigma, "coeff_sigma"), _dev_ptr(resid, "resid"),
                                    _dev_ptr(thresholds, "thresholds"), ctypes.c_float(rms_max), N, R,
                                    ctypes.c_void_p(mask.data_ptr()), ctypes.c_void_p(counts.data_ptr()), _stream()))
    return mask, counts


def second_pass(A, Y, sigma, keep, *, constraint=0, cov=None):
    """linmin_second_pass: keep (R,) uint8 / bool.  Returns (coeffs, coeff_sigma, resid, status)."""
    torch = _torch()
    L, R = int(A.shape[0]), int(A.shape[1])
    N = int(Y.shape[0])
    _check_tensor(A, "A", (L, R), torch.float32, True)
    _check_tensor(Y, "Y", (N, L), torch.float32, True, A.device)
    _check_sigma(sigma, N, L, True, A.device)
    keep = keep.to(torch.uint8)
    _check_tensor(keep, "keep", (R,), torch.uint8, True, A.device)
    coeffs, csig, resid, _ = _alloc_outputs(N, R, A.device, True, True, False, None)
    weighting, cov_ptr = _weighting_of(cov, L, True, A.device)
    with torch.cuda.device(A.device):
        o = _make_opts(stream=torch.cuda.current_stream().cuda_stream, sigma_pixel_stride=_sigma_stride(sigma, N, L),
                       constraint=constraint, weighting=weighting, cov_ptr=cov_ptr)
        st = _check(load().linmin_second_pass(_dev_ptr(A, "A"), _dev_ptr(Y, "Y"), _dev_ptr(sigma, "sigma"), N, L, R,
                                              ctypes.c_void_p(keep.data_ptr()), ctypes.byref(o), _dev_ptr(coeffs, "coeffs"),
                                              _dev_ptr(csig, "coeff_sigma"), _dev_ptr(resid, "resid")))
    return coeffs, csig, resid, st


def autofit(A):
    """linmin_autofit (eq. 7): (E_ls, E_nn), each (L, R): residues of every endmember against the others."""
    torch = _torch()
    L, R = int(A.shape[0]), int(A.shape[1])
    _check_tensor(A, "A", (L, R), torch.float32, True)
    E_ls = torch.empty((L, R), dtype=torch.float32, device=A.device)
    E_nn = torch.empty((L, R), dtype=torch.float32, device=A.device)
    with torch.cuda.device(A.device):
        _check(load().linmin_autofit(_dev_ptr(A, "A"), L, R, _stream(), _dev_ptr(E_ls, "E_ls"), _dev_ptr(E_nn, "E_nn")))
    return E_ls, E_nn
