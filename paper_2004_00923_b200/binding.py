"""ctypes binding of libholo_b200.so -- same names as include/holo.h, marshalling only."""
import ctypes as C
import os

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIB = None

HOLO_OK, HOLO_ERR_ARG, HOLO_ERR_ALLOC, HOLO_ERR_CUDA, HOLO_ERR_STATE, HOLO_ERR_NOCONV = 0, -1, -2, -3, -4, -5
HOLO_WS_SUM, HOLO_WS_H, HOLO_WS_C, HOLO_WS_EVALS, HOLO_WS_V, HOLO_WS_STATUS, HOLO_WS_QX, HOLO_WS_QY = range(8)

EXPORTED_SYMBOLS = [
    "holo_create", "holo_destroy", "holo_process", "holo_submit", "holo_flush", "holo_submit_host", "holo_flush_host", "holo_push", "holo_process_host", "holo_fresnel", "holo_covariance",
    "holo_raw_covariance", "holo_set_mode", "holo_eig", "holo_project", "holo_fourier_demod", "holo_svd_filter", "holo_normalize", "holo_normalize_static", "holo_fftshift", "holo_set_range", "holo_set_assume_unitary",
    "holo_workspace", "holo_workspace_copy", "holo_status", "holo_launches_per_process", "holo_tune", "holo_profile_read", "holo_fft_group",
    "holo_last_error", "holo_version",
]


class HoloError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"holo error {code}: {msg}")
        self.code = code


def library_path():
    return os.path.join(_HERE, "libholo_b200.so")


def load_library():
    """Loads the in-tree CUDA library; fails loudly if it has not been built (no fallback)."""
    global _LIB
    if _LIB is not None:
        return _LIB
    path = library_path()
    if not os.path.exists(path):
        raise ImportError(f"{path} not found: build it with `python -m paper_2004_00923_b200.build` "
                          "(or __graft_entry__.build()); there is no CPU fallback")
    L = C.CDLL(path)
    vp, ip, dbl = C.c_void_p, C.c_int, C.c_double
    L.holo_create.restype = vp
    L.holo_create.argtypes = [ip, ip, ip, dbl, dbl, dbl, ip, ip]
    L.holo_destroy.restype = None
    L.holo_destroy.argtypes = [vp]
    L.holo_process.argtypes = [vp, vp, vp, vp]
    L.holo_process_host.argtypes = [vp, vp, vp, vp]
    L.holo_submit.argtypes = [vp, vp, vp, vp]
    L.holo_flush.argtypes = [vp, vp]
    L.holo_push.argtypes = [vp, vp, ip, vp, vp]
    L.holo_submit_host.argtypes = [vp, vp, vp, vp]
    L.holo_flush_host.argtypes = [vp, vp]
    L.holo_fresnel.argtypes = [vp, vp, vp, vp]
    L.holo_covariance.argtypes = [vp, vp, vp, vp]
    L.holo_raw_covariance.argtypes = [vp, vp, vp, vp]
    L.holo_set_mode.argtypes = [vp, ip]
    L.holo_eig.argtypes = [vp, vp, vp, vp, vp]
    L.holo_project.argtypes = [vp, vp, vp, vp, vp]
    L.holo_fourier_demod.argtypes = [vp, vp, ip, ip, vp, vp]
    L.holo_svd_filter.argtypes = [vp, vp, vp, vp, vp]
    L.holo_normalize.argtypes = [vp, vp, vp]
    L.holo_normalize_static.argtypes = [vp, vp, ip, ip, vp]
    L.holo_fftshift.argtypes = [vp, vp, vp, vp]
    L.holo_set_range.argtypes = [vp, ip, ip]
    L.holo_set_assume_unitary.argtypes = [vp, ip]
    L.holo_workspace.restype = vp
    L.holo_workspace.argtypes = [vp, ip]
    L.holo_workspace_copy.argtypes = [vp, ip, vp, C.c_ulonglong, vp]
    L.holo_status.argtypes = [vp, C.POINTER(C.c_int32), vp]
    L.holo_launches_per_process.argtypes = [vp]
    L.holo_tune.argtypes = [vp, ip, ip]
    L.holo_profile_read.argtypes = [vp, C.POINTER(C.c_double), C.POINTER(C.c_int)]
    L.holo_fft_group.argtypes = [vp]
    L.holo_last_error.restype = C.c_char_p
    L.holo_version.restype = ip
    _LIB = L
    return L


def _stream_ptr(stream):
    if stream is None:
        import torch
        return torch.cuda.current_stream().cuda_stream
    if isinstance(stream, int):
        return stream
    return stream.cuda_stream


def normalize_static(in_dev, out_dev, nx, ny, stream=None):
    """holo_normalize_static: out = in / mean(in) without a handle and without any allocation (include/holo.h)."""
    L = load_library()
    rc = L.holo_normalize_static(Holo._p(in_dev), Holo._p(out_dev), nx, ny, _stream_ptr(stream))
    if rc != 0:
        raise HoloError(rc, L.holo_last_error().decode())


class Holo:
    """One handle = one (nx, ny, T, lambda, pitch, z, k_lo, k_hi) configuration on the current device."""

    def __init__(self, nx, ny, T, lam, pitch, z, k_lo, k_hi):
        self._L = load_library()
        self._h = None
        h = self._L.holo_create(nx, ny, T, lam, pitch, z, k_lo, k_hi)
        if not h:
            raise HoloError(HOLO_ERR_ARG, self._L.holo_last_error().decode())
        self._h = h
        self.nx, self.ny, self.T = nx, ny, T

    def close(self):
        if self._h:
            self._L.holo_destroy(self._h)
            self._h = None

    __del__ = close

    def _chk(self, rc):
        if rc != 0:
            raise HoloError(rc, self._L.holo_last_error().decode())

    @staticmethod
    def _p(t):
        return t if isinstance(t, int) else t.data_ptr()

    # --- same names as the C ABI -------------------------------------------------------------
    def process(self, frames_dev, image_dev, stream=None):
        self._chk(self._L.holo_process(self._h, self._p(frames_dev), self._p(image_dev), _stream_ptr(stream)))

    def submit(self, frames_dev, image_dev, stream=None):
        self._chk(self._L.holo_submit(self._h, self._p(frames_dev), self._p(image_dev), _stream_ptr(stream)))

    def flush(self, stream=None):
        self._chk(self._L.holo_flush(self._h, _stream_ptr(stream)))

    def push(self, new_frames_dev, n_new, image_dev, stream=None):
        self._chk(self._L.holo_push(self._h, self._p(new_frames_dev), n_new, self._p(image_dev), _stream_ptr(stream)))

    def submit_host(self, frames_host, image_host, stream=None):
        self._chk(self._L.holo_submit_host(self._h, self._p(frames_host), self._p(image_host), _stream_ptr(stream)))

    def flush_host(self, stream=None):
        self._chk(self._L.holo_flush_host(self._h, _stream_ptr(stream)))

    def process_host(self, frames_host, image_host, stream=None):
        self._chk(self._L.holo_process_host(self._h, self._p(frames_host), self._p(image_host), _stream_ptr(stream)))

    def fresnel(self, frames_dev, H_dev, stream=None):
        self._chk(self._L.holo_fresnel(self._h, self._p(frames_dev), self._p(H_dev), _stream_ptr(stream)))

    def covariance(self, H_dev, C_dev, stream=None):
        self._chk(self._L.holo_covariance(self._h, self._p(H_dev), self._p(C_dev), _stream_ptr(stream)))

    def raw_covariance(self, frames_dev, C_dev, stream=None):
        self._chk(self._L.holo_raw_covariance(self._h, self._p(frames_dev), self._p(C_dev), _stream_ptr(stream)))

    def set_mode(self, mode):
        self._chk(self._L.holo_set_mode(self._h, mode))

    def eig(self, C_dev, evals_dev, V_dev, stream=None):
        self._chk(self._L.holo_eig(self._h, self._p(C_dev), self._p(evals_dev), self._p(V_dev), _stream_ptr(stream)))

    def project(self, H_dev, V_dev, image_dev, stream=None):
        self._chk(self._L.holo_project(self._h, self._p(H_dev), self._p(V_dev), self._p(image_dev), _stream_ptr(stream)))

    def fourier_demod(self, H_dev, n1, n2, image_dev, stream=None):
        self._chk(self._L.holo_fourier_demod(self._h, self._p(H_dev), n1, n2, self._p(image_dev), _stream_ptr(stream)))

    def svd_filter(self, H_dev, V_dev, Hf_dev, stream=None):
        self._chk(self._L.holo_svd_filter(self._h, self._p(H_dev), self._p(V_dev), self._p(Hf_dev), _stream_ptr(stream)))

    def normalize(self, image_dev, stream=None):
        self._chk(self._L.holo_normalize(self._h, self._p(image_dev), _stream_ptr(stream)))

    def fftshift(self, in_dev, out_dev, stream=None):
        self._chk(self._L.holo_fftshift(self._h, self._p(in_dev), self._p(out_dev), _stream_ptr(stream)))

    def set_range(self, k_lo, k_hi):
        self._chk(self._L.holo_set_range(self._h, k_lo, k_hi))

    def set_assume_unitary(self, on):
        self._chk(self._L.holo_set_assume_unitary(self._h, int(bool(on))))

    def workspace_ptr(self, which):
        return self._L.holo_workspace(self._h, which)

    def status(self, stream=None):
        buf = (C.c_int32 * 4)()
        rc = self._L.holo_status(self._h, buf, _stream_ptr(stream))
        return rc, list(buf)

    def launches_per_process(self):
        return int(self._L.holo_launches_per_process(self._h))

    def tune(self, key, value):
        self._chk(self._L.holo_tune(self._h, key, value))

    def profile_read(self):
        """[(ms, launches)] per kernel class (sum, fft_rows, fft_cols, cov_partial, cov_reduce, eig, project)."""
        ms = (C.c_double * 7)()
        cnt = (C.c_int * 7)()
        self._chk(self._L.holo_profile_read(self._h, ms, cnt))
        return [(float(ms[i]), int(cnt[i])) for i in range(7)]

    def fft_group(self):
        return int(self._L.holo_fft_group(self._h))

    # --- conveniences for tests (allocation only) ---------------------------------------------
    def workspace_tensor(self, which):
        """Copy of a workspace array as a torch tensor (test hook)."""
        import torch
        T, ny, nx = self.T, self.ny, self.nx
        shapes = {HOLO_WS_SUM: ((ny, nx), torch.int32), HOLO_WS_H: ((T, ny, nx), torch.complex64),
                  HOLO_WS_C: ((T, T), torch.complex64), HOLO_WS_EVALS: ((T,), torch.float32),
                  HOLO_WS_V: ((T, T), torch.complex64), HOLO_WS_STATUS: ((8,), torch.int32),
                  HOLO_WS_QX: ((nx,), torch.complex64), HOLO_WS_QY: ((ny,), torch.complex64)}
        shape, dtype = shapes[which]
        out = torch.empty(shape, dtype=dtype, device="cuda")
        nbytes = out.numel() * out.element_size()
        self._chk(self._L.holo_workspace_copy(self._h, which, out.data_ptr(), nbytes, _stream_ptr(None)))
        torch.cuda.current_stream().synchronize()
        return out
