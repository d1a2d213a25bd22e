"""ctypes loader for oracle/libholo_oracle.so (double-precision C++ oracle; see holo_oracle.h).

TEST INFRASTRUCTURE ONLY.  Argument marshalling only -- all arithmetic is in holo_oracle.cpp.
Complex arrays cross the boundary as numpy complex128 (interleaved doubles).
"""
import ctypes as C
import os
import subprocess
import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIB = None


def build(force=False):
    """Compile the oracle with g++ (idempotent)."""
    so = os.path.join(_HERE, "libholo_oracle.so")
    src = os.path.join(_HERE, "holo_oracle.cpp")
    hdr = os.path.join(_HERE, "holo_oracle.h")
    if force or not os.path.exists(so) or os.path.getmtime(so) < max(os.path.getmtime(src), os.path.getmtime(hdr)):
        subprocess.check_call(["g++", "-O2", "-std=c++17", "-fopenmp", "-fPIC", "-shared", "-o", so, src], cwd=_HERE)
    return so


def _lib():
    global _LIB
    if _LIB is None:
        _LIB = C.CDLL(build())
        dp, u16p, ip = C.POINTER(C.c_double), C.POINTER(C.c_uint16), C.c_int
        L = _LIB
        L.oracle_fft2.argtypes = [dp, ip, ip]
        L.oracle_chirp.argtypes = [ip, ip, C.c_double, C.c_double, C.c_double, dp]
        L.oracle_mean_subtract.argtypes = [u16p, ip, ip, ip, dp]
        L.oracle_fresnel.argtypes = [u16p, ip, ip, ip, C.c_double, C.c_double, C.c_double, dp]
        L.oracle_fresnel_field.argtypes = [dp, ip, ip, C.c_double, C.c_double, C.c_double, dp]
        L.oracle_covariance.argtypes = [dp, C.c_longlong, ip, dp]
        L.oracle_eig.argtypes = [dp, ip, dp, dp]
        L.oracle_project.argtypes = [dp, C.c_longlong, ip, dp, dp]
        L.oracle_envelope.argtypes = [dp, C.c_longlong, ip, ip, ip, dp]
        L.oracle_dft_basis.argtypes = [ip, dp]
        L.oracle_svd_filter.argtypes = [dp, C.c_longlong, ip, dp, ip, ip, dp]
        L.oracle_normalize.argtypes = [dp, C.c_longlong, dp]
        L.oracle_fftshift.argtypes = [dp, ip, ip, dp]
        L.oracle_process.argtypes = [u16p, ip, ip, ip, C.c_double, C.c_double, C.c_double, ip, ip, dp, dp, dp, dp, dp]
    return _LIB


def _d(a):
    return a.ctypes.data_as(C.POINTER(C.c_double))


def _u16(a):
    return a.ctypes.data_as(C.POINTER(C.c_uint16))


def _chk(rc):
    if rc < 0:
        raise ValueError("oracle call failed (bad arguments)")
    return rc


def fft2(a):
    """Unnormalised forward 2-D DFT of a (ny, nx) complex array (oracle's own radix-2)."""
    out = np.ascontiguousarray(a, dtype=np.complex128).copy()
    _chk(_lib().oracle_fft2(_d(out), out.shape[0], out.shape[1]))
    return out


def chirp(nx, ny, lam, pitch, z):
    q = np.empty((ny, nx), np.complex128)
    _chk(_lib().oracle_chirp(nx, ny, lam, pitch, z, _d(q)))
    return q


def mean_subtract(frames):
    f = np.ascontiguousarray(frames, dtype=np.uint16)
    T, ny, nx = f.shape
    d = np.empty((T, ny, nx), np.float64)
    _chk(_lib().oracle_mean_subtract(_u16(f), nx, ny, T, _d(d)))
    return d


def fresnel(frames, lam, pitch, z):
    """uint16 (T, ny, nx) -> H complex128 (T, ny, nx)."""
    f = np.ascontiguousarray(frames, dtype=np.uint16)
    T, ny, nx = f.shape
    H = np.empty((T, ny, nx), np.complex128)
    _chk(_lib().oracle_fresnel(_u16(f), nx, ny, T, lam, pitch, z, _d(H)))
    return H


def fresnel_field(g, lam, pitch, z):
    g = np.ascontiguousarray(g, dtype=np.complex128)
    ny, nx = g.shape
    H = np.empty((ny, nx), np.complex128)
    _chk(_lib().oracle_fresnel_field(_d(g), nx, ny, lam, pitch, z, _d(H)))
    return H


def covariance(H):
    """H complex (T, ...) -> C complex128 (T, T), C_ts = sum_p conj(H_t) H_s."""
    H = np.ascontiguousarray(H, dtype=np.complex128)
    T = H.shape[0]
    n_pix = H.size // T
    Cm = np.empty((T, T), np.complex128)
    _chk(_lib().oracle_covariance(_d(H), n_pix, T, _d(Cm)))
    return Cm


def eig(Cm):
    """Hermitian C (T,T) -> (evals descending float64 (T,), V complex128 (T,T) columns, sweeps)."""
    Cm = np.ascontiguousarray(Cm, dtype=np.complex128)
    T = Cm.shape[0]
    ev = np.empty(T, np.float64)
    V = np.empty((T, T), np.complex128)
    sw = _chk(_lib().oracle_eig(_d(Cm), T, _d(ev), _d(V)))
    return ev, V, sw


def project(H, V):
    """P_k = sum_t H_t V_tk for all k; returns complex128 with H's shape (k-planar)."""
    H = np.ascontiguousarray(H, dtype=np.complex128)
    V = np.ascontiguousarray(V, dtype=np.complex128)
    T = H.shape[0]
    P = np.empty_like(H)
    _chk(_lib().oracle_project(_d(H), H.size // T, T, _d(V), _d(P)))
    return P


def envelope(P, k_lo, k_hi):
    P = np.ascontiguousarray(P, dtype=np.complex128)
    T = P.shape[0]
    M = np.empty(P.shape[1:], np.float64)
    _chk(_lib().oracle_envelope(_d(P), P.size // T, T, k_lo, k_hi, _d(M)))
    return M


def dft_basis(T):
    W = np.empty((T, T), np.complex128)
    _chk(_lib().oracle_dft_basis(T, _d(W)))
    return W


def svd_filter(H, V, k_lo, k_hi):
    """Eq. 3: Hf = H V I_f V^H, complex128 with H's shape."""
    H = np.ascontiguousarray(H, dtype=np.complex128)
    V = np.ascontiguousarray(V, dtype=np.complex128)
    T = H.shape[0]
    Hf = np.empty_like(H)
    _chk(_lib().oracle_svd_filter(_d(H), H.size // T, T, _d(V), k_lo, k_hi, _d(Hf)))
    return Hf


def normalize(M):
    """image divided by its spatial average."""
    M = np.ascontiguousarray(M, dtype=np.float64)
    out = np.empty_like(M)
    _chk(_lib().oracle_normalize(_d(M), M.size, _d(out)))
    return out


def fftshift(M):
    M = np.ascontiguousarray(M, dtype=np.float64)
    out = np.empty_like(M)
    _chk(_lib().oracle_fftshift(_d(M), M.shape[0], M.shape[1], _d(out)))
    return out


def process(frames, lam, pitch, z, k_lo, k_hi, want_H=False):
    """Whole path.  Returns dict(M, C, evals, V, sweeps[, H])."""
    f = np.ascontiguousarray(frames, dtype=np.uint16)
    T, ny, nx = f.shape
    M = np.empty((ny, nx), np.float64)
    H = np.empty((T, ny, nx), np.complex128) if want_H else None
    Cm = np.empty((T, T), np.complex128)
    ev = np.empty(T, np.float64)
    V = np.empty((T, T), np.complex128)
    sw = _chk(_lib().oracle_process(_u16(f), nx, ny, T, lam, pitch, z, k_lo, k_hi, _d(M),
                                    _d(H) if want_H else None, _d(Cm), _d(ev), _d(V)))
    out = dict(M=M, C=Cm, evals=ev, V=V, sweeps=sw)
    if want_H:
        out["H"] = H
    return out


def num_threads():
    return int(_lib().oracle_num_threads())
