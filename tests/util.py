"""Shared test helpers (numpy only; neither the oracle's nor the CUDA path's arithmetic)."""
import numpy as np


def rel_l2(a, b):
    a = np.asarray(a)
    b = np.asarray(b)
    den = np.linalg.norm(b.ravel())
    return float(np.linalg.norm((a - b).ravel()) / (den if den > 0 else 1.0))


def dft_matrix(n):
    k = np.arange(n)
    return np.exp(-2j * np.pi * np.outer(k, k) / n)


def brute_dft2(a):
    """O(N^4)-equivalent direct 2-D DFT via explicit DFT matrices (no FFT anywhere)."""
    ny, nx = a.shape
    return dft_matrix(ny) @ a @ dft_matrix(nx).T


def integer_gram(frames):
    """Exact G_ts = sum_p (T I_t - S)(T I_s - S) in Python integers (object dtype on overflow risk)."""
    T = frames.shape[0]
    I = frames.reshape(T, -1).astype(np.int64)
    S = I.sum(axis=0)
    D = T * I - S[None, :]
    peak = int(np.abs(D).max())
    if peak * peak * D.shape[1] < 2 ** 62:
        return D @ D.T, D
    return (D.astype(object) @ D.T.astype(object)), D


def eig_gaps(frames):
    """Descending eigenvalues of the (scaled) covariance via the integer Gram; for qualifying inputs."""
    G, _ = integer_gram(frames)
    ev = np.linalg.eigvalsh(np.asarray(G, dtype=np.float64))[::-1]
    gaps = (ev[:-1] - ev[1:]) / np.maximum(ev[:-1], 1e-300)
    return ev, gaps


def projector(V, k_lo, k_hi):
    Vs = V[:, k_lo - 1:k_hi]
    return Vs @ Vs.conj().T
