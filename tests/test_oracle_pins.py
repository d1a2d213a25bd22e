"""Pins for the CPU oracle (oracle/holo_oracle.cpp) against what the paper and the mathematics fix.

None of these re-types the oracle's own formula or re-calls its routine: brute-force DFT matrices,
closed forms, exact integer arithmetic, LAPACK on tiny inputs, and algebraic invariants
(SURVEY.md section 8(c) "What pins each part").  All CPU, all `-m "not gpu"`.
"""
import os
import numpy as np
import pytest

import oracle
from gen import holo_gen as G
from tests.util import rel_l2, brute_dft2, dft_matrix, integer_gram

LAM, PITCH, Z = G.LAMBDA_M, G.PITCH_M, G.Z_M
rng0 = np.random.default_rng(1234)


# ---------------------------------------------------------------- A2: FFT (Eq. 1)
@pytest.mark.parametrize("ny,nx", [(1, 8), (8, 1), (4, 16), (16, 32), (32, 32)])
def test_fft2_vs_bruteforce_dft(ny, nx):
    a = rng0.standard_normal((ny, nx)) + 1j * rng0.standard_normal((ny, nx))
    assert rel_l2(oracle.fft2(a), brute_dft2(a)) <= 1e-12


def test_fft2_impulse_and_constant():
    ny, nx, j0, i0 = 16, 64, 5, 37
    a = np.zeros((ny, nx), complex)
    a[j0, i0] = 2.5
    ky, kx = np.mgrid[0:ny, 0:nx]
    ramp = 2.5 * np.exp(-2j * np.pi * (i0 * kx / nx + j0 * ky / ny))      # forward sign, unnormalised
    assert np.abs(oracle.fft2(a) - ramp).max() <= 1e-12
    c = oracle.fft2(np.full((ny, nx), 3.0 + 1j))
    assert abs(c[0, 0] - (3.0 + 1j) * nx * ny) <= 1e-10
    c[0, 0] = 0
    assert np.abs(c).max() <= 1e-10


def test_fft2_linearity_and_nonsquare_axes():
    a = rng0.standard_normal((8, 32)) + 0j
    b = rng0.standard_normal((8, 32)) * 1j
    assert rel_l2(oracle.fft2(2 * a - 3j * b), 2 * oracle.fft2(a) - 3j * oracle.fft2(b)) <= 1e-13
    # axis convention: x is the fast axis; a pure x-harmonic lands in row 0
    ny, nx, u = 8, 32, 5
    h = np.exp(2j * np.pi * u * np.arange(nx) / nx)[None, :].repeat(ny, 0)
    F = oracle.fft2(h)
    assert abs(F[0, u] - nx * ny) <= 1e-9 and np.abs(F).sum() - abs(F[0, u]) <= 1e-8
    with pytest.raises(ValueError):
        oracle.fft2(np.zeros((8, 12), complex))


# ---------------------------------------------------------------- A1: chirp (Eq. 1)
def test_chirp_golden_constants():
    path = os.path.join(os.path.dirname(__file__), "golden", "chirp_constants.txt")
    n = 2048
    q = oracle.chirp(n, n, LAM, PITCH, Z)
    assert q[n // 2, n // 2] == 1.0
    for line in open(path):
        if line.startswith("#"):
            continue
        dx, dy, ph = line.split()
        dx, dy, ph = int(dx), int(dy), float(ph)
        v = q[n // 2 + dy, n // 2 + dx]
        assert abs(v - np.exp(1j * ph)) <= 5e-12, (dx, dy)      # + sign: Im > 0 for small positive phase
    assert q[n // 2, n // 2 + 1].imag > 0
    assert np.abs(np.abs(q) - 1).max() <= 1e-15


def test_chirp_nonsquare_axes():
    q = oracle.chirp(16, 64, LAM, PITCH, Z)     # nx=16, ny=64 -> shape (64, 16)
    assert q.shape == (64, 16)
    assert q[32, 8] == 1.0
    ph = np.pi * (3 ** 2) * PITCH ** 2 / (LAM * Z)
    assert abs(q[32 + 3, 8] - np.exp(1j * ph)) <= 1e-13 and abs(q[32, 8 + 3] - np.exp(1j * ph)) <= 1e-13


@pytest.mark.parametrize("n,u0,v0", [(64, 5, 40), (128, 0, 0), (256, 255, 17)])
def test_point_source_refocuses_to_one_pixel(n, u0, v0):
    """A diverging spherical wave conj(q)*plane-wave refocuses to a single output bin:
    FFT2[q * conj(q) e^{+2 pi i (i u0/n + j v0/n)}] = n^2 delta(k-(u0,v0)).  Pins sign AND centre
    of the oracle's chirp against the generator's independently written one."""
    qg = G.chirp_np(n, n, LAM, PITCH, Z)
    j, i = np.mgrid[0:n, 0:n]
    g = np.conj(qg) * np.exp(2j * np.pi * (i * u0 + j * v0) / n)
    H = oracle.fresnel_field(g, LAM, PITCH, Z)
    assert abs(H[v0, u0] - n * n) <= 1e-6 * n * n
    H[v0, u0] = 0
    assert np.abs(H).max() <= 1e-7 * n * n
    # wrong sign (twin image) must NOT focus: the check above has teeth
    Hw = oracle.fresnel_field(np.conj(g), LAM, PITCH, Z)
    assert np.abs(Hw).max() < 0.5 * n * n


def test_uint16_single_bright_pixel_closed_form():
    """One bright pixel of amplitude A at (i0,j0) in frame 0 only =>
    H_0(k) = A(1-1/T) q(i0,j0) e^{-2 pi i(i0 kx/nx + j0 ky/ny)},  H_{t>0} = -(A/T) (same)."""
    nx, ny, T, A, i0, j0 = 32, 16, 4, 1000, 21, 3
    fr = np.full((T, ny, nx), 700, np.uint16)
    fr[0, j0, i0] += A
    H = oracle.fresnel(fr, LAM, PITCH, Z)
    x, y = (i0 - nx // 2) * PITCH, (j0 - ny // 2) * PITCH
    q00 = np.exp(1j * np.pi * (x * x + y * y) / (LAM * Z))
    ky, kx = np.mgrid[0:ny, 0:nx]
    ramp = q00 * np.exp(-2j * np.pi * (i0 * kx / nx + j0 * ky / ny))
    assert np.abs(H[0] - A * (1 - 1 / T) * ramp).max() <= 1e-9
    for t in range(1, T):
        assert np.abs(H[t] + (A / T) * ramp).max() <= 1e-9


# ---------------------------------------------------------------- A0: mean
def test_mean_subtraction_sums_to_zero_and_is_per_pixel_temporal():
    fr = rng0.integers(0, 65536, (5, 8, 16)).astype(np.uint16)     # T=5: not a power of two, full range
    d = oracle.mean_subtract(fr)
    assert np.abs(d.sum(axis=0)).max() <= 1e-9
    T = fr.shape[0]
    exact = (T * fr.astype(np.int64) - fr.astype(np.int64).sum(0)[None]) / T
    assert np.abs(d - exact).max() <= 1e-10


def test_parseval_and_trace():
    cfg = G.small_config(n=32, T=8)
    fr = G.stack_np(cfg, 7)
    H = oracle.fresnel(fr, LAM, PITCH, Z)
    d = oracle.mean_subtract(fr)
    assert abs((np.abs(H) ** 2).sum() - 32 * 32 * (d ** 2).sum()) <= 1e-10 * (np.abs(H) ** 2).sum()
    C = oracle.covariance(H)
    assert abs(np.trace(C).real - (np.abs(H) ** 2).sum()) <= 1e-10 * np.trace(C).real
    assert np.abs(H.sum(axis=0)).max() <= 1e-7            # sum_t H_t = 0 (mean subtraction)


# ---------------------------------------------------------------- A3: covariance (Eq. 4)
def test_covariance_definition_tiny_bruteforce():
    T, npix = 3, 5
    H = rng0.standard_normal((T, npix)) + 1j * rng0.standard_normal((T, npix))
    C = oracle.covariance(H)
    for t in range(T):
        for s in range(T):
            ref = sum(H[t, p].conjugate() * H[s, p] for p in range(npix))     # python loop, H^{t*}H
            assert abs(C[t, s] - ref) <= 1e-13
    assert np.abs(C - C.conj().T).max() <= 1e-13
    # not the transposed/conjugated variant: Im C must have the sign of conj(H_t) H_s
    assert abs(C[0, 1].imag - (H[0].conj() * H[1]).sum().imag) <= 1e-13


@pytest.mark.parametrize("n,T,seed", [(32, 8, 3), (64, 16, 4)])
def test_covariance_exact_integer_gram(n, T, seed):
    """C = (nx ny / T^2) G with G_ts = sum_p (T I_t - S)(T I_s - S) in exact integers: pins A0-A3
    jointly (q unimodular, DFT unitary up to nx*ny)."""
    fr = G.stack_np(G.small_config(n=n, T=T), seed)
    C = oracle.covariance(oracle.fresnel(fr, LAM, PITCH, Z))
    Gm, _ = integer_gram(fr)
    Cx = np.asarray(Gm, dtype=np.float64) * (n * n) / (T * T)
    assert rel_l2(C.real, Cx) <= 1e-11
    assert np.abs(C.imag).max() <= 1e-11 * np.abs(C.real).max()
    w = np.linalg.eigvalsh(C)
    assert w.min() >= -1e-9 * w.max()                 # PSD
    assert np.abs(C @ np.ones(T)).max() <= 1e-9 * np.abs(C).max()      # C.1 = 0


# ---------------------------------------------------------------- A4: eig (Eq. 5)
def _rand_herm(T, rng, psd=False):
    X = rng.standard_normal((T, T)) + 1j * rng.standard_normal((T, T))
    return X.conj().T @ X if psd else (X + X.conj().T) / 2


@pytest.mark.parametrize("T", [1, 2, 3, 5, 16, 32, 64])
def test_eig_invariants_and_lapack(T):
    rng = np.random.default_rng(100 + T)
    C = _rand_herm(T, rng, psd=(T % 2 == 0))
    ev, V, sw = oracle.eig(C)
    nC = np.linalg.norm(C)
    assert np.all(np.diff(ev) <= 0)                                  # descending (reading R1)
    assert np.linalg.norm(V.conj().T @ V - np.eye(T)) <= 1e-13 * T
    assert np.linalg.norm(C @ V - V * ev[None, :]) <= 1e-13 * nC * T
    D = V.conj().T @ C @ V
    assert np.linalg.norm(D - np.diag(np.diag(D))) <= 1e-13 * nC * T
    assert abs(ev.sum() - np.trace(C).real) <= 1e-12 * nC
    assert np.abs(ev - np.linalg.eigvalsh(C)[::-1]).max() <= 1e-12 * nC        # LAPACK cross-check
    assert sw <= 12


def test_eig_2x2_closed_form_and_diagonal():
    a, c, b = 3.0, -1.0, 0.7 - 1.9j
    ev, V, _ = oracle.eig(np.array([[a, b], [np.conj(b), c]]))
    r = np.sqrt(((a - c) / 2) ** 2 + abs(b) ** 2)
    assert np.allclose(ev, [(a + c) / 2 + r, (a + c) / 2 - r], atol=1e-14)
    # eigenvector of the larger eigenvalue is proportional to (b, lambda1 - a)
    v = np.array([b, ev[0] - a])
    v /= np.linalg.norm(v)
    assert abs(abs(np.vdot(v, V[:, 0])) - 1) <= 1e-13
    ev, V, sw = oracle.eig(np.diag([1.0, 5.0, -2.0, 5.0]).astype(complex))
    assert np.allclose(ev, [5, 5, 1, -2]) and sw == 0
    assert np.allclose(np.abs(V).sum(0), 1) and np.allclose(np.abs(V).sum(1), 1)     # a permutation


def test_eig_zero_matrix_no_nan():
    ev, V, sw = oracle.eig(np.zeros((8, 8), complex))
    assert np.all(ev == 0) and np.array_equal(V, np.eye(8)) and sw == 0      # reading R11


def test_eig_matches_svd_of_H():
    """Eq. 2 vs Eq. 5: Lambda = Delta^2."""
    H = oracle.fresnel(G.stack_np(G.small_config(n=16, T=6), 11), LAM, PITCH, Z)
    sv = np.linalg.svd(H.reshape(6, -1).T, compute_uv=False)
    ev, _, _ = oracle.eig(oracle.covariance(H))
    assert np.abs(ev - sv ** 2).max() <= 1e-10 * ev[0]


def test_T2_stack_closed_form():
    """T=2: d_0 = -d_1, so lambda = {2 nx ny sum d_0^2, 0}, v_1 = (1,-1)/sqrt2, M_[1,1] = 2|H_0|^2."""
    n = 16
    fr = rng0.integers(900, 1500, (2, n, n)).astype(np.uint16)
    out = oracle.process(fr, LAM, PITCH, Z, 1, 1, want_H=True)
    d0 = (fr[0].astype(float) - fr[1].astype(float)) / 2
    assert abs(out["evals"][0] - 2 * n * n * (d0 ** 2).sum()) <= 1e-10 * out["evals"][0]
    assert abs(out["evals"][1]) <= 1e-10 * out["evals"][0]
    assert abs(abs(np.vdot(np.array([1, -1]) / np.sqrt(2), out["V"][:, 0])) - 1) <= 1e-12
    assert rel_l2(out["M"], 2 * np.abs(out["H"][0]) ** 2) <= 1e-12


# ---------------------------------------------------------------- A5/A6: projection + envelope (Eq. 6-7)
def test_projection_definition_and_index_convention():
    T, npix = 4, 6
    H = rng0.standard_normal((T, npix)) + 1j * rng0.standard_normal((T, npix))
    V = rng0.standard_normal((T, T)) + 1j * rng0.standard_normal((T, T))      # any matrix: P = H V
    P = oracle.project(H, V)
    assert rel_l2(P, (H.T @ V).T) <= 1e-14                 # Hc = H V with H as (pixels, T)
    M = oracle.envelope(P, 2, 3)
    assert rel_l2(M, np.abs(P[1]) ** 2 + np.abs(P[2]) ** 2) <= 1e-14          # 1-based inclusive (R13)
    with pytest.raises(ValueError):
        oracle.envelope(P, 0, 3)
    with pytest.raises(ValueError):
        oracle.envelope(P, 3, 2)


def test_energy_conservation_and_component_energies():
    cfg = G.small_config(n=32, T=8)
    out = oracle.process(G.stack_np(cfg, 5), LAM, PITCH, Z, 2, 8, want_H=True)
    H, V, ev = out["H"], out["V"], out["evals"]
    P = oracle.project(H, V)
    tot = (np.abs(H) ** 2).sum(axis=0)
    assert rel_l2((np.abs(P) ** 2).sum(axis=0), tot) <= 1e-12          # per-pixel energy conservation
    assert np.abs((np.abs(P) ** 2).sum(axis=(1, 2)) - ev).max() <= 1e-10 * ev[0]   # sum_p |P_k|^2 = lambda_k
    assert abs(out["M"].sum() - ev[1:].sum()) <= 1e-10 * ev[0]
    full = oracle.envelope(P, 1, 8)
    assert rel_l2(full, tot) <= 1e-12                       # k_lo=1,k_hi=T -> sum_t |H_t|^2
    assert rel_l2(out["M"], tot - np.abs(P[0]) ** 2) <= 1e-12           # complement identity (R12)


def test_pure_tone_spans_dft_bins():
    """I_t = a + b cos(2 pi m t/T + phi(x,y)): the two dominant principal components span DFT bins
    m and T-m of Eq. 8's W, so sum_{k<=2}|P_k|^2 = |Ht_m|^2 + |Ht_{T-m}|^2."""
    n, T, m = 16, 8, 3
    phi = rng0.uniform(0, 2 * np.pi, (n, n))
    t = np.arange(T)[:, None, None]
    fr = np.round(2000 + 800 * np.cos(2 * np.pi * m * t / T + phi[None])).astype(np.uint16)
    out = oracle.process(fr, LAM, PITCH, Z, 1, 2, want_H=True)
    W = oracle.dft_basis(T)
    Ht = oracle.project(out["H"], W)
    ref = np.abs(Ht[m]) ** 2 + np.abs(Ht[T - m]) ** 2
    # rounding to uint16 leaks ~1e-7 of the energy into other bins
    assert rel_l2(out["M"], ref) <= 1e-5
    assert out["evals"][2] <= 1e-5 * out["evals"][1]


def test_dft_basis_eq8():
    T = 8
    W = oracle.dft_basis(T)
    assert np.abs(W - dft_matrix(T) / np.sqrt(T)).max() <= 1e-15         # w_mn, 1-based (m-1)(n-1)
    assert np.linalg.norm(W.conj().T @ W - np.eye(T)) <= 1e-14
    # Fourier demodulation of a constant stack: only bin n=1 is non-zero
    H = np.ones((T, 5), complex)
    P = oracle.project(H, W)
    assert abs(P[0, 0] - np.sqrt(T)) <= 1e-14 and np.abs(P[1:]).max() <= 1e-14


def test_constant_stack_is_all_zero():
    fr = np.full((4, 16, 16), 1234, np.uint16)            # reading R11
    out = oracle.process(fr, LAM, PITCH, Z, 1, 4)
    assert np.all(out["M"] == 0) and np.all(out["evals"] == 0) and np.all(np.isfinite(out["V"].view(float)))


# ---------------------------------------------------------------- generator <-> operator (sign/centre)
def test_generator_refocuses_inside_vessel_mask():
    """The generator is the inverse of FFT2[q .]: vessels (amplitude x3, fast Doppler) come back
    in focus at their object-plane pixels; with the mirrored mask there is no contrast."""
    cfg = G.small_config(n=128, T=16, n_stripes=3)
    scene = G.make_scene(cfg, 21)
    fr = G.frames_np(scene, 0, cfg.T)
    M = oracle.process(fr, LAM, PITCH, Z, 2, 16)["M"]
    inside, outside = M[scene.mask].mean(), M[~scene.mask].mean()
    assert inside / outside > 1.5
    mirror = np.roll(scene.mask[::-1, ::-1], (1, 1), (0, 1))           # x -> -x mod n
    assert M[mirror].mean() / M[~mirror].mean() < 1.15


# ---------------------------------------------------------------- Eq. 3 SVD filter, normalisation (:86), fftshift
def test_svd_filter_matches_library_svd_eq3():
    """Eq. 3 literally: H = U Delta V^H (LAPACK, on H as an n_pix x T matrix), Hf = U Delta I_f V^H."""
    rs = np.random.default_rng(7)
    T, n = 6, 40
    H = rs.standard_normal((T, n)) + 1j * rs.standard_normal((T, n))
    ev, V, _ = oracle.eig(oracle.covariance(H))
    U, sv, Vh = np.linalg.svd(H.T, full_matrices=False)          # H.T: rows = pixels, columns = frames
    for k_lo, k_hi in ((1, T), (2, T), (2, 4), (3, 3)):
        keep = np.zeros(T)
        keep[k_lo - 1:k_hi] = 1.0                                 # singular values come in descending order too
        ref = ((U * (sv * keep)) @ Vh).T
        assert rel_l2(oracle.svd_filter(H, V, k_lo, k_hi), ref) <= 1e-10, (k_lo, k_hi)


def test_svd_filter_identities():
    rs = np.random.default_rng(8)
    T, n = 8, 64
    H = rs.standard_normal((T, n)) + 1j * rs.standard_normal((T, n))
    ev, V, _ = oracle.eig(oracle.covariance(H))
    assert rel_l2(oracle.svd_filter(H, V, 1, T), H) <= 1e-12       # I_f = identity: nothing is removed
    Hf = oracle.svd_filter(H, V, 3, 6)
    M = oracle.envelope(oracle.project(H, V), 3, 6)
    assert rel_l2((np.abs(Hf) ** 2).sum(axis=0), M) <= 1e-12       # frame-basis energy = component energy (V unitary)
    # idempotent, and the two complementary filters add up to H
    assert rel_l2(oracle.svd_filter(Hf, V, 3, 6), Hf) <= 1e-12
    rest = oracle.svd_filter(H, V, 1, 2) + oracle.svd_filter(H, V, 7, 8)
    assert rel_l2(Hf + rest, H) <= 1e-12


def test_normalize_mean_is_one_and_zero_image():
    rs = np.random.default_rng(9)
    M = rs.random((12, 20)) * 5 + 0.1
    out = oracle.normalize(M)
    assert abs(out.mean() - 1.0) <= 1e-14
    assert rel_l2(out * M.sum() / M.size, M) <= 1e-14              # a pure rescaling
    assert abs(oracle.normalize(3.0 * M) - out).max() <= 1e-14      # scale invariant
    assert not np.any(oracle.normalize(np.zeros((4, 4))))


def test_fftshift_matches_numpy_and_centres_dc():
    rs = np.random.default_rng(10)
    for shape in ((8, 8), (4, 16), (16, 2)):
        M = rs.random(shape)
        assert np.array_equal(oracle.fftshift(M), np.fft.fftshift(M))
    a = np.abs(oracle.fft2(np.ones((8, 16)) + 0j)) ** 2             # all energy in bin (0, 0)
    s = oracle.fftshift(a)
    assert s[4, 8] == a[0, 0] and s.sum() == a[0, 0]
