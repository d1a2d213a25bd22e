"""Seeded synthetic inline-interferogram generator (inputs only -- none of the method's arithmetic).

Serves BOTH the oracle-side tests and the CUDA-side tests/bench; imports neither.  It stands in
for the paper's in-vivo retinal recordings (1024x1024, 16-bit container, 500 fps,
stacks of 32), which are not available.  Recipe = BASELINE.json:configs, made precise in
SURVEY.md section 8(d) and restated in DESIGN.md "Input recipe":

  phi ~ U[0,2pi), A ~ Rayleigh(1), f ~ U[0,0.02] cycles/frame per pixel (background);
  n_s straight 'vessel' stripes of half-width 4 px, random orientation/offset: amplitude x3,
  f ~ U[0.1,0.4] per pixel;  O = A*amp*exp(i phi);
  psi_t = cumulative sum of N(0, sigma_psi) over the GLOBAL frame index;
  E_t = O * exp(2 pi i f t + i psi_t)  in the object plane;
  sensor field Es_t = conj(q) * IFFT2(E_t) * sqrt(nx ny)  (the unitary inverse of the
  reconstruction operator FFT2[q * .], q = exp(+i pi (x^2+y^2)/(lambda z)), centred coordinates);
  Ibar_t = 1000 + 40*|1 + Es_t|^2 [+ 40*|Es_t|^2 if self_beating];
  I_t = clip(Poisson(Ibar_t), 0, 4095) as uint16.

Two back ends with the same formulas: numpy (canonical, used for parity fixtures) and torch on a
device (bench streams only; not bit-identical to numpy -- parity always copies the actual bytes).
"""
from dataclasses import dataclass, field
import numpy as np

LAMBDA_M = 785e-9
PITCH_M = 20e-6
Z_M = 0.2


@dataclass(frozen=True)
class Config:
    name: str
    n: int            # nx = ny
    T: int
    n_frames: int     # length of the stream
    stride: int       # frames between consecutive stacks (== T: non-overlapping)
    n_stripes: int
    sigma_psi: float
    self_beating: bool
    k_lo: int
    k_hi: int
    lam: float = LAMBDA_M
    pitch: float = PITCH_M
    z: float = Z_M

    @property
    def n_stacks(self):
        return (self.n_frames - self.T) // self.stride + 1


# BASELINE.json:configs[0..4]
CONFIGS = {
    1: Config("cfg1_256x16", 256, 16, 16, 16, 3, 0.3, False, 2, 16),
    2: Config("cfg2_512x32", 512, 32, 256, 32, 5, 0.3, False, 2, 32),
    3: Config("cfg3_1024x32", 1024, 32, 2048, 32, 8, 0.5, True, 2, 32),
    4: Config("cfg4_1024x32_slide8", 1024, 32, 2048, 8, 8, 0.5, True, 2, 32),
    5: Config("cfg5_2048x64", 2048, 64, 1024, 64, 12, 0.3, False, 3, 64),
}


def small_config(n=64, T=8, n_stripes=2, k_lo=2, k_hi=None, sigma_psi=0.3, self_beating=False, n_frames=None):
    """A reduced-size config of the same recipe, for CPU tests."""
    return Config(f"small_{n}x{T}", n, T, n_frames or T, T, n_stripes, sigma_psi, self_beating,
                  k_lo, k_hi if k_hi is not None else T)


def chirp_np(nx, ny, lam, pitch, z):
    x = (np.arange(nx, dtype=np.float64) - nx // 2) * pitch
    y = (np.arange(ny, dtype=np.float64) - ny // 2) * pitch
    ph = np.pi * (x[None, :] ** 2 + y[:, None] ** 2) / (lam * z)
    return np.exp(1j * ph)


@dataclass
class Scene:
    cfg: Config
    seed: int
    O: np.ndarray        # complex128 (n, n)   object field
    f: np.ndarray        # float64 (n, n)      Doppler frequency, cycles/frame
    psi: np.ndarray      # float64 (n_frames,) global phase walk
    mask: np.ndarray     # bool (n, n)         union of vessel stripes
    rng: np.random.Generator = field(repr=False, default=None)


def make_scene(cfg: Config, seed: int) -> Scene:
    rng = np.random.default_rng(seed)
    n = cfg.n
    phi = rng.uniform(0.0, 2 * np.pi, (n, n))
    A = rng.rayleigh(1.0, (n, n))
    f = rng.uniform(0.0, 0.02, (n, n))
    amp = np.ones((n, n))
    mask_all = np.zeros((n, n), bool)
    yy, xx = np.mgrid[0:n, 0:n].astype(np.float64)
    for _ in range(cfg.n_stripes):
        theta = rng.uniform(0.0, np.pi)
        rho = rng.uniform(0.2 * n, 0.8 * n)
        dist = (xx - n / 2) * np.cos(theta) + (yy - n / 2) * np.sin(theta) - (rho - n / 2)
        mask = np.abs(dist) <= 4.0
        amp[mask] = 3.0
        f[mask] = rng.uniform(0.1, 0.4, int(mask.sum()))
        mask_all |= mask
    O = A * amp * np.exp(1j * phi)
    psi = np.cumsum(rng.normal(0.0, cfg.sigma_psi, cfg.n_frames))
    return Scene(cfg, seed, O, f, psi, mask_all, rng)


def frames_np(scene: Scene, t0: int, count: int) -> np.ndarray:
    """uint16 (count, n, n) frames t0 .. t0+count-1 of the stream (numpy, canonical).
    Poisson noise is drawn from the scene's generator in call order."""
    cfg = scene.cfg
    n = cfg.n
    qc = np.conj(chirp_np(n, n, cfg.lam, cfg.pitch, cfg.z))
    out = np.empty((count, n, n), np.uint16)
    for i in range(count):
        t = t0 + i
        E = scene.O * np.exp(2j * np.pi * scene.f * t + 1j * scene.psi[t])
        Es = qc * np.fft.ifft2(E) * n          # ifft2 carries 1/n^2; * sqrt(n*n) makes it unitary
        Ibar = 1000.0 + 40.0 * np.abs(1.0 + Es) ** 2
        if cfg.self_beating:
            Ibar = Ibar + 40.0 * np.abs(Es) ** 2
        out[i] = np.clip(scene.rng.poisson(Ibar), 0, 4095).astype(np.uint16)
    return out


def stack_np(cfg: Config, seed: int, stack_index: int = 0) -> np.ndarray:
    """Convenience: the stack_index-th stack (T frames) of a fresh scene.  Deterministic in
    (cfg, seed, stack_index): noise for earlier frames is drawn and discarded."""
    scene = make_scene(cfg, seed)
    t0 = stack_index * cfg.stride
    if t0 > 0:
        frames_np(scene, 0, t0)
    return frames_np(scene, t0, cfg.T)


def stream_torch(cfg: Config, seed: int, device, n_frames=None, chunk=32):
    """uint16 torch tensor (n_frames, n, n) on `device` -- same formulas, torch RNG for the shot
    noise (scene parameters still come from numpy's default_rng(seed)).  Bench harness only."""
    import torch
    import dataclasses
    n_frames = n_frames or cfg.n_frames
    if n_frames > cfg.n_frames:                          # a longer stream of the same recipe (the phase walk continues)
        cfg = dataclasses.replace(cfg, n_frames=n_frames)
    scene = make_scene(cfg, seed)
    n = cfg.n
    g = torch.Generator(device=device)
    g.manual_seed(seed)
    O = torch.from_numpy(scene.O).to(device=device, dtype=torch.complex64)
    f = torch.from_numpy(scene.f).to(device=device, dtype=torch.float64)
    psi = torch.from_numpy(scene.psi).to(device=device, dtype=torch.float64)
    qc = torch.from_numpy(np.conj(chirp_np(n, n, cfg.lam, cfg.pitch, cfg.z))).to(device=device, dtype=torch.complex64)
    out = torch.empty((n_frames, n, n), dtype=torch.int16, device=device)   # values <= 4095
    for t0 in range(0, n_frames, chunk):
        c = min(chunk, n_frames - t0)
        t = torch.arange(t0, t0 + c, device=device, dtype=torch.float64)
        ph = 2 * np.pi * f[None] * t[:, None, None] + psi[t0:t0 + c, None, None]
        ph = torch.remainder(ph, 2 * np.pi).to(torch.float32)
        E = O[None] * torch.polar(torch.ones_like(ph), ph)
        Es = qc[None] * torch.fft.ifft2(E) * n
        Ibar = 1000.0 + 40.0 * (1.0 + Es).abs() ** 2
        if cfg.self_beating:
            Ibar = Ibar + 40.0 * Es.abs() ** 2
        I = torch.poisson(Ibar, generator=g).clamp_(0, 4095)
        out[t0:t0 + c] = I.to(torch.int16)
    return out.view(torch.uint16)
