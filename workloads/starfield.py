"""Seeded star-field image pairs in the shapes of BASELINE.json's five configs.

Recipe:
  * reference R = sky + sum of pixel-integrated circular Gaussian stars
    (steps (i)-(v)), positions uniform, fluxes log-uniform
    (BASELINE.json states log-uniform instead of the paper's F^-3/2 law);
  * target I = [R (x) K_true] + B0 on the valid region (Eq. 2 used
    as the *simulation* step, computed with a library correlation), plus
    Gaussian noise of variance sigma0^2/F^2 + I_nl/(G F) (Eq. 6 with
    M := I_noiseless, as PAPER.md:298 Eq. 25; Eq. 26);
  * config 2 replaces 0.1 % of pixels by cosmic-ray hits, config 3 saturates and
    masks 2 % of pixels and draws a per-pixel flat field.
RNG streams: reference `default_rng(c)`; target epoch e `default_rng(10000*(c+1)+e)`.
All images are computed in float64 and stored as float32.
"""
from __future__ import annotations

import dataclasses
import math
from typing import Optional, Sequence

import numpy as np
from scipy import signal, special

FWHM_TO_SIGMA = 1.0 / 2.35482


@dataclasses.dataclass(frozen=True)
class Config:
    index: int
    n: int
    m: int
    n_stars: int
    fwhm: float
    flux_lo: float
    flux_hi: float
    sky: float
    sigma0: float
    gain: float
    loss: str            # "gaussian" | "huber"
    n_epochs: int = 1
    flat: bool = False   # per-pixel flat field drawn U(0.95, 1.05)
    cosmic_frac: float = 0.0
    saturate_frac: float = 0.0
    kernel: str = "gauss"


CONFIGS = (
    Config(0, 128, 7, 50, 2.0, 1e2, 1e5, 100.0, 5.0, 1.0, "gaussian", kernel="c0"),
    Config(1, 512, 15, 2000, 2.5, 1e2, 1e6, 200.0, 5.0, 1.0, "gaussian", kernel="c1"),
    Config(2, 1024, 19, 20000, 3.0, 1e2, 1e6, 500.0, 8.0, 2.0, "huber",
           cosmic_frac=0.001, kernel="c2"),
    Config(3, 2048, 25, 60000, 2.8, 1e2, 1e6, 300.0, 6.0, 1.5, "gaussian",
           flat=True, saturate_frac=0.02, kernel="c3"),
    Config(4, 4096, 19, 200000, 2.5, 1e2, 1e6, 400.0, 5.0, 1.0, "gaussian",
           n_epochs=16, kernel="c4"),
)


@dataclasses.dataclass
class Workload:
    """One reference and E target epochs, ready for either implementation."""
    config: Config
    n: int
    m: int
    R: np.ndarray                 # [n][n] float32
    I: np.ndarray                 # [E][n][n] float32
    theta_true: np.ndarray        # [E][m*m+1] float64 (K row-major, then B0)
    theta0: np.ndarray            # [E][m*m+1] float32, flat-kernel init (R11)
    flat: Optional[np.ndarray]    # [n][n] float32 or None
    mask: Optional[np.ndarray]    # [E][n][n] uint8 (1 = use) or None
    sigma0: float
    gain: float
    loss: str

    @property
    def n_epochs(self) -> int:
        return self.I.shape[0]


def n_valid(n: int, m: int) -> int:
    """N_data = (N - 2h)^2 with h = (m-1)/2."""
    return (n - m + 1) ** 2


# --------------------------------------------------------------------------
# reference image
# --------------------------------------------------------------------------
def render_stars(n: int, xs, ys, fluxes, fwhm: float, sky: float) -> np.ndarray:
    """sky + sum of pixel-integrated circular Gaussians, float64 [n][n].

    Pixel (i, j) covers [j, j+1) x [i, i+1); a star at (x, y) of flux f gives
    f/4 * [erf((j+1-x)/(s√2)) - erf((j-x)/(s√2))] * [same in y] inside a stamp of
    radius ceil(6 sigma)+1.
    """
    sigma = fwhm * FWHM_TO_SIGMA
    rad = int(math.ceil(6.0 * sigma)) + 1
    w = 2 * rad + 1
    img = np.zeros(n * n, dtype=np.float64)
    xs = np.asarray(xs, dtype=np.float64)
    ys = np.asarray(ys, dtype=np.float64)
    fluxes = np.asarray(fluxes, dtype=np.float64)
    s2 = sigma * math.sqrt(2.0)
    offs = np.arange(-rad, rad + 2, dtype=np.float64)  # w+1 pixel edges
    chunk = 20000
    for c0 in range(0, xs.size, chunk):
        x = xs[c0:c0 + chunk]
        y = ys[c0:c0 + chunk]
        f = fluxes[c0:c0 + chunk]
        j0 = np.floor(x).astype(np.int64)
        i0 = np.floor(y).astype(np.int64)
        ex = special.erf((j0[:, None] + offs[None, :] - x[:, None]) / s2)
        ey = special.erf((i0[:, None] + offs[None, :] - y[:, None]) / s2)
        gx = 0.5 * (ex[:, 1:] - ex[:, :-1])          # [S][w]
        gy = 0.5 * (ey[:, 1:] - ey[:, :-1])          # [S][w]
        stamp = f[:, None, None] * gy[:, :, None] * gx[:, None, :]   # [S][w][w]
        jj = j0[:, None] + np.arange(-rad, rad + 1)[None, :]         # [S][w]
        ii = i0[:, None] + np.arange(-rad, rad + 1)[None, :]
        ok = ((ii >= 0) & (ii < n))[:, :, None] & ((jj >= 0) & (jj < n))[:, None, :]
        flat_idx = (ii[:, :, None] * n + jj[:, None, :])[ok]
        img += np.bincount(flat_idx, weights=stamp[ok], minlength=n * n)
        del stamp, ex, ey, gx, gy
    return img.reshape(n, n) + sky


REF_NOISE_VARIANCE_RATIO = 0.1     # "10 times less variance than the target"


def add_reference_noise(cfg: Config, R_noiseless: np.ndarray) -> np.ndarray:
    """The paper's S10 reference noise: sigma_R = 10^-1/2 sqrt(sigma0^2 + R_noiseless / G) (Eq. 22, PAPER.md:280,
    with the config's sigma0 and gain in place of the paper's 5 and 1) and R_noisy = R_noiseless + W sigma_R,
    W ~ N(0, 1) (Eq. 23).  Own RNG stream `default_rng(777000 + c)`, so that the streams of the
    noiseless recipe are untouched.  float64 in, float32 out."""
    rng = np.random.default_rng(777000 + cfg.index)
    R64 = np.asarray(R_noiseless, dtype=np.float64)
    sig = np.sqrt(REF_NOISE_VARIANCE_RATIO * (cfg.sigma0 ** 2 + np.maximum(R64, 0.0) / cfg.gain))
    return (R64 + rng.standard_normal(R64.shape) * sig).astype(np.float32)


def make_reference(cfg: Config, n: Optional[int] = None) -> np.ndarray:
    """Reference image of config `cfg` (optionally at a reduced size n, keeping
    the stellar density), float32 [n][n]."""
    n = cfg.n if n is None else n
    n_stars = cfg.n_stars if n == cfg.n else max(1, int(round(cfg.n_stars * (n / cfg.n) ** 2)))
    rng = np.random.default_rng(cfg.index)
    xs = rng.uniform(0.0, n, n_stars)
    ys = rng.uniform(0.0, n, n_stars)
    lf = rng.uniform(math.log10(cfg.flux_lo), math.log10(cfg.flux_hi), n_stars)
    R = render_stars(n, xs, ys, 10.0 ** lf, cfg.fwhm, cfg.sky)
    return R.astype(np.float32)


# --------------------------------------------------------------------------
# planted kernels
# --------------------------------------------------------------------------
def _grid(m: int):
    h = (m - 1) // 2
    d = np.arange(m, dtype=np.float64) - h
    dy, dx = np.meshgrid(d, d, indexing="ij")   # row = dy, column = dx
    return dx, dy


def _scaled(K: np.ndarray, total: float) -> np.ndarray:
    return K * (total / K.sum())


def planted_kernel(cfg: Config, m: int, rng: np.random.Generator):
    """(K_true [m][m] float64, B0_true) for one target epoch."""
    dx, dy = _grid(m)
    r2 = dx * dx + dy * dy
    if cfg.kernel == "c0":
        return _scaled(np.exp(-r2 / (2.0 * 1.0 ** 2)), 1.2), 5.0
    if cfg.kernel == "c1":
        t = math.radians(-30.0)
        ux, uy = dx - 0.3, dy + 0.2
        qx = math.cos(t) * ux - math.sin(t) * uy
        qy = math.sin(t) * ux + math.cos(t) * uy
        return _scaled(np.exp(-0.5 * (qx ** 2 / 1.5 ** 2 + qy ** 2 / 1.2 ** 2)), 0.9), -10.0
    if cfg.kernel == "c2":
        g1 = np.exp(-r2 / (2.0 * 1.2 ** 2))
        g2 = np.exp(-r2 / (2.0 * 3.0 ** 2))
        return _scaled(0.8 * g1 / g1.sum() + 0.2 * g2 / g2.sum(), 1.1), 20.0
    if cfg.kernel == "c3":
        return _scaled((1.0 + r2 / 2.5 ** 2) ** (-3.0), 1.05), 7.0
    if cfg.kernel == "c4":
        sig = rng.uniform(1.0, 2.5)
        scale = rng.uniform(0.8, 1.2)
        b0 = rng.uniform(-20.0, 20.0)
        return _scaled(np.exp(-r2 / (2.0 * sig ** 2)), scale), b0
    raise ValueError(cfg.kernel)


# --------------------------------------------------------------------------
# target images
# --------------------------------------------------------------------------
def correlate_valid(R: np.ndarray, K: np.ndarray) -> np.ndarray:
    """sum_ab K[a][b] R[i+a][j+b] for the (n-m+1)^2 valid outputs, float64.

    Library routine only (scipy.signal): direct correlation for small images,
    FFT-based for large ones.  This is the simulation step of the generator.
    """
    R = np.asarray(R, dtype=np.float64)
    K = np.asarray(K, dtype=np.float64)
    if R.shape[0] <= 256:
        return signal.correlate2d(R, K, mode="valid")
    return signal.fftconvolve(R, K[::-1, ::-1], mode="valid")


def make_target(cfg: Config, epoch: int, R: np.ndarray, m: Optional[int] = None,
                noise: bool = True):
    """One target epoch: (I float32 [n][n], theta_true float64 [m*m+1],
    flat float32|None, mask uint8|None)."""
    n = R.shape[0]
    m = cfg.m if m is None else m
    h = (m - 1) // 2
    rng = np.random.default_rng(10000 * (cfg.index + 1) + epoch)
    K, b0 = planted_kernel(cfg, m, rng)
    P = K.sum()
    R64 = R.astype(np.float64)
    I_nl = P * R64 + b0                      # border filler, never read by a fit
    I_nl[h:n - h, h:n - h] = correlate_valid(R64, K) + b0
    flat = rng.uniform(0.95, 1.05, (n, n)) if cfg.flat else None
    F = flat if flat is not None else 1.0
    I = I_nl
    if noise:
        var = cfg.sigma0 ** 2 / (F * F) + np.maximum(I_nl, 0.0) / (cfg.gain * F)
        I = I_nl + rng.standard_normal((n, n)) * np.sqrt(var)
    mask = None
    if cfg.cosmic_frac > 0.0:
        k = int(round(cfg.cosmic_frac * n * n))
        idx = rng.choice(n * n, size=k, replace=False)
        I = I.copy()
        I.reshape(-1)[idx] = rng.uniform(1e3, 1e4, k)
    if cfg.saturate_frac > 0.0:
        k = int(round(cfg.saturate_frac * n * n))
        idx = rng.choice(n * n, size=k, replace=False)
        I = I.copy()
        I.reshape(-1)[idx] = 6.5e4
        mask = np.ones(n * n, dtype=np.uint8)
        mask[idx] = 0
        mask = mask.reshape(n, n)
    theta = np.concatenate([K.reshape(-1), [b0]])
    return (I.astype(np.float32), theta,
            None if flat is None else flat.astype(np.float32), mask)


def theta_init(R: np.ndarray, I: np.ndarray, m: int) -> np.ndarray:
    """Flat-kernel initial guess [m*m+1] float32: K = 1/N_K and
    B0 = median(I over the valid region) - median(R) * sum(K_init), which is the
    paper's B0 = median(I) when R is background-subtracted (R11)."""
    n = R.shape[0]
    h = (m - 1) // 2
    th = np.full(m * m + 1, 1.0 / (m * m), dtype=np.float64)
    th[-1] = float(np.median(I[h:n - h, h:n - h])) - float(np.median(R)) * 1.0
    return th.astype(np.float32)


def gaussian_kernel_init(m: int, phi_k: float, b0: float) -> np.ndarray:
    """Symmetric Gaussian initial kernel of width phi_k summing to 1
     followed by b0, float32 [m*m+1]."""
    dx, dy = _grid(m)
    K = np.exp(-(dx * dx + dy * dy) / (2.0 * phi_k ** 2))
    K /= K.sum()
    return np.concatenate([K.reshape(-1), [b0]]).astype(np.float32)


def make_workload(c: int, n: Optional[int] = None, n_epochs: Optional[int] = None,
                  m: Optional[int] = None, noise: bool = True, ref_noise: bool = False,
                  epochs: Optional[Sequence[int]] = None, sky_subtract: bool = False) -> Workload:
    """Config `c` of BASELINE.json; n / n_epochs / m may be reduced for tests
    (same recipe, same stellar density, same RNG streams).  `epochs` selects target epochs by index (default
    0 .. n_epochs-1).  `ref_noise`: the targets are simulated from the noiseless reference as
    always, and the reference handed to the fit carries the paper's S10 noise (Eq. 22-23) -- the situation of
    every image pair of the paper; BASELINE.json's configs are the ref_noise = False case.  `sky_subtract`: the
    reference handed to the fit has its sky level removed ("we always background subtract the reference image",
    PAPER.md:240) -- the targets are unchanged, so the planted B0 becomes B0 + P sky in theta_true; BASELINE.json's
    configs leave the sky in (sky_subtract = False)."""
    cfg = CONFIGS[c]
    n = cfg.n if n is None else n
    m = cfg.m if m is None else m
    E = cfg.n_epochs if n_epochs is None else n_epochs
    R_true = make_reference(cfg, n)
    R = add_reference_noise(cfg, R_true) if ref_noise else R_true
    if sky_subtract:
        R = (R.astype(np.float64) - cfg.sky).astype(np.float32)
    Is, thetas, masks, theta0s = [], [], [], []
    flat = None
    for e in (range(E) if epochs is None else epochs):
        I, th, fl, mk = make_target(cfg, e, R_true, m, noise)
        if sky_subtract:
            th = th.copy()
            th[-1] += th[:-1].sum() * cfg.sky
        Is.append(I)
        thetas.append(th)
        theta0s.append(theta_init(R, I, m))
        if fl is not None and flat is None:
            flat = fl            # one master flat per handle: epoch 0's draw
        if mk is not None:
            masks.append(mk)
    return Workload(cfg, n, m, R, np.stack(Is), np.stack(thetas), np.stack(theta0s),
                    flat, np.stack(masks) if masks else None,
                    cfg.sigma0, cfg.gain, cfg.loss)
