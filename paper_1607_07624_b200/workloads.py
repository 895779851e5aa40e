"""Seeded synthetic inputs for the five BASELINE.json configs.

This module serves BOTH the oracle-side tests and the CUDA-side tests/bench and
therefore holds none of the method's arithmetic: it only makes pupils
(amplitude masks) and von Karman phase screens, i.e. the data PASSATA's
atmosphere / propagation / pupil-stop objects would hand to the pyramid
(PAPER.md:L192-219, L233-235, L309-310, L341).  The paper uses no public
dataset; these stand in for its atmosphere object.  Recipe: SURVEY.md 8(d),
restated in DESIGN.md ("Input recipe").

numpy only (numpy.fft is used here to colour white noise -- generator code, not
the product path).
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field
from typing import Dict, List, Optional, Tuple

import numpy as np

ARCSEC = math.pi / (180.0 * 3600.0)


@dataclass(frozen=True)
class WfsConfig:
    """Geometry + workload of one BASELINE.json config."""
    name: str
    D: float                 # telescope diameter [m]
    n_pupil: int             # N
    m_grid: int              # M
    obstruction: float       # central obstruction, diameter ratio
    spiders: int             # number of spider arms (0 = none)
    spider_width: float      # [m]
    mod_radius: float        # r [lambda/D]
    mod_points: int          # K
    n_subap: int             # n_sub
    wavelengths_nm: Tuple[float, ...]
    r0_500: float            # [m] at 500 nm
    L0: float                # [m]
    steps: int
    screen_px: int           # G
    layer_weights: Tuple[float, ...] = (1.0,)
    layer_heights: Tuple[float, ...] = (0.0,)
    wind_speed: Tuple[float, ...] = (0.0,)          # [m/s]
    wind_dir_deg: Tuple[float, ...] = (0.0,)
    n_stars: int = 1
    star_radius_arcsec: float = 0.0
    independent_screens: bool = False               # cfg 1: 10 independent screens
    seed: int = 0
    dt: float = 1e-3                                 # loop period [s]

    @property
    def pitch(self) -> float:
        return self.D / self.n_pupil

    @property
    def instances(self) -> int:
        return self.n_stars * len(self.wavelengths_nm)

    @property
    def batch(self) -> int:
        """B = steps x sensor instances (frames per full workload)."""
        return self.steps * self.instances

    @property
    def det_size(self) -> int:
        return 2 * self.n_subap


CONFIGS: Dict[str, WfsConfig] = {
    # configs[0]: tiny, the case the oracle finishes in seconds.
    "cfg1_tiny": WfsConfig(
        name="cfg1_tiny", D=8.0, n_pupil=64, m_grid=128, obstruction=0.10, spiders=0,
        spider_width=0.0, mod_radius=3.0, mod_points=12, n_subap=16,
        wavelengths_nm=(750.0,), r0_500=0.15, L0=25.0, steps=10, screen_px=256,
        independent_screens=True, seed=1000),
    # configs[1]: LBT FLAO-like (Table 1: 160 px, 0.05 m pitch, 3 l/D, 750 nm, 1 kHz).
    "cfg2_flao": WfsConfig(
        name="cfg2_flao", D=8.2, n_pupil=160, m_grid=320, obstruction=0.11, spiders=0,
        spider_width=0.0, mod_radius=3.0, mod_points=24, n_subap=40,
        wavelengths_nm=(750.0,), r0_500=0.12, L0=40.0, steps=1000, screen_px=1024,
        wind_speed=(15.0,), wind_dir_deg=(0.0,), seed=2000),
    # configs[2]: non-power-of-two grid (radix 2/3/5).
    "cfg3_npot": WfsConfig(
        name="cfg3_npot", D=8.0, n_pupil=240, m_grid=480, obstruction=0.0, spiders=0,
        spider_width=0.0, mod_radius=2.0, mod_points=36, n_subap=40,
        wavelengths_nm=(1650.0,), r0_500=0.10, L0=25.0, steps=500, screen_px=1024,
        wind_speed=(10.0,), wind_dir_deg=(0.0,), seed=3000),
    # configs[3]: 40 m class -- the configuration the metric's target is quoted on.
    "cfg4_elt": WfsConfig(
        name="cfg4_elt", D=39.0, n_pupil=480, m_grid=1024, obstruction=0.28, spiders=6,
        spider_width=0.5, mod_radius=4.0, mod_points=48, n_subap=92,
        wavelengths_nm=(1650.0,), r0_500=0.157, L0=25.0, steps=100, screen_px=1024,
        layer_weights=(0.6, 0.25, 0.15), layer_heights=(0.0, 0.0, 0.0),
        wind_speed=(10.0, 20.0, 30.0), wind_dir_deg=(0.0, 120.0, 240.0), seed=4000),
    # configs[4]: 6 guide stars x 2 wavelengths = 12 sensor instances per step.
    "cfg5_multi": WfsConfig(
        name="cfg5_multi", D=39.0, n_pupil=400, m_grid=800, obstruction=0.0, spiders=0,
        spider_width=0.0, mod_radius=3.0, mod_points=32, n_subap=80,
        wavelengths_nm=(1650.0, 2200.0), r0_500=0.13, L0=30.0, steps=50, screen_px=1024,
        layer_weights=(0.6, 0.25, 0.15), layer_heights=(0.0, 5000.0, 12000.0),
        wind_speed=(10.0, 20.0, 30.0), wind_dir_deg=(0.0, 120.0, 240.0),
        n_stars=6, star_radius_arcsec=60.0, seed=5000),
}
CONFIG_ORDER: List[str] = ["cfg1_tiny", "cfg2_flao", "cfg3_npot", "cfg4_elt", "cfg5_multi"]


def make_pupil(cfg: WfsConfig) -> np.ndarray:
    """Binary amplitude A[N][N] (float32): pixel-centre test eps*D/2 <= rho <= D/2
    with coordinates (i-(N-1)/2)*pitch, minus `spiders` radial arms of
    `spider_width` starting at angle 0 every 360/spiders degrees (a pixel is
    masked when its centre is within width/2 of the ray)."""
    N, pitch = cfg.n_pupil, cfg.pitch
    c = (np.arange(N) - (N - 1) / 2.0) * pitch
    X, Y = np.meshgrid(c, c)                     # Y rows, X columns
    rho = np.hypot(X, Y)
    A = (rho <= cfg.D / 2.0) & (rho >= cfg.obstruction * cfg.D / 2.0)
    for j in range(cfg.spiders):
        ang = 2.0 * math.pi * j / cfg.spiders
        ux, uy = math.cos(ang), math.sin(ang)
        along = X * ux + Y * uy                  # distance along the ray
        across = np.abs(-X * uy + Y * ux)        # distance from the ray's line
        A &= ~((along >= 0.0) & (across <= cfg.spider_width / 2.0))
    return A.astype(np.float32)


def vk_screen(G: int, pitch: float, r0: float, L0: float, seed: int) -> np.ndarray:
    """Periodic von Karman phase screen [rad] at the wavelength r0 refers to:
    FFT-filtered seeded Gaussian white noise,
    Phi(f) = 0.0229 r0^(-5/3) (|f|^2 + L0^-2)^(-11/6), Phi(0) = 0."""
    rng = np.random.default_rng(seed)
    w = rng.standard_normal((G, G)) + 1j * rng.standard_normal((G, G))
    f = np.fft.fftfreq(G, d=pitch)
    fx, fy = np.meshgrid(f, f)
    psd = 0.0229 * r0 ** (-5.0 / 3.0) * (fx * fx + fy * fy + 1.0 / (L0 * L0)) ** (-11.0 / 6.0)
    psd[0, 0] = 0.0
    df = 1.0 / (G * pitch)
    return np.real(np.fft.ifft2(w * np.sqrt(psd) * df)) * (G * G)


def _bilinear_periodic(screen: np.ndarray, xs: np.ndarray, ys: np.ndarray) -> np.ndarray:
    """Sample a periodic screen at fractional pixel coordinates (xs, ys grids)."""
    G = screen.shape[0]
    x0 = np.floor(xs).astype(np.int64)
    y0 = np.floor(ys).astype(np.int64)
    fx = xs - x0
    fy = ys - y0
    x0 %= G
    y0 %= G
    x1 = (x0 + 1) % G
    y1 = (y0 + 1) % G
    return ((1 - fy) * ((1 - fx) * screen[y0, x0] + fx * screen[y0, x1])
            + fy * ((1 - fx) * screen[y1, x0] + fx * screen[y1, x1]))


def r0_at(r0_500: float, lam_nm: float) -> float:
    return r0_500 * (lam_nm / 500.0) ** 1.2


def phase_batch(cfg: WfsConfig, steps: Optional[int] = None, first_step: int = 0) -> np.ndarray:
    """Pupil-plane phase [rad at the sensing wavelength], float32 [B][N][N] with
    B = steps x instances, step-major then star-major then wavelength-minor.
    Layers are generated as phase at 500 nm and scaled by 500/lambda."""
    steps = cfg.steps if steps is None else steps
    N, G, pitch = cfg.n_pupil, cfg.screen_px, cfg.pitch
    out = np.empty((steps * cfg.instances, N, N), dtype=np.float32)
    if cfg.independent_screens:
        for t in range(steps):
            scr = vk_screen(G, pitch, cfg.r0_500, cfg.L0, cfg.seed + first_step + t)
            for wi, lam in enumerate(cfg.wavelengths_nm):
                out[t * cfg.instances + wi] = (scr[:N, :N] * (500.0 / lam)).astype(np.float32)
        return out
    layers = [vk_screen(G, pitch, cfg.r0_500 * w ** (-3.0 / 5.0), cfg.L0, cfg.seed + li)
              for li, w in enumerate(cfg.layer_weights)]
    ii = np.arange(N, dtype=np.float64)
    X0, Y0 = np.meshgrid(ii, ii)
    for t in range(steps):
        time = (first_step + t) * cfg.dt
        for si in range(cfg.n_stars):
            az = 2.0 * math.pi * si / max(cfg.n_stars, 1)
            tan_r = math.tan(cfg.star_radius_arcsec * ARCSEC)
            opd500 = np.zeros((N, N))
            for li, scr in enumerate(layers):
                wd = math.radians(cfg.wind_dir_deg[li])
                sx = (-cfg.wind_speed[li] * time * math.cos(wd)
                      + cfg.layer_heights[li] * tan_r * math.cos(az)) / pitch
                sy = (-cfg.wind_speed[li] * time * math.sin(wd)
                      + cfg.layer_heights[li] * tan_r * math.sin(az)) / pitch
                opd500 += _bilinear_periodic(scr, X0 + sx, Y0 + sy)
            for wi, lam in enumerate(cfg.wavelengths_nm):
                idx = (t * cfg.n_stars + si) * len(cfg.wavelengths_nm) + wi
                out[idx] = (opd500 * (500.0 / lam)).astype(np.float32)
    return out


def atmosphere(cfg: WfsConfig) -> dict:
    """Inputs of the f1 propagation step for a frozen-flow config: the
    same seeded layers phase_batch() samples, stored as float32 [L][G][G] phase at 500 nm,
    plus the geometry in plain numbers -- wind velocity vectors [m/s], layer heights [m],
    tangents of the source directions, wavelength scale factors 500/lambda.  No
    interpolation or shifting happens here (that is the method, not the input)."""
    if cfg.independent_screens:
        raise ValueError(f"{cfg.name} uses independent screens, not a frozen-flow atmosphere")
    screens = np.stack([vk_screen(cfg.screen_px, cfg.pitch, cfg.r0_500 * w ** (-3.0 / 5.0), cfg.L0, cfg.seed + li)
                        for li, w in enumerate(cfg.layer_weights)]).astype(np.float32)
    wind = np.array([[v * math.cos(math.radians(d)), v * math.sin(math.radians(d))]
                     for v, d in zip(cfg.wind_speed, cfg.wind_dir_deg)], dtype=np.float64)
    tan_r = math.tan(cfg.star_radius_arcsec * ARCSEC)
    dirs = np.array([[tan_r * math.cos(2.0 * math.pi * si / max(cfg.n_stars, 1)),
                      tan_r * math.sin(2.0 * math.pi * si / max(cfg.n_stars, 1))]
                     for si in range(cfg.n_stars)], dtype=np.float64)
    return dict(screens=screens, pitch=cfg.pitch, wind_vxy=wind,
                heights=np.array(cfg.layer_heights, dtype=np.float64), dirs_tan=dirs,
                wl_scale=np.array([500.0 / lam for lam in cfg.wavelengths_nm], dtype=np.float64),
                dt=cfg.dt, n_pupil=cfg.n_pupil)


def zernike_ifs(A: np.ndarray, n_modes: int) -> Tuple[np.ndarray, np.ndarray]:
    """Test / bench input for the DM (Table 1 `dm`: type 'zernike', nmodes 54): the first n_modes
    Zernike polynomials after piston (Noll order j = 2 ..), sampled at the centres of the lit pixels of the
    pupil A[N][N] (unit disc = the N-px pupil, same coordinates as make_pupil), each scaled to unit rms over
    those pixels.  Returns (ifs float32 [n_modes][n_pix], pix int32 [n_pix] = flat indices y*N + x).
    An input generator only: how the DM uses it is the method, which lives elsewhere."""
    N = A.shape[0]
    c = (np.arange(N) - (N - 1) / 2.0) / (N / 2.0)
    X, Y = np.meshgrid(c, c)
    lit = np.flatnonzero(A.ravel() > 0)
    rho, th = np.hypot(X, Y).ravel()[lit], np.arctan2(Y, X).ravel()[lit]
    out = np.empty((n_modes, lit.size), dtype=np.float64)
    j, n = 1, 0
    rows = 0
    while rows < n_modes:
        n += 1
        for m in range(n % 2, n + 1, 2):                     # |m| = n, n-2, ... (ascending |m|: Noll-like order)
            rad = np.zeros_like(rho)
            for k in range((n - m) // 2 + 1):
                rad += ((-1) ** k * math.factorial(n - k)
                        / (math.factorial(k) * math.factorial((n + m) // 2 - k) * math.factorial((n - m) // 2 - k))) * rho ** (n - 2 * k)
            for trig in ((None,) if m == 0 else (np.cos, np.sin)):
                if rows >= n_modes:
                    break
                z = rad if trig is None else rad * trig(m * th)
                out[rows] = z / np.sqrt(np.mean(z * z))
                rows += 1
    return out.astype(np.float32), lit.astype(np.int32)


def tilt_phase(N: int, alpha_x: float, alpha_y: float = 0.0) -> np.ndarray:
    """Test input: a pure tilt of (alpha_x, alpha_y) lambda/D across the N-px
    pupil, phi = 2 pi (alpha_x (x-c) + alpha_y (y-c)) / N, float32."""
    c = (N - 1) / 2.0
    i = np.arange(N) - c
    X, Y = np.meshgrid(i, i)
    return (2.0 * math.pi * (alpha_x * X + alpha_y * Y) / N).astype(np.float32)


def shard_range(n_items: int, rank: int, world: int) -> Tuple[int, int]:
    """Contiguous block partition of n_items over `world` ranks: [lo, hi)."""
    base, rem = divmod(n_items, world)
    lo = rank * base + min(rank, rem)
    return lo, lo + base + (1 if rank < rem else 0)
