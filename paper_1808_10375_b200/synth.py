"""Seeded synthetic fly-scan ptychography inputs (the five BASELINE.json configs).

This module is the ONLY code shared by the CUDA path's tests/bench and the oracle's
tests: it makes inputs, nothing else.  It holds none of the difference-map arithmetic
(no psi update, no modulus projection, no overlap projection); it does evaluate the
paper's *forward model* eq. (1)-(2) with a library FFT to synthesise
intensities, because that is what "synthetic data" means for this method
("generate the hypothetical diffraction pattern").

Recipe (restated in DESIGN.md):
  * one numpy Generator (PCG64) per config, seed 0 unless stated, draws in the fixed
    order: jitter-y, jitter-x, object amplitude, object phase field(s), start field(s)
    of object modes l >= 2, Poisson noise.
  * positions: y0 = margin_y + iy*step + U{-jit..+jit}, x likewise, j = iy*nx + ix.
  * object: amplitude iid U[0.8,1]; phase = Gaussian-smoothed white normal field mapped
    affinely to [-pi/2, pi/2]; object mode 2 = 0.3*exp(i*phi2).
  * probe: Gaussian amplitude (sigma) times quadratic phase exp(i*c*r^2), centre
    (N/2, N/2); mode k = sqrt(w_k) * roll(P_base, shift_k, axis=x).
  * I_j = sum_kl |FFT2(P_k * O_l|window)|^2 in float64, DC at [0,0], Poisson-scaled so
    that the mean frame holds `photons` counts (data stay in |FFT|^2 units), float32.
  * start state: P0 = 0.9*P_true; O0_1 = 1; O0_l (l>=2) = 0.1 * unit-RMS smoothed
    complex normal field.
Everything returned is float32 / complex64 / int32: both sides start from bit-identical
numbers.
"""
from __future__ import annotations

import dataclasses
import numpy as np

try:  # multi-threaded batched FFT for the big configs; numpy.fft is the fallback
    import scipy.fft as _fft
    _FFT_KW = {"workers": -1}
except Exception:  # pragma: no cover
    import numpy.fft as _fft
    _FFT_KW = {}


@dataclasses.dataclass(frozen=True)
class DMConfig:
    name: str
    N: int
    ny: int
    nx: int
    step: int
    jit: int
    obj_h: int
    obj_w: int
    K: int
    L: int
    probe_sigma: float
    probe_c: float
    shifts: tuple
    weights: tuple
    phase_sigma: float
    photons: float | None
    n_iter: int

    @property
    def n_views(self) -> int:
        return self.ny * self.nx

    @property
    def mode_views(self) -> int:
        return self.n_views * self.K * self.L

    def scaled(self, ny: int, nx: int, name: str | None = None) -> "DMConfig":
        """Same N, K, L, step, jitter, probe and noise; a smaller raster and the object
        cropped to fit it with the config's own margins (used for parity cases the
        oracle finishes in seconds)."""
        my = (self.obj_h - ((self.ny - 1) * self.step + self.N)) // 2
        mx = (self.obj_w - ((self.nx - 1) * self.step + self.N)) // 2
        h = (ny - 1) * self.step + self.N + 2 * my
        w = (nx - 1) * self.step + self.N + 2 * mx
        w += w & 1
        return dataclasses.replace(self, ny=ny, nx=nx, obj_h=h, obj_w=w,
                                   name=name or f"{self.name}-{ny}x{nx}")


CONFIGS = (
    DMConfig("c0-tiny", 64, 10, 10, 8, 1, 160, 160, 1, 1, 10.0, 0.02, (0,), (1.0,), 4.0, None, 50),
    DMConfig("c1-flyscan2", 128, 50, 50, 10, 2, 640, 640, 2, 1, 20.0, 0.005, (0, 3), (0.8, 0.2), 6.0, 1e6, 100),
    DMConfig("c2-dense4", 128, 100, 100, 6, 1, 760, 760, 4, 1, 20.0, 0.005, (0, 1, 3, 4),
             (0.4, 0.3, 0.2, 0.1), 6.0, 1e5, 100),
    DMConfig("c3-probe4obj2", 256, 64, 64, 16, 2, 1300, 1300, 4, 2, 40.0, 0.00125, (0, 4, 8, 12),
             (0.4, 0.3, 0.2, 0.1), 6.0, 1e6, 100),
    DMConfig("c4-large512", 512, 40, 50, 32, 3, 1800, 2100, 3, 1, 60.0, 0.0003125, (0, 10, 21),
             (0.6, 0.3, 0.1), 6.0, 1e7, 50),
)


@dataclasses.dataclass
class DMProblem:
    cfg: DMConfig
    positions: np.ndarray      # int32 [n_views][2] = (y0, x0), top-left corner of the window
    intensities: np.ndarray    # float32 [n_views][N][N], DC at [0,0]
    probe0: np.ndarray         # complex64 [K][N][N]
    object0: np.ndarray        # complex64 [L][H][W]
    probe_true: np.ndarray     # complex64 [K][N][N]
    object_true: np.ndarray    # complex64 [L][H][W]


def _smooth_field(rng: np.random.Generator, h: int, w: int, sigma: float, complex_: bool = False):
    """White normal field circularly convolved with a Gaussian of width sigma (pixels)."""
    white = rng.standard_normal((h, w))
    if complex_:
        white = white + 1j * rng.standard_normal((h, w))
    fy = np.fft.fftfreq(h)[:, None]
    fx = np.fft.fftfreq(w)[None, :]
    kern = np.exp(-2.0 * np.pi ** 2 * sigma ** 2 * (fy ** 2 + fx ** 2))
    out = _fft.ifft2(_fft.fft2(white, **_FFT_KW) * kern, **_FFT_KW)
    return out if complex_ else out.real


def _phase_field(rng, h, w, sigma):
    f = _smooth_field(rng, h, w, sigma)
    lo, hi = f.min(), f.max()
    return (f - lo) / (hi - lo) * np.pi - np.pi / 2.0


def make_positions(cfg: DMConfig, rng: np.random.Generator) -> np.ndarray:
    my = (cfg.obj_h - ((cfg.ny - 1) * cfg.step + cfg.N)) // 2
    mx = (cfg.obj_w - ((cfg.nx - 1) * cfg.step + cfg.N)) // 2
    jy = rng.integers(-cfg.jit, cfg.jit + 1, size=(cfg.ny, cfg.nx))
    jx = rng.integers(-cfg.jit, cfg.jit + 1, size=(cfg.ny, cfg.nx))
    iy, ix = np.meshgrid(np.arange(cfg.ny), np.arange(cfg.nx), indexing="ij")
    y0 = my + iy * cfg.step + jy
    x0 = mx + ix * cfg.step + jx
    pos = np.stack([y0.ravel(), x0.ravel()], axis=1).astype(np.int32)
    assert pos[:, 0].min() >= 0 and pos[:, 0].max() + cfg.N <= cfg.obj_h
    assert pos[:, 1].min() >= 0 and pos[:, 1].max() + cfg.N <= cfg.obj_w
    return pos


def make_probe(cfg: DMConfig) -> np.ndarray:
    n = cfg.N
    y = np.arange(n)[:, None] - n / 2
    x = np.arange(n)[None, :] - n / 2
    r2 = y * y + x * x
    base = np.exp(-r2 / (2.0 * cfg.probe_sigma ** 2)) * np.exp(1j * cfg.probe_c * r2)
    modes = [np.sqrt(w) * np.roll(base, s, axis=1) for w, s in zip(cfg.weights, cfg.shifts)]
    return np.stack(modes).astype(np.complex128)


def make_problem(cfg: DMConfig | int, seed: int = 0, view_batch: int = 256) -> DMProblem:
    if isinstance(cfg, int):
        cfg = CONFIGS[cfg]
    rng = np.random.default_rng(seed)
    n, h, w = cfg.N, cfg.obj_h, cfg.obj_w
    pos = make_positions(cfg, rng)

    amp = rng.uniform(0.8, 1.0, size=(h, w))
    obj = [amp * np.exp(1j * _phase_field(rng, h, w, cfg.phase_sigma))]
    for _ in range(1, cfg.L):
        obj.append(0.3 * np.exp(1j * _phase_field(rng, h, w, cfg.phase_sigma)))
    obj = np.stack(obj)
    obj0 = [np.ones((h, w), dtype=np.complex128)]
    for _ in range(1, cfg.L):
        f = _smooth_field(rng, h, w, cfg.phase_sigma, complex_=True)
        obj0.append(0.1 * f / np.sqrt(np.mean(np.abs(f) ** 2)))
    obj0 = np.stack(obj0)

    probe = make_probe(cfg)

    inten = np.empty((cfg.n_views, n, n), dtype=np.float64)
    ar = np.arange(n)
    for b0 in range(0, cfg.n_views, view_batch):
        b1 = min(b0 + view_batch, cfg.n_views)
        yy = pos[b0:b1, 0][:, None, None] + ar[None, :, None]
        xx = pos[b0:b1, 1][:, None, None] + ar[None, None, :]
        acc = np.zeros((b1 - b0, n, n))
        for l in range(cfg.L):
            win = obj[l][yy, xx]                                    # [b][N][N]
            for k in range(cfg.K):
                f = _fft.fft2(win * probe[k][None], axes=(-2, -1), **_FFT_KW)
                acc += f.real ** 2 + f.imag ** 2
        inten[b0:b1] = acc

    if cfg.photons is not None:
        s = cfg.photons / inten.sum(axis=(1, 2)).mean()
        inten = rng.poisson(inten * s).astype(np.float64) / s

    return DMProblem(
        cfg=cfg,
        positions=pos,
        intensities=np.ascontiguousarray(inten, dtype=np.float32),
        probe0=np.ascontiguousarray(0.9 * probe, dtype=np.complex64),
        object0=np.ascontiguousarray(obj0, dtype=np.complex64),
        probe_true=np.ascontiguousarray(probe, dtype=np.complex64),
        object_true=np.ascontiguousarray(obj, dtype=np.complex64),
    )


def rel_l2(a: np.ndarray, b: np.ndarray) -> float:
    """Relative L2 distance ||a-b|| / ||b|| in float64 (comparison utility, no method arithmetic)."""
    a = np.asarray(a).astype(np.complex128 if np.iscomplexobj(a) or np.iscomplexobj(b) else np.float64)
    b = np.asarray(b).astype(a.dtype)
    den = np.linalg.norm(b.ravel())
    num = np.linalg.norm((a - b).ravel())
    return float(num / den) if den > 0 else float(num)


def make_sampled_problem(cfg: DMConfig | int, sample_views, seed: int = 0) -> DMProblem:
    """Full-size inputs for parity on SAMPLED views (tests at BASELINE.json's full sizes, where the
    oracle cannot hold every view): positions, probe and object as in make_problem, but noise-free
    intensities are synthesised for `sample_views` only (all other frames are zero) and the start
    state is the near-truth one, P0 = 0.9 P_true, O0 = O_true, whose spectrum has the data's own
    shape (an FP32-well-conditioned first step)."""
    if isinstance(cfg, int):
        cfg = CONFIGS[cfg]
    rng = np.random.default_rng(seed)
    n, h, w = cfg.N, cfg.obj_h, cfg.obj_w
    pos = make_positions(cfg, rng)
    amp = rng.uniform(0.8, 1.0, size=(h, w))
    obj = [amp * np.exp(1j * _phase_field(rng, h, w, cfg.phase_sigma))]
    for _ in range(1, cfg.L):
        obj.append(0.3 * np.exp(1j * _phase_field(rng, h, w, cfg.phase_sigma)))
    obj = np.stack(obj)
    probe = make_probe(cfg)
    inten = np.zeros((cfg.n_views, n, n), dtype=np.float32)
    ar = np.arange(n)
    for j in sample_views:
        yy = pos[j, 0] + ar[:, None]
        xx = pos[j, 1] + ar[None, :]
        acc = np.zeros((n, n))
        for l in range(cfg.L):
            for k in range(cfg.K):
                f = _fft.fft2(obj[l][yy, xx] * probe[k])
                acc += f.real ** 2 + f.imag ** 2
        inten[j] = acc
    return DMProblem(
        cfg=cfg, positions=pos, intensities=inten,
        probe0=np.ascontiguousarray(0.9 * probe, dtype=np.complex64),
        object0=np.ascontiguousarray(obj, dtype=np.complex64),
        probe_true=np.ascontiguousarray(probe, dtype=np.complex64),
        object_true=np.ascontiguousarray(obj, dtype=np.complex64),
    )
