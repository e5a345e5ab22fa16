"""Seeded synthetic scans that stand in for the paper's workloads.

This module serves BOTH the tests of the CPU oracle and the CUDA path and belongs to neither: it holds no
step of the reconstruction method.  It only draws numbers from a counter-based generator and, to make
physically consistent diffraction data, evaluates the forward model Eq. (1) ONCE with
numpy's FFT (a library routine shared with neither side).  Everything is produced in float64, then rounded
once to the float32 / complex64 arrays both sides consume.

The paper's own data (SEM-derived gold-ball phantom, zone-plate illumination, ALS scans)
are not available; BASELINE.json `configs` defines these stand-ins with the paper's shapes (128x128 frames,
50x50 scans, 10,000-frame simulations).
"""
from __future__ import annotations

from dataclasses import dataclass, replace

import numpy as np

_MASK = np.uint64(0xFFFFFFFFFFFFFFFF)
BASE_SEED = 1602014480

# random streams
S_AMP, S_PHASE, S_JITTER, S_POISSON, S_MISC = 1, 2, 3, 4, 5


def _splitmix64(x: np.ndarray) -> np.ndarray:
    """One splitmix64 output step on uint64 arrays (wrap-around arithmetic)."""
    with np.errstate(over="ignore"):
        x = (x + np.uint64(0x9E3779B97F4A7C15)) & _MASK
        z = x
        z = ((z ^ (z >> np.uint64(30))) * np.uint64(0xBF58476D1CE4E5B9)) & _MASK
        z = ((z ^ (z >> np.uint64(27))) * np.uint64(0x94D049BB133111EB)) & _MASK
        return z ^ (z >> np.uint64(31))


def uniform(seed: int, stream: int, index) -> np.ndarray:
    """U[0,1) doubles, a pure function of (seed, stream, index): hash = sm64(sm64(sm64(seed)+stream)+index)."""
    idx = np.asarray(index, dtype=np.uint64)
    with np.errstate(over="ignore"):
        k = _splitmix64(np.asarray([seed], dtype=np.uint64))
        k = _splitmix64((k + np.uint64(stream)) & _MASK)
        h = _splitmix64((k + idx) & _MASK)
    return (h >> np.uint64(11)).astype(np.float64) * (1.0 / 9007199254740992.0)


def poisson(lam: np.ndarray, seed: int, stream: int, index0: int = 0) -> np.ndarray:
    """Poisson(lam) counts driven by one or two counter-based uniforms per element.

    lam < 32: inversion by sequential search on one uniform.  lam >= 32: rounded normal approximation
    (Box-Muller on two uniforms), clamped at 0.  A stand-in for detector shot noise, not a statistics library.
    """
    lam = np.asarray(lam, dtype=np.float64)
    flat = lam.ravel()
    n = flat.size
    idx = np.arange(index0, index0 + n, dtype=np.uint64)
    u = uniform(seed, stream, idx)
    out = np.zeros(n, dtype=np.float64)
    small = flat < 32.0
    # inversion for the small-rate elements
    sel = np.nonzero(small)[0]
    if sel.size:
        l = flat[sel]; us = u[sel]
        p = np.exp(-l); cdf = p.copy(); k = np.zeros(sel.size)
        active = np.nonzero(us > cdf)[0]
        it = 0
        while active.size and it < 200:
            it += 1
            k[active] += 1.0
            p[active] *= l[active] / k[active]
            cdf[active] += p[active]
            active = active[us[active] > cdf[active]]
        out[sel] = k
    big = np.nonzero(~small)[0]
    if big.size:
        u1 = u[big]
        u2 = uniform(seed, stream + 100, idx[big])
        g = np.sqrt(-2.0 * np.log(1.0 - u1)) * np.cos(2.0 * np.pi * u2)
        out[big] = np.maximum(0.0, np.rint(flat[big] + np.sqrt(flat[big]) * g))
    return out.reshape(lam.shape)


@dataclass(frozen=True)
class ScanConfig:
    """One synthetic scan.  `kind`: 'raster' (grid x grid, step, +-jitter) or 'fermat' (K spiral points)."""
    name: str
    m: int
    kind: str
    grid: int            # raster: points per side; fermat: total number of points
    step: int            # raster step / fermat radial scale (px)
    jitter: int          # raster: integer jitter amplitude J (uniform in {-J..J}, offset +J keeps pos >= 0)
    pupil_radius: float  # R, Fourier pixels; phase 0.01*rho^2 (reading G18-A)
    photons: float       # per frame; 0 = noise-free
    beta: float
    iters: int
    refine_every: int
    seed: int
    blind_start: bool = False   # start probe = Gaussian sigma=m/8 (configs 3, 5)
    phase_coeff: float = 0.01   # pupil phase = phase_coeff * rho^2 (the configs say 0.01)
    periodic: int = 0           # > 0: periodic boundary on a periodic x periodic image (the paper's Fig. 3 simulation)

    @property
    def K(self) -> int:
        return self.grid * self.grid if self.kind == "raster" else self.grid

    @property
    def shape(self):
        if self.periodic:
            return (self.periodic, self.periodic)
        if self.kind == "raster":
            n = (self.grid - 1) * self.step + self.m + 2 * self.jitter
            return (n, n)
        r = self.step * np.sqrt(self.grid - 1.0)
        c = int(np.ceil(r / 64.0)) * 64          # centre; cfg 5: 48*sqrt(1599)=1919.4 -> 1920
        return (2 * c + self.m, 2 * c + self.m)


def config(n: int) -> ScanConfig:
    """BASELINE.json configs[n-1] (n = 1..5) as read in SURVEY.md section 8(d)."""
    s = BASE_SEED + n
    if n == 1:
        return ScanConfig("tiny", 64, "raster", 10, 16, 0, 12.0, 1e4, 0.75, 100, 0, s)
    if n == 2:
        return ScanConfig("medium", 128, "raster", 50, 32, 4, 24.0, 1e5, 0.75, 200, 0, s)
    if n == 3:
        return ScanConfig("medium-blind", 128, "raster", 50, 32, 4, 24.0, 1e5, 0.75, 200, 1, s, True)
    if n == 4:
        return ScanConfig("large", 256, "raster", 100, 48, 6, 48.0, 0.0, 0.9, 100, 0, s)
    if n == 5:
        return ScanConfig("very-large", 512, "fermat", 1600, 48, 0, 96.0, 1e6, 0.75, 100, 1, s, True)
    if n == 6:
        # the paper's own Fig. 3 shape: 10,000 frames 128x128 on a 1000x1000 image, periodic boundary,
        # 164 frames per pixel, exact illumination given, noise-free; beta is the paper's default
        return ScanConfig("fig3-periodic", 128, "raster", 100, 10, 0, 24.0, 0.0, 0.75, 100, 0, s, periodic=1000)
    raise ValueError("config number must be 1..6")


def reduced(cfg: ScanConfig, grid: int, **kw) -> ScanConfig:
    """The same recipe on a smaller raster / fewer spiral points (sizes the oracle finishes in seconds).  A periodic
    scan keeps its step and shrinks the image with the raster (grid * step pixels), so it still tiles the torus."""
    if cfg.periodic and "periodic" not in kw:
        kw["periodic"] = grid * cfg.step
    return replace(cfg, grid=grid, name=f"{cfg.name}-g{grid}", **kw)


def positions(cfg: ScanConfig) -> np.ndarray:
    """int32 (K,2) (row, col) of each frame's top-left pixel, all within {0..n-m}."""
    if cfg.kind == "raster":
        i, j = np.meshgrid(np.arange(cfg.grid), np.arange(cfg.grid), indexing="ij")
        pos = np.stack([i.ravel() * cfg.step, j.ravel() * cfg.step], axis=1).astype(np.int64)
        if cfg.jitter:
            J = cfg.jitter
            u = uniform(cfg.seed, S_JITTER, np.arange(2 * cfg.K)).reshape(cfg.K, 2)
            pos += np.floor(u * (2 * J + 1)).astype(np.int64) - J + J
        return pos.astype(np.int32)
    k = np.arange(cfg.grid, dtype=np.float64)
    rad = cfg.step * np.sqrt(k)
    ang = k * np.pi * (3.0 - np.sqrt(5.0))
    c = (cfg.shape[0] - cfg.m) // 2
    pos = np.stack([np.floor(c + rad * np.cos(ang) + 0.5), np.floor(c + rad * np.sin(ang) + 0.5)], axis=1)
    return pos.astype(np.int32)


def true_object(cfg: ScanConfig) -> np.ndarray:
    """complex64 (n_r, n_c): i.i.d. amplitude U[0.8,1], phase U[-pi/2, pi/2]."""
    nr, nc = cfg.shape
    idx = np.arange(nr * nc)
    amp = 0.8 + 0.2 * uniform(cfg.seed, S_AMP, idx)
    ph = (uniform(cfg.seed, S_PHASE, idx) - 0.5) * np.pi
    return (amp * np.exp(1j * ph)).reshape(nr, nc).astype(np.complex64)


def true_probe(cfg: ScanConfig) -> np.ndarray:
    """complex64 (m,m): w = fftshift(F*(ifftshift D)), D = [rho<=R] exp(i 0.01 rho^2), rho from (m/2,m/2)
    (readings G18-A, G19); unitary, so sum|w|^2 = number of pupil pixels."""
    m = cfg.m
    u = np.arange(m) - m // 2
    rho2 = (u[:, None] ** 2 + u[None, :] ** 2).astype(np.float64)
    D = np.where(rho2 <= cfg.pupil_radius ** 2, np.exp(1j * cfg.phase_coeff * rho2), 0.0)
    w = np.fft.fftshift(np.fft.ifft2(np.fft.ifftshift(D), norm="ortho"))
    return w.astype(np.complex64)


def start_probe(cfg: ScanConfig, intensities: np.ndarray | None = None) -> np.ndarray:
    """The probe handed to the library: the true one, or for blind configs a Gaussian sigma = m/8 at the
    frame centre scaled so that sum|w|^2 = mean_i sum_q I_i."""
    if not cfg.blind_start:
        return true_probe(cfg)
    m = cfg.m
    u = np.arange(m) - m // 2
    g = np.exp(-(u[:, None] ** 2 + u[None, :] ** 2) / (2.0 * (m / 8.0) ** 2))
    if intensities is not None:
        tot = float(np.asarray(intensities, dtype=np.float64).reshape(-1, m * m).sum(axis=1).mean())
    else:
        tot = float(np.sum(np.abs(true_probe(cfg).astype(np.complex128)) ** 2))
    g *= np.sqrt(tot / np.sum(g * g))
    return g.astype(np.complex64)


def exit_waves(cfg: ScanConfig, obj: np.ndarray, probe: np.ndarray, pos: np.ndarray, lo=0, hi=None):
    """float64-complex frames w * psi(. + x_i) for frames lo..hi (used to build data and fixed-point tests)."""
    hi = len(pos) if hi is None else hi
    m = cfg.m
    r = np.arange(m)
    rows = pos[lo:hi, 0, None, None] + r[None, :, None]
    cols = pos[lo:hi, 1, None, None] + r[None, None, :]
    if cfg.periodic:
        rows, cols = rows % obj.shape[0], cols % obj.shape[1]
    return probe.astype(np.complex128)[None] * obj.astype(np.complex128)[rows, cols]


def intensities(cfg: ScanConfig, obj=None, probe=None, pos=None, chunk: int = 256) -> np.ndarray:
    """float32 (K,m,m): I_i = |F(w psi(.+x_i))|^2, unitary DFT with kernel e^{-2 pi i q.r}, DC at [0,0]
    (Eq. 1; readings G2, G3), then Poisson(s I)/s with s = photons / mean_i sum_q I_i when photons > 0."""
    obj = true_object(cfg) if obj is None else obj
    probe = true_probe(cfg) if probe is None else probe
    pos = positions(cfg) if pos is None else pos
    K, m = len(pos), cfg.m
    out = np.empty((K, m, m), dtype=np.float32)
    tot = 0.0
    for lo in range(0, K, chunk):
        hi = min(K, lo + chunk)
        Z = np.fft.fft2(exit_waves(cfg, obj, probe, pos, lo, hi), norm="ortho")
        Iq = Z.real ** 2 + Z.imag ** 2
        tot += float(Iq.sum())
        if cfg.photons > 0:
            out[lo:hi] = 0  # filled in the second pass
        else:
            out[lo:hi] = Iq.astype(np.float32)
    if cfg.photons > 0:
        s = cfg.photons / (tot / K)
        for lo in range(0, K, chunk):
            hi = min(K, lo + chunk)
            Z = np.fft.fft2(exit_waves(cfg, obj, probe, pos, lo, hi), norm="ortho")
            Iq = Z.real ** 2 + Z.imag ** 2
            cnt = poisson(s * Iq, cfg.seed, S_POISSON, index0=lo * m * m)
            out[lo:hi] = (cnt / s).astype(np.float32)
    return out


def make(cfg: ScanConfig):
    """(pos int32 (K,2), shape, intensities f32 (K,m,m), start probe c64 (m,m), true object c64, true probe c64)."""
    pos = positions(cfg)
    obj = true_object(cfg)
    wt = true_probe(cfg)
    I = intensities(cfg, obj, wt, pos)
    w0 = start_probe(cfg, I)
    return pos, cfg.shape, I, w0, obj, wt
