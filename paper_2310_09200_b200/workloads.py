"""Seeded synthetic workloads (the five configs of BASELINE.json) — inputs only.

This module serves BOTH the CUDA path and the oracle and therefore holds none of the method's
arithmetic: no Gram matrix, no eigensolve, no synthesis. It simulates what a telescope would
hand to ``collect``: antenna positions per epoch, beamforming weights, the visibility matrix S
(data model of PAPER.md Eq. 3, 5, 23: a_i(r) = exp(+j 2 pi <p_i, r>/lambda_w),
S = W^H (sum_q sigma_q a(r_q) a(r_q)^H + sigma_n^2 I) W, exact expectation, fp64, rounded once to
complex64), the pixel unit vectors and a deterministic placement of level edges given a list
of eigenvalues that the caller obtained elsewhere.

The paper measures on OSKAR-simulated SKA-Low MeasurementSets and LOFAR/MWA data
(PAPER.md:455, :510, :607); none of that is available here, so these generators stand in for it
with the same shapes (512 / 37x48 stations, 20-100 epochs over 6-8 h, 256^2-2048^2 pixels,
point-source skies). Recipe: DESIGN.md "Synthetic inputs". numpy only; no torch, no CUDA.
"""
from __future__ import annotations

from dataclasses import dataclass, field

import numpy as np

C_LIGHT = 299792458.0
BASE_SEED = 23100920          # arXiv id 2310.09200; seed = BASE_SEED + config index (1..5)


@dataclass(frozen=True)
class Config:
    idx: int
    name: str
    n_ant: int
    n_beam: int
    n_eig: int
    n_levels: int
    n_side: int                 # image is n_side x n_side
    fov_deg: float
    n_epochs: int
    wavelengths: tuple          # one per channel (metres)
    n_sources: int
    flux_range: tuple           # (lo, hi); log-uniform unless cfg 1 (uniform)
    noise: float                # sigma_n^2 added as noise * I before beamforming
    h_span_hours: float
    latitude_deg: float
    beamformed: bool = False

    @property
    def n_pix(self) -> int:
        return self.n_side * self.n_side

    @property
    def n_chan(self) -> int:
        return len(self.wavelengths)

    @property
    def n_collects(self) -> int:
        return self.n_epochs * self.n_chan

    @property
    def terms_per_collect(self) -> int:
        return self.n_ant * self.n_eig * self.n_pix

    @property
    def total_terms(self) -> int:
        return self.terms_per_collect * self.n_collects


CONFIGS = {
    1: Config(1, "tiny", 16, 16, 8, 2, 32, 10.0, 1, (2.0,), 3, (1.0, 5.0), 0.1, 0.0, 90.0),
    2: Config(2, "lofar_like", 1776, 37, 12, 4, 256, 20.0, 60, (5.0,), 20, (0.1, 10.0), 0.0, 8.0, 52.9,
              beamformed=True),
    3: Config(3, "ska_low_like", 512, 512, 32, 4, 512, 15.0, 100, (3.0,), 50, (0.01, 10.0), 0.5, 6.0, -26.8),
    4: Config(4, "ska_low_wide", 512, 512, 64, 8, 1024, 30.0, 20, (2.5,), 200, (0.01, 10.0), 0.5, 6.0, -26.8),
    5: Config(5, "ska_low_multichannel", 512, 512, 64, 8, 2048, 40.0, 50,
              tuple(299.792458 / (100.0 + c) for c in range(16)), 200, (0.01, 10.0), 0.5, 6.0, -26.8),
}


# ------------------------------------------------------------------------------------ geometry
def _disk_points(rng, n, radius, min_sep, existing=None):
    """n points uniform in a disk with pairwise separation >= min_sep (sequential rejection)."""
    pts = [] if existing is None else list(existing)
    n0 = len(pts)
    while len(pts) - n0 < n:
        r = radius * np.sqrt(rng.random())
        a = 2.0 * np.pi * rng.random()
        p = np.array([r * np.cos(a), r * np.sin(a)])
        if all(np.hypot(*(p - q)) >= min_sep for q in pts):
            pts.append(p)
    return np.array(pts[n0:])


def _enu_to_equatorial(enu, lat_rad):
    e, n, u = enu[:, 0], enu[:, 1], enu[:, 2]
    x = -np.sin(lat_rad) * n + np.cos(lat_rad) * u
    y = e
    z = np.cos(lat_rad) * n + np.sin(lat_rad) * u
    return np.stack([x, y, z], axis=1)


def _rot_z(h):
    c, s = np.cos(h), np.sin(h)
    return np.array([[c, -s, 0.0], [s, c, 0.0], [0.0, 0.0, 1.0]])


def _layout_tiny(rng):
    xy = _disk_points(rng, 16, 100.0, 5.0)                      # 200 m diameter
    z = rng.normal(0.0, 1.0, size=16)
    return np.column_stack([xy, z])


def _layout_lofar(rng):
    centres = []
    while len(centres) < 37:
        p = rng.normal(0.0, 2000.0, size=2)
        if all(np.hypot(*(p - q)) >= 100.0 for q in centres):
            centres.append(p)
    centres = np.array(centres)
    up = rng.normal(0.0, 1.0, size=37)
    enu = np.zeros((37 * 48, 3))
    for s in range(37):
        d = _disk_points(rng, 48, 20.0, 2.5)
        enu[s * 48:(s + 1) * 48, :2] = centres[s] + d
        enu[s * 48:(s + 1) * 48, 2] = up[s]
    return enu


def _layout_ska(rng):
    core = _disk_points(rng, 224, 1000.0, 35.0)
    arms = []
    radii = 1100.0 * (35000.0 / 1100.0) ** (np.arange(96) / 95.0)
    for k in range(3):
        az = 2.0 * np.pi * k / 3.0 + np.log(radii / 1000.0)
        xy = np.column_stack([radii * np.cos(az), radii * np.sin(az)]) + rng.normal(0.0, 20.0, size=(96, 2))
        arms.append(xy)
    xy = np.vstack([core] + arms)
    u = rng.normal(0.0, 5.0, size=512) - (xy[:, 0] ** 2 + xy[:, 1] ** 2) / (2.0 * 6371000.0)
    return np.column_stack([xy, u])


@dataclass
class Workload:
    cfg: Config
    enu: np.ndarray                      # (n_ant, 3) local East-North-Up metres
    xyz0: np.ndarray                     # (n_ant, 3) sky-frame positions at hour angle 0
    r_c: np.ndarray                      # field centre unit vector
    e_l: np.ndarray
    e_m: np.ndarray
    src_dir: np.ndarray                  # (n_sources, 3) unit vectors
    src_lm: np.ndarray                   # (n_sources, 2)
    src_flux: np.ndarray                 # (n_sources,)
    src_pixel: np.ndarray | None = None  # cfg 1: pixel index of each source
    _pix: np.ndarray | None = field(default=None, repr=False)

    # -------------------------------------------------------------------------- pixel grid
    @property
    def pix_step(self) -> float:
        return 2.0 * np.sin(np.radians(self.cfg.fov_deg) / 2.0) / self.cfg.n_side

    def lm_grid(self):
        n = self.cfg.n_side
        return (np.arange(n) - n // 2) * self.pix_step

    def pixels(self, index=None) -> np.ndarray:
        """Pixel unit vectors, (n_pix, 3) float64 Fortran order; j = a + n_side * b."""
        if self._pix is None:
            g = self.lm_grid()
            l = np.tile(g, self.cfg.n_side)
            m = np.repeat(g, self.cfg.n_side)
            n = np.sqrt(1.0 - l * l - m * m)
            pix = l[:, None] * self.e_l + m[:, None] * self.e_m + n[:, None] * self.r_c
            self._pix = np.asfortranarray(pix)
        if index is None:
            return self._pix
        return np.asfortranarray(self._pix[np.asarray(index)])

    # -------------------------------------------------------------------------- per collect
    def hour_angle(self, t: int) -> float:
        c = self.cfg
        return (-0.5 + (t + 0.5) / c.n_epochs) * np.radians(15.0 * c.h_span_hours)

    def xyz(self, t: int) -> np.ndarray:
        if self.cfg.idx == 1:
            return np.asfortranarray(self.xyz0)
        return np.asfortranarray(self.xyz0 @ _rot_z(self.hour_angle(t)).T)

    def beam_weights(self, xyz: np.ndarray, wavelength: float):
        """cfg 2: W (n_ant, n_beam) complex64, block diagonal, unit modulus, phased at r_c."""
        if not self.cfg.beamformed:
            return None
        W = np.zeros((self.cfg.n_ant, self.cfg.n_beam), dtype=np.complex128)
        for s in range(self.cfg.n_beam):
            blk = slice(s * 48, (s + 1) * 48)
            c_s = xyz[blk].mean(axis=0)
            W[blk, s] = np.exp(2j * np.pi * ((xyz[blk] - c_s) @ self.r_c) / wavelength)
        return np.asfortranarray(W.astype(np.complex64))

    def collect_inputs(self, n: int) -> dict:
        """Inputs of collect number n (n = t * n_chan + c): dict(S, W, xyz, wavelength)."""
        c = self.cfg
        t, ch = divmod(n, c.n_chan)
        wl = float(c.wavelengths[ch])
        xyz = self.xyz(t)
        W = self.beam_weights(xyz, wl)
        A = np.exp(2j * np.pi * (xyz @ self.src_dir.T) / wl)            # a_i(r_q), Eq. 3
        if W is not None:
            W128 = W.astype(np.complex128)
            A = W128.conj().T @ A                                        # Phi^* = W^H Psi^*, Eq. 23
            S = (A * self.src_flux) @ A.conj().T
            if c.noise:
                S = S + c.noise * (W128.conj().T @ W128)
        else:
            S = (A * self.src_flux) @ A.conj().T + c.noise * np.eye(c.n_ant)
        S = 0.5 * (S + S.conj().T)
        return dict(S=np.asfortranarray(S.astype(np.complex64)), W=W, xyz=xyz, wavelength=wl)

    def mid_collect(self) -> int:
        return (self.cfg.n_epochs // 2) * self.cfg.n_chan

    def sample_pixels(self, stride: int = 16, full_tiles: bool = False) -> np.ndarray:
        """Deterministic pixel subset: every stride-th row and column + pixel nearest each of the
        10 brightest sources (pixels are independent, so a subset image is exact for them).
        full_tiles: also 1024 CONSECUTIVE pixels from a 256-aligned index near the image centre and the last 256
        pixels of the image. A strided grid only ever lands on pixel indices that are multiples of the stride; a
        kernel that maps consecutive pixels to the threads (lanes) of a tile is then compared on a few lanes only."""
        n = self.cfg.n_side
        rows = np.arange(0, n, stride)
        idx = (rows[None, :] + n * rows[:, None]).ravel()
        if full_tiles:
            start = ((n * n // 2 + n // 3) // 256) * 256
            idx = np.concatenate([idx, np.arange(start, min(start + 1024, n * n)), np.arange(max(n * n - 256, 0), n * n)])
        g0 = -(n // 2) * self.pix_step
        bright = np.argsort(self.src_flux)[::-1][:10]
        a = np.clip(np.rint((self.src_lm[bright, 0] - g0) / self.pix_step), 0, n - 1).astype(np.int64)
        b = np.clip(np.rint((self.src_lm[bright, 1] - g0) / self.pix_step), 0, n - 1).astype(np.int64)
        return np.unique(np.concatenate([idx, a + n * b]))


def make_workload(idx: int) -> Workload:
    cfg = CONFIGS[idx]
    seed = BASE_SEED + idx
    if idx == 1:
        rng = np.random.default_rng(seed)
        enu = _layout_tiny(rng)
        xyz0 = enu.copy()
        r_c, e_l, e_m = np.array([0.0, 0.0, 1.0]), np.array([1.0, 0.0, 0.0]), np.array([0.0, 1.0, 0.0])
    else:
        if idx == 2:
            rng = np.random.default_rng(seed)
            enu = _layout_lofar(rng)
        else:
            lay_rng = np.random.default_rng(BASE_SEED + 3)      # cfgs 3-5 share the cfg-3 layout stream
            enu = _layout_ska(lay_rng)
            rng = lay_rng if idx == 3 else np.random.default_rng(seed)
        lat = np.radians(cfg.latitude_deg)
        xyz0 = _enu_to_equatorial(enu, lat)
        r_c = np.array([np.cos(lat), 0.0, np.sin(lat)])
        e_l = np.array([0.0, 1.0, 0.0])
        e_m = np.array([-np.sin(lat), 0.0, np.cos(lat)])

    wl = Workload(cfg, enu, xyz0, r_c, e_l, e_m, None, None, None)
    if idx == 1:
        g = wl.lm_grid()
        n = cfg.n_side
        cells = rng.choice(24 * 24, size=cfg.n_sources, replace=False)      # distinct pixel centres
        a = n // 2 - 12 + cells % 24
        b = n // 2 - 12 + cells // 24
        lm = np.column_stack([g[a], g[b]])
        flux = rng.uniform(*cfg.flux_range, size=cfg.n_sources)
        wl.src_pixel = a + n * b
    else:
        half = 0.9 * np.sin(np.radians(cfg.fov_deg) / 2.0)
        lm = rng.uniform(-half, half, size=(cfg.n_sources, 2))
        lo, hi = cfg.flux_range
        flux = np.exp(rng.uniform(np.log(lo), np.log(hi), size=cfg.n_sources))
    nn = np.sqrt(1.0 - np.sum(lm * lm, axis=1))
    wl.src_lm = lm
    wl.src_flux = flux
    wl.src_dir = lm[:, :1] * e_l + lm[:, 1:] * e_m + nn[:, None] * r_c
    return wl


# ------------------------------------------------------------------------------ level edges
def choose_intervals(mu_desc, n_levels: int, lam_max=None, lam_min=None) -> np.ndarray:
    """Deterministic level edges from a list of eigenvalues (obtained by the caller).

    mu_desc: the N_eig selected eigenvalues of the reference collect, sorted descending. Interior
    edge q (q = 1..L-1) is the geometric mean across the widest log-gap among the rank boundaries
    within +-w of q*N/L, w = clamp(N/(2L), 1, 3); the outer edges are 2 x lam_max and lam_min / 2.
    Returns (L, 2) float64 [min, max]; level 0 is the highest-energy level.
    """
    mu = np.asarray(mu_desc, dtype=np.float64)
    n = mu.size
    assert n >= n_levels >= 1 and np.all(np.diff(mu) <= 0) and mu[-1] > 0
    lam_max = float(mu[0]) if lam_max is None else float(lam_max)
    lam_min = float(mu[-1]) if lam_min is None else float(lam_min)
    w = int(min(3, max(1, n // (2 * n_levels))))
    edges = []
    prev_rank = 0
    for q in range(1, n_levels):
        centre = (q * n) // n_levels
        lo_r = max(prev_rank + 1, centre - w, 1)
        hi_r = max(lo_r, min(centre + w, n - 1 - (n_levels - 1 - q)))
        ranks = np.arange(lo_r, hi_r + 1)                   # boundary r sits between mu[r-1], mu[r]
        gaps = np.log(mu[ranks - 1] / mu[ranks])
        r = int(ranks[int(np.argmax(gaps))])
        edges.append(float(np.sqrt(mu[r - 1] * mu[r])))
        prev_rank = r
    bounds = [2.0 * lam_max] + edges + [0.5 * lam_min]
    return np.array([[bounds[l + 1], bounds[l]] for l in range(n_levels)], dtype=np.float64)
