"""Seeded synthetic inputs for the matched-filter trajectory search.

Stand-ins for TESS residual stacks (the paper's Sector 18/19/5 full-frame images are not
available offline).  Shapes follow the paper: 2048x2048 CCDs, 1000-3888 frames
per 27-day sector (L33, L152), 256x256 cutouts (L130), sigma-unit residuals after background
subtraction and clipping (L106).  The five configurations are those of BASELINE.json:configs;
the recipe is SURVEY.md section 8(d) and is restated in DESIGN.md.

This module is the ONLY code shared by the CPU oracle (``oracle/``) and the CUDA path
(``paper_2209_09848_b200/``).  It holds no arithmetic of the method itself: no PRF, no
trajectory rounding, no filter weights, no scores.  Injected sources are returned as
*parameters* (trajectory index, start pixel, amplitude); rendering them into the frames is
done by the caller with ``oracle.inject`` (tests) or ``tno_mf_inject`` (CUDA library).

Seeds: ``seed_c = 220909848 + c`` for config c = 1..5.  Small parameters come from
``numpy.random.default_rng(seed_c)`` in the order sigma_t, outlier positions, hot-pixel
positions, sources.  Pixel noise comes from a per-frame generator seeded ``(seed_c, t)`` so any
frame can be regenerated alone.
"""
from __future__ import annotations

import dataclasses
import math
from typing import Optional

import numpy as np

SEED_BASE = 220909848


@dataclasses.dataclass(frozen=True)
class Config:
    """One entry of BASELINE.json:configs (index = position + 1)."""
    idx: int
    name: str
    T: int
    H: int
    W: int
    t0: float
    prf_sigma: float
    grid_n: int                 # velocity grid is grid_n x grid_n
    v_max: float                # vx, vy in linspace(-v_max, v_max, grid_n)
    accels: tuple               # tuple of (ax, ay); trajectories are acceleration-major
    n_sources: int
    amp_lo: float
    amp_hi: float
    outlier_frac: float         # fixed positions, fresh Laplace(0, outlier_scale) draw per frame
    outlier_scale: float
    hot_frac: float             # fixed positions, constant +hot_value in every frame
    hot_value: float
    sigma_drift: float          # sigma_t *= 1 + sigma_drift * sin(2 pi t / drift_period)
    drift_period: float
    topk: int
    threshold: float
    want_maps: bool

    @property
    def seed(self) -> int:
        return SEED_BASE + self.idx

    @property
    def n_traj(self) -> int:
        return self.grid_n * self.grid_n * len(self.accels)

    @property
    def evals(self) -> int:
        """trajectory x frame x pixel evaluations of one search."""
        return self.n_traj * self.T * self.H * self.W


CONFIGS = {
    1: Config(1, "tiny", 16, 64, 64, 0.0, 1.0, 3, 0.1, ((0.0, 0.0),), 2, 3.0, 3.0,
              0.0, 5.0, 0.0, 50.0, 0.0, 1000.0, 5, 5.0, True),
    2: Config(2, "cutout", 100, 256, 256, 50.0, 1.0, 5, 0.2, ((0.0, 0.0),), 10, 0.5, 3.0,
              0.005, 5.0, 0.0, 50.0, 0.0, 1000.0, 20, 5.0, True),
    3: Config(3, "headline", 1000, 2048, 2048, 500.0, 1.0, 10, 0.05, ((0.0, 0.0),), 50, 0.3, 2.0,
              0.005, 5.0, 0.0001, 50.0, 0.0, 1000.0, 100, 5.0, True),
    4: Config(4, "long", 3888, 2048, 2048, 1944.0, 1.0, 8, 0.015, ((0.0, 0.0),), 30, 0.2, 1.5,
              0.005, 5.0, 0.0, 50.0, 0.2, 1000.0, 100, 5.0, True),
    5: Config(5, "curved", 1000, 2048, 2048, 500.0, 1.2, 16, 0.05,
              ((0.0, 0.0), (2e-5, 0.0), (-2e-5, 0.0), (0.0, 2e-5)), 200, 0.3, 2.0,
              0.005, 5.0, 0.0001, 50.0, 0.0, 1000.0, 100, 5.0, False),
}


def scaled(cfg: Config, *, T: Optional[int] = None, H: Optional[int] = None,
           W: Optional[int] = None, **kw) -> Config:
    """A reduced copy of a config (same recipe, smaller stack); t0 stays at the same
    relative epoch (0 stays 0, T/2 stays T/2)."""
    T2 = cfg.T if T is None else T
    t0 = 0.0 if cfg.t0 == 0.0 else float(T2 // 2)
    return dataclasses.replace(cfg, T=T2, H=cfg.H if H is None else H,
                               W=cfg.W if W is None else W, t0=t0, **kw)


def trajectories(cfg: Config) -> np.ndarray:
    """float32 [n_traj, 4] rows (vx, vy, ax, ay) in px/frame and px/frame^2.
    Index k = ia * n*n + iy * n + ix (acceleration-major, then vy, then vx)."""
    v = np.linspace(-cfg.v_max, cfg.v_max, cfg.grid_n)
    out = np.empty((cfg.n_traj, 4), dtype=np.float32)
    k = 0
    for (ax, ay) in cfg.accels:
        for iy in range(cfg.grid_n):
            for ix in range(cfg.grid_n):
                out[k] = (v[ix], v[iy], ax, ay)
                k += 1
    return out


@dataclasses.dataclass
class Params:
    """Everything about a stack except its pixel noise."""
    cfg: Config
    sigma_t: np.ndarray          # float32 [T]
    traj: np.ndarray             # float32 [n_traj, 4]
    outlier_pos: np.ndarray      # int64 [n_out] flat pixel index y*W+x, sorted
    hot_pos: np.ndarray          # int64 [n_hot]
    src_k: np.ndarray            # int32 [n_src] trajectory index of each injected source
    src_x: np.ndarray            # int32 [n_src] start pixel at the reference epoch t0
    src_y: np.ndarray            # int32 [n_src]
    src_amp: np.ndarray          # float32 [n_src] amplitude in absolute flux units


def _track_margin(cfg: Config, traj_row: np.ndarray, keep: int) -> int:
    """Conservative bound (px) on how far a track wanders from its start pixel, plus `keep`."""
    dt = max(abs(0.0 - cfg.t0), abs((cfg.T - 1) - cfg.t0))
    reach = max(abs(float(traj_row[0])) * dt + abs(float(traj_row[2])) * dt * dt,
                abs(float(traj_row[1])) * dt + abs(float(traj_row[3])) * dt * dt)
    return int(math.ceil(reach)) + keep


def make_params(cfg: Config) -> Params:
    rng = np.random.default_rng(cfg.seed)
    sigma = rng.uniform(0.8, 1.2, size=cfg.T)
    if cfg.sigma_drift != 0.0:
        t = np.arange(cfg.T, dtype=np.float64)
        sigma = sigma * (1.0 + cfg.sigma_drift * np.sin(2.0 * np.pi * t / cfg.drift_period))
    sigma_t = sigma.astype(np.float32)
    npx = cfg.H * cfg.W
    n_out = int(round(cfg.outlier_frac * npx))
    outlier_pos = np.sort(rng.choice(npx, size=n_out, replace=False)) if n_out else \
        np.zeros(0, dtype=np.int64)
    n_hot = int(round(cfg.hot_frac * npx))
    hot_pos = np.sort(rng.choice(npx, size=n_hot, replace=False)) if n_hot else \
        np.zeros(0, dtype=np.int64)
    traj = trajectories(cfg)
    # sources: distinct trajectories when there are few of them (config 1), random otherwise
    if cfg.n_sources <= 2:
        src_k = rng.choice(cfg.n_traj, size=cfg.n_sources, replace=False)
    else:
        src_k = rng.integers(0, cfg.n_traj, size=cfg.n_sources)
    keep = 4
    sx = np.empty(cfg.n_sources, dtype=np.int32)
    sy = np.empty(cfg.n_sources, dtype=np.int32)
    for i, k in enumerate(src_k):
        m = _track_margin(cfg, traj[k], keep)
        m = min(m, (min(cfg.H, cfg.W) - 1) // 2)
        sx[i] = rng.integers(m, cfg.W - m)
        sy[i] = rng.integers(m, cfg.H - m)
    amp = rng.uniform(cfg.amp_lo, cfg.amp_hi, size=cfg.n_sources).astype(np.float32)
    return Params(cfg, sigma_t, traj, outlier_pos.astype(np.int64), hot_pos.astype(np.int64),
                  src_k.astype(np.int32), sx, sy, amp)


def frame_numpy(p: Params, t: int) -> np.ndarray:
    """float32 [H, W] residual frame t WITHOUT injected sources (numpy generator)."""
    cfg = p.cfg
    rng = np.random.default_rng([cfg.seed, t])
    f = rng.standard_normal((cfg.H, cfg.W)) * float(p.sigma_t[t])
    if p.outlier_pos.size:
        f.reshape(-1)[p.outlier_pos] += rng.laplace(0.0, cfg.outlier_scale, size=p.outlier_pos.size)
    if p.hot_pos.size:
        f.reshape(-1)[p.hot_pos] += cfg.hot_value
    return f.astype(np.float32)


def stack_numpy(p: Params) -> np.ndarray:
    """float32 [T, H, W] without injected sources; for configs the oracle finishes in seconds."""
    return np.stack([frame_numpy(p, t) for t in range(p.cfg.T)], axis=0)


def stack_torch(p: Params, device, chunk: int = 16):
    """float32 [T, H, W] torch tensor generated ON `device` (no host copy of the stack), without
    injected sources.  Values differ from ``stack_numpy`` (different generator) but follow the
    same recipe; they are consistent within a process for a given (seed, t)."""
    import torch
    cfg = p.cfg
    out = torch.empty((cfg.T, cfg.H, cfg.W), dtype=torch.float32, device=device)
    sig = torch.from_numpy(p.sigma_t.astype(np.float32)).to(device)
    opos = torch.from_numpy(p.outlier_pos).to(device) if p.outlier_pos.size else None
    hpos = torch.from_numpy(p.hot_pos).to(device) if p.hot_pos.size else None
    gen = torch.Generator(device=device)
    for t in range(cfg.T):
        gen.manual_seed((cfg.seed << 20) + t)
        f = out[t]
        f.normal_(0.0, 1.0, generator=gen)
        f.mul_(sig[t])
        flat = f.view(-1)
        if opos is not None:
            u = torch.rand(opos.numel(), device=device, generator=gen, dtype=torch.float32)
            u = u.clamp_(1e-7, 1.0 - 1e-7) - 0.5
            lap = -cfg.outlier_scale * torch.sign(u) * torch.log1p(-2.0 * u.abs())
            flat.index_add_(0, opos, lap)
        if hpos is not None:
            flat.index_add_(0, hpos, torch.full((hpos.numel(),), cfg.hot_value, device=device))
    return out
