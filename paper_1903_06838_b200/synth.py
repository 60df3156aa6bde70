"""Seeded synthetic detector frames (input generator only — none of the method's arithmetic).

Serves both sides of the parity tests: the CUDA path and the oracle read the SAME
uint16 frames and float32 maps produced here.  Nothing in this module calibrates,
finds photons or touches a threshold; it is the forward model of DESIGN.md §4
(BASELINE.json `configs`): pedestal + gain * (photon charge clouds + per-segment
common-mode offset + read noise), rounded and clamped to uint16.

Randomness is counter based: every random number is a SplitMix64-style hash of
(seed, config id, purpose, frame, element), evaluated with wrapping int64 torch
ops, so any frame can be generated alone, in any order, on any torch device, and
the integer streams are identical on CPU and GPU (libm-level float differences can
still flip a rounding; parity never depends on that because both sides read the
same generated buffer).
"""
from __future__ import annotations

import math
from dataclasses import dataclass, replace

import torch

_MASK63 = (1 << 63) - 1


@dataclass(frozen=True)
class DetectorConfig:
    """One BASELINE.json workload (fields not restated there inherit config 0)."""
    name: str
    cfg_id: int
    n_frames: int
    panels: int
    rows: int
    cols: int
    seg_cols: int
    occupancy: float       # photons per pixel per frame (Poisson process), or P(pixel hit) if dense
    photon_adu: float      # E_ph
    cloud_sigma: float     # charge-cloud sigma in pixel pitches
    noise_sigma: float     # read noise, gain-corrected ADU
    cm_sigma: float        # per (frame, panel, row, segment) common-mode offset sigma
    dense_mean: float = 0.0  # >0: pixel hit with prob `occupancy`, k ~ Poisson(dense_mean) | k>=1
    seed_adu: float = 50.0
    cm_adu: float = 20.0
    ped_mean: float = 1000.0
    ped_sigma: float = 20.0
    gain_lo: float = 0.9
    gain_hi: float = 1.1
    seed: int = 0

    @property
    def npix(self) -> int:
        return self.panels * self.rows * self.cols

    @property
    def max_hits(self) -> int:
        return ((self.rows + 1) // 2) * ((self.cols + 1) // 2) * self.panels

    def scaled(self, n_frames: int) -> "DetectorConfig":
        return replace(self, n_frames=n_frames)


# BASELINE.json configs[0..4]; S for configs 3 and 4 is W/2 (reading R7).
CONFIGS = (
    DetectorConfig("tiny", 0, 100, 1, 185, 388, 194, 0.005, 100.0, 0.3, 3.0, 5.0),
    DetectorConfig("epix", 1, 2000, 1, 704, 768, 384, 0.01, 80.0, 0.4, 2.5, 5.0),
    DetectorConfig("cspad", 2, 500, 32, 185, 388, 194, 0.002, 120.0, 0.3, 4.0, 8.0),
    DetectorConfig("dense", 3, 500, 1, 1024, 1024, 512, 0.10, 100.0, 0.6, 3.0, 5.0, dense_mean=1.5),
    DetectorConfig("lcls2", 4, 4000, 16, 512, 512, 256, 0.005, 100.0, 0.3, 3.0, 5.0),
)


def _lsr(x: torch.Tensor, s: int) -> torch.Tensor:
    """Logical shift right of an int64 tensor."""
    return (x >> s) & ((1 << (64 - s)) - 1)


def _to_i64(v: int) -> int:
    v &= (1 << 64) - 1
    return v - (1 << 64) if v >= (1 << 63) else v


_C1 = _to_i64(0xBF58476D1CE4E5B9)
_C2 = _to_i64(0x94D049BB133111EB)
_GOLD = _to_i64(0x9E3779B97F4A7C15)


def _mix(x: torch.Tensor) -> torch.Tensor:
    x = (x ^ _lsr(x, 30)) * _C1
    x = (x ^ _lsr(x, 27)) * _C2
    return x ^ _lsr(x, 31)


def _key(cfg: DetectorConfig, purpose: int, frame: int) -> int:
    k = (cfg.seed * 0x100000001B3 + cfg.cfg_id * 1315423911 + purpose * 2654435761 + frame * 0x9E3779B1) \
        & ((1 << 64) - 1)
    # one scalar SplitMix round in Python ints
    k = (k + 0x9E3779B97F4A7C15) & ((1 << 64) - 1)
    k = ((k ^ (k >> 30)) * 0xBF58476D1CE4E5B9) & ((1 << 64) - 1)
    k = ((k ^ (k >> 27)) * 0x94D049BB133111EB) & ((1 << 64) - 1)
    return _to_i64(k ^ (k >> 31))


def _uniform(key: int, counter: torch.Tensor, stream: int) -> torch.Tensor:
    """float64 uniform in (0, 1), one per counter element."""
    x = _mix((counter * 4 + stream) * _GOLD + key)
    return (_lsr(x, 11).to(torch.float64) + 0.5) * (1.0 / 9007199254740992.0)


def _normal(key: int, counter: torch.Tensor) -> torch.Tensor:
    u1 = _uniform(key, counter, 0)
    u2 = _uniform(key, counter, 1)
    return torch.sqrt(-2.0 * torch.log(u1)) * torch.cos((2.0 * math.pi) * u2)


def make_maps(cfg: DetectorConfig, device="cpu"):
    """pedestal ~ N(ped_mean, ped_sigma), gain ~ U(gain_lo, gain_hi); float32 [P, H, W]."""
    idx = torch.arange(cfg.npix, dtype=torch.int64, device=device)
    ped = cfg.ped_mean + cfg.ped_sigma * _normal(_key(cfg, 0, 0), idx)
    gain = cfg.gain_lo + (cfg.gain_hi - cfg.gain_lo) * _uniform(_key(cfg, 0, 1), idx, 2)
    shape = (cfg.panels, cfg.rows, cfg.cols)
    return ped.to(torch.float32).reshape(shape), gain.to(torch.float32).reshape(shape)


def _photon_counts(cfg: DetectorConfig, u: torch.Tensor, u2: torch.Tensor) -> torch.Tensor:
    """Photons landing in each pixel: Poisson(occupancy) by CDF inversion, or the dense rule."""
    if cfg.dense_mean > 0.0:
        lam = cfg.dense_mean
        norm = 1.0 - math.exp(-lam)
        k = torch.ones_like(u, dtype=torch.int64)
        cdf, term = 0.0, math.exp(-lam)
        for j in range(1, 16):
            term = term * lam / j
            cdf += term / norm
            k = k + (u2 > cdf).to(torch.int64)
        return torch.where(u < cfg.occupancy, k, torch.zeros_like(k))
    lam = cfg.occupancy
    k = torch.zeros_like(u, dtype=torch.int64)
    term = math.exp(-lam)
    cdf = term
    for j in range(1, 12):
        k = k + (u > cdf).to(torch.int64)
        term = term * lam / j
        cdf += term
    return k


def _phi(z: torch.Tensor) -> torch.Tensor:
    return 0.5 * (1.0 + torch.special.erf(z * (1.0 / math.sqrt(2.0))))


def _keys(cfg: DetectorConfig, purpose: int, frames, device) -> torch.Tensor:
    """One key per frame as an int64 column [F, 1] (broadcasts against per-element counters)."""
    return torch.tensor([_key(cfg, purpose, f) for f in frames], dtype=torch.int64, device=device).reshape(-1, 1)


def _signal(cfg: DetectorConfig, frames, device) -> torch.Tensor:
    """Deposited photon charge of the given frames, gain-corrected ADU, float64 [F, P*H*W]."""
    P, H, W = cfg.panels, cfg.rows, cfg.cols
    F = len(frames)
    idx = torch.arange(cfg.npix, dtype=torch.int64, device=device)
    key = _keys(cfg, 3, frames, device)
    k = _photon_counts(cfg, _uniform(key, idx, 0), _uniform(key, idx, 1))      # [F, npix]
    sig = torch.zeros(F * cfg.npix, dtype=torch.float64, device=device)
    hit = torch.nonzero(k.reshape(-1) > 0).flatten()            # flat (frame, pixel), frame-major
    if hit.numel() == 0:
        return sig.reshape(F, cfg.npix)
    reps = k.reshape(-1)[hit]
    ph = torch.repeat_interleave(hit, reps)
    # ordinal of the photon inside its pixel
    start = torch.cumsum(reps, 0) - reps
    ordinal = torch.arange(ph.numel(), device=device) - torch.repeat_interleave(start, reps)
    ph_frame = ph // cfg.npix
    ph_pix = ph - ph_frame * cfg.npix
    ctr = ph_pix * 16 + ordinal
    pkey = _keys(cfg, 4, frames, device).flatten()[ph_frame]
    col = ph_pix % W
    row = (ph_pix // W) % H
    pan = ph_pix // (W * H)
    x0 = col.to(torch.float64) + _uniform(pkey, ctr, 0)   # pixel j covers [j, j+1)
    y0 = row.to(torch.float64) + _uniform(pkey, ctr, 1)
    s = cfg.cloud_sigma
    base = ph_frame * cfg.npix
    for dr in range(-3, 4):
        rr = row + dr
        wy = _phi((rr.to(torch.float64) + 1.0 - y0) / s) - _phi((rr.to(torch.float64) - y0) / s)
        okr = (rr >= 0) & (rr < H)
        for dc in range(-3, 4):
            cc = col + dc
            wx = _phi((cc.to(torch.float64) + 1.0 - x0) / s) - _phi((cc.to(torch.float64) - x0) / s)
            ok = okr & (cc >= 0) & (cc < W)          # charge falling off the panel is lost
            tgt = base + (pan * H + rr) * W + cc
            sig.index_put_((tgt[ok],), (cfg.photon_adu * wy * wx)[ok], accumulate=True)
    return sig.reshape(F, cfg.npix)


def _make_block(cfg: DetectorConfig, frames, ped: torch.Tensor, gain: torch.Tensor) -> torch.Tensor:
    """Raw frames `frames` (a list of frame numbers) as int32 values in [0, 65535]; shape [F, P, H, W]."""
    device = ped.device
    P, H, W, S = cfg.panels, cfg.rows, cfg.cols, cfg.seg_cols
    F = len(frames)
    idx = torch.arange(cfg.npix, dtype=torch.int64, device=device)
    noise = cfg.noise_sigma * _normal(_keys(cfg, 1, frames, device), idx)          # [F, npix]
    nseg = W // S
    sidx = torch.arange(P * H * nseg, dtype=torch.int64, device=device)
    cm = cfg.cm_sigma * _normal(_keys(cfg, 2, frames, device), sidx).reshape(F, P * H * nseg, 1)
    s = (_signal(cfg, frames, device) + noise).reshape(F, P * H * nseg, S) + cm
    raw = torch.round(ped.to(torch.float64).reshape(1, -1) + gain.to(torch.float64).reshape(1, -1) * s.reshape(F, -1))
    return raw.clamp_(0.0, 65535.0).to(torch.int32).reshape(F, P, H, W)   # round: half-to-even


def make_frame(cfg: DetectorConfig, frame: int, ped: torch.Tensor, gain: torch.Tensor) -> torch.Tensor:
    """One raw frame, uint16 stored as int32 tensor values in [0, 65535]; shape [P, H, W]."""
    return _make_block(cfg, [frame], ped, gain)[0]


def make_frames(cfg: DetectorConfig, first: int, count: int, ped: torch.Tensor, gain: torch.Tensor,
                out: torch.Tensor | None = None, block_pixels: int = 1 << 25) -> torch.Tensor:
    """raw[count, P, H, W] as torch.uint16 on ped.device (frames first .. first+count-1).  Frames are
    generated in blocks of ~block_pixels pixels (every frame depends only on its own number, so the
    block size never changes a value)."""
    if out is None:
        out = torch.empty((count, cfg.panels, cfg.rows, cfg.cols), dtype=torch.uint16, device=ped.device)
    B = max(1, block_pixels // cfg.npix)
    for i in range(0, count, B):
        m = min(B, count - i)
        out[i:i + m].copy_(_make_block(cfg, list(range(first + i, first + i + m)), ped, gain).to(torch.uint16))
    return out


def checksum(t: torch.Tensor) -> int:
    """FNV-1a-64 of the tensor's bytes (CPU; for logs only)."""
    data = t.detach().cpu().contiguous().view(torch.uint8).numpy().tobytes()
    h = 0xCBF29CE484222325
    for b in data:
        h = ((h ^ b) * 0x100000001B3) & ((1 << 64) - 1)
    return h
