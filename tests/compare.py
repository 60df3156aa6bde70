"""Hit-list comparator: CUDA path vs oracle, with the exemption protocol of DESIGN.md §3.4.

Integer outputs must be bit-exact except at pixels the ORACLE flags as fragile (an fp64 value
within 1e-4 ADU of a deciding comparison, BASELINE.json north_star); those are matched leniently
and counted per class.  Floats must satisfy |g - o| <= 1e-4 + 1e-4*|o|; the count failing the
stricter absolute-only reading is reported too.

Lenient matching is BOUNDED: a hit present on both sides may differ
  * in n by +-1 only when the oracle flags F4 on it or F1 in its window (E itself may have moved);
  * in E, dx, dy beyond the float tolerance only when a segment of its 3x3 window is F1-flagged (one
    mask pixel may flip, moving that segment's c), and then by at most 9*T_cm/#M in E (#M = the
    smallest number of segmented pixels among the window's segments, from the oracle) and 0.02 px in
    dx, dy.
Anything larger is a failure even on a flagged pixel.
"""
from __future__ import annotations

from dataclasses import dataclass, field

import numpy as np

F1, F2, F3, F4 = 1, 2, 4, 8
ATOL = 1e-4
RTOL = 1e-4


@dataclass
class Report:
    frames: int = 0
    hits_oracle: int = 0
    hits_gpu: int = 0
    matched: int = 0
    exempt: dict = field(default_factory=lambda: {"F1": 0, "F2": 0, "F3": 0, "F4": 0})
    exempt_hits: int = 0
    failures: list = field(default_factory=list)
    strict_abs_fail: int = 0
    max_err: dict = field(default_factory=lambda: {"E": 0.0, "dx": 0.0, "dy": 0.0})

    @property
    def ok(self) -> bool:
        return not self.failures

    def summary(self) -> str:
        return (f"frames={self.frames} hits(oracle/gpu)={self.hits_oracle}/{self.hits_gpu} matched={self.matched} "
                f"exempt_hits={self.exempt_hits} {self.exempt} failures={len(self.failures)} "
                f"strict_abs_fail={self.strict_abs_fail} max_err={self.max_err}")


def _window_flags(frag, idx, P, H, W):
    """OR of the pixel's own F2|F3|F4 flags and F1 of every in-panel pixel of its 3x3 window."""
    idx = np.asarray(idx, np.int64)
    c = idx % W
    r = (idx // W) % H
    p = idx // (W * H)
    out = frag[idx] & (F2 | F3 | F4)
    for dr in (-1, 0, 1):
        for dc in (-1, 0, 1):
            rr, cc = r + dr, c + dc
            ok = (rr >= 0) & (rr < H) & (cc >= 0) & (cc < W)
            q = (p * H + np.clip(rr, 0, H - 1)) * W + np.clip(cc, 0, W - 1)
            out = out | np.where(ok, frag[q] & (F1 | F3), 0).astype(frag.dtype)
    return out


def _window_min_count(cm_count, idx, P, H, W, S):
    """Smallest #M among the row segments touched by the in-panel 3x3 window of each pixel."""
    idx = np.asarray(idx, np.int64)
    c = idx % W
    r = (idx // W) % H
    p = idx // (W * H)
    nseg = W // S
    out = np.full(idx.shape, np.iinfo(np.int64).max, np.int64)
    for dr in (-1, 0, 1):
        for dc in (-1, 0, 1):
            rr, cc = r + dr, c + dc
            ok = (rr >= 0) & (rr < H) & (cc >= 0) & (cc < W)
            q = (p * H + np.clip(rr, 0, H - 1)) * nseg + np.clip(cc, 0, W - 1) // S
            out = np.where(ok, np.minimum(out, cm_count[q]), out)
    return out


LENIENT_DXY = 0.02      # px, SURVEY.md §8(c)


def compare(oracle_res, gpu, *, panels, rows, cols, frames=None, check_accum=True, seg_cols=None,
            cm_adu=20.0) -> Report:
    """gpu: dict of numpy arrays hit_count[n], hit_pixel[n,cap], hit_charge, hit_nphot, hit_dx, hit_dy,
    frame_photons[n], accum[npix].  oracle_res: oracle.pdp_oracle.OracleResult with fragile flags.
    frames: optional list mapping oracle frame i -> gpu frame index."""
    rep = Report()
    n = len(oracle_res.hit_count)
    cap = gpu["hit_pixel"].shape[1]
    frames = list(range(n)) if frames is None else list(frames)
    any_exempt = False
    for i in range(n):
        gf = frames[i]
        rep.frames += 1
        frag = oracle_res.fragile[i]
        oi = oracle_res.hit_pixel[i].astype(np.int64)
        gcount = int(gpu["hit_count"][gf])
        k = min(gcount, cap)
        gi = gpu["hit_pixel"][gf, :k].astype(np.int64) & 0xFFFFFFFF
        rep.hits_oracle += len(oi)
        rep.hits_gpu += gcount
        if k > 1 and not np.all(np.diff(gi) > 0):
            rep.failures.append((gf, "gpu list not strictly increasing"))
            continue
        gn = gpu["hit_nphot"][gf, :k]
        if gcount <= cap and int(gpu["frame_photons"][gf]) != int(gn.astype(np.int64).sum()):
            rep.failures.append((gf, "frame_photons != sum of listed n"))
        common, io, ig = np.intersect1d(oi, gi, return_indices=True)
        only_o = np.setdiff1d(oi, gi)
        only_g = np.setdiff1d(gi, oi)
        for name, arr in (("only_oracle", only_o), ("only_gpu", only_g)):
            if len(arr):
                fl = _window_flags(frag, arr, panels, rows, cols)
                for px, f in zip(arr, fl):
                    if f == 0:
                        rep.failures.append((gf, name, int(px)))
                    else:
                        any_exempt = True
                        rep.exempt_hits += 1
                        for b, nm in ((F1, "F1"), (F2, "F2"), (F3, "F3"), (F4, "F4")):
                            rep.exempt[nm] += 1 if f & b else 0
        if len(common):
            oE = oracle_res.hit_charge[i][io]; gE = gpu["hit_charge"][gf, ig].astype(np.float64)
            ox = oracle_res.hit_dx[i][io]; gx = gpu["hit_dx"][gf, ig].astype(np.float64)
            oy = oracle_res.hit_dy[i][io]; gy = gpu["hit_dy"][gf, ig].astype(np.float64)
            on = oracle_res.hit_nphot[i][io]; gnn = gn[ig]
            bad_n = on != gnn
            eE, ex, ey = np.abs(gE - oE), np.abs(gx - ox), np.abs(gy - oy)
            # float32 storage of the result adds half an ulp of the stored value
            ulpE = np.abs(oE) * 2.0 ** -24
            bad_f = (eE > ATOL + RTOL * np.abs(oE) + ulpE) | (ex > ATOL + RTOL * np.abs(ox)) | (ey > ATOL + RTOL * np.abs(oy))
            rep.strict_abs_fail += int(((eE > ATOL + ulpE) | (ex > ATOL) | (ey > ATOL)).sum())
            rep.max_err["E"] = max(rep.max_err["E"], float(eE.max()))
            rep.max_err["dx"] = max(rep.max_err["dx"], float(ex.max()))
            rep.max_err["dy"] = max(rep.max_err["dy"], float(ey.max()))
            bad = bad_n | bad_f
            rep.matched += int((~bad).sum())
            if bad.any():
                fl = _window_flags(frag, common[bad], panels, rows, cols)
                if seg_cols and oracle_res.cm_count is not None:
                    m = np.maximum(1, _window_min_count(oracle_res.cm_count[i], common[bad], panels, rows, cols, seg_cols))
                    boundE = 9.0 * float(cm_adu) / m
                else:                               # no segment information: the loosest bound, one whole T_cm per pixel
                    boundE = np.full(int(bad.sum()), 9.0 * float(cm_adu))
                for px, f, bn, dn, bf, dE, dX, dY, oe, bE in zip(
                        common[bad], fl, bad_n[bad], (on.astype(np.int64) - gnn)[bad], bad_f[bad], eE[bad], ex[bad],
                        ey[bad], oE[bad], boundE):
                    ok_n = (not bn) or (abs(int(dn)) <= 1 and (f & (F1 | F4)) != 0)
                    ok_f = (not bf) or ((f & F1) != 0 and dE <= bE + ATOL + RTOL * abs(oe)
                                        and dX <= LENIENT_DXY and dY <= LENIENT_DXY)
                    lenient = f != 0 and ok_n and ok_f
                    if not lenient:
                        rep.failures.append((gf, "mismatch", int(px)))
                    else:
                        any_exempt = True
                        rep.exempt_hits += 1
                        for b, nm in ((F1, "F1"), (F2, "F2"), (F3, "F3"), (F4, "F4")):
                            rep.exempt[nm] += 1 if f & b else 0
        if len(only_o) == 0 and len(only_g) == 0 and gcount != len(oi):
            rep.failures.append((gf, "hit_count differs", gcount, len(oi)))
    if check_accum and frames == list(range(len(gpu["hit_count"]))):
        acc = np.zeros_like(gpu["accum"], dtype=np.int64)
        for f in range(n):
            k = min(int(gpu["hit_count"][f]), cap)
            np.add.at(acc, gpu["hit_pixel"][f, :k].astype(np.int64) & 0xFFFFFFFF, gpu["hit_nphot"][f, :k].astype(np.int64))
        if np.all(gpu["hit_count"] <= cap) and not np.array_equal(acc, gpu["accum"].astype(np.int64) & 0xFFFFFFFF):
            rep.failures.append((-1, "accum != scatter of gpu hit lists"))
        if not any_exempt and not np.array_equal(gpu["accum"].astype(np.int64) & 0xFFFFFFFF, oracle_res.accum.astype(np.int64)):
            rep.failures.append((-1, "accum != oracle accum"))
    return rep
