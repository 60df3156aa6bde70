"""The comparator is part of the parity claim: these CPU tests feed it an oracle result and a copy of
it perturbed the way a wrong kernel would be, and check what it accepts."""
import copy
import dataclasses

import numpy as np
import pytest

from tests.compare import compare, F1, F4


def _as_gpu(res, npix, cap):
    n = len(res.hit_count)
    g = {"hit_count": res.hit_count.copy(), "frame_photons": res.frame_photons.astype(np.int64),
         "accum": res.accum.copy(), "hit_pixel": np.zeros((n, cap), np.uint32), "hit_charge": np.zeros((n, cap), np.float32),
         "hit_nphot": np.zeros((n, cap), np.int32), "hit_dx": np.zeros((n, cap), np.float32),
         "hit_dy": np.zeros((n, cap), np.float32)}
    for f in range(n):
        k = len(res.hit_pixel[f])
        g["hit_pixel"][f, :k] = res.hit_pixel[f]
        g["hit_charge"][f, :k] = res.hit_charge[f]
        g["hit_nphot"][f, :k] = res.hit_nphot[f]
        g["hit_dx"][f, :k] = res.hit_dx[f]
        g["hit_dy"][f, :k] = res.hit_dy[f]
    return g


@pytest.fixture(scope="module")
def case(oracle):
    from paper_1903_06838_b200 import synth
    cfg = dataclasses.replace(synth.CONFIGS[0], rows=40, cols=128, seg_cols=64, occupancy=0.02)
    ped, gain = synth.make_maps(cfg)
    raw = synth.make_frames(cfg, 0, 2, ped, gain).numpy()
    res = oracle.process(raw, ped.numpy(), gain.numpy(), panels=1, rows=cfg.rows, cols=cfg.cols, seg_cols=cfg.seg_cols,
                         seed_adu=cfg.seed_adu, cm_adu=cfg.cm_adu, photon_adu=cfg.photon_adu, want_fragile=True)
    assert res.hit_count.min() > 20
    return cfg, res


def _cmp(cfg, res, g):
    return compare(res, g, panels=1, rows=cfg.rows, cols=cfg.cols, seg_cols=cfg.seg_cols, cm_adu=cfg.cm_adu)


def test_identical_passes(case):
    cfg, res = case
    rep = _cmp(cfg, res, _as_gpu(res, cfg.npix, cfg.max_hits))
    assert rep.ok and rep.exempt_hits == 0 and rep.matched == res.hit_count.sum()


def test_unflagged_mismatches_fail(case):
    cfg, res = case
    res = copy.deepcopy(res)
    res.fragile[:] = 0
    for field, delta in (("hit_charge", 0.05), ("hit_dx", 5e-4), ("hit_dy", -5e-4), ("hit_nphot", 1)):
        g = _as_gpu(res, cfg.npix, cfg.max_hits)
        g[field][0, 3] += delta
        if field == "hit_nphot":
            g["frame_photons"][0] += 1
            g["accum"][g["hit_pixel"][0, 3]] += 1
        assert not _cmp(cfg, res, g).ok, field
    g = _as_gpu(res, cfg.npix, cfg.max_hits)          # a hit missing on the GPU side
    k = int(res.hit_count[0])
    g["hit_pixel"][0, 3:k - 1] = g["hit_pixel"][0, 4:k]
    g["hit_count"][0] -= 1
    assert not _cmp(cfg, res, g).ok


def test_flagged_mismatch_is_bounded(case):
    """A flagged hit is matched leniently only inside the SURVEY §8(c) bounds."""
    cfg, res = case
    res = copy.deepcopy(res)
    res.fragile[:] = 0
    px = int(res.hit_pixel[0][3])
    seg_first = (px // cfg.seg_cols) * cfg.seg_cols
    res.fragile[0, seg_first:seg_first + cfg.seg_cols] |= F1           # the hit's own segment may flip a mask pixel
    m = int(res.cm_count[0][px // cfg.seg_cols])
    bound = 9.0 * cfg.cm_adu / m
    g = _as_gpu(res, cfg.npix, cfg.max_hits)
    g["hit_charge"][0, 3] += 0.5 * bound                               # inside 9*T_cm/#M: exempt, counted
    rep = _cmp(cfg, res, g)
    assert rep.ok and rep.exempt_hits == 1 and rep.exempt["F1"] == 1
    g["hit_charge"][0, 3] += 2.0 * bound                               # beyond the bound: failure although flagged
    assert not _cmp(cfg, res, g).ok
    g = _as_gpu(res, cfg.npix, cfg.max_hits)
    g["hit_dx"][0, 3] += 0.05                                          # beyond 0.02 px
    assert not _cmp(cfg, res, g).ok
    # n may differ by one only with F4 (or F1) on the hit, never by two
    res.fragile[:] = 0
    res.fragile[0, px] |= F4
    g = _as_gpu(res, cfg.npix, cfg.max_hits)
    g["hit_nphot"][0, 3] += 1
    g["frame_photons"][0] += 1
    g["accum"][px] += 1
    assert _cmp(cfg, res, g).ok
    g["hit_nphot"][0, 3] += 1
    g["frame_photons"][0] += 1
    g["accum"][px] += 1
    assert not _cmp(cfg, res, g).ok
    # F4 alone does not excuse a float mismatch
    g = _as_gpu(res, cfg.npix, cfg.max_hits)
    g["hit_charge"][0, 3] += 0.05
    assert not _cmp(cfg, res, g).ok
