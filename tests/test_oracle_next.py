"""Pins of the oracle's extensions beyond the hot path, CPU only:
stacked / other-shape common-mode stages, histogram summarization (L99, L109, L113)
and dense photon counting by division and rounding (L83, L91).  Hand-worked values, closed forms,
symmetries and library routines; none of the expectations comes from the oracle or the CUDA path."""
import math

import numpy as np
import pytest

TH = dict(seed_adu=50.0, cm_adu=20.0, photon_adu=100.0)
MEDIAN, MEAN, NONE = 0, 1, 2


def v2_of(oracle, raw, ped=0.0, gain=1.0, stages=None, panels=1, seg_cols=None, **kw):
    raw = np.asarray(raw, np.uint16)
    P = panels
    H, W = raw.shape[-2], raw.shape[-1]
    args = dict(TH)
    args.update(kw)
    return oracle.frame_v2(raw, np.full((P, H, W), ped, np.float32), np.full((P, H, W), gain, np.float32), panels=P,
                           rows=H, cols=W, seg_cols=seg_cols or W, stages=stages, **args)


# ---------------------------------------------------------------- O3': stages ----
def test_row_then_column_mean_removes_additive_pattern(oracle):
    """Hand-worked 4x4: v1[i][j] = row_off[i] + col_off[j].  Row stage (1x4 mean): c = row_off[i] + 4, residue
    col_off[j] - 4 = [-4, -2, 0, 6]; column stage (4x1 mean) removes it exactly: v2 == 0 (PAPER.md:L55 'row, column
    ... by reshaping'; L117 stacked stages)."""
    row_off, col_off = np.array([1, 2, 3, 4]), np.array([0, 2, 4, 10])
    raw = row_off[:, None] + col_off[None, :]
    v2, cm = v2_of(oracle, raw, stages=[(1, 4, MEAN), (4, 1, MEAN)])
    assert np.array_equal(v2[0], np.zeros((4, 4)))
    assert cm.reshape(-1).tolist() == [-4.0, -2.0, 0.0, 6.0]            # estimates of the LAST stage, per column
    # the stages are applied in order, each on the previous one's output: a single row stage leaves the residue
    v2, cm = v2_of(oracle, raw, stages=[(1, 4, MEAN)])
    assert np.array_equal(v2[0], np.tile(col_off - 4.0, (4, 1)))
    assert cm.reshape(-1).tolist() == [5.0, 6.0, 7.0, 8.0]
    # median estimator: row medians are row_off[i] + (2+4)/2, residue [-3, -1, 1, 7], columns constant -> 0
    v2, cm = v2_of(oracle, raw, stages=[(1, 4, MEDIAN), (4, 1, MEDIAN)])
    assert np.array_equal(v2[0], np.zeros((4, 4)))
    assert cm.reshape(-1).tolist() == [-3.0, -1.0, 1.0, 7.0]


def test_block_stage_and_three_stacked(oracle):
    """2x2 blocks with offsets [[10, 20], [30, 0]] on a 4x4 panel: the block stage removes them exactly; stacked
    after a row and a column stage of an additive pattern (three stages) the result is still 0."""
    blk = np.kron(np.array([[10, 20], [30, 0]]), np.ones((2, 2), int))
    v2, cm = v2_of(oracle, blk, stages=[(2, 2, MEAN)], cm_adu=40.0)
    assert np.array_equal(v2[0], np.zeros((4, 4))) and cm.reshape(-1).tolist() == [10.0, 20.0, 30.0, 0.0]
    add = np.array([1, 2, 3, 4])[:, None] + np.array([0, 2, 4, 10])[None, :]
    raw = add + 1                                                         # + a panel-wide offset for the third stage
    v2, cm = v2_of(oracle, raw, stages=[(1, 4, MEAN), (4, 1, MEAN), (4, 4, MEAN)])
    assert np.array_equal(v2[0], np.zeros((4, 4))) and cm.reshape(-1).tolist() == [0.0]
    # a single 16 ADU pixel at (0, 0), hand-worked: row stage -> row 0 = [12, -4, -4, -4]; 2x2 block stage ->
    # top-left block mean 2, top-right block mean -2
    raw = np.zeros((4, 4), int)
    raw[0, 0] = 16
    a, _ = v2_of(oracle, raw, stages=[(1, 4, MEAN), (2, 2, MEAN)])
    assert a[0].tolist() == [[10, -6, -2, -2], [-2, -2, 2, 2], [0, 0, 0, 0], [0, 0, 0, 0]]


def test_frame_stage_guard_sqrt_hw(oracle):
    """The paper's frame-wise stage with its sqrt(HW) term: 4x4 panel, only two quiet pixels
    (3 and 5 ADU), fourteen at 250: c = 8 / max(2, sqrt(16)) = 2, not 4 (reading R4); with twelve quiet
    pixels the plain mean."""
    raw = np.full((4, 4), 250)
    raw[0, 0], raw[3, 3] = 3, 5
    v2, cm = v2_of(oracle, raw, stages=[(4, 4, MEAN)])
    assert cm.reshape(-1).tolist() == [2.0] and v2[0][0, 0] == 1.0 and v2[0][1, 1] == 248.0
    raw = np.full((4, 4), 6)
    raw[0, :] = 250
    v2, cm = v2_of(oracle, raw, stages=[(4, 4, MEAN)])
    assert cm.reshape(-1).tolist() == [6.0]
    # median on the same group shape: 2 quiet pixels < ceil(sqrt(16)) = 4 -> c = 0
    raw = np.full((4, 4), 250)
    raw[0, 0], raw[3, 3] = 3, 5
    _, cm = v2_of(oracle, raw, stages=[(4, 4, MEDIAN)])
    assert cm.reshape(-1).tolist() == [0.0]


def test_single_stage_equals_hot_path_and_transpose_symmetry(oracle):
    """(a) one stage of 1 x seg_cols groups IS the hot path's common mode (ties the staged code to the pinned
    one); (b) a column stage on a frame equals the row stage on the transposed frame, transposed (a swapped
    gh/gw or a wrong stride fails); (c) groups never mix panels."""
    rng = np.random.default_rng(4)
    P, H, W, S = 2, 6, 8, 4
    ped = rng.normal(100, 5, (P, H, W)).astype(np.float32)
    gain = rng.uniform(0.9, 1.1, (P, H, W)).astype(np.float32)
    raw = np.clip(np.rint(ped + gain * (rng.normal(0, 4, (P, H, W)) + 90.0 * (rng.random((P, H, W)) < 0.1))), 0, 65535).astype(np.uint16)
    kw = dict(panels=P, rows=H, cols=W, seg_cols=S, **TH)
    for mode in (MEDIAN, MEAN):
        a, ca = oracle.frame_v2(raw, ped, gain, cm_mode=mode, **kw)
        b, cb = oracle.frame_v2(raw, ped, gain, stages=[(1, S, mode)], **kw)
        assert np.array_equal(a, b) and np.array_equal(ca.reshape(-1), cb.reshape(-1))
        # column stage (3 x 1 groups) vs row stage (1 x 3) on the transposed panels
        c, _ = oracle.frame_v2(raw, ped, gain, stages=[(3, 1, mode)], **kw)
        rt, pt, gt = (np.ascontiguousarray(x.transpose(0, 2, 1)) for x in (raw, ped, gain))
        d, _ = oracle.frame_v2(rt, pt, gt, panels=P, rows=W, cols=H, seg_cols=H, stages=[(1, 3, mode)], **TH)
        assert np.array_equal(c, d.transpose(0, 2, 1))
        # panel-wise stage: each panel's estimate only depends on its own pixels
        e, ce = oracle.frame_v2(raw, ped, gain, stages=[(H, W, mode)], **kw)
        e0, ce0 = oracle.frame_v2(raw[:1], ped[:1], gain[:1], panels=1, rows=H, cols=W, seg_cols=S, stages=[(H, W, mode)], **TH)
        assert np.array_equal(e[0], e0[0]) and ce.reshape(-1)[0] == ce0.reshape(-1)[0]
    # a stage that does not tile the panel is refused
    with pytest.raises(Exception):
        oracle.frame_v2(raw, ped, gain, stages=[(4, 4, MEAN)], **kw)


def test_last_mean_stage_leaves_zero_group_means(oracle):
    """Invariant: after a mean stage whose groups are fully inside the mask, every group of that stage has zero
    mean, whatever came before (three stacked stages on noise)."""
    rng = np.random.default_rng(8)
    H, W = 12, 16
    raw = (1000 + np.rint(rng.normal(0, 3, (H, W)))).astype(np.uint16)
    v2, _ = v2_of(oracle, raw, ped=1000.0, stages=[(1, 8, MEAN), (4, 1, MEDIAN), (3, 4, MEAN)])
    g = v2[0].reshape(H // 3, 3, W // 4, 4).mean(axis=(1, 3))
    assert np.abs(g).max() < 1e-12


def test_stages_drive_the_hit_finder(oracle):
    """The seed finder runs on the output of the LAST stage: a 60 ADU pixel on a +30 ADU column offset seeds
    after (row, column) stages but its E is 60, not 90; with the row stage alone the whole column seeds nothing
    different... checked through process()."""
    H, W = 8, 8
    raw = np.zeros((H, W), np.uint16) + 100
    raw[:, 5] += 30                                   # column offset above T_cm: the row stage masks it out
    raw[3, 2] += 60
    ped = np.full((H, W), 100.0, np.float32)
    gain = np.ones((H, W), np.float32)
    res = oracle.process(raw[None], ped, gain, panels=1, rows=H, cols=W, seg_cols=W, stages=[(1, 8, MEAN), (8, 1, MEAN)],
                         cm_adu=40.0, seed_adu=50.0, photon_adu=100.0)
    # hand-worked: row means over the 8 masked pixels: rows != 3: 30/8 = 3.75; row 3 (60 is unmasked, 7 masked): 30/7.
    # after the row stage column 5 holds 26.25 (rows != 3) / 25.714 (row 3), masked by T_cm = 40; the column stage
    # removes each column's mean; pixel (3, 2): 60 - 30/7 minus the column-2 mean ((-3.75*7 - 30/7 + 60)/8 is NOT
    # used: 55.71 > 40 is unmasked, so the column mean is over the 7 others: -3.75) = 60 - 30/7 + 3.75
    assert res.hit_pixel[0].tolist() == [3 * 8 + 2]
    v2, _ = oracle.frame_v2(raw, ped, gain, panels=1, rows=H, cols=W, seg_cols=W, stages=[(1, 8, MEAN), (8, 1, MEAN)],
                            cm_adu=40.0, seed_adu=50.0, photon_adu=100.0)
    assert v2[0][3, 2] == pytest.approx(60 - 30 / 7 + 3.75, abs=1e-12)
    assert res.hit_charge[0][0] == pytest.approx(v2[0][2:5, 1:4].sum(), abs=1e-9)
    # the ORDER of the stages matters: column stage first removes the 30 ADU column exactly (it is inside the mask),
    # column 2 has mean 0 over its 7 masked pixels, and the row stage then finds nothing: v2(3, 2) = 60 exactly
    v2r, _ = oracle.frame_v2(raw, ped, gain, panels=1, rows=H, cols=W, seg_cols=W, stages=[(8, 1, MEAN), (1, 8, MEAN)],
                             cm_adu=40.0, seed_adu=50.0, photon_adu=100.0)
    assert v2r[0][3, 2] == 60.0 and np.count_nonzero(v2r[0]) == 1


# ---------------------------------------------------------------- O11: histograms ----
def test_histogram_handworked_edges(oracle):
    """Uniform bins [lo + b w, lo + (b+1) w): a value on an edge belongs to the bin it opens; below lo and at or
    above lo + nbins w it is dropped."""
    x = [0.0, 9.999, 10.0, 49.99, 50.0, -0.001, 25.0, 1e9, -1e9]
    h = oracle.histogram(x, lo=0.0, width=10.0, nbins=5)
    assert h.tolist() == [2, 1, 1, 0, 1]
    h = oracle.histogram([-1.0, -0.75, -0.5, 0.0, 0.49, 0.5, 0.999, 1.0], lo=-1.0, width=0.5, nbins=4)   # dx, dy range
    assert h.tolist() == [2, 1, 2, 2]
    # accumulates into a given histogram
    h2 = oracle.histogram([0.0, 0.6], lo=-1.0, width=0.5, nbins=4, hist=h)
    assert h2.tolist() == [2, 1, 3, 3]
    assert oracle.histogram([], 0.0, 1.0, 3).tolist() == [0, 0, 0]
    # values just outside must not land in a neighbouring memory word either (guard elements around the bins)
    big = np.zeros(7, np.uint64)
    oracle.histogram(x, lo=0.0, width=10.0, nbins=5, hist=big[1:6])
    assert big.tolist() == [0, 2, 1, 1, 0, 1, 0]


def test_histogram_matches_numpy(oracle):
    """Reduces to numpy.histogram on values that avoid numpy's closed last edge."""
    rng = np.random.default_rng(2)
    x = rng.normal(80, 30, 20000)
    lo, w, nb = np.float32(5.0), np.float32(2.5), 64
    want, _ = np.histogram(x[x < float(lo) + nb * float(w) - 1e-9], bins=float(lo) + float(w) * np.arange(nb + 1))
    assert oracle.histogram(x, lo, w, nb).tolist() == want.tolist()


# ---------------------------------------------------------------- O12: dense photon counting ----
def test_dense_counting_handworked(oracle):
    """n_px = max(0, rint(v2 / E_ph)) half-to-even: v2 = 0, 49, 50, 51, 150, 250, -50, 160 at
    E_ph = 100 -> 0, 0, 0, 1, 2, 2, 0, 2; zeroing below a noise threshold (L91); accumulation over frames."""
    raw = np.array([[100, 149, 150, 151, 250, 350, 50, 260]], np.uint16)
    ped = np.full((1, 8), 100.0, np.float32)
    gain = np.ones((1, 8), np.float32)
    kw = dict(panels=1, rows=1, cols=8, seg_cols=8, cm_adu=20.0, photon_adu=100.0)
    img, tot, _ = oracle.dense(raw[None], ped, gain, cm_mode=NONE, **kw)
    assert img.tolist() == [0, 0, 0, 1, 2, 2, 0, 2] and tot.tolist() == [7]
    img, tot, _ = oracle.dense(raw[None], ped, gain, cm_mode=NONE, zero_below_adu=51.0, **kw)
    assert img.tolist() == [0, 0, 0, 1, 2, 2, 0, 2]                     # 51 is not below 51
    img, tot, _ = oracle.dense(raw[None], ped, gain, cm_mode=NONE, zero_below_adu=155.0, **kw)
    assert img.tolist() == [0, 0, 0, 0, 0, 2, 0, 2] and tot.tolist() == [4]
    img, tot, _ = oracle.dense(np.stack([raw, raw, raw]), ped, gain, cm_mode=NONE, **kw)
    assert img.tolist() == [0, 0, 0, 3, 6, 6, 0, 6] and tot.tolist() == [7, 7, 7]
    # on top of the common mode: the median_1x8 fixture (v2 = -2, 3, 1, 145, -1, 4, 0, -3) counts one photon
    raw = np.array([[103, 108, 106, 250, 104, 109, 105, 102]], np.uint16)
    img, tot, _ = oracle.dense(raw[None], ped, gain, cm_mode=MEDIAN, **kw)
    assert img.tolist() == [0, 0, 0, 1, 0, 0, 0, 0] and tot.tolist() == [1]
    # gain division happens before the rounding: (310 - 10) / 2 = 150 -> 2
    img, _, _ = oracle.dense(np.array([[[10, 310]]], np.uint16), np.full((1, 2), 10.0, np.float32),
                             np.full((1, 2), 2.0, np.float32), panels=1, rows=1, cols=2, seg_cols=2, cm_adu=20.0,
                             photon_adu=100.0, cm_mode=NONE)
    assert img.tolist() == [0, 2]


def test_dense_counting_matches_numpy_and_flags(oracle):
    """Against numpy.rint on the oracle-independent v2 = (raw - ped)/gain (no common mode), and the fragile flag at
    a rounding boundary."""
    rng = np.random.default_rng(6)
    P, H, W = 2, 5, 8
    ped = rng.normal(1000, 20, (P, H, W)).astype(np.float32)
    gain = rng.uniform(0.9, 1.1, (P, H, W)).astype(np.float32)
    raw = rng.integers(900, 1600, (3, P, H, W)).astype(np.uint16)
    img, tot, frag = oracle.dense(raw, ped, gain, panels=P, rows=H, cols=W, seg_cols=4, cm_adu=20.0, photon_adu=120.0,
                                  cm_mode=NONE, want_fragile=True)
    v = (raw.astype(np.float64) - ped.astype(np.float64)) / gain.astype(np.float64)
    n = np.maximum(0, np.rint(v / 120.0)).astype(np.int64)
    assert np.array_equal(img.reshape(P, H, W), n.sum(0)) and tot.tolist() == n.reshape(3, -1).sum(1).tolist()
    assert not frag.any()
    # v2 = 150 + 5e-5 at E_ph = 100: flagged; 150 + 2e-4: not
    for e, want in ((150.0 + 5e-5, True), (150.0 + 2e-4, False)):
        g1 = np.ones((1, 2), np.float32)
        g1[0, 1] = np.float32(1.0 / e)
        _, _, fr = oracle.dense(np.array([[[0, 1]]], np.uint16), np.zeros((1, 2), np.float32), g1, panels=1, rows=1, cols=2,
                                seg_cols=2, cm_adu=20.0, photon_adu=100.0, cm_mode=NONE, want_fragile=True)
        assert bool(fr[0, 1] & 8) == want
