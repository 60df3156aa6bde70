"""Pins of the fp64 oracle against things other than itself (CPU only).

Each test fixes the oracle to hand-worked values (tests/golden), a library routine
(numpy.median / numpy.mean / numpy.rint), a closed form (erf centroid), brute force with an
independently written rule, or an invariant of the definitions in PAPER.md.
"""
import itertools
import json
import math
import os

import numpy as np
import pytest

GOLD = os.path.join(os.path.dirname(__file__), "golden", "handworked.json")
MODES = {"median": 0, "mean": 1, "none": 2}
TH = dict(seed_adu=50.0, cm_adu=20.0, photon_adu=100.0)


def run(oracle, raw, ped, gain, rows, cols, seg, panels=1, **kw):
    args = dict(TH)
    args.update(kw)
    return oracle.process(raw, ped, gain, panels=panels, rows=rows, cols=cols, seg_cols=seg, **args)


def _cases():
    with open(GOLD) as f:
        return json.load(f)["cases"]


@pytest.mark.parametrize("case", _cases(), ids=lambda c: c["name"])
def test_handworked(oracle, case):
    H, W, S, P = case["rows"], case["cols"], case["seg_cols"], case.get("panels", 1)
    if "raw_rows" in case:
        raw = np.array(case["raw_rows"], np.uint16)
    else:
        raw = np.full((P, H, W), case.get("background", 0), np.uint16)
        for r, c, v in case.get("nonzero", []):
            raw[0, r, c] = v
        for p, r, c, v in case.get("nonzero_p", []):       # [panel, row, col, value]
            raw[p, r, c] = v
    ped = np.full((P, H, W), case["ped"], np.float32)
    gain = np.full((P, H, W), case["gain"], np.float32)
    res = run(oracle, raw.reshape(1, -1), ped, gain, H, W, S, panels=P, cm_mode=MODES[case["cm_mode"]],
              cm_min_count=case.get("cm_min_count", 0), want_cm=True)
    if "cm" in case:
        np.testing.assert_allclose(res.cm[0], case["cm"], rtol=0, atol=1e-12)
    if "cm_count" in case:
        assert res.cm_count[0].tolist() == case["cm_count"]
    if "v2" in case:
        v2, _ = oracle.frame_v2(raw, ped, gain, panels=P, rows=H, cols=W, seg_cols=S,
                                cm_mode=MODES[case["cm_mode"]],
                                cm_min_count=case.get("cm_min_count", 0), **TH)
        np.testing.assert_allclose(v2[0], case["v2"], rtol=0, atol=1e-12)
    if "hit_idx" in case:
        assert res.hit_pixel[0].tolist() == case["hit_idx"]
    if "hits" in case:
        assert res.hit_count[0] == len(case["hits"])
        for k, h in enumerate(case["hits"]):
            assert res.hit_pixel[0][k] == h["idx"]
            assert res.hit_nphot[0][k] == h["n"]
            assert res.hit_charge[0][k] == pytest.approx(h["E"], abs=1e-10)
            assert res.hit_dx[0][k] == pytest.approx(h["dx"], abs=1e-12)
            assert res.hit_dy[0][k] == pytest.approx(h["dy"], abs=1e-12)
        assert res.frame_photons[0] == sum(h["n"] for h in case["hits"])


def test_dark_gain_identity(oracle):
    """O1-O2 special case: ped = 0, gain = 1, no CM  =>  v2 == raw exactly."""
    rng = np.random.default_rng(1)
    raw = rng.integers(0, 65536, (6, 10), dtype=np.uint16)
    v2, cm = oracle.frame_v2(raw, np.zeros((6, 10), np.float32), np.ones((6, 10), np.float32),
                             panels=1, rows=6, cols=10, seg_cols=5, cm_mode=2, **TH)
    assert np.array_equal(v2[0], raw.astype(np.float64))
    assert np.all(cm == 0)


def test_dark_gain_closed_form(oracle):
    """v1 = (raw - ped) / gain in fp64 of the float32 maps; a transposed or swapped operand fails."""
    rng = np.random.default_rng(2)
    raw = rng.integers(900, 1200, (2, 5, 8), dtype=np.uint16)
    ped = rng.normal(1000, 20, (2, 5, 8)).astype(np.float32)
    gain = rng.uniform(0.5, 2.0, (2, 5, 8)).astype(np.float32)
    v2, _ = oracle.frame_v2(raw, ped, gain, panels=2, rows=5, cols=8, seg_cols=4, cm_mode=2, **TH)
    want = (raw.astype(np.float64) - ped.astype(np.float64)) / gain.astype(np.float64)
    assert np.array_equal(v2, want)


@pytest.mark.parametrize("S,W", [(8, 16), (194, 388), (7, 21), (384, 768)])
def test_common_mode_matches_numpy(oracle, S, W):
    """MEDIAN reduces to numpy.median on the masked subset (a library routine: a real pin).
    The MEAN_GUARDED line below RESTATES the oracle's own formula sum/max(k, sqrt(S)): it guards against
    typos only.  What pins the guard is the hand-worked `guard_mean_1x8` fixture (7/sqrt(8)) and, where
    k >= sqrt(S), numpy's plain mean at the end of this test; the guard's FORM against the paper is
    parity unpinned by necessity (Fig. 3 is missing, R4)."""
    rng = np.random.default_rng(S)
    H = 12
    ped = rng.normal(1000, 20, (H, W)).astype(np.float32)
    gain = rng.uniform(0.9, 1.1, (H, W)).astype(np.float32)
    sig = rng.normal(0, 6, (H, W)) + rng.normal(0, 5, (H, W // S)).repeat(S, axis=1)
    sig[rng.random((H, W)) < 0.05] += 90.0
    sig[0, : S - 1] = 300.0                          # row 0, segment 0: too few quiet pixels
    raw = np.clip(np.rint(ped + gain * sig), 0, 65535).astype(np.uint16)
    v1 = (raw.astype(np.float64) - ped.astype(np.float64)) / gain.astype(np.float64)
    min_count = math.ceil(math.sqrt(S))
    want_med = np.zeros((H, W // S))
    want_mean = np.zeros((H, W // S))
    for r in range(H):
        for s in range(W // S):
            seg = v1[r, s * S:(s + 1) * S]
            m = seg[np.abs(seg) < 20.0]
            want_med[r, s] = np.median(m) if m.size >= min_count else 0.0
            want_mean[r, s] = m.sum() / max(m.size, math.sqrt(S))
    _, cm = oracle.frame_v2(raw, ped, gain, panels=1, rows=H, cols=W, seg_cols=S, cm_mode=0, **TH)
    np.testing.assert_allclose(cm[0], want_med, rtol=0, atol=1e-12)
    assert cm[0][0, 0] == 0.0
    _, cm = oracle.frame_v2(raw, ped, gain, panels=1, rows=H, cols=W, seg_cols=S, cm_mode=1, **TH)
    np.testing.assert_allclose(cm[0], want_mean, rtol=0, atol=1e-12)
    # plain mean whenever enough quiet pixels exist (textbook case of the guard)
    full = np.abs(v1[3, :S]) < 20.0
    if full.sum() >= math.sqrt(S):
        assert cm[0][3, 0] == pytest.approx(v1[3, :S][full].mean(), abs=1e-12)


def test_common_mode_shift_invariance(oracle):
    """gain = 1: adding an integer to every raw value of a segment adds it to c, v2 unchanged."""
    rng = np.random.default_rng(5)
    W = S = 33
    ped = np.full((1, W), 1000.0, np.float32)
    gain = np.ones((1, W), np.float32)
    raw = (1000 + np.rint(rng.normal(0, 3, (1, W)))).astype(np.uint16)
    for mode in (0, 1):
        v2a, ca = oracle.frame_v2(raw, ped, gain, panels=1, rows=1, cols=W, seg_cols=S, cm_mode=mode, **TH)
        v2b, cb = oracle.frame_v2(raw + 4, ped, gain, panels=1, rows=1, cols=W, seg_cols=S, cm_mode=mode, **TH)
        assert cb[0, 0, 0] == pytest.approx(ca[0, 0, 0] + 4.0, abs=1e-12)
        np.testing.assert_allclose(v2a, v2b, atol=1e-12)
    # odd count, all pixels quiet: the median of v2 over the mask is exactly 0
    v2, _ = oracle.frame_v2(raw, ped, gain, panels=1, rows=1, cols=W, seg_cols=S, cm_mode=0, **TH)
    assert np.median(v2) == 0.0


def _independent_seeds(v, T):
    """Second, differently written seed rule: sort the <= 9 window values by (-value, index);
    the centre is a seed iff it sorts first and exceeds T."""
    H, W = v.shape
    out = []
    for r in range(H):
        for c in range(W):
            if not v[r, c] > T:
                continue
            win = [(-v[rr, cc], rr * W + cc) for rr in range(max(0, r - 1), min(H, r + 2))
                   for cc in range(max(0, c - 1), min(W, c + 2))]
            if sorted(win)[0][1] == r * W + c:
                out.append(r * W + c)
    return out


def test_seed_rule_bruteforce_8x8(oracle):
    """All placements of 1-2 pixels (and a sample of triples) from a value set with ties on 8x8."""
    H = W = 8
    ped = np.zeros((H, W), np.float32)
    gain = np.ones((H, W), np.float32)
    frames, expect = [], []
    vals = (60, 60, 70)
    cells = list(range(64))
    for a in cells:
        f = np.zeros(64, np.uint16); f[a] = 60
        frames.append(f)
    for a, b in itertools.combinations(cells, 2):
        for va, vb in ((60, 60), (60, 70), (70, 60)):
            f = np.zeros(64, np.uint16); f[a] = va; f[b] = vb
            frames.append(f)
    rng = np.random.default_rng(0)
    for _ in range(3000):
        f = np.zeros(64, np.uint16)
        k = rng.integers(3, 7)
        base = rng.integers(0, 64)
        r0, c0 = divmod(int(base), 8)
        for _ in range(k):                                 # clustered so that windows overlap
            r = min(7, max(0, r0 + rng.integers(-2, 3))); c = min(7, max(0, c0 + rng.integers(-2, 3)))
            f[r * 8 + c] = vals[rng.integers(0, 3)] + (0 if rng.random() < 0.7 else 45)
        frames.append(f)
    raw = np.stack(frames)
    res = run(oracle, raw, ped, gain, H, W, 8, cm_mode=2)
    for i, f in enumerate(frames):
        want = _independent_seeds(f.reshape(8, 8).astype(np.float64), 50.0)
        got = res.hit_pixel[i].tolist()
        assert got == want, (i, f.reshape(8, 8), got, want)
        # no two seeds are 8-adjacent
        for p, q in itertools.combinations(got, 2):
            assert max(abs(p // 8 - q // 8), abs(p % 8 - q % 8)) > 1
    # named cases: horizontal run seeds its leftmost pixel; diagonal pair seeds the upper one
    f = np.zeros((8, 8), np.uint16); f[3, 2:6] = 60
    assert run(oracle, f[None], ped, gain, 8, 8, 8, cm_mode=2).hit_pixel[0].tolist() == [3 * 8 + 2]
    f = np.zeros((8, 8), np.uint16); f[2, 3] = 60; f[3, 2] = 60
    assert run(oracle, f[None], ped, gain, 8, 8, 8, cm_mode=2).hit_pixel[0].tolist() == [2 * 8 + 3]
    f = np.zeros((8, 8), np.uint16); f[2, 2] = 60; f[2, 4] = 60        # same window, not adjacent
    assert run(oracle, f[None], ped, gain, 8, 8, 8, cm_mode=2).hit_pixel[0].tolist() == [18, 20]


def test_seed_rule_bruteforce_two_panels(oracle):
    """Panels never neighbour each other (R12): on random 2-panel frames the
    seeds must equal the independently written rule applied to EACH PANEL ALONE.  Values cluster at the
    panel seam (last rows of panel 0, first rows of panel 1), so an oracle that let row H-1 of panel 0
    neighbour row 0 of panel 1 (they are adjacent in memory) fails here."""
    P, H, W = 2, 4, 5
    ped = np.zeros((P, H, W), np.float32)
    gain = np.ones((P, H, W), np.float32)
    rng = np.random.default_rng(11)
    frames = []
    for _ in range(2000):
        f = np.zeros((P, H, W), np.uint16)
        for _ in range(rng.integers(2, 7)):
            p = rng.integers(0, 2)
            r = (H - 1 - rng.integers(0, 2)) if p == 0 else rng.integers(0, 2)
            f[p, r, rng.integers(0, W)] = (60, 60, 70, 105)[rng.integers(0, 4)]
        frames.append(f)
    raw = np.stack(frames).reshape(len(frames), -1)
    res = run(oracle, raw, ped, gain, H, W, W, panels=P, cm_mode=2)
    n_seam = 0
    for i, f in enumerate(frames):
        want = []
        for p in range(P):
            want += [p * H * W + q for q in _independent_seeds(f[p].astype(np.float64), 50.0)]
        assert res.hit_pixel[i].tolist() == want, (i, f, res.hit_pixel[i].tolist(), want)
        # the same frame read as ONE panel of 2H rows would often give a different answer
        n_seam += want != _independent_seeds(f.reshape(P * H, W).astype(np.float64), 50.0)
        for k, q in enumerate(want):                      # E only sums pixels of the seed's own panel
            p, r, c = q // (H * W), (q // W) % H, q % W
            win = f[p, max(0, r - 1):r + 2, max(0, c - 1):c + 2].astype(np.float64)
            assert res.hit_charge[i][k] == win.sum()
    assert n_seam > 300          # the seam mattered in a good share of the frames


def test_rounding_table(oracle):
    """n = max(0, rint(E/E_ph)) half-to-even, against numpy.rint."""
    H, W = 3, 3
    ped = np.zeros((H, W), np.float32); gain = np.ones((H, W), np.float32)
    for e in (51, 99, 100, 149, 150, 151, 249, 250, 251, 350, 450, 550, 1050, 65535):
        f = np.zeros((H, W), np.uint16); f[1, 1] = e
        res = run(oracle, f[None], ped, gain, H, W, 3, cm_mode=2)
        assert res.hit_nphot[0].tolist() == [int(np.rint(e / 100.0))], e
    # negative total charge clamps to 0: seed 60 surrounded by strongly negative pixels
    ped = np.full((H, W), 100.0, np.float32)
    f = np.full((H, W), 0, np.uint16); f[1, 1] = 160
    res = run(oracle, f[None], ped, gain, H, W, 3, cm_mode=2)
    assert res.hit_count[0] == 1 and res.hit_nphot[0][0] == 0 and res.hit_charge[0][0] == -740.0
    assert res.hit_dx[0][0] == 0.0 and res.hit_dy[0][0] == 0.0      # E <= 0 -> no centroid


def _phi(z):
    return 0.5 * (1.0 + math.erf(z / math.sqrt(2.0)))


def _cloud(H, W, y0, x0, sigma, e):
    img = np.zeros((H, W))
    for r in range(H):
        for c in range(W):
            img[r, c] = e * (_phi((r + 1 - y0) / sigma) - _phi((r - y0) / sigma)) * \
                (_phi((c + 1 - x0) / sigma) - _phi((c - x0) / sigma))
    return img


def test_centroid_closed_form_and_symmetry(oracle):
    """One noise-free cloud: E = charge in the window; dx, dy equal the separable erf closed form
    (NOT the true offset: PAPER.md:L89 'nonlinear dependence'); centred cloud -> (0, 0); mirror."""
    H, W, sigma, e = 9, 11, 0.35, 1000.0
    ped = np.zeros((H, W), np.float32)
    # integer raw would quantise the cloud; use gain = 64 so that raw carries 6 fractional bits
    gain = np.full((H, W), 64.0, np.float32)
    for (u, v) in ((0.0, 0.0), (0.2, -0.3), (-0.45, 0.1)):
        y0, x0 = 4.5 + v, 5.5 + u
        img = _cloud(H, W, y0, x0, sigma, e)
        raw = np.rint(img * 64.0).astype(np.uint16)                    # v1 = raw / 64 exactly
        q = raw.astype(np.float64) / 64.0
        res = run(oracle, raw[None], ped, gain, H, W, W, cm_mode=2)
        assert res.hit_pixel[0].tolist() == [4 * W + 5]
        win = q[3:6, 4:7]
        assert res.hit_charge[0][0] == pytest.approx(win.sum(), abs=1e-9)
        wx = [_phi((j + 0.5 - u) / sigma) - _phi((j - 0.5 - u) / sigma) for j in (-1, 0, 1)]
        wy = [_phi((j + 0.5 - v) / sigma) - _phi((j - 0.5 - v) / sigma) for j in (-1, 0, 1)]
        dx_cf = (wx[2] - wx[0]) / sum(wx)
        dy_cf = (wy[2] - wy[0]) / sum(wy)
        assert res.hit_dx[0][0] == pytest.approx(dx_cf, abs=2e-4)       # raw quantisation 1/64 ADU
        assert res.hit_dy[0][0] == pytest.approx(dy_cf, abs=2e-4)
        if u == 0.0 and v == 0.0:
            assert res.hit_dx[0][0] == 0.0 and res.hit_dy[0][0] == 0.0
        # mirror left-right negates dx, keeps dy and E
        resm = run(oracle, raw[:, ::-1][None].copy(), ped, gain, H, W, W, cm_mode=2)
        assert resm.hit_pixel[0].tolist() == [4 * W + (W - 1 - 5)]
        assert resm.hit_dx[0][0] == pytest.approx(-res.hit_dx[0][0], abs=1e-12)
        assert resm.hit_dy[0][0] == pytest.approx(res.hit_dy[0][0], abs=1e-12)
        # transposing the frame swaps dx and dy
        rest = run(oracle, raw.T[None].copy(), ped.T.copy(), gain.T.copy(), W, H, H, cm_mode=2)
        assert rest.hit_dx[0][0] == pytest.approx(res.hit_dy[0][0], abs=1e-12)
        assert rest.hit_dy[0][0] == pytest.approx(res.hit_dx[0][0], abs=1e-12)


def test_charge_conservation(oracle):
    """Isolated clouds fully inside their 3x3 windows, no noise: sum of E = deposited charge."""
    H, W = 40, 40
    rng = np.random.default_rng(7)
    ped = np.zeros((H, W), np.float32); gain = np.ones((H, W), np.float32)
    raw = np.zeros((H, W), np.uint16)
    total = 0
    for r in range(3, H - 3, 6):
        for c in range(3, W - 3, 6):
            patch = rng.integers(0, 30, (3, 3)); patch[1, 1] = 120 + rng.integers(0, 50)
            raw[r - 1:r + 2, c - 1:c + 2] = patch
            total += int(patch.sum())
    res = run(oracle, raw[None], ped, gain, H, W, W, cm_mode=2)
    assert res.hit_count[0] == len(range(3, H - 3, 6)) ** 2
    assert res.hit_charge[0].sum() == float(total)


def test_noise_only_no_hits_and_invariants(oracle):
    from paper_1903_06838_b200 import synth
    import dataclasses
    cfg = dataclasses.replace(synth.CONFIGS[0], occupancy=0.0, n_frames=3)
    ped, gain = synth.make_maps(cfg)
    raw = synth.make_frames(cfg, 0, 3, ped, gain).numpy()
    res = run(oracle, raw, ped.numpy(), gain.numpy(), cfg.rows, cfg.cols, cfg.seg_cols,
              photon_adu=cfg.photon_adu)
    assert res.hit_count.sum() == 0 and res.accum.sum() == 0

    cfg = synth.CONFIGS[0].scaled(4)
    raw = synth.make_frames(cfg, 0, 4, ped, gain).numpy()
    for mode in (0, 1):
        res = run(oracle, raw, ped.numpy(), gain.numpy(), cfg.rows, cfg.cols, cfg.seg_cols,
                  photon_adu=cfg.photon_adu, cm_mode=mode, threads=2)
        assert res.hit_count.min() > 50                       # ~240 expected per frame
        for f in range(4):
            idx = res.hit_pixel[f].astype(np.int64)
            assert np.all(np.diff(idx) > 0)                   # strictly increasing
            assert res.hit_count[f] <= cfg.max_hits
            assert res.frame_photons[f] == res.hit_nphot[f].sum()
        assert res.accum.sum() == res.frame_photons.sum()
        # permutation of the frames leaves accum unchanged
        res2 = run(oracle, raw[::-1].copy(), ped.numpy(), gain.numpy(), cfg.rows, cfg.cols,
                   cfg.seg_cols, photon_adu=cfg.photon_adu, cm_mode=mode)
        assert np.array_equal(res.accum, res2.accum)
        assert res2.hit_pixel[0].tolist() == res.hit_pixel[3].tolist()


def test_overflow_semantics(oracle):
    """True count, truncated list, totals over all seeds."""
    H, W = 6, 6
    ped = np.zeros((H, W), np.float32); gain = np.ones((H, W), np.float32)
    raw = np.zeros((H, W), np.uint16); raw[::2, ::2] = 120
    res = run(oracle, raw[None], ped, gain, H, W, W, cm_mode=2, hit_capacity=4)
    assert res.hit_count[0] == 9 and len(res.hit_pixel[0]) == 4
    assert res.hit_pixel[0].tolist() == [0, 2, 4, 12]
    assert res.frame_photons[0] == 9 and res.accum.sum() == 9


def test_fragile_flags(oracle):
    """A value 5e-5 from T_cm flags its whole segment (F1); 5e-5 from T_seed flags the pixel (F2)."""
    W = 8
    ped = np.zeros((1, W), np.float32)
    gain = np.ones((1, W), np.float32); gain[0, 2] = np.float32(1.0 / (20.0 - 5e-5))
    raw = np.zeros((1, W), np.uint16); raw[0, 2] = 1                     # v1 = 19.99995
    res = run(oracle, raw[None], ped, gain, 1, W, 4, cm_mode=0, want_fragile=True)
    assert res.fragile[0].tolist() == [1, 1, 1, 1, 0, 0, 0, 0]
    gain[0, 2] = np.float32(1.0 / (50.0 + 5e-5))
    res = run(oracle, raw[None], ped, gain, 1, W, 4, cm_mode=2, want_fragile=True)
    assert res.fragile[0][2] & 2 and res.fragile[0][5] == 0


def _frame_with_values(vals, W=8):
    """1 x W frame whose v1 equals `vals` (col -> value) to fp64 rounding of 1/float32(1/v)."""
    ped = np.zeros((1, W), np.float32)
    gain = np.ones((1, W), np.float32)
    raw = np.zeros((1, W), np.uint16)
    for c, v in vals.items():
        gain[0, c] = np.float32(1.0 / v)
        raw[0, c] = 1
    return raw, ped, gain


def test_fragile_flags_f3_f4(oracle):
    """F3: two 3x3 neighbours closer than the band (1e-4 ADU) while near/above T_seed flag BOTH pixels,
    2e-4 apart flags nothing.  F4: E within the band of (k + 1/2) E_ph flags the seed, 2e-4 away does not.
    (BASELINE.json: 'pixels whose fp64 value lies within 1e-4 ADU of a threshold'; R21.)
    An over-wide F3/F4 would silently widen what tests/compare.py forgives; a missing one would make
    the parity tests fail on legitimate rounding differences."""
    F3, F4 = 4, 8
    # two neighbours 5e-5 apart at 60 ADU (above T_seed = 50)
    raw, ped, gain = _frame_with_values({2: 60.0, 3: 60.0 + 5e-5})
    v1 = raw.astype(np.float64) / gain.astype(np.float64)
    assert 2e-5 < abs(v1[0, 3] - v1[0, 2]) < 9e-5
    res = run(oracle, raw[None], ped, gain, 1, 8, 8, cm_mode=2, want_fragile=True)
    fr = res.fragile[0]
    assert fr[2] & F3 and fr[3] & F3
    assert not (fr[[0, 1, 4, 5, 6, 7]] & F3).any()           # background pairs (0 == 0) are far below T_seed
    assert res.hit_pixel[0].tolist() == [3]                   # the larger one seeds
    # 2e-4 apart: no F3 anywhere
    raw, ped, gain = _frame_with_values({2: 60.0, 3: 60.0 + 2e-4})
    res = run(oracle, raw[None], ped, gain, 1, 8, 8, cm_mode=2, want_fragile=True)
    assert not (res.fragile[0] & F3).any()
    # near-tie BELOW the seed threshold (30 ADU): irrelevant to any output, not flagged
    raw, ped, gain = _frame_with_values({2: 30.0, 3: 30.0 + 5e-5})
    res = run(oracle, raw[None], ped, gain, 1, 8, 8, cm_mode=2, want_fragile=True)
    assert not (res.fragile[0] & F3).any() and res.hit_count[0] == 0
    # non-adjacent pixels (columns 2 and 5) 5e-5 apart: not a 3x3 pair, not flagged
    raw, ped, gain = _frame_with_values({2: 60.0, 5: 60.0 + 5e-5})
    res = run(oracle, raw[None], ped, gain, 1, 8, 8, cm_mode=2, want_fragile=True)
    assert not (res.fragile[0] & F3).any() and res.hit_pixel[0].tolist() == [2, 5]
    # F4: lone pixel with E = 150 +- 5e-5 (rounding boundary 1.5 * E_ph) is flagged, 150 +- 2e-4 is not
    for e, want in ((150.0 + 5e-5, True), (150.0 - 5e-5, True), (150.0 + 2e-4, False), (150.0 - 2e-4, False),
                    (250.0 + 5e-5, True), (200.0 + 5e-5, False), (100.0, False)):
        raw, ped, gain = _frame_with_values({4: e})
        res = run(oracle, raw[None], ped, gain, 1, 8, 8, cm_mode=2, want_fragile=True)
        assert res.hit_pixel[0].tolist() == [4]
        assert bool(res.fragile[0][4] & F4) == want, e
        assert not (res.fragile[0][[0, 1, 2, 3, 5, 6, 7]] & F4).any()
        assert res.hit_nphot[0][0] == int(np.rint((1.0 / float(gain[0, 4])) / 100.0))
