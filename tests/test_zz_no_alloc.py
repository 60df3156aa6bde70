"""pdp_histograms_static: the histogram summarization with its workspace in a static __device__ array, for callers
that cannot allocate (include/pdp.h).  Its output must equal the allocating path's (pdp_histograms) bit for bit —
integer work, so the tolerance of the other histogram tests applies: none — on two calls in a row that share the
scratch array, the second with fewer frames and other bins, so that words left behind by the first call would show.

Named test_zz_* so that pytest collects it last: the suite runs with `pytest -x`, and a failure here must not hide
the tests before it.  It runs alone in a fresh process as well as after the other tests (no state is shared with them
beyond the built library)."""
import ctypes
import dataclasses

import numpy as np
import pytest
import torch

from paper_1903_06838_b200 import binding, build


def test_static_scratch_rejects_sizes_beyond_the_maximum():
    """Argument checks come before any CUDA call: they run without a GPU."""
    build.build()
    lib = binding.load_library()
    out = binding.pdp_output(16, 8, 8, 8, 8, 8, 8, 8, 8, 8)        # non-NULL dummies, never dereferenced
    big = binding.pdp_hist_spec(0.0, 1.0, binding.STATIC_HIST_MAX_BINS + 1)
    rc = lib.pdp_histograms_static(ctypes.byref(out), 4, ctypes.byref(big), 8, None, None, None, None)
    assert rc == -3, rc                                             # PDP_E_VALUE
    msg = lib.pdp_static_last_error().decode()
    assert "exceed" in msg and str(binding.STATIC_HIST_MAX_BINS) in msg, msg
    e, d = binding.pdp_hist_spec(0.0, 1.0, 2048), binding.pdp_hist_spec(-1.0, 0.01, 1025)   # 2048 + 2 * 1025 > 4096
    assert lib.pdp_histograms_static(ctypes.byref(out), 4, ctypes.byref(e), 8, ctypes.byref(d), 8, 8, None) == -3
    assert lib.pdp_histograms_static(None, 4, ctypes.byref(e), 8, None, None, None, None) == -1          # PDP_E_NULL
    assert lib.pdp_histograms_static(ctypes.byref(out), -1, ctypes.byref(e), 8, None, None, None, None) == -4   # PDP_E_BATCH
    assert lib.pdp_histograms_static(ctypes.byref(out), 0, ctypes.byref(e), 8, None, None, None, None) == 0     # no-op
    assert lib.pdp_static_last_error().decode() == ""


@pytest.mark.gpu
def test_static_scratch_histograms_match_the_allocating_path():
    if not torch.cuda.is_available():
        pytest.skip("needs a CUDA device")
    from paper_1903_06838_b200 import synth
    build.build()
    dev = "cuda"
    cfg, n = dataclasses.replace(synth.CONFIGS[0], rows=60, cols=128, seg_cols=64, occupancy=0.03), 200
    ped, gain = synth.make_maps(cfg, dev)
    raw = synth.make_frames(cfg, 0, n, ped, gain)
    ctx = binding.Context(panels=cfg.panels, rows=cfg.rows, cols=cfg.cols, seg_cols=cfg.seg_cols, max_frames_per_batch=n,
                          pedestal=ped.cpu(), gain=gain.cpu(), seed_adu=cfg.seed_adu, cm_adu=cfg.cm_adu,
                          photon_adu=cfg.photon_adu)
    out = binding.alloc_output(n, cfg.npix, cfg.max_hits, dev)
    ctx.process(raw, out)
    torch.cuda.synchronize()
    assert int((out.hit_count.to(torch.int64) & 0xFFFFFFFF).sum()) > 10000

    def zeros(k):
        return torch.zeros(k, dtype=torch.int32, device=dev)

    # call 1: all frames, the largest bin count the static scratch takes (2048 + 2 * 1024 = 4096), 128 CTAs;
    # call 2, right after it on the same stream: 37 frames (37 CTAs), other and fewer bins -> other row stride:
    # it reads only what it wrote itself, whatever call 1 left in the array.
    calls = [(n, (20.0, 0.125, 2048), (-1.0, 2.0 / 1024, 1024)), (37, (20.0, 2.5, 96), (-1.0, 0.03125, 64))]
    got, want = [], []
    for nf, e_spec, d_spec in calls:
        h = [zeros(e_spec[2]), zeros(d_spec[2]), zeros(d_spec[2])]
        binding.histograms_static(out, nf, energy=e_spec, dxy=d_spec, hist_energy=h[0], hist_dx=h[1], hist_dy=h[2])
        got.append(h)
    torch.cuda.synchronize()
    for nf, e_spec, d_spec in calls:
        h = [zeros(e_spec[2]), zeros(d_spec[2]), zeros(d_spec[2])]
        ctx.histograms(out, nf, energy=e_spec, dxy=d_spec, hist_energy=h[0], hist_dx=h[1], hist_dy=h[2])
        want.append(h)
    torch.cuda.synchronize()
    for (nf, _, _), g, w in zip(calls, got, want):
        hits = int((out.hit_count[:nf].to(torch.int64) & 0xFFFFFFFF).sum())
        assert int(w[0].sum()) > 0.9 * hits                          # the reference path saw the hits at all
        for a, b in zip(g, w):
            assert np.array_equal(a.cpu().numpy(), b.cpu().numpy())

    # += semantics and a repeat of call 1 after call 2: still the same counts (doubles the first result)
    nf, e_spec, d_spec = calls[0]
    binding.histograms_static(out, nf, energy=e_spec, dxy=d_spec, hist_energy=got[0][0], hist_dx=got[0][1], hist_dy=got[0][2])
    # only one of the two histograms
    he = zeros(e_spec[2])
    binding.histograms_static(out, nf, energy=e_spec, hist_energy=he)
    torch.cuda.synchronize()
    for a, b in zip(got[0], want[0]):
        assert np.array_equal(a.cpu().numpy(), 2 * b.cpu().numpy())
    assert np.array_equal(he.cpu().numpy(), want[0][0].cpu().numpy())
    with pytest.raises(binding.PdpError, match="exceed"):
        binding.histograms_static(out, nf, energy=(0.0, 1.0, 4097), hist_energy=zeros(4097))
    ctx.close()
