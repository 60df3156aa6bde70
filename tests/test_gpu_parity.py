"""GPU parity: the CUDA path (through the C ABI) against the fp64 oracle, element by element, on the
same seeded inputs.  Integers bit-exact except oracle-flagged fragile pixels (counted), floats within
1e-4 + 1e-4*|ref| (tests/compare.py)."""
import dataclasses
import os

import numpy as np
import pytest
import torch

from tests.compare import compare

pytestmark = pytest.mark.gpu

if not torch.cuda.is_available():  # collected everywhere, run only where a GPU exists
    pytest.skip("needs a CUDA device", allow_module_level=True)

from paper_1903_06838_b200 import binding, build, synth  # noqa: E402

build.build()
DEV = "cuda"
LAUNCHES_PER_CALL = 2      # kernels one pdp_process call enqueues on the throughput path (chain + accumulated image)


def small(cfg_id, **kw):
    return dataclasses.replace(synth.CONFIGS[cfg_id], **kw)


KERNELS = {None: 0, "auto": 0, "lookback": 1, "chain": 2}
LAUNCHES = {"lookback": 1, "chain": 2}       # chain kernel + accumulated-image pass


def gpu_run(cfg, raw, ped, gain, cm_mode, *, cap=None, cm_min_count=0, keep_cm=False, host_chunk=None,
            n_calls=1, kernel=None, variant=0, sparse_warps=0, chunk_frames=0):
    # the library picks its kernel by batch size (frame-owner throughput kernel for large batches, band x
    # chunk items with look-back for small ones); pdp_debug_set pins one so that both are tested on every case
    ctx = binding.Context(panels=cfg.panels, rows=cfg.rows, cols=cfg.cols, seg_cols=cfg.seg_cols,
                          max_frames_per_batch=max(1, raw.shape[0]), pedestal=ped.cpu(), gain=gain.cpu(),
                          seed_adu=cfg.seed_adu, cm_adu=cfg.cm_adu, photon_adu=cfg.photon_adu,
                          cm_mode=cm_mode, cm_min_count=cm_min_count)
    ctx.debug_set("kernel", KERNELS[kernel])
    if variant:
        ctx.debug_set("variant", variant)
    if sparse_warps:
        ctx.debug_set("sparse_warps", sparse_warps)
    if chunk_frames:
        ctx.debug_set("chunk_frames", chunk_frames)
    if keep_cm:
        ctx.keep_common_mode(True)
    out = binding.alloc_output(raw.shape[0], cfg.npix, cap or cfg.max_hits, DEV)
    for _ in range(n_calls):
        if host_chunk:
            ctx.process_host(raw.cpu().pin_memory(), out, host_chunk)
        else:
            ctx.process(raw, out)
    torch.cuda.synchronize()
    res = {k: getattr(out, k).cpu().numpy() for k in
           ("hit_count", "hit_pixel", "hit_charge", "hit_nphot", "hit_dx", "hit_dy", "frame_photons", "accum", "status")}
    res["hit_count"] = res["hit_count"].astype(np.int64) & 0xFFFFFFFF
    res["frame_photons"] = res["frame_photons"].astype(np.int64) & 0xFFFFFFFF
    if keep_cm:
        res["cm"] = ctx.common_mode(raw.shape[0]).cpu().numpy()
    res["launches"] = ctx.last_launch_count
    res["kernel"] = ctx.last_kernel_name
    ctx.close()
    return res


def oracle_run(oracle, cfg, raw, ped, gain, cm_mode, **kw):
    return oracle.process(raw.cpu().numpy(), ped.cpu().numpy(), gain.cpu().numpy(), panels=cfg.panels,
                          rows=cfg.rows, cols=cfg.cols, seg_cols=cfg.seg_cols, seed_adu=cfg.seed_adu,
                          cm_adu=cfg.cm_adu, photon_adu=cfg.photon_adu, cm_mode=cm_mode, threads=os.cpu_count() or 1,
                          want_fragile=True, **kw)


def make(cfg, n):
    ped, gain = synth.make_maps(cfg, DEV)
    raw = synth.make_frames(cfg, 0, n, ped, gain)
    return raw, ped, gain


CASES = {
    "tiny_185x388": (small(0), 6),
    "epix_704x768": (small(1), 3),
    "epix_T30": (small(1, seed_adu=30.0), 2),
    "cspad_3x185x388": (small(2, panels=3), 3),
    "dense_96x1024": (small(3, rows=96), 3),
    "lcls2_2x70x512": (small(4, panels=2, rows=70), 3),
    "ragged_2x11x72_s24": (small(0, panels=2, rows=11, cols=72, seg_cols=24, occupancy=0.02), 5),
    "narrow_5x60_s30": (small(0, rows=5, cols=60, seg_cols=30, occupancy=0.03), 7),
    "one_row": (small(0, rows=1, cols=128, seg_cols=64, occupancy=0.03), 4),
    "single_segment_40x256": (small(4, panels=1, rows=40, cols=256, seg_cols=256), 3),
}


@pytest.mark.parametrize("kernel", ["chain", "lookback"])
@pytest.mark.parametrize("cm_mode", [0, 1, 2], ids=["median", "mean", "none"])
@pytest.mark.parametrize("case", list(CASES), ids=list(CASES))
def test_parity(oracle, case, cm_mode, kernel):
    cfg, n = CASES[case]
    raw, ped, gain = make(cfg, n)
    g = gpu_run(cfg, raw, ped, gain, cm_mode, kernel=kernel)
    o = oracle_run(oracle, cfg, raw, ped, gain, cm_mode)
    rep = compare(o, g, panels=cfg.panels, rows=cfg.rows, cols=cfg.cols, seg_cols=cfg.seg_cols, cm_adu=cfg.cm_adu)
    print(case, cm_mode, rep.summary())
    assert rep.ok, rep.failures[:10]
    assert rep.hits_oracle > 0
    assert rep.exempt_hits <= max(3, rep.hits_oracle // 200)       # exemptions stay rare
    assert g["status"][0] == 0 and g["launches"] == LAUNCHES[kernel]
    assert g["kernel"].startswith("pdp_chain_kernel" if kernel == "chain" else "pdp_fused_kernel")


# layouts of the throughput kernel (V pixels per vector, NV vectors per lane, LPS lanes per row segment):
# every layout that covers the geometry must give bit-identical results
VARIANTS = {
    "epix_704x768": (80608, 80316, 80232, 80332),
    "lcls2_2x70x512": (80408, 80216, 80132, 80416),
    "dense_96x1024": (80416, 80232, 80332),
    "tiny_185x388": (21308, 20432, 20832),
    "narrow_5x60_s30": (20132, 20232),
    "single_segment_40x256": (80408, 80132, 80216),
}


@pytest.mark.parametrize("cm_mode", [0, 1], ids=["median", "mean"])
@pytest.mark.parametrize("case", list(VARIANTS), ids=list(VARIANTS))
def test_chain_layout_variants(oracle, case, cm_mode):
    cfg, n = CASES[case]
    n = 2 * n + 1
    raw, ped, gain = make(cfg, n)
    o = oracle_run(oracle, cfg, raw, ped, gain, cm_mode)
    ref = None
    for variant in VARIANTS[case]:
        g = gpu_run(cfg, raw, ped, gain, cm_mode, kernel="chain", variant=variant)
        rep = compare(o, g, panels=cfg.panels, rows=cfg.rows, cols=cfg.cols, seg_cols=cfg.seg_cols, cm_adu=cfg.cm_adu)
        print(case, cm_mode, variant, g["kernel"], rep.summary())
        assert rep.ok, (variant, rep.failures[:10])
        assert "%d,%d,%d" % (variant // 10000, variant // 100 % 100, variant % 100) in g["kernel"]
        if ref is None:
            ref = g
        elif cm_mode == 0:    # the median is an order statistic: identical in every layout
            for k in ("hit_count", "hit_pixel", "hit_charge", "hit_nphot", "hit_dx", "hit_dy", "frame_photons", "accum"):
                assert np.array_equal(ref[k], g[k]), (variant, k)


@pytest.mark.parametrize("kernel,variant", [("chain", 0), ("chain", 80316), ("chain", 80232), ("lookback", 0)])
@pytest.mark.parametrize("cm_mode", [0, 1], ids=["median", "mean"])
def test_common_mode_values(oracle, cm_mode, kernel, variant):
    """c of every segment against the oracle: the kernel's fp32 order statistic / mean."""
    cfg, n = small(1, rows=64), 5
    raw, ped, gain = make(cfg, n)
    g = gpu_run(cfg, raw, ped, gain, cm_mode, keep_cm=True, kernel=kernel, variant=variant)
    o = oracle.process(raw.cpu().numpy(), ped.cpu().numpy(), gain.cpu().numpy(), panels=1, rows=cfg.rows,
                       cols=cfg.cols, seg_cols=cfg.seg_cols, seed_adu=50, cm_adu=20, photon_adu=80,
                       cm_mode=cm_mode, want_cm=True, want_fragile=True)
    cm_o = o.cm.reshape(g["cm"].shape)
    frag_seg = (o.fragile.reshape(n, 1, cfg.rows, cfg.cols // cfg.seg_cols, cfg.seg_cols) & 1).any(-1)
    err = np.abs(g["cm"] - cm_o)[~frag_seg]
    assert err.max() < 1e-5, err.max()                # |c_gpu - c_oracle| <= ~7e-6


def test_integer_exact_suite(oracle):
    """Integer pedestals, power-of-two gains, thresholds at x.5: fp32 == fp64, frequent ties,
    nothing can sit within 1e-4 of a threshold => ZERO exemptions allowed."""
    rng = np.random.default_rng(3)
    P, H, W, S, n = 2, 37, 96, 48, 12
    ped = torch.tensor(rng.integers(900, 1100, (P, H, W)).astype(np.float32))
    gain = torch.tensor(rng.choice([0.5, 1.0, 2.0], (P, H, W)).astype(np.float32))
    sig = rng.integers(-6, 7, (n, P, H, W)) * 2 + rng.integers(-3, 4, (n, P, H, W // S)).repeat(S, -1) * 2
    ph = rng.random((n, P, H, W)) < 0.02
    sig = sig + ph * rng.choice([40, 60, 60, 80, 150, 250], (n, P, H, W))
    ph2 = np.roll(ph, 1, -1) | np.roll(ph, 1, -2)
    sig = sig + ph2 * rng.choice([0, 20, 60], (n, P, H, W))                  # neighbours, ties
    raw = torch.tensor((ped.numpy() + gain.numpy() * sig).astype(np.uint16))
    cfg = small(0, panels=P, rows=H, cols=W, seg_cols=S, seed_adu=50.5, cm_adu=20.5, photon_adu=100.0)
    for cm_mode, kernel, variant in ((0, "chain", 0), (1, "chain", 0), (2, "chain", 0), (0, "lookback", 0), (2, "lookback", 0),
                                     (0, "chain", 80132), (0, "chain", 80216), (1, "chain", 80216)):
        g = gpu_run(cfg, raw.to(DEV), ped, gain, cm_mode, kernel=kernel, variant=variant)
        o = oracle_run(oracle, cfg, raw, ped, gain, cm_mode)
        rep = compare(o, g, panels=P, rows=H, cols=W, seg_cols=S, cm_adu=cfg.cm_adu)
        print(cm_mode, kernel, rep.summary())
        assert rep.ok, rep.failures[:10]
        if cm_mode != 1:
            # exact ties (F3) and exact half-integers (F4) do occur here, and must still match exactly
            assert rep.exempt_hits == 0 and (o.fragile & 3).max() == 0
            assert rep.max_err["E"] == 0.0
        assert rep.hits_oracle > 200


@pytest.mark.parametrize("kernel", ["chain", "lookback"])
def test_overflow_and_empty(oracle, kernel):
    cfg, n = small(0, rows=40, cols=128, seg_cols=64, occupancy=0.03), 3
    raw, ped, gain = make(cfg, n)
    full = gpu_run(cfg, raw, ped, gain, 0, kernel=kernel)
    cap = int(full["hit_count"].min()) // 2
    g = gpu_run(cfg, raw, ped, gain, 0, cap=cap, kernel=kernel)
    assert g["status"][0] & 1
    assert np.array_equal(g["hit_count"], full["hit_count"])                 # true counts
    assert np.array_equal(g["frame_photons"], full["frame_photons"])         # totals over ALL hits
    assert np.array_equal(g["accum"], full["accum"])
    assert np.array_equal(g["hit_pixel"][:, :cap], full["hit_pixel"][:, :cap])
    assert np.array_equal(g["hit_charge"][:, :cap], full["hit_charge"][:, :cap])
    # zero frames: a no-op
    ctx = binding.Context(panels=1, rows=40, cols=128, seg_cols=64, max_frames_per_batch=4, pedestal=ped.cpu(),
                          gain=gain.cpu(), seed_adu=50, cm_adu=20, photon_adu=100)
    out = binding.alloc_output(1, cfg.npix, 8, DEV)
    ctx.process(raw[:0], out, n_frames=0)
    torch.cuda.synchronize()
    assert ctx.last_launch_count == 0 and int(out.accum.sum()) == 0
    with pytest.raises(binding.PdpError):
        ctx.process(raw, out, n_frames=5)                                    # > max_frames_per_batch
    ctx.close()


def test_chunking_determinism_accumulation_and_host_feed(oracle):
    cfg, n = small(0, rows=50, cols=128, seg_cols=64, occupancy=0.02), 21
    raw, ped, gain = make(cfg, n)
    OUT = ("hit_count", "hit_pixel", "hit_charge", "hit_nphot", "hit_dx", "hit_dy", "frame_photons", "accum", "status")
    ref = gpu_run(cfg, raw, ped, gain, 0, kernel="chain")
    again = gpu_run(cfg, raw, ped, gain, 0, kernel="chain")
    for k in OUT:
        assert np.array_equal(ref[k], again[k]), k                           # bit-identical run to run
    small_k = gpu_run(cfg, raw, ped, gain, 0, kernel="lookback")
    chunked = gpu_run(cfg, raw, ped, gain, 0, kernel="lookback", chunk_frames=4)   # 6 chunks, ragged last one
    for k in OUT:
        assert np.array_equal(small_k[k], chunked[k]), k
    # the two kernels calibrate with different (equally accurate) fp32 formulas: same hits, floats within tolerance
    for k in ("hit_count", "hit_pixel", "hit_nphot", "frame_photons", "accum"):
        assert np.array_equal(ref[k], small_k[k]), k
    twice = gpu_run(cfg, raw, ped, gain, 0, n_calls=2, kernel="chain")        # accum persists across calls
    assert np.array_equal(twice["accum"], 2 * ref["accum"])
    twice = gpu_run(cfg, raw, ped, gain, 0, n_calls=2, kernel="lookback")
    assert np.array_equal(twice["accum"], 2 * ref["accum"])
    host = gpu_run(cfg, raw, ped, gain, 0, host_chunk=8, kernel="chain")     # 3 chunks through the side stream
    for k in OUT:
        assert np.array_equal(ref[k], host[k]), k
    assert host["launches"] == 3 * LAUNCHES["chain"]
    o = oracle_run(oracle, cfg, raw, ped, gain, 0)
    assert compare(o, ref, panels=1, rows=cfg.rows, cols=cfg.cols, seg_cols=cfg.seg_cols, cm_adu=cfg.cm_adu).ok


def test_occupancy_independence_of_lists(oracle):
    """Noise-only frames: zero hits, zero accum (sigma far below threshold)."""
    cfg = small(0, occupancy=0.0)
    raw, ped, gain = make(cfg, 4)
    g = gpu_run(cfg, raw, ped, gain, 0)
    assert g["hit_count"].sum() == 0 and g["accum"].sum() == 0 and g["frame_photons"].sum() == 0


@pytest.mark.parametrize("cm_mode", [0, 1], ids=["median", "mean"])
def test_many_frames_dense(oracle, cm_mode):
    cfg, n = small(3, rows=50, cols=256, seg_cols=128), 300     # dense, wide clouds: many non-maximum candidates
    raw, ped, gain = make(cfg, n)
    g = gpu_run(cfg, raw, ped, gain, cm_mode, sparse_warps=8)
    o = oracle_run(oracle, cfg, raw, ped, gain, cm_mode)
    rep = compare(o, g, panels=cfg.panels, rows=cfg.rows, cols=cfg.cols, seg_cols=cfg.seg_cols, cm_adu=cfg.cm_adu)
    print(rep.summary())
    assert rep.ok, rep.failures[:10]
    assert rep.hits_oracle > 10000 and rep.exempt_hits <= rep.hits_oracle // 200


@pytest.mark.parametrize("path", ["chain", "lookback", "staged"])
def test_process_path_allocates_nothing(path):
    """include/pdp.h: no allocation on the pdp_process path.  The workspaces are taken in pdp_create (throughput
    kernel: seed scratch, density hint) and pdp_set_cm_stages (working image): the device's free memory is the
    same before the first pdp_process call and after it."""
    cfg, n = small(0, panels=2, occupancy=0.02), 160
    raw, ped, gain = make(cfg, n)
    ctx = binding.Context(panels=cfg.panels, rows=cfg.rows, cols=cfg.cols, seg_cols=cfg.seg_cols, max_frames_per_batch=n,
                          pedestal=ped.cpu(), gain=gain.cpu(), seed_adu=cfg.seed_adu, cm_adu=cfg.cm_adu,
                          photon_adu=cfg.photon_adu, cm_mode=0)
    if path == "staged":
        ctx.set_cm_stages([(1, cfg.seg_cols, 1), (cfg.rows, 1, 1)])
    else:
        ctx.debug_set("kernel", KERNELS[path])
    out = binding.alloc_output(n, cfg.npix, cfg.max_hits, DEV)
    torch.cuda.synchronize()
    free0, _ = torch.cuda.mem_get_info()
    for _ in range(2):
        ctx.process(raw, out)
    torch.cuda.synchronize()
    free1, _ = torch.cuda.mem_get_info()
    assert free1 == free0, (free0, free1)
    assert int((out.hit_count.to(torch.int64) & 0xFFFFFFFF).sum()) > 1000
    ctx.close()


def test_set_params_switches_estimator_and_layout(oracle):
    """One context, estimator changed with pdp_set_params: the throughput kernel's layout preference depends on the
    estimator (194-pixel segments: <2,13,8> for the median, <2,7,16> otherwise), so the plans are rebuilt; every call
    must match the oracle for the estimator in force.  The second call of each estimator runs with the sparse-warp
    count chosen from the first call's hit density and must give the same lists."""
    cfg, n = small(0, panels=2, occupancy=0.02), 160
    raw, ped, gain = make(cfg, n)
    ctx = binding.Context(panels=cfg.panels, rows=cfg.rows, cols=cfg.cols, seg_cols=cfg.seg_cols, max_frames_per_batch=n,
                          pedestal=ped.cpu(), gain=gain.cpu(), seed_adu=cfg.seed_adu, cm_adu=cfg.cm_adu,
                          photon_adu=cfg.photon_adu, cm_mode=0)
    names = {}
    for cm_mode in (0, 1, 0, 2):
        ctx.set_params(seed_adu=cfg.seed_adu, cm_adu=cfg.cm_adu, photon_adu=cfg.photon_adu, cm_mode=cm_mode)
        o = oracle_run(oracle, cfg, raw, ped, gain, cm_mode)
        prev = None
        for call in range(2):
            out = binding.alloc_output(n, cfg.npix, cfg.max_hits, DEV)
            ctx.process(raw, out)
            torch.cuda.synchronize()
            g = {k: getattr(out, k).cpu().numpy() for k in
                 ("hit_count", "hit_pixel", "hit_charge", "hit_nphot", "hit_dx", "hit_dy", "frame_photons", "accum", "status")}
            g["hit_count"] = g["hit_count"].astype(np.int64) & 0xFFFFFFFF
            g["frame_photons"] = g["frame_photons"].astype(np.int64) & 0xFFFFFFFF
            rep = compare(o, g, panels=cfg.panels, rows=cfg.rows, cols=cfg.cols, seg_cols=cfg.seg_cols, cm_adu=cfg.cm_adu)
            assert rep.ok, (cm_mode, call, rep.failures[:10])
            if prev is not None:
                for k in g:
                    assert np.array_equal(prev[k], g[k]), (cm_mode, k)
            prev = g
        names[cm_mode] = ctx.last_kernel_name
    ctx.close()
    assert names[0] == "pdp_chain_kernel<2,13,8,0>" and names[1] == "pdp_chain_kernel<2,7,16,1>" \
        and names[2] == "pdp_chain_kernel<2,7,16,2>", names


@pytest.mark.parametrize("cm_mode", [0, 1], ids=["median", "mean"])
def test_many_frames_auto_kernel(oracle, cm_mode):
    """More frames than SMs: the library picks the frame-owner kernel, every CTA owns ~3 frames
    and walks all bands for them (ragged last band, two panels)."""
    cfg, n = small(0, panels=2, rows=43, cols=128, seg_cols=64, occupancy=0.02), 437
    raw, ped, gain = make(cfg, n)
    g = gpu_run(cfg, raw, ped, gain, cm_mode)
    o = oracle_run(oracle, cfg, raw, ped, gain, cm_mode)
    rep = compare(o, g, panels=cfg.panels, rows=cfg.rows, cols=cfg.cols, seg_cols=cfg.seg_cols, cm_adu=cfg.cm_adu)
    print(rep.summary())
    assert rep.ok, rep.failures[:10]
    assert rep.hits_oracle > 10000 and rep.exempt_hits <= rep.hits_oracle // 200


def _gpu_invariants(out, cfg, n):
    """Any-size invariants over ALL frames, evaluated on the device (the lists of the big configs are GBs):
    strictly increasing pixel lists, frame_photons == sum of listed n, accum == scatter of all lists."""
    cap = out.hit_capacity
    hc = out.hit_count.to(torch.int64) & 0xFFFFFFFF
    assert int(hc.max()) <= cap and int(out.status.item()) == 0
    for f0 in range(0, n, 64):                                  # blocks of frames bound the temporaries
        f1 = min(n, f0 + 64)
        k = torch.arange(cap, device=hc.device)[None, :] < hc[f0:f1, None]
        px = out.hit_pixel[f0:f1].to(torch.int64) & 0xFFFFFFFF
        assert bool(((px[:, 1:] > px[:, :-1]) | ~k[:, 1:]).all()), "lists not strictly increasing"
        assert bool((px[k] < cfg.npix).all())
        nph = torch.where(k, out.hit_nphot[f0:f1], 0).to(torch.int64)
        assert torch.equal(nph.sum(1), out.frame_photons[f0:f1].to(torch.int64) & 0xFFFFFFFF)
        if f0 == 0:
            acc = torch.zeros(cfg.npix, dtype=torch.int64, device=hc.device)
        acc.index_add_(0, px[k], nph[k])
    assert torch.equal(acc, out.accum.to(torch.int64) & 0xFFFFFFFF), "accum != scatter of all lists"
    return hc


def _full_size_sampled(oracle, cfg_id, cm_mode, min_hits, *, host_chunk=None, extra_sample=()):
    """One BASELINE.json config at FULL size in the launch configuration bench.py times (one pdp_process
    call over all frames, auto kernel choice, capacity chosen like the bench does): frames sampled at the
    start, the end and around CTA / chunk ownership boundaries are compared hit by hit with the oracle;
    invariants that hold at any size cover every frame."""
    cfg = synth.CONFIGS[cfg_id]
    n = cfg.n_frames
    raw, ped, gain = make(cfg, n)
    ctx = binding.Context(panels=cfg.panels, rows=cfg.rows, cols=cfg.cols, seg_cols=cfg.seg_cols,
                          max_frames_per_batch=n, pedestal=ped.cpu(), gain=gain.cpu(), seed_adu=cfg.seed_adu,
                          cm_adu=cfg.cm_adu, photon_adu=cfg.photon_adu, cm_mode=cm_mode)
    probe = binding.alloc_output(8, cfg.npix, cfg.max_hits, DEV)
    ctx.process(raw[:8], probe)
    torch.cuda.synchronize()
    cap = min(cfg.max_hits, max(256, 4 * int(probe.hit_count.max())))
    del probe
    out = binding.alloc_output(n, cfg.npix, cap, DEV)
    if host_chunk:
        try:
            host = torch.empty(raw.shape, dtype=torch.uint16).pin_memory()
        except RuntimeError:                                     # the box cannot pin the whole batch
            host = torch.empty(raw.shape, dtype=torch.uint16)
        host.copy_(raw)
        ctx.process_host(host, out, host_chunk)
    else:
        ctx.process(raw, out)
    torch.cuda.synchronize()
    launches = ctx.last_launch_count
    assert launches == (-(-n // host_chunk) if host_chunk else 1) * LAUNCHES_PER_CALL
    hc = _gpu_invariants(out, cfg, n)
    per_cta = n / 148.0
    sample = {0, 1, n // 2, n - 2, n - 1}
    for b in (1, 2, 74, 147):                                    # last/first frames of neighbouring CTAs
        e = int(b * per_cta)
        sample |= {max(0, e - 1), e, min(n - 1, e + 1)}
    sample |= {15, 16, 17} if per_cta > 16 else set()            # chunk boundary inside a CTA's range
    sample = sorted(x for x in sample | set(extra_sample) if 0 <= x < n)
    assert len(sample) >= 12
    idx = torch.tensor(sample, device=raw.device)
    picked = raw.view(torch.int16)[idx].view(torch.uint16)       # uint16 has no index kernel
    o = oracle_run(oracle, cfg, picked, ped, gain, cm_mode)
    g = {k: getattr(out, k)[idx].cpu().numpy() for k in ("hit_count", "hit_pixel", "hit_charge", "hit_nphot",
                                                          "hit_dx", "hit_dy", "frame_photons")}
    g["hit_count"] = g["hit_count"].astype(np.int64) & 0xFFFFFFFF
    g["frame_photons"] = g["frame_photons"].astype(np.int64) & 0xFFFFFFFF
    g["accum"] = np.zeros(1, np.int32)
    rep = compare(o, g, panels=cfg.panels, rows=cfg.rows, cols=cfg.cols, seg_cols=cfg.seg_cols, cm_adu=cfg.cm_adu,
                  check_accum=False)
    print(cfg.name, "cm", cm_mode, "cap", cap, "hits/frame %.0f" % float(hc.double().mean()), rep.summary())
    ctx.close()
    assert rep.ok, rep.failures[:10]
    assert rep.hits_oracle > min_hits and rep.exempt_hits <= max(3, rep.hits_oracle // 200)


def test_full_size_config1_sampled(oracle):
    """configs[1]: 2000 frames of 704x768 (13.5 frames per CTA)."""
    _full_size_sampled(oracle, 1, 0, 3000)


def test_full_size_config2_sampled(oracle):
    """configs[2]: 500 frames of 32 panels x 185x388 (S = 194: 4-byte vectors, frames only 8-byte aligned,
    3.4 frames per CTA, panel edges every 185 rows)."""
    _full_size_sampled(oracle, 2, 0, 30000)


def test_full_size_config3_sampled(oracle):
    """configs[3]: 500 frames of 1024x1024 at 10 % occupancy (42 k hits per frame: the sparse stage and the
    ordered emission under real load)."""
    _full_size_sampled(oracle, 3, 0, 400000)


@pytest.mark.parametrize("host", [False, True], ids=["device", "streamed"])
def test_full_size_config4_sampled(oracle, host):
    """configs[4]: 4000 frames of 16 panels x 512x512 (33.5 GB, 27 frames per CTA: multi-chunk path), device
    resident and streamed from (pinned) host memory in 296-frame chunks (2 frames per CTA and chunk, 2.5 GB per copy)
    through the double-buffered side stream."""
    _full_size_sampled(oracle, 4, 0, 150000, host_chunk=296 if host else None)


@pytest.mark.parametrize("n", [148 * 6 + 3, 148 * 17, 148 * 20, 148 * 24 + 5, 148 * 33],
                         ids=["6perCTA", "17perCTA", "20perCTA", "24perCTA", "33perCTA"])
def test_frames_per_cta_paths(oracle, n):
    """Every frame against the oracle on a small, DENSE geometry with 6 ... 33 frames per CTA: partial
    frame groups, a second and third chunk of frame slots per CTA (ring reuse, barrier phase carry-over),
    a short last chunk (slot ownership must not change between chunks), with the sparse
    stage as the bottleneck (5 % of the pixels are photon centres)."""
    cfg = small(0, panels=2, rows=21, cols=128, seg_cols=64, occupancy=0.05)
    raw, ped, gain = make(cfg, n)
    for cm_mode in (0, 1):
        g = gpu_run(cfg, raw, ped, gain, cm_mode)
        o = oracle_run(oracle, cfg, raw, ped, gain, cm_mode)
        rep = compare(o, g, panels=cfg.panels, rows=cfg.rows, cols=cfg.cols, seg_cols=cfg.seg_cols, cm_adu=cfg.cm_adu)
        print(n, cm_mode, rep.summary())
        assert rep.ok, rep.failures[:10]
        assert rep.hits_oracle > 100 * n and rep.exempt_hits <= max(3, rep.hits_oracle // 200)


def test_full_size_config0(oracle):
    """configs[0] at full size (100 frames of 185x388, S = 194: padded lanes, 4-byte vectors), every frame."""
    cfg, n = small(0), 100
    raw, ped, gain = make(cfg, n)
    for cm_mode in (0, 1):
        g = gpu_run(cfg, raw, ped, gain, cm_mode)
        o = oracle_run(oracle, cfg, raw, ped, gain, cm_mode)
        rep = compare(o, g, panels=cfg.panels, rows=cfg.rows, cols=cfg.cols, seg_cols=cfg.seg_cols, cm_adu=cfg.cm_adu)
        print(rep.summary())
        assert rep.ok, rep.failures[:10]
        assert rep.hits_oracle > 20000 and rep.exempt_hits <= rep.hits_oracle // 200


@pytest.mark.parametrize("kernel", ["chain", "lookback"])
def test_seed_threshold_below_mask_threshold(oracle, kernel):
    """T_seed < T_cm: pixels INSIDE the common-mode mask can seed (the kernels' rare 'low' candidate path)."""
    cfg, n = small(0, rows=40, cols=256, seg_cols=128, occupancy=0.01, photon_adu=30.0, seed_adu=12.0), 80
    raw, ped, gain = make(cfg, n)
    for cm_mode in (0, 1):
        g = gpu_run(cfg, raw, ped, gain, cm_mode, kernel=kernel)
        o = oracle_run(oracle, cfg, raw, ped, gain, cm_mode)
        rep = compare(o, g, panels=cfg.panels, rows=cfg.rows, cols=cfg.cols, seg_cols=cfg.seg_cols, cm_adu=cfg.cm_adu)
        print(rep.summary())
        assert rep.ok, rep.failures[:10]
        assert rep.hits_oracle > 2000 and rep.exempt_hits <= max(3, rep.hits_oracle // 200)


def test_wide_gain_range_and_min_count(oracle):
    """Gains from 0.25 to 4 (BIG grows with max |v1|), and a cm_min_count that most segments miss (c = 0)."""
    cfg, n = small(4, panels=1, rows=48, gain_lo=0.25, gain_hi=4.0), 90
    raw, ped, gain = make(cfg, n)
    for cm_min_count in (0, 250):
        g = gpu_run(cfg, raw, ped, gain, 0, cm_min_count=cm_min_count, kernel="chain")
        o = oracle_run(oracle, cfg, raw, ped, gain, 0, cm_min_count=cm_min_count)
        rep = compare(o, g, panels=cfg.panels, rows=cfg.rows, cols=cfg.cols, seg_cols=cfg.seg_cols, cm_adu=cfg.cm_adu)
        print(cm_min_count, rep.summary())
        assert rep.ok, rep.failures[:10]
        assert rep.hits_oracle > 1000 and rep.exempt_hits <= max(3, rep.hits_oracle // 200)


def test_wide_panel(oracle):
    """W = 1280 (40 bitmap words per row, S = 640: padded lane runs) on the throughput kernel."""
    cfg, n = small(0, rows=24, cols=1280, seg_cols=640, occupancy=0.004), 90
    raw, ped, gain = make(cfg, n)
    g = gpu_run(cfg, raw, ped, gain, 0)                 # auto choice
    o = oracle_run(oracle, cfg, raw, ped, gain, 0)
    rep = compare(o, g, panels=cfg.panels, rows=cfg.rows, cols=cfg.cols, seg_cols=cfg.seg_cols, cm_adu=cfg.cm_adu)
    print(rep.summary())
    assert rep.ok, rep.failures[:10]
    assert rep.hits_oracle > 3000 and g["kernel"].startswith("pdp_chain_kernel")
    with pytest.raises(binding.PdpError):
        gpu_run(cfg, raw, ped, gain, 0, kernel="chain", variant=80608)   # a layout that cannot cover S = 640 must fail loudly


def test_histograms(oracle):
    """NEXT-2: energy spectrum and centroid histograms of the finished lists.  Bit-exact
    against the oracle's histogram function applied to the SAME lists (the bin rule is evaluated in double on the
    stored float32 values on both sides), and, against the oracle's own hits, equal except for hits whose value
    lies within the float tolerance of a bin edge."""
    cfg, n = small(0, rows=60, cols=128, seg_cols=64, occupancy=0.03), 200
    raw, ped, gain = make(cfg, n)
    ctx = binding.Context(panels=cfg.panels, rows=cfg.rows, cols=cfg.cols, seg_cols=cfg.seg_cols, max_frames_per_batch=n,
                          pedestal=ped.cpu(), gain=gain.cpu(), seed_adu=cfg.seed_adu, cm_adu=cfg.cm_adu, photon_adu=cfg.photon_adu)
    out = binding.alloc_output(n, cfg.npix, cfg.max_hits, DEV)
    ctx.process(raw, out)
    e_spec, d_spec = (20.0, 2.5, 96), (-1.0, 0.03125, 64)
    he = torch.zeros(e_spec[2], dtype=torch.int32, device=DEV)
    hx = torch.zeros(d_spec[2], dtype=torch.int32, device=DEV)
    hy = torch.zeros(d_spec[2], dtype=torch.int32, device=DEV)
    for _ in range(2):                                                   # += semantics: two calls double every bin
        ctx.histograms(out, n, energy=e_spec, dxy=d_spec, hist_energy=he, hist_dx=hx, hist_dy=hy)
    torch.cuda.synchronize()
    assert ctx.last_launch_count == 2
    hc = out.hit_count.cpu().numpy().astype(np.int64)
    k = np.arange(out.hit_capacity)[None, :] < hc[:, None]
    E, X, Y = (getattr(out, f).cpu().numpy()[k].astype(np.float64) for f in ("hit_charge", "hit_dx", "hit_dy"))
    assert np.array_equal(he.cpu().numpy(), 2 * oracle.histogram(E, *e_spec).astype(np.int64))
    assert np.array_equal(hx.cpu().numpy(), 2 * oracle.histogram(X, *d_spec).astype(np.int64))
    assert np.array_equal(hy.cpu().numpy(), 2 * oracle.histogram(Y, *d_spec).astype(np.int64))
    assert he.sum() > 2 * 0.9 * hc.sum()                                # the spectrum window holds nearly every hit
    # against the oracle's own hit values: identical up to hits within 1e-4 (+1e-4 rel.) of a bin edge
    o = oracle_run(oracle, cfg, raw, ped, gain, 0)
    oE = np.concatenate(o.hit_charge)
    want = oracle.histogram(oE, *e_spec).astype(np.int64)
    edge = np.abs((oE - e_spec[0]) / e_spec[1] - np.rint((oE - e_spec[0]) / e_spec[1])) * e_spec[1] < 1e-4 + 1e-4 * np.abs(oE)
    assert np.abs(he.cpu().numpy() // 2 - want).sum() <= 2 * int(edge.sum()) + 2 * (len(oE) - int(hc.sum())) ** 2
    # only one of the two specs: the other histograms stay untouched
    he2 = torch.zeros_like(he)
    ctx.histograms(out, n, energy=e_spec, hist_energy=he2)
    torch.cuda.synchronize()
    assert np.array_equal(2 * he2.cpu().numpy(), he.cpu().numpy())
    ctx.close()


@pytest.mark.parametrize("cm_mode", [0, 1, 2], ids=["median", "mean", "none"])
@pytest.mark.parametrize("case", ["epix_704x768", "tiny_185x388", "dense_96x1024", "ragged_2x11x72_s24"])
def test_dense_photon_counting(oracle, case, cm_mode):
    """NEXT-4: per-pixel divide-and-round photon counting, image summed over the frames and
    per-frame totals, bit-exact against the oracle except at pixels it flags (v2/E_ph within 1e-4 ADU of a rounding
    boundary or of the zeroing threshold, or a mask pixel about to flip in the pixel's row segment)."""
    cfg, n = CASES[case]
    n = 3 * n
    raw, ped, gain = make(cfg, n)
    for zero_below in (float("-inf"), 30.0):
        ctx = binding.Context(panels=cfg.panels, rows=cfg.rows, cols=cfg.cols, seg_cols=cfg.seg_cols, max_frames_per_batch=n,
                              pedestal=ped.cpu(), gain=gain.cpu(), seed_adu=cfg.seed_adu, cm_adu=cfg.cm_adu,
                              photon_adu=cfg.photon_adu, cm_mode=cm_mode)
        img = torch.zeros(cfg.npix, dtype=torch.int32, device=DEV)
        tot = torch.zeros(n, dtype=torch.int32, device=DEV)
        ctx.process_dense(raw, img, tot, zero_below_adu=zero_below)
        ctx.process_dense(raw, img, None, zero_below_adu=zero_below)          # += : twice the image, totals optional
        torch.cuda.synchronize()
        assert ctx.last_kernel_name.startswith("pdp_dense_kernel")
        ctx.close()
        o_img, o_tot, frag = oracle.dense(raw.cpu().numpy(), ped.cpu().numpy(), gain.cpu().numpy(), panels=cfg.panels,
                                          rows=cfg.rows, cols=cfg.cols, seg_cols=cfg.seg_cols, cm_adu=cfg.cm_adu,
                                          photon_adu=cfg.photon_adu, cm_mode=cm_mode, zero_below_adu=zero_below,
                                          want_fragile=True)
        g_img = img.cpu().numpy().astype(np.int64)
        assert np.all(g_img % 2 == 0)
        diff = g_img // 2 != o_img.astype(np.int64)
        fragile_px = frag.any(axis=0)
        print(case, cm_mode, zero_below, "photons", int(o_img.sum()), "pixels differing", int(diff.sum()), "fragile pixels", int(fragile_px.sum()))
        assert o_img.sum() > 5 * n
        assert not (diff & ~fragile_px).any()                              # differences only where the oracle says fragile
        assert diff.sum() <= max(3, int(fragile_px.sum()))
        clean = ~frag.reshape(n, -1).any(axis=1)                           # frames without any fragile pixel: exact totals
        assert np.array_equal(tot.cpu().numpy().astype(np.int64)[clean], o_tot.astype(np.int64)[clean])
        assert np.abs(tot.cpu().numpy().astype(np.int64) - o_tot.astype(np.int64)).max() <= max(3, int(frag.reshape(n, -1).any(axis=1).sum() and frag.sum()))


@pytest.mark.parametrize("cm_mode", [0, 1], ids=["median", "mean"])
def test_dense_photon_counting_sliced(oracle, cm_mode):
    """Few row segments and many frames: the frames of a segment are split into slices that run on different warps
    and accumulate into their own images (merged by pdp_dense_merge_kernel); ragged last slice (301 frames)."""
    cfg, n = small(0, panels=2, rows=12, cols=128, seg_cols=64, occupancy=0.02), 301
    raw, ped, gain = make(cfg, n)
    ctx = binding.Context(panels=cfg.panels, rows=cfg.rows, cols=cfg.cols, seg_cols=cfg.seg_cols, max_frames_per_batch=n,
                          pedestal=ped.cpu(), gain=gain.cpu(), seed_adu=cfg.seed_adu, cm_adu=cfg.cm_adu,
                          photon_adu=cfg.photon_adu, cm_mode=cm_mode)
    img = torch.zeros(cfg.npix, dtype=torch.int32, device=DEV)
    tot = torch.zeros(n, dtype=torch.int32, device=DEV)
    ctx.process_dense(raw, img, tot)
    assert ctx.last_launch_count == 3                                     # counting, slice merge, per-frame totals
    ctx.process_dense(raw, img, None)                                     # += : twice the image
    torch.cuda.synchronize()
    ctx.close()
    o_img, o_tot, frag = oracle.dense(raw.cpu().numpy(), ped.cpu().numpy(), gain.cpu().numpy(), panels=cfg.panels,
                                      rows=cfg.rows, cols=cfg.cols, seg_cols=cfg.seg_cols, cm_adu=cfg.cm_adu,
                                      photon_adu=cfg.photon_adu, cm_mode=cm_mode, zero_below_adu=float("-inf"),
                                      want_fragile=True)
    g_img = img.cpu().numpy().astype(np.int64)
    assert np.all(g_img % 2 == 0)
    diff = g_img // 2 != o_img.astype(np.int64)
    fragile_px = frag.any(axis=0)
    print(cm_mode, "photons", int(o_img.sum()), "pixels differing", int(diff.sum()), "fragile pixels", int(fragile_px.sum()))
    assert o_img.sum() > 5 * n
    assert not (diff & ~fragile_px).any()
    clean = ~frag.reshape(n, -1).any(axis=1)
    assert np.array_equal(tot.cpu().numpy().astype(np.int64)[clean], o_tot.astype(np.int64)[clean])


STAGE_SETS = {
    "row_col_mean": [(1, 64, 1), (8, 1, 1)],
    "paper_3_stacked_mean": [(1, 128, 1), (8, 1, 1), (40, 128, 1)],          # row, column, panel-wise: PAPER.md:L117
    "row_median_block_mean": [(1, 64, 0), (8, 16, 1)],
    "panel_median": [(40, 128, 0)],
    "col_median_then_none": [(10, 1, 0), (1, 128, 2)],
    "narrow_mean_groups": [(2, 2, 1), (8, 4, 1), (40, 1, 1)],
    "median_groups_in_registers": [(4, 128, 0), (20, 32, 0), (8, 128, 0)],   # 512, 640, 1024 pixels: 16, 24, 32 per lane
}


@pytest.mark.parametrize("name", list(STAGE_SETS), ids=list(STAGE_SETS))
def test_stacked_common_mode_stages(oracle, name):
    """NEXT-1: up to three stacked common-mode stages on row, column, block and panel-wise
    groups, mean and median estimators, against the oracle's staged chain: hits bit-exact outside the pixels the
    oracle flags, floats within tolerance."""
    stages = STAGE_SETS[name]
    cfg, n = small(0, panels=2, rows=40, cols=128, seg_cols=64, occupancy=0.01), 9
    raw, ped, gain = make(cfg, n)
    ctx = binding.Context(panels=cfg.panels, rows=cfg.rows, cols=cfg.cols, seg_cols=cfg.seg_cols, max_frames_per_batch=n,
                          pedestal=ped.cpu(), gain=gain.cpu(), seed_adu=cfg.seed_adu, cm_adu=cfg.cm_adu, photon_adu=cfg.photon_adu)
    ctx.set_cm_stages(stages)
    out = binding.alloc_output(n, cfg.npix, cfg.max_hits, DEV)
    ctx.process(raw, out)
    torch.cuda.synchronize()
    assert ctx.last_launch_count == 1 + len(stages) + 1 + 1            # calibrate, stages, finder, accumulated image
    g = {k: getattr(out, k).cpu().numpy() for k in
         ("hit_count", "hit_pixel", "hit_charge", "hit_nphot", "hit_dx", "hit_dy", "frame_photons", "accum", "status")}
    g["hit_count"] = g["hit_count"].astype(np.int64) & 0xFFFFFFFF
    g["frame_photons"] = g["frame_photons"].astype(np.int64) & 0xFFFFFFFF
    o = oracle_run(oracle, cfg, raw, ped, gain, 0, stages=stages)
    rep = compare(o, g, panels=cfg.panels, rows=cfg.rows, cols=cfg.cols, cm_adu=cfg.cm_adu)
    print(name, rep.summary())
    assert rep.ok, rep.failures[:10]
    assert rep.hits_oracle > 300 and rep.exempt_hits <= 3
    # back to the hot path: [] restores the fused single row-segment stage
    ctx.set_cm_stages([])
    out2 = binding.alloc_output(n, cfg.npix, cfg.max_hits, DEV)
    ctx.process(raw, out2)
    torch.cuda.synchronize()
    o1 = oracle_run(oracle, cfg, raw, ped, gain, 0)
    assert np.array_equal(out2.hit_count.cpu().numpy().astype(np.int64), o1.hit_count)
    with pytest.raises(binding.PdpError):
        ctx.set_cm_stages([(7, 128, 1)])                                # does not tile 40 rows
    ctx.close()


def test_stacked_stages_large_groups(oracle):
    """The coalesced guarded-mean kernels on groups that need their large forms: a panel-wise group of 49152 pixels
    (1024-thread CTAs), columns of 256 rows in two column chunks (128 + 64), full rows."""
    stages = [(1, 192, 1), (256, 1, 1), (256, 192, 1)]
    cfg, n = small(0, panels=2, rows=256, cols=192, seg_cols=96, occupancy=0.01), 5
    raw, ped, gain = make(cfg, n)
    ctx = binding.Context(panels=cfg.panels, rows=cfg.rows, cols=cfg.cols, seg_cols=cfg.seg_cols, max_frames_per_batch=n,
                          pedestal=ped.cpu(), gain=gain.cpu(), seed_adu=cfg.seed_adu, cm_adu=cfg.cm_adu, photon_adu=cfg.photon_adu)
    ctx.set_cm_stages(stages)
    out = binding.alloc_output(n, cfg.npix, cfg.max_hits, DEV)
    ctx.process(raw, out)
    torch.cuda.synchronize()
    g = {k: getattr(out, k).cpu().numpy() for k in
         ("hit_count", "hit_pixel", "hit_charge", "hit_nphot", "hit_dx", "hit_dy", "frame_photons", "accum", "status")}
    g["hit_count"] = g["hit_count"].astype(np.int64) & 0xFFFFFFFF
    g["frame_photons"] = g["frame_photons"].astype(np.int64) & 0xFFFFFFFF
    o = oracle_run(oracle, cfg, raw, ped, gain, 0, stages=stages)
    rep = compare(o, g, panels=cfg.panels, rows=cfg.rows, cols=cfg.cols, cm_adu=cfg.cm_adu)
    print(rep.summary())
    assert rep.ok, rep.failures[:10]
    assert rep.hits_oracle > 1000 and rep.exempt_hits <= 5
    ctx.close()
