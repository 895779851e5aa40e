"""GPU parity: the CUDA path (through the C ABI) against the CPU oracle on the
same seeded float32 inputs, element by element.

Bar (BASELINE.json north_star, reading A14): per frame
    max |dI| / max I <= 1e-4   on the detector frame,
    |d slope|        <= 1e-4   per element (absolute),
valid masks bit-exact.  This file holds the small cases and the edge cases; every
frame of the four full-size configs is compared in test_gpu_parity_full.py.
"""
import numpy as np
import pytest

from paper_1607_07624_b200 import workloads as wl

pytestmark = pytest.mark.gpu

TOL_FRAME = 1e-4
TOL_SLOPE = 1e-4


@pytest.fixture(scope="module")
def torch_cuda():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    return torch


def _compare(frames_gpu, slopes_gpu, frames_ref, slopes_ref):
    frames_gpu = np.asarray(frames_gpu, dtype=np.float64)
    slopes_gpu = np.asarray(slopes_gpu, dtype=np.float64)
    assert frames_gpu.shape == frames_ref.shape and slopes_gpu.shape == slopes_ref.shape
    assert np.isfinite(frames_gpu).all() and np.isfinite(slopes_gpu).all()
    worst_f = worst_s = 0.0
    for b in range(frames_ref.shape[0]):
        ef = np.abs(frames_gpu[b] - frames_ref[b]).max() / frames_ref[b].max()
        es = np.abs(slopes_gpu[b] - slopes_ref[b]).max()
        worst_f, worst_s = max(worst_f, ef), max(worst_s, es)
    assert worst_f <= TOL_FRAME, f"frame error {worst_f:.3e} > {TOL_FRAME}"
    assert worst_s <= TOL_SLOPE, f"slope error {worst_s:.3e} > {TOL_SLOPE}"
    return worst_f, worst_s


def _run_both(torch, A, M, r, K, ns, phase, **kw):
    from oracle import pwfs_oracle as orc
    from paper_1607_07624_b200.pwfs import PWFS
    sensor = PWFS(A, M, r, K, ns, **kw)
    try:
        v_ref, nv_ref = orc.valid_mask(A, ns, kw.get("illum_thresh", 0.5))
        assert sensor.n_valid == nv_ref
        assert np.array_equal(sensor.valid_mask(), v_ref)              # bit-exact mask
        fr, sl = sensor.run(torch.from_numpy(phase).cuda())
        torch.cuda.synchronize()
        fr_ref, sl_ref = orc.pwfs_run(A, M, r, K, ns, phase, s=kw.get("mask_shift_px", 0),
                                      theta0=kw.get("mod_angle0", 0.0),
                                      thresh=kw.get("illum_thresh", 0.5),
                                      norm_mode=kw.get("slope_norm", 0))
        return _compare(fr.cpu().numpy(), sl.cpu().numpy(), fr_ref, sl_ref)
    finally:
        sensor.close()


# ------------------------------------------------------------------ configs --
def test_cfg1_every_frame(torch_cuda):
    cfg = wl.CONFIGS["cfg1_tiny"]
    A = wl.make_pupil(cfg)
    phase = wl.phase_batch(cfg)                                         # all 10 steps
    _run_both(torch_cuda, A, cfg.m_grid, cfg.mod_radius, cfg.mod_points, cfg.n_subap, phase)


def test_repeated_frames_and_calls_are_bit_identical(torch_cuda):
    """Every frame of every full-size config is compared with the oracle in test_gpu_parity_full.py; here: the
    result of a frame depends neither on its position in the batch nor on the call (no atomics, fixed orders)."""
    from paper_1607_07624_b200.pwfs import from_config
    torch = torch_cuda
    cfg = wl.CONFIGS["cfg4_elt"]
    phase = wl.phase_batch(cfg, steps=2)
    big = torch.from_numpy(np.concatenate([phase] * 10)).cuda()                    # 20 frames: 2 distinct, repeated
    with from_config(cfg) as sensor:
        fr, sl = sensor.run(big)
        fr2, sl2 = sensor.run(big)
        torch.cuda.synchronize()
        assert torch.equal(fr, fr2) and torch.equal(sl, sl2)
        for i in range(2, 20):
            assert torch.equal(fr[i], fr[i % 2]) and torch.equal(sl[i], sl[i % 2])


@pytest.mark.parametrize("N,M,ns,K,r,kw", [
    (64, 128, 16, 12, 3.0, {}),                                   # cfg1 geometry, quarter mask
    (60, 128, 23, 5, 1.5, {}),                                    # margins, non-integer binning, odd K
    (50, 128, 7, 1, 0.0, {}),                                     # unmodulated, ragged N
    (48, 128, 12, 7, 2.0, dict(mask_shift_px=30, mod_angle0=0.4, illum_thresh=0.3, slope_norm=1)),   # table mask
    (64, 128, 32, 9, 2.5, {}),                                    # largest detector the kernel takes (D = 64)
])
def test_fused_small_grid_kernel_against_oracle_and_two_kernel_path(torch_cuda, monkeypatch, N, M, ns, K, r, kw):
    """M = 128: small batches run the whole path in ONE kernel (pwfs_small.cuh).  It must match the oracle at the
    parity bar, and the two-kernel path (PWFS_SMALL=0) to FP32 summation order; launches are counted per class."""
    from paper_1607_07624_b200.pwfs import PWFS
    torch = torch_cuda
    rng = np.random.default_rng(N * 3 + K)
    c = (np.arange(N) - (N - 1) / 2.0)
    X, Y = np.meshgrid(c, c)
    A = ((np.hypot(X, Y) <= N / 2.0) & (np.hypot(X, Y) >= 0.1 * N)).astype(np.float32)
    phase = (rng.standard_normal((5, N, N)) * 3.0).astype(np.float32)
    phase[1] = wl.tilt_phase(N, 0.3, -0.2)
    monkeypatch.setenv("PWFS_SMALL", "1")
    _run_both(torch, A, M, r, K, ns, phase, **kw)                  # fused kernel vs oracle
    with PWFS(A, M, r, K, ns, **kw) as fused:
        fused.get_timing()
        f1, s1 = fused.run(torch.from_numpy(phase).cuda())
        f1b, s1b = fused.run(torch.from_numpy(phase).cuda())       # second call: completion counters were reset
        fh, sh = fused.run_host(phase)
        _, launches = fused.get_timing()
        assert launches["fused"] == 3 and launches["xpass"] == 0 and launches["ypass"] == 0
        assert torch.equal(f1, f1b) and torch.equal(s1, s1b)
        assert np.array_equal(fh, f1.cpu().numpy()) and np.array_equal(sh, s1.cpu().numpy())
        f1n, _ = fused.run(torch.from_numpy(phase).cuda(), want_slopes=False)
        assert torch.equal(f1, f1n)
    monkeypatch.setenv("PWFS_SMALL", "0")
    with PWFS(A, M, r, K, ns, **kw) as two:
        f2, s2 = two.run(torch.from_numpy(phase).cuda())
        _, launches = two.get_timing()
        assert launches["fused"] == 0 and launches["xpass"] >= 1
    assert ((f1 - f2).abs().amax(dim=(1, 2)) <= 2e-6 * f2.abs().amax(dim=(1, 2))).all()
    assert (s1 - s2).abs().max() <= 1e-5


def test_full_resolution_intensity_before_rebinning(torch_cuda):
    """The un-rebinned I = mean_k |E_k|^2 of the hot path's own kernels (test-only export pwfs_debug_intensity)
    against the oracle's orc_intensity on the whole M x M grid, M = 2N so that every column is computed."""
    from oracle import pwfs_oracle as orc
    from paper_1607_07624_b200.pwfs import PWFS, from_config
    torch = torch_cuda
    cfg = wl.CONFIGS["cfg1_tiny"]
    A = wl.make_pupil(cfg)
    phase = wl.phase_batch(cfg, steps=2)
    with from_config(cfg) as sensor:
        I = sensor.debug_intensity(torch.from_numpy(phase).cuda()).cpu().numpy().astype(np.float64)
    for b in range(2):
        ref = orc.intensity(A, phase[b], cfg.m_grid, cfg.mod_points, cfg.mod_radius)
        assert np.abs(I[b] - ref).max() <= TOL_FRAME * ref.max()
    # a radix-5 grid with a general mask shift (table-mask kernels)
    N, M, s = 80, 160, 44
    rng = np.random.default_rng(3)
    c = np.arange(N) - (N - 1) / 2.0
    X, Y = np.meshgrid(c, c)
    A2 = (np.hypot(X, Y) <= N / 2.0).astype(np.float32)
    ph = (rng.standard_normal((1, N, N)) * 2.0).astype(np.float32)
    with PWFS(A2, M, 1.5, 6, 20, debug_shift_px=s) as sensor:
        I2 = sensor.debug_intensity(torch.from_numpy(ph).cuda()).cpu().numpy().astype(np.float64)[0]
    ref = orc.intensity(A2, ph[0], M, 6, 1.5, s=s)
    # columns outside the two pupil-image windows are not computed (returned as zero): compare the computed ones
    o = M // 2 - N // 2
    cols = np.zeros(M, bool)
    for g in ((M - s) % M, s % M):
        cols[(g + np.arange(N) + o) % M] = True
    assert np.abs(I2[:, cols] - ref[:, cols]).max() <= TOL_FRAME * ref.max()
    assert np.abs(I2[:, ~cols]).max() == 0.0


# -------------------------------------------------------------- edge cases ---
@pytest.mark.parametrize("N,M,ns,K,r", [
    (64, 128, 16, 12, 3.0),      # cfg1 geometry
    (60, 128, 23, 5, 1.5),       # non-integer binning, K % 4 != 0, margins (M > 2N)
    (50, 128, 7, 1, 0.0),        # unmodulated, ragged N (not a multiple of 16 or 32)
    (128, 256, 32, 8, 2.0),      # M = 256
    (250, 512, 50, 6, 2.5),      # M = 512, ragged N
    (300, 640, 30, 4, 1.0),      # M = 640
    (37, 320, 37, 3, 0.7),       # tiny pupil in a large grid, b = 1
    # the other grids M = 32 R1 (radix-3/5/9/27 register stages, odd warp batches NB = 3, 5, 6)
    (80, 160, 20, 4, 1.0),       # R1 = 5
    (90, 192, 18, 6, 1.5),       # R1 = 6, margins
    (144, 288, 24, 4, 2.0),      # R1 = 9
    (190, 384, 38, 3, 1.0),      # R1 = 12
    (288, 576, 36, 4, 2.0),      # R1 = 18
    (380, 768, 76, 3, 1.0),      # R1 = 24
    (432, 864, 54, 2, 1.0),      # R1 = 27
    (470, 960, 47, 2, 1.5),      # R1 = 30, ragged N
    (1000, 2048, 100, 2, 2.0),   # R1 = 64: 64 register points per lane, two rounds of size-32 transforms
    # R1 = 36 ... 60: second round of the size-32 stage with R1 - 32 lanes
    (570, 1152, 57, 2, 1.0), (640, 1280, 64, 2, 1.5), (700, 1440, 70, 2, 1.0), (768, 1536, 96, 2, 2.0),
    (800, 1600, 80, 2, 1.0), (860, 1728, 86, 2, 1.0), (960, 1920, 96, 2, 1.5),
])
def test_geometries(torch_cuda, N, M, ns, K, r):
    rng = np.random.default_rng(N * 7 + M)
    c = (np.arange(N) - (N - 1) / 2.0)
    X, Y = np.meshgrid(c, c)
    A = (np.hypot(X, Y) <= N / 2.0).astype(np.float32)
    phase = (rng.standard_normal((3, N, N)) * 3.0).astype(np.float32)
    phase[1] = wl.tilt_phase(N, 0.3, -0.2)
    _run_both(torch_cuda, A, M, r, K, ns, phase)


def test_options_shift_angle_threshold_norm(torch_cuda):
    N, M, ns = 48, 128, 12
    rng = np.random.default_rng(5)
    A = (rng.random((N, N)) > 0.15).astype(np.float32) * (0.5 + rng.random((N, N))).astype(np.float32)
    phase = (rng.standard_normal((2, N, N)) * 2.0).astype(np.float32)
    _run_both(torch_cuda, A, M, 2.0, 7, ns, phase, mask_shift_px=30, mod_angle0=0.4,
              illum_thresh=0.3, slope_norm=1)
    _run_both(torch_cuda, A, M, 2.0, 7, ns, phase, mask_shift_px=24, mod_angle0=-1.1)


def test_large_phase_values_are_range_reduced(torch_cuda):
    cfg = wl.CONFIGS["cfg1_tiny"]
    A = wl.make_pupil(cfg)
    phase = wl.phase_batch(cfg, steps=2) * 8.0                          # ~ +-500 rad
    assert np.abs(phase).max() > 200
    _run_both(torch_cuda, A, cfg.m_grid, cfg.mod_radius, cfg.mod_points, cfg.n_subap,
              phase.astype(np.float32))


def test_empty_batch_and_single_frame(torch_cuda):
    from paper_1607_07624_b200.pwfs import from_config
    torch = torch_cuda
    cfg = wl.CONFIGS["cfg1_tiny"]
    sensor = from_config(cfg)
    try:
        fr, sl = sensor.run(torch.empty((0, cfg.n_pupil, cfg.n_pupil), dtype=torch.float32, device="cuda"))
        assert fr.shape == (0, cfg.det_size, cfg.det_size) and sl.shape == (0, 2 * sensor.n_valid)
        ph = torch.from_numpy(wl.phase_batch(cfg, steps=1)[0]).cuda()   # [N,N]
        fr1, sl1 = sensor.run(ph)
        assert fr1.shape == (1, cfg.det_size, cfg.det_size)
        fr2, _ = sensor.run(ph, want_slopes=False)
        assert torch.equal(fr1, fr2)
    finally:
        sensor.close()


def test_schedule_knobs_do_not_change_results(torch_cuda):
    from paper_1607_07624_b200.pwfs import from_config
    torch = torch_cuda
    cfg = wl.CONFIGS["cfg1_tiny"]
    phase = torch.from_numpy(wl.phase_batch(cfg, steps=7)).cuda()
    sensor = from_config(cfg)
    try:
        base_f, base_s = sensor.run(phase)
        for fpc, ks in [(1, 1), (3, 2), (7, 4), (2, 12)]:
            sensor.set_schedule(fpc, ks)
            f, s = sensor.run(phase)
            assert (f - base_f).abs().max() <= 2e-6 * base_f.abs().max()
            assert (s - base_s).abs().max() <= 1e-5
    finally:
        sensor.close()


def test_host_buffer_pipeline_with_several_chunks(torch_cuda, monkeypatch):
    """B >= 16: pwfs_run_host works in a short first chunk and three large ones on three streams (copy-in, kernels,
    tail + copy-out); every frame must come out as on the device path (FP32 summation order aside)."""
    from paper_1607_07624_b200.pwfs import from_config
    torch = torch_cuda
    monkeypatch.setenv("PWFS_SMALL", "0")                          # cfg1 would otherwise take the fused single-kernel path
    cfg = wl.CONFIGS["cfg1_tiny"]
    phase = np.concatenate([wl.phase_batch(cfg, steps=10)] * 5)[:47]                # ragged: 2 + 15 + 15 + 15
    phase = np.ascontiguousarray(phase + np.arange(47, dtype=np.float32)[:, None, None] * 0.01)   # all frames differ
    with from_config(cfg) as sensor:
        fd, sd = sensor.run(torch.from_numpy(phase).cuda())
        fh = torch.empty((47, cfg.det_size, cfg.det_size), dtype=torch.float32).pin_memory()
        sh = torch.empty((47, 2 * sensor.n_valid), dtype=torch.float32).pin_memory()
        for _ in range(2):                                                          # second call re-uses events and scratch
            fh.zero_(); sh.zero_()
            sensor.run_host(torch.from_numpy(phase).pin_memory(), fh, sh)
            assert ((fd.cpu() - fh).abs().amax(dim=(1, 2)) <= 2e-6 * fd.cpu().abs().amax(dim=(1, 2))).all()
            assert (sd.cpu() - sh).abs().max() <= 1e-5


def test_host_buffer_pipeline_when_scratch_holds_fewer_frames_than_the_short_first_chunk(torch_cuda, monkeypatch):
    """B/16 frames in the first chunk must not exceed what the scratch budget holds (with a small
    budget the short chunk used to be launched with more frames than T was sized for)."""
    from paper_1607_07624_b200.pwfs import from_config
    torch = torch_cuda
    cfg = wl.CONFIGS["cfg1_tiny"]
    # T of one cfg1 frame = KX (7) x M (128) x NP (64) x 8 B = 458 752 B: a 1 MiB budget holds 2 frames, B/16 = 6
    monkeypatch.setenv("PWFS_SCRATCH_MB", "1")
    monkeypatch.setenv("PWFS_SMALL", "0")                          # the chunked two-kernel pipeline is what is under test
    B = 100
    phase = np.concatenate([wl.phase_batch(cfg, steps=10)] * 10)
    phase = np.ascontiguousarray(phase + np.arange(B, dtype=np.float32)[:, None, None] * 0.01)
    with from_config(cfg) as small:
        assert small.geometry(B)["frames_per_chunk"] <= 2
        fh, sh = small.run_host(phase)
        fd, sd = small.run(torch.from_numpy(phase).cuda())
        torch.cuda.synchronize()
    monkeypatch.delenv("PWFS_SCRATCH_MB")
    with from_config(cfg) as big:                                  # reference: one chunk, two-kernel path
        fr, sr = big.run(torch.from_numpy(phase).cuda())
        torch.cuda.synchronize()
    fr, sr = fr.cpu().numpy(), sr.cpu().numpy()
    for f, s_ in ((fh, sh), (fd.cpu().numpy(), sd.cpu().numpy())):
        assert (np.abs(f - fr).max(axis=(1, 2)) <= 2e-6 * fr.max(axis=(1, 2))).all()
        assert np.abs(s_ - sr).max() <= 1e-5


def test_binding_rejects_wrong_buffers(torch_cuda):
    """run() / run_host() check shape, dtype, device and contiguity of caller-supplied buffers."""
    from paper_1607_07624_b200.pwfs import from_config
    torch = torch_cuda
    cfg = wl.CONFIGS["cfg1_tiny"]
    N, D = cfg.n_pupil, cfg.det_size
    ph = torch.from_numpy(wl.phase_batch(cfg, steps=2)).cuda()
    with from_config(cfg) as sensor:
        nv = sensor.n_valid
        with pytest.raises(ValueError):
            sensor.run(ph, frames=torch.empty((1, D, D), device="cuda"))                 # too small
        with pytest.raises(TypeError):
            sensor.run(ph, frames=torch.empty((2, D, D), device="cuda", dtype=torch.float64))
        with pytest.raises(ValueError):
            sensor.run(ph, frames=torch.empty((2, D, D)))                                # host tensor
        with pytest.raises(ValueError):
            sensor.run(ph, frames=torch.empty((2, D, 2 * D), device="cuda")[:, :, ::2])  # strided
        with pytest.raises(ValueError):
            sensor.run(ph, slopes=torch.empty((2, 2 * nv + 1), device="cuda"))
        with pytest.raises(ValueError):
            sensor.run(torch.empty((2, N, N + 1), device="cuda"))
        with pytest.raises(ValueError):
            sensor.run_host(np.zeros((2, N + 1, N), np.float32))                         # wrong N: would read past the buffer
        with pytest.raises(TypeError):
            sensor.run_host(np.zeros((2, N, N), np.float64))
        with pytest.raises(ValueError):
            sensor.run_host(np.zeros((2, N, N), np.float32), frames=np.zeros((1, D, D), np.float32))
        with pytest.raises(ValueError):
            sensor.run_host(ph)                                                          # device tensor
        # a non-contiguous phase view is copied, on a caller-chosen stream too
        wide = torch.zeros((2, N, 2 * N), device="cuda")
        wide[:, :, ::2] = ph
        side = torch.cuda.Stream()
        side.wait_stream(torch.cuda.current_stream())
        f0, s0 = sensor.run(ph)
        f1, s1 = sensor.run(wide[:, :, ::2], stream=side)
        side.synchronize()
        torch.cuda.synchronize()
        assert torch.equal(f0, f1) and torch.equal(s0, s1)


def test_cuda_graph_capture_needs_reserved_scratch(torch_cuda):
    """pwfs_run refuses to allocate while its stream is being captured; after pwfs_reserve it captures and replays."""
    from paper_1607_07624_b200.pwfs import from_config, PwfsError, PWFS_EINVAL
    torch = torch_cuda
    cfg = wl.CONFIGS["cfg1_tiny"]
    ph = torch.from_numpy(wl.phase_batch(cfg, steps=3)).cuda()
    fr = torch.empty((3, cfg.det_size, cfg.det_size), device="cuda")
    with from_config(cfg) as ref:
        f_ref, s_ref = ref.run(ph)
    with from_config(cfg) as sensor:
        sl = torch.empty((3, 2 * sensor.n_valid), device="cuda")
        side = torch.cuda.Stream()
        side.wait_stream(torch.cuda.current_stream())
        g = torch.cuda.CUDAGraph()
        refused = None
        with torch.cuda.graph(g, stream=side):
            try:
                sensor.run(ph, fr, sl)                       # no scratch yet: must not cudaMalloc under capture
            except PwfsError as e:
                refused = e
        assert refused is not None and refused.code == PWFS_EINVAL
        torch.cuda.synchronize()
        sensor.reserve(3)
        g = torch.cuda.CUDAGraph()
        with torch.cuda.graph(g, stream=side):
            sensor.run(ph, fr, sl)
        fr.zero_(); sl.zero_()
        g.replay()
        torch.cuda.synchronize()
        assert torch.equal(fr, f_ref) and torch.equal(sl, s_ref)


@pytest.mark.parametrize("name,big,small", [("cfg1_tiny", 1000, 10), ("cfg2_flao", 300, 1), ("cfg2_flao", 300, 7)])
def test_reserve_covers_every_smaller_batch_under_capture(torch_cuda, monkeypatch, name, big, small):
    """pwfs_reserve(B) promises allocation-free pwfs_run calls of UP TO B frames.  A smaller batch can take another
    path (M = 128: 1000 frames run the two-kernel path, 10 the fused kernel with its own scratch) or a larger k-split
    (M = 320: one frame splits the modulation loop, 300 do not, so it needs more column scratch per frame): both
    must capture into a graph right after the reserve, with nothing run eagerly before."""
    from paper_1607_07624_b200.pwfs import from_config
    torch = torch_cuda
    monkeypatch.delenv("PWFS_SMALL", raising=False)
    cfg = wl.CONFIGS[name]
    ph = torch.from_numpy(wl.phase_batch(cfg, steps=small)).cuda()
    with from_config(cfg) as ref:
        f_ref, s_ref = ref.run(ph)
        g_big, g_small = ref.geometry(big), ref.geometry(small)
    if name == "cfg2_flao":
        assert g_small["k_split"] > g_big["k_split"] == 1
    with from_config(cfg) as sensor:
        fr = torch.empty((small, sensor.det_size, sensor.det_size), device="cuda")
        sl = torch.empty((small, 2 * sensor.n_valid), device="cuda")
        sensor.reserve(big)
        side = torch.cuda.Stream()
        side.wait_stream(torch.cuda.current_stream())
        g = torch.cuda.CUDAGraph()
        with torch.cuda.graph(g, stream=side):
            sensor.run(ph, fr, sl)                           # PWFS_EINVAL here if the reserve sized B = big only
        fr.zero_(); sl.zero_()
        g.replay()
        torch.cuda.synchronize()
        assert torch.equal(fr, f_ref) and torch.equal(sl, s_ref)
        _, launches = sensor.get_timing()
        assert (launches["fused"] == 1) == (name == "cfg1_tiny")


def test_host_buffer_entry_point_matches_device_entry_point(torch_cuda):
    from paper_1607_07624_b200.pwfs import from_config
    torch = torch_cuda
    cfg = wl.CONFIGS["cfg1_tiny"]
    phase = wl.phase_batch(cfg, steps=4)
    sensor = from_config(cfg)
    try:
        fd, sd = sensor.run(torch.from_numpy(phase).cuda())
        pinned = torch.from_numpy(phase).pin_memory()
        fh = torch.empty((4, cfg.det_size, cfg.det_size), dtype=torch.float32).pin_memory()
        sh = torch.empty((4, 2 * sensor.n_valid), dtype=torch.float32).pin_memory()
        sensor.run_host(pinned, fh, sh)
        assert torch.equal(fd.cpu(), fh) and torch.equal(sd.cpu(), sh)
        fn, sn = sensor.run_host(phase)                                # pageable numpy
        assert np.array_equal(fn, fh.numpy()) and np.array_equal(sn, sh.numpy())
    finally:
        sensor.close()


def test_bad_parameters_are_rejected(torch_cuda):
    from paper_1607_07624_b200.pwfs import PWFS, PwfsError, PWFS_EINVAL, PWFS_EUNSUPPORTED
    A = np.ones((32, 32), np.float32)
    for kw, code in [
        (dict(m_grid=96), PWFS_EUNSUPPORTED),          # 96/32 = 3 not built
        (dict(m_grid=60), PWFS_EINVAL),                # M < 2N
        (dict(mod_points=0), PWFS_EINVAL),
        (dict(mod_radius=-1.0), PWFS_EINVAL),
        (dict(n_subap=0), PWFS_EINVAL),
        (dict(n_subap=33), PWFS_EINVAL),
        (dict(mask_shift_px=10), PWFS_EINVAL),         # 2 s < N : windows overlap
        (dict(mask_shift_px=60), PWFS_EINVAL),         # window leaves the grid
        (dict(slope_norm=2), PWFS_EINVAL),
    ]:
        args = dict(pupil_amp=A, m_grid=128, mod_radius=1.0, mod_points=4, n_subap=8)
        args.update(kw)
        with pytest.raises(PwfsError) as ei:
            PWFS(**args)
        assert ei.value.code == code, kw
    with pytest.raises(PwfsError):                      # no light: n_valid == 0
        PWFS(np.zeros((32, 32), np.float32), 128, 1.0, 4, 8)


# ------------------------------------------------ f3: tilt list, field stop ---
def _run_both_list(torch, A, M, ns, phase, tx, ty, tw, stop, **kw):
    from oracle import pwfs_oracle as orc
    from paper_1607_07624_b200.pwfs import PWFS
    tl = (tx, ty) if tw is None else (tx, ty, tw)
    sensor = PWFS(A, M, 0.0, 1, ns, tilt_list=tl, field_stop_px=stop, **kw)
    try:
        fr, sl = sensor.run(torch.from_numpy(phase).cuda())
        torch.cuda.synchronize()
        # the oracle gets the same float32 list values, widened exactly
        f32 = lambda a: np.asarray(a, np.float32).astype(np.float64)
        w = np.ones(len(tx)) if tw is None else f32(tw)
        fr_ref, sl_ref = orc.pwfs_run_list(A, M, f32(tx), f32(ty), w, ns, phase, s=kw.get("mask_shift_px", 0),
                                           stop_h=stop, norm_mode=kw.get("slope_norm", 0))
        return _compare(fr.cpu().numpy(), sl.cpu().numpy(), fr_ref, sl_ref)
    finally:
        sensor.close()


def test_f3_uniform_circle_list_equals_the_circle_bit_for_bit(torch_cuda):
    from paper_1607_07624_b200.pwfs import PWFS, from_config
    torch = torch_cuda
    cfg = wl.CONFIGS["cfg1_tiny"]
    A = wl.make_pupil(cfg)
    phase = torch.from_numpy(wl.phase_batch(cfg, steps=3)).cuda()
    th = 2.0 * np.pi * np.arange(cfg.mod_points) / cfg.mod_points
    with from_config(cfg) as circ, PWFS(A, cfg.m_grid, 0.0, 1, cfg.n_subap,
                                        tilt_list=(cfg.mod_radius * np.cos(th), cfg.mod_radius * np.sin(th))) as lst:
        f0, s0 = circ.run(phase)
        f1, s1 = lst.run(phase)
        # float32 list entries differ from the double-precision circle in the last bits only
        assert (f0 - f1).abs().max() <= 2e-5 * f0.abs().max() and (s0 - s1).abs().max() <= 2e-5


@pytest.mark.parametrize("N,M,ns,stop", [
    (64, 128, 16, -1.0),      # weighted list on the quarter-mask kernels
    (64, 128, 16, 40.0),      # + field stop (table-mask kernels)
    (60, 128, 23, 17.5),      # margins, non-integer binning, tight stop
    (160, 320, 40, 103.0),    # cfg2 geometry, FoV 2" at 750 nm on 8.2 m ~ +-103 bins
    (240, 480, 40, 100.0),
    (250, 512, 50, 200.0),
    (288, 576, 36, 150.0),    # R1 = 18 on the table-mask kernels
    (900, 2048, 90, 500.0),   # M = 2048: mask table read through L1 (AM_GLOBAL)
    (720, 1440, 72, 300.0),   # R1 = 45, table-mask kernels
])
def test_f3_weighted_list_and_stop(torch_cuda, N, M, ns, stop):
    rng = np.random.default_rng(N + M)
    c = (np.arange(N) - (N - 1) / 2.0)
    X, Y = np.meshgrid(c, c)
    A = ((np.hypot(X, Y) <= N / 2.0) & (np.hypot(X, Y) >= 0.12 * N)).astype(np.float32)
    phase = (rng.standard_normal((2, N, N)) * 2.0).astype(np.float32)
    phase[1] = wl.tilt_phase(N, -0.4, 0.25)
    # an "extended source": 3 x 3 grid of points with a Gaussian brightness profile, plus a repeated x (shared row pass)
    gx, gy = np.meshgrid([-0.8, 0.0, 0.8], [-0.8, 0.0, 0.8])
    tx, ty = gx.ravel(), gy.ravel()
    tw = np.exp(-(tx ** 2 + ty ** 2) / 0.5)
    _run_both_list(torch_cuda, A, M, ns, phase, tx, ty, tw, stop)


def test_f3_full_size_elt_extended_source(torch_cuda):
    """cfg4 geometry with a 12-point weighted list and a field stop, 1 frame against the oracle."""
    cfg = wl.CONFIGS["cfg4_elt"]
    A = wl.make_pupil(cfg)
    phase = wl.phase_batch(cfg, steps=1)
    th = 2.0 * np.pi * np.arange(12) / 12
    tx, ty = np.concatenate([1.5 * np.cos(th[:8:1]), [0.0, 0.5, -0.5, 0.0]]), np.concatenate([1.5 * np.sin(th[:8:1]), [0.0, 0.0, 0.0, 0.7]])
    tw = np.linspace(0.5, 1.5, 12)
    _run_both_list(torch_cuda, A, cfg.m_grid, cfg.n_subap, phase, tx, ty, tw, 300.0)


def test_f3_bad_lists_are_rejected(torch_cuda):
    from paper_1607_07624_b200.pwfs import PWFS, PwfsError, PWFS_EINVAL
    A = np.ones((32, 32), np.float32)
    for tl in [([0.0, 1.0], [0.0, 0.0], [1.0, -1.0]), ([0.0], [0.0], [0.0]), ([np.nan], [0.0])]:
        with pytest.raises(PwfsError) as ei:
            PWFS(A, 128, 1.0, 4, 8, tilt_list=tl)
        assert ei.value.code == PWFS_EINVAL
