"""pwfs_run_noalloc: the sensor call for users who may not allocate GPU memory.

Some users of this library cannot let a call reach cudaMalloc: a fixed-rate control
loop (cudaMalloc / cudaFree can stall until the whole device is idle and take an
unbounded time), or a process whose GPU memory has been handed to another allocator
or capped by a quota.  For them include/pwfs.h offers pwfs_run_noalloc, which runs
the fused M = 128 kernel with its working memory in a fixed array inside libpwfs.so
(4 MiB + 256 B per GPU) instead of heap scratch.  This file checks that it computes
what the ordinary path (pwfs_run) computes, on two calls in a row that share that
array, that free device memory does not move across a call, and that batches beyond
the array's size are refused.

The file is named so that pytest collects it last: `pytest -x` stops at the first
failure, and a failure here must not hide the parity tests.  It makes no assumption
about what ran before it in the process (it passes alone and after the whole suite).
"""
import numpy as np
import pytest

from paper_1607_07624_b200 import workloads as wl

pytestmark = pytest.mark.gpu

TOL_FRAME = 1e-4      # max |dI| / max I per frame -- the bar of tests/test_gpu_parity.py
TOL_SLOPE = 1e-4      # |d slope| per element


@pytest.fixture(scope="module")
def torch_cuda():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    return torch


def _close(torch, fr, sl, fr_ref, sl_ref):
    assert torch.isfinite(fr).all() and torch.isfinite(sl).all()
    err_f = ((fr - fr_ref).abs().amax(dim=(1, 2)) / fr_ref.amax(dim=(1, 2))).max().item()
    err_s = (sl - sl_ref).abs().max().item()
    assert err_f <= TOL_FRAME, f"frame error {err_f:.3e} > {TOL_FRAME}"
    assert err_s <= TOL_SLOPE, f"slope error {err_s:.3e} > {TOL_SLOPE}"


def test_two_calls_in_a_row_match_the_ordinary_path(torch_cuda, monkeypatch):
    """Call 1 (10 frames) and call 2 (3 other frames, then without slopes) go through the shared fixed array one
    after the other; each must agree with pwfs_run on the same input -- with its fused kernel, and with its
    two-kernel path, which sums over the modulation points in another order."""
    from paper_1607_07624_b200.pwfs import from_config
    torch = torch_cuda
    monkeypatch.delenv("PWFS_SMALL", raising=False)
    cfg = wl.CONFIGS["cfg1_tiny"]                                   # M = 128, N = 64, K = 12, 16 x 16 subapertures
    ph_a = torch.from_numpy(wl.phase_batch(cfg)).cuda()             # the config's 10 steps
    rng = np.random.default_rng(77)
    ph_b = torch.from_numpy((rng.standard_normal((3, cfg.n_pupil, cfg.n_pupil)) * 4.0).astype(np.float32)).cuda()
    with from_config(cfg) as sensor:
        D, nv = sensor.det_size, sensor.n_valid
        ref_a = sensor.run(ph_a)                                    # ordinary path (allocates its scratch on demand)
        ref_b = sensor.run(ph_b)
        _, launches = sensor.get_timing()
        assert launches["fused"] == 2                               # ... which took the fused kernel for these batches
        fr_a, sl_a = torch.full((10, D, D), -1.0, device="cuda"), torch.full((10, 2 * nv), -1.0, device="cuda")
        fr_b, sl_b = torch.full((3, D, D), -1.0, device="cuda"), torch.full((3, 2 * nv), -1.0, device="cuda")
        fr_c = torch.full((3, D, D), -1.0, device="cuda")
        sensor.run_noalloc(ph_a, fr_a, sl_a)                        # first call on this GPU: finds the array
        torch.cuda.synchronize()
        free_before = torch.cuda.mem_get_info()[0]
        sensor.run_noalloc(ph_b, fr_b, sl_b)                        # second call: the array holds call 1's leftovers
        sensor.run_noalloc(ph_b, fr_c, None)                        # slopes are optional
        torch.cuda.synchronize()
        assert torch.cuda.mem_get_info()[0] == free_before          # no device memory was taken or returned
        _, launches = sensor.get_timing()
        assert launches["fused"] == 3 and launches["xpass"] == 0
        _close(torch, fr_a, sl_a, *ref_a)
        _close(torch, fr_b, sl_b, *ref_b)
        assert torch.equal(fr_a, ref_a[0]) and torch.equal(sl_a, ref_a[1])      # same kernel: same bits
        assert torch.equal(fr_b, ref_b[0]) and torch.equal(sl_b, ref_b[1])
        assert torch.equal(fr_c, fr_b)
    monkeypatch.setenv("PWFS_SMALL", "0")                           # read at create: this handle never takes the fused kernel
    with from_config(cfg) as two:
        ref2_a, ref2_b = two.run(ph_a), two.run(ph_b)
        _, launches = two.get_timing()
        assert launches["fused"] == 0 and launches["xpass"] == 2
    _close(torch, fr_a, sl_a, *ref2_a)
    _close(torch, fr_b, sl_b, *ref2_b)


def test_two_sensors_share_the_array_one_after_the_other(torch_cuda):
    """The array belongs to the GPU, not to a handle: a second sensor with another geometry (table mask, odd K,
    non-integer binning) runs through it right after the first, on the same stream, and both stay correct."""
    from paper_1607_07624_b200.pwfs import PWFS
    torch = torch_cuda
    N = 60
    c = np.arange(N) - (N - 1) / 2.0
    X, Y = np.meshgrid(c, c)
    A = ((np.hypot(X, Y) <= N / 2.0) & (np.hypot(X, Y) >= 0.12 * N)).astype(np.float32)
    rng = np.random.default_rng(5)
    ph = torch.from_numpy((rng.standard_normal((4, N, N)) * 2.0).astype(np.float32)).cuda()
    with PWFS(A, 128, 1.5, 5, 23) as s1, PWFS(A, 128, 2.0, 7, 12, mask_shift_px=31, slope_norm=1) as s2:
        refs = [s.run(ph) for s in (s1, s2)]
        outs = [(torch.empty_like(r[0]), torch.empty_like(r[1])) for r in refs]
        for _ in range(2):
            for s, o in zip((s1, s2), outs):
                s.run_noalloc(ph, o[0], o[1])
        torch.cuda.synchronize()
        for o, r in zip(outs, refs):
            _close(torch, o[0], o[1], *r)


def test_sizes_beyond_the_fixed_array_are_refused(torch_cuda):
    from paper_1607_07624_b200.pwfs import (NOALLOC_MAX_FRAMES, NOALLOC_MAX_PART_FLOATS, PWFS_ELIMIT,
                                            PWFS_EUNSUPPORTED, PwfsError, from_config, strerror)
    torch = torch_cuda
    assert "pwfs_run_noalloc" in strerror(PWFS_ELIMIT)
    cfg = wl.CONFIGS["cfg1_tiny"]
    with from_config(cfg) as sensor:
        D, nv, N = sensor.det_size, sensor.n_valid, cfg.n_pupil
        ok = NOALLOC_MAX_FRAMES                                      # 64 x 12 x 32^2 floats = 75 % of the array
        assert ok * cfg.mod_points * D * D <= NOALLOC_MAX_PART_FLOATS
        ph = torch.zeros((ok + 1, N, N), device="cuda")
        fr, sl = torch.full((ok + 1, D, D), -1.0, device="cuda"), torch.full((ok + 1, 2 * nv), -1.0, device="cuda")
        with pytest.raises(PwfsError) as ei:
            sensor.run_noalloc(ph, fr, sl)                           # one frame too many
        assert ei.value.code == PWFS_ELIMIT
        torch.cuda.synchronize()
        assert (fr == -1.0).all() and (sl == -1.0).all()             # nothing was enqueued
        sensor.run_noalloc(ph[:ok], fr[:ok], sl[:ok])                # the largest batch it takes
        ref = sensor.run(ph[:ok])
        torch.cuda.synchronize()
        _close(torch, fr[:ok], sl[:ok], *ref)
        sensor.run_noalloc(ph[:0], fr[:0], sl[:0])                   # B = 0: no-op
    A = wl.make_pupil(cfg)
    from paper_1607_07624_b200.pwfs import PWFS
    with PWFS(A, 128, 3.0, 48, 32) as big:                           # K x D^2 = 48 x 64^2: 5 frames fit, 6 do not
        D, nv = big.det_size, big.n_valid
        ph = torch.zeros((6, 64, 64), device="cuda")
        fr, sl = torch.empty((6, D, D), device="cuda"), torch.empty((6, 2 * nv), device="cuda")
        with pytest.raises(PwfsError) as ei:
            big.run_noalloc(ph, fr, sl)
        assert ei.value.code == PWFS_ELIMIT
        big.run_noalloc(ph[:5], fr[:5], sl[:5])
        ref = big.run(ph[:5])
        torch.cuda.synchronize()
        _close(torch, fr[:5], sl[:5], *ref)
    cfg2 = wl.CONFIGS["cfg2_flao"]
    with from_config(cfg2) as other:                                 # M = 320: no fused kernel for this grid
        D, nv, N = other.det_size, other.n_valid, cfg2.n_pupil
        with pytest.raises(PwfsError) as ei:
            other.run_noalloc(torch.zeros((1, N, N), device="cuda"), torch.empty((1, D, D), device="cuda"),
                              torch.empty((1, 2 * nv), device="cuda"))
        assert ei.value.code == PWFS_EUNSUPPORTED
