"""GPU parity of f2 (CCD detector, slope computer with reference, modal reconstructor) against
oracle/chain_oracle.py (+ the hot-path oracle's slopes), on the same seeded inputs.

Bars:
  * photon counts are integers decided in double precision on both sides: bit-exact;
  * pixels with read noise / without noise are doubles rounded to float32 once: <= 1 float32 ulp;
  * slopes: float32 arithmetic on O(10^0..10^4) pixel values, |d| <= 1e-5 (1 + |s|);
  * modes: float32 dot products of length n, |d| <= 1e-5 * sum_j |R_mj| |s_j|
    (worst-case bound (n/32 + 6) eps for the lane-strided FMA order is 2.2e-5 at n = 11712;
    typical error is ~sqrt of that).
The oracle's own frames (cast to float32) are the detector's input: nothing here is produced by
the CUDA path and fed to the oracle."""
import numpy as np
import pytest

from paper_1607_07624_b200 import workloads as wl

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def torch_cuda():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    return torch


def _dev(torch, a):
    return torch.from_numpy(np.ascontiguousarray(a, dtype=np.float32)).to("cuda:0")


def _ulp32(x):
    return np.spacing(np.abs(x).astype(np.float32)).astype(np.float64)


def _frames(seed, B, D, lo=0.0, hi=300.0):
    """Intensity-like frames spanning both photon-noise branches (lam from ~0 to hi), with
    exact zeros (unlit corners) in them."""
    rng = np.random.default_rng(seed)
    f = rng.gamma(0.7, 1.0, size=(B, D, D)) * rng.uniform(lo, hi, size=(B, 1, 1)) / 0.7
    f[:, : D // 5, : D // 5] = 0.0
    return f.astype(np.float32)


# ---------------------------------------------------------------------- CCD ---
@pytest.mark.parametrize("D,n_inst,n_int,n_steps", [(37, 3, 2, 4), (32, 1, 1, 3), (80, 2, 5, 5), (5, 1, 4, 8)])
def test_ccd_photon_counts_are_bit_exact(torch_cuda, D, n_inst, n_int, n_steps):
    from oracle import chain_oracle as co
    from paper_1607_07624_b200.chain import CCD
    fr = _frames(D * 1000 + n_int, n_steps * n_inst, D, hi=200.0 / n_int)
    kw = dict(n_inst=n_inst, n_int=n_int, gain=1.7, quantum_eff=0.32, photon_noise=True, seed=0xDEADBEEF12345)
    want = co.ccd(fr, first_out_frame=7, **kw)
    with CCD(D, **kw) as ccd:
        got = ccd.run(_dev(torch_cuda, fr), first_out_frame=7).cpu().numpy().astype(np.float64)
    assert got.shape == want.shape
    lam = 0.32 * 1.7 * co.integrate(fr, n_inst, n_int)
    assert (lam < 128).any() and (lam >= 128).any() and (lam == 0).any()      # both branches and the zero case ran
    assert np.array_equal(got, want)


def test_ccd_full_noise_and_no_noise_within_one_float_ulp(torch_cuda):
    from oracle import chain_oracle as co
    from paper_1607_07624_b200.chain import CCD
    D, n_inst, n_int, n_steps = 41, 2, 3, 6
    fr = _frames(3, n_steps * n_inst, D, hi=120.0)
    for kw in (dict(photon_noise=True, readout_noise=True, readout_level=2.5, seed=99),
               dict(readout_noise=True, readout_level=0.7, seed=5),
               dict()):
        kw = dict(n_inst=n_inst, n_int=n_int, gain=0.9, quantum_eff=0.8, **kw)
        want = co.ccd(fr, **kw)
        with CCD(D, **kw) as ccd:
            got = ccd.run(_dev(torch_cuda, fr)).cpu().numpy().astype(np.float64)
        assert (np.abs(got - want) <= _ulp32(want)).all(), kw
    # noise off: exactly qe * gain * sum, rounded once
    assert np.array_equal(got.astype(np.float32), (0.8 * 0.9 * co.integrate(fr, n_inst, n_int)).astype(np.float32))


def test_ccd_stream_is_indexed_by_output_frame_and_seed(torch_cuda):
    from paper_1607_07624_b200.chain import CCD
    D = 24
    fr = _dev(torch_cuda, _frames(8, 8, D, hi=50.0))
    kw = dict(n_inst=2, n_int=1, gain=1.0, photon_noise=True, readout_noise=True, readout_level=1.0)
    with CCD(D, seed=1, **kw) as a, CCD(D, seed=2, **kw) as b:
        whole = a.run(fr, first_out_frame=10)
        again = a.run(fr, first_out_frame=10)
        parts = torch_cuda.cat([a.run(fr[:4], first_out_frame=10), a.run(fr[4:], first_out_frame=14)])
        other = b.run(fr, first_out_frame=10)
    assert torch_cuda.equal(whole, again) and torch_cuda.equal(whole, parts)
    assert not torch_cuda.equal(whole, other)
    with CCD(D, n_inst=2, n_int=3) as c:
        with pytest.raises(Exception):
            c.run(fr)                                  # 4 steps is not a multiple of n_int = 3
        assert c.run(fr[:0]).shape[0] == 0             # empty batch is a no-op


def test_ccd_at_bench_size_on_oracle_frames(torch_cuda):
    """cfg4 detector (184^2), the oracle's own noiseless frame as input, faint and bright star."""
    from oracle import chain_oracle as co
    from oracle import pwfs_oracle as orc
    from paper_1607_07624_b200.chain import CCD
    cfg = wl.CONFIGS["cfg4_elt"]
    A = wl.make_pupil(cfg)
    phase = wl.phase_batch(cfg, steps=1)
    fr, _ = orc.pwfs_run(A, cfg.m_grid, cfg.mod_radius, cfg.mod_points, cfg.n_subap, phase)
    fr32 = fr.astype(np.float32)
    for n_ph in (3.0e4, 3.0e6):                        # ~1 and ~100 photons per lit pixel
        kw = dict(gain=n_ph / fr.sum(), quantum_eff=0.32, photon_noise=True, seed=2024)
        want = co.ccd(fr32, **kw)
        with CCD(2 * cfg.n_subap, **kw) as ccd:
            got = ccd.run(_dev(torch_cuda, fr32)).cpu().numpy().astype(np.float64)
        assert np.array_equal(got, want)
        assert abs(got.sum() / (0.32 * n_ph) - 1.0) < 0.05


# ----------------------------------------------------------- slope computer ---
@pytest.mark.parametrize("name,norm", [("cfg1_tiny", 0), ("cfg1_tiny", 1), ("cfg2_flao", 0), ("cfg4_elt", 0)])
def test_slopec_matches_oracle_on_noisy_pixels(torch_cuda, name, norm):
    from oracle import chain_oracle as co
    from oracle import pwfs_oracle as orc
    from paper_1607_07624_b200.chain import SlopeComputer
    cfg = wl.CONFIGS[name]
    A = wl.make_pupil(cfg)
    valid, nv = orc.valid_mask(A, cfg.n_subap)
    D = 2 * cfg.n_subap
    rng = np.random.default_rng(nv)
    # detector-like pixels: a lit level plus noise, strictly positive so both normalisations are safe
    pix = (200.0 + 30.0 * rng.standard_normal((3, D, D))).astype(np.float32)
    sn = (0.05 * rng.standard_normal(2 * nv)).astype(np.float32)
    raw = np.stack([orc.slopes(p.astype(np.float64), valid, norm) for p in pix])
    with SlopeComputer(valid, slope_norm=norm, sn=sn) as sc:
        assert sc.n_slopes == 2 * nv
        got = sc.run(_dev(torch_cuda, pix)).cpu().numpy().astype(np.float64)
        want = co.slopes_with_reference(raw, sn)
        assert (np.abs(got - want) <= 1e-5 * (1 + np.abs(want))).all()
        sc.set_reference(None)
        got0 = sc.run(_dev(torch_cuda, pix)).cpu().numpy().astype(np.float64)
        assert (np.abs(got0 - raw) <= 1e-5 * (1 + np.abs(raw))).all()
        sc.set_reference(2 * sn)
        got2 = sc.run(_dev(torch_cuda, pix)).cpu().numpy().astype(np.float64)
        assert (np.abs(got2 - (raw - 2.0 * sn)) <= 1e-5 * (1 + np.abs(raw))).all()


def test_slopec_agrees_with_the_hot_path_slopes(torch_cuda):
    """Same frames through pwfs_run's slope kernel and through the stand-alone slope computer."""
    from paper_1607_07624_b200.chain import SlopeComputer
    from paper_1607_07624_b200.pwfs import from_config
    cfg = wl.CONFIGS["cfg1_tiny"]
    phase = wl.phase_batch(cfg, steps=4)
    with from_config(cfg, device=0) as sensor:
        fr, sl = sensor.run(torch_cuda.from_numpy(phase).to("cuda:0"))
        with SlopeComputer(sensor.valid_mask()) as sc:
            sl2 = sc.run(fr)
    assert (sl - sl2).abs().max().item() <= 1e-6


# ------------------------------------------------------------ reconstructor ---
@pytest.mark.parametrize("n_modes,ns,B", [(54, 2512, 1), (5, 416, 3), (37, 1030, 17), (1, 1, 1), (33, 7, 2),
                                          (300, 2528, 40), (1200, 416, 9), (4096, 11712, 1),
                                          # single frames: the streaming GEMV kernel (4, 8, 12 slope registers per thread,
                                          # ragged rows, more rows than CTAs), and one row longer than it takes
                                          (700, 1030, 1), (100, 6001, 1), (64, 12288, 1), (65, 12290, 1), (2500, 2049, 1),
                                          # batches >= 24 frames run on the tensor cores (rec_tc.cu): ragged tiles in
                                          # every dimension, K not a multiple of 32, two frame tiles, one K block
                                          (130, 1000, 24), (257, 515, 130), (128, 2048, 128), (2100, 31, 33),
                                          (64, 4100, 300)])
def test_reconstructor_matches_matrix_product(torch_cuda, n_modes, ns, B):
    from oracle import chain_oracle as co
    from paper_1607_07624_b200.chain import Reconstructor
    rng = np.random.default_rng(n_modes * 7 + ns + B)
    R = rng.standard_normal((n_modes, ns)).astype(np.float32)
    S = (0.1 * rng.standard_normal((B, ns))).astype(np.float32)
    want = co.reconstruct(R, S)
    bound = 1e-5 * (np.abs(S.astype(np.float64)) @ np.abs(R.astype(np.float64)).T) + 1e-30
    with Reconstructor(R) as rec:
        got = rec.run(_dev(torch_cuda, S)).cpu().numpy().astype(np.float64)
        assert got.shape == (B, n_modes)
        assert (np.abs(got - want) <= bound).all(), np.abs(got - want).max()
        # slopes not 16-byte aligned: the scalar-load variant
        buf = torch_cuda.zeros(B * ns + 1, dtype=torch_cuda.float32, device="cuda:0")
        buf[1:] = _dev(torch_cuda, S).reshape(-1)
        got_u = rec.run(buf[1:].view(B, ns)).cpu().numpy().astype(np.float64)
        assert (np.abs(got_u - want) <= bound).all()
        assert rec.run(_dev(torch_cuda, S)[:0]).shape == (0, n_modes)


def test_reconstructor_at_bench_size(torch_cuda):
    """cfg4: 11712 slopes -> 4096 modes, 100 frames (the batch bench.py times)."""
    from paper_1607_07624_b200.chain import Reconstructor
    n_modes, ns, B = 4096, 11712, 100
    rng = np.random.default_rng(4)
    R = rng.standard_normal((n_modes, ns), dtype=np.float32)
    S = (0.1 * rng.standard_normal((B, ns))).astype(np.float32)
    with Reconstructor(R) as rec:
        got = rec.run(_dev(torch_cuda, S)).cpu().numpy().astype(np.float64)
    rows = rng.choice(n_modes, 64, replace=False)              # sampled outputs, computed one by one in double
    R64, S64 = R[rows].astype(np.float64), S.astype(np.float64)
    want = S64 @ R64.T
    bound = 1e-5 * (np.abs(S64) @ np.abs(R64).T)
    assert (np.abs(got[:, rows] - want) <= bound).all()
    assert np.isfinite(got).all()


# ------------------------------------------------------------- whole chain ---
def test_device_chain_f1_to_modes_matches_oracle_chain(torch_cuda):
    """atmosphere -> pyramid -> CCD -> slopes - sn -> modes, all on the device, against the same
    chain of oracles.  Noise off: float tolerances add up; photon noise on: counts may differ by
    one where the two intensities (1e-4 apart at most) straddle a decision boundary."""
    from oracle import atmo_oracle as ao
    from oracle import chain_oracle as co
    from oracle import pwfs_oracle as orc
    from paper_1607_07624_b200.atmo import Atmosphere
    from paper_1607_07624_b200.chain import CCD, Reconstructor, SlopeComputer
    from paper_1607_07624_b200.pwfs import from_config
    cfg = wl.CONFIGS["cfg1_tiny"]
    A = wl.make_pupil(cfg)
    rng = np.random.default_rng(11)
    G, N, L = 96, cfg.n_pupil, 2
    atm = dict(screens=(rng.standard_normal((L, G, G)) * 2).astype(np.float32), pitch=0.125,
               wind_vxy=[[7.0, -3.0], [-12.0, 5.0]], heights=[0.0, 4000.0], dirs_tan=[[0.0, 0.0], [2e-4, -1e-4]],
               wl_scale=[1.0], n_pupil=N)
    n_steps, n_int, dt = 4, 2, 1e-3
    valid, nv = orc.valid_mask(A, cfg.n_subap)
    sn = (0.01 * rng.standard_normal(2 * nv)).astype(np.float32)
    R = rng.standard_normal((20, 2 * nv)).astype(np.float32) / nv
    n_ph = 5.0e4

    phase = ao.propagate(atm["screens"], atm["pitch"], atm["wind_vxy"], atm["heights"], atm["dirs_tan"],
                         atm["wl_scale"], 3, n_steps, dt, N).astype(np.float32)
    fr, _ = orc.pwfs_run(A, cfg.m_grid, cfg.mod_radius, cfg.mod_points, cfg.n_subap, phase)
    gain = n_ph / float((A.astype(np.float64) ** 2).sum())          # sum I = sum A^2 per step
    for photon in (False, True):
        kw = dict(n_inst=2, n_int=n_int, gain=gain, quantum_eff=0.5, photon_noise=photon, seed=77)
        pix = co.ccd(fr, **kw)
        s = co.slopes_with_reference(np.stack([orc.slopes(p, valid) for p in pix]), sn)
        modes = co.reconstruct(R, s)
        with Atmosphere(**atm) as a, from_config(cfg, device=0) as sensor, CCD(2 * cfg.n_subap, **kw) as ccd, \
                SlopeComputer(sensor.valid_mask(), sn=sn) as sc, Reconstructor(R) as rec:
            d_fr, _ = sensor.run(a.propagate(3, n_steps, dt))
            d_pix = ccd.run(d_fr)
            d_modes = rec.run(sc.run(d_pix))
            torch_cuda.cuda.synchronize()
        g_pix, g_modes = d_pix.cpu().numpy().astype(np.float64), d_modes.cpu().numpy().astype(np.float64)
        assert g_pix.shape == pix.shape == (n_steps // n_int * 2, 2 * cfg.n_subap, 2 * cfg.n_subap)
        if photon:
            diff = np.abs(g_pix - pix)
            assert diff.max() <= 1.0 and (diff != 0).mean() <= 5e-3
        else:
            assert (np.abs(g_pix - pix) <= 1e-4 * pix.max()).all()
            tol = 1e-4 * np.abs(R.astype(np.float64)).sum(axis=1).max() * 2
            assert np.abs(g_modes - modes).max() <= tol


def test_batched_reconstructor_is_capturable_after_reserve(torch_cuda):
    """pwfs_rec_reserve sizes the tensor-core path's scratch, so a batched pwfs_rec_run neither allocates nor
    synchronises and can be captured into a CUDA graph; without it the capture is refused (PWFS_EINVAL), not broken."""
    from paper_1607_07624_b200.chain import Reconstructor
    from paper_1607_07624_b200.pwfs import PwfsError, PWFS_EINVAL
    torch = torch_cuda
    rng = np.random.default_rng(9)
    R = rng.standard_normal((200, 700)).astype(np.float32)
    S = _dev(torch, 0.1 * rng.standard_normal((40, 700)))
    out = torch.zeros((40, 200), device="cuda")
    side = torch.cuda.Stream()
    side.wait_stream(torch.cuda.current_stream())
    with Reconstructor(R) as rec:
        refused = None
        g = torch.cuda.CUDAGraph()
        with torch.cuda.graph(g, stream=side):
            try:
                rec.run(S, out=out, stream=side)
            except PwfsError as e:
                refused = e
        assert refused is not None and refused.code == PWFS_EINVAL
        torch.cuda.synchronize()
        rec.reserve(40)
        want = rec.run(S).clone()
        g = torch.cuda.CUDAGraph()
        with torch.cuda.graph(g, stream=side):
            rec.run(S, out=out, stream=side)
        out.zero_()
        g.replay()
        torch.cuda.synchronize()
        assert torch.equal(out, want)


def test_reconstructor_reserve_covers_smaller_batches(torch_cuda):
    """pwfs_rec_reserve(B) must serve every batch up to B.  A smaller batch fills fewer frame tiles and is split
    further along K: with 10 048 slopes on 148 SMs, 200 frames (2 tiles x 74 splits) write more split-K partials than
    300 (3 tiles x 49), so a reserve sized for exactly 300 frames would refuse the capture of 200."""
    from paper_1607_07624_b200.chain import Reconstructor
    torch = torch_cuda
    rng = np.random.default_rng(10)
    R = (rng.standard_normal((128, 10048)) / 100.0).astype(np.float32)
    S = _dev(torch, 0.1 * rng.standard_normal((300, 10048)))
    side = torch.cuda.Stream()
    side.wait_stream(torch.cuda.current_stream())
    with Reconstructor(R) as ref:
        want = {b: ref.run(S[:b]).clone() for b in (200, 100, 300)}
    with Reconstructor(R) as rec:
        rec.reserve(300)
        for b in (200, 100, 300):
            out = torch.zeros((b, 128), device="cuda")
            g = torch.cuda.CUDAGraph()
            with torch.cuda.graph(g, stream=side):
                rec.run(S[:b], out=out, stream=side)
            g.replay()
            torch.cuda.synchronize()
            assert torch.equal(out, want[b]), b
