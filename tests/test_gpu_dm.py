"""GPU parity of the deformable mirror (influence-function multiply) and the integrator control against
oracle/dm_oracle.py, through the C ABI (include/pwfs_dm.h), and the closed loop they make possible on the device:
pyramid -> slopes -> modes -> integrator -> DM -> phase, no host round trip (Table 2).

Bars: DM layer |d| <= 1e-5 * sum_m |ifs||cmd| per pixel (FP32 FMA against a double sum); integrator 1e-6 relative."""
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
    return torch.from_numpy(np.ascontiguousarray(a, dtype=np.float32)).cuda()


@pytest.mark.parametrize("name,n_act,B", [("cfg1_tiny", 20, 1), ("cfg1_tiny", 54, 3), ("cfg2_flao", 54, 8),
                                          ("cfg2_flao", 300, 13), ("cfg4_elt", 257, 2)])
def test_dm_layer_matches_oracle(torch_cuda, name, n_act, B):
    from oracle import dm_oracle as dmo
    from paper_1607_07624_b200.dm import DeformableMirror
    torch = torch_cuda
    cfg = wl.CONFIGS[name]
    A = wl.make_pupil(cfg)
    N = cfg.n_pupil
    ifs, pix = wl.zernike_ifs(A, n_act)
    rng = np.random.default_rng(n_act + B)
    cmd = rng.standard_normal((B, n_act)).astype(np.float32)
    phase = rng.standard_normal((B, N, N)).astype(np.float32)
    bound = np.zeros((B, N * N))
    bound[:, pix] = 1e-5 * (np.abs(cmd.astype(np.float64)) @ np.abs(ifs.astype(np.float64))) + 1e-12
    bound = bound.reshape(B, N, N)
    with DeformableMirror(ifs, pix, N) as dm:
        lay = dm.apply(_dev(torch, cmd)).cpu().numpy().astype(np.float64)                  # beta = 0: the layer itself
        want = dmo.dm_layer(ifs, pix, N, cmd)
        assert (np.abs(lay - want) <= bound).all(), np.abs(lay - want).max()
        assert (lay.reshape(B, -1)[:, np.setdiff1d(np.arange(N * N), pix)] == 0).all()     # zero outside the IFs
        ph = _dev(torch, phase)
        out = dm.apply(_dev(torch, cmd), ph, alpha=-0.7, beta=1.0).cpu().numpy().astype(np.float64)
        want2 = dmo.dm_apply(ifs, pix, phase, cmd, alpha=-0.7, beta=1.0)
        assert (np.abs(out - want2) <= 0.7 * bound + 1e-6 * np.abs(want2) + 1e-7).all()
        assert dm.apply(_dev(torch, cmd)[:0]).shape == (0, N, N)


def test_dm_rejects_bad_arguments(torch_cuda):
    from paper_1607_07624_b200.dm import DeformableMirror
    from paper_1607_07624_b200.pwfs import PwfsError, PWFS_EINVAL
    ifs = np.ones((2, 3), np.float32)
    for pix in ([0, 1, 1], [0, 1, 16], [-1, 0, 1]):                    # repeated, out of range, negative
        with pytest.raises(PwfsError) as ei:
            DeformableMirror(ifs, np.array(pix, np.int32), 4)
        assert ei.value.code == PWFS_EINVAL
    bad = ifs.copy(); bad[1, 2] = np.nan
    with pytest.raises(PwfsError):
        DeformableMirror(bad, np.array([0, 1, 2], np.int32), 4)
    with DeformableMirror(ifs, np.array([0, 5, 15], np.int32), 4) as dm:
        with pytest.raises(PwfsError):
            dm.apply(_dev(torch_cuda, np.zeros((1, 2))), _dev(torch_cuda, np.zeros((1, 4, 4))), beta=0.5)


@pytest.mark.parametrize("n,delay,T", [(54, 0, 7), (54, 2, 9), (4096, 1, 5), (1, 3, 6)])
def test_integrator_matches_oracle_eagerly_and_from_a_graph(torch_cuda, n, delay, T):
    from oracle import dm_oracle as dmo
    from paper_1607_07624_b200.dm import Integrator
    torch = torch_cuda
    rng = np.random.default_rng(n + delay)
    gain = rng.uniform(0.1, 0.9, n).astype(np.float32)
    deltas = rng.standard_normal((T, n)).astype(np.float32)
    want = dmo.integrator(gain, delay, deltas)
    with Integrator(gain, delay) as integ:
        got = np.stack([integ.step(_dev(torch, deltas[t])).cpu().numpy() for t in range(T)]).astype(np.float64)
        assert np.abs(got - want).max() <= 1e-6 * max(1.0, np.abs(want).max())
        # the step counter lives on the device: one captured step, replayed, walks through the same sequence
        integ.reset()
        d_in = torch.zeros(n, device="cuda")
        d_out = torch.zeros(n, device="cuda")
        side = torch.cuda.Stream()
        side.wait_stream(torch.cuda.current_stream())
        g = torch.cuda.CUDAGraph()
        with torch.cuda.graph(g, stream=side):
            integ.step(d_in, out=d_out)
        integ.reset()
        torch.cuda.synchronize()
        rows = []
        for t in range(T):
            d_in.copy_(_dev(torch, deltas[t]))
            g.replay()
            rows.append(d_out.cpu().numpy().copy())
        assert np.abs(np.stack(rows).astype(np.float64) - want).max() <= 1e-6 * max(1.0, np.abs(want).max())


def test_closed_loop_on_the_device_flattens_a_static_aberration(torch_cuda):
    """PASSATA's SCAO loop of Table 2 with every object on the device: residual phase -> pyramid (pwfs_run) ->
    reconstructor -> integrator -> DM -> residual phase.  The reconstructor is the pseudo-inverse of a push-pull
    interaction matrix measured through the same device chain.  A static aberration made of the first 10 Zernike modes
    must be driven to < 5 % of its rms in 25 steps (gain 0.4, one frame of delay); every array stays in device memory."""
    from paper_1607_07624_b200.chain import Reconstructor
    from paper_1607_07624_b200.dm import DeformableMirror, Integrator
    from paper_1607_07624_b200.pwfs import from_config
    torch = torch_cuda
    cfg = wl.CONFIGS["cfg1_tiny"]
    A = wl.make_pupil(cfg)
    N, n_modes = cfg.n_pupil, 10
    ifs, pix = wl.zernike_ifs(A, n_modes)
    amp = 0.05                                                          # rad rms per mode: linear regime of the pyramid
    with from_config(cfg) as sensor, DeformableMirror(ifs, pix, N) as dm:
        pokes = torch.cat([amp * torch.eye(n_modes, device="cuda"), -amp * torch.eye(n_modes, device="cuda")])
        _, sl = sensor.run(dm.apply(pokes))
        imat = ((sl[:n_modes] - sl[n_modes:]) / (2 * amp)).T.cpu().numpy().astype(np.float64)     # [n_slopes][n_modes]
        recmat = np.linalg.pinv(imat).astype(np.float32)
        rng = np.random.default_rng(5)
        a = (0.3 * rng.standard_normal(n_modes)).astype(np.float32)
        atmo = dm.apply(_dev(torch, a[None]))                           # the static aberration as a phase screen [1,N,N]
        rms0 = float(atmo.reshape(-1)[torch.from_numpy(pix.astype(np.int64)).cuda()].std())
        with Reconstructor(recmat) as rec, Integrator(np.full(n_modes, -0.4, np.float32), delay=1) as integ:
            cmd = torch.zeros((1, n_modes), device="cuda")
            resid = torch.empty_like(atmo)
            rms = []
            for _ in range(25):
                resid.copy_(atmo)
                dm.apply(cmd, resid, alpha=1.0, beta=1.0)               # residual = atmosphere + DM layer
                _, sl = sensor.run(resid)
                modes = rec.run(sl)
                integ.step(modes.reshape(-1), out=cmd)                  # negative gains: the DM opposes what is measured
                rms.append(float(resid.reshape(-1)[torch.from_numpy(pix.astype(np.int64)).cuda()].std()))
    assert rms[0] == pytest.approx(rms0, rel=1e-5)
    assert rms[-1] < 0.05 * rms0, rms
