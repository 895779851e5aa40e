"""Pins of the DM / integrator oracle (oracle/dm_oracle.py) against what does not depend on it: a library
matrix product, closed forms of the integrator recursion, the tilt phase the input module defines on its own,
and a closed loop whose convergence rate is known in closed form."""
import numpy as np
import pytest

from oracle import dm_oracle as dmo
from paper_1607_07624_b200 import workloads as wl


@pytest.fixture(scope="module")
def zern():
    cfg = wl.CONFIGS["cfg1_tiny"]
    A = wl.make_pupil(cfg)
    ifs, pix = wl.zernike_ifs(A, 20)
    return dict(A=A, N=cfg.n_pupil, ifs=ifs, pix=pix)


def test_layer_is_the_matrix_product_scattered_into_the_pupil(zern):
    rng = np.random.default_rng(0)
    cmd = rng.standard_normal((3, 20)).astype(np.float32)
    lay = dmo.dm_layer(zern["ifs"], zern["pix"], zern["N"], cmd)
    want = np.zeros((3, zern["N"] ** 2))
    want[:, zern["pix"]] = cmd.astype(np.float64) @ zern["ifs"].astype(np.float64)      # library routine
    assert np.abs(lay.reshape(3, -1) - want).max() < 1e-12
    assert (lay.reshape(3, -1)[:, np.setdiff1d(np.arange(zern["N"] ** 2), zern["pix"])] == 0).all()


def test_single_actuator_and_linearity(zern):
    e = np.zeros(20, np.float32); e[7] = 2.5
    lay = dmo.dm_layer(zern["ifs"], zern["pix"], zern["N"], e).ravel()
    assert np.abs(lay[zern["pix"]] - 2.5 * zern["ifs"][7].astype(np.float64)).max() < 1e-12
    rng = np.random.default_rng(1)
    a, b = rng.standard_normal((2, 20)).astype(np.float32)
    la, lb = (dmo.dm_layer(zern["ifs"], zern["pix"], zern["N"], v) for v in (a, b))
    lab = dmo.dm_layer(zern["ifs"], zern["pix"], zern["N"], (a.astype(np.float64) + b).astype(np.float32))
    assert np.abs(lab - (la + lb)).max() < 1e-5                       # float32 rounding of a + b only


def test_tilt_modes_reproduce_the_tilt_phase_of_the_input_module(zern):
    """Zernike 2 and 3 are x and y tilts: a command on them gives the plane wl.tilt_phase defines independently."""
    N, ifs, pix = zern["N"], zern["ifs"], zern["pix"]
    for mode, (ax, ay) in ((0, (1.0, 0.0)), (1, (0.0, 1.0))):
        plane = wl.tilt_phase(N, ax, ay).astype(np.float64).ravel()[pix]
        coeff = (plane @ ifs[mode].astype(np.float64)) / (ifs[mode].astype(np.float64) @ ifs[mode].astype(np.float64))
        cmd = np.zeros(20, np.float32); cmd[mode] = coeff
        lay = dmo.dm_layer(ifs, pix, N, cmd).ravel()[pix]
        assert np.abs(lay - plane).max() < 1e-5 * np.abs(plane).max()


def test_apply_scales_and_accumulates(zern):
    rng = np.random.default_rng(2)
    ph = rng.standard_normal((2, zern["N"], zern["N"])).astype(np.float32)
    cmd = rng.standard_normal((2, 20)).astype(np.float32)
    lay = dmo.dm_layer(zern["ifs"], zern["pix"], zern["N"], cmd)
    out = dmo.dm_apply(zern["ifs"], zern["pix"], ph, cmd, alpha=-0.5, beta=1.0)
    assert np.abs(out - (ph.astype(np.float64) - 0.5 * lay)).max() < 1e-12
    assert np.abs(dmo.dm_apply(zern["ifs"], zern["pix"], ph, cmd, alpha=2.0, beta=0.0) - 2.0 * lay).max() < 1e-12


def test_integrator_closed_forms():
    g = np.array([0.5, 0.25, 1.0], np.float32)
    const = np.tile(np.array([2.0, -4.0, 1.0], np.float32), (6, 1))
    out = dmo.integrator(g, 0, const)
    for t in range(6):                                                # constant input -> ramp (t + 1) g d
        assert np.allclose(out[t], (t + 1) * g * const[0])
    out2 = dmo.integrator(g, 2, const)                                # delay 2: same ramp, two frames late, zero before
    assert (out2[:2] == 0).all() and np.allclose(out2[2:], out[:4])
    imp = np.zeros((5, 3), np.float32); imp[1] = 1.0                  # impulse -> step (the integrator holds)
    assert np.allclose(dmo.integrator(g, 0, imp), np.array([[0, 0, 0]] + [list(g)] * 4))


@pytest.mark.parametrize("gain,delay", [(0.5, 0), (0.3, 1)])
def test_closed_loop_on_a_static_aberration_converges_at_the_known_rate(zern, gain, delay):
    """Loop: residual_t = a + layer(c_{t-1-delay'}), delta_t = -modal coefficients of the residual, integrator.
    With an exact modal 'sensor' (projection on the orthogonalised IFs) and delay 0 the residual coefficients obey
    e_t = (1 - g) e_{t-1}; with one frame of delay e_t = e_{t-1} - g e_{t-2}: both closed forms are checked."""
    N, ifs, pix = zern["N"], zern["ifs"].astype(np.float64), zern["pix"]
    P = np.linalg.pinv(ifs.T)                                         # modal coefficients of a pupil-plane phase
    rng = np.random.default_rng(3)
    a = rng.standard_normal(20)                                       # static aberration, in modes
    T = 12
    deltas = np.zeros((T, 20), np.float32)
    e_hist = []
    for t in range(T):
        cmds = dmo.integrator(np.full(20, gain, np.float32), delay, deltas[:t]) if t > 0 else np.zeros((0, 20))
        c_applied = cmds[t - 1] if t > 0 else np.zeros(20)            # the command computed after step t-1
        resid = (a @ ifs) + dmo.dm_layer(zern["ifs"], pix, N, c_applied.astype(np.float32)).ravel()[pix]
        e = P @ resid
        e_hist.append(e)
        deltas[t] = (-e).astype(np.float32)
    e_hist = np.array(e_hist)
    if delay == 0:
        for t in range(1, T):
            assert np.allclose(e_hist[t], (1 - gain) * e_hist[t - 1], atol=1e-5)
    else:
        for t in range(2, T):
            assert np.allclose(e_hist[t], e_hist[t - 1] - gain * e_hist[t - 2], atol=1e-5)
    assert np.abs(e_hist[-1]).max() < 0.05 * np.abs(e_hist[0]).max()


def test_zernike_generator_gives_unit_rms_and_known_low_orders():
    cfg = wl.CONFIGS["cfg2_flao"]
    A = wl.make_pupil(cfg)
    ifs, pix = wl.zernike_ifs(A, 54)                                  # PAPER.md Table 1: 54 Zernike modes
    assert ifs.shape == (54, int(A.sum())) and pix.size == int(A.sum())
    assert np.allclose((ifs.astype(np.float64) ** 2).mean(axis=1), 1.0, atol=1e-5)
    N = cfg.n_pupil
    c = (np.arange(N) - (N - 1) / 2.0)
    X, Y = np.meshgrid(c, c)
    x, y = X.ravel()[pix], Y.ravel()[pix]
    assert abs(np.corrcoef(ifs[0], x)[0, 1]) > 0.999999 and abs(np.corrcoef(ifs[1], y)[0, 1]) > 0.999999
    r2 = x * x + y * y
    assert abs(np.corrcoef(ifs[3], r2)[0, 1]) > 0.9999 or abs(np.corrcoef(ifs[2], r2)[0, 1]) > 0.9999   # defocus among n = 2
