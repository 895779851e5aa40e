"""ORACLE (test infrastructure, NOT the product) for SURVEY.md 8(f) row f1:
wavefront propagation through phase screens.

Plain numpy, float64, written from the definition; shares nothing with the CUDA
path (paper_1607_07624_b200/csrc/atmo_api.cu) and is imported only by
tests/, __graft_entry__.smoke() and bench.py's cpu_baseline leg.

What it follows.  The paper names the object and its wiring only: "Wavefront
propagation through phasescreens" is the first GPU-accelerated routine it lists
(section 6); `prop = factory.get_atmo_propagation(atmo, source)`
(PAPER.md:L235), layers are added to it one by one (L254-257) and its output
`prop.pupil_list` is the pyramid's input electric field (L317); the atmosphere
is a stack of layers with heights, wind speed and wind direction
(Table 1 `atmo`, `wind_speed`, `wind_direction`) seen from a
source at polar coordinates (L175-183).  The paper gives no formula; the
readings taken:

  F1a  frozen flow: layer l is a periodic G x G screen translated rigidly with
       velocity (vx_l, vy_l) [m/s]; at time t the pupil pixel (x, y) looks at
       screen coordinate  X = x + (-vx_l t + h_l tan_x) / pitch  (Y likewise),
       h_l the layer height and (tan_x, tan_y) the tangent of the source
       direction.  Source at infinity: no cone effect, no magnification; pupil
       and screens share the pixel pitch.
  F1b  the screen is sampled by BILINEAR interpolation of its four neighbours,
       indices taken modulo G (periodic screen).
  F1c  the layers are summed with unit weight (their strength is in the
       screens), then multiplied by one scale factor per sensing wavelength
       (screens hold phase at a reference wavelength; scale = lambda_ref/lambda).
  F1d  frame order: step-major, then source direction, then wavelength
       (SURVEY.md 8(d) cfg 5: "instance order star-major, lambda-minor").

Pins (tests/test_oracle_atmo.py): integer shifts equal numpy.roll; a linear ramp
is reproduced exactly; half-pixel shift equals the neighbour average; layer sum
and wavelength scale are linear; and the whole thing agrees with the independent
frozen-flow sampler of the input generator (workloads.phase_batch), which was
written before this file for the hot path's inputs.
"""
from __future__ import annotations

import numpy as np


def sample_coordinates(N, v_xy, height, tan_xy, t, pitch):
    """F1a: screen coordinates (X[x], Y[y]) [px] that the N pupil pixels see."""
    sx = (-float(v_xy[0]) * t + float(height) * float(tan_xy[0])) / pitch
    sy = (-float(v_xy[1]) * t + float(height) * float(tan_xy[1])) / pitch
    i = np.arange(N, dtype=np.float64)
    return i + sx, i + sy


def bilinear_periodic(screen, X, Y):
    """F1b: out[y][x] = bilinear sample of the periodic `screen` at (X[x], Y[y])."""
    scr = np.asarray(screen, dtype=np.float64)
    G = scr.shape[0]
    out = np.empty((Y.size, X.size), dtype=np.float64)
    for yi, Yv in enumerate(Y):
        y0 = int(np.floor(Yv))
        fy = Yv - y0
        r0 = scr[y0 % G]
        r1 = scr[(y0 + 1) % G]
        for xi, Xv in enumerate(X):
            x0 = int(np.floor(Xv))
            fx = Xv - x0
            a, b = x0 % G, (x0 + 1) % G
            out[yi, xi] = ((1.0 - fy) * ((1.0 - fx) * r0[a] + fx * r0[b])
                           + fy * ((1.0 - fx) * r1[a] + fx * r1[b]))
    return out


def bilinear_periodic_rows(screen, X, Y):
    """Same definition with the x loop written as numpy index arithmetic (the y
    loop stays): used for the larger parity samples.  Pinned to the scalar
    version above in the tests."""
    scr = np.asarray(screen, dtype=np.float64)
    G = scr.shape[0]
    x0 = np.floor(X).astype(np.int64)
    fx = X - x0
    a, b = x0 % G, (x0 + 1) % G
    out = np.empty((Y.size, X.size), dtype=np.float64)
    for yi, Yv in enumerate(Y):
        y0 = int(np.floor(Yv))
        fy = Yv - y0
        r0 = scr[y0 % G]
        r1 = scr[(y0 + 1) % G]
        out[yi] = ((1.0 - fy) * ((1.0 - fx) * r0[a] + fx * r0[b])
                   + fy * ((1.0 - fx) * r1[a] + fx * r1[b]))
    return out


def propagate(screens, pitch, wind_vxy, heights, dirs_tan, wl_scale, first_step, n_steps, dt, N,
              scalar=False):
    """F1a-F1d: phase[b][y][x], b = (step * n_dirs + dir) * n_wl + wl, float64.

    screens [L][G][G] (float32 values, widened exactly), wind_vxy [L][2] m/s,
    heights [L] m, dirs_tan [S][2], wl_scale [W]."""
    screens = np.asarray(screens)
    L = screens.shape[0]
    S, W = len(dirs_tan), len(wl_scale)
    out = np.empty((n_steps * S * W, N, N), dtype=np.float64)
    interp = bilinear_periodic if scalar else bilinear_periodic_rows
    for i in range(n_steps):
        t = (first_step + i) * dt
        for d in range(S):
            acc = np.zeros((N, N), dtype=np.float64)
            for l in range(L):
                X, Y = sample_coordinates(N, wind_vxy[l], heights[l], dirs_tan[d], t, pitch)
                acc += interp(screens[l], X, Y)
            for w in range(W):
                out[(i * S + d) * W + w] = acc * float(wl_scale[w])
    return out
