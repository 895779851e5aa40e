"""CPU ORACLE of the deformable mirror (influence-function multiply) and the integrator
control -- the two objects that close PASSATA's loop after the reconstructor.

TEST INFRASTRUCTURE, NOT THE PRODUCT: only tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline leg may import this; the CUDA path (csrc/dm_api.cu) shares nothing with it.

What the paper says (it gives object names, wiring and parameters only):
  DM   Table 1 `dm`: type 'zernike', nmodes 54, npixels 160, obsratio,
       height; `dm = factory.get_dm(params.dm)`, input "dm.in_command = intc.out_comm"
       (L246, L265-266), output `dm.out_layer`, added to the propagation's layer list
       (`prop.add_layer_to_layer_list, dm.out_layer`, L257).  Sec. 6: "Influence function
       multiplication (from DM commands to applied wavefront)" is a GPU routine (L343); for
       an EELT "the influence functions matrix alone occupies between 4 and 5 GB" (L350).
  INT  Table 1 `control` (L144-152): type 'INT', delay (frames), int_gain (vector);
       "intc.in_delta_comm = rec.out_modes" (L265).
Readings:
  D1  layer[y][x] = sum_m ifs[m][p] * cmd[m] at the pixels p -> (y, x) = divmod(pix[p], N) the
      influence functions are defined on, zero elsewhere; ifs is [n_act][n_pix] row-major.
      Plain double-precision sum in the order m = 0, 1, ...
  D2  the layer is ADDED to the phase seen by the sensor with a scale alpha (the caller's
      sign convention and unit conversion): phase_out = beta * phase_in + alpha * layer.
  C1  integrator: state c_t = c_{t-1} + gain (.) delta_t, c_{-1} = 0 (element-wise gains).
  C2  delay d >= 0 whole frames: the command that leaves the control at step t is c_{t-d};
      zero while t < d.
"""
from __future__ import annotations

import numpy as np


def dm_layer(ifs, pix, n_pupil, cmd):
    """D1.  ifs [n_act][n_pix], pix [n_pix] flat indices y*N + x, cmd [B][n_act] -> [B][N][N] (float64)."""
    ifs = np.asarray(ifs, dtype=np.float32).astype(np.float64)
    cmd = np.atleast_2d(np.asarray(cmd, dtype=np.float32)).astype(np.float64)
    pix = np.asarray(pix, dtype=np.int64)
    n_act, n_pix = ifs.shape
    out = np.zeros((cmd.shape[0], n_pupil * n_pupil))
    for b in range(cmd.shape[0]):
        acc = np.zeros(n_pix)
        for m in range(n_act):                       # the definition, term by term
            acc += ifs[m] * cmd[b, m]
        out[b, pix] = acc
    return out.reshape(cmd.shape[0], n_pupil, n_pupil)


def dm_apply(ifs, pix, phase, cmd, alpha=1.0, beta=1.0):
    """D2.  phase [B][N][N] -> beta * phase + alpha * layer."""
    phase = np.asarray(phase, dtype=np.float32).astype(np.float64)
    return beta * phase + alpha * dm_layer(ifs, pix, phase.shape[-1], cmd)


def integrator(gain, delay, deltas):
    """C1, C2.  deltas [T][n_modes] -> commands [T][n_modes] that leave the control at steps 0..T-1."""
    gain = np.asarray(gain, dtype=np.float32).astype(np.float64)
    deltas = np.asarray(deltas, dtype=np.float32).astype(np.float64)
    T, n = deltas.shape
    c = np.zeros(n)
    hist = []
    out = np.zeros((T, n))
    for t in range(T):
        c = c + gain * deltas[t]
        hist.append(c.copy())
        if t - delay >= 0:
            out[t] = hist[t - delay]
    return out
