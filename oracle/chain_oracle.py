"""ORACLE (test infrastructure, NOT the product) for SURVEY.md 8(f) row f2: the
steps downstream of the pyramid -- CCD detector (integration, quantum
efficiency, photon and read-out noise), slope reference subtraction, modal
reconstructor.

Plain numpy / pure Python, float64, step by step; shares nothing with the CUDA
path (paper_1607_07624_b200/csrc/chain_api.cu) and is imported only by tests/,
__graft_entry__.smoke() and bench.py's cpu_baseline leg.

What it follows.  The paper names the objects, their wiring and their
parameters, no formula:
  * CCD: "a CCD processing object might integrate its input data for several
    simulation steps, and produce output data (pixel frames) at a lower rate"
    (section 2); Table 1 `detector`:
    size, dt "[s] Detector integration time", bandw, photon_noise "activate
    photon noise", readout_noise, readout_level "readout noise in
    [e-/pix/frame]", quantum_eff "quantum efficiency * total transmission";
    ccd.in_i = pyr.out_i (L318).
  * slope computer: Table 1 `slopec` (L137-143): pupdata_tag "tag of the pyramid
    WFS pupils", sn_tag "tag of the slope reference vector";
    sc.in_pixels = ccd.out_pixels (L261).
  * modal reconstructor: Table 1 `modalrec` (L212-215) recmat_tag
    "reconstruction matrix tag"; rec.in_slopes = sc.out_slopes (L262),
    intc.in_delta_comm = rec.out_modes (L265).

Readings taken:
  F2a  frames arrive step-major / instance-minor, b = step * n_inst + inst (the
       order f1 and pwfs_run use).  The detector sums n_int = dt_ccd / dt_loop
       consecutive steps of the same instance; output frame
       p = (step // n_int) * n_inst + inst.  n_steps must be a multiple of n_int.
  F2b  expected electrons per pixel: lam = quantum_eff * gain * sum_steps I,
       gain = photons per unit of intensity per step (the source object, which
       turns magnitude / bandw / dt into photons, is out of scope: its product
       enters as this one number).
  F2c  photon noise: k ~ Poisson(lam) from ONE uniform u by inversion (smallest
       k with u <= CDF(k), sequential search from 0) when lam < 128; for
       lam >= 128 the normal approximation k = max(0, floor(lam + sqrt(lam) z + 1/2)),
       z by Box-Muller.  lam <= 0 gives k = 0.  Off: k = lam (not rounded).
  F2d  read-out noise: + readout_level * z', z' a second Box-Muller normal.
       Pixels stay in electrons, float (no ADC, no clipping: the paper lists neither).
  F2e  random numbers: Philox4x32-10 (Salmon et al., SC'11), key = the 64-bit
       seed (lo, hi), counter = (pixel index y*D+x, output frame index lo, hi,
       0); of the four 32-bit words r0..r3, u = (r + 1/2) / 2^32 in (0, 1):
       u0 = inversion uniform or Box-Muller radius of z, u1 = angle of z,
       u2 = radius of z', u3 = angle of z';
       z = sqrt(-2 ln ua) cos(2 pi ub), all in double.
  F2f  slopes with reference: s = slopes(pixels) - sn, sn a vector of 2 n_valid
       numbers in the slope order of O9 (slopes() itself is the hot path's O9,
       oracle/pwfs_oracle.c orc_slopes, applied to the detector pixels).
  F2g  reconstructor: modes = recmat @ s, recmat [n_modes][2 n_valid] row-major.

Pins (tests/test_oracle_chain.py): Philox against the published known-answer
vectors of Random123; inversion against scipy.stats.poisson.ppf; Box-Muller
against the identity z^2 + z~^2 = -2 ln u and normal moments / KS; Poisson and
read-noise mean and variance; integration against a reshape-sum; noise off ==
qe * gain * sum; reference == slopes of the flat wavefront cancels; the
reconstructor against a pseudo-inverse of an interaction matrix measured with
the hot-path oracle (closed chain recovers small modal inputs).
"""
from __future__ import annotations

import math

import numpy as np

POISSON_SWITCH = 128.0   # F2c

_M0, _M1 = 0xD2511F53, 0xCD9E8D57          # Philox4x32 multipliers
_W0, _W1 = 0x9E3779B9, 0xBB67AE85          # Weyl key increments
_MASK = 0xFFFFFFFF


def philox4x32_10(counter, key):
    """F2e: ten rounds of Philox-4x32 on one counter (4 words) and key (2 words),
    pure Python integers.  Returns the 4 output words."""
    c0, c1, c2, c3 = (int(c) & _MASK for c in counter)
    k0, k1 = (int(k) & _MASK for k in key)
    for _ in range(10):
        p0 = _M0 * c0
        p1 = _M1 * c2
        hi0, lo0 = p0 >> 32, p0 & _MASK
        hi1, lo1 = p1 >> 32, p1 & _MASK
        c0, c1, c2, c3 = hi1 ^ c1 ^ k0, lo1, hi0 ^ c3 ^ k1, lo0
        k0 = (k0 + _W0) & _MASK
        k1 = (k1 + _W1) & _MASK
    return c0, c1, c2, c3


def philox_block(n_px, frame_index, seed):
    """F2e for every pixel of one output frame: uint32 array [n_px][4]
    (vectorised copy of philox4x32_10 over the pixel index; uint64 arithmetic)."""
    c0 = np.arange(n_px, dtype=np.uint64)
    c1 = np.full(n_px, int(frame_index) & _MASK, dtype=np.uint64)
    c2 = np.full(n_px, (int(frame_index) >> 32) & _MASK, dtype=np.uint64)
    c3 = np.zeros(n_px, dtype=np.uint64)
    k0, k1 = int(seed) & _MASK, (int(seed) >> 32) & _MASK
    m = np.uint64(_MASK)
    s32 = np.uint64(32)
    for _ in range(10):
        p0 = np.uint64(_M0) * c0
        p1 = np.uint64(_M1) * c2
        hi0, lo0 = p0 >> s32, p0 & m
        hi1, lo1 = p1 >> s32, p1 & m
        c0, c1, c2, c3 = hi1 ^ c1 ^ np.uint64(k0), lo1, hi0 ^ c3 ^ np.uint64(k1), lo0
        k0 = (k0 + _W0) & _MASK
        k1 = (k1 + _W1) & _MASK
    return np.stack([c0, c1, c2, c3], axis=1).astype(np.uint32)


def uniform01(r):
    """F2e: u = (r + 1/2) / 2^32, strictly inside (0, 1)."""
    return (np.asarray(r, dtype=np.float64) + 0.5) / 4294967296.0


def box_muller(ua, ub):
    """F2e: z = sqrt(-2 ln ua) cos(2 pi ub)."""
    return np.sqrt(-2.0 * np.log(ua)) * np.cos(2.0 * np.pi * ub)


def poisson_inversion(lam, u):
    """F2c, lam < POISSON_SWITCH: smallest k with u <= sum_{j<=k} e^-lam lam^j / j!,
    by sequential search from k = 0 (scalar, pure Python)."""
    if lam <= 0.0:
        return 0
    p = math.exp(-lam)
    s = p
    k = 0
    while u > s and k < 4096:      # the bound only guards against u beyond the rounded CDF's end
        k += 1
        p *= lam / k
        s += p
    return k


def poisson_counts(lam, u0, u1):
    """F2c for arrays: inversion below the switch, normal approximation above."""
    lam = np.asarray(lam, dtype=np.float64)
    out = np.zeros(lam.shape, dtype=np.float64)
    flat_l, flat_o = lam.ravel(), out.ravel()
    flat_u0, flat_u1 = np.asarray(u0).ravel(), np.asarray(u1).ravel()
    for i in range(flat_l.size):
        l = flat_l[i]
        if l <= 0.0:
            flat_o[i] = 0.0
        elif l < POISSON_SWITCH:
            flat_o[i] = poisson_inversion(float(l), float(flat_u0[i]))
        else:
            z = math.sqrt(-2.0 * math.log(flat_u0[i])) * math.cos(2.0 * math.pi * flat_u1[i])
            flat_o[i] = max(0.0, math.floor(l + math.sqrt(l) * z + 0.5))
    return out


def integrate(frames, n_inst, n_int):
    """F2a: frames [n_steps*n_inst][D][D] -> [n_steps/n_int * n_inst][D][D]."""
    frames = np.asarray(frames, dtype=np.float64)
    B, D = frames.shape[0], frames.shape[1]
    if B % n_inst or (B // n_inst) % n_int:
        raise ValueError("n_steps must be a multiple of n_int")
    n_out_steps = B // n_inst // n_int
    out = np.zeros((n_out_steps * n_inst, D, frames.shape[2]))
    for step in range(B // n_inst):
        for inst in range(n_inst):
            out[(step // n_int) * n_inst + inst] += frames[step * n_inst + inst]
    return out


def ccd(frames, n_inst=1, n_int=1, gain=1.0, quantum_eff=1.0, photon_noise=False,
        readout_noise=False, readout_level=0.0, seed=0, first_out_frame=0):
    """F2a-F2e: intensity frames -> detector pixels [electrons], float64."""
    acc = integrate(frames, n_inst, n_int)
    lam = quantum_eff * gain * acc
    P, D, D2 = lam.shape
    pix = np.empty_like(lam)
    for p in range(P):
        r = philox_block(D * D2, first_out_frame + p, seed)
        u = uniform01(r)
        l = lam[p].ravel()
        k = poisson_counts(l, u[:, 0], u[:, 1]) if photon_noise else l.copy()
        if readout_noise:
            k = k + readout_level * box_muller(u[:, 2], u[:, 3])
        pix[p] = k.reshape(D, D2)
    return pix


def slopes_with_reference(slopes, sn=None):
    """F2f: subtract the slope reference vector (sn_tag) from every frame's slopes."""
    s = np.asarray(slopes, dtype=np.float64)
    return s if sn is None else s - np.asarray(sn, dtype=np.float64)[None, :]


def reconstruct(recmat, slopes):
    """F2g: modes[b] = recmat @ slopes[b]."""
    R = np.asarray(recmat, dtype=np.float64)
    s = np.asarray(slopes, dtype=np.float64)
    return s @ R.T
