"""Pins P2-P10 and P13 of SURVEY.md 8(c): the oracle's optics (O0-O6) and its
end-to-end output held against what the mathematics and the physics fix.
None of these re-types the oracle's formula: each is a conservation law, a
symmetry, a special case with a closed form, a different factorisation of the
operator, or a value stated in SURVEY.md before the oracle existed
(tests/golden/survey_scratch_values.json)."""
import math

import numpy as np
import pytest

from oracle import pwfs_oracle as orc
from paper_1607_07624_b200 import workloads as wl

CFG1 = wl.CONFIGS["cfg1_tiny"]


@pytest.fixture(scope="module")
def c1():
    cfg = CFG1
    A = wl.make_pupil(cfg)
    valid, nv = orc.valid_mask(A, cfg.n_subap)
    phi = wl.phase_batch(cfg, steps=1)[0]
    return dict(cfg=cfg, A=A, N=cfg.n_pupil, M=cfg.m_grid, K=cfg.mod_points,
                r=cfg.mod_radius, ns=cfg.n_subap, valid=valid.astype(bool), nv=nv, phi=phi)


def _to2d(vec, valid):
    g = np.zeros(valid.shape)
    g[valid] = vec
    return g


# ---------------------------------------------------------------- P2 --------
def test_parseval_through_both_transforms(c1, golden):
    A, phi, N, M = c1["A"], c1["phi"], c1["N"], c1["M"]
    mask = orc.pyramid_mask(M, M // 4)
    assert np.abs(np.abs(mask) - 1.0).max() < 1e-14            # phase-only mask
    dx, dy = orc.mod_offsets(c1["K"], c1["r"])
    E, F = orc.field(A, phi, M, dx[1], dy[1], mask, want_focal=True)
    lit = float((A.astype(np.float64) ** 2).sum())
    assert lit == golden["P2_cfg1_total_flux"]
    assert abs((np.abs(F) ** 2).sum() - M * M * lit) <= 1e-10 * M * M * lit   # forward unnormalised
    assert abs((np.abs(E) ** 2).sum() - lit) <= 1e-10 * lit                    # inverse has 1/M^2
    I = orc.intensity(A, phi, M, c1["K"], c1["r"])
    assert abs(I.sum() - lit) <= 1e-10 * lit                                   # mean over k, not sum


# ---------------------------------------------------------------- P3, P4 ----
def test_flat_phase_mirror_symmetry_and_equal_flux(c1, golden):
    A, N, M, ns = c1["A"], c1["N"], c1["M"], c1["ns"]
    flat = np.zeros((N, N), np.float32)
    I = orc.intensity(A, flat, M, c1["K"], c1["r"])
    scale = I.max()
    assert np.abs(I - I[:, ::-1]).max() <= 1e-12 * scale       # x -> M-1-x
    assert np.abs(I - I[::-1, :]).max() <= 1e-12 * scale       # y -> M-1-y
    assert np.abs(I - I.T).max() <= 1e-12 * scale              # K % 4 == 0, A symmetric under x<->y
    fr = orc.frame(I, N, M // 4, ns)
    a, b = fr[:ns, :ns], fr[:ns, ns:]
    c, d = fr[ns:, :ns], fr[ns:, ns:]
    # the four pupil images are mirror copies with equal flux (SURVEY P3 correction)
    assert np.abs(b - a[:, ::-1]).max() <= 1e-12 * fr.max()
    assert np.abs(c - a[::-1, :]).max() <= 1e-12 * fr.max()
    assert np.abs(d - a[::-1, ::-1]).max() <= 1e-12 * fr.max()
    for t in (a, b, c, d):
        assert abs(t.sum() - golden["P3_cfg1_flat_flux_per_pupil_image"]) < 1e-9
    # not pixel-identical: the images are not left-right symmetric individually
    assert np.abs(a - a[:, ::-1]).max() > 1e-3 * fr.max()
    s = orc.slopes(fr, c1["valid"].astype(np.uint8))
    assert np.abs(s).max() <= 1e-13                             # P4


def test_cfg4_pupil_is_mirror_but_not_transpose_symmetric():
    A = wl.make_pupil(wl.CONFIGS["cfg4_elt"])
    assert np.array_equal(A, A[:, ::-1]) and np.array_equal(A, A[::-1, :])
    assert not np.array_equal(A, A.T)


# ---------------------------------------------------------------- P5 --------
def test_tilt_sign_and_antisymmetry(c1):
    A, N, M, K, r, ns, valid, nv = (c1[k] for k in ("A", "N", "M", "K", "r", "ns", "valid", "nv"))
    _, sp = orc.pwfs_run(A, M, r, K, ns, wl.tilt_phase(N, +0.1))
    _, sm = orc.pwfs_run(A, M, r, K, ns, wl.tilt_phase(N, -0.1))
    sxp, syp = sp[0, :nv], sp[0, nv:]
    sxm = sm[0, :nv]
    assert sxp.mean() > 0.01                                   # reading A12: +x tilt => Sx > 0
    assert abs(syp.mean()) < 1e-12
    assert np.abs(_to2d(sxp, valid) + _to2d(sxm, valid)[:, ::-1]).max() < 1e-12
    _, sy = orc.pwfs_run(A, M, r, K, ns, wl.tilt_phase(N, 0.0, +0.1))
    assert sy[0, nv:].mean() > 0.01 and abs(sy[0, :nv].mean()) < 1e-12      # +y tilt => Sy > 0
    # x<->y exchange of the input transposes the response (A symmetric, K % 4 == 0)
    assert np.abs(_to2d(sy[0, nv:], valid) - _to2d(sxp, valid).T).max() < 1e-12


# ---------------------------------------------------------------- P6 --------
def test_small_tilt_linearity_and_survey_values(c1, golden):
    A, N, M, K, r, ns, nv = (c1[k] for k in ("A", "N", "M", "K", "r", "ns", "nv"))
    got = {}
    for alpha in (0.05, 0.1, 0.2):
        _, s = orc.pwfs_run(A, M, r, K, ns, wl.tilt_phase(N, alpha))
        got[alpha] = s[0, :nv].mean()
    for key, val in golden["P6_cfg1_mean_sx_vs_alpha"].items():
        assert abs(got[float(key)] - val) < 2e-6               # values stated to 6 decimals
    assert abs(got[0.1] / got[0.05] - 2.0) < 0.03
    assert got[0.2] / got[0.1] < 2.0                           # saturating, not growing


# ---------------------------------------------------------------- P7 --------
def test_identity_mask_returns_the_embedded_pupil(c1):
    A, phi, N, M = c1["A"], c1["phi"], c1["N"], c1["M"]
    I = orc.intensity(A, phi, M, 1, 0.0, s=0)                  # mask == 1, no modulation
    o = M // 2 - N // 2
    ref = np.zeros((M, M))
    ref[o:o + N, o:o + N] = A.astype(np.float64) ** 2
    assert np.abs(I - ref).max() < 1e-12


# ---------------------------------------------------------------- P8 --------
@pytest.mark.parametrize("s", [5, 32])
def test_single_face_ramp_is_a_circular_shift(c1, s):
    A, phi, N, M = c1["A"], c1["phi"], c1["N"], c1["M"]
    u = np.arange(M)
    us = np.where(u < M // 2, u, u - M)
    ramp_x = np.exp(2j * np.pi * s * us / M)                   # no |.|: one face along x
    mask = np.ones((M, 1)) * ramp_x[None, :]
    E = orc.field(A, phi, M, 0.3, -0.2, mask)
    G = orc.embed(orc.phasor(A, phi, 0.3, -0.2), M)
    assert np.abs(E - np.roll(G, -s, axis=1)).max() < 1e-12    # E[y][x] = G[y][x+s]
    mask_y = ramp_x[:, None] * np.ones((1, M))
    E = orc.field(A, phi, M, 0.3, -0.2, mask_y)
    assert np.abs(E - np.roll(G, -s, axis=0)).max() < 1e-12


# ---------------------------------------------------------------- P9 --------
def test_integer_bin_tilt_shifts_the_focal_plane(c1):
    A, phi, N, M = c1["A"], c1["phi"], c1["N"], c1["M"]
    ones = np.ones((M, M), complex)
    _, F0 = orc.field(A, phi, M, 0.0, 0.0, ones, want_focal=True)
    dx, dy = 3.0, -2.0                                         # M/N = 2 -> 6 and -4 bins
    _, Fk = orc.field(A, phi, M, dx, dy, ones, want_focal=True)
    o, c = M // 2 - N // 2, (N - 1) / 2.0
    const = np.exp(-2j * np.pi * (dx + dy) * (o + c) / N)
    ref = const * np.roll(np.roll(F0, int(dx * M / N), axis=1), int(dy * M / N), axis=0)
    assert np.abs(Fk - ref).max() <= 1e-10 * np.abs(F0).max()
    # +x tilt moves light towards +u: centroid check on a flat wavefront
    flat = np.zeros((N, N), np.float32)
    _, Ft = orc.field(A, flat, M, 2.0, 0.0, ones, want_focal=True)
    P = np.abs(Ft) ** 2
    v_pk, u_pk = np.unravel_index(np.argmax(P), P.shape)
    assert (v_pk, u_pk) == (0, 4)                              # PSF core at u = +2 l/D * M/N


# ---------------------------------------------------------------- P10 -------
@pytest.mark.parametrize("alpha", [0.1, 0.5, 1.0])
def test_geometric_optics_gain_with_well_sampled_modulation(c1, golden, alpha):
    A, N, M, ns, nv = (c1[k] for k in ("A", "N", "M", "ns", "nv"))
    _, s = orc.pwfs_run(A, M, 3.0, 48, ns, wl.tilt_phase(N, alpha))
    geo = 2.0 / math.pi * math.asin(alpha / 3.0)
    ratio = s[0, :nv].mean() / geo
    assert 0.95 < ratio < 1.10
    if alpha == 0.1:
        assert abs(ratio - golden["P10_geometric_gain"]["ratio_N64_M128_K48_r3"]) < 2e-3


def test_undersampled_modulation_value_from_survey(c1, golden):
    g = golden["P10_geometric_gain"]
    assert abs(2 / math.pi * math.asin(0.1 / 3.0) - g["cfg1_K12_alpha0.1_geometric"]) < 1e-6


# ---------------------------------------------------------------- P13 -------
@pytest.mark.parametrize("N,M", [(4, 8), (6, 12), (8, 16), (5, 12)])
def test_separable_circulant_operator_on_tiny_grids(N, M):
    """E = C G C^T with C = IDFT diag(a) DFT built by brute force: pins padding
    placement, both transform signs/scales, mask symmetry and [y][x] ordering
    in one identity that is factorised differently from the oracle."""
    rng = np.random.default_rng(N * 100 + M)
    A = (rng.random((N, N)) > 0.2).astype(np.float32)
    phi = rng.standard_normal((N, N)).astype(np.float32) * 2.0
    s = M // 4
    dx, dy = 0.7, -1.3
    j = np.arange(M)
    Wf = np.exp(-2j * np.pi * np.outer(j, j) / M)
    us = np.where(j < M // 2, j, j - M)
    a = np.exp(2j * np.pi * s * np.abs(us) / M)
    Cm = (np.conj(Wf) / M) @ np.diag(a) @ Wf
    c = (N - 1) / 2.0
    xx = np.arange(N) - c
    P = A.astype(np.float64) * np.exp(1j * (phi.astype(np.float64)
        + 2 * np.pi * (dx * xx[None, :] + dy * xx[:, None]) / N))
    o = M // 2 - N // 2
    G = np.zeros((M, M), complex)
    G[o:o + N, o:o + N] = P
    ref = Cm @ G @ Cm.T
    E = orc.field(A, phi, M, dx, dy, orc.pyramid_mask(M, s))
    assert np.abs(E - ref).max() < 1e-12
    En = orc.field(A, phi, M, dx, dy, orc.pyramid_mask(M, s), naive=True)
    assert np.abs(En - ref).max() < 1e-12


def test_mask_values_for_quarter_shift_are_powers_of_i():
    M = 16
    m = orc.pyramid_mask(M, M // 4)
    j = np.arange(M)
    us = np.abs(np.where(j < M // 2, j, j - M))
    ref = (1j) ** (us[None, :] + us[:, None])
    assert np.abs(m - ref).max() < 1e-14


def test_modulation_points(c1):
    dx, dy = orc.mod_offsets(12, 3.0, 0.0)
    assert abs(dx[0] - 3.0) < 1e-15 and abs(dy[0]) < 1e-15     # starts on +x
    assert abs(dx[3]) < 1e-15 and abs(dy[3] - 3.0) < 1e-15     # counter-clockwise
    assert np.allclose(np.hypot(dx, dy), 3.0)
    dx2, dy2 = orc.mod_offsets(12, 3.0, math.pi / 2)
    assert abs(dx2[0]) < 1e-15 and abs(dy2[0] - 3.0) < 1e-15


def test_unmodulated_single_point_equals_k_average_of_itself(c1):
    A, phi, N, M = c1["A"], c1["phi"], c1["N"], c1["M"]
    I1 = orc.intensity(A, phi, M, 1, 0.0)
    mask = orc.pyramid_mask(M, M // 4)
    E = orc.field(A, phi, M, 0.0, 0.0, mask)
    assert np.abs(I1 - np.abs(E) ** 2).max() < 1e-13
    # modulation is an average: K points at radius 0 give the same image
    I4 = orc.intensity(A, phi, M, 4, 0.0)
    assert np.abs(I4 - I1).max() < 1e-13


def test_whole_path_equals_composition_of_its_steps(c1):
    A, phi, N, M, K, r, ns, nv = (c1[k] for k in ("A", "phi", "N", "M", "K", "r", "ns", "nv"))
    frames, sl = orc.pwfs_run(A, M, r, K, ns, phi)
    I = orc.intensity(A, phi, M, K, r)
    fr = orc.frame(I, N, M // 4, ns)
    assert np.abs(frames[0] - fr).max() <= 1e-12 * fr.max()
    assert np.abs(sl[0] - orc.slopes(fr, c1["valid"].astype(np.uint8))).max() < 1e-12
    assert sl.shape == (1, 2 * nv)


def test_cfg4_geometry_values_from_survey(golden):
    """Full 40 m-class geometry (N480/M1024/K48/r4, spiders, b = 120/23): the
    fraction of a flat wavefront's flux that lands inside the four windows and
    the mean x-slope for a 0.1 l/D tilt, both stated in SURVEY.md P3/P10."""
    cfg = wl.CONFIGS["cfg4_elt"]
    A = wl.make_pupil(cfg)
    N, M, ns = cfg.n_pupil, cfg.m_grid, cfg.n_subap
    _, nv = orc.valid_mask(A, ns)
    frames, sl = orc.pwfs_run(A, M, cfg.mod_radius, cfg.mod_points, ns,
                              np.stack([np.zeros((N, N), np.float32), wl.tilt_phase(N, 0.1)]))
    lit = float(A.sum())
    assert abs(frames[0].sum() / lit - golden["P3_cfg4_flat_fraction_inside_windows"]) < 1e-4
    assert np.abs(sl[0]).max() < 1e-12                         # flat => zero slopes, mirror-symmetric pupil
    g = golden["P10_geometric_gain"]
    assert abs(sl[1, :nv].mean() - g["cfg4_alpha0.1_mean_sx"]) < 2e-6
    assert abs(2 / math.pi * math.asin(0.1 / 4.0) - g["cfg4_alpha0.1_geometric"]) < 1e-6
