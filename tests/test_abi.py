"""The C-ABI library loads here (no GPU) and exports every symbol include/pwfs.h
declares; entry points that need no device behave as documented and the ones
that do fail loudly instead of falling back to a CPU path."""
import ctypes as C
import os
import re

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_1607_07624_b200 import build, pwfs
    build.build()                                   # nvcc cross-compiles without a GPU
    return pwfs.load_library()


def _declared_functions(header):
    src = open(os.path.join(ROOT, "include", header)).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(pwfs_[a-z0-9_]+)\s*\(", src)))


def test_header_symbols_are_exported(lib):
    from paper_1607_07624_b200 import atmo, chain, dm, peak, psf, pwfs, sh
    bindings = {"pwfs.h": pwfs.EXPORTS, "pwfs_atmo.h": atmo.EXPORTS, "pwfs_chain.h": chain.EXPORTS,
                "pwfs_psf.h": psf.EXPORTS, "pwfs_sh.h": sh.EXPORTS, "pwfs_dm.h": dm.EXPORTS,
                "pwfs_peak.h": peak.EXPORTS}
    assert sorted(os.listdir(os.path.join(ROOT, "include"))) == sorted(bindings)
    for header, exports in bindings.items():
        names = _declared_functions(header)
        so = peak.load_library() if header == "pwfs_peak.h" else lib    # the micro-benchmark is a library of its own
        for n in names:
            assert hasattr(so, n), f"{header}: {n} is not exported"
        assert sorted(exports) == names, header       # the binding covers the whole header
    assert not hasattr(lib, "pwfs_peak_fp32")         # ... and is NOT in the sensor library
    names = _declared_functions("pwfs.h")
    assert len(names) >= 14 and "pwfs_create" in names and "pwfs_run" in names and "pwfs_destroy" in names


def test_atmo_entry_points_reject_bad_arguments_without_a_device(lib):
    from paper_1607_07624_b200 import atmo, pwfs
    atmo._lib()
    h = C.c_void_p()
    assert lib.pwfs_atmo_create(None, C.byref(h)) == pwfs.PWFS_EINVAL
    scr = np.zeros((1, 8, 8), np.float32)
    z2, z1, one = np.zeros(2), np.zeros(1), np.ones(1)
    dp, fp = C.POINTER(C.c_double), C.POINTER(C.c_float)
    mk = lambda **kw: atmo.pwfs_atmo_params(**{**dict(
        n_layers=1, screen_px=8, screens=scr.ctypes.data_as(fp), pitch=0.1, wind_vxy=z2.ctypes.data_as(dp),
        heights=z1.ctypes.data_as(dp), n_dirs=1, dirs_tan=z2.ctypes.data_as(dp), n_wl=1,
        wl_scale=one.ctypes.data_as(dp), n_pupil=8, device=0), **kw})
    for bad in (dict(n_layers=0), dict(n_pupil=9), dict(pitch=0.0), dict(n_dirs=0), dict(n_wl=0), dict(pitch=float("nan"))):
        prm = mk(**bad)
        assert lib.pwfs_atmo_create(C.byref(prm), C.byref(h)) == pwfs.PWFS_EINVAL, bad
        assert h.value is None
    lib.pwfs_atmo_destroy(None)
    assert lib.pwfs_atmo_propagate(None, 0, 1, 1e-3, None, None) == pwfs.PWFS_EINVAL


def test_chain_entry_points_reject_bad_arguments_without_a_device(lib):
    from paper_1607_07624_b200 import chain, pwfs
    chain._lib()
    h = C.c_void_p()
    mk = lambda **kw: chain.pwfs_ccd_params(**{**dict(det_size=8, n_inst=1, n_int=1, gain=1.0, quantum_eff=0.5,
                                                      photon_noise=1, readout_noise=1, readout_level=1.0, seed=1,
                                                      device=0), **kw})
    assert lib.pwfs_ccd_create(None, C.byref(h)) == pwfs.PWFS_EINVAL
    for bad in (dict(det_size=0), dict(n_inst=0), dict(n_int=0), dict(gain=-1.0), dict(quantum_eff=1.5),
                dict(readout_level=float("nan")), dict(gain=float("inf"))):
        prm = mk(**bad)
        assert lib.pwfs_ccd_create(C.byref(prm), C.byref(h)) == pwfs.PWFS_EINVAL, bad
        assert h.value is None
    assert lib.pwfs_ccd_run(None, None, 1, 0, None, None) == pwfs.PWFS_EINVAL
    v = np.zeros((4, 4), np.uint8)
    assert lib.pwfs_slopec_create(4, C.c_void_p(v.ctypes.data), 0, None, 0, C.byref(h)) == pwfs.PWFS_EINVAL   # none valid
    v[1, 1] = 1
    assert lib.pwfs_slopec_create(4, C.c_void_p(v.ctypes.data), 2, None, 0, C.byref(h)) == pwfs.PWFS_EINVAL   # bad norm
    assert lib.pwfs_slopec_create(0, C.c_void_p(v.ctypes.data), 0, None, 0, C.byref(h)) == pwfs.PWFS_EINVAL
    assert lib.pwfs_slopec_run(None, None, 1, None, None) == pwfs.PWFS_EINVAL
    assert lib.pwfs_rec_create(0, 4, C.c_void_p(v.ctypes.data), 0, C.byref(h)) == pwfs.PWFS_EINVAL
    assert lib.pwfs_rec_create(4, 4, None, 0, C.byref(h)) == pwfs.PWFS_EINVAL
    assert lib.pwfs_rec_run(None, None, 1, None, None) == pwfs.PWFS_EINVAL
    for n in ("pwfs_ccd_destroy", "pwfs_slopec_destroy", "pwfs_rec_destroy"):
        getattr(lib, n)(None)                                                    # NULL-safe
    import torch
    if not torch.cuda.is_available():                                            # no device: loud failure, no fallback
        prm = mk()
        assert lib.pwfs_ccd_create(C.byref(prm), C.byref(h)) == pwfs.PWFS_ECUDA
        R = np.ones((2, 4), np.float32)
        assert lib.pwfs_rec_create(2, 4, C.c_void_p(R.ctypes.data), 0, C.byref(h)) in (pwfs.PWFS_ECUDA, pwfs.PWFS_ENOMEM)
        assert lib.pwfs_slopec_create(4, C.c_void_p(v.ctypes.data), 0, None, 0, C.byref(h)) in (pwfs.PWFS_ECUDA, pwfs.PWFS_ENOMEM)
        assert h.value is None


def test_psf_entry_points_reject_bad_arguments_without_a_device(lib):
    from paper_1607_07624_b200 import psf, pwfs
    psf._lib()
    h = C.c_void_p()
    amp = np.ones((16, 16), np.float32)
    fp = C.POINTER(C.c_float)
    mk = lambda **kw: psf.pwfs_psf_params(**{**dict(n_pupil=16, m_grid=128, pupil_amp=amp.ctypes.data_as(fp),
                                                    phase_scale=1.0, device=0), **kw})
    assert lib.pwfs_psf_create(None, C.byref(h)) == pwfs.PWFS_EINVAL
    for bad, code in ((dict(n_pupil=1), pwfs.PWFS_EINVAL), (dict(n_pupil=100), pwfs.PWFS_EINVAL),      # M < 2N
                      (dict(m_grid=96), pwfs.PWFS_EUNSUPPORTED), (dict(phase_scale=float("nan")), pwfs.PWFS_EINVAL),
                      (dict(pupil_amp=(0 * amp).ctypes.data_as(fp)), pwfs.PWFS_EINVAL)):
        prm = mk(**bad)
        assert lib.pwfs_psf_create(C.byref(prm), C.byref(h)) == code, bad
        assert h.value is None
    assert lib.pwfs_psf_accumulate(None, None, 1, None, None) == pwfs.PWFS_EINVAL
    assert lib.pwfs_psf_read(None, None, None, None) == pwfs.PWFS_EINVAL
    assert lib.pwfs_psf_reset(None, None) == pwfs.PWFS_EINVAL
    lib.pwfs_psf_destroy(None)
    import torch
    if not torch.cuda.is_available():
        prm = mk()
        assert lib.pwfs_psf_create(C.byref(prm), C.byref(h)) in (pwfs.PWFS_ECUDA, pwfs.PWFS_ENOMEM)
        assert h.value is None


def test_sh_entry_points_reject_bad_arguments_without_a_device(lib):
    from paper_1607_07624_b200 import pwfs, sh
    sh._lib()
    h = C.c_void_p()
    amp = np.ones((16, 16), np.float32)
    fp = C.POINTER(C.c_float)
    mk = lambda **kw: sh.pwfs_sh_params(**{**dict(n_pupil=16, n_subap=4, pupil_amp=amp.ctypes.data_as(fp), fft_px=8,
                                                  n_px=4, bin=2, illum_thresh=0.5, phase_scale=1.0, device=0), **kw})
    assert lib.pwfs_sh_create(None, C.byref(h)) == pwfs.PWFS_EINVAL
    for bad, code in ((dict(n_subap=5), pwfs.PWFS_EINVAL), (dict(fft_px=7), pwfs.PWFS_EINVAL),
                      (dict(fft_px=2), pwfs.PWFS_EINVAL),                      # P < b
                      (dict(n_px=5, bin=2), pwfs.PWFS_EINVAL),                 # window larger than the FFT grid
                      (dict(n_px=3, bin=1), pwfs.PWFS_EINVAL),                 # parity
                      (dict(fft_px=128), pwfs.PWFS_EUNSUPPORTED),
                      (dict(pupil_amp=(0 * amp).ctypes.data_as(fp)), pwfs.PWFS_EINVAL)):
        prm = mk(**bad)
        assert lib.pwfs_sh_create(C.byref(prm), C.byref(h)) == code, bad
        assert h.value is None
    assert lib.pwfs_sh_run(None, None, 1, None, None, None) == pwfs.PWFS_EINVAL
    assert lib.pwfs_sh_info(None, None, None) == pwfs.PWFS_EINVAL
    assert lib.pwfs_sh_valid_mask(None, None) == pwfs.PWFS_EINVAL
    lib.pwfs_sh_destroy(None)
    import torch
    if not torch.cuda.is_available():
        prm = mk()
        assert lib.pwfs_sh_create(C.byref(prm), C.byref(h)) in (pwfs.PWFS_ECUDA, pwfs.PWFS_ENOMEM)
        assert h.value is None


def test_ccd_params_struct_layout_matches_header():
    from paper_1607_07624_b200.chain import pwfs_ccd_params
    src = open(os.path.join(ROOT, "include", "pwfs_chain.h")).read()
    body = src[src.index("typedef struct {"):src.index("} pwfs_ccd_params;")]
    body = re.sub(r"/\*.*?\*/", "", body, flags=re.S)
    declared = re.findall(r"\b(?:int32_t|uint64_t|double)\s*(\w+);", body)
    assert declared == [f[0] for f in pwfs_ccd_params._fields_]
    assert C.sizeof(pwfs_ccd_params) == 64


def test_params_struct_layout_matches_header():
    from paper_1607_07624_b200.pwfs import pwfs_params
    fields = [f[0] for f in pwfs_params._fields_]
    src = open(os.path.join(ROOT, "include", "pwfs.h")).read()
    body = src[src.index("typedef struct {"):src.index("} pwfs_params;")]
    body = re.sub(r"/\*.*?\*/", "", body, flags=re.S)
    declared = re.findall(r"\b(?:int32_t|float|const float \*)\s*(\w+);", body)
    assert declared == fields
    assert C.sizeof(pwfs_params) == 48


def test_strerror_and_supported_grid(lib):
    from paper_1607_07624_b200 import pwfs
    assert pwfs.strerror(0) == "ok"
    assert "invalid" in pwfs.strerror(pwfs.PWFS_EINVAL)
    assert "memory" in pwfs.strerror(pwfs.PWFS_ENOMEM)
    assert "CUDA" in pwfs.strerror(pwfs.PWFS_ECUDA)
    assert "unknown" in pwfs.strerror(-99)
    for m in (128, 160, 192, 256, 288, 320, 384, 480, 512, 576, 640, 768, 800, 864, 960, 1024, 1152, 1280, 1440, 1536, 1600, 1728, 1920,
              2048):
        assert pwfs.supported_grid(m)
    for m in (0, 96, 100, 4096, 1000, 224, 352, 416, 448, 1056, 1088, 1664, 1792, 2016):
        assert not pwfs.supported_grid(m)


def test_null_and_invalid_arguments_do_not_crash(lib):
    from paper_1607_07624_b200 import pwfs
    h = C.c_void_p()
    assert lib.pwfs_create(None, C.byref(h)) == pwfs.PWFS_EINVAL
    amp = np.ones((8, 8), np.float32)
    prm = pwfs.pwfs_params(8, 10, amp.ctypes.data_as(C.POINTER(C.c_float)), 0, 1.0, 4, 0.0, 2, 0.5, 0, 0)
    assert lib.pwfs_create(C.byref(prm), C.byref(h)) == pwfs.PWFS_EINVAL      # M < 2N
    assert h.value is None
    prm.m_grid = 96
    assert lib.pwfs_create(C.byref(prm), C.byref(h)) == pwfs.PWFS_EUNSUPPORTED
    lib.pwfs_destroy(None)                                                      # NULL-safe
    assert lib.pwfs_info(None, None, None) == pwfs.PWFS_EINVAL
    assert lib.pwfs_run(None, None, 1, None, None, None) == pwfs.PWFS_EINVAL
    assert lib.pwfs_run_noalloc(None, None, 1, None, None, None) == pwfs.PWFS_EINVAL
    assert lib.pwfs_reserve(None, 1) == pwfs.PWFS_EINVAL
    assert "pwfs_run_noalloc" in pwfs.strerror(pwfs.PWFS_ELIMIT)
    assert lib.pwfs_last_cuda_error(None) == 0


def test_no_cpu_fallback_without_a_device(lib):
    """Without a CUDA device construction must raise (PWFS_ECUDA), never compute."""
    import torch
    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    from paper_1607_07624_b200.pwfs import PWFS, PwfsError, PWFS_ECUDA
    with pytest.raises(PwfsError) as ei:
        PWFS(np.ones((32, 32), np.float32), 128, 1.0, 4, 8)
    assert ei.value.code == PWFS_ECUDA


def test_result_changing_hooks_are_not_in_the_production_library(lib):
    """PWFS_DEBUG_T_ALIAS (wrong frames, PWFS_OK returned) and PWFS_REC_KSPLIT exist in -DPWFS_TUNING builds only
    (build.py --tuning -> libpwfs_tuning.so): the strings must not occur in libpwfs.so."""
    from paper_1607_07624_b200 import pwfs
    blob = open(pwfs.LIB_PATH, "rb").read()
    for name in (b"PWFS_DEBUG_T_ALIAS", b"PWFS_REC_KSPLIT"):
        assert name not in blob, name


def test_product_path_does_not_touch_the_oracle():
    pkg = os.path.join(ROOT, "paper_1607_07624_b200")
    for dirpath, _, files in os.walk(pkg):
        for fn in files:
            if fn.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, fn)).read()
                assert "_oracle" not in txt and "from oracle" not in txt and "import oracle" not in txt, fn
    otxt = "".join(open(os.path.join(ROOT, "oracle", fn)).read() for fn in os.listdir(os.path.join(ROOT, "oracle"))
                   if fn.endswith((".py", ".c", ".h")))
    assert "import paper_1607_07624_b200" not in otxt and "from paper_1607_07624_b200" not in otxt and "libpwfs.so" not in otxt
