#!/usr/bin/env python
"""bench.py -- pyramid-WFS frames/s and fraction of roofline on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference]
                    [--config cfg4_elt] [--no-cpu-baseline] [--no-stages] [--no-configs] [--no-loops]

--gpus N > 1 without a launcher starts N ranks itself (torch.distributed.run on
127.0.0.1, one per GPU); under a launcher (WORLD_SIZE set) it must equal WORLD_SIZE.

One "step" = one pass of the whole hot path (phasor+tilt -> pad -> FFT2 -> mask
-> IFFT2 -> sum_k |E|^2 -> rebin -> slopes) over the full batch of the named
config (cfg4_elt: 100 frames x 48 modulation points), through the C ABI.
Prints ONE JSON line (rank 0).  See DESIGN.md "Measurement" for every field.
"""
from __future__ import annotations

import argparse
import json
import math
import os
import statistics
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from paper_1607_07624_b200 import workloads as wl  # noqa: E402

METRIC = "pyramid_wfs_frames_per_s"
UNIT = "frames/s"
# FP32 "alu" roofline: 148 SMs x 128 FP32 lanes x 2 flop/FMA x 1.965 GHz
FP32_PEAK_TFLOPS = 148 * 128 * 2 * 1.965e9 / 1e12
L2_FLUSH_BYTES = 256 << 20


def nominal_flops_per_modpoint(M: int) -> float:
    """2 transforms x 5 M^2 log2(M^2) per modulation point."""
    return 2.0 * 5.0 * M * M * math.log2(M * M)


class ClockSampler:
    """Samples SM clock and throttle reasons during the timed region (NVML)."""

    def __init__(self, index: int):
        self.index, self.samples, self.reasons, self.max_mhz = index, [], set(), None
        self._stop = threading.Event()
        self._thr = None
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM)
        except Exception:
            self.nv = None

    def _loop(self):
        nv = self.nv
        names = {}
        for nm in dir(nv):
            if nm.startswith("nvmlClocksThrottleReason") and isinstance(getattr(nv, nm), int):
                names[getattr(nv, nm)] = nm.replace("nvmlClocksThrottleReason", "")
        while not self._stop.is_set():
            try:
                self.samples.append(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM))
                mask = nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h)
                for bit, nm in names.items():
                    if bit and (mask & bit) == bit and nm not in ("None", "All"):
                        self.reasons.add(nm)
            except Exception:
                pass
            self._stop.wait(0.05)

    def start(self):
        if self.nv is not None:
            self._thr = threading.Thread(target=self._loop, daemon=True)
            self._thr.start()

    def stop(self) -> dict:
        self._stop.set()
        if self._thr is not None:
            self._thr.join()
        norm = {"GpuIdle": "gpu_idle", "ApplicationsClocksSetting": "applications_clocks_setting",
                "SwPowerCap": "sw_power_cap", "HwSlowdown": "hw_slowdown", "SyncBoost": "sync_boost",
                "SwThermalSlowdown": "sw_thermal_slowdown", "HwThermalSlowdown": "hw_thermal_slowdown",
                "HwPowerBrakeSlowdown": "hw_power_brake_slowdown", "DisplayClockSetting": "display_clock_setting"}
        return {"sm_mhz": statistics.median(self.samples) if self.samples else None,
                "sm_max_mhz": self.max_mhz, "samples": len(self.samples),
                "reasons": sorted(norm.get(r, r) for r in self.reasons if r != "GpuIdle")}


def time_oracle(cfg, frames: int):
    """The oracle as it stands on the host cores: seconds for `frames` frames."""
    from oracle import pwfs_oracle as orc
    A = wl.make_pupil(cfg)
    steps = max(1, math.ceil(frames / cfg.instances))
    phase = wl.phase_batch(cfg, steps=steps)[:frames]
    orc.valid_mask(A, cfg.n_subap)                       # library load / build outside the clock
    t0 = time.perf_counter()
    orc.pwfs_run(A, cfg.m_grid, cfg.mod_radius, cfg.mod_points, cfg.n_subap, phase)
    return time.perf_counter() - t0, orc.num_threads()


def oracle_sample_frames(cfg) -> int:
    """Frames the oracle gets through in roughly 10-30 s on ~8 cores."""
    cost = cfg.mod_points * 2 * cfg.m_grid ** 2 * math.log2(cfg.m_grid)      # ~ relative cost/frame
    ref = 48 * 2 * 1024 ** 2 * 10                                            # cfg4: ~3.5 s/frame on 8 cores
    return max(1, min(cfg.batch, int(round(4 * ref / cost))))


def measured_hbm_peak():
    """HBM GB/s from the driver-written MEASURED_PEAKS.json, else the profiling guide's fallback."""
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as fh:
            return float(json.load(fh)["hbm_gbs"]), "MEASURED_PEAKS.json hbm_gbs"
    except Exception:
        return 6550.0, "fallback (B200_PROFILING.md)"


def bench_stages(cfg, dev, phase, frames, flush, reps: int = 5, loops: bool = True) -> dict:
    """The rows of SURVEY.md 8(f) on this config's geometry, each timed alone with CUDA events on the
    launching stream (L2 flushed before every timed call) and set against the roofline that bounds it:
    algorithmic bytes / measured HBM copy bandwidth, or nominal flop / derived FP32 peak."""
    import torch
    from paper_1607_07624_b200.atmo import Atmosphere
    from paper_1607_07624_b200.chain import CCD, Reconstructor, SlopeComputer
    from paper_1607_07624_b200.dm import DeformableMirror, Integrator
    from paper_1607_07624_b200.psf import PsfCamera
    from paper_1607_07624_b200.sh import ShackHartmann
    from paper_1607_07624_b200.pwfs import from_config
    hbm, hbm_src = measured_hbm_peak()
    stream = torch.cuda.current_stream(dev)
    B, N, M = phase.shape[0], cfg.n_pupil, cfg.m_grid
    D = frames.shape[1]

    def timed(fn):
        for _ in range(2):
            fn()
        best = []
        for _ in range(reps):
            flush.zero_()
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record(stream)
            fn()
            b.record(stream)
            torch.cuda.synchronize(dev)
            best.append(a.elapsed_time(b))
        return statistics.median(best)

    def hbm_row(ms, nbytes, launches, note):
        gbs = nbytes / (ms * 1e-3) / 1e9
        return {"ms": ms, "bound": "hbm", "algorithmic_bytes": int(nbytes), "achieved": gbs, "peak": hbm, "unit": "GB/s",
                "frac": gbs / hbm, "launches": launches, "note": note}

    def alu_row(ms, flop, launches, note):
        tf = flop / (ms * 1e-3) / 1e12
        return {"ms": ms, "bound": "alu", "nominal_flop": float(flop), "achieved": tf, "peak": FP32_PEAK_TFLOPS,
                "unit": "TFLOP/s", "frac": tf / FP32_PEAK_TFLOPS, "launches": launches, "note": note}

    out = {"peak_source": {"hbm": hbm_src, "alu": "derived FP32 peak (DESIGN.md 7)"}, "frames": B}
    # f1: propagation through phase screens (frozen-flow configs only)
    if not cfg.independent_screens:
        atm = wl.atmosphere(cfg)
        L, S, W = atm["screens"].shape[0], len(atm["dirs_tan"]), len(atm["wl_scale"])
        n_steps = B // (S * W)
        with Atmosphere(**{k: v for k, v in atm.items() if k != "dt"}, device=dev.index) as a:
            buf = torch.empty_like(phase)
            ms = timed(lambda: a.propagate(0, n_steps, atm["dt"], out=buf))
        nbytes = n_steps * S * (W * N * N * 4 + L * (N + 1) * (N + 1) * 4)
        out["f1_atmo_propagate"] = hbm_row(ms, nbytes, 1, f"{L} layers, {S} dir x {W} wl, {n_steps} steps: N^2 floats out per "
                                           "frame + L (N+1)^2 screen samples in per direction")
    # f2: detector, slope computer, reconstructor
    with from_config(cfg, device=dev.index) as sensor:
        valid = sensor.valid_mask()
    nv = int(valid.sum())
    n_ph = 100.0 * D * D / 4                                       # ~100 photons per lit pixel
    with CCD(D, gain=n_ph / float((wl.make_pupil(cfg).astype(np.float64) ** 2).sum()), quantum_eff=0.32,
             photon_noise=True, readout_noise=True, readout_level=1.0, seed=1, device=dev.index) as ccd:
        pix = torch.empty_like(frames)
        ms = timed(lambda: ccd.run(frames, out=pix))
        out["f2_ccd"] = hbm_row(ms, B * D * D * 8, 1, "photon + read noise, n_int = 1: 4 B in + 4 B out per pixel")
    with SlopeComputer(valid, sn=np.zeros(2 * nv, np.float32), device=dev.index) as sc:
        sl = torch.empty((B, 2 * nv), dtype=torch.float32, device=dev)
        ms = timed(lambda: sc.run(pix, out=sl))
        out["f2_slopec"] = hbm_row(ms, B * (4 * nv * 4 + 2 * nv * 4), 1, "4 valid pixels in + 2 slopes out per subaperture")
    n_modes = min(4096, 2 * nv)
    rng = np.random.default_rng(0)
    R = rng.standard_normal((n_modes, 2 * nv), dtype=np.float32) / nv
    with Reconstructor(R, device=dev.index) as rec:
        modes = torch.empty((B, n_modes), dtype=torch.float32, device=dev)
        ms = timed(lambda: rec.run(sl, out=modes))
        ns = 2 * nv
        if B >= 24 and os.environ.get("PWFS_REC_TC", "1") != "0":   # chain_api.cu: batches run the tcgen05 TF32x3 kernel
            row = hbm_row(ms, n_modes * ns * 4 + B * ns * 4 + B * n_modes * 4, 3,
                          f"{n_modes} modes x {ns} slopes x {B} frames, tcgen05 TF32x3 (FP32 bar): algorithmic bytes = "
                          "recmat once + slopes in + modes out; the kernel streams recmat once as FP32 (TMA) and splits it "
                          "into TF32 hi/lo planes in tensor memory (A operand from TMEM), slope planes from a split kernel")
            row["tf32_tflops"] = 3 * 2.0 * B * n_modes * ns / (ms * 1e-3) / 1e12
            out["f2_rec_batch"] = row
        else:
            out["f2_rec_batch"] = alu_row(ms, 2.0 * B * n_modes * ns, 1, f"{n_modes} modes x {ns} slopes x {B} frames, FP32 FMA")
        m1 = torch.empty((1, n_modes), dtype=torch.float32, device=dev)
        ms = timed(lambda: rec.run(sl[:1], out=m1))
        out["f2_rec_gemv"] = hbm_row(ms, n_modes * 2 * nv * 4, 1, "one frame: recmat streamed once")
    # DM: influence-function multiply, one frame of commands -> phase layer added to the phase.
    # Random influence functions on the lit pixels (synthetic; 1024 actuators keep the matrix at ~0.6 GB here)
    Apup = wl.make_pupil(cfg)
    pix = np.flatnonzero(Apup.ravel() > 0).astype(np.int32)
    n_act = min(1024, n_modes)
    ifs = rng.standard_normal((n_act, pix.size), dtype=np.float32)
    with DeformableMirror(ifs, pix, N, device=dev.index) as dm:
        cmd1 = torch.zeros((1, n_act), dtype=torch.float32, device=dev)
        ph1 = phase[:1].clone()
        ms = timed(lambda: dm.apply(cmd1, ph1, alpha=1.0, beta=1.0))
        out["dm_apply"] = hbm_row(ms, n_act * pix.size * 4 + 2 * pix.size * 4, 1,
                                  f"{n_act} actuators x {pix.size} pupil pixels, one frame: the influence matrix streamed once")
    del ifs
    # the whole device chain as a loop runs it: one simulation step per iteration (f1 -> a1-a8 -> f2), n_inst frames
    if loops and not cfg.independent_screens:
        atm = wl.atmosphere(cfg)
        n_inst = len(atm["dirs_tan"]) * len(atm["wl_scale"])
        with Atmosphere(**{k: v for k, v in atm.items() if k != "dt"}, device=dev.index) as a, \
                from_config(cfg, device=dev.index) as sensor, \
                CCD(D, n_inst=n_inst, gain=n_ph / float((wl.make_pupil(cfg).astype(np.float64) ** 2).sum()), quantum_eff=0.32,
                    photon_noise=True, readout_noise=True, readout_level=1.0, seed=1, device=dev.index) as ccd, \
                SlopeComputer(valid, sn=np.zeros(2 * nv, np.float32), device=dev.index) as sc, \
                Reconstructor(R, device=dev.index) as rec:
            ph = torch.empty((n_inst, N, N), dtype=torch.float32, device=dev)
            fr = torch.empty((n_inst, D, D), dtype=torch.float32, device=dev)
            px, s1 = torch.empty_like(fr), torch.empty((n_inst, 2 * nv), dtype=torch.float32, device=dev)
            md = torch.empty((n_inst, n_modes), dtype=torch.float32, device=dev)
            n_loop = 50
            step = [0]

            def loop():
                for _ in range(n_loop):
                    a.propagate(step[0], 1, atm["dt"], out=ph)
                    sensor.run(ph, fr, want_slopes=False)
                    ccd.run(fr, first_out_frame=step[0] * n_inst, out=px)
                    sc.run(px, out=s1)
                    rec.run(s1, out=md)
                    step[0] += 1
            ms = timed(loop) / n_loop
            out["chain_loop_step"] = {"ms": ms, "steps_per_s": 1e3 / ms, "frames_per_step": n_inst, "launches": 8,
                                      "note": "closed-loop order, one step per iteration, all on the device: propagate -> "
                                              "pyramid (4 kernels) -> CCD -> slopes - reference -> modes (GEMV); eager "
                                              "launches, device time per step over 50 consecutive steps"}
            # the same 8 launches per step replayed from one CUDA graph of 10 consecutive steps (their own step indices
            # and noise frames): what a loop that submits whole blocks of steps pays per step
            n_cap = 10
            step[0] = 0
            sensor.reserve(n_inst)
            g = torch.cuda.CUDAGraph()
            side = torch.cuda.Stream(dev)
            side.wait_stream(stream)
            with torch.cuda.graph(g, stream=side):
                for _ in range(n_cap):
                    a.propagate(step[0], 1, atm["dt"], out=ph, stream=side)
                    sensor.run(ph, fr, want_slopes=False, stream=side)
                    ccd.run(fr, first_out_frame=step[0] * n_inst, out=px, stream=side)
                    sc.run(px, out=s1, stream=side)
                    rec.run(s1, out=md, stream=side)
                    step[0] += 1
            torch.cuda.synchronize(dev)

            def replay():
                for _ in range(n_loop // n_cap):
                    g.replay()
            ms_g = timed(replay) / n_loop
            out["chain_loop_step_graph"] = {"ms": ms_g, "steps_per_s": 1e3 / ms_g, "frames_per_step": n_inst,
                                            "steps_per_graph": n_cap,
                                            "note": "the same step captured 10 times (consecutive step indices) in one CUDA "
                                                    "graph; device time per step over 50 steps = 5 replays"}
            del g
        # the CLOSED loop of PAPER.md Table 2 (rec -> INT -> DM -> prop.add_layer): the DM layer of the delayed integrator
        # command is added to the propagated phase before the sensor; n_cl modes drive n_cl actuators
        n_cl = min(1024, n_modes)
        Rc = rng.standard_normal((n_cl, 2 * nv), dtype=np.float32) / nv
        ifc = rng.standard_normal((n_cl, pix.size), dtype=np.float32) * 1e-3
        with Atmosphere(**{k: v for k, v in atm.items() if k != "dt"}, device=dev.index) as a, \
                from_config(cfg, device=dev.index) as sensor, \
                CCD(D, n_inst=n_inst, gain=n_ph / float((Apup.astype(np.float64) ** 2).sum()), quantum_eff=0.32,
                    photon_noise=True, readout_noise=True, readout_level=1.0, seed=1, device=dev.index) as ccd, \
                SlopeComputer(valid, sn=np.zeros(2 * nv, np.float32), device=dev.index) as sc, \
                Reconstructor(Rc, device=dev.index) as rec, \
                Integrator(np.full(n_cl, -0.3, np.float32), delay=1, device=dev.index) as integ, \
                DeformableMirror(ifc, pix, N, device=dev.index) as dm:
            if n_inst == 1:                                    # single-conjugate loop: one sensor drives the mirror
                ph = torch.empty((1, N, N), dtype=torch.float32, device=dev)
                fr = torch.empty((1, D, D), dtype=torch.float32, device=dev)
                px, s1 = torch.empty_like(fr), torch.empty((1, 2 * nv), dtype=torch.float32, device=dev)
                md = torch.empty((1, n_cl), dtype=torch.float32, device=dev)
                cmd = torch.zeros((1, n_cl), dtype=torch.float32, device=dev)
                sensor.reserve(1)

                def cl_step(i, st=None):
                    a.propagate(i, 1, atm["dt"], out=ph, stream=st)
                    dm.apply(cmd, ph, alpha=1.0, beta=1.0, stream=st)
                    sensor.run(ph, fr, want_slopes=False, stream=st)
                    ccd.run(fr, first_out_frame=i, out=px, stream=st)
                    sc.run(px, out=s1, stream=st)
                    rec.run(s1, out=md, stream=st)
                    integ.step(md.reshape(-1), out=cmd, stream=st)
                for i in range(3):
                    cl_step(i)
                side = torch.cuda.Stream(dev)
                side.wait_stream(stream)
                g = torch.cuda.CUDAGraph()
                with torch.cuda.graph(g, stream=side):
                    for i in range(10):
                        cl_step(3 + i, side)
                torch.cuda.synchronize(dev)
                ms_e = timed(lambda: [cl_step(20 + i) for i in range(50)]) / 50
                ms_g = timed(lambda: [g.replay() for _ in range(5)]) / 50
                out["closed_loop_step"] = {"ms": ms_e, "ms_cuda_graph": ms_g, "steps_per_s": 1e3 / ms_g, "launches": 11,
                                           "modes": n_cl,
                                           "note": "PASSATA's SCAO loop, every object on the device: propagate -> + DM layer "
                                                   "(influence-function multiply, 2 launches) -> pyramid (4) -> CCD -> "
                                                   "slopes -> modes (GEMV) -> integrator (delay 1); eager / one CUDA graph of "
                                                   "10 steps, device time per step over 50 steps"}
                del g
        del Rc, ifc
    del R
    # f4: PSF camera on the same grid, Shack-Hartmann on the same pupil
    with PsfCamera(wl.make_pupil(cfg), M, phase_scale=0.45, device=dev.index) as cam:
        ms = timed(lambda: cam.accumulate(phase, want_sr=True))
        chunks = -(-B * M * ((N + 31) // 32 * 32) * 8 // (2 << 30))
        out["f4_psf"] = alu_row(ms, B * 5.0 * M * M * math.log2(M * M), 3 * chunks,
                                "one forward 2-D transform per frame, nominal 5 M^2 log2 M^2")
    b = next((c for c in (6, 5, 4, 8, 3, 2) if N % c == 0), 1)
    P, n_px, bin_ = (16, 8, 2) if b <= 8 else (32, 8, 4)
    with ShackHartmann(wl.make_pupil(cfg), N // b, P, n_px, bin_, phase_scale=0.45, device=dev.index) as sh:
        ms = timed(lambda: sh.run(phase))
        Dsh, Pc = sh.det_size, n_px * bin_
        flop = B * (N // b) ** 2 * 8.0 * b * Pc * (b + Pc)
        row_h = hbm_row(ms, B * (N * N * 4 + Dsh * Dsh * 4), 1, "")
        row_a = alu_row(ms, flop, 1, "")
        row = row_h if row_h["frac"] >= row_a["frac"] else row_a
        row["note"] = (f"{N // b}^2 subapertures of {b} px, P = {P}, {n_px}^2 detector px each: phase in + frame out "
                       f"({row_h['frac']:.3f} of HBM) vs direct-DFT FMAs ({row_a['frac']:.3f} of FP32)")
        out["f4_shack_hartmann"] = row
    return out


def run_reference(args, cfg):
    """--impl reference: the CPU oracle (this tier's reference arm), rank 0 only."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    frames = 1 if cfg.m_grid >= 800 else oracle_sample_frames(cfg)
    for _ in range(args.warmup):
        time_oracle(cfg, 1)
    tot, cores = 0.0, 0
    for _ in range(args.steps):
        dt, cores = time_oracle(cfg, frames)
        tot += dt
    value = frames * args.steps / tot
    sample = f"{frames} frame(s) of {cfg.name} per step, all {cfg.mod_points} modulation points"
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * tot / args.steps,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
            "data": "synthetic", "config": {"workload": cfg.name, "frames_per_step": frames},
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


class DryRunSensor:
    """--dry-run only: a CPU stand-in with the sensor's interface, so that the launch / sharding / timing /
    reporting plumbing of this file can be driven by a world-size-2 gloo test on a box without GPUs.  It
    computes nothing of the method (its "frames" are per-frame means of the phase) and its line says so."""

    def __init__(self, cfg):
        self.det_size, self.n_valid, self.cfg = cfg.det_size, 4, cfg

    def geometry(self, batch):
        return dict(n_cols=2 * self.cfg.n_pupil, k_unique=self.cfg.mod_points // 2 + 1, frames_per_chunk=batch, k_split=1)

    def run(self, phase, frames, slopes):
        frames[:] = phase.mean(dim=(1, 2))[:, None, None]
        slopes.zero_()
        return frames, slopes

    def set_timing(self, on):
        pass

    def get_timing(self):
        ks = ("xpass", "ypass", "xrebin", "slopes", "fused")
        return {k: 0.0 for k in ks}, {k: 0 for k in ks}

    def close(self):
        pass


def time_hot_path(sensor, phase, frames, slopes, steps, warmup, flush, stream, barrier, sampler=None):
    """W untimed calls, then K timed calls of sensor.run over the whole batch, each bracketed by CUDA events on the
    launching stream with the L2 flushed (untimed) before it; barrier + synchronize on both sides.  Returns
    (summed ms over the K steps on this rank, per-kernel ms, per-kernel launch counts, clock record)."""
    import torch
    for _ in range(warmup):
        sensor.run(phase, frames, slopes)
    barrier()
    sensor.get_timing()                                  # reset counters
    sensor.set_timing(True)
    if sampler is not None:
        sampler.start()
    barrier()
    if stream is None:                                   # --dry-run: no device, wall clock
        t0 = time.perf_counter()
        for _ in range(steps):
            sensor.run(phase, frames, slopes)
        ms_total = (time.perf_counter() - t0) * 1e3
        barrier()
    else:
        ev0 = [torch.cuda.Event(enable_timing=True) for _ in range(steps)]
        ev1 = [torch.cuda.Event(enable_timing=True) for _ in range(steps)]
        for i in range(steps):
            flush.zero_()                                # evict L2 between timed steps (not timed)
            ev0[i].record(stream)
            sensor.run(phase, frames, slopes)
            ev1[i].record(stream)
        barrier()
        ms_total = sum(a.elapsed_time(b) for a, b in zip(ev0, ev1))
    clocks = sampler.stop() if sampler is not None else None
    kernel_ms, launches = sensor.get_timing()
    sensor.set_timing(False)
    return ms_total, kernel_ms, launches, clocks


def roofline_numbers(cfg, geo, B, steps, ms_per_step, kernel_ms, launches, peak_tflops):
    """Fractions of the FP32 roofline from one timed run: the whole path against the nominal 2 x 5 M^2 log2 M^2
    flop per modulation point, and the dominant kernel against its half of that."""
    M, K = cfg.m_grid, cfg.mod_points
    dom = max(kernel_ms, key=kernel_ms.get)
    n_launch = max(1, launches[dom])
    units_per_launch = B * K * steps / n_launch                          # modulation points per launch
    share = {"xpass": 0.5, "ypass": 0.5, "fused": 1.0}.get(dom, 0.0)
    flops_per_launch = share * nominal_flops_per_modpoint(M) * units_per_launch
    avg_launch_s = kernel_ms[dom] * 1e-3 / n_launch
    achieved = flops_per_launch / avg_launch_s / 1e12 if avg_launch_s > 0 else 0.0
    path_tflops = nominal_flops_per_modpoint(M) * B * K / (ms_per_step * 1e-3) / 1e12
    return {"kernel": dom, "achieved": achieved, "frac": achieved / peak_tflops, "launch_ms": avg_launch_s * 1e3,
            "launches": n_launch, "nominal_flops_per_launch": flops_per_launch, "path_achieved": path_tflops,
            "path_frac": path_tflops / peak_tflops,
            # 1-D transform pairs executed / the 2 K M pairs the nominal count assumes (shared x-pass, pupil rows
            # and window columns only): path_frac above this ratio x pipe utilisation is algorithmic saving
            "executed_pair_ratio": (geo["k_unique"] * cfg.n_pupil + K * geo["n_cols"]) / (2.0 * K * M),
            "kernel_ms_per_step": {k: v / steps for k, v in kernel_ms.items()}}


def latency_per_call(sensor, phase_b, dev, stream, reps: int = 100) -> dict:
    """Device time of ONE pwfs_run call on a small batch (the closed loop's per-step call: 1 frame, or a config's
    sensor instances), back to back on one stream: eager launches, and the same call replayed from a CUDA graph."""
    import torch
    b = phase_b.shape[0]
    fr = torch.empty((b, sensor.det_size, sensor.det_size), dtype=torch.float32, device=dev)
    sl = torch.empty((b, 2 * sensor.n_valid), dtype=torch.float32, device=dev)

    def timed(fn):
        for _ in range(5):
            fn()
        torch.cuda.synchronize(dev)
        a, e = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record(stream)
        for _ in range(reps):
            fn()
        e.record(stream)
        torch.cuda.synchronize(dev)
        return a.elapsed_time(e) / reps

    eager_ms = timed(lambda: sensor.run(phase_b, fr, sl))
    graph = torch.cuda.CUDAGraph()
    with torch.cuda.graph(graph):                        # pwfs_run only enqueues kernels: capturable as is
        sensor.run(phase_b, fr, sl)
    graph_ms = timed(graph.replay)
    del graph
    geo = sensor.geometry(b)
    return {"frames_per_call": b, "eager_ms": eager_ms, "cuda_graph_ms": graph_ms, "calls": reps,
            "k_split": geo["k_split"], "us_per_frame_cuda_graph": 1e3 * graph_ms / b,
            "note": "back-to-back calls on one stream, device time per call (CUDA events)"}


def bench_other_configs(main_name, dev, flush, steps, warmup) -> dict:
    """Every BASELINE.json config timed like the headline one (full batch per step, warm-up, L2 flushed before each
    timed step, CUDA events, per-kernel brackets): frames/s, ms per step, fraction of the FP32 roofline for the path
    and for the dominant kernel.  Frozen-flow inputs come from the f1 device kernel on the same seeded screens."""
    import torch
    from paper_1607_07624_b200.atmo import Atmosphere
    from paper_1607_07624_b200.pwfs import from_config
    stream = torch.cuda.current_stream(dev)
    out = {}
    for name in wl.CONFIG_ORDER:
        if name == main_name:
            continue
        cfg = wl.CONFIGS[name]
        if cfg.independent_screens:
            phase = torch.from_numpy(wl.phase_batch(cfg)).to(dev)
            src = "numpy generator (independent screens)"
        else:
            atm = wl.atmosphere(cfg)
            with Atmosphere(**{k: v for k, v in atm.items() if k != "dt"}, device=dev.index) as a:
                phase = a.propagate(0, cfg.steps, atm["dt"])
                torch.cuda.synchronize(dev)
            src = "f1 device propagation of the seeded screens"
        B = phase.shape[0]
        with from_config(cfg, device=dev.index) as sensor:
            geo = sensor.geometry(B)
            D, nv = sensor.det_size, sensor.n_valid
            frames = torch.empty((B, D, D), dtype=torch.float32, device=dev)
            slopes = torch.empty((B, 2 * nv), dtype=torch.float32, device=dev)
            sync = lambda: torch.cuda.synchronize(dev)
            ms_total, kernel_ms, launches, _ = time_hot_path(sensor, phase, frames, slopes, steps, warmup, flush, stream, sync)
            lat_step = latency_per_call(sensor, phase[:cfg.instances].contiguous(), dev, stream)   # one simulation step
        ms = ms_total / steps
        r = roofline_numbers(cfg, geo, B, steps, ms, kernel_ms, launches, FP32_PEAK_TFLOPS)
        out[name] = {"frames_per_step": B, "frames_per_s": B / (ms * 1e-3), "ms_per_step": ms,
                     "modpoint_ffts_per_s": B * cfg.mod_points / (ms * 1e-3), "m_grid": cfg.m_grid, "n_pupil": cfg.n_pupil,
                     "mod_points": cfg.mod_points, "frames_per_chunk": geo["frames_per_chunk"], "k_split": geo["k_split"],
                     "path_frac": r["path_frac"], "dominant_kernel": r["kernel"], "dominant_frac": r["frac"],
                     "executed_pair_ratio": r["executed_pair_ratio"], "kernel_ms_per_step": r["kernel_ms_per_step"],
                     "steps": steps, "warmup": warmup, "input": src, "latency_step": lat_step}
        del phase, frames, slopes
    return out


def measure_fp32_peak(local: int) -> dict:
    """pwfs_peak_fp32 (FFMA and FFMA2 streams on every SM) with the SM clock sampled while it runs."""
    from paper_1607_07624_b200.peak import peak_fp32
    sampler = ClockSampler(local)
    sampler.start()
    res = {}
    for _ in range(3):                                   # ~50 ms each: long enough for a few clock samples
        for nm, packed in (("ffma", False), ("ffma2", True)):
            tf, ms = peak_fp32(local, packed)
            res[nm] = max(res.get(nm, 0.0), tf)
    clk = sampler.stop()
    best = max(res.values())
    return {"tflops": best, "ffma_tflops": res["ffma"], "ffma2_tflops": res["ffma2"], "sm_mhz": clk["sm_mhz"],
            "how": "pwfs_peak_fp32 (libpwfs_peak.so): independent FFMA / FFMA2 chains, 64 warps per SM, best of 3 x 5 launches, CUDA events"}


def run_ours(args, cfg):
    import torch
    import torch.distributed as dist
    from paper_1607_07624_b200 import sharding

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if world != args.gpus:
        raise SystemExit(f"bench.py: --gpus {args.gpus} but WORLD_SIZE={world}: launch one rank per GPU "
                         f"(python bench.py --gpus N starts them itself)")
    dry = args.dry_run
    if dry:
        dev = torch.device("cpu")
    else:
        if not torch.cuda.is_available():
            raise SystemExit("bench.py: no CUDA device (the product path has no CPU fallback)")
        if torch.cuda.device_count() < world:
            raise SystemExit(f"bench.py: --gpus {world} needs {world} CUDA devices, this node has {torch.cuda.device_count()}")
        torch.cuda.set_device(local)
        dev = torch.device("cuda", local)
    if world > 1:
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        if dry:
            dist.init_process_group("gloo")
        else:
            dist.init_process_group("nccl", device_id=dev)

    # weak scaling: the job is world x (the config's batch); rank r owns the contiguous block of frames
    # sharding.my_frames gives it (whole simulation steps), i.e. its own seeded slice of time.  No data-path
    # collective: outputs stay on the GPU that holds their inputs.
    B_cfg = cfg.batch
    lo, hi = sharding.my_frames(world * B_cfg)
    assert lo % cfg.instances == 0 and hi - lo == B_cfg
    phase_np = wl.phase_batch(cfg, steps=(hi - lo) // cfg.instances, first_step=lo // cfg.instances)
    B = phase_np.shape[0]
    if dry:
        sensor = DryRunSensor(cfg)
    else:
        from paper_1607_07624_b200.pwfs import from_config
        sensor = from_config(cfg, device=local)
    geo = sensor.geometry(B)
    phase = torch.from_numpy(phase_np).to(dev)
    D, nv = sensor.det_size, sensor.n_valid
    frames = torch.empty((B, D, D), dtype=torch.float32, device=dev)
    slopes = torch.empty((B, 2 * nv), dtype=torch.float32, device=dev)
    flush = None if dry else torch.empty(L2_FLUSH_BYTES, dtype=torch.uint8, device=dev)
    stream = None if dry else torch.cuda.current_stream(dev)

    def barrier():
        if not dry:
            torch.cuda.synchronize(dev)
        if world > 1:
            dist.barrier()
            if not dry:
                torch.cuda.synchronize(dev)

    def max_over_ranks(x: float) -> float:
        return sharding.max_over_ranks(x, dev)

    # ---- device-resident timing (value) -------------------------------------
    sampler = None if dry else ClockSampler(local)
    ms_rank, kernel_ms, launches, clocks = time_hot_path(sensor, phase, frames, slopes, args.steps, args.warmup, flush,
                                                         stream, barrier, sampler)
    ms_total = max_over_ranks(ms_rank)
    ms_per_step = ms_total / args.steps
    value = world * B * args.steps / (ms_total * 1e-3)
    per_rank = None
    if world > 1:                                        # every rank's own frames/s, gathered for the report
        t = torch.tensor([B * args.steps / (ms_rank * 1e-3)], dtype=torch.float64, device=dev)
        allv = [torch.zeros_like(t) for _ in range(world)]
        dist.all_gather(allv, t)
        per_rank = [float(v.item()) for v in allv]

    if dry:
        if rank == 0:
            print(json.dumps({"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
                              "warmup": args.warmup, "ms_per_step": ms_per_step, "higher_is_better": True,
                              "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
                              "dry_run": True, "per_rank_frames_per_s": per_rank,
                              "config": {"workload": cfg.name, "frames_per_step": world * B, "frames_per_rank": B,
                                         "first_frame_of_rank0": lo,
                                         "parallelism": f"frames sharded over {world} rank(s), no collective"},
                              "note": "--dry-run: CPU stand-in sensor, plumbing test only, NOT a measurement",
                              "gpu_launches": 0}), flush=True)
        if world > 1:
            dist.barrier()
            dist.destroy_process_group()
        return

    # ---- closed-loop latency: one frame per call (B = 1), eager and replayed from a CUDA graph
    latency = None
    if rank == 0:
        latency = latency_per_call(sensor, phase[:1].contiguous(), dev, stream)
        latency_step = latency if cfg.instances == 1 else latency_per_call(sensor, phase[:cfg.instances].contiguous(), dev, stream)

    # ---- end to end through the host-buffer entry point (e2e) ----------------
    h_phase = torch.from_numpy(phase_np).pin_memory()
    h_frames = torch.empty((B, D, D), dtype=torch.float32).pin_memory()
    h_slopes = torch.empty((B, 2 * nv), dtype=torch.float32).pin_memory()
    for _ in range(max(1, args.warmup // 2)):
        sensor.run_host(h_phase, h_frames, h_slopes)
    barrier()
    t0 = time.perf_counter()
    for _ in range(args.steps):
        sensor.run_host(h_phase, h_frames, h_slopes)     # synchronous: returns when results are on the host
    barrier()
    e2e_s = max_over_ranks(time.perf_counter() - t0)
    e2e_value = world * B * args.steps / e2e_s
    same = bool(np.array_equal(h_frames.numpy(), frames.cpu().numpy()))

    if rank == 0:
        M, K = cfg.m_grid, cfg.mod_points
        r = roofline_numbers(cfg, geo, B, args.steps, ms_per_step, kernel_ms, launches, FP32_PEAK_TFLOPS)
        dom, n_launch = r["kernel"], r["launches"]
        traffic, traffic_src = None, None                                # dram bytes per launch, from the committed ncu capture
        tpath = os.path.join(ROOT, "profiles", "traffic.csv")
        if os.path.exists(tpath):
            import csv
            with open(tpath) as fh:
                for row in csv.DictReader(fh):
                    if row["config"] == cfg.name and row["kernel"] == dom:
                        per_frame = float(row["dram_bytes_per_launch"]) / float(row["frames_per_launch"])
                        traffic = per_frame * B * args.steps / n_launch
                        traffic_src = ("copied from profiles/traffic.csv, not measured by this run -- " + row["source"])
        peak_m = measure_fp32_peak(local)
        roof = {"bound": "alu", "kernel": dom, "achieved": r["achieved"], "peak": FP32_PEAK_TFLOPS,
                "unit": "TFLOP/s", "frac": r["frac"], "traffic": traffic, "traffic_source": traffic_src,
                "peak_source": "derived: 148 SM x 128 FP32 lanes x 2 x 1.965 GHz (guide unit counts/clocks)",
                "peak_measured": peak_m["tflops"], "peak_measured_detail": peak_m,
                "frac_vs_measured": r["achieved"] / peak_m["tflops"],
                "path_frac_vs_measured": r["path_achieved"] / peak_m["tflops"]}
        roof.update({k: r[k] for k in ("launch_ms", "launches", "nominal_flops_per_launch", "path_achieved", "path_frac",
                                       "executed_pair_ratio", "kernel_ms_per_step")})
        roof["kernel_ms_note"] = ("CUDA events around every launch; xrebin and slopes of chunk c run on a side stream "
                                  "under the row pass of chunk c+1, so their bracketed times include waiting for SM "
                                  "slots and overlap xpass")
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": ms_per_step, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
            "config": {"workload": cfg.name, "n_pupil": cfg.n_pupil, "m_grid": M, "mod_points": K,
                       "mod_radius": cfg.mod_radius, "n_subap": cfg.n_subap, "frames_per_step": world * B,
                       "frames_per_rank": B,
                       "frames_per_chunk": geo["frames_per_chunk"], "k_split": geo["k_split"],
                       "k_unique_xtilts": geo["k_unique"], "columns_computed": geo["n_cols"],
                       "l2": f"flushed between timed steps ({L2_FLUSH_BYTES >> 20} MiB memset, untimed)",
                       "parallelism": f"frames sharded over {world} GPU(s), no collective"},
            "modpoint_ffts_per_s": value * K,
            "transforms_2d_per_s": 2 * value * K,
            "per_rank_frames_per_s": per_rank,
            "roofline": roof,
            "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": int(h_phase.numel() * 4) * world,
                    "d2h_bytes_per_step": int(h_frames.numel() * 4 + h_slopes.numel() * 4) * world,
                    "matches_device_path": same},
            "gpu_launches": int(sum(launches.values())),
            "latency_b1": latency,
            "clocks": clocks,
        }
        if not args.no_configs and world == 1:
            line["configs"] = bench_other_configs(cfg.name, dev, flush, steps=max(3, min(args.steps, 5)), warmup=3)
            line["configs"][cfg.name] = {
                "frames_per_step": B, "frames_per_s": value, "ms_per_step": ms_per_step, "modpoint_ffts_per_s": value * K,
                "m_grid": M, "n_pupil": cfg.n_pupil, "mod_points": K, "frames_per_chunk": geo["frames_per_chunk"],
                "k_split": geo["k_split"], "path_frac": r["path_frac"], "dominant_kernel": dom, "dominant_frac": r["frac"],
                "executed_pair_ratio": r["executed_pair_ratio"], "kernel_ms_per_step": r["kernel_ms_per_step"],
                "steps": args.steps, "warmup": args.warmup, "input": "numpy generator (the headline run above)",
                "latency_step": latency_step}
        if not args.no_stages:
            line["stages"] = bench_stages(cfg, dev, phase, frames, flush, loops=not args.no_loops)
        if not args.no_cpu_baseline:
            nfr = oracle_sample_frames(cfg)
            dt, cores = time_oracle(cfg, nfr)
            line["cpu_baseline"] = {"value": nfr / dt, "unit": UNIT, "cores": cores, "kind": "oracle",
                                    "sample": f"{nfr} frame(s) of {cfg.name}, all {K} modulation points, {dt:.1f} s"}
        print(json.dumps(line), flush=True)
    sensor.close()
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()


def spawn_ranks(args) -> None:
    """`python bench.py --gpus N` without a launcher: start N ranks of this file on this node (one per GPU) the way
    the driver does -- torch.distributed.run, rendezvous on 127.0.0.1 -- and replace this process by the launcher."""
    import socket
    if not args.dry_run:
        import torch
        n_dev = torch.cuda.device_count() if torch.cuda.is_available() else 0
        if n_dev < args.gpus:
            raise SystemExit(f"bench.py: --gpus {args.gpus} needs {args.gpus} CUDA devices, this node has {n_dev}")
    with socket.socket() as sk:
        sk.bind(("127.0.0.1", 0))
        port = sk.getsockname()[1]
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}",
           "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:]
    sys.stdout.flush()
    os.execv(sys.executable, cmd)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", choices=["ours", "reference"], default="ours")
    ap.add_argument("--config", default="cfg4_elt", choices=wl.CONFIG_ORDER)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-stages", action="store_true", help="skip the per-stage timings of the 8(f) rows")
    ap.add_argument("--no-configs", action="store_true", help="skip the timings of the other four configs")
    ap.add_argument("--no-loops", action="store_true",
                    help="stage timings without the chain / closed-loop rows (thousands of single-frame launches; for profiling runs)")
    ap.add_argument("--dry-run", action="store_true",
                    help="CPU stand-in sensor on gloo: exercises launch/sharding/timing/report plumbing only")
    args = ap.parse_args()
    if args.steps < 1 or args.warmup < 0:
        raise SystemExit("bench.py: need --steps >= 1 and --warmup >= 0")
    cfg = wl.CONFIGS[args.config]
    if args.gpus < 1:
        raise SystemExit("bench.py: need --gpus >= 1")
    if args.impl == "reference":
        run_reference(args, cfg)
    elif args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        spawn_ranks(args)
    else:
        run_ours(args, cfg)


if __name__ == "__main__":
    main()
