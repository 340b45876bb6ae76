#!/usr/bin/env python
"""bench.py — throughput of the Shifted-Fresnel hot path on B200 (BASELINE.json `metric`).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl sfd|reference] [--config 1|2|4]
    python bench.py --peaks          # measured pipe rates of this GPU (sfd_measure_pipes), one JSON line

Started bare with --gpus N > 1 (no WORLD_SIZE in the environment) it launches its N ranks itself, one
process per GPU, rendezvous on 127.0.0.1; under torchrun it is one of the ranks.

A *step* is one pass of the whole hot path (convert, pre-chirp,
zero-pad, forward FFT, kernel-spectrum multiply, inverse FFT, crop, post-chirp, |u|^2) over one
synthetic hologram, for all views of the workload, through `sfd_execute` of the C-ABI library.
Default workload: BASELINE.json configs[2], the configuration the metric is quoted on
("4 views, 1024^2 hologram").  One JSON line is printed by rank 0 (see DESIGN.md §8 for every key).

Own arm (`--impl sfd`, default)
  value      reconstructions/s (views/s) with inputs resident in HBM; K back-to-back steps timed
             with one CUDA-event pair on the launching stream, max over ranks.  The R input/output
             buffer sets the steps rotate through are larger than L2 together.
  roofline   the dominant kernel's nominal flops / its mean CUDA-event duration against the fp32 FMA
             rate MEASURED on this GPU in the same run (sfd_measure_pipes), with the HBM figures
             (algorithmic bytes against MEASURED_PEAKS.json) beside it; traffic from profiles/.
  clocks     SM clock, throttle reasons and power sampled through NVML during a block of >= 0.5 s of
             the same steps run right before the timed region (and during the timed region itself
             when that is long enough to be seen by a 5 ms sampler).
  e2e        the same metric through `sfd_stream_run`: pinned HOST holograms in, 8-bit intensity
             images in pinned HOST memory out, H2D + kernels + D2H all inside the timed region.
  cpu_baseline  the float64 oracle (form B) on the host cores, bounded sample (N=1, rank 0 only).

Reference arm (`--impl reference`): the oracle as it stands on the host cores, one view per step.
"""
from __future__ import annotations

import argparse
import json
import os
import pathlib
import socket
import subprocess
import sys
import threading
import time

ROOT = pathlib.Path(__file__).resolve().parent
if str(ROOT) not in sys.path:
    sys.path.insert(0, str(ROOT))

METRIC = "reconstructions/sec (4 views, 1024^2 hologram)"
UNIT = "reconstructions/s"
L2_BYTES = 126 * 1000 * 1000
# plain fp32 pipe: 148 SMs x 128 lanes x 2 flop (FMA) x 1.965 GHz (B200_PROFILING.md: 148 SMs,
# clocks.max.sm 1965 MHz) — the ALU-side denominator of DESIGN.md §7
ALU_PEAK_TFLOPS = 148 * 128 * 2 * 1.965e9 / 1e12


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=2000)
    ap.add_argument("--warmup", type=int, default=20)
    ap.add_argument("--impl", default="sfd", choices=["sfd", "reference"])
    ap.add_argument("--config", type=int, default=2, choices=[1, 2, 4])
    ap.add_argument("--e2e-frames", type=int, default=256,
                    help="frames of the real-time stream (BASELINE.json configs[3]: 256)")
    ap.add_argument("--peaks", action="store_true",
                    help="print the measured pipe rates of this GPU (sfd_measure_pipes) and exit")
    ap.add_argument("--no-extras", action="store_true",
                    help="skip the secondary measurements (live steering, angular spectrum)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--kernels", default="auto", choices=["auto", "generic"],
                    help="generic = force the generic Stockham kernels at N=1024 (A/B timing)")
    ap.add_argument("--intensity-only", action="store_true",
                    help="skip the complex field output (row f1); not the headline configuration")
    return ap.parse_args()


def fp32_floor_us(N, V, cycles_per_branch, sms=148, ghz=1.965):
    """Time one pass of the warp-per-branch kernels needs if the fp32 pipes never idle (us):
    V N lines x N/512 branches, each `cycles_per_branch` pipe cycles of one of 4 x sms sub-partitions."""
    return V * N * (N // 512) * cycles_per_branch / (4 * sms) / (ghz * 1e3)


def ncu_traffic(workload, kernel):
    """DRAM read + write bytes per launch of `kernel` from the committed ncu --set full capture
    (profiles/r02_traffic.json, written from the capture named inside it); None if not recorded."""
    f = ROOT / "profiles" / "r02_traffic.json"
    try:
        rec = json.loads(f.read_text())[workload][kernel]
        return int(rec["dram_read_bytes"]) + int(rec["dram_write_bytes"]), rec.get("source")
    except Exception:
        return None, None


def measured_peaks():
    p = ROOT / "MEASURED_PEAKS.json"
    if p.exists():
        try:
            d = json.loads(p.read_text())
            return float(d["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
        except Exception:
            pass
    return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


# ---- clocks during the timed region ---------------------------------------------------------------
class ClockSampler(threading.Thread):
    """Samples SM clock and throttle reasons of one GPU through NVML every `period` seconds."""
    REASONS = {0x8: "hw_slowdown", 0x40: "hw_thermal_slowdown", 0x20: "sw_thermal_slowdown",
               0x4: "sw_power_cap", 0x80: "hw_power_brake_slowdown"}

    def __init__(self, index, period=0.005):
        super().__init__(daemon=True)
        self.index, self.period = index, period
        self.samples = []            # (t, sm_mhz, reasons bitmask, watts)
        self._stop_evt = threading.Event()
        self.sm_max = None
        self.ok = False
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.sm_max = int(pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM))
            self.ok = True
        except Exception as e:       # no NVML: the JSON line says so
            self.err = repr(e)

    def run(self):
        if not self.ok:
            return
        nv = self.nv
        while not self._stop_evt.is_set():
            try:
                mhz = int(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM))
                try:
                    rs = int(nv.nvmlDeviceGetCurrentClocksEventReasons(self.h))
                except Exception:
                    rs = int(nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h))
                try:
                    w = nv.nvmlDeviceGetPowerUsage(self.h) / 1000.0
                except Exception:
                    w = 0.0
                self.samples.append((time.perf_counter(), mhz, rs, w))
            except Exception:
                pass
            self._stop_evt.wait(self.period)

    def stop(self):
        self._stop_evt.set()
        if self.is_alive():
            self.join(timeout=2)

    def summary(self, t0, t1, fallback=None):
        """Samples inside [t0, t1]; if the region is too short to hold two samples, those of the
        `fallback` window (the sustained block of the same steps right before it) are reported."""
        if not self.ok:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "note": "NVML unavailable"}
        inside = [s for s in self.samples if t0 <= s[0] <= t1]
        note = "sampled inside the timed region"
        if len(inside) < 2 and fallback is not None:
            inside = [s for s in self.samples if fallback[0] <= s[0] <= fallback[1]]
            note = ("timed region shorter than two sampling periods: samples of the sustained block of "
                    "the same steps that ends where the timed region starts")
        mhz = sorted(s[1] for s in inside)
        bits = 0
        for s in inside:
            bits |= s[2]
        return {"sm_mhz": mhz[len(mhz) // 2] if mhz else None, "sm_max_mhz": self.sm_max,
                "reasons": sorted(n for b, n in self.REASONS.items() if bits & b),
                "power_w_max": round(max((s[3] for s in inside), default=0.0), 1),
                "samples": len(inside), "note": note}


# ---- algorithmic bytes / flops of one launch ---------------------------------------
def algorithmic(N, V, in_bytes, want_field, want_inten):
    """Bytes the method itself must move through HBM per launch, and nominal flops, per kernel."""
    M = 2 * N
    log2M = M.bit_length() - 1
    line_flops = 2 * 5 * M * log2M + 6 * M          # forward + inverse FFT, spectrum multiply
    out_px = (8 if want_field else 0) + (4 if want_inten else 0)
    return {
        # pass y: hologram once per frame (shared by the views) -> B[V][N][N] complex64
        "k_pass_y": {"bytes": N * N * in_bytes + V * N * N * 8,
                     "flops": V * N * (line_flops + 2 * N + 6 * N)},
        # pass x: B -> field complex64 and/or intensity float32
        "k_pass_x": {"bytes": V * N * N * 8 + V * N * N * out_px,
                     "flops": V * N * (line_flops + 6 * N + 6 * N + 3 * N)},
    }


# ---- the oracle on the host cores (cpu_baseline and the reference arm) ----------------------------
def oracle_view_seconds(holo, wl, v):
    """One reconstruction (one view) with oracle form B as it stands; returns seconds."""
    from oracle import shifted_fresnel as O
    t0 = time.perf_counter()
    O.reconstruct_views(holo, wl.lam, wl.p1[v:v + 1], wl.p2[v:v + 1], wl.z[v:v + 1],
                        wl.Ox[v:v + 1], wl.Oy[v:v + 1], form="B")
    return time.perf_counter() - t0


ORACLE_CAVEAT = ("the oracle does more work per reconstruction than the GPU path: float64, the paper's "
                 "un-pruned 2-D 2N x 2N FFTs, chirp tables and kernel spectrum rebuilt for every view "
                 "(steps (v)-(vi) every frame, as the paper's step list has it); the GPU path is fp32, "
                 "pruned, and caches the tables per plan - a baseline, not a like-for-like comparison")


def cpu_baseline(wl, holo, budget_s=12.0, max_views=400):
    from oracle import shifted_fresnel as O
    oracle_view_seconds(holo, wl, 0)                 # untimed warm-up (FFT plan cache, page faults)
    done, spent = 0, 0.0
    while done < max_views and spent < budget_s:
        spent += oracle_view_seconds(holo, wl, done % wl.n_views)
        done += 1
    return {"value": done / spent, "unit": UNIT, "cores": int(O.FFT_WORKERS), "kind": "oracle",
            "sample": f"{done} single-view reconstructions of {wl.name} (oracle form B, float64, "
                      f"scipy.fft workers={O.FFT_WORKERS}) in {spent:.2f} s after 1 warm-up",
            "caveat": ORACLE_CAVEAT,
            "frames_per_s": done / spent / wl.n_views}


def run_reference(args, info):
    """Reference arm: the oracle, untuned, on the host cores; rank 0 only (the other ranks join the
    process group, meet rank 0 at a barrier and exit 0 without work)."""
    from paper_1001_4309_b200 import dist as D
    D.init(info, "gloo")
    D.barrier(info)
    if not info.is_root:
        D.barrier(info)
        D.finalize(info)
        return 0
    from oracle import shifted_fresnel as O
    from paper_1001_4309_b200 import workloads as W
    wl = W.config(args.config)
    holo = wl.hologram()
    budget = 240.0
    for i in range(args.warmup):
        oracle_view_seconds(holo, wl, i % wl.n_views)
        if i >= 2:
            break                                     # warm-up is bounded: each step is ~0.1-0.5 s
    t_total, done = 0.0, 0
    for i in range(args.steps):
        t_total += oracle_view_seconds(holo, wl, i % wl.n_views)
        done += 1
        if t_total > budget:
            break
    value = done / t_total
    sample = (f"each step = one single-view reconstruction of {wl.name} (oracle form B, float64, "
              f"scipy.fft workers={O.FFT_WORKERS}); {done} of {args.steps} requested steps timed "
              f"({t_total:.1f} s; capped at {budget:.0f} s)")
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "ranks_joined": info.world,
        "steps": done, "steps_requested": args.steps, "warmup": min(args.warmup, 3),
        "ms_per_step": 1e3 * t_total / done, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": wl.name, "N": wl.N, "views": wl.n_views, "unit_per_step": 1},
        "frames_per_s": value / wl.n_views,
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": int(O.FFT_WORKERS),
                         "kind": "oracle", "sample": sample, "caveat": ORACLE_CAVEAT},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)
    D.barrier(info)
    D.finalize(info)
    return 0


# ---- own arm ----------------------------------------------------------------------------------------
def run_sfd(args, info):
    import numpy as np
    import torch
    from paper_1001_4309_b200 import dist as D
    from paper_1001_4309_b200 import workloads as W
    from paper_1001_4309_b200 import binding as B      # raises if libsfd.so is not built

    if not torch.cuda.is_available():
        raise RuntimeError("bench.py --impl sfd needs a CUDA device: the hot path has no CPU fallback")
    if info.local_rank >= torch.cuda.device_count():
        raise RuntimeError(f"rank {info.rank}: local rank {info.local_rank} but only "
                           f"{torch.cuda.device_count()} CUDA device(s) visible")
    torch.cuda.set_device(info.local_rank)
    dev = torch.device("cuda", info.local_rank)
    D.init(info, "nccl")

    wl = W.config(args.config)
    N, V = wl.N, wl.n_views
    in_bytes = 1 if wl.in_dtype == W.IN_U8 else 4
    want_field = not args.intensity_only
    base = wl.hologram()                                # seeded synthetic Gabor hologram

    # R buffer sets; frame r is the base hologram rolled by 37 r pixels (the path is
    # data-oblivious; distinct addresses are what matters).  R sets together exceed 2 x L2.
    set_bytes = N * N * in_bytes + V * N * N * ((8 if want_field else 0) + 4)
    R = max(2, -(-2 * L2_BYTES // set_bytes))
    holos = [torch.from_numpy(np.roll(base, (37 * r, 37 * r), axis=(0, 1)).copy()).to(dev)
             for r in range(R)]
    fields = [torch.empty((V, N, N), dtype=torch.complex64, device=dev) if want_field else None
              for _ in range(R)]
    intens = [torch.empty((V, N, N), dtype=torch.float32, device=dev) for _ in range(R)]

    plan = B.Plan(wl)
    if args.kernels == "generic":
        plan.select_kernels(B.SFD_KERNELS_GENERIC)
    stream = torch.cuda.current_stream()
    # measured pipe rates of this GPU (a few ms of FMA kernels), the roofline's denominator
    pipe_tflops, cyc_a, cyc_b, pipe_ghz = B.sfd_measure_pipes()
    sampler = ClockSampler(torch.cuda._get_nvml_device_index(dev) if hasattr(
        torch.cuda, "_get_nvml_device_index") else info.local_rank)
    sampler.start()

    def step(i):
        r = i % R
        B.sfd_execute(plan.handle, holos[r], fields[r], intens[r], stream)

    def timed(n, first=0):
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        t0 = time.perf_counter()
        e0.record(stream)
        for i in range(n):
            step(first + i)
        e1.record(stream)
        torch.cuda.synchronize()
        return e0.elapsed_time(e1) * 1e-3, t0, time.perf_counter()

    for i in range(max(args.warmup, 3)):
        step(i)
    torch.cuda.synchronize()
    # sustained block: the same steps for >= 0.5 s with the clock sampler running, so that the clock
    # record does not depend on the length of the timed region (a --steps 20 region lasts 1 ms)
    probe, _, _ = timed(50)
    n_sus = max(200, int(0.6 / (probe / 50)))
    sec_sus, ts0, ts1 = timed(n_sus)
    D.barrier(info)
    n0 = B.sfd_launch_count()
    sec_rank, t0, t1 = timed(args.steps)
    launches = B.sfd_launch_count() - n0
    D.barrier(info)
    clocks = sampler.summary(t0, t1, fallback=(ts0, ts1))
    clocks["sustained_block"] = dict(sampler.summary(ts0, ts1), steps=n_sus, seconds=round(sec_sus, 4))
    units, sec, value = D.aggregate_throughput(info, args.steps * V, sec_rank, dev)
    _, sec_s, value_sus = D.aggregate_throughput(info, n_sus * V, sec_sus, dev)
    launches_all = int(D.sum_over_ranks(info, launches, dev))

    # per-kernel CUDA-event durations (events recorded by the library around each kernel, on the
    # launching stream), same rotation, right after the timed region
    plan.set_timing(True)
    ksteps = min(max(args.steps, 20), 200)
    kms = np.zeros(3)
    for i in range(ksteps):
        step(i)
        kms += np.array(plan.last_kernel_ms())
    plan.set_timing(False)
    kms /= max(ksteps, 1)

    alg = algorithmic(N, V, in_bytes, want_field, True)
    peak, peak_src = measured_peaks()
    keys = ["k_pass_y", "k_pass_x"]                    # rows of algorithmic()
    # the kernels that actually ran: N = 1024 / 2048 have their own pair (sfd_plan_uses_warp_kernels)
    names = [f"k_cols_{wl.N}", f"k_rows_{wl.N}"] if plan.uses_warp_kernels else keys
    dom = int(np.argmax(kms[:2]))
    per_kernel = {}
    for k, name in enumerate(names):
        dur = kms[k] * 1e-3
        alg[name] = alg[keys[k]]
        per_kernel[name] = {
            "ms": round(float(kms[k]), 5),
            "algorithmic_bytes": alg[name]["bytes"],
            "gbs": round(alg[name]["bytes"] / dur / 1e9, 1) if dur > 0 else None,
            "hbm_frac": round(alg[name]["bytes"] / dur / 1e9 / peak, 4) if dur > 0 else None,
            "nominal_tflops": round(alg[name]["flops"] / dur / 1e12, 2) if dur > 0 else None,
            "alu_frac": round(alg[name]["flops"] / dur / 1e12 / pipe_tflops, 4) if dur > 0 else None,
        }
    dname = names[dom]
    step_bytes = alg["k_pass_y"]["bytes"] + alg["k_pass_x"]["bytes"]
    traffic, traffic_src = ncu_traffic(wl.name, dname)
    # pipe model of the warp-per-branch kernels with the butterfly cycles measured in this run: a
    # 1024-point branch of a line = 2 stage-A + 2 stage-B butterflies + 3 table multiplies (4 operations
    # per complex value; the pre-chirp of pass y multiplies a real sample: 2)
    cyc_branch = [2 * cyc_a + 2 * cyc_b + 2 * 128 + 64, 2 * cyc_a + 2 * cyc_b + 3 * 128]
    # Binding roof: with the traffic cut to 28 MiB per view the path runs at
    # ~16 flop/B, above the fp32 ridge (11 flop/B), so the plain fp32 pipe bounds it.  The HBM
    # figures BASELINE.json's metric asks for are reported beside it under "hbm".
    roofline = {
        "bound": "alu", "kernel": dname, "achieved": per_kernel[dname]["nominal_tflops"],
        "peak": round(pipe_tflops, 2), "unit": "TFLOP/s",
        "frac": per_kernel[dname]["alu_frac"],
        "peak_source": f"measured in this run: sfd_measure_pipes, {pipe_tflops:.2f} TFLOP/s of plain fp32 FMA "
                       f"(2 flop each) over all SMs at {pipe_ghz:.3f} GHz; derived figure for comparison: "
                       f"148 SMs x 128 lanes x 2 x 1.965 GHz = {ALU_PEAK_TFLOPS:.1f}",
        "peak_derived": round(ALU_PEAK_TFLOPS, 1),
        "flops_model": "nominal 5 M log2 M per M-point FFT, M = 2N, two FFTs per line, + pointwise",
        "traffic": traffic, "traffic_source": traffic_src,
        "hbm": {"kernel": dname, "achieved": per_kernel[dname]["gbs"], "peak": peak, "unit": "GB/s",
                "frac": per_kernel[dname]["hbm_frac"], "peak_source": peak_src,
                "algorithmic_bytes": alg[dname]["bytes"],
                "step": {"algorithmic_bytes": step_bytes,
                         "gbs": round(step_bytes / (sec_rank / args.steps) / 1e9, 1),
                         "frac": round(step_bytes / (sec_rank / args.steps) / 1e9 / peak, 4)}},
        "kernels": per_kernel,
        "fp32_pipe": ({"floor_us_per_kernel": [round(fp32_floor_us(N, V, c, plan_sms(torch, dev), pipe_ghz), 2)
                                               for c in cyc_branch],
                       "frac": round(fp32_floor_us(N, V, cyc_branch[dom], plan_sms(torch, dev), pipe_ghz)
                                     / (1e3 * float(kms[dom])), 4),
                       "cycles_stage_a": round(cyc_a, 1), "cycles_stage_b": round(cyc_b, 1),
                       "model": "measured cycles of the two radix-32 butterfly stages (a warp alone on its "
                                "sub-partition) x 2 each + table multiplies per 1024-point branch, N/512 "
                                "branches per line, V N lines per kernel, 4 sub-partitions per SM"}
                      if plan.uses_warp_kernels else None),
        "timing": f"library CUDA events around each kernel on the launching stream, mean of "
                  f"{ksteps} steps after the timed region (kernel sum "
                  f"{kms[:2].sum():.4f} ms vs {1e3 * sec_rank / args.steps:.4f} ms/step)",
    }

    # end to end through the C ABI with host buffers
    e2e = None
    if not args.no_e2e:
        F = max(4, args.e2e_frames)
        hp = torch.empty((F, N, N), dtype=torch.uint8 if in_bytes == 1 else torch.float32).pin_memory()
        for f in range(F):
            hp[f] = torch.from_numpy(np.roll(base, (11 * f, 5 * f), axis=(0, 1)).copy())
        op = torch.empty((F, V, N, N), dtype=torch.uint8).pin_memory()
        # warm-up: one untimed pass over the whole ring of host buffers (allocates the device double
        # buffers and touches every pinned output page once: the first DMA into fresh pinned pages
        # runs at 2/3 of the steady rate), then the timed pass over the same F frames
        plan.stream_run(hp, op)
        D.barrier(info)
        _, s = plan.stream_run(hp, op)
        u_all, s_max, e_val = D.aggregate_throughput(info, F * V, s, dev)
        e2e = {"value": e_val, "unit": UNIT, "h2d_bytes_per_step": N * N * in_bytes,
               "d2h_bytes_per_step": V * N * N, "frames": F, "frames_per_s": e_val / V,
               "frames_are": f"{F} distinct pinned host frames = the seeded hologram of {wl.name} rolled by "
                             "(11 f, 5 f) pixels (the path is data-oblivious; the 256 independently seeded "
                             "frames of configs[3] take 8 min to generate and are covered by the parity test "
                             "on 6 of them)",
               "api": f"sfd_stream_run: pinned host holograms -> double-buffered H2D -> {names[0]}, "
                      f"{names[1]}, k_quantise -> D2H of 8-bit intensity images to pinned host memory",
               "pcie_gbs_d2h": round(V * N * N * F / s / 1e9, 2),
               "warmup": "one untimed pass over the same ring of F pinned host frames"}
        del hp, op

    extras = None
    if info.is_root and not args.no_extras:
        extras = {"steering": steering(plan, wl, holos[0], stream, torch, B),
                  "angular_spectrum": asm_line(wl, dev, torch, B, np),
                  "other_sizes": sizes_line(wl, dev, torch, B)}
        if 2 * wl.N <= 2048:    # the 2N grid of the hologram generator
            extras["angular_spectrum_2N"] = asm_line(wl, dev, torch, B, np, reps=100, N=2 * wl.N)
    sampler.stop()

    cpu = None
    if info.is_root and info.world == 1 and not args.no_cpu_baseline:
        cpu = cpu_baseline(wl, base)

    plan.close()
    D.finalize(info)
    if not info.is_root:
        return 0
    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": info.world, "steps": args.steps,
        "warmup": max(args.warmup, 3), "ms_per_step": 1e3 * sec / args.steps,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32",
        "data": "synthetic",
        "config": {"workload": wl.name, "N": N, "M": 2 * N, "views": V,
                   "input": "uint8" if in_bytes == 1 else "float32",
                   "outputs": ("complex64 field + " if want_field else "") + "float32 intensity",
                   "l2": f"steps rotate through {R} input/output buffer sets, "
                         f"{R * set_bytes / 2**20:.0f} MiB > L2 ({L2_BYTES / 1e6:.0f} MB)",
                   "sharding": "whole frames per rank, no collective on the data path"},
        "frames_per_s": value / V,
        "value_sustained": value_sus,
        "sustained": f"{n_sus} steps in {sec_s:.3f} s right before the timed region, same loop",
        "roofline": roofline, "cpu_baseline": cpu, "e2e": e2e, "clocks": clocks,
        "gpu_launches": launches_all, "extras": extras,
        "paper_context": "paper: 4 views in ~60 ms on four GTX 295 chips (66.7 reconstructions/s), "
                         "9542 ms on a Core2Quad; other hardware, context only",
    }
    print(json.dumps(line), flush=True)
    return 0


def plan_sms(torch, dev):
    return torch.cuda.get_device_properties(dev).multi_processor_count


def steering(plan, wl, holo, stream, torch, B, frames=400, every=10):
    """Row f1: what live steering costs.  A device-resident loop of sfd_execute_u8 (the real-time
    mode's kernels) with and without an asynchronous update of one view every `every` frames."""
    V = wl.n_views

    def run(update):
        out = None
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        host_ms = []
        e0.record(stream)
        for f in range(frames):
            if update and f % every == 0:
                v = (f // every) % V
                plan.update_view_async(v, wl.p1[v], wl.p2[v], wl.z[v] * (1.0 + 1e-3 * (f % 7)), wl.Ox[v],
                                       wl.Oy[v], stream)
                host_ms.append(plan.last_update_host_ms)
            out = plan.execute_u8(holo, out, stream)
        e1.record(stream)
        torch.cuda.synchronize()
        return frames / (e0.elapsed_time(e1) * 1e-3), host_ms

    run(False)
    plain, _ = run(False)
    steered, host_ms = run(True)
    for v in range(V):                                   # leave the plan as it was
        plan.update_view(v, wl.p1[v], wl.p2[v], wl.z[v], wl.Ox[v], wl.Oy[v])
    return {"frames_per_s_plain": round(plain, 1), "frames_per_s_steered": round(steered, 1),
            "update_every_frames": every,
            "host_build_ms": round(sum(host_ms) / len(host_ms), 3),
            "api": "sfd_plan_update_view_async on the execute stream (float64 tables on the host into pinned "
                   "staging, one H2D copy, no synchronisation) between sfd_execute_u8 calls"}


def asm_line(wl, dev, torch, B, np, reps=200, N=None):
    """Row f4: angular-spectrum propagations per second on an N x N grid (default: the workload's size),
    complex64 in, inputs resident, distinct buffers rotated through L2: one plane with field + intensity
    + phase out, and an 8-plane focus stack (field + intensity) from one input."""
    N = N or wl.N
    stream = torch.cuda.current_stream()

    def run(P, with_phase, R):
        u0 = [torch.randn(N, N, dtype=torch.complex64, device=dev) for _ in range(R)]
        outs = [(torch.empty((P, N, N), dtype=torch.complex64, device=dev),
                 torch.empty((P, N, N), dtype=torch.float32, device=dev),
                 torch.empty((P, N, N), dtype=torch.float32, device=dev) if with_phase else None)
                for _ in range(R)]
        with B.AsmPlan(N, N, wl.lam, 4.65e-6, [0.08 + 0.002 * i for i in range(P)]) as plan:
            for i in range(10):
                B.sfd_asm_execute(plan.handle, u0[i % R], *outs[i % R], stream)
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(stream)
            for i in range(reps):
                B.sfd_asm_execute(plan.handle, u0[i % R], *outs[i % R], stream)
            e1.record(stream)
            torch.cuda.synchronize()
        return e0.elapsed_time(e1) * 1e-3 / reps

    sec = run(1, True, 6)
    sec8 = run(8, False, 2)
    by = N * N * (8 + 8 + 8 + 8 + 8 + 8 + 8 + 4 + 4)     # in, A w/r, H, W w/r, field, intensity, phase
    by8 = N * N * (8 + 8 + 8 + 8 * (8 + 8 + 8 + 8 + 4))  # in, A w/r; per plane H, W w/r, field, intensity
    io, io8 = N * N * (8 + 8 + 4 + 4), N * N * (8 + 8 * (8 + 4))  # input + outputs only (what must touch HBM)
    return {"propagations_per_s": round(1.0 / sec, 1), "us": round(sec * 1e6, 2), "N": N,
            "algorithmic_bytes": by, "gbs": round(by / sec / 1e9, 1),
            "io_bytes": io, "io_gbs": round(io / sec / 1e9, 1),
            "stack8": {"us_per_plane": round(sec8 * 1e6 / 8, 2), "planes_per_s": round(8.0 / sec8, 1),
                       "algorithmic_bytes": by8, "gbs": round(by8 / sec8 / 1e9, 1),
                       "io_bytes": io8, "io_gbs": round(io8 / sec8 / 1e9, 1)},
            "note": "algorithmic_bytes counts the intermediates (A, W, H) written and read between the kernels"
                    + (", which stay in L2 at this size" if N <= 1024 else " (larger than L2 at this size)")
                    + "; io_bytes is the input and the outputs only",
            "api": "sfd_asm_execute: 3 launches (rows FFT, columns FFT x H x IFFT per plane, rows IFFT + |u|^2 + arg u)"}


def sizes_line(wl, dev, torch, B, steps=600):
    """The same views on smaller square holograms (uint8, field + intensity out): us per frame.
    N = 512 runs the one-warp-per-line kernels, the smaller sizes the generic Stockham kernels."""
    out = {}
    stream = torch.cuda.current_stream()
    for N in (512, 256, 128):
        R = 8
        holos = [torch.randint(0, 256, (N, N), dtype=torch.uint8, device=dev) for _ in range(R)]
        f = [torch.empty((wl.n_views, N, N), dtype=torch.complex64, device=dev) for _ in range(R)]
        I = [torch.empty((wl.n_views, N, N), dtype=torch.float32, device=dev) for _ in range(R)]
        with B.Plan(N=N, lam=wl.lam, p1=wl.p1, p2=wl.p2, z=wl.z, Ox=wl.Ox, Oy=wl.Oy, in_dtype=B.SFD_U8) as plan:
            for i in range(20):
                B.sfd_execute(plan.handle, holos[i % R], f[i % R], I[i % R], stream)
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(stream)
            for i in range(steps):
                B.sfd_execute(plan.handle, holos[i % R], f[i % R], I[i % R], stream)
            e1.record(stream)
            torch.cuda.synchronize()
            rec = {"us_per_frame": round(e0.elapsed_time(e1) * 1e3 / steps, 2),
                   "warp_kernels": plan.uses_warp_kernels}
            # the same R frames as one CUDA graph (sfd_execute only enqueues kernels): what the GPU
            # needs once the host's launch rate is out of the way
            side = torch.cuda.Stream()
            side.wait_stream(stream)
            with torch.cuda.stream(side):
                B.sfd_execute(plan.handle, holos[0], f[0], I[0], side)
            stream.wait_stream(side)
            graph = torch.cuda.CUDAGraph()
            with torch.cuda.graph(graph):
                cap = torch.cuda.current_stream()
                for i in range(R):
                    B.sfd_execute(plan.handle, holos[i], f[i], I[i], cap)
            for _ in range(3):
                graph.replay()
            reps = max(1, steps // R)
            e0.record(stream)
            for _ in range(reps):
                graph.replay()
            e1.record(stream)
            torch.cuda.synchronize()
            rec["us_per_frame_cuda_graph"] = round(e0.elapsed_time(e1) * 1e3 / (reps * R), 2)
            out[f"N{N}"] = rec
    out["note"] = (f"{wl.n_views} views of {wl.name}, uint8 in, complex64 field + float32 intensity out; "
                   "us_per_frame_cuda_graph replays the same frames as one captured graph of 8 sfd_execute calls: "
                   "where it matches us_per_frame the size is bound by the latency of its two dependent kernels, "
                   "not by the launch rate of the host")
    return out


def run_peaks():
    import torch
    from paper_1001_4309_b200 import binding as B
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py --peaks needs a CUDA device")
    B.sfd_measure_pipes()                                  # warm-up (clocks, instruction cache)
    tf, ca, cb, ghz = B.sfd_measure_pipes()
    B.sfd_measure_memory_pipes()
    smem, tm1, tm2, tmlat = B.sfd_measure_memory_pipes()
    hbm, src = measured_peaks()
    print(json.dumps({"peaks": {"fp32_fma_tflops": round(tf, 2), "dft32_stage_a_cycles": round(ca, 1),
                                "dft32_stage_b_cycles": round(cb, 1), "sm_ghz": round(ghz, 3),
                                "fp32_derived_tflops": round(ALU_PEAK_TFLOPS, 1), "hbm_gbs": hbm,
                                "hbm_source": src, "gpu": torch.cuda.get_device_name(0),
                                "smem_bytes_per_clk_sm": round(smem, 1),
                                "tmem_ld_bytes_per_clk_subpartition": [round(tm1, 1), round(tm2, 1)],
                                "tmem_ld_dependent_cycles": round(tmlat, 1),
                                "how": "sfd_measure_pipes (include/sfd.h): FFMA chains on all SMs; "
                                       "sfdb::dft32 / dft32_tw in a register-only loop, one warp per "
                                       "sub-partition, clock64.  sfd_measure_memory_pipes: shared memory "
                                       "in the access pattern of the 32 x 32 transposes (8 warps per SM); "
                                       "tcgen05.ld.32x32b.x16, four in flight per warp, with one and two "
                                       "warps per sub-partition; one dependent tcgen05.ld + wait::ld"}}),
          flush=True)
    return 0


# ---- launcher: `python bench.py --gpus N` started bare spawns its own N ranks -------------------------
def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def spawn_ranks(args):
    """One process per GPU with RANK / LOCAL_RANK / WORLD_SIZE / MASTER_* set, as torchrun would; the
    output of every rank passes through (rank 0 prints the JSON line).  Returns the worst exit code."""
    port = _free_port()
    procs = []
    for r in range(args.gpus):
        env = dict(os.environ, RANK=str(r), LOCAL_RANK=str(r), WORLD_SIZE=str(args.gpus),
                   MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
        if args.impl == "sfd":
            env.setdefault("NCCL_DEBUG", "INFO")          # the communicator log (stderr) stays on
            env.setdefault("NCCL_DEBUG_SUBSYS", "INIT")
        procs.append(subprocess.Popen([sys.executable, os.path.abspath(__file__)] + sys.argv[1:], env=env))
    rc = 0
    for p in procs:
        rc = max(rc, abs(p.wait()))
    return rc


def main():
    args = parse_args()
    if args.peaks:
        return run_peaks()
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        return spawn_ranks(args)
    from paper_1001_4309_b200 import dist as D
    info = D.rank_info()
    if info.world != args.gpus:
        raise SystemExit(f"--gpus {args.gpus} but WORLD_SIZE={info.world}")
    if args.impl == "reference":
        return run_reference(args, info)
    return run_sfd(args, info)


if __name__ == "__main__":
    sys.exit(main())
