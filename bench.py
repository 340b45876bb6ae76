#!/usr/bin/env python
"""bench.py — throughput of the Shifted-Fresnel hot path on B200 (BASELINE.json `metric`).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl sfd|reference] [--config 1|2|4]

A *step* is one pass of the whole hot path (convert, pre-chirp,
zero-pad, forward FFT, kernel-spectrum multiply, inverse FFT, crop, post-chirp, |u|^2) over one
synthetic hologram, for all views of the workload, through `sfd_execute` of the C-ABI library.
Default workload: BASELINE.json configs[2], the configuration the metric is quoted on
("4 views, 1024^2 hologram").  One JSON line is printed by rank 0 (see DESIGN.md §8 for every key).

Own arm (`--impl sfd`, default)
  value      reconstructions/s (views/s) with inputs resident in HBM; K back-to-back steps timed
             with one CUDA-event pair on the launching stream, max over ranks.  The R input/output
             buffer sets the steps rotate through are larger than L2 together.
  roofline   the dominant kernel's algorithmic bytes / its mean CUDA-event duration, against the
             measured HBM copy bandwidth of MEASURED_PEAKS.json, plus an ALU-side figure.
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
    ap.add_argument("--e2e-frames", type=int, default=128)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--kernels", default="auto", choices=["auto", "generic"],
                    help="generic = force the generic Stockham kernels at N=1024 (A/B timing)")
    ap.add_argument("--intensity-only", action="store_true",
                    help="skip the complex field output (row f1); not the headline configuration")
    return ap.parse_args()


def fp32_floor_us(N, V, sms=148, ghz=1.965):
    """Time one pass of the warp-per-branch kernels needs if the fp32 pipes never idle (us)."""
    return V * N * (N // 512) * 2730.0 / (4 * sms) / (ghz * 1e3)


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

    def __init__(self, index, period=0.01):
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

    def summary(self, t0, t1):
        if not self.ok:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "note": "NVML unavailable"}
        inside = [s for s in self.samples if t0 <= s[0] <= t1]
        note = "sampled inside the timed region"
        if not inside:               # region shorter than one sampling period
            inside = [s for s in self.samples if t0 - 0.5 <= s[0] <= t1 + 0.5] or self.samples
            note = "timed region shorter than the sampling period; nearest samples under load"
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
            "frames_per_s": done / spent / wl.n_views}


def run_reference(args, info):
    """Reference arm: the oracle, untuned, on the host cores; rank 0 only."""
    if not info.is_root:
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
        "steps": done, "steps_requested": args.steps, "warmup": min(args.warmup, 3),
        "ms_per_step": 1e3 * t_total / done, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": wl.name, "N": wl.N, "views": wl.n_views, "unit_per_step": 1},
        "frames_per_s": value / wl.n_views,
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": int(O.FFT_WORKERS),
                         "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)
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
    sampler = ClockSampler(torch.cuda._get_nvml_device_index(dev) if hasattr(
        torch.cuda, "_get_nvml_device_index") else info.local_rank)
    sampler.start()

    def step(i):
        r = i % R
        B.sfd_execute(plan.handle, holos[r], fields[r], intens[r], stream)

    for i in range(max(args.warmup, 3)):
        step(i)
    torch.cuda.synchronize()
    D.barrier(info)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    n0 = B.sfd_launch_count()
    t0 = time.perf_counter()
    e0.record(stream)
    for i in range(args.steps):
        step(i)
    e1.record(stream)
    torch.cuda.synchronize()
    t1 = time.perf_counter()
    launches = B.sfd_launch_count() - n0
    D.barrier(info)
    sec_rank = e0.elapsed_time(e1) * 1e-3
    clocks = sampler.summary(t0, t1)
    units, sec, value = D.aggregate_throughput(info, args.steps * V, sec_rank, dev)
    launches_all = int(D.sum_over_ranks(info, launches, dev))

    # per-kernel CUDA-event durations (events recorded by the library around each kernel, on the
    # launching stream), same rotation, right after the timed region
    plan.set_timing(True)
    ksteps = min(args.steps, 200)
    kms = np.zeros(3)
    for i in range(ksteps):
        step(i)
        kms += np.array(plan.last_kernel_ms())
    plan.set_timing(False)
    kms /= max(ksteps, 1)

    alg = algorithmic(N, V, in_bytes, want_field, True)
    peak, peak_src = measured_peaks()
    keys = ["k_pass_y", "k_pass_x"]                    # rows of algorithmic()
    # the kernels that actually ran: N = 1024 has its own pair (sfd_plan_uses_warp_kernels)
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
            "alu_frac": round(alg[name]["flops"] / dur / 1e12 / ALU_PEAK_TFLOPS, 4) if dur > 0 else None,
        }
    dname = names[dom]
    step_bytes = alg["k_pass_y"]["bytes"] + alg["k_pass_x"]["bytes"]
    # Binding roof: with the traffic cut to 28 MiB per view the path runs at
    # ~16 flop/B, above the fp32 ridge (11.4 flop/B), so the plain fp32 pipe bounds it.  The HBM
    # figures BASELINE.json's metric asks for are reported beside it under "hbm".
    roofline = {
        "bound": "alu", "kernel": dname, "achieved": per_kernel[dname]["nominal_tflops"],
        "peak": round(ALU_PEAK_TFLOPS, 1), "unit": "TFLOP/s",
        "frac": per_kernel[dname]["alu_frac"],
        "peak_source": "derived: 148 SMs x 128 fp32 lanes x 2 flop x 1.965 GHz (DESIGN.md section 7)",
        "flops_model": "nominal 5 M log2 M per M-point FFT, M = 2N, two FFTs per line, + pointwise",
        "traffic": NCU_TRAFFIC.get((wl.name, dname)),
        "traffic_source": "profiles/ (ncu --set full, dram__bytes_read.sum + dram__bytes_write.sum, "
                          "per launch, caches flushed by ncu before the launch)"
        if NCU_TRAFFIC.get((wl.name, dname)) else None,
        "hbm": {"kernel": dname, "achieved": per_kernel[dname]["gbs"], "peak": peak, "unit": "GB/s",
                "frac": per_kernel[dname]["hbm_frac"], "peak_source": peak_src,
                "algorithmic_bytes": alg[dname]["bytes"],
                "step": {"algorithmic_bytes": step_bytes,
                         "gbs": round(step_bytes / (sec_rank / args.steps) / 1e9, 1),
                         "frac": round(step_bytes / (sec_rank / args.steps) / 1e9 / peak, 4)}},
        "kernels": per_kernel,
        # measured pipe model of the warp-per-branch kernels: a 1024-point
        # branch of a line costs 2730 fp32-pipe cycles of one of the 4 x 148 sub-partitions
        "fp32_pipe": ({"floor_us_per_kernel": round(fp32_floor_us(N, V), 2),
                       "frac": round(fp32_floor_us(N, V) / (1e3 * float(kms[dom])), 4),
                       "model": "2730 pipe cycles per 1024-point branch and line (4 radix-32 butterflies of "
                                "464 cycles, 2 twiddle and 3 table multiplies), N/512 branches per line, "
                                "V N lines per kernel, 592 sub-partitions at 1.965 GHz"}
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
               "api": f"sfd_stream_run: pinned host holograms -> double-buffered H2D -> {names[0]}, "
                      f"{names[1]}, k_quantise -> D2H of 8-bit intensity images to pinned host memory",
               "pcie_gbs_d2h": round(V * N * N * F / s / 1e9, 2),
               "warmup": "one untimed pass over the same ring of F pinned host frames"}
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
        "roofline": roofline, "cpu_baseline": cpu, "e2e": e2e, "clocks": clocks,
        "gpu_launches": launches_all,
        "paper_context": "paper: 4 views in ~60 ms on four GTX 295 chips (66.7 reconstructions/s), "
                         "9542 ms on a Core2Quad; other hardware, context only",
    }
    print(json.dumps(line), flush=True)
    return 0


# ncu `--set full` DRAM traffic per launch (bytes), copied from profiles/ by hand after each capture;
# key = (workload name, kernel).  Absent = null in the JSON line.
NCU_TRAFFIC = {
    # profiles/r01_final_launches.md (final round-1 kernels, config 2)
    ("paper_4view_1024", "k_cols_1024"): 16894720 + 15644928,
    ("paper_4view_1024", "k_rows_1024"): 33795584 + 3111168,
    # profiles/r01_v9_config4.md (N = 2048 warp kernels, config 4)
    ("scale_stress_2048", "k_cols_2048"): 10770688 + 533581050,
    ("scale_stress_2048", "k_rows_2048"): 539547390 + 753424640,
}


def main():
    args = parse_args()
    from paper_1001_4309_b200 import dist as D
    info = D.rank_info()
    if info.world != args.gpus and info.world > 1:
        raise SystemExit(f"--gpus {args.gpus} but WORLD_SIZE={info.world}")
    if args.impl == "reference":
        return run_reference(args, info)
    return run_sfd(args, info)


if __name__ == "__main__":
    sys.exit(main())
