#!/usr/bin/env python
"""bench.py -- throughput of the fast-mode hot path (BASELINE.json:metric) on synthetic SRAL-shaped input.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload NAME] [--impl ours|reference]

One "step" = one pass of the whole hot path over one batch: U surface updates accumulated (steps A1-A7)
and U*P pulses synthesised (steps S1-S3).  Prints ONE JSON line (rank 0).  See DESIGN.md "Measurement".
"""
from __future__ import annotations

import argparse
import csv
import json
import os
import statistics
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import torch  # noqa: E402

from paper_2408_11472_b200 import dist as D  # noqa: E402
from paper_2408_11472_b200 import workloads as W  # noqa: E402

DEFAULT_WORKLOAD = "sar_footprint_268m"   # configs[2]: the config north_star quotes the roofline target on
BYTES_PER_SCATTERER = 28                  # 7 fp32 SoA arrays
FALLBACK_HBM_GBS = 6650.0                 # B200_PROFILING.md fallback when MEASURED_PEAKS.json is absent


# ----------------------------------------------------------------------------------------------------
def measured_peak():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(p) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:
        return FALLBACK_HBM_GBS, "fallback (B200_PROFILING.md 6.65 TB/s)"


def committed_traffic(workload):
    """dram bytes per accumulation launch from the committed ncu --set full capture, or None."""
    p = os.path.join(ROOT, "profiles", "acc_kernel_traffic.csv")
    try:
        with open(p) as f:
            for row in csv.DictReader(f):
                if row["workload"] == workload:
                    return float(row["dram_bytes_read"]) + float(row["dram_bytes_write"])
    except Exception:
        pass
    return None


class NvmlSampler:
    """SM clock and throttle reasons of the device, read in-process through NVML every 5 ms DURING the timed region
    (a timed region of 10 ms is over before `nvidia-smi -lms 100` prints its first line)."""
    REASONS = ((0x8, "hw_slowdown"), (0x40, "hw_thermal_slowdown"), (0x20, "sw_thermal_slowdown"), (0x4, "sw_power_cap"))

    def __init__(self, dev):
        import pynvml
        self.nv = pynvml
        pynvml.nvmlInit()
        try:
            uuid = "GPU-" + str(torch.cuda.get_device_properties(dev).uuid)
            self.h = pynvml.nvmlDeviceGetHandleByUUID(uuid.encode() if hasattr(uuid, "encode") else uuid)
        except Exception:
            self.h = pynvml.nvmlDeviceGetHandleByIndex(dev.index or 0)
        self.mx = float(pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM))
        self.sm, self.mask, self.stop = [], 0, threading.Event()

    def _reasons(self):
        f = getattr(self.nv, "nvmlDeviceGetCurrentClocksEventReasons", None) or self.nv.nvmlDeviceGetCurrentClocksThrottleReasons
        return int(f(self.h))

    def _loop(self):
        while not self.stop.is_set():
            try:
                self.sm.append(float(self.nv.nvmlDeviceGetClockInfo(self.h, self.nv.NVML_CLOCK_SM)))
                self.mask |= self._reasons()
            except Exception:
                pass
            self.stop.wait(0.005)

    def __enter__(self):
        self.t = threading.Thread(target=self._loop, daemon=True)
        self.t.start()
        return self

    def __exit__(self, *a):
        self.stop.set()
        self.t.join(timeout=1)

    def summary(self):
        if not self.sm:
            return {"sm_mhz": None, "sm_max_mhz": self.mx, "reasons": [], "samples": 0, "source": "nvml"}
        return {"sm_mhz": statistics.median(self.sm), "sm_min_mhz": min(self.sm), "sm_max_mhz": self.mx,
                "reasons": sorted(n for b, n in self.REASONS if self.mask & b), "samples": len(self.sm),
                "source": "nvml, 5 ms period, in-process"}


def clock_sampler(dev):
    try:
        return NvmlSampler(dev)
    except Exception:
        return ClockSampler(dev.index or 0)


class ClockSampler:
    """Fallback when NVML cannot be loaded: nvidia-smi clocks and throttle reasons DURING the timed region
    (B200_PROFILING.md recipe)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.rows, self.proc, self.index = [], None, index

    def __enter__(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
        except Exception:
            self.proc = None
        return self

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([c.strip() for c in line.split(",")])

    def __exit__(self, *a):
        if self.proc:
            time.sleep(0.15)
            self.proc.terminate()
            try:
                self.proc.wait(timeout=2)
            except Exception:
                self.proc.kill()

    def summary(self):
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            try:
                sm.append(float(r[0]))
                mx.append(float(r[1]))
                for n, v in zip(names, r[3:7]):
                    if v.lower().startswith("active"):
                        reasons.add(n)
            except Exception:
                continue
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        return {"sm_mhz": statistics.median(sm), "sm_max_mhz": max(mx), "reasons": sorted(reasons),
                "samples": len(sm), "source": "nvidia-smi -lms 100"}


# ----------------------------------------------------------------------------------------------------
def strided_rows(wl, n_target):
    """Row indices of a sample of about n_target scatterers drawn as whole rows spread evenly over the scene, so that
    dark and illuminated parts appear in scene proportion."""
    rows = max(1, min(wl.n_along, n_target // wl.n_cross))
    step = wl.n_along / rows
    return [min(wl.n_along - 1, int((i + 0.5) * step)) for i in range(rows)]


def cpu_oracle_sample(wl, sample, nthreads, target_s=12.0):
    """Times the oracle, as it stands, on a bounded sample of the workload: passes of one update over `sample`
    (strided rows of the scene; satellite states of successive updates) until about target_s seconds of wall time are
    spent, and one segment (2 spectra -> P pulses x G gates) of synthesis.
    Returns (scatterers/s extrapolated to a whole step, description, threads used, seconds spent, in-window fraction
    of the sample)."""
    import numpy as np
    from oracle import oracle as orc
    cfg = orc.make_config(wl.n_gates, wl.n_doppler, wl.pulses_per_update, wl.wavelength_m, wl.prf_hz,
                          wl.gate_spacing_m, wl.antenna_alpha)

    def sat(u):
        st = W.sat_state(wl, u % wl.n_updates)
        return orc.make_sat(st["pos"], st["vel"], st["boresight"], st["range_gate0_m"])

    arrs = [sample[f].numpy() for f in W.FIELDS]
    ns = arrs[0].size
    g0, _ = orc.indices(cfg, sat(0), *arrs[:6])
    in_window = float((g0 != orc.GATE_NONE).mean())
    orc.spectrum(cfg, sat(0), *arrs, nthreads=nthreads)        # page in, spin up the threads (untimed)
    t_acc, passes, used, T = 0.0, 0, nthreads, None
    while t_acc < target_s and passes < 4096:
        t0 = time.perf_counter()
        T, used = orc.spectrum(cfg, sat(passes), *arrs, nthreads=nthreads)
        t_acc += time.perf_counter() - t0
        passes += 1
    T2 = np.stack([T, T])
    t0 = time.perf_counter()
    orc.synthesize(cfg, T2, 0, wl.pulses_per_update, final=False)
    t_syn = time.perf_counter() - t0
    tau = t_acc / (ns * passes)
    S = wl.n_scatterers
    value = S / (S * tau + t_syn)
    desc = (f"accumulate: {passes} passes of 1 update over {ns} of {S} scatterers (whole rows spread evenly over the "
            f"scene, {100 * in_window:.1f} % of them in the gate window) in {t_acc:.2f} s; synthesize: 1 segment "
            f"({wl.pulses_per_update} pulses x {wl.n_gates} gates, naive O(N^2) iDFT) in {t_syn:.2f} s; extrapolated "
            f"to a whole step (U updates x S scatterers + U segments)")
    return value, desc, used, t_acc + t_syn, in_window


def reduced_scene(wl, n_target):
    """A scene of the same recipe with only the rows of strided_rows(): the rows are generated as a block and then
    placed at their along-track positions (for the PM sea the field loses its along-track correlation: irrelevant for
    the oracle's cost)."""
    rows = strided_rows(wl, n_target)
    wl_s = wl.scaled(n_along=len(rows))
    scat = W.scatterers(wl_s)
    x_rows = torch.tensor([(r - (wl.n_along - 1) / 2.0) * wl.spacing_m for r in rows], dtype=torch.float32)
    scat["x"] = x_rows[:, None].expand(len(rows), wl.n_cross).reshape(-1).contiguous()
    return scat


def run_reference(args, wl):
    """--impl reference: the oracle (oracle/), as it stands, on the host cores; each step a bounded sample."""
    from oracle import oracle as orc
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    orc.build()
    nthreads = orc.max_threads()
    scat = reduced_scene(wl, 1 << 22)
    vals, descs, step_s = [], [], []
    t_all0 = time.perf_counter()
    for i in range(args.warmup + args.steps):
        v, desc, used, spent, inw = cpu_oracle_sample(wl, scat, nthreads, target_s=2.0)   # extrapolates with the full S
        if i >= args.warmup:
            vals.append(v)
            descs.append(desc)
            step_s.append(spent)
    t_all = time.perf_counter() - t_all0
    value = statistics.mean(vals)
    out = {
        "impl": "reference", "metric": "scatterers accumulated + IQ synthesised per second (whole step)",
        "value": value, "unit": "scatterers/s", "n_gpus": args.gpus, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": 1e3 * statistics.mean(step_s), "ms_per_full_step_extrapolated": 1e3 * wl.n_updates * wl.n_scatterers / value,
        "higher_is_better": True, "scaling": "strong",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": wl.name, "scatterers": wl.n_scatterers, "gates": wl.n_gates, "doppler_bins": wl.n_doppler,
                   "pulses_per_update": wl.pulses_per_update, "updates": wl.n_updates,
                   "note": "oracle on host cores; each step is a bounded sample of this workload "
                   f"(same recipe, {scat['x'].numel()} scatterers as whole rows spread evenly over the scene); "
                   "ms_per_step is the measured time of a sampled step, value the rate extrapolated to whole steps"},
        "cpu_baseline": {"value": value, "unit": "scatterers/s", "cores": nthreads, "kind": "oracle",
                         "sample": descs[-1]},
        "e2e": {"value": value, "unit": "scatterers/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0, "wall_s": t_all,
    }
    print(json.dumps(out), flush=True)


# ----------------------------------------------------------------------------------------------------
def in_window_fraction(sim, S, scat, sat):
    """Fraction of the scatterers that land in the gate window (the production kernel's own index export)."""
    g0, _ = sim.debug_indices(scat, sat)
    n = g0.numel()
    return float((g0 != S.GATE_NONE).sum().item()) / n if n else 0.0


def empty_launch_us(dev, reps=200):
    """Latency floor of a launch: back-to-back one-element fills on the stream, per launch (CUDA events)."""
    t = torch.zeros(1, device=dev)
    for _ in range(20):
        t.zero_()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    torch.cuda.synchronize(dev)
    e0.record()
    for _ in range(reps):
        t.zero_()
    e1.record()
    torch.cuda.synchronize(dev)
    return 1e3 * e0.elapsed_time(e1) / reps


def scene_copies(scat):
    """Identical device copies of a scene that successive updates cycle through, so that no update finds part of its
    input in the 126 MB L2 from the update before: three copies when the scene is below 4 GB (>= 1.4 GB in rotation),
    the scene itself when it is larger (7.5 GB per pass: nothing survives)."""
    nbytes = sum(v.numel() * v.element_size() for v in scat.values())
    if nbytes >= 4e9 or nbytes == 0:
        return [scat]
    return [scat] + [{k: v.clone() for k, v in scat.items()} for _ in range(2)]


def timed_run(S, wl, scats, dev, local_rank, steps, warmup, world, dist, opts, peak, doppler_mode=0, lut=None):
    """warmup + steps passes of the whole hot path over device-resident input, timed on the device.
    scats: identical copies of the (local) scene, used in rotation (scene_copies).
    Returns a dict of measurements (times are the max over ranks)."""
    U, P, G, N = wl.n_updates, wl.pulses_per_update, wl.n_gates, wl.n_doppler
    scat = scats[0]
    n_local = scat["x"].numel()
    sats = [S.sat_for(wl, u) for u in range(U)]
    sim = S.Sim(S.config_for(wl, max_pending_updates=U + 1, device=local_rank, doppler_mode=doppler_mode))
    if lut is not None:
        sim.set_antenna_lut(*lut)
    turn = [0]
    for kv in opts:
        k, v = kv.split("=")
        sim.set_option(int(k), int(v))
    iq = torch.empty((U * P, G), dtype=torch.complex64, device=dev)
    stream = torch.cuda.current_stream(dev)
    acc_events, syn_events = [], []

    # Accumulation time: on one GPU ONE event pair brackets the U back-to-back accumulations of a step (mean = elapsed / U):
    # an event record between two launches costs about 3 us of GPU time per update and serialises launches that the
    # library lets overlap (the prologue of an accumulation kernel runs under the finalize kernel of the update before).
    # With several ranks the all-reduce sits between the updates, so every update gets its own pair.
    per_update_events = world > 1

    def step(record):
        if record and not per_update_events:
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(stream)
        for u in range(U):
            if record and per_update_events:
                e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                e0.record(stream)
            sim.accumulate_update(scats[turn[0] % len(scats)], sats[u])
            turn[0] += 1
            if record and per_update_events:
                e1.record(stream)
                acc_events.append((e0, e1, 1))
            if world > 1:   # the one exchange step: partial spectra -> full spectrum
                D.allreduce_spectrum(sim.spectrum_view(sim.stats()["updates_accumulated"] - 1))
        if record and not per_update_events:
            e1.record(stream)
            acc_events.append((e0, e1, U))
        if record:
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(stream)
        sim.synthesize_pulses(U * P, iq, flags=S.SYN_FINAL)
        if record:
            e1.record(stream)
            syn_events.append((e0, e1))

    def barrier():
        torch.cuda.synchronize(dev)
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize(dev)

    for _ in range(warmup):
        step(False)
    barrier()
    sim.read_counters(reset=True)
    launches0 = sim.stats()["kernel_launches"]
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    with clock_sampler(dev) as clk:
        barrier()
        ev0.record(stream)
        for _ in range(steps):
            step(True)
        ev1.record(stream)
        barrier()
    total_ms = ev0.elapsed_time(ev1)
    launches = sim.stats()["kernel_launches"] - launches0
    counters = sim.read_counters()
    acc_ms_mean = statistics.mean(a.elapsed_time(b) / n for a, b, n in acc_events)
    syn_ms_mean = statistics.mean(a.elapsed_time(b) for a, b in syn_events)
    if world > 1:
        t = torch.tensor([total_ms, acc_ms_mean, syn_ms_mean], device=dev, dtype=torch.float64)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        total_ms, acc_ms_mean, syn_ms_mean = float(t[0]), float(t[1]), float(t[2])
    ms_per_step = total_ms / steps
    achieved = BYTES_PER_SCATTERER * n_local / (acc_ms_mean * 1e-3) / 1e9
    inw = in_window_fraction(sim, S, scat, sats[0])
    syn_bytes = U * 24 * G * N      # per segment and gate: two spectra rows read + one IQ row written
    return {
        "ms_per_step": ms_per_step, "value": U * wl.n_scatterers / (ms_per_step * 1e-3),
        "iq_samples_per_s": U * P * G / (ms_per_step * 1e-3),
        "split_ms": {"accumulate_per_update": acc_ms_mean, "synthesize_per_step": syn_ms_mean,
                     "launch_gaps_per_step": ms_per_step - U * acc_ms_mean - syn_ms_mean},
        "roofline": {"bound": "hbm", "kernel": "acc_kernel", "achieved": achieved, "peak": peak, "unit": "GB/s",
                     "frac": achieved / peak, "traffic": committed_traffic(wl.name),
                     "traffic_source": "committed ncu --set full capture of this kernel on this workload "
                                       "(profiles/acc_kernel_traffic.csv); not measured in this run",
                     "l2": (f"{len(scats)} identical device copies of the scene used in rotation "
                            f"({len(scats) * BYTES_PER_SCATTERER * n_local / 1e9:.2f} GB >> 126 MB L2): every update reads from DRAM"
                            if len(scats) > 1 else "one pass reads more than the L2 holds many times over: no flush needed"),
                     "algorithmic_bytes_per_launch": BYTES_PER_SCATTERER * n_local, "launch_ms": acc_ms_mean,
                     "frac_of_8TBs_nominal": achieved / 8000.0},
        "synthesis": {"kernel": "synth_kernel", "ms": syn_ms_mean, "algorithmic_bytes": syn_bytes,
                      "achieved_gbs": syn_bytes / (syn_ms_mean * 1e-3) / 1e9, "floor_us_at_peak": 1e6 * syn_bytes / (peak * 1e9)},
        "in_window_fraction_update0": inw, "gpu_launches": launches, "clocks": clk.summary(),
        "escapes_per_step": counters["escapes"] / max(1, steps),
        "index_fallbacks_per_step": counters["index_fallbacks"] / max(1, steps),
        "steps": steps, "warmup": warmup,
    }


def next_row(name, what, wl, r):
    """One SURVEY.md 8(f) row measured like the main line (same events, same clock sampler)."""
    return {"row": name, "what": what, "workload": wl.name, "ms_per_update": r["split_ms"]["accumulate_per_update"],
            "value": wl.n_scatterers / (r["split_ms"]["accumulate_per_update"] * 1e-3), "unit": "scatterers/s",
            "frac_of_hbm_peak": r["roofline"]["frac"], "steps": r["steps"], "clocks": r["clocks"]}


def gaussian_table(wl, dev, n=512):
    """A synthetic u-v antenna table for the timing of the tabulated-gain path: the analytic Gaussian of the workload
    sampled on n x n points over the directions the scene spans (the paper's tables are not available)."""
    half = 1.05 * max(wl.n_along, wl.n_cross) * wl.spacing_m / 2.0 / W.ALTITUDE_M
    step = 2.0 * half / (n - 1)
    u = -half + step * torch.arange(n, device=dev, dtype=torch.float64)
    g = torch.exp(-wl.antenna_alpha * (u[None, :] ** 2 + u[:, None] ** 2))
    return torch.complex(g, torch.zeros_like(g)).to(torch.complex64).contiguous(), -half, step, -half, step


def event_ms(dev, fn, reps=5):
    """Median device time of fn() over reps runs after one untimed run, with the clock sampler around them."""
    stream = torch.cuda.current_stream(dev)
    fn()
    torch.cuda.synchronize(dev)
    ts = []
    with clock_sampler(dev) as clk:
        for _ in range(reps):
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(stream)
            fn()
            e1.record(stream)
            torch.cuda.synchronize(dev)
            ts.append(e0.elapsed_time(e1))
    return statistics.median(ts), clk.summary()


def regular_row(S, wl, scat, dev, n_pulses=256):
    """sim_regular_pulses: every scatterer at every pulse, the scene resident on the device."""
    sim = S.Sim(S.config_for(wl, device=dev.index or 0))
    out = torch.empty((n_pulses, wl.n_gates), dtype=torch.complex64, device=dev)
    ms, clk = event_ms(dev, lambda: sim.regular_pulses(scat, S.sat_for(wl, 0), 0, n_pulses, out=out))
    return {"row": "regular_mode", "what": f"sim_regular_pulses, {n_pulses} pulses (PAPER.md:27, :33)", "workload": wl.name,
            "ms": ms, "value": wl.n_scatterers * n_pulses / (ms * 1e-3), "unit": "scatterer-pulses/s", "clocks": clk}


def burst_row(S, wl, dev, burst=64):
    """sim_burst_beams on an IQ stream of the track config's shape (random values)."""
    sim = S.Sim(S.config_for(wl, device=dev.index or 0))
    iq = torch.randn((wl.n_pulses, wl.n_gates, 2), device=dev, generator=torch.Generator(device=dev).manual_seed(5))
    iq = torch.view_as_complex(iq).contiguous()
    ms, clk = event_ms(dev, lambda: sim.burst_beams(iq, burst), reps=20)
    nbytes = 2 * iq.numel() * 8
    return {"row": "burst_fft", "what": f"sim_burst_beams, bursts of {burst} pulses (PAPER.md:145-149)", "workload": wl.name,
            "ms": ms, "value": iq.numel() / (ms * 1e-3), "unit": "IQ samples/s", "algorithmic_bytes": nbytes,
            "achieved_gbs": nbytes / (ms * 1e-3) / 1e9, "clocks": clk}


OTHER_WORKLOADS = ["nadir_patch_16m", "sweep_p16", "sweep_p32", "sweep_p64", "sweep_p128", "sweep_p256", "sweep_p512",
                   "track_segment_67m"]


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--workload", default=DEFAULT_WORKLOAD, choices=sorted(W.WORKLOADS))
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-others", action="store_true", help="skip the short runs of the other configs")
    ap.add_argument("--opt", action="append", default=[], help="KEY=VALUE library option (SIM_OPT_* number)")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup
    wl = W.get(args.workload)

    if args.impl == "reference":
        run_reference(args, wl)
        return

    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the product has no CPU fallback")
    if "WORLD_SIZE" not in os.environ and args.gpus > 1:
        # `python bench.py --gpus N` by itself: start the N ranks here (one process per GPU under torchrun, the same
        # command line the driver uses), instead of quietly measuring one GPU
        if torch.cuda.device_count() < args.gpus:
            raise SystemExit(f"bench.py --gpus {args.gpus}: this node shows {torch.cuda.device_count()} CUDA device(s)")
        import socket
        with socket.socket() as so:
            so.bind(("127.0.0.1", 0))
            port = so.getsockname()[1]
        env = dict(os.environ)
        env.setdefault("NCCL_DEBUG", "INFO")          # the init lines name every rank, its GPU and the transport
        env.setdefault("NCCL_DEBUG_SUBSYS", "INIT")
        cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}",
               "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__), *sys.argv[1:]]
        sys.stdout.flush()
        os.execve(sys.executable, cmd, env)
    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if world != args.gpus and rank == 0:
        print(f"bench.py: --gpus {args.gpus} but WORLD_SIZE = {world}: n_gpus reports the {world} rank(s) that run",
              file=sys.stderr)
    if local_rank >= torch.cuda.device_count():
        raise SystemExit(f"bench.py: rank {rank} has no GPU (LOCAL_RANK {local_rank}, {torch.cuda.device_count()} visible)")
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=dev)

    from paper_2408_11472_b200 import sim as S
    S.load_library()
    peak, peak_src = measured_peak()

    U, P, G, N = wl.n_updates, wl.pulses_per_update, wl.n_gates, wl.n_doppler
    scat_full = W.scatterers(wl, device=dev)
    scat = D.shard_scatterers(scat_full, wl.n_cross, rank, world)
    if world > 1:
        del scat_full
    n_local = scat["x"].numel()
    sats = [S.sat_for(wl, u) for u in range(U)]
    stream = torch.cuda.current_stream(dev)

    def barrier():
        torch.cuda.synchronize(dev)
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize(dev)

    scats = scene_copies(scat)
    main_run = timed_run(S, wl, scats, dev, local_rank, args.steps, args.warmup, world, dist, args.opt, peak)
    main_run["roofline"]["peak_source"] = peak_src
    del scats[1:]

    # ---- end to end through the C ABI with HOST buffers (pinned), copies inside the timed region ----
    e2e = None
    if not args.no_e2e:
        chunk = 1 << 22
        cfg_h = S.config_for(wl, max_pending_updates=U + 1, device=local_rank, host_stage_scatterers=chunk,
                             host_stage_pulses=U * P)
        sim_h = S.Sim(cfg_h)
        host = {k: torch.empty(v.shape, dtype=v.dtype, pin_memory=True).copy_(v) for k, v in scat.items()}
        iq_h = torch.empty((U * P, G), dtype=torch.complex64, pin_memory=True)
        k_e2e = max(1, min(args.steps, 3))

        def step_h():
            for u in range(U):
                sim_h.accumulate_update_host(host, sats[u])
                if world > 1:
                    D.allreduce_spectrum(sim_h.spectrum_view(sim_h.stats()["updates_accumulated"] - 1))
            sim_h.synthesize_pulses_host(U * P, iq_h, flags=S.SYN_FINAL)

        step_h()
        sim_h.synchronize()
        barrier()
        t0 = time.perf_counter()
        h0, h1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        h0.record(stream)
        for _ in range(k_e2e):
            step_h()
        h1.record(stream)
        sim_h.synchronize()
        barrier()
        e2e_ms = h0.elapsed_time(h1) / k_e2e
        e2e_wall_ms = (time.perf_counter() - t0) * 1e3 / k_e2e
        e2e_ms = max(e2e_ms, e2e_wall_ms)   # the host-side enqueue can be the longer leg
        if world > 1:
            t = torch.tensor([e2e_ms], device=dev, dtype=torch.float64)
            dist.all_reduce(t, op=dist.ReduceOp.MAX)
            e2e_ms = float(t[0])
        e2e = {"value": U * wl.n_scatterers / (e2e_ms * 1e-3), "unit": "scatterers/s",
               "h2d_bytes_per_step": U * BYTES_PER_SCATTERER * n_local * world,
               "d2h_bytes_per_step": U * P * G * 8 * world, "ms_per_step": e2e_ms, "steps": k_e2e,
               "note": "sim_accumulate_update_host / sim_synthesize_pulses_host from pinned host buffers, "
                       f"{chunk}-scatterer double-buffered H2D chunks"}
        del sim_h, host

    cpu_baseline = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        from oracle import oracle as orc
        orc.build()
        # whole rows spread evenly over the scene (dark and illuminated parts in scene proportion), oracle as it stands
        rows = strided_rows(wl, 1 << 22)
        idx = torch.tensor(rows, device=dev)
        sub = {k: v.view(wl.n_along, wl.n_cross)[idx].reshape(-1).cpu() for k, v in scat.items()}
        v, desc, used, _, inw = cpu_oracle_sample(wl, sub, orc.max_threads(), target_s=12.0)
        v1, _, _, _, _ = cpu_oracle_sample(wl, sub, 1, target_s=3.0)     # the same oracle on one core (BASELINE.md plan)
        cpu_baseline = {"value": v, "unit": "scatterers/s", "cores": used, "kind": "oracle", "sample": desc,
                        "single_thread_value": v1, "sample_in_window_fraction": inw,
                        "scene_in_window_fraction_update0": main_run["in_window_fraction_update0"]}

    # ---- SURVEY.md 8(f) rows on this box: pulse-pair Doppler and the tabulated gain on this workload ----
    next_rows = []
    if world == 1 and not args.no_others:
        k_next = max(3, min(args.steps, 5))
        r = timed_run(S, wl, [scat], dev, local_rank, k_next, 3, 1, None, args.opt, peak, doppler_mode=S.DOPPLER_PULSE_PAIR)
        next_rows.append(next_row("pulse_pair_doppler", "sim_accumulate_update, SIM_DOPPLER_PULSE_PAIR (PAPER.md:81-83)", wl, r))
        tab = gaussian_table(wl, dev)
        r = timed_run(S, wl, [scat], dev, local_rank, k_next, 3, 1, None, args.opt, peak, lut=tab)
        next_rows.append(next_row("tabulated_antenna_gain", "sim_accumulate_update after sim_set_antenna_lut, 512 x 512 "
                                  "complex u-v table (PAPER.md:35)", wl, r))
        del tab

    # ---- the other configs, short runs with the same event timing (configs[1], [3], [4]) ----
    others = []
    if world == 1 and not args.no_others and args.workload == DEFAULT_WORKLOAD:
        del scat, scat_full
        torch.cuda.empty_cache()
        scenes = {}
        for name in OTHER_WORKLOADS:
            w2 = W.get(name)
            key = (w2.n_along, w2.n_cross, w2.seed, w2.sea)
            if key not in scenes:
                scenes.clear()
                torch.cuda.empty_cache()
                scenes[key] = W.scatterers(w2, device=dev)
                scenes[key] = scene_copies(scenes[key])
            r = timed_run(S, w2, scenes[key], dev, local_rank, 3 if w2.n_updates > 16 else 10, 3, 1, None, args.opt, peak)
            others.append({"workload": name, "scatterers": w2.n_scatterers, "gates": w2.n_gates, "doppler_bins": w2.n_doppler,
                           "pulses_per_update": w2.pulses_per_update, "updates": w2.n_updates, **r})
            if name == "nadir_patch_16m":     # regular mode on the same resident scene
                next_rows.append(regular_row(S, w2, scenes[key][0], dev))
        scenes.clear()
        torch.cuda.empty_cache()
        next_rows.append(burst_row(S, W.get("track_segment_67m"), dev))

    if rank == 0:
        out = {
            "metric": "scatterers accumulated + IQ synthesised per second (whole step)",
            "value": main_run["value"], "unit": "scatterers/s", "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": main_run["ms_per_step"], "higher_is_better": True, "scaling": "strong", "vs_baseline": None,
            "vs_baseline_note": "BASELINE.md holds no published number for this metric and workload (the paper quotes wall "
                                "times of its own scenario on its own GPUs); cpu_baseline is the oracle on this box",
            "dtype": "f32", "dtype_note": "fp32 amplitudes, accumulation (block-floating int32 tiles, fp64 global accumulator) and FFT; fp64 range, gate/bin index and phase reduction",
            "data": "synthetic",
            "config": {"workload": wl.name, "scatterers": wl.n_scatterers, "gates": G, "doppler_bins": N,
                       "pulses_per_update": P, "updates": U, "l2": main_run["roofline"]["l2"],
                       "parallelism": f"scatterer-sharded x{world}, all-reduce of spectra" if world > 1 else "1 GPU",
                       "in_window_fraction_update0": main_run["in_window_fraction_update0"]},
            "iq_samples_per_s": main_run["iq_samples_per_s"],
            "split_ms": main_run["split_ms"],
            "roofline": main_run["roofline"], "synthesis": main_run["synthesis"],
            "empty_launch_us": empty_launch_us(dev),
            "cpu_baseline": cpu_baseline, "e2e": e2e, "gpu_launches": main_run["gpu_launches"],
            "clocks": main_run["clocks"], "escapes_per_step": main_run["escapes_per_step"],
            "index_fallbacks_per_step": main_run["index_fallbacks_per_step"],
            "other_workloads": others, "next_rows": next_rows,
        }
        print(json.dumps(out), flush=True)
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
