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


class ClockSampler:
    """nvidia-smi clocks and throttle reasons DURING the timed region (B200_PROFILING.md recipe)."""
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
                "samples": len(sm)}


# ----------------------------------------------------------------------------------------------------
def cpu_oracle_sample(wl, scat_cpu, nthreads, target_s=12.0):
    """Times the oracle, as it stands, on a bounded sample of the workload: passes of one update over the
    central block of ns scatterers (satellite states of successive updates) until about target_s seconds of
    wall time are spent, and one segment (2 spectra -> P pulses x G gates) of synthesis.
    Returns (scatterers/s extrapolated to a whole step, description, threads used, seconds spent)."""
    import numpy as np
    from oracle import oracle as orc
    cfg = orc.make_config(wl.n_gates, wl.n_doppler, wl.pulses_per_update, wl.wavelength_m, wl.prf_hz,
                          wl.gate_spacing_m, wl.antenna_alpha)

    def sat(u):
        st = W.sat_state(wl, u % wl.n_updates)
        return orc.make_sat(st["pos"], st["vel"], st["boresight"], st["range_gate0_m"])

    n = scat_cpu["x"].numel()
    ns = min(n, 1 << 22)
    lo = max(0, n // 2 - ns // 2)
    arrs = [scat_cpu[f][lo:lo + ns].numpy() for f in W.FIELDS]
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
    desc = (f"accumulate: {passes} passes of 1 update over the central {ns} of {S} scatterers in {t_acc:.2f} s; "
            f"synthesize: 1 segment ({wl.pulses_per_update} pulses x {wl.n_gates} gates, naive O(N^2) iDFT) in "
            f"{t_syn:.2f} s; extrapolated to a whole step (U updates x S scatterers + U segments)")
    return value, desc, used, t_acc + t_syn


def run_reference(args, wl):
    """--impl reference: the oracle (oracle/), as it stands, on the host cores; each step a bounded sample."""
    from oracle import oracle as orc
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    orc.build()
    nthreads = orc.max_threads()
    # the sample never needs more than the central rows: generate a reduced scene with the same recipe
    rows = min(wl.n_along, max(64, (1 << 23) // wl.n_cross))
    wl_s = wl.scaled(n_along=rows) if wl.sea != "pm" else wl.scaled(n_along=min(wl.n_along, 1024), n_cross=min(wl.n_cross, 4096))
    scat = W.scatterers(wl_s)
    vals, descs = [], []
    t_all0 = time.perf_counter()
    for i in range(args.warmup + args.steps):
        v, desc, used, _ = cpu_oracle_sample(wl, scat, nthreads, target_s=2.0)   # extrapolates with the full S
        if i >= args.warmup:
            vals.append(v)
            descs.append(desc)
    t_all = time.perf_counter() - t_all0
    value = statistics.mean(vals)
    out = {
        "impl": "reference", "metric": "scatterers accumulated + IQ synthesised per second (whole step)",
        "value": value, "unit": "scatterers/s", "n_gpus": args.gpus, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": 1e3 * wl.n_updates * wl.n_scatterers / value, "higher_is_better": True, "scaling": "strong",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": wl.name, "note": "oracle on host cores; each step a bounded sample of this workload "
                   f"(same recipe, {wl_s.n_along}x{wl_s.n_cross} scatterers generated)"},
        "cpu_baseline": {"value": value, "unit": "scatterers/s", "cores": nthreads, "kind": "oracle",
                         "sample": descs[-1]},
        "e2e": {"value": value, "unit": "scatterers/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0, "wall_s": t_all,
    }
    print(json.dumps(out), flush=True)


# ----------------------------------------------------------------------------------------------------
def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--workload", default=DEFAULT_WORKLOAD, choices=sorted(W.WORKLOADS))
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--opt", action="append", default=[], help="KEY=VALUE library option (SIM_OPT_* number)")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup
    wl = W.get(args.workload)

    if args.impl == "reference":
        run_reference(args, wl)
        return

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the product has no CPU fallback")
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=dev)

    from paper_2408_11472_b200 import sim as S
    S.load_library()

    U, P, G, N = wl.n_updates, wl.pulses_per_update, wl.n_gates, wl.n_doppler
    scat_full = W.scatterers(wl, device=dev)
    scat = D.shard_scatterers(scat_full, wl.n_cross, rank, world)
    if world > 1:
        del scat_full
    n_local = scat["x"].numel()
    sats = [S.sat_for(wl, u) for u in range(U)]

    cfg = S.config_for(wl, max_pending_updates=U + 1, device=local_rank)
    sim = S.Sim(cfg)
    for kv in args.opt:
        k, v = kv.split("=")
        sim.set_option(int(k), int(v))
    iq = torch.empty((U * P, G), dtype=torch.complex64, device=dev)
    stream = torch.cuda.current_stream(dev)

    acc_events = []

    def step(record):
        for u in range(U):
            if record:
                e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                e0.record(stream)
            sim.accumulate_update(scat, sats[u])
            if record:
                e1.record(stream)
                acc_events.append((e0, e1))
            if world > 1:   # the one exchange step: partial spectra -> full spectrum
                D.allreduce_spectrum(sim.spectrum_view(sim.stats()["updates_accumulated"] - 1))
        sim.synthesize_pulses(U * P, iq, flags=S.SYN_FINAL)

    def barrier():
        torch.cuda.synchronize(dev)
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize(dev)

    for _ in range(args.warmup):
        step(False)
    barrier()
    sim.read_counters(reset=True)
    launches0 = sim.stats()["kernel_launches"]
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    syn_ev = []
    with ClockSampler(local_rank) as clk:
        barrier()
        ev0.record(stream)
        for _ in range(args.steps):
            step(True)
        ev1.record(stream)
        barrier()
    total_ms = ev0.elapsed_time(ev1)
    launches = sim.stats()["kernel_launches"] - launches0
    counters = sim.read_counters()
    acc_ms = [a.elapsed_time(b) for a, b in acc_events]
    acc_ms_mean = statistics.mean(acc_ms)
    if world > 1:
        t = torch.tensor([total_ms, acc_ms_mean], device=dev, dtype=torch.float64)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        total_ms, acc_ms_mean = float(t[0]), float(t[1])
    ms_per_step = total_ms / args.steps
    value = U * wl.n_scatterers / (ms_per_step * 1e-3)
    iq_rate = U * P * G / (ms_per_step * 1e-3)
    syn_ms = ms_per_step - U * acc_ms_mean

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

    peak, peak_src = measured_peak()
    achieved = BYTES_PER_SCATTERER * n_local / (acc_ms_mean * 1e-3) / 1e9
    roofline = {"bound": "hbm", "kernel": "acc_ws3_kernel", "achieved": achieved, "peak": peak, "unit": "GB/s",
                "frac": achieved / peak, "traffic": committed_traffic(wl.name), "peak_source": peak_src,
                "algorithmic_bytes_per_launch": BYTES_PER_SCATTERER * n_local, "launch_ms": acc_ms_mean,
                "frac_of_8TBs_nominal": achieved / 8000.0}

    cpu_baseline = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        from oracle import oracle as orc
        orc.build()
        # the central 2048 rows of the scene on the host (bounded copy), oracle as it stands
        rows = min(wl.n_along, max(8, (1 << 24) // wl.n_cross))
        lo = (wl.n_along - rows) // 2 * wl.n_cross
        sub = {k: v[lo:lo + rows * wl.n_cross].cpu() for k, v in scat.items()}
        v, desc, used, _ = cpu_oracle_sample(wl, sub, orc.max_threads(), target_s=12.0)
        v1, _, _, _ = cpu_oracle_sample(wl, sub, 1, target_s=3.0)     # the same oracle on one core (BASELINE.md plan)
        cpu_baseline = {"value": v, "unit": "scatterers/s", "cores": used, "kind": "oracle", "sample": desc,
                        "single_thread_value": v1}

    if rank == 0:
        out = {
            "metric": "scatterers accumulated + IQ synthesised per second (whole step)",
            "value": value, "unit": "scatterers/s", "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "strong", "vs_baseline": None,
            "dtype": "f32", "dtype_note": "fp32 amplitudes, accumulation (block-floating int32 tiles) and FFT; fp64 range, gate/bin index and phase reduction",
            "data": "synthetic",
            "config": {"workload": wl.name, "scatterers": wl.n_scatterers, "gates": G, "doppler_bins": N,
                       "pulses_per_update": P, "updates": U, "l2": "inputs larger than L2 (no flush needed)"
                       if BYTES_PER_SCATTERER * n_local > 2.5e8 else "inputs fit L2: not a bench workload",
                       "parallelism": f"scatterer-sharded x{world}, all-reduce of spectra" if world > 1 else "1 GPU"},
            "iq_samples_per_s": iq_rate,
            "split_ms": {"accumulate_per_update": acc_ms_mean, "synthesize_per_step": syn_ms},
            "roofline": roofline, "cpu_baseline": cpu_baseline, "e2e": e2e, "gpu_launches": launches,
            "clocks": clk.summary(), "escapes_per_step": counters["escapes"] / max(1, args.steps),
            "index_fallbacks_per_step": counters["index_fallbacks"] / max(1, args.steps),
        }
        print(json.dumps(out), flush=True)
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
