#!/usr/bin/env python
"""Throughput of the regular-mode kernel (sim_regular_pulses, reading R5): the
16.8M-scatterer nadir patch evaluated at 256 pulses.  Prints one JSON line.  (bench.py measures the hot path.)
    python -m paper_2408_11472_b200.bench_regular [n_pulses]"""
import json
import statistics
import sys

import torch

from paper_2408_11472_b200 import sim as S, workloads as W


def main():
    n_pulses = int(sys.argv[1]) if len(sys.argv) > 1 else 256
    S.load_library()
    wl = W.get("nadir_patch_16m")
    scat = W.scatterers(wl, device="cuda")
    sim = S.Sim(S.config_for(wl))
    out = torch.empty((n_pulses, wl.n_gates), dtype=torch.complex64, device="cuda")
    stream = torch.cuda.current_stream()
    ts = []
    for rep in range(6):
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(stream)
        sim.regular_pulses(scat, S.sat_for(wl, 0), 0, n_pulses, out=out)
        e1.record(stream)
        torch.cuda.synchronize()
        ts.append(e0.elapsed_time(e1))
    ms = statistics.median(ts[1:])
    print(json.dumps({"metric": "scatterer-pulses/s (regular mode)", "value": wl.n_scatterers * n_pulses / (ms * 1e-3),
                      "ms": ms, "config": {"workload": wl.name, "pulses": n_pulses, "scatterers": wl.n_scatterers}}))


if __name__ == "__main__":
    main()
