"""The seeded input generators: shapes, determinism, statistics."""
import math

import numpy as np
import torch

from paper_2408_11472_b200 import workloads as W


def test_registry_matches_baseline_configs():
    t = W.get("tiny")
    assert (t.n_scatterers, t.n_gates, t.n_doppler, t.pulses_per_update, t.n_updates, t.seed) == (65536, 64, 64, 64, 2, 0)
    n = W.get("nadir_patch_16m")
    assert (n.n_scatterers, n.n_gates, n.n_doppler, n.n_updates, n.n_pulses, n.seed) == (16777216, 128, 256, 8, 2048, 1)
    s = W.get("sar_footprint_268m")
    assert (s.n_scatterers, s.n_doppler, s.n_updates, s.n_pulses, s.sea, s.seed) == (268435456, 512, 4, 2048, "pm", 2)
    k = W.get("track_segment_67m")
    assert (k.n_scatterers, k.n_updates, k.n_pulses, k.seed) == (67108864, 64, 16384, 4)
    for p in (16, 32, 64, 128, 256, 512):
        w = W.get(f"sweep_p{p}")
        assert w.n_doppler == p and w.pulses_per_update == p and w.n_scatterers == 16777216 and w.seed == 3
    assert abs(t.range_gate0_m - 814485.024) < 1e-9 and abs(n.range_gate0_m - 814470.048) < 1e-9


def test_white_scene_statistics_and_determinism():
    wl = W.get("tiny")
    a, b = W.scatterers(wl), W.scatterers(wl)
    for f in W.FIELDS:
        assert a[f].dtype == torch.float32 and a[f].shape == (65536,) and torch.equal(a[f], b[f])
    assert float(a["x"][0]) == -127.5 and float(a["y"][1]) == -126.5 and float(a["x"][256]) == -126.5
    assert abs(float(a["z"].std()) - 0.5) < 0.01 and abs(float(a["vz"].std()) - 0.3) < 0.01
    assert abs(float(a["vx"].std()) - 1.0) < 0.02
    ln = torch.log(a["s0dA"])
    assert abs(float(ln.mean()) - math.log(10)) < 0.01 and abs(float(ln.std()) - 0.3) < 0.01
    c = W.scatterers(wl.scaled(seed=5))
    assert not torch.equal(a["z"], c["z"])


def test_pm_scene_is_a_wave_field():
    wl = W.get("sar_footprint_268m").scaled(n_along=512, n_cross=512)
    s = W.scatterers(wl)
    z = s["z"].double().reshape(512, 512)
    assert abs(float(z.std(unbiased=False)) - 0.5) < 1e-4           # rescaled to 2 m SWH exactly
    # spatially correlated (a white field would give ~0), waves run along x
    zx = float((z[1:] * z[:-1]).mean() / z.var())
    assert zx > 0.5
    # orbital velocities: magnitude ~ omega_p * sigma, vertical and along-track comparable
    om = math.sqrt(W.GRAVITY * 0.0805)
    assert 0.2 * om * 0.5 < float(s["vz"].std()) < 5 * om * 0.5
    assert float(s["vx"].std()) > float(s["vy"].std())


def test_satellite_track():
    wl = W.get("track_segment_67m")
    s0, s63 = W.sat_state(wl, 0), W.sat_state(wl, 63)
    assert abs(s0["pos"][0] + 3185.7777) < 1e-3 and abs(s63["pos"][0] - 3086.222) < 1e-2
    assert s0["pos"][2] == 814500.0 and s0["vel"] == (7000.0, 0.0, 0.0) and s0["boresight"] == (0.0, 0.0, -1.0)
