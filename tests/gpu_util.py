"""Helpers shared by the GPU parity tests: run the CUDA path through the C ABI and the oracle on the
same seeded arrays, and compare."""
from __future__ import annotations

import numpy as np
import torch

from paper_2408_11472_b200 import workloads as W

TOL = 1e-4   # BASELINE.json:north_star: relative L2 <= 1e-4 per spectrum grid and per IQ block


def rel_l2(a, ref):
    a = np.asarray(a, dtype=np.complex128)
    ref = np.asarray(ref, dtype=np.complex128)
    den = np.linalg.norm(ref.ravel())
    num = np.linalg.norm((a - ref).ravel())
    if den == 0.0:
        return 0.0 if num == 0.0 else float("inf")
    return float(num / den)


def to_numpy(scat):
    return {k: v.detach().cpu().numpy() for k, v in scat.items()}


def to_cuda(scat):
    return {k: v.cuda().contiguous() for k, v in scat.items()}


def oracle_cfg(orc, wl, weight_mode=0, doppler_mode=0):
    return orc.make_config(wl.n_gates, wl.n_doppler, wl.pulses_per_update, wl.wavelength_m, wl.prf_hz,
                           wl.gate_spacing_m, wl.antenna_alpha, weight_mode, doppler_mode)


def oracle_sat(orc, wl, u):
    s = W.sat_state(wl, u)
    return orc.make_sat(s["pos"], s["vel"], s["boresight"], s["range_gate0_m"])


def oracle_spectra(orc, wl, scat_np, updates, weight_mode=0, nthreads=None, doppler_mode=0):
    cfg = oracle_cfg(orc, wl, weight_mode, doppler_mode)
    nthreads = nthreads or orc.max_threads()
    out = []
    for u in updates:
        T, _ = orc.spectrum(cfg, oracle_sat(orc, wl, u), *[scat_np[f] for f in W.FIELDS], nthreads=nthreads)
        out.append(T)
    return np.stack(out)


def gpu_run(sim_mod, wl, scat_cuda, weight_mode=0, options=None, pulses_per_call=None, final=True,
            max_pending=None):
    """Whole stream through the C ABI: U accumulations, U*P pulses.  Returns (spectra, iq, sim)."""
    cfg = sim_mod.config_for(wl, weight_mode=weight_mode,
                             max_pending_updates=max_pending or max(2, wl.n_updates))
    sim = sim_mod.Sim(cfg)
    for k, v in (options or {}).items():
        sim.set_option(k, v)
    spectra = []
    for u in range(wl.n_updates):
        sim.accumulate_update(scat_cuda, sim_mod.sat_for(wl, u))
        spectra.append(sim.get_spectrum(u))
    n = wl.n_pulses
    iq = torch.empty((n, wl.n_gates), dtype=torch.complex64, device="cuda")
    step = pulses_per_call or n
    done = 0
    while done < n:
        m = min(step, n - done)
        sim.synthesize_pulses(m, iq[done:done + m], flags=sim_mod.SYN_FINAL if final else 0)
        done += m
    torch.cuda.synchronize()
    return torch.stack(spectra).cpu().numpy(), iq.cpu().numpy(), sim


def check_stream(orc, wl, T_gpu, iq_gpu, T_ref, weight_mode=0, tol=TOL):
    """Per-spectrum and per-IQ-block relative L2 against the oracle.  Returns the worst errors."""
    worst_T = 0.0
    for u in range(T_ref.shape[0]):
        e = rel_l2(T_gpu[u], T_ref[u])
        worst_T = max(worst_T, e)
        assert e <= tol, f"spectrum {u}: rel L2 {e:.3e} > {tol}"
    cfg = oracle_cfg(orc, wl, weight_mode)
    Y = orc.synthesize(cfg, T_ref, 0, wl.n_pulses, final=True)
    P = wl.pulses_per_update
    worst_Y = 0.0
    for s in range(wl.n_updates):
        e = rel_l2(iq_gpu[s * P:(s + 1) * P], Y[s * P:(s + 1) * P])
        worst_Y = max(worst_Y, e)
        assert e <= tol, f"IQ block {s}: rel L2 {e:.3e} > {tol}"
    return worst_T, worst_Y
