"""GPU parity at the stated size of every BASELINE.json config, in the launch configuration bench.py times
(library defaults), and the bin decisions of the PRODUCTION accumulation kernel read back out of the spectrum.

* configs[3] (update-interval sweep on the 16.8M patch): for each P = N in {16 ... 512}: the spectra of all 8
  updates, all 8 IQ blocks (<= 1e-4 each) and all 16.8M index pairs of two updates (bit-exact).
* configs[4] (track): 64 updates over the 67M strip, then ONE sim_synthesize_pulses(16384, SIM_SYN_FINAL) - the
  64-segment single launch bench.py uses - compared per 256-pulse block with the oracle's stream.
* configs[1], [2]: IQ blocks at full size (spectra and indices are in test_gpu_parity.py).
* cells: sparse scenes with one scatterer per (gate, bin) cell, on gate boundaries, on Doppler ties and in ordinary
  positions: the non-zero pattern of sim_get_spectrum must be the oracle's cells (analytic and pulse-pair Doppler,
  guard widths 1 / 16 / 2^18, canonical-only path)."""
import numpy as np
import pytest
import torch

from paper_2408_11472_b200 import workloads as W
from tests import gpu_util as U

pytestmark = [pytest.mark.gpu, pytest.mark.timeout(1800)]


@pytest.fixture(scope="module")
def sim_mod():
    if not torch.cuda.is_available():
        pytest.fail("GPU tests need a CUDA device")
    from paper_2408_11472_b200 import sim
    sim.load_library()
    return sim


@pytest.fixture(scope="module")
def sweep_scene():
    wl = W.get("sweep_p16")                       # the six sweep settings share one scene (seed 3)
    scat = W.scatterers(wl)
    return U.to_numpy(scat), U.to_cuda(scat)


def _indices_exact(orc, sim_mod, wl, scat_cuda, scat_np, sim, u):
    g0, k = sim.debug_indices(scat_cuda, sim_mod.sat_for(wl, u))
    g0r, kr = orc.indices(U.oracle_cfg(orc, wl), U.oracle_sat(orc, wl, u), *[scat_np[f] for f in W.FIELDS[:6]])
    assert np.array_equal(g0.cpu().numpy(), g0r) and np.array_equal(k.cpu().numpy(), kr)


@pytest.mark.parametrize("P", [16, 32, 64, 128, 256, 512])
def test_config4_sweep_full_size(oracle, sim_mod, sweep_scene, P):
    wl = W.get(f"sweep_p{P}")
    scat_np, scat_cuda = sweep_scene
    T_ref = U.oracle_spectra(oracle, wl, scat_np, range(wl.n_updates))
    T, iq, sim = U.gpu_run(sim_mod, wl, scat_cuda)
    eT, eY = U.check_stream(oracle, wl, T, iq, T_ref)
    for u in (0, wl.n_updates - 1):
        _indices_exact(oracle, sim_mod, wl, scat_cuda, scat_np, sim, u)
    print(f"sweep P={P}: worst spectrum rel L2 {eT:.2e}, worst IQ block rel L2 {eY:.2e}")


def test_config5_track_full_stream(oracle, sim_mod):
    wl = W.get("track_segment_67m")
    scat_cuda = W.scatterers(wl, device="cuda")
    scat_np = U.to_numpy(scat_cuda)
    U_, P = wl.n_updates, wl.pulses_per_update
    sim = sim_mod.Sim(sim_mod.config_for(wl, max_pending_updates=U_ + 1))
    T_ref = np.empty((U_, wl.n_gates, wl.n_doppler), np.complex128)
    worst_T = 0.0
    for u in range(U_):
        sim.accumulate_update(scat_cuda, sim_mod.sat_for(wl, u))
        T_ref[u] = U.oracle_spectra(oracle, wl, scat_np, [u])[0]
        e = U.rel_l2(sim.get_spectrum(u).cpu().numpy(), T_ref[u])
        worst_T = max(worst_T, e)
        assert e <= U.TOL, f"update {u}: {e}"
    iq = sim.synthesize_pulses(U_ * P, flags=sim_mod.SYN_FINAL).cpu().numpy()    # ONE launch over 64 segments
    assert iq.shape == (16384, 128) and iq.dtype == np.complex64
    Y = oracle.synthesize(U.oracle_cfg(oracle, wl), T_ref, 0, U_ * P, final=True)
    worst_Y = 0.0
    for s in range(U_):
        e = U.rel_l2(iq[s * P:(s + 1) * P], Y[s * P:(s + 1) * P])
        worst_Y = max(worst_Y, e)
        assert e <= U.TOL, f"IQ block {s}: {e}"
    print(f"track: worst spectrum rel L2 {worst_T:.2e}, worst IQ block rel L2 {worst_Y:.2e}")


def test_config2_nadir_patch_full_stream(oracle, sim_mod):
    wl = W.get("nadir_patch_16m")
    scat = W.scatterers(wl)
    scat_np, scat_cuda = U.to_numpy(scat), U.to_cuda(scat)
    T_ref = U.oracle_spectra(oracle, wl, scat_np, range(wl.n_updates))
    T, iq, _ = U.gpu_run(sim_mod, wl, scat_cuda)
    U.check_stream(oracle, wl, T, iq, T_ref)


def test_config3_sar_footprint_full_stream(oracle, sim_mod):
    wl = W.get("sar_footprint_268m")
    scat_cuda = W.scatterers(wl, device="cuda")
    scat_np = U.to_numpy(scat_cuda)
    T_ref = U.oracle_spectra(oracle, wl, scat_np, range(wl.n_updates))
    T, iq, _ = U.gpu_run(sim_mod, wl, scat_cuda)
    U.check_stream(oracle, wl, T, iq, T_ref)


# ---- bins of the production kernel, read back out of the accumulated spectrum -----------------------------------
def _sparse_scene(wl, kind, seed):
    """<= 4096 scatterers on the nadir column, one per (gate, bin) cell.  kind: 'plain' (well inside the cells),
    'gate_edge' (R - rg0 an exact multiple of the dyadic gate spacing), 'tie' (kf = j + 1/2 exactly)."""
    G, N = wl.n_gates, wl.n_doppler
    r = np.random.default_rng(seed)
    cells = r.permutation((G - 2) * N)[:4096]
    g, k = cells // N + 1, cells % N
    kk = np.where(k >= N // 2, k - N, k).astype(np.float64)           # signed bin
    h0 = 814500.0 - wl.range_gate0_m
    lam_prf = float(np.float32(wl.wavelength_m * wl.prf_hz / (2 * N)))   # m/s per bin, as an fp32 value
    if kind == "plain":
        gf, kf = g + r.uniform(0.2, 0.8, g.size), kk + r.uniform(-0.3, 0.3, g.size)
    elif kind == "gate_edge":
        gf, kf = g.astype(np.float64), kk + r.uniform(-0.3, 0.3, g.size)
    else:
        gf, kf = g + r.uniform(0.2, 0.8, g.size), np.where(kk < N // 2 - 1, kk + 0.5, kk - 0.5)
    z = (h0 - gf * wl.gate_spacing_m).astype(np.float32)             # R = H - z on the nadir column
    vz = (kf * lam_prf).astype(np.float32)
    n = g.size
    zeros = np.zeros(n, np.float32)
    return {"x": zeros.copy(), "y": zeros.copy(), "z": z, "vx": np.full(n, 7000.0, np.float32), "vy": zeros.copy(),
            "vz": vz, "s0dA": np.full(n, 10.0, np.float32)}


@pytest.mark.parametrize("doppler_mode", [0, 1])
@pytest.mark.parametrize("kind", ["plain", "gate_edge", "tie"])
def test_cells_of_the_production_kernel(oracle, sim_mod, kind, doppler_mode):
    wl = W.get("tiny").scaled(n_updates=1, gate_spacing_m=0.5, n_gates=64, n_doppler=128, pulses_per_update=128)
    scat_np = _sparse_scene(wl, kind, seed=17)
    scat_cuda = {k: torch.from_numpy(v).cuda() for k, v in scat_np.items()}
    sat_args = ((0.0, 0.0, 814500.0), (7000.0, 0.0, 0.0), (0.0, 0.0, -1.0), wl.range_gate0_m)   # exactly overhead
    cfg = U.oracle_cfg(oracle, wl, doppler_mode=doppler_mode)
    T_ref, _ = oracle.spectrum(cfg, oracle.make_sat(*sat_args), *[scat_np[f] for f in W.FIELDS])
    g0r, kr = oracle.indices(cfg, oracle.make_sat(*sat_args), *[scat_np[f] for f in W.FIELDS[:6]])
    assert (g0r >= 0).all() and len(set(zip(g0r.tolist(), kr.tolist()))) > 2500     # sparse: mostly one cell each (ties may pair up)
    big = np.abs(T_ref) > 1e-6 * np.abs(T_ref).max()      # (a weight of 1e-11 leaking over a gate edge is below fp32)
    for path, guard in ((1, 16), (1, 1), (1, 1 << 18), (0, 16)):
        sim = sim_mod.Sim(sim_mod.config_for(wl, doppler_mode=doppler_mode))
        sim.set_option(sim_mod.OPT_INDEX_PATH, path)
        sim.set_option(sim_mod.OPT_GUARD_LSB, guard)
        sim.accumulate_update(scat_cuda, sim_mod.make_sat(*sat_args))
        T = sim.get_spectrum(0).cpu().numpy()
        nz = np.abs(T) > 0
        assert not (big & ~nz).any(), (kind, path, guard, "a cell of the oracle is empty on the GPU")
        assert not (nz & (np.abs(T_ref) == 0)).any(), (kind, path, guard, "the GPU filled a cell the oracle leaves empty")
        assert U.rel_l2(T, T_ref) <= U.TOL
