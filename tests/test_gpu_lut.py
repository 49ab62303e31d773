"""GPU parity of the tabulated antenna pattern (sim_set_antenna_lut, reading R9) against
oracle.spectrum_lut on the same seeded scenes and synthetic tables: relative L2 <= 1e-4 per spectrum grid."""
import numpy as np
import pytest
import torch

from paper_2408_11472_b200 import workloads as W
from tests import gpu_util as U

pytestmark = pytest.mark.gpu


def pattern(nu, nv, half_u, half_v, alpha):
    """Synthetic complex pattern: Gaussian main lobe, a ripple and a phase ramp, sampled on the grid."""
    u0, v0 = -half_u, -half_v
    du, dv = 2 * half_u / (nu - 1), 2 * half_v / (nv - 1)
    u = (u0 + du * np.arange(nu))[None, :]
    v = (v0 + dv * np.arange(nv))[:, None]
    g = np.exp(-alpha * (u * u + v * v)) * (1.0 + 0.3 * np.cos(900.0 * u)) * np.exp(1j * (200.0 * u - 150.0 * v))
    return g.astype(np.complex64), u0, du, v0, dv


def run(sim_mod, orc, wl, tab, u0, du, v0, dv, sat_kw=None, variants=(0, 4), tol=U.TOL, doppler_mode=0):
    scat = W.scatterers(wl)
    scat_np, scat_cuda = U.to_numpy(scat), U.to_cuda(scat)
    st = W.sat_state(wl, 0)
    st.update(sat_kw or {})
    sat_o = orc.make_sat(st["pos"], st["vel"], st["boresight"], st["range_gate0_m"])
    sat_g = sim_mod.make_sat(st["pos"], st["vel"], st["boresight"], st["range_gate0_m"])
    T_ref = orc.spectrum_lut(U.oracle_cfg(orc, wl, doppler_mode=doppler_mode), sat_o, tab, u0, du, v0, dv, *[scat_np[f] for f in W.FIELDS],
                             nthreads=orc.max_threads())
    assert np.abs(T_ref).max() > 0
    worst = 0.0
    for variant in variants:
        sim = sim_mod.Sim(sim_mod.config_for(wl, doppler_mode=doppler_mode))
        sim.set_option(sim_mod.OPT_ACC_VARIANT, variant)
        sim.set_antenna_lut(torch.from_numpy(tab).cuda(), u0, du, v0, dv)
        sim.accumulate_update(scat_cuda, sat_g)
        T = sim.get_spectrum(0).cpu().numpy()
        e = U.rel_l2(T, T_ref)
        assert e <= tol, (variant, e)
        worst = max(worst, e)
        # clearing the table restores the analytic gain
        sim.set_antenna_lut(None)
        sim.accumulate_update(scat_cuda, sat_g)
        T_an = sim.get_spectrum(1).cpu().numpy()
        T_an_ref = U.oracle_spectra(orc, wl, scat_np, [0], doppler_mode=doppler_mode)[0] if not sat_kw else None
        if T_an_ref is not None:
            assert U.rel_l2(T_an, T_an_ref) <= U.TOL
    return worst


@pytest.fixture(scope="module")
def sim_mod():
    if not torch.cuda.is_available():
        pytest.fail("GPU tests need a CUDA device")
    from paper_2408_11472_b200 import sim
    sim.load_library()
    return sim


def test_lut_whole_footprint(oracle, sim_mod):
    # SAR footprint recipe (PM sea) at 32 m spacing: spans +-8 km, u and v up to +-0.0101; table covers it
    wl = W.get("sar_footprint_268m").scaled(n_along=512, n_cross=512, spacing_m=32.0, n_updates=2)
    tab, u0, du, v0, dv = pattern(257, 193, 0.0112, 0.0108, wl.antenna_alpha)
    run(sim_mod, oracle, wl, tab, u0, du, v0, dv)


def test_lut_nadir_patch_off_nadir_boresight_and_tilted_velocity(oracle, sim_mod):
    wl = W.get("nadir_patch_16m").scaled(n_along=1000, n_cross=1021, n_updates=2)
    tab, u0, du, v0, dv = pattern(129, 129, 0.004, 0.004, wl.antenna_alpha)
    run(sim_mod, oracle, wl, tab, u0, du, v0, dv, sat_kw={"boresight": (0.0012, -0.0007, -1.0), "vel": (6990.0, 120.0, -3.0)})


def test_lut_with_pulse_pair_doppler(oracle, sim_mod):
    wl = W.get("nadir_patch_16m").scaled(n_along=600, n_cross=700, n_updates=2)
    tab, u0, du, v0, dv = pattern(129, 97, 0.004, 0.004, wl.antenna_alpha)
    run(sim_mod, oracle, wl, tab, u0, du, v0, dv, doppler_mode=1)


def test_lut_partly_outside_the_recorded_pattern(oracle, sim_mod):
    # the table covers only +-0.004 of a +-0.0101 footprint: everything outside contributes exactly nothing
    wl = W.get("sar_footprint_268m").scaled(n_along=512, n_cross=512, spacing_m=32.0, n_updates=2)
    tab, u0, du, v0, dv = pattern(65, 65, 0.004, 0.004, wl.antenna_alpha)
    run(sim_mod, oracle, wl, tab, u0, du, v0, dv)


def test_lut_errors(sim_mod):
    wl = W.get("tiny")
    sim = sim_mod.Sim(sim_mod.config_for(wl))
    tab = torch.ones((4, 4), dtype=torch.complex64, device="cuda")
    with pytest.raises(sim_mod.SimError):
        sim.set_antenna_lut(tab, 0.0, 0.0, 0.0, 1.0)           # du = 0
    with pytest.raises(sim_mod.SimError):
        sim.set_antenna_lut(tab[:1], 0.0, 1.0, 0.0, 1.0)       # n_v = 1
    sim.set_antenna_lut(tab, -1.0, 1.0, -1.0, 1.0)
    scat = U.to_cuda(W.scatterers(wl))
    st = W.sat_state(wl, 0)
    with pytest.raises(sim_mod.SimError):                      # velocity parallel to the boresight
        sim.accumulate_update(scat, sim_mod.make_sat(st["pos"], (0.0, 0.0, -7000.0), (0.0, 0.0, -1.0), st["range_gate0_m"]))
    assert sim.stats()["updates_accumulated"] == 0
    with pytest.raises(sim_mod.SimError):                      # regular mode has no table
        sim.regular_pulses(scat, sim_mod.sat_for(wl, 0), 0, 4)
