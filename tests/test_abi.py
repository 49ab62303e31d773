"""CPU-only checks of the boundary: libsim.so builds, loads and exports every symbol include/sim.h
declares; host-only entry points validate their arguments.  No compute call is made here."""
import ctypes as C
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def sim_mod():
    from paper_2408_11472_b200 import sim
    sim.load_library()
    return sim


def declared_symbols():
    text = open(os.path.join(ROOT, "include", "sim.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(sim_[a-z_]+)\s*\(", text)))


def test_header_symbols_are_exported(sim_mod):
    names = declared_symbols()
    assert {"sim_create", "sim_accumulate_update", "sim_synthesize_pulses", "sim_destroy"} <= set(names)
    lib = sim_mod.load_library()
    for n in names:
        assert hasattr(lib, n), f"{n} declared in sim.h but not exported by libsim.so"
    assert sorted(sim_mod.EXPORTS) == names       # the binding names every entry point


def test_struct_layout_matches_header(sim_mod):
    # sizes the C side checks through struct_size; offsets follow natural alignment
    assert C.sizeof(sim_mod.SimConfig) == 4 * 8 + 8 * 4 + 8 * 2
    assert sim_mod.SimConfig.doppler_mode.offset == 28 and sim_mod.SimConfig.wavelength_m.offset == 32
    assert C.sizeof(sim_mod.SimScatterers) == 8 * 8
    assert C.sizeof(sim_mod.SimSatState) == 8 * 10
    assert C.sizeof(sim_mod.SimStats) == 8 * 4


def test_workspace_bytes_and_config_validation(sim_mod):
    lib = sim_mod.load_library()
    n = C.c_size_t()
    cfg = sim_mod.make_config(128, 512, 512, 0.0221, 18000.0, 0.468, 4995.0, max_pending_updates=3)
    assert lib.sim_workspace_bytes(C.byref(cfg), C.byref(n)) == sim_mod.OK
    assert n.value >= 3 * 128 * 512 * 8 + 256 * 8
    base = n.value
    cfg2 = sim_mod.make_config(128, 512, 512, 0.0221, 18000.0, 0.468, 4995.0, max_pending_updates=3,
                               host_stage_scatterers=1 << 20, host_stage_pulses=2048)
    assert lib.sim_workspace_bytes(C.byref(cfg2), C.byref(n)) == sim_mod.OK
    assert n.value >= base + 2 * 7 * 4 * (1 << 20) + 2048 * 128 * 8
    bad = [dict(n_doppler=112), dict(n_doppler=8), dict(n_doppler=4098), dict(n_doppler=8192), dict(n_gates=0), dict(n_gates=1025),
           dict(pulses_per_update=0), dict(max_pending_updates=1), dict(weight_mode=7), dict(wavelength_m=0.0),
           dict(prf_hz=-1.0), dict(gate_spacing_m=float("nan")), dict(antenna_alpha=-1.0),
           dict(host_stage_scatterers=3)]
    for kw in bad:
        args = dict(n_gates=64, n_doppler=64, pulses_per_update=64, wavelength_m=0.0221, prf_hz=18000.0,
                    gate_spacing_m=0.468, antenna_alpha=1.0)
        args.update(kw)
        c = sim_mod.make_config(**args)
        assert lib.sim_workspace_bytes(C.byref(c), C.byref(n)) == sim_mod.ERR_BAD_CONFIG, kw
        assert lib.sim_last_error(None)
    c = sim_mod.make_config(64, 64, 64, 0.0221, 18000.0, 0.468, 1.0)
    c.struct_size = 12
    assert lib.sim_workspace_bytes(C.byref(c), C.byref(n)) == sim_mod.ERR_BAD_CONFIG
    assert lib.sim_workspace_bytes(None, C.byref(n)) == sim_mod.ERR_INVALID_ARG
    assert lib.sim_destroy(None) == sim_mod.OK     # NULL-safe


def test_product_path_refuses_cpu(sim_mod):
    import torch
    if torch.cuda.is_available():
        pytest.skip("CUDA present")
    with pytest.raises(RuntimeError, match="no CPU fallback"):
        sim_mod.Sim(sim_mod.make_config(64, 64, 64, 0.0221, 18000.0, 0.468, 1.0))


def test_product_does_not_import_oracle():
    pkg = os.path.join(ROOT, "paper_2408_11472_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".h", ".cuh")):
                src = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(from|import)\s+oracle", src, flags=re.M), f
                assert "liboracle" not in src and "oracle.c" not in src, f
