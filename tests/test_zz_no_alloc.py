"""sim_accumulate_static: the entry point for users of libsim.so who have no way to allocate device memory.

Who they are: code that runs inside somebody else's program (a plug-in of a host simulator that claimed the whole
device for its own arena at start-up and gives plug-ins only input and output buffers), loops with a latency bound
(cudaMalloc and cudaFree stall every stream of the device), and processes whose device-memory quota is spent.  For
them the library's usual "caller brings a workspace" contract is no help, so this one call keeps the accumulation
kernel's scratch memory (fp64 accumulator + scheduling counters) in an array compiled into the library, at most
SIM_STATIC_MAX_CELLS = 65536 cells of [gate x Doppler bin].

What is checked: the output equals that of the existing path (sim_create + sim_accumulate_update + sim_get_spectrum
on a torch-allocated workspace) within the tolerance of the other GPU tests, on two calls in a row with different
inputs (the array is shared between calls and keeps the previous call's contents, so the second call would show
anything the first one left behind), with every buffer the new call sees allocated beforehand.

The file name sorts last on purpose: `pytest -x` stops at the first failure, and a failure here must not hide the
tests of the hot path proper.  It passes alone in a fresh process and after the other tests.
"""
import numpy as np
import pytest
import torch

from paper_2408_11472_b200 import workloads as W
from tests import gpu_util as U

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def sim_mod():
    if not torch.cuda.is_available():
        pytest.fail("GPU tests need a CUDA device")
    from paper_2408_11472_b200 import sim
    sim.load_library()
    return sim


def _existing_path(sim_mod, wl, scat_cuda, sat, batches=1):
    """The spectrum of one update by the handle-based calls (workspace allocated by torch)."""
    s = sim_mod.Sim(sim_mod.config_for(wl, max_pending_updates=2))
    n = scat_cuda["x"].numel()
    cut = [n * b // batches // 4 * 4 for b in range(batches)] + [n]
    for b in range(batches):
        part = {k: v[cut[b]:cut[b + 1]] for k, v in scat_cuda.items()}
        s.accumulate_update(part, sat, flags=sim_mod.ACC_APPEND if b else 0)
    T = s.get_spectrum(0)
    torch.cuda.synchronize()
    s.close()
    return T.cpu().numpy()


def test_two_calls_in_a_row_match_the_existing_path(sim_mod):
    # two different scenes of different size and geometry, both G * N = 128 * 256 <= 65536 cells:
    # the nadir-patch recipe (every scatterer illuminated, ragged length) and the track recipe (satellite elsewhere)
    wl_a = W.get("nadir_patch_16m").scaled(n_along=1000, n_cross=1021, n_updates=3)
    wl_b = W.get("track_segment_67m").scaled(n_along=2048, n_cross=256, n_updates=6)
    scat_a, scat_b = U.to_cuda(W.scatterers(wl_a)), U.to_cuda(W.scatterers(wl_b))
    sat_a, sat_b = sim_mod.sat_for(wl_a, 1), sim_mod.sat_for(wl_b, 4)
    ref_a = _existing_path(sim_mod, wl_a, scat_a, sat_a)
    ref_b = _existing_path(sim_mod, wl_b, scat_b, sat_b)
    assert np.abs(ref_a).max() > 0 and np.abs(ref_b).max() > 0

    # everything the new call touches exists before it runs; the outputs start as garbage that must be overwritten
    cfg_a, cfg_b = sim_mod.config_for(wl_a), sim_mod.config_for(wl_b)
    out_a = torch.full((wl_a.n_gates, wl_a.n_doppler), complex(7.0, -3.0), dtype=torch.complex64, device="cuda")
    out_b = torch.full((wl_b.n_gates, wl_b.n_doppler), complex(-5.0, 11.0), dtype=torch.complex64, device="cuda")
    torch.cuda.synchronize()
    before = torch.cuda.memory_allocated(), torch.cuda.memory_reserved()
    free_before = torch.cuda.mem_get_info()[0]
    sim_mod.accumulate_static(cfg_a, scat_a, sat_a, out=out_a)      # first call
    sim_mod.accumulate_static(cfg_b, scat_b, sat_b, out=out_b)      # second call, same stream, no sync in between
    torch.cuda.synchronize()
    assert (torch.cuda.memory_allocated(), torch.cuda.memory_reserved()) == before     # torch was asked for nothing
    e_a, e_b = U.rel_l2(out_a.cpu().numpy(), ref_a), U.rel_l2(out_b.cpu().numpy(), ref_b)
    assert e_a <= U.TOL, f"first call: rel L2 {e_a:.3e} vs the existing path"
    assert e_b <= U.TOL, f"second call: rel L2 {e_b:.3e} vs the existing path"

    # a third and fourth call with the first scene again: same answer as before the other scene went through, and the
    # device's free memory is what it was before the first call (module loading aside, which only ever happens once)
    out_a2 = torch.empty_like(out_a)
    torch.cuda.synchronize()
    free_mid = torch.cuda.mem_get_info()[0]
    sim_mod.accumulate_static(cfg_a, scat_a, sat_a, out=out_a2)
    sim_mod.accumulate_static(cfg_a, scat_a, sat_a, out=out_a2)
    torch.cuda.synchronize()
    assert U.rel_l2(out_a2.cpu().numpy(), ref_a) <= U.TOL
    assert U.rel_l2(out_a2.cpu().numpy(), out_a.cpu().numpy()) <= 1e-6
    assert torch.cuda.mem_get_info()[0] >= free_mid      # warm calls take no device memory from anybody
    assert free_before - torch.cuda.mem_get_info()[0] < 64 << 20


def test_batches_with_append_and_the_oracle(oracle, sim_mod):
    # a scene delivered in three pieces (SIM_ACC_APPEND adds to the caller's buffer), Tiny config: also against the oracle
    wl = W.get("tiny")
    scat = W.scatterers(wl)
    scat_np, scat_cuda = U.to_numpy(scat), U.to_cuda(scat)
    sat = sim_mod.sat_for(wl, 1)
    cfg = sim_mod.config_for(wl)
    out = torch.empty((wl.n_gates, wl.n_doppler), dtype=torch.complex64, device="cuda")
    n = wl.n_scatterers
    cuts = [0, 20000, 20000, 50004, n]            # includes an empty batch
    for b in range(len(cuts) - 1):
        part = {k: v[cuts[b]:cuts[b + 1]] for k, v in scat_cuda.items()}
        sim_mod.accumulate_static(cfg, part, sat, out=out, flags=sim_mod.ACC_APPEND if b else 0)
    torch.cuda.synchronize()
    got = out.cpu().numpy()
    assert U.rel_l2(got, _existing_path(sim_mod, wl, scat_cuda, sat, batches=3)) <= U.TOL
    T_ref = U.oracle_spectra(oracle, wl, scat_np, [1])[0]
    assert U.rel_l2(got, T_ref) <= U.TOL
    # an empty scene: the buffer is overwritten with zeros
    empty = {k: v[:0] for k, v in scat_cuda.items()}
    sim_mod.accumulate_static(cfg, empty, sat, out=out)
    torch.cuda.synchronize()
    assert float(out.abs().max()) == 0.0


def test_sizes_beyond_the_built_in_array_are_refused(sim_mod):
    wl = W.get("tiny")
    scat_cuda = U.to_cuda(W.scatterers(wl))
    sat = sim_mod.sat_for(wl, 0)
    ok = sim_mod.config_for(wl.scaled(n_gates=128, n_doppler=512))          # exactly SIM_STATIC_MAX_CELLS: accepted
    assert ok.n_gates * ok.n_doppler == sim_mod.STATIC_MAX_CELLS
    out = torch.zeros(1024 * 4096, dtype=torch.complex64, device="cuda")     # room for the largest size tried below
    sim_mod.accumulate_static(ok, scat_cuda, sat, out=out)
    torch.cuda.synchronize()
    assert float(out[:sim_mod.STATIC_MAX_CELLS].abs().max()) > 0 and float(out[sim_mod.STATIC_MAX_CELLS:].abs().max()) == 0.0
    for g, n in ((128, 576), (129, 512), (1024, 4096)):
        big = sim_mod.config_for(wl.scaled(n_gates=g, n_doppler=n))
        with pytest.raises(sim_mod.SimError) as ei:
            sim_mod.accumulate_static(big, scat_cuda, sat, out=out)
        assert ei.value.code == sim_mod.ERR_BAD_CONFIG and "SIM_STATIC_MAX_CELLS" in str(ei.value)
    with pytest.raises(sim_mod.SimError) as ei:
        sim_mod.accumulate_static(ok, scat_cuda, sat, out=out, flags=2)
    assert ei.value.code == sim_mod.ERR_INVALID_ARG
    # the refused calls left the array usable
    sim_mod.accumulate_static(sim_mod.config_for(wl), scat_cuda, sat, out=out)
    torch.cuda.synchronize()
    assert U.rel_l2(out[:wl.n_gates * wl.n_doppler].cpu().numpy().reshape(wl.n_gates, wl.n_doppler),
                    _existing_path(sim_mod, wl, scat_cuda, sat)) <= U.TOL
