"""The multi-GPU exchange path ("the available devices divide up the batch of tiles ... a
final thread gathers") on the GPU side: each rank accumulates its rows into the spectrum slot of ITS workspace, the
slots are summed in place (Sim.spectrum_view is the all-reduce buffer), and synthesis then reads the reduced slot.
One GPU: two handles stand for two ranks and a plain in-place add stands for the all-reduce (no rank waits on
another).  Two GPUs or more: the same through NCCL, two processes."""
import os
import socket

import numpy as np
import pytest
import torch

from paper_2408_11472_b200 import dist as D
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


def test_partial_spectra_summed_in_place_then_synthesised(oracle, sim_mod):
    wl = W.get("track_segment_67m").scaled(n_along=1024, n_cross=256, n_updates=4)
    scat = W.scatterers(wl)
    scat_np = U.to_numpy(scat)
    T_ref = U.oracle_spectra(oracle, wl, scat_np, range(wl.n_updates))
    world = 2
    parts = [U.to_cuda(D.shard_scatterers(scat, wl.n_cross, r, world)) for r in range(world)]
    sims = [sim_mod.Sim(sim_mod.config_for(wl, max_pending_updates=wl.n_updates)) for _ in range(world)]
    for u in range(wl.n_updates):
        for r in range(world):
            sims[r].accumulate_update(parts[r], sim_mod.sat_for(wl, u))
        views = [s.spectrum_view(u) for s in sims]
        assert views[0].data_ptr() != views[1].data_ptr() and views[0].shape == (wl.n_gates, wl.n_doppler, 2)
        total = views[0] + views[1]
        for v in views:                        # what the all-reduce leaves on every rank: the sum, in the slot itself
            v.copy_(total)
    for r in range(world):
        T = torch.stack([sims[r].get_spectrum(u) for u in range(wl.n_updates)]).cpu().numpy()
        iq = sims[r].synthesize_pulses(wl.n_pulses, flags=sim_mod.SYN_FINAL).cpu().numpy()
        U.check_stream(oracle, wl, T, iq, T_ref)
    # a partial spectrum alone is not the answer (the halves really were different)
    lone = sim_mod.Sim(sim_mod.config_for(wl))
    lone.accumulate_update(parts[0], sim_mod.sat_for(wl, 0))
    assert U.rel_l2(lone.get_spectrum(0).cpu().numpy(), T_ref[0]) > 0.1


def _nccl_worker(rank, world, port, out):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    import torch.distributed as dist
    torch.cuda.set_device(rank)
    dist.init_process_group("nccl", rank=rank, world_size=world, device_id=torch.device("cuda", rank))
    try:
        from paper_2408_11472_b200 import sim as S
        wl = W.get("track_segment_67m").scaled(n_along=1024, n_cross=256, n_updates=3)
        scat = W.scatterers(wl)
        mine = {k: v.cuda(rank).contiguous() for k, v in D.shard_scatterers(scat, wl.n_cross, rank, world).items()}
        sim = S.Sim(S.config_for(wl, max_pending_updates=wl.n_updates, device=rank))
        for u in range(wl.n_updates):
            sim.accumulate_update(mine, S.sat_for(wl, u))
            D.allreduce_spectrum(sim.spectrum_view(u))
        T = torch.stack([sim.get_spectrum(u) for u in range(wl.n_updates)]).cpu()
        iq = sim.synthesize_pulses(wl.n_pulses, flags=S.SYN_FINAL).cpu()
        torch.save({"T": T, "iq": iq}, f"{out}.{rank}")
    finally:
        dist.destroy_process_group()


@pytest.mark.skipif(torch.cuda.device_count() < 2, reason="needs two GPUs")
def test_nccl_world2(oracle, sim_mod, tmp_path):
    import torch.multiprocessing as mp
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    out = str(tmp_path / "rank")
    mp.spawn(_nccl_worker, args=(2, port, out), nprocs=2, join=True)
    wl = W.get("track_segment_67m").scaled(n_along=1024, n_cross=256, n_updates=3)
    T_ref = U.oracle_spectra(oracle, wl, U.to_numpy(W.scatterers(wl)), range(wl.n_updates))
    for rank in range(2):
        r = torch.load(f"{out}.{rank}")
        U.check_stream(oracle, wl, r["T"].numpy(), r["iq"].numpy(), T_ref)
