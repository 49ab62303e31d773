"""Host logic of the multi-GPU path on CPU: world_size-2 gloo.  The per-rank partial spectra come from the
oracle here (the CUDA kernels need a GPU); what is under test is the partition and the exchange step."""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2408_11472_b200 import dist as D
from paper_2408_11472_b200 import workloads as W


def test_shard_rows_partition():
    for n, world in ((16384, 8), (4096, 3), (7, 2), (5, 8), (1, 1)):
        edges = [D.shard_rows(n, r, world) for r in range(world)]
        assert edges[0][0] == 0 and edges[-1][1] == n
        assert all(a[1] == b[0] for a, b in zip(edges, edges[1:]))
        sizes = [hi - lo for lo, hi in edges]
        assert max(sizes) - min(sizes) <= 1
    with pytest.raises(ValueError):
        D.shard_rows(8, 2, 2)


def test_shard_scatterers_alignment_and_cover():
    wl = W.get("tiny").scaled(n_along=30, n_cross=8)
    scat = W.scatterers(wl)
    parts = [D.shard_scatterers(scat, wl.n_cross, r, 4) for r in range(4)]
    for f in W.FIELDS:
        assert torch.equal(torch.cat([p[f] for p in parts]), scat[f])
    assert all(p["x"].numel() % 4 == 0 for p in parts)           # bulk copies stay 16-byte aligned
    assert D.shard_scatterers(scat, wl.n_cross, 0, 1) is scat


def _worker(rank, world, port, out):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        from oracle import oracle as orc
        wl = W.get("tiny").scaled(n_along=96, n_cross=64, n_updates=2)
        scat = W.scatterers(wl)
        mine = {k: v.numpy() for k, v in D.shard_scatterers(scat, wl.n_cross, rank, world).items()}
        cfg = orc.make_config(wl.n_gates, wl.n_doppler, wl.pulses_per_update, wl.wavelength_m, wl.prf_hz,
                              wl.gate_spacing_m, wl.antenna_alpha)
        errs = []
        for u in range(wl.n_updates):
            st = W.sat_state(wl, u)
            sat = orc.make_sat(st["pos"], st["vel"], st["boresight"], st["range_gate0_m"])
            part, _ = orc.spectrum(cfg, sat, *[mine[f] for f in W.FIELDS], nthreads=1)
            T = torch.from_numpy(part.astype(np.complex64))
            D.allreduce_spectrum(T)                                # the one exchange step
            full, _ = orc.spectrum(cfg, sat, *[scat[f].numpy() for f in W.FIELDS], nthreads=1)
            errs.append(float(np.linalg.norm(T.numpy() - full) / np.linalg.norm(full)))
        if rank == 0:
            torch.save(errs, out)
    finally:
        dist.destroy_process_group()


def test_gloo_world2_allreduce_of_partial_spectra(tmp_path, oracle):
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    out = str(tmp_path / "errs.pt")
    mp.spawn(_worker, args=(2, port, out), nprocs=2, join=True)
    errs = torch.load(out)
    assert len(errs) == 2 and max(errs) < 1e-6                     # complex64 rounding of the partial sums only
