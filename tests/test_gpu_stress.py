"""Randomised (seeded) sweep over scene shapes, sizes, Doppler modes and every tuning knob of the production
accumulation kernel: each draw must match the oracle (rel L2 <= 1e-4) and, above all, terminate: the kernel's
warps talk through mbarriers and shared-memory counters only, so a missed arrival would hang, not fail."""
import os
import random

import numpy as np
import pytest
import torch

from paper_2408_11472_b200 import workloads as W
from tests import gpu_util as U

pytestmark = [pytest.mark.gpu, pytest.mark.timeout(600)]

SHAPES = [(8, 2, 2), (8, 4, 4), (16, 4, 4)]


@pytest.mark.parametrize("seed", [11, 12, 13])
def test_random_shapes_and_options(oracle, seed):
    if not torch.cuda.is_available():
        pytest.fail("GPU tests need a CUDA device")
    from paper_2408_11472_b200 import sim as S
    S.load_library()
    rnd = random.Random(seed)
    for trial in range(int(os.environ.get("SIM_STRESS_TRIALS", "40"))):   # (fewer under compute-sanitizer: profiles/r03_sanitizer.md)
        G = rnd.choice([1, 7, 64, 128, 300])
        N = rnd.choice([16, 64, 256, 2048, 48, 250, 1000])   # powers of two and mixed-radix sizes (bins are taken mod N)
        na, nc = rnd.randint(1, 300), rnd.randint(1, 400)
        sea = rnd.choice(["white", "white", "pm"]) if na >= 8 and nc >= 8 else "white"
        wl = W.get("tiny").scaled(n_along=na, n_cross=nc, n_gates=G, n_doppler=N, pulses_per_update=N, n_updates=1,
                                  spacing_m=rnd.choice([1.0, 8.0, 40.0]), sea=sea, seed=seed * 1000 + trial)
        scat = W.scatterers(wl)
        n = wl.n_scatterers
        if rnd.random() < 0.3:                                    # ragged sizes, including empty
            n = rnd.randint(0, n)
            scat = {a: v[:n].contiguous() for a, v in scat.items()}
        if rnd.random() < 0.2 and n > 10:
            scat["s0dA"][rnd.randint(0, n - 1):] = 0.0            # a dead tail
        dm = rnd.choice([0, 0, 1])
        sim = S.Sim(S.config_for(wl, doppler_mode=dm))
        ncw, pt, il = rnd.choice(SHAPES)
        opts = [(S.OPT_ACC_SHAPE, (ncw << 16) | (pt << 8) | il),
                (S.OPT_ACC_EPOCH, rnd.choice([64, 500, 1024, 2047, 8191, 16383])),
                (None, rnd.choice([0, 2, 3, 4, 8])),      # draw of an option that no longer exists: the seeds keep their scenes
                (S.OPT_ACC_BLOCKS, rnd.choice([0, 1, 2, 5, 37, 296, 1000])),
                (S.OPT_ACC_SUPERCHUNK, rnd.choice([0, 1, 4096, 100000])),
                (S.OPT_ACC_WINDOW_BINS, rnd.choice([0, 1, 3, 7, 12, 16])),
                (S.OPT_ACC_SCATTER, rnd.choice([0, 1])), (S.OPT_INDEX_PATH, rnd.choice([0, 1, 1])),
                (None, rnd.choice([0, 0, 300]))]         # (the same)
        for k, v in opts:
            if k is not None:
                sim.set_option(k, v)
        sim.accumulate_update(U.to_cuda(scat), S.sat_for(wl, 0))
        T = sim.get_spectrum(0).cpu().numpy()
        T_ref = U.oracle_spectra(oracle, wl, U.to_numpy(scat), [0], doppler_mode=dm, nthreads=4)[0]
        e = U.rel_l2(T, T_ref)
        assert e <= U.TOL, (seed, trial, e, G, N, n, sea, dm, (ncw, pt, il), opts[1:])
