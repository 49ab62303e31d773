"""Pins of the oracle's REGULAR mode against things other than itself:
a 40-digit closed form of one moving scatterer at several pulses, the independent long-double gate-summed
restatement tests/brute.regular_mode_sum, the identity with the fast mode at the update pulse (pin P7), and the
fast mode itself for on-bin scatterers (pin P5 seen from the other side).  CPU only."""
import math

import mpmath as mp
import numpy as np
import pytest

from tests import brute

LAM, PRF, DR, H = 0.0221, 18000.0, 0.468, 814500.0
ALPHA = 4.0 * math.log(2.0) / math.sin(math.radians(1.35)) ** 2
V = 7000.0


def scen(orc, G=64, N=64, alpha=ALPHA):
    rg0 = H - (G // 2) * DR
    return orc.make_config(G, N, N, LAM, PRF, DR, alpha), orc.make_sat((0, 0, H), (V, 0, 0), (0, 0, -1), rg0), rg0


def test_r1_single_moving_scatterer_closed_form(oracle):
    mp.mp.dps = 40
    cfg, sat, rg0 = scen(oracle)
    s = (37.5, -21.25, 0.625, 1.5, -0.75, 0.4375, 8.0)
    arrs = [np.array([v], np.float32) for v in s]
    j0, n = -5, 40
    Y = oracle.regular(cfg, sat, *arrs, j0, n)
    for jj in (0, 5, 17, 39):
        t = mp.mpf(j0 + jj) / mp.mpf(PRF)
        d = [mp.mpf(s[0]) + (mp.mpf(s[3]) - V) * t, mp.mpf(s[1]) + mp.mpf(s[4]) * t,
             mp.mpf(s[2]) - mp.mpf(H) + mp.mpf(s[5]) * t]
        R = mp.sqrt(sum(a * a for a in d))
        gf = (R - mp.mpf(rg0)) / mp.mpf(DR)
        g0 = int(mp.floor(gf))
        w1 = gf - g0
        sin2 = (d[0] ** 2 + d[1] ** 2) / R ** 2                      # boresight (0,0,-1)
        c = mp.sqrt(mp.mpf(s[6])) * mp.exp(-mp.mpf(ALPHA) * sin2) / R ** 2 * mp.expj(-4 * mp.pi * R / mp.mpf(LAM))
        row = Y[jj]
        assert (np.abs(row) > 0).sum() == 2
        for g, w in ((g0, 1 - w1), (g0 + 1, w1)):
            want = complex(w * c)
            assert abs(row[g] - want) < 2e-7 * abs(complex(c)), (jj, g)   # ulp(2R/lambda) = 1.5e-8 cycles = 9e-8 rad


def test_r2_gate_sum_equals_independent_restatement(oracle):
    rng = np.random.default_rng(4)
    n = 300
    cfg, sat, _ = scen(oracle, G=64, alpha=0.0)                      # brute.regular_mode_sum has no antenna
    x = rng.uniform(-50, 50, n).astype(np.float32)
    y = rng.uniform(-50, 50, n).astype(np.float32)
    z = rng.normal(0, 0.5, n).astype(np.float32)
    vx, vy = rng.normal(0, 1, (2, n)).astype(np.float32)
    vz = rng.normal(0, 0.3, n).astype(np.float32)
    s0 = rng.uniform(5, 15, n).astype(np.float32)
    j0, npul = -8, 48
    Y = oracle.regular(cfg, sat, x, y, z, vx, vy, vz, s0, j0, npul, nthreads=3)
    direct = brute.regular_mode_sum(np.stack([x, y, z], 1), np.stack([vx, vy, vz], 1), s0, (0, 0, H), (V, 0, 0),
                                    LAM, PRF, range(j0, j0 + npul))
    assert np.abs(Y.sum(axis=1) - direct).max() <= 2e-7 * np.abs(direct).max()
    assert np.array_equal(Y, oracle.regular(cfg, sat, x, y, z, vx, vy, vz, s0, j0, npul, nthreads=1)) or \
        np.allclose(Y, oracle.regular(cfg, sat, x, y, z, vx, vy, vz, s0, j0, npul, nthreads=1), rtol=1e-12, atol=0)


def test_r3_pulse_zero_is_the_fast_mode_update_pulse(oracle):
    """Reading A2: y_u[g][0] = sum_k T_u[g][k] is the regular-mode coherent sum at the update pulse."""
    from paper_2408_11472_b200 import workloads as W
    wl = W.get("tiny").scaled(n_along=64, n_cross=64)
    scat = {k: v.numpy() for k, v in W.scatterers(wl).items()}
    cfg = oracle.make_config(wl.n_gates, wl.n_doppler, wl.pulses_per_update, wl.wavelength_m, wl.prf_hz,
                             wl.gate_spacing_m, wl.antenna_alpha)
    st = W.sat_state(wl, 1)
    sat = oracle.make_sat(st["pos"], st["vel"], st["boresight"], st["range_gate0_m"])
    T, _ = oracle.spectrum(cfg, sat, *[scat[f] for f in W.FIELDS])
    Y0 = oracle.regular(cfg, sat, *[scat[f] for f in W.FIELDS], 0, 1)[0]
    assert np.abs(T.sum(axis=1) - Y0).max() <= 1e-12 * np.abs(Y0).max()


@pytest.mark.parametrize("N,P", [(16, 16), (32, 16)])
def test_r4_fast_mode_reproduces_regular_mode_for_on_bin_scatterers(oracle, N, P):
    """Nadir-column scatterers with on-bin vertical speeds: the fast mode (LINEAR weights, gate-summed) is the
    regular mode (pin P5, here against oracle_regular instead of the brute force)."""
    rng = np.random.default_rng(12)
    n, G, U = 40, 32, 3
    rg0 = H - (G // 2) * DR
    cfg = oracle.make_config(G, N, P, LAM, PRF, DR, 0.0, oracle.W_LINEAR)
    z0 = rng.uniform(-1.0, 1.0, n)
    vz = rng.integers(-N // 4, N // 4, n) * LAM * PRF / (2 * N)
    s0 = rng.uniform(5, 15, n).astype(np.float32)
    T_all = []
    for u in range(U):
        t = u * P / PRF
        sat = oracle.make_sat((V * t, 0, H), (V, 0, 0), (0, 0, -1), rg0)
        zt = (z0 + vz * t).astype(np.float32)
        T_all.append(oracle.spectrum(cfg, sat, np.full(n, V * t, np.float32), np.zeros(n, np.float32), zt,
                                     np.full(n, V, np.float32), np.zeros(n, np.float32), vz.astype(np.float32), s0)[0])
    Yf = oracle.synthesize(cfg, np.stack(T_all), 0, (U - 1) * P, final=False).sum(axis=1)
    sat0 = oracle.make_sat((0, 0, H), (V, 0, 0), (0, 0, -1), rg0)
    Yr = oracle.regular(cfg, sat0, np.zeros(n, np.float32), np.zeros(n, np.float32), z0.astype(np.float32),
                        np.full(n, V, np.float32), np.zeros(n, np.float32), vz.astype(np.float32), s0,
                        0, (U - 1) * P).sum(axis=1)
    # fp32 rounding of the advanced heights (1e-7 m = 1e-5 cycles) bounds the agreement
    assert np.abs(Yf - Yr).max() <= 2e-4 * np.abs(Yr).max()


# ---- Delay-Doppler burst step ------------------------------------------
@pytest.mark.parametrize("B", [16, 64, 256])
def test_b1_burst_dft_is_numpy_fft_along_pulses(oracle, B):
    rng = np.random.default_rng(B)
    G, nb = 5, 3
    Y = rng.normal(size=(nb * B, G)) + 1j * rng.normal(size=(nb * B, G))
    Z = oracle.burst_dft(Y, B)
    want = np.fft.fft(Y.reshape(nb, B, G), axis=1)                 # library special case
    assert np.allclose(Z, want, rtol=1e-12, atol=1e-12)
    assert np.allclose((np.abs(Z) ** 2).sum(axis=1), B * (np.abs(Y.reshape(nb, B, G)) ** 2).sum(axis=1))   # Parseval


def test_b2_an_on_bin_scatterer_focuses_into_one_beam(oracle):
    """Whole chain: a nadir scatterer whose Doppler sits on bin k of a 64-pulse burst (v_z = k lambda PRF / 128) gives,
    through the regular mode and the burst DFT, one beam: k."""
    B, G = 64, 16
    rg0 = H - (G // 2) * DR
    cfg = oracle.make_config(G, B, B, LAM, PRF, DR, 0.0)
    sat = oracle.make_sat((0, 0, H), (V, 0, 0), (0, 0, -1), rg0)
    for k in (0, 5, -9):
        vz = k * LAM * PRF / (2 * B)
        a = [np.array([v], np.float32) for v in (0.0, 0.0, 0.05, V, 0.0, vz, 10.0)]
        Y = oracle.regular(cfg, sat, *a, 0, B)
        Z = oracle.burst_dft(Y, B)[0]
        p = (np.abs(Z) ** 2).sum(axis=1)
        assert np.argmax(p) == k % B and p[k % B] > 0.97 * p.sum()      # the range changes by < 1 gate over the burst
