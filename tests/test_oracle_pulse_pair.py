"""Pins of the oracle's pulse-pair Doppler mode (Algorithm 1 lines 5-7)
against things other than itself: the LITERAL estimator arg(C_{i+1} C_i^*) PRF / 2 pi evaluated at 50 digits,
the analytic f_D plus its closed-form second-order term, natural aliasing, and the spectrum cell a single
scatterer lands in.  CPU only."""
import math

import mpmath as mp
import numpy as np
import pytest

LAM, PRF, DR, H = 0.0221, 18000.0, 0.468, 814500.0
ALPHA = 4.0 * math.log(2.0) / math.sin(math.radians(1.35)) ** 2


def scen(orc, mode, G=64, N=64, sat_pos=(0.0, 0.0, H), sat_vel=(7000.0, 0.0, 0.0)):
    rg0 = H - (G // 2) * DR
    return (orc.make_config(G, N, N, LAM, PRF, DR, ALPHA, 0, mode), orc.make_sat(sat_pos, sat_vel, (0, 0, -1), rg0))


def scene(n, seed, spread=120.0, vz_sigma=0.3):
    g = np.random.default_rng(seed)
    x = g.uniform(-spread, spread, n).astype(np.float32)
    y = g.uniform(-spread, spread, n).astype(np.float32)
    z = g.normal(0, 0.5, n).astype(np.float32)
    vx = g.normal(0, 1, n).astype(np.float32)
    vy = g.normal(0, 1, n).astype(np.float32)
    vz = g.normal(0, vz_sigma, n).astype(np.float32)
    return x, y, z, vx, vy, vz


def literal_kf(N, sat_pos, sat_vel, s):
    """f_D N / PRF from arg(C_{i+1} conj(C_i)) with C = exp(-i 4 pi R / lambda), 50 digits (PAPER.md:83 in its
    physical form, reading A6): principal value, i.e. in (-N/2, N/2]."""
    mp.mp.dps = 50
    x, y, z, vx, vy, vz = [mp.mpf(float(v)) for v in s]
    tau = 1 / mp.mpf(PRF)
    lam = mp.mpf(LAM)
    d0 = [x - mp.mpf(sat_pos[0]), y - mp.mpf(sat_pos[1]), z - mp.mpf(sat_pos[2])]
    dv = [vx - mp.mpf(sat_vel[0]), vy - mp.mpf(sat_vel[1]), vz - mp.mpf(sat_vel[2])]
    d1 = [a + b * tau for a, b in zip(d0, dv)]
    R0 = mp.sqrt(sum(a * a for a in d0))
    R1 = mp.sqrt(sum(a * a for a in d1))
    C0 = mp.expj(-4 * mp.pi * R0 / lam)
    C1 = mp.expj(-4 * mp.pi * R1 / lam)
    return float(mp.arg(C1 * mp.conj(C0)) / (2 * mp.pi) * N)


def wrap(kf, N):
    return (kf + N / 2) % N - N / 2


@pytest.mark.parametrize("N", [64, 512])
def test_pp1_matches_literal_estimator(oracle, N):
    cfg, sat = scen(oracle, oracle.DOPPLER_PULSE_PAIR, N=N)
    s = scene(60, 11)
    kf = oracle.doppler_coordinate(cfg, sat, *s)
    assert np.isfinite(kf).all()
    for i in range(60):
        lit = literal_kf(N, (0, 0, H), (7000.0, 0, 0), [a[i] for a in s])
        # fp64 cancellation in R' - R (ulp(R) = 1.2e-10 m) is worth 2N/lambda * 2.4e-10 = 1e-5 bins at N = 512
        assert abs(wrap(kf[i] - lit, N)) < 4e-5, (i, kf[i], lit)


def test_pp2_analytic_plus_second_order_term(oracle):
    """R(t + tau) - R(t) = Rdot tau + (|dv|^2 - Rdot^2) tau^2 / (2R) + O(tau^3): pulse-pair equals the analytic
    f_D to O(PRI), and the difference is this closed form."""
    N = 512
    cfg_a, sat = scen(oracle, oracle.DOPPLER_ANALYTIC, N=N)
    cfg_p, _ = scen(oracle, oracle.DOPPLER_PULSE_PAIR, N=N)
    s = scene(4000, 5, spread=3000.0)
    ka = oracle.doppler_coordinate(cfg_a, sat, *s)
    kp = oracle.doppler_coordinate(cfg_p, sat, *s)
    ok = np.isfinite(ka)
    assert ok.sum() > 3000 and np.array_equal(ok, np.isfinite(kp))
    x, y, z, vx, vy, vz = [a.astype(np.float64) for a in s]
    d = np.stack([x, y, z - H])
    dv = np.stack([vx - 7000.0, vy, vz])
    R = np.sqrt((d * d).sum(0))
    rdot = (d * dv).sum(0) / R
    second = -(2.0 * N / LAM) * ((dv * dv).sum(0) - rdot ** 2) / (2.0 * R) / PRF ** 2
    diff = (kp - ka)[ok]
    assert np.abs(diff).max() < 0.01                          # O(PRI): a hundredth of a bin at most here
    assert np.abs(diff).max() > 1e-3                          # ... and not zero: the two estimators differ
    assert np.abs(diff - second[ok]).max() < 5e-5            # closed form (+ the fp64 cancellation noise)


def test_pp3_natural_aliasing_and_bins(oracle):
    """A radial speed beyond lambda PRF / 4 aliases: arg() wraps, the bin is kf mod N in both modes."""
    N = 64
    cfg_p, sat = scen(oracle, oracle.DOPPLER_PULSE_PAIR, N=N)
    for vz, expect in ((0.0, 0), (3.1078125 * 5, 5), (-3.1078125 * 7, N - 7), (3.1078125 * (N + 3), 3),
                       (3.1078125 * 40, 40)):   # bin 40 is the alias of -24: upward = positive Doppler
        a = [np.array([v], np.float32) for v in (0.0, 0.0, 0.0, 7000.0, 0.0, vz)]
        g0, k = oracle.indices(cfg_p, sat, *a)
        assert g0[0] == 32 and k[0] == expect, (vz, k[0], expect)
        lit = literal_kf(N, (0, 0, H), (7000.0, 0, 0), [v[0] for v in a])
        assert int(math.floor(lit + 0.5)) % N == expect


def test_pp4_single_scatterer_cell_and_amplitude_unchanged(oracle):
    """The mode changes the Doppler coordinate only: same gate split, same complex amplitude, other bin."""
    N = 64
    cfg_a, sat = scen(oracle, oracle.DOPPLER_ANALYTIC, N=N)
    cfg_p, _ = scen(oracle, oracle.DOPPLER_PULSE_PAIR, N=N)
    s = [np.array([v], np.float32) for v in (100.0, 30.0, 0.2, 0.5, -0.5, 3.1078125 * 9.5 + 0.004, 10.0)]
    Ta, _ = oracle.spectrum(cfg_a, sat, *s)
    Tp, _ = oracle.spectrum(cfg_p, sat, *s)
    assert (np.abs(Ta) > 0).sum() == 2 and (np.abs(Tp) > 0).sum() == 2
    assert np.allclose(Ta.sum(axis=1), Tp.sum(axis=1), rtol=0, atol=0)     # per-gate sums are identical
    ka = oracle.doppler_coordinate(cfg_a, sat, *s[:6])[0]
    kp = oracle.doppler_coordinate(cfg_p, sat, *s[:6])[0]
    assert np.nonzero(np.abs(Ta).sum(0))[0][0] == int(math.floor(ka + 0.5)) % N
    assert np.nonzero(np.abs(Tp).sum(0))[0][0] == int(math.floor(kp + 0.5)) % N
