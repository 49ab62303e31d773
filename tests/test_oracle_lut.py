"""Pins of the oracle's tabulated antenna gain (oracle_spectrum_lut; "recorded on a u-v grid ...
obtained through interpolation in the u-v grid", reading R9) against things other than itself:
a constant table (= the isotropic spectrum), a table that is linear in u and v (bilinear interpolation
reproduces it exactly: an independent numpy restatement evaluates a + b u + c v at every scatterer), a finely
sampled Gaussian (= the analytic pattern within the interpolation bound), single scatterers at 40 digits with a
random table, the orientation of the frame and the edge rule.  CPU only."""
import math

import mpmath as mp
import numpy as np
import pytest

from tests import brute

LAM, PRF, DR, H = 0.0221, 18000.0, 0.468, 814500.0
ALPHA = 4.0 * math.log(2.0) / math.sin(math.radians(1.35)) ** 2
G, N = 64, 64
RG0 = H - (G // 2) * DR


def scene(n, seed, half=4000.0):
    r = np.random.default_rng(seed)
    x = r.uniform(-half, half, n).astype(np.float32)
    y = r.uniform(-half, half, n).astype(np.float32)
    z = r.normal(0, 0.5, n).astype(np.float32)
    vx, vy = r.normal(0, 1, n).astype(np.float32), r.normal(0, 1, n).astype(np.float32)
    vz = r.normal(0, 0.3, n).astype(np.float32)
    s0 = np.exp(r.normal(math.log(10.0), 0.3, n)).astype(np.float32)
    return x, y, z, vx, vy, vz, s0


def setup(orc, alpha=0.0, pos=(0.0, 0.0, H), vel=(7000.0, 0.0, 0.0), bore=(0.0, 0.0, -1.0)):
    return orc.make_config(G, N, N, LAM, PRF, DR, alpha), orc.make_sat(pos, vel, bore, RG0), pos, vel, bore


def grid(nu, nv, half=0.008):
    du, dv = 2 * half / (nu - 1), 2 * half / (nv - 1)
    return -half, du, -half, dv


def test_constant_table_is_isotropic_times_constant(oracle):
    cfg, sat, *_ = setup(oracle)
    sc = scene(3000, 1)
    u0, du, v0, dv = grid(9, 7)
    g = 0.75 - 0.5j          # exactly representable in complex64
    T = oracle.spectrum_lut(cfg, sat, np.full((7, 9), g, np.complex64), u0, du, v0, dv, *sc)
    T_iso, _ = oracle.spectrum(cfg, sat, *sc)
    assert np.abs(T_iso).max() > 0
    assert np.abs(T - g * T_iso).max() <= 1e-13 * np.abs(T_iso).max()


@pytest.mark.parametrize("bore", [(0.0, 0.0, -1.0), (0.004, -0.003, -1.0)])
def test_table_linear_in_u_and_v_is_reproduced_exactly(oracle, bore):
    # dyadic grid and coefficients: every table value is exact in fp32, so the only difference from the direct
    # evaluation of a + b u + c v is fp64 rounding
    cfg, sat, pos, vel, _ = setup(oracle, bore=bore)
    sc = scene(4000, 2)
    nu, nv, du, dv = 33, 17, 2.0 ** -10, 2.0 ** -9
    u0, v0 = -16 * du, -8 * dv
    a, b, c = 0.5 + 0.25j, 8.0 - 4.0j, -2.0 + 16.0j
    uu, vv = u0 + du * np.arange(nu), v0 + dv * np.arange(nv)
    tab = (a + b * uu[None, :] + c * vv[:, None]).astype(np.complex64)
    assert np.array_equal(tab.astype(np.complex128), a + b * uu[None, :] + c * vv[:, None])
    T = oracle.spectrum_lut(cfg, sat, tab, u0, du, v0, dv, *sc)
    T_ref = brute.numpy_spectrum(*sc, pos, vel, bore, RG0, LAM, PRF, DR, G, N, 0.0, gain_fn=lambda u, v: a + b * u + c * v)[0]
    assert np.abs(T_ref).max() > 0
    assert np.linalg.norm(T - T_ref) <= 1e-7 * np.linalg.norm(T_ref)   # fp64 phase of the oracle: 7.4e7 cycles * 2^-53 (as pin P10)


def test_finely_sampled_gaussian_matches_the_analytic_pattern(oracle):
    # sin^2(theta) = u^2 + v^2 exactly, so G(u, v) = exp(-alpha (u^2 + v^2)) IS the analytic pattern of reading A10;
    # bilinear interpolation error <= (du^2 + dv^2)/8 * max|G''| = (du^2 + dv^2)/8 * 2 alpha, plus fp32 table rounding
    cfg_a, sat, *_ = setup(oracle, alpha=ALPHA)
    cfg_0, *_ = setup(oracle, alpha=0.0)
    sc = scene(5000, 3)
    nu = nv = 513
    u0, du, v0, dv = grid(nu, nv)
    uu, vv = u0 + du * np.arange(nu), v0 + dv * np.arange(nv)
    tab = np.exp(-ALPHA * (uu[None, :] ** 2 + vv[:, None] ** 2)).astype(np.complex64)
    T = oracle.spectrum_lut(cfg_0, sat, tab, u0, du, v0, dv, *sc)
    T_ref, _ = oracle.spectrum(cfg_a, sat, *sc)
    bound = (du * du + dv * dv) / 8 * 2 * ALPHA + 2.0 ** -23
    err = np.linalg.norm(T - T_ref) / np.linalg.norm(T_ref)
    assert err <= 2 * bound, (err, bound)
    # and a coarse grid is visibly worse (the test can fail): 17 nodes
    u0c, duc, v0c, dvc = grid(17, 17)
    uc, vc = u0c + duc * np.arange(17), v0c + dvc * np.arange(17)
    Tc = oracle.spectrum_lut(cfg_0, sat, np.exp(-ALPHA * (uc[None, :] ** 2 + vc[:, None] ** 2)).astype(np.complex64),
                             u0c, duc, v0c, dvc, *sc)
    assert np.linalg.norm(Tc - T_ref) / np.linalg.norm(T_ref) > 50 * err


def test_single_scatterers_against_mpmath_with_a_random_table(oracle):
    pos, vel, bore = (12.5, -3.0, H), (6990.0, 50.0, -2.0), (0.002, 0.001, -1.0)
    cfg, sat, *_ = setup(oracle, pos=pos, vel=vel, bore=bore)
    r = np.random.default_rng(7)
    nu, nv = 11, 13
    u0, du, v0, dv = -0.006, 0.0012, -0.0065, 0.0011
    tab = (r.normal(size=(nv, nu)) + 1j * r.normal(size=(nv, nu))).astype(np.complex64)
    mp.mp.dps = 40
    b = [mp.mpf(c) for c in bore]
    nb = mp.sqrt(sum(c * c for c in b))
    b = [c / nb for c in b]
    vb = sum(mp.mpf(a) * c for a, c in zip(vel, b))
    t = [mp.mpf(a) - vb * c for a, c in zip(vel, b)]
    nt = mp.sqrt(sum(c * c for c in t))
    e1 = [c / nt for c in t]
    e2 = [b[1] * e1[2] - b[2] * e1[1], b[2] * e1[0] - b[0] * e1[2], b[0] * e1[1] - b[1] * e1[0]]
    done = 0
    for trial in range(60):
        s = [float(np.float32(v)) for v in (r.uniform(-4500, 4500), r.uniform(-4500, 4500), r.normal(0, 0.5),
                                            r.normal(), r.normal(), r.normal(0, 0.3), 10.0)]
        ref = brute.closed_form(s, pos, vel, bore, RG0, LAM, PRF, DR, N, 0.0)
        d = [mp.mpf(s[0]) - mp.mpf(pos[0]), mp.mpf(s[1]) - mp.mpf(pos[1]), mp.mpf(s[2]) - mp.mpf(pos[2])]
        u = sum(a * c for a, c in zip(d, e1)) / ref["R"]
        v = sum(a * c for a, c in zip(d, e2)) / ref["R"]
        fu, fv = (u - mp.mpf(u0)) / mp.mpf(du), (v - mp.mpf(v0)) / mp.mpf(dv)
        T = oracle.spectrum_lut(cfg, sat, tab, u0, du, v0, dv, *[np.array([c], np.float32) for c in s])
        if not (0 <= fu <= nu - 1 and 0 <= fv <= nv - 1):
            assert np.abs(T).max() == 0.0
            continue
        i, j = int(mp.floor(fu)), int(mp.floor(fv))
        a_, b_ = fu - i, fv - j
        gm = ((1 - a_) * (1 - b_) * complex(tab[j, i]) + a_ * (1 - b_) * complex(tab[j, i + 1]) +
              (1 - a_) * b_ * complex(tab[j + 1, i]) + a_ * b_ * complex(tab[j + 1, i + 1]))
        if not (-1 <= ref["gf"] < G):
            continue
        want = complex(gm) * ref["c"]
        assert abs(T.sum() - want) <= 1e-7 * abs(want) + 1e-25   # fp64 phase of the oracle: 7.4e7 cycles * 2^-53
        done += 1
    assert done >= 20


def test_frame_orientation_and_edge_rule(oracle):
    cfg, sat, *_ = setup(oracle)
    # u along +velocity (+x); v = (b x e1) = -y for a nadir boresight
    nu = nv = 3
    u0, du, v0, dv = -0.004, 0.004, -0.004, 0.004      # nodes at -0.004, 0, +0.004
    one = lambda s: oracle.spectrum_lut(cfg, sat, tab, u0, du, v0, dv, *[np.array([c], np.float32) for c in s]).sum()
    tab = np.zeros((nv, nu), np.complex64)
    tab[:, 2] = 1.0                                    # non-zero only towards u = +0.004
    ahead, behind = (1600.0, 0, 0, 0, 0, 0, 10.0), (-1600.0, 0, 0, 0, 0, 0, 10.0)
    assert abs(one(ahead)) > 0 and one(behind) == 0
    tab = np.zeros((nv, nu), np.complex64)
    tab[2, :] = 1.0                                    # non-zero only towards v = +0.004, i.e. y < 0
    assert abs(one((0, -1600.0, 0, 0, 0, 0, 10.0))) > 0 and one((0, 1600.0, 0, 0, 0, 0, 10.0)) == 0
    # outside the recorded pattern: nothing; u = 0.0045 > 0.004
    tab = np.ones((nv, nu), np.complex64)
    assert one((3700.0, 0, 0, 0, 0, 0, 10.0)) == 0 and abs(one((3200.0, 0, 0, 0, 0, 0, 10.0))) > 0
    # velocity parallel to the boresight: no along-track axis
    with pytest.raises(RuntimeError):
        oracle.spectrum_lut(cfg, oracle.make_sat((0, 0, H), (0, 0, -7000.0), (0, 0, -1.0), RG0), tab, u0, du, v0, dv,
                            *[np.array([c], np.float32) for c in ahead])
