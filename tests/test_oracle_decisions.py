"""Pins of the three integer DECISIONS of the oracle's geometry() with literal expected values (CPU only):
where a Doppler coordinate exactly half-way between two bins goes (reading A7: up), where a range exactly on a gate
boundary goes (reading A8: to the upper gate with weight 1, nothing to the lower one), and which edge of the gate
window and of the Doppler range is inside (readings A8, A3: gf = -1 in, gf = G out, |kf| = 2^30 out).

The scenes are built from powers of two so that every intermediate of the canonical sequence is exact in fp64 and
the coordinate lands ON the tie / boundary / edge with no rounding at all (asserted first, through
oracle.doppler_coordinate and the weights).  With the configs' lambda = 0.0221 m and PRF = 18 kHz that never
happens: c_D = -2N / (lambda PRF) is not dyadic.  The expected bins and gates are written out as numbers: a rint()
(ties to even), a round() (ties away from zero), a `<=` for the `<` of the window, or a ceil()-based gate would each
fail at least one line.  Ref: PAPER.md:53 ("range gate and Doppler interval"), :94 (rasterize); A3/A7/A8.
"""
import numpy as np
import pytest

LAM = 2.0 ** -6          # wavelength, m
PRF = 2.0 ** 14          # Hz
N = 64                   # c_D = -2 N / (LAM PRF) = -1/2 exactly;  c_P = -2 N / LAM = -8192 exactly
G = 16
DR = 0.5                 # gate spacing, m: 1 / DR = 2 exactly
H = 814500.0             # satellite altitude: H^2 < 2^53, so R = sqrt(H^2) = H exactly
SAT_VEL = (7000.0, 0.0, 0.0)
BORE = (0.0, 0.0, -1.0)


def _scene(orc, mode, rg0):
    cfg = orc.make_config(G, N, N, LAM, PRF, DR, 0.0, 0, mode)
    sat = orc.make_sat((0.0, 0.0, H), SAT_VEL, BORE, rg0)
    return cfg, sat


def _arr(v):
    return np.array([v], np.float32)


def _nadir(z=0.0, vz=0.0):
    """A scatterer straight below the satellite, moving with it horizontally: d = (0, 0, z - H), dv = (0, 0, vz)."""
    return _arr(0.0), _arr(0.0), _arr(z), _arr(SAT_VEL[0]), _arr(SAT_VEL[1]), _arr(vz)


# j -> bin of kf = j + 1/2 with ties UP: floor(j + 1).  rint gives 0, 2, 4, -2, -2, 32; round() gives 1, 3, 4, -2, -3, 32.
TIES = [(0, 1), (2, 3), (3, 4), (-2, N - 1), (-3, N - 2), (N // 2 - 1, N // 2)]


@pytest.mark.parametrize("mode", [0, 1], ids=["analytic", "pulse_pair"])
@pytest.mark.parametrize("j,expected_bin", TIES)
def test_doppler_tie_goes_up(oracle, mode, j, expected_bin):
    # analytic:   rdot = dv.d / R = vz (z - H) / (H - z) = -vz,  kf = rdot c_D = vz / 2
    # pulse pair: R' = H - vz / PRF (sqrt(x^2) = |x| in binary fp),  kf = (R' - R) c_P = vz 8192 / 16384 = vz / 2
    cfg, sat = _scene(oracle, mode, rg0=H - 4.0)
    s = _nadir(vz=float(2 * j + 1))
    kf = oracle.doppler_coordinate(cfg, sat, *s)
    assert kf[0] == j + 0.5                      # exactly on the tie, no rounding anywhere
    g0, k = oracle.indices(cfg, sat, *s)
    assert int(g0[0]) == 8                       # gf = (H - (H - 4)) * 2 = 8 exactly
    assert int(k[0]) == expected_bin
    T, _ = oracle.spectrum(cfg, sat, *s, _arr(1.0))
    nz = {tuple(int(v) for v in c) for c in np.argwhere(T != 0)}
    assert nz == {(8, expected_bin)}


@pytest.mark.parametrize("m", [0, 1, 5, G - 1])
def test_gate_boundary_goes_to_the_upper_gate(oracle, m):
    # R - rg0 = m dR exactly: gf = m, g0 = m with w0 = 1, w1 = 0: ONE non-zero cell, in gate m (not split, not m - 1)
    cfg, sat = _scene(oracle, 0, rg0=H)
    s = _nadir(z=-0.5 * m, vz=3.0)               # kf = 1.5 -> bin 2 (tie, up)
    g0, k = oracle.indices(cfg, sat, *s)
    assert (int(g0[0]), int(k[0])) == (m, 2)
    T, _ = oracle.spectrum(cfg, sat, *s, _arr(1.0))
    nz = {tuple(int(v) for v in c) for c in np.argwhere(T != 0)}
    assert nz == {(m, 2)}
    # the whole amplitude is there: |c| = sqrt(s0dA) / R^2 with the isotropic antenna of this scene
    R = H + 0.5 * m
    assert abs(T[m, 2]) == pytest.approx(1.0 / (R * R), rel=1e-14)


def test_gate_quarter_way_is_split_three_to_one(oracle):
    # the complement of the boundary case: gf = m + 1/4 exactly -> 3/4 in gate m, 1/4 in gate m + 1
    cfg, sat = _scene(oracle, 0, rg0=H)
    s = _nadir(z=-(0.5 * 5 + 0.125), vz=3.0)
    g0, k = oracle.indices(cfg, sat, *s)
    assert (int(g0[0]), int(k[0])) == (5, 2)
    T, _ = oracle.spectrum(cfg, sat, *s, _arr(1.0))
    assert {tuple(int(v) for v in c) for c in np.argwhere(T != 0)} == {(5, 2), (6, 2)}
    assert abs(T[5, 2]) / abs(T[6, 2]) == pytest.approx(3.0, rel=1e-14)


def test_window_edges(oracle):
    cfg, sat = _scene(oracle, 0, rg0=H)
    GATE_NONE = oracle.GATE_NONE
    # gf = -1 exactly: still inside (g0 = -1), its whole weight belongs to gate -1, so gate 0 receives exactly nothing
    s = _nadir(z=+0.5, vz=3.0)
    g0, k = oracle.indices(cfg, sat, *s)
    assert (int(g0[0]), int(k[0])) == (-1, 2)
    T, _ = oracle.spectrum(cfg, sat, *s, _arr(1.0))
    assert not np.any(T != 0)
    # one fp32 step above gf = -1 (z = 0.5 - 2^-25 is a float32; R, gf exact in fp64): a sliver in gate 0
    s = _nadir(z=0.5 - 2.0 ** -25, vz=3.0)
    g0, k = oracle.indices(cfg, sat, *s)
    assert int(g0[0]) == -1
    T, _ = oracle.spectrum(cfg, sat, *s, _arr(1.0))
    assert {tuple(int(v) for v in c) for c in np.argwhere(T != 0)} == {(0, 2)}
    assert abs(T[0, 2]) == pytest.approx(2.0 ** -24 / (H - 0.5) ** 2, rel=1e-6)
    # just below -1: dropped
    g0, k = oracle.indices(cfg, sat, *_nadir(z=0.5 + 2.0 ** -24, vz=3.0))
    assert (int(g0[0]), int(k[0])) == (GATE_NONE, -1)
    # gf = G exactly: outside (neither gate G nor G + 1 exists)
    g0, k = oracle.indices(cfg, sat, *_nadir(z=-0.5 * G, vz=3.0))
    assert (int(g0[0]), int(k[0])) == (GATE_NONE, -1)
    T, _ = oracle.spectrum(cfg, sat, *_nadir(z=-0.5 * G, vz=3.0), _arr(1.0))
    assert not np.any(T != 0)
    # one fp32 step inside: the last gate, nearly all of the weight lost beyond the window
    s = _nadir(z=-0.5 * G + 2.0 ** -21, vz=3.0)
    g0, k = oracle.indices(cfg, sat, *s)
    assert (int(g0[0]), int(k[0])) == (G - 1, 2)
    T, _ = oracle.spectrum(cfg, sat, *s, _arr(1.0))
    assert {tuple(int(v) for v in c) for c in np.argwhere(T != 0)} == {(G - 1, 2)}


@pytest.mark.parametrize("mode", [0, 1], ids=["analytic", "pulse_pair"])
def test_doppler_range_edge(oracle, mode):
    cfg, sat = _scene(oracle, mode, rg0=H - 4.0)
    # kf = vz / 2: vz = +-2^31 gives |kf| = 2^30 exactly: dropped; the next float32 below, 2^31 - 128, is kept
    for vz in (2.0 ** 31, -(2.0 ** 31)):
        s = _nadir(vz=vz)
        kf = oracle.doppler_coordinate(cfg, sat, *s)
        g0, k = oracle.indices(cfg, sat, *s)
        assert (int(g0[0]), int(k[0])) == (oracle.GATE_NONE, -1)
        assert np.isnan(kf[0])
    s = _nadir(vz=2.0 ** 31 - 128.0)
    assert oracle.doppler_coordinate(cfg, sat, *s)[0] == 2.0 ** 30 - 64.0
    g0, k = oracle.indices(cfg, sat, *s)
    assert (int(g0[0]), int(k[0])) == (8, 0)             # (2^30 - 64) mod 64 = 0
    s = _nadir(vz=-(2.0 ** 31 - 128.0))
    assert oracle.doppler_coordinate(cfg, sat, *s)[0] == -(2.0 ** 30) + 64.0
    g0, k = oracle.indices(cfg, sat, *s)
    assert (int(g0[0]), int(k[0])) == (8, 0)
