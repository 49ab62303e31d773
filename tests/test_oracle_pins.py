"""Pins of the fp64 oracle against things OTHER than itself (SURVEY.md section 8(c) pins P1-P10):
closed forms at 40 digits, the printed worked values, numpy.fft as a library special case, Parseval,
a brute-force regular-mode coherent sum, linearity, the weights of eq. (1) and an independent
numpy/long-double restatement.  CPU only."""
import math
import os

import numpy as np
import pytest

from tests import brute

LAM, PRF, DR, H = 0.0221, 18000.0, 0.468, 814500.0
ALPHA = 4.0 * math.log(2.0) / math.sin(math.radians(1.35)) ** 2
SAT_POS, SAT_VEL, BORE = (0.0, 0.0, H), (7000.0, 0.0, 0.0), (0.0, 0.0, -1.0)


def scen(orc, G=64, N=64, P=64, lam=LAM, alpha=ALPHA, mode=0, sat_pos=SAT_POS, sat_vel=SAT_VEL,
         bore=BORE, rg0=None):
    rg0 = H - (G // 2) * DR if rg0 is None else rg0
    return (orc.make_config(G, N, P, lam, PRF, DR, alpha, mode),
            orc.make_sat(sat_pos, sat_vel, bore, rg0), rg0)


def one(orc, cfg, sat, s):
    a = [np.array([v], np.float32) for v in s]
    T, _ = orc.spectrum(cfg, sat, *a)
    return T


def golden_rows():
    path = os.path.join(os.path.dirname(__file__), "golden", "worked_values.txt")
    rows = []
    for line in open(path):
        line = line.split("#")[0].strip()
        if line:
            rows.append([float(v) for v in line.split()])
    return rows


def test_alpha_constant():
    assert abs(ALPHA - 4995.09267381) < 1e-7


# ---- P1: closed form, single scatterer (invariant (a): a delta in one (gate, bin)) -------------
def test_p1_worked_values_golden(oracle):
    cfg, sat, rg0 = scen(oracle)
    for row in golden_rows():
        x, y, z, vx, vy, vz, R, gf, fD, kf, fr, gain, amp = row
        T = one(oracle, cfg, sat, (x, y, z, vx, vy, vz, 10.0))
        g0, k = int(math.floor(gf)), int(math.floor(kf + 0.5)) % 64
        # range_gate0 = 814485.024 is not a binary fraction: gf = 32 comes out as 32 +- 1e-11, so a
        # weight ~1e-11 may leak into the neighbouring gate; count cells above 1e-6 of the peak.
        nz = np.argwhere(np.abs(T) > 1e-6 * np.abs(T).max())
        w1 = gf - g0
        expect_cells = {(g0, k)} | ({(g0 + 1, k)} if w1 > 1e-9 else set())
        assert {tuple(int(v) for v in c) for c in nz} == expect_cells
        c = T.sum()
        assert abs(abs(c) - amp) / amp < 2e-9
        phase_cyc = (-np.angle(c) / (2 * np.pi)) % 1.0
        # the table assumes exact decimal inputs; fp32(-0.7) is off by 1.2e-8 m = 1.1e-6 cycles
        assert abs((phase_cyc - fr + 0.5) % 1.0 - 0.5) < 3e-6
        assert abs(abs(T[g0, k]) / abs(c) - (1 - w1)) < 1e-7
        if w1 > 1e-9:
            assert abs(abs(T[g0 + 1, k]) / abs(c) - w1) < 1e-7


def test_p1_row1_single_cell_value(oracle):
    cfg, sat, _ = scen(oracle)
    T = one(oracle, cfg, sat, (0, 0, 0, 0, 0, 0, 10.0))
    assert np.count_nonzero(np.abs(T) > 1e-6 * np.abs(T).max()) == 1
    assert np.count_nonzero(T[:, 1:]) == 0 and np.count_nonzero(T[:31]) == 0 and np.count_nonzero(T[34:]) == 0
    expect = 4.766700032e-12 * np.exp(-2j * np.pi * 0.2398190)
    assert abs(T[32, 0] - expect) / abs(expect) < 1e-6


def test_p1_row2_half_split(oracle):
    cfg, sat, _ = scen(oracle)
    T = one(oracle, cfg, sat, (0, 0, 0.234, 0, 0, 0, 10.0))
    assert np.count_nonzero(T) == 2
    assert abs(abs(T[31, 0]) / abs(T[32, 0]) - 1.0) < 1e-6   # z = fp32(0.234): w1 = 0.5 + 5.6e-9


def test_p1_closed_form_mpmath_random(oracle):
    """Every term of O1 against a 40-digit evaluation of the definitions, off-nadir boresight too."""
    rng = np.random.default_rng(11)
    for trial in range(60):
        bore = BORE if trial % 2 == 0 else (0.003, -0.002, -1.0)
        N = [64, 256, 512][trial % 3]
        cfg, sat, rg0 = scen(oracle, G=64, N=N, P=N, bore=bore)
        s = np.array([rng.uniform(-4000, 4000), rng.uniform(-4000, 4000), rng.normal(0, 0.5),
                      rng.normal(0, 1), rng.normal(0, 1), rng.normal(0, 3),
                      math.exp(rng.normal(math.log(10), 0.3))], np.float32)
        cf = brute.closed_form(s, SAT_POS, SAT_VEL, bore, rg0, LAM, PRF, DR, N, ALPHA)
        gf, kf = float(cf["gf"]), float(cf["kf"])
        if not (0.0 <= gf < 63.0) or abs(gf - round(gf)) < 1e-6 or abs(kf + 0.5 - round(kf + 0.5)) < 1e-6:
            continue
        T = one(oracle, cfg, sat, s)
        g0, k = math.floor(gf), math.floor(kf + 0.5) % N
        w1 = gf - g0
        c = cf["c"]
        # phase is limited by fp64 q = 2R/lambda ~ 7.4e7 cycles: ~1e-8 cycles
        assert abs(T[g0, k] - (1 - w1) * c) <= 2e-7 * abs(c)
        assert abs(T[g0 + 1, k] - w1 * c) <= 2e-7 * abs(c)
        assert abs(abs(T.sum()) - float(cf["A"])) <= 1e-12 * float(cf["A"])
        assert np.count_nonzero(T) == 2


def test_p1_indices_match_closed_form(oracle):
    rng = np.random.default_rng(5)
    n = 300
    cfg, sat, rg0 = scen(oracle, G=128, N=256, P=256)
    a = [rng.uniform(-6000, 6000, n), rng.uniform(-6000, 6000, n), rng.normal(0, 0.5, n),
         rng.normal(0, 1, n), rng.normal(0, 1, n), rng.normal(0, 0.3, n)]
    a = [v.astype(np.float32) for v in a]
    g0, k = oracle.indices(cfg, sat, *a)
    for p in range(n):
        cf = brute.closed_form([v[p] for v in a] + [1.0], SAT_POS, SAT_VEL, BORE, rg0, LAM, PRF, DR,
                               256, ALPHA)
        gf, kf = float(cf["gf"]), float(cf["kf"])
        if abs(gf - round(gf)) < 1e-6 or abs(kf + 0.5 - round(kf + 0.5)) < 1e-6:
            continue
        if -1.0 <= gf < 128:
            assert g0[p] == math.floor(gf) and k[p] == math.floor(kf + 0.5) % 256
        else:
            assert g0[p] == oracle.GATE_NONE and k[p] == -1


def test_dropped_scatterers(oracle):
    cfg, sat, _ = scen(oracle)
    # s0dA <= 0, out of window (too far / too near), NaN position: nothing accumulates
    for s in [(0, 0, 0, 0, 0, 0, 0.0), (0, 0, 0, 0, 0, 0, -1.0), (0, 0, -40.0, 0, 0, 0, 10.0),
              (0, 0, 16.0, 0, 0, 0, 10.0), (float("nan"), 0, 0, 0, 0, 0, 10.0),
              (0, 0, 0, float("inf"), 0, 0, 10.0), (0, 0, 0, 0, 0, 0, float("nan"))]:
        assert np.count_nonzero(one(oracle, cfg, sat, s)) == 0
    # half-in: gf in [-1, 0) -> only the upper half lands in gate 0; gf in [G-1, G) -> only lower half
    T = one(oracle, cfg, sat, (0, 0, 32 * DR + 0.25 * DR, 0, 0, 0, 10.0))   # gf = -0.25
    assert np.count_nonzero(T) == 1 and abs(T[0, 0]) > 0
    T = one(oracle, cfg, sat, (0, 0, -31.25 * DR, 0, 0, 0, 10.0))           # gf = 63.25
    assert np.count_nonzero(T) == 1 and abs(T[63, 0]) > 0


def test_negative_doppler_wraps(oracle):
    cfg, sat, _ = scen(oracle)
    vz = -3 * LAM * PRF / (2 * 64)            # bin -3 -> 61
    T = one(oracle, cfg, sat, (0, 0, -0.234, 0, 0, vz, 10.0))   # gf = 32.5: gates 32 and 33
    assert np.argwhere(np.abs(T) > 0).tolist() == [[32, 61], [33, 61]]
    vz = (64 + 5) * LAM * PRF / (2 * 64)      # aliased: bin 69 -> 5
    T = one(oracle, cfg, sat, (0, 0, -0.234, 0, 0, vz, 10.0))
    assert np.argwhere(np.abs(T) > 0).tolist() == [[32, 5], [33, 5]]


# ---- P2: pure tone after synthesis (invariant (a)) -----------------------------------------------
@pytest.mark.parametrize("k", [0, 1, 7, 33, 63])
def test_p2_pure_tone(oracle, k):
    cfg, sat, _ = scen(oracle)
    kk = k if k < 32 else k - 64
    vz = kk * LAM * PRF / (2 * 64)
    T = one(oracle, cfg, sat, (0, 0, -0.234, 0, 0, vz, 10.0))   # gf = 32.5: gates 32 and 33
    assert np.argwhere(np.abs(T) > 0).tolist() == [[32, k], [33, k]]
    y = oracle.idft(T)
    m = np.arange(64)
    for g in (32, 33):
        c = T[g, k]
        assert np.allclose(y[g], c * np.exp(2j * np.pi * k * m / 64), rtol=0, atol=1e-13 * abs(c))
    assert np.count_nonzero(np.abs(y[(np.arange(64) != 32) & (np.arange(64) != 33)])) == 0


# ---- P3 / P4: library special case and Parseval (invariant (d)) ----------------------------------
@pytest.mark.parametrize("N", [16, 64, 512, 12, 1, 250, 750, 1250])   # (the paper's n_fast values: any N)
def test_p3_idft_is_N_times_numpy_ifft(oracle, N):
    rng = np.random.default_rng(N)
    T = rng.normal(size=(5, N)) + 1j * rng.normal(size=(5, N))
    y = oracle.idft(T)
    ref = N * np.fft.ifft(T, axis=-1)
    assert np.abs(y - ref).max() <= 1e-12 * np.abs(ref).max()


def test_p4_parseval(oracle):
    rng = np.random.default_rng(3)
    T = rng.normal(size=(7, 128)) + 1j * rng.normal(size=(7, 128))
    y = oracle.idft(T)
    assert np.allclose((np.abs(y) ** 2).sum(1), 128 * (np.abs(T) ** 2).sum(1), rtol=1e-12)


# ---- P6: weights of eq. (1) (invariant (e), reading A1) ------------------------------------------
@pytest.mark.parametrize("P", [1, 12, 16, 256])
def test_p6_weights(oracle, P):
    for m in range(P + 1):
        ws, wn = oracle.weight(0, P, m), oracle.weight(0, P, P - m)
        assert abs(ws * ws + wn * wn - 1.0) < 1e-15          # paper: variance conserved
        assert abs(ws - math.sqrt(1 - m / P)) < 1e-15         # eq. (1)
        ls, ln = oracle.weight(1, P, m), oracle.weight(1, P, P - m)
        assert abs(ls + ln - 1.0) < 1e-15                     # partition of unity
    assert oracle.weight(0, P, 0) == 1.0 and oracle.weight(0, P, P) == 0.0


# ---- P5: brute-force regular mode on tiny inputs (invariant (b)) ---------------------------------
@pytest.mark.parametrize("N,P", [(16, 16), (32, 16), (16, 12)])
@pytest.mark.parametrize("mode", [0, 1])
def test_p5_fast_mode_equals_regular_mode_for_on_bin_scatterers(oracle, N, P, mode):
    """Scatterers in the nadir column co-moving with the satellite along x and moving vertically at an
    on-bin velocity: R(t) is exactly linear, so the fast mode must reproduce the per-pulse coherent sum
     -- times (sqrt(1-a)+sqrt(a)) with the paper's weights (reading A1).  lambda = 2^-6 m
    and dyadic z make every fp32 input and every phase exact, so the tolerance is tight."""
    lam = 2.0 ** -6
    V = 6750.0                      # V P / PRF is dyadic: satellite and scatterer x stay exact in fp32
    rng = np.random.default_rng(100 * N + P)
    n, U, G = 40, 4, 64
    kbin = rng.integers(-N // 2, N // 2, n)
    vzs = kbin * lam * PRF / (2 * N)
    z0 = rng.integers(-4096, 4096, n) * 2.0 ** -12
    s0 = rng.uniform(5, 20, n).astype(np.float32)
    cfg, _, rg0 = scen(oracle, G=G, N=N, P=P, lam=lam, alpha=0.0, mode=mode)
    T_all = np.zeros((U + 1, G, N), np.complex128)
    for u in range(U + 1):
        t = u * P / PRF
        sat = oracle.make_sat((V * t, 0.0, H), (V, 0.0, 0.0), BORE, rg0)
        zu = z0 + vzs * t
        assert np.array_equal(zu.astype(np.float32).astype(np.float64), zu)      # exact in fp32
        xs = np.full(n, np.float32(V * t))
        assert float(xs[0]) == V * t
        T_all[u], _ = oracle.spectrum(cfg, sat, xs, np.zeros(n), zu, np.full(n, V), np.zeros(n),
                                      vzs, s0)
        assert np.array_equal(vzs.astype(np.float32).astype(np.float64), vzs)
    Y = oracle.synthesize(cfg, T_all, 0, U * P, final=False)
    fast = Y.sum(axis=1)                                                         # gate sum removes the split
    pos0 = np.stack([np.zeros(n), np.zeros(n), z0], 1)
    vel = np.stack([np.full(n, V), np.zeros(n), vzs], 1)
    direct = brute.regular_mode_sum(pos0, vel, s0, SAT_POS, (V, 0.0, 0.0), lam, PRF, range(U * P))
    a = (np.arange(U * P) % P) / P
    gain = np.sqrt(1 - a) + np.sqrt(a) if mode == 0 else np.ones_like(a)
    assert np.abs(fast - gain * direct).max() <= 2e-6 * np.abs(direct).max()
    assert np.abs(direct).max() > 0


# ---- P7: update-pulse identity (reading A2) -----------------------------------------------------
def test_p7_update_pulse_is_coherent_sum(oracle):
    rng = np.random.default_rng(8)
    G, N, P, U = 8, 32, 32, 3
    cfg, _, _ = scen(oracle, G=G, N=N, P=P)
    T_all = rng.normal(size=(U, G, N)) + 1j * rng.normal(size=(U, G, N))
    Y = oracle.synthesize(cfg, T_all, 0, U * P, final=True)
    for u in range(U):
        assert np.allclose(Y[u * P], T_all[u].sum(axis=1), rtol=1e-12, atol=1e-12)


def test_synthesize_tail_and_not_ready(oracle):
    rng = np.random.default_rng(9)
    G, N, P = 4, 16, 16
    cfg, _, _ = scen(oracle, G=G, N=N, P=P)
    T_all = rng.normal(size=(2, G, N)) + 1j * rng.normal(size=(2, G, N))
    with pytest.raises(LookupError):
        oracle.synthesize(cfg, T_all, 0, 2 * P, final=False)
    Y = oracle.synthesize(cfg, T_all, 0, 2 * P, final=True)
    y1 = N * np.fft.ifft(T_all[1], axis=-1)
    assert np.allclose(Y[P:], y1.T, rtol=1e-12, atol=1e-12)        # tail: lone spectrum at weight 1
    # arbitrary start / length gives the same samples as the full stream
    Yp = oracle.synthesize(cfg, T_all, 5, 20, final=True)
    assert np.array_equal(Yp, Y[5:25])


@pytest.mark.parametrize("N,P", [(16, 16), (32, 16), (16, 12), (64, 100), (250, 250), (500, 250)])
def test_o3_definition_against_numpy(oracle, N, P):
    """O3 written a second time with numpy.fft and explicit eq. (1) weights (periodic extension, A4)."""
    rng = np.random.default_rng(N + P)
    G, U = 3, 4
    for mode in (0, 1):
        cfg, _, _ = scen(oracle, G=G, N=N, P=P, mode=mode)
        T_all = rng.normal(size=(U, G, N)) + 1j * rng.normal(size=(U, G, N))
        ysig = N * np.fft.ifft(T_all, axis=-1)
        Y = oracle.synthesize(cfg, T_all, 0, (U - 1) * P, final=False)
        for x in range((U - 1) * P):
            acc = np.zeros(G, complex)
            for u in range(U):
                d = abs(u * P - x)
                if d < P:
                    w = (1 - d / P) ** (0.5 if mode == 0 else 1.0)
                    acc += w * ysig[u][:, (x - u * P) % N]
            assert np.allclose(Y[x], acc, rtol=1e-12, atol=1e-12)


# ---- P8: linearity in scatterer sets (invariant (c)) --------------------------------------------
def _random_scene(rng, n, half=3000.0):
    return [rng.uniform(-half, half, n).astype(np.float32), rng.uniform(-half, half, n).astype(np.float32),
            rng.normal(0, 0.5, n).astype(np.float32), rng.normal(0, 1, n).astype(np.float32),
            rng.normal(0, 1, n).astype(np.float32), rng.normal(0, 0.3, n).astype(np.float32),
            np.exp(rng.normal(math.log(10), 0.3, n)).astype(np.float32)]


def test_p8_linearity_and_accumulate_flag(oracle):
    rng = np.random.default_rng(21)
    cfg, sat, _ = scen(oracle, G=128, N=256, P=256)
    a = _random_scene(rng, 5000)
    T, _ = oracle.spectrum(cfg, sat, *a)
    TA, _ = oracle.spectrum(cfg, sat, *[v[:2000] for v in a])
    TB, _ = oracle.spectrum(cfg, sat, *[v[2000:] for v in a])
    scale = np.abs(T).max()
    assert np.abs(T - (TA + TB)).max() <= 1e-12 * scale
    Tacc, _ = oracle.spectrum(cfg, sat, *[v[2000:] for v in a], out=TA.copy(), accumulate=True)
    assert np.abs(T - Tacc).max() <= 1e-12 * scale
    Tmt, used = oracle.spectrum(cfg, sat, *a, nthreads=4)
    assert used == 4 and np.abs(T - Tmt).max() <= 1e-12 * scale


# ---- P9: variance conservation -- why eq. (1) has the 1/2 power -------------------
def test_p9_variance_conservation(oracle):
    rng = np.random.default_rng(31)
    G, N, P = 256, 64, 64
    T_all = (rng.normal(size=(2, G, N)) + 1j * rng.normal(size=(2, G, N))) / math.sqrt(2)
    prof = {}
    for mode in (0, 1):
        cfg, _, _ = scen(oracle, G=G, N=N, P=P, mode=mode)
        Y = oracle.synthesize(cfg, T_all, 0, P, final=False)
        prof[mode] = (np.abs(Y) ** 2).mean(axis=1) / N
    assert np.all(np.abs(prof[0] - 1.0) < 0.2)                    # flat (independent spectra)
    mid = prof[1][P // 2 - 4:P // 2 + 4].mean()
    assert 0.4 < mid < 0.6                                        # linear weights lose half the power
    assert abs(prof[0][P // 2 - 4:P // 2 + 4].mean() - 1.0) < 0.1


# ---- P10: independent numpy / long-double restatement -------------------------------------------
@pytest.mark.parametrize("bore", [BORE, (0.004, 0.001, -1.0)])
def test_p10_numpy_restatement(oracle, bore):
    rng = np.random.default_rng(41)
    G, N = 128, 512
    cfg, sat, rg0 = scen(oracle, G=G, N=N, P=N, bore=bore)
    a = _random_scene(rng, 1000, half=7000.0)
    a[6][::17] = 0.0                                              # some dead scatterers
    T, _ = oracle.spectrum(cfg, sat, *a)
    Tn, g0n, kn, gf, kf = brute.numpy_spectrum(*a, SAT_POS, SAT_VEL, bore, rg0, LAM, PRF, DR, G, N, ALPHA)
    assert np.abs(T - Tn).max() <= 1e-7 * np.abs(Tn).max()        # fp64 phase: 7.4e7 cycles * 2^-53
    g0, k = oracle.indices(cfg, sat, *a[:6])
    safe = (np.abs(gf - np.round(gf)) > 1e-6) & (np.abs(kf + 0.5 - np.round(kf + 0.5)) > 1e-6)
    inwin = (gf >= -1) & (gf < G)
    assert np.array_equal(g0[safe & inwin], g0n[safe & inwin])
    assert np.array_equal(k[safe & inwin], kn[safe & inwin])
    assert np.all(g0[~inwin] == oracle.GATE_NONE)
    assert inwin.sum() > 300 and (~inwin).sum() > 100


def test_fp64_phase_accuracy_vs_mpmath(oracle):
    """q = 2R/lambda ~ 7.4e7 cycles: the fp64 oracle holds the phase to ~1e-8 cycles."""
    cfg, sat, rg0 = scen(oracle)
    worst = 0.0
    rng = np.random.default_rng(51)
    for _ in range(40):
        s = np.array([rng.uniform(-2000, 2000), rng.uniform(-2000, 2000), rng.normal(0, 0.5), 0, 0, 0, 10.0],
                     np.float32)
        cf = brute.closed_form(s, SAT_POS, SAT_VEL, BORE, rg0, LAM, PRF, DR, 64, ALPHA)
        c = one(oracle, cfg, sat, s).sum()
        worst = max(worst, abs(np.angle(c * np.conj(cf["c"]))))
    assert worst < 2e-7
