"""Independent restatements used to PIN the oracle (tests only; imports neither oracle/ nor the CUDA path).

* closed_form():      one scatterer, evaluated with mpmath at 40 digits from the definitions.
* numpy_spectrum():   vectorised numpy/longdouble restatement of step O1 (different code shape).
* regular_mode_sum(): the paper's regular mode -- "summing the complex contributions from all the
                      facets" at every pulse -- for point scatterers in uniform motion.
"""
from __future__ import annotations

import mpmath as mp
import numpy as np

mp.mp.dps = 40


def closed_form(scat, sat_pos, sat_vel, boresight, range_gate0, lam, prf, dR, N, alpha):
    """scat = (x, y, z, vx, vy, vz, s0dA) as Python floats (already fp32-representable)."""
    x, y, z, vx, vy, vz, s0dA = [mp.mpf(float(v)) for v in scat]
    d = [x - mp.mpf(sat_pos[0]), y - mp.mpf(sat_pos[1]), z - mp.mpf(sat_pos[2])]
    dv = [vx - mp.mpf(sat_vel[0]), vy - mp.mpf(sat_vel[1]), vz - mp.mpf(sat_vel[2])]
    R = mp.sqrt(sum(c * c for c in d))
    u = [c / R for c in d]
    fD = -2 * sum(a * b for a, b in zip(dv, u)) / mp.mpf(lam)
    kf = fD * N / mp.mpf(prf)
    gf = (R - mp.mpf(range_gate0)) / mp.mpf(dR)
    q = 2 * R / mp.mpf(lam)
    fr = q - mp.floor(q)
    b = [mp.mpf(c) for c in boresight]
    nb = mp.sqrt(sum(c * c for c in b))
    b = [c / nb for c in b]
    cosang = sum(a * c for a, c in zip(u, b))
    sin2 = 1 - cosang * cosang  # safe at 40 digits
    gain = mp.exp(-mp.mpf(alpha) * sin2)
    A = mp.sqrt(s0dA) * gain / (R * R)
    c = A * mp.exp(-1j * 4 * mp.pi * R / mp.mpf(lam))
    return {"R": R, "gf": gf, "fD": fD, "kf": kf, "fr": fr, "gain": gain, "A": A, "c": complex(c)}


def uv_frame(sat_vel, boresight):
    """Antenna frame of DESIGN.md reading R9, restated: b unit boresight, e1 the unit along-track
    vector normal to b, e2 = b x e1."""
    b = np.asarray(boresight, np.float64)
    b = b / np.linalg.norm(b)
    v = np.asarray(sat_vel, np.float64)
    t = v - np.dot(v, b) * b
    e1 = t / np.linalg.norm(t)
    return b, e1, np.cross(b, e1)


def numpy_spectrum(x, y, z, vx, vy, vz, s0dA, sat_pos, sat_vel, boresight, range_gate0, lam, prf,
                   dR, G, N, alpha, gain_fn=None):
    """[G][N] complex128 spectrum, vectorised; phases reduced in 80-bit long double.
    gain_fn(u, v) -> complex gain replaces the analytic pattern (u, v: direction cosines in uv_frame)."""
    L = np.longdouble
    d = np.stack([np.asarray(x, L) - L(sat_pos[0]), np.asarray(y, L) - L(sat_pos[1]),
                  np.asarray(z, L) - L(sat_pos[2])])
    dv = np.stack([np.asarray(vx, L) - L(sat_vel[0]), np.asarray(vy, L) - L(sat_vel[1]),
                   np.asarray(vz, L) - L(sat_vel[2])])
    R = np.sqrt((d * d).sum(0))
    u = d / R
    fD = -2 * (dv * u).sum(0) / L(lam)
    kf = fD * N / L(prf)
    k = np.mod(np.floor(kf + L(0.5)).astype(np.int64), N)
    gf = (R - L(range_gate0)) / L(dR)
    g0 = np.floor(gf).astype(np.int64)
    w1 = (gf - g0).astype(np.float64)
    w0 = 1.0 - w1
    cycles = 2 * R / L(lam)
    fr = (cycles - np.floor(cycles)).astype(np.float64)
    b = np.asarray(boresight, np.float64)
    b = b / np.linalg.norm(b)
    cr = np.cross(d.astype(np.float64).T, b)
    sin2 = (cr * cr).sum(1) / (R * R).astype(np.float64)
    if gain_fn is None:
        gain = np.exp(-alpha * sin2)
    else:
        _, e1, e2 = uv_frame(sat_vel, boresight)
        d64 = d.astype(np.float64).T
        gain = gain_fn(d64 @ e1 / R.astype(np.float64), d64 @ e2 / R.astype(np.float64))
    A = np.sqrt(np.asarray(s0dA, np.float64)) * gain / (R * R).astype(np.float64)
    A = np.where(np.asarray(s0dA) > 0, A, 0.0)
    c = A * np.exp(-2j * np.pi * fr)
    T = np.zeros((G, N), np.complex128)
    lo = (g0 >= 0) & (g0 < G)
    hi = (g0 + 1 >= 0) & (g0 + 1 < G)
    np.add.at(T, (g0[lo], k[lo]), (w0 * c)[lo])
    np.add.at(T, (g0[hi] + 1, k[hi]), (w1 * c)[hi])
    return T, g0, k, gf.astype(np.float64), kf.astype(np.float64)


def regular_mode_sum(pos0, vel, s0dA, sat_pos0, sat_vel, lam, prf, pulses, alpha=0.0):
    """sum_p a_p(t) exp(-i 4 pi R_p(t) / lambda) at t = pulse/PRF, scatterers and satellite in uniform
    motion from their t = 0 states.  Long double throughout.  pos0, vel: [n][3]."""
    L = np.longdouble
    pos0 = np.asarray(pos0, L)
    vel = np.asarray(vel, L)
    out = np.zeros(len(pulses), np.complex128)
    for j, xp in enumerate(pulses):
        t = L(xp) / L(prf)
        d = pos0 + vel * t - (np.asarray(sat_pos0, L) + np.asarray(sat_vel, L) * t)
        R = np.sqrt((d * d).sum(1))
        cyc = 2 * R / L(lam)
        fr = (cyc - np.floor(cyc)).astype(np.float64)
        a = np.sqrt(np.asarray(s0dA, np.float64)) / (R * R).astype(np.float64)
        assert alpha == 0.0
        out[j] = (a * np.exp(-2j * np.pi * fr)).sum()
    return out
