"""ctypes binding of oracle/oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this module.  It holds no arithmetic of the method: it compiles oracle.c with gcc and
marshals numpy arrays.  It imports nothing from paper_2408_11472_b200.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "oracle.c")
_LIB = os.path.join(_HERE, "liboracle.so")

W_SQRT = 0
W_LINEAR = 1
DOPPLER_ANALYTIC = 0
DOPPLER_PULSE_PAIR = 1
GATE_NONE = -(2**31)


class OracleConfig(C.Structure):
    _fields_ = [
        ("n_gates", C.c_int32),
        ("n_doppler", C.c_int32),
        ("pulses_per_update", C.c_int32),
        ("weight_mode", C.c_int32),
        ("wavelength_m", C.c_double),
        ("prf_hz", C.c_double),
        ("gate_spacing_m", C.c_double),
        ("antenna_alpha", C.c_double),
        ("doppler_mode", C.c_int32),
    ]


class OracleSat(C.Structure):
    _fields_ = [
        ("pos", C.c_double * 3),
        ("vel", C.c_double * 3),
        ("boresight", C.c_double * 3),
        ("range_gate0_m", C.c_double),
    ]


class OracleLut(C.Structure):
    _fields_ = [
        ("table", C.POINTER(C.c_float)),
        ("nu", C.c_int32),
        ("nv", C.c_int32),
        ("u0", C.c_double),
        ("du", C.c_double),
        ("v0", C.c_double),
        ("dv", C.c_double),
    ]


def build(force: bool = False) -> str:
    """Compile oracle.c -> liboracle.so (gcc, -ffp-contract=off, OpenMP)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        cmd = ["gcc", "-std=c11", "-O2", "-ffp-contract=off", "-fopenmp", "-shared", "-fPIC",
               _SRC, "-o", _LIB, "-lm"]
        subprocess.run(cmd, check=True)
    return _LIB


_lib = None


def lib():
    global _lib
    if _lib is None:
        build()
        L = C.CDLL(_LIB)
        fp = C.POINTER(C.c_float)
        dp = C.POINTER(C.c_double)
        ip = C.POINTER(C.c_int32)
        L.oracle_spectrum.argtypes = [C.POINTER(OracleConfig), C.POINTER(OracleSat), C.c_int64,
                                      fp, fp, fp, fp, fp, fp, fp, dp, C.c_int, C.c_int]
        L.oracle_spectrum.restype = C.c_int
        L.oracle_spectrum_lut.argtypes = [C.POINTER(OracleConfig), C.POINTER(OracleSat), C.POINTER(OracleLut), C.c_int64,
                                          fp, fp, fp, fp, fp, fp, fp, dp, C.c_int, C.c_int]
        L.oracle_spectrum_lut.restype = C.c_int
        L.oracle_indices.argtypes = [C.POINTER(OracleConfig), C.POINTER(OracleSat), C.c_int64,
                                     fp, fp, fp, fp, fp, fp, ip, ip]
        L.oracle_indices.restype = C.c_int
        L.oracle_doppler_coordinate.argtypes = [C.POINTER(OracleConfig), C.POINTER(OracleSat), C.c_int64,
                                                fp, fp, fp, fp, fp, fp, dp]
        L.oracle_doppler_coordinate.restype = C.c_int
        L.oracle_regular.argtypes = [C.POINTER(OracleConfig), C.POINTER(OracleSat), C.c_int64,
                                     fp, fp, fp, fp, fp, fp, fp, C.c_int64, C.c_int64, dp, C.c_int, C.c_int]
        L.oracle_regular.restype = C.c_int
        L.oracle_burst_dft.argtypes = [C.c_int32, C.c_int32, C.c_int64, dp, dp]
        L.oracle_burst_dft.restype = C.c_int
        L.oracle_idft.argtypes = [C.c_int32, C.c_int32, dp, dp]
        L.oracle_idft.restype = C.c_int
        L.oracle_weight.argtypes = [C.c_int32, C.c_int32, C.c_int64]
        L.oracle_weight.restype = C.c_double
        L.oracle_synthesize.argtypes = [C.POINTER(OracleConfig), C.c_int32, dp, C.c_int64,
                                        C.c_int64, C.c_int, dp]
        L.oracle_synthesize.restype = C.c_int
        L.oracle_max_threads.restype = C.c_int
        _lib = L
    return _lib


def make_config(n_gates, n_doppler, pulses_per_update, wavelength_m, prf_hz, gate_spacing_m,
                antenna_alpha, weight_mode=W_SQRT, doppler_mode=DOPPLER_ANALYTIC) -> OracleConfig:
    return OracleConfig(int(n_gates), int(n_doppler), int(pulses_per_update), int(weight_mode),
                        float(wavelength_m), float(prf_hz), float(gate_spacing_m),
                        float(antenna_alpha), int(doppler_mode))


def make_sat(pos, vel, boresight, range_gate0_m) -> OracleSat:
    s = OracleSat()
    for i in range(3):
        s.pos[i] = float(pos[i])
        s.vel[i] = float(vel[i])
        s.boresight[i] = float(boresight[i])
    s.range_gate0_m = float(range_gate0_m)
    return s


def _f32(a):
    a = np.ascontiguousarray(a, dtype=np.float32)
    return a, a.ctypes.data_as(C.POINTER(C.c_float))


def max_threads() -> int:
    return int(lib().oracle_max_threads())


def spectrum(cfg: OracleConfig, sat: OracleSat, x, y, z, vx, vy, vz, s0dA, out=None,
             accumulate=False, nthreads=1):
    """O1: one update's [G][N] complex128 spectrum.  Returns (T, threads_used)."""
    arrs = [_f32(a) for a in (x, y, z, vx, vy, vz, s0dA)]
    n = arrs[0][0].size
    assert all(a[0].size == n for a in arrs)
    if out is None:
        out = np.zeros((cfg.n_gates, cfg.n_doppler), dtype=np.complex128)
    assert out.dtype == np.complex128 and out.flags.c_contiguous
    rc = lib().oracle_spectrum(C.byref(cfg), C.byref(sat), n, *[a[1] for a in arrs],
                               out.ctypes.data_as(C.POINTER(C.c_double)), int(accumulate),
                               int(nthreads))
    if rc < 0:
        raise RuntimeError(f"oracle_spectrum failed: {rc}")
    return out, rc


def spectrum_lut(cfg: OracleConfig, sat: OracleSat, table, u0, du, v0, dv, x, y, z, vx, vy, vz, s0dA, nthreads=1):
    """O1 with the antenna gain interpolated in a complex u-v table [nv][nu] (reading R9)."""
    tab = np.ascontiguousarray(table, dtype=np.complex64)
    assert tab.ndim == 2
    lut = OracleLut(tab.view(np.float32).ctypes.data_as(C.POINTER(C.c_float)), tab.shape[1], tab.shape[0],
                    float(u0), float(du), float(v0), float(dv))
    arrs = [_f32(a) for a in (x, y, z, vx, vy, vz, s0dA)]
    n = arrs[0][0].size
    out = np.zeros((cfg.n_gates, cfg.n_doppler), dtype=np.complex128)
    rc = lib().oracle_spectrum_lut(C.byref(cfg), C.byref(sat), C.byref(lut), n, *[a[1] for a in arrs],
                                   out.ctypes.data_as(C.POINTER(C.c_double)), 0, int(nthreads))
    if rc < 0:
        raise RuntimeError(f"oracle_spectrum_lut failed: {rc}")
    return out


def indices(cfg: OracleConfig, sat: OracleSat, x, y, z, vx, vy, vz):
    """Canonical (g0, k) per scatterer; dropped scatterers: (GATE_NONE, -1)."""
    arrs = [_f32(a) for a in (x, y, z, vx, vy, vz)]
    n = arrs[0][0].size
    g0 = np.empty(n, dtype=np.int32)
    k = np.empty(n, dtype=np.int32)
    rc = lib().oracle_indices(C.byref(cfg), C.byref(sat), n, *[a[1] for a in arrs],
                              g0.ctypes.data_as(C.POINTER(C.c_int32)),
                              k.ctypes.data_as(C.POINTER(C.c_int32)))
    if rc < 0:
        raise RuntimeError(f"oracle_indices failed: {rc}")
    return g0, k


def doppler_coordinate(cfg: OracleConfig, sat: OracleSat, x, y, z, vx, vy, vz):
    """kf = f_D N / PRF per scatterer before rounding to a bin (NaN when dropped)."""
    arrs = [_f32(a) for a in (x, y, z, vx, vy, vz)]
    n = arrs[0][0].size
    kf = np.empty(n, dtype=np.float64)
    rc = lib().oracle_doppler_coordinate(C.byref(cfg), C.byref(sat), n, *[a[1] for a in arrs],
                                         kf.ctypes.data_as(C.POINTER(C.c_double)))
    if rc < 0:
        raise RuntimeError(f"oracle_doppler_coordinate failed: {rc}")
    return kf


def regular(cfg: OracleConfig, sat: OracleSat, x, y, z, vx, vy, vz, s0dA, j0, n_pulses, nthreads=1):
    """Regular mode: [n_pulses][G] complex128 for pulses j0..j0+n_pulses-1 relative to the instant of `sat`."""
    arrs = [_f32(a) for a in (x, y, z, vx, vy, vz, s0dA)]
    n = arrs[0][0].size
    Y = np.zeros((int(n_pulses), cfg.n_gates), dtype=np.complex128)
    rc = lib().oracle_regular(C.byref(cfg), C.byref(sat), n, *[a[1] for a in arrs], int(j0), int(n_pulses),
                              Y.ctypes.data_as(C.POINTER(C.c_double)), 0, int(nthreads))
    if rc < 0:
        raise RuntimeError(f"oracle_regular failed: {rc}")
    return Y


def burst_dft(Y, burst):
    """Delay-Doppler burst step: forward DFT along the pulses of each burst.  Y [n_pulses][G] -> [n_bursts][burst][G]."""
    Y = np.ascontiguousarray(Y, dtype=np.complex128)
    n, G = Y.shape
    assert n % burst == 0
    Z = np.empty((n // burst, burst, G), dtype=np.complex128)
    rc = lib().oracle_burst_dft(G, int(burst), n // burst, Y.ctypes.data_as(C.POINTER(C.c_double)),
                                Z.ctypes.data_as(C.POINTER(C.c_double)))
    if rc < 0:
        raise RuntimeError(f"oracle_burst_dft failed: {rc}")
    return Z


def idft(T):
    """O2: unnormalised inverse DFT along the last axis of a [G][N] complex128 array."""
    T = np.ascontiguousarray(T, dtype=np.complex128)
    G, N = T.shape
    y = np.empty_like(T)
    rc = lib().oracle_idft(G, N, T.ctypes.data_as(C.POINTER(C.c_double)),
                           y.ctypes.data_as(C.POINTER(C.c_double)))
    if rc < 0:
        raise RuntimeError(f"oracle_idft failed: {rc}")
    return y


def weight(weight_mode, P, d) -> float:
    return float(lib().oracle_weight(int(weight_mode), int(P), int(d)))


def synthesize(cfg: OracleConfig, T_all, x0, n_pulses, final=False):
    """O3: blended IQ [n_pulses][G] complex128 for pulses x0..x0+n_pulses-1."""
    T_all = np.ascontiguousarray(T_all, dtype=np.complex128)
    U, G, N = T_all.shape
    assert G == cfg.n_gates and N == cfg.n_doppler
    Y = np.empty((n_pulses, G), dtype=np.complex128)
    rc = lib().oracle_synthesize(C.byref(cfg), U, T_all.ctypes.data_as(C.POINTER(C.c_double)),
                                 int(x0), int(n_pulses), int(final),
                                 Y.ctypes.data_as(C.POINTER(C.c_double)))
    if rc == -3:
        raise LookupError("oracle_synthesize: a needed spectrum is missing (not ready)")
    if rc < 0:
        raise RuntimeError(f"oracle_synthesize failed: {rc}")
    return Y
