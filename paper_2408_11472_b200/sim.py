"""Thin ctypes binding of libsim.so (include/sim.h).  Argument marshalling only: every step of the
path runs in the CUDA kernels under csrc/.  PyTorch is used for device memory and streams.

There is no CPU fallback: if csrc/libsim.so is missing and cannot be built, or the device is not
CUDA, every entry point raises.
"""
from __future__ import annotations

import ctypes as C
import os

import torch

from . import build as _build

OK = 0
ERR_INVALID_ARG, ERR_BAD_CONFIG, ERR_WORKSPACE, ERR_NOT_READY, ERR_OVERFLOW, ERR_CUDA = -1, -2, -3, -4, -5, -6
W_SQRT, W_LINEAR = 0, 1
ACC_APPEND = 1
DOPPLER_ANALYTIC, DOPPLER_PULSE_PAIR = 0, 1
SYN_FINAL = 1
GATE_NONE = -(2**31)
OPT_ACC_VARIANT, OPT_ACC_BLOCKS, OPT_ACC_SUPERCHUNK, OPT_ACC_WINDOW_BINS, OPT_GUARD_LSB, OPT_INDEX_PATH = 1, 2, 3, 4, 5, 6
OPT_ACC_WARPS = 9
OPT_ACC_PER_LANE, OPT_ACC_EPOCH, OPT_ACC_SCATTER, OPT_ACC_INTERLEAVE, OPT_ACC_SHAPE = 11, 12, 14, 15, 16

EXPORTS = [
    "sim_workspace_bytes", "sim_create", "sim_accumulate_update", "sim_synthesize_pulses",
    "sim_accumulate_update_host", "sim_synthesize_pulses_host", "sim_synchronize", "sim_destroy",
    "sim_get_spectrum", "sim_spectrum_offset", "sim_debug_indices", "sim_set_option", "sim_get_stats",
    "sim_read_counters", "sim_last_error", "sim_regular_pulses", "sim_burst_beams", "sim_set_antenna_lut",
    "sim_accumulate_static",
]
STATIC_MAX_CELLS = 65536


class SimError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"libsim error {code}: {msg}")
        self.code = code


class SimConfig(C.Structure):
    _fields_ = [
        ("struct_size", C.c_uint32), ("n_gates", C.c_int32), ("n_doppler", C.c_int32),
        ("pulses_per_update", C.c_int32), ("max_pending_updates", C.c_int32), ("weight_mode", C.c_int32),
        ("device", C.c_int32), ("doppler_mode", C.c_int32), ("wavelength_m", C.c_double), ("prf_hz", C.c_double),
        ("gate_spacing_m", C.c_double), ("antenna_alpha", C.c_double),
        ("host_stage_scatterers", C.c_int64), ("host_stage_pulses", C.c_int64),
    ]


class SimScatterers(C.Structure):
    _fields_ = [(n, C.c_void_p) for n in ("x", "y", "z", "vx", "vy", "vz", "s0dA")] + [("n", C.c_uint64)]


class SimSatState(C.Structure):
    _fields_ = [("pos", C.c_double * 3), ("vel", C.c_double * 3), ("boresight", C.c_double * 3),
                ("range_gate0_m", C.c_double)]


class SimStats(C.Structure):
    _fields_ = [("kernel_launches", C.c_uint64), ("updates_accumulated", C.c_uint64),
                ("scatterers_seen", C.c_uint64), ("pulses_emitted", C.c_int64)]


_lib = None


def load_library(build_if_missing: bool = True):
    """dlopen csrc/libsim.so (building it in-tree first if needed).  Raises if that is impossible."""
    global _lib
    if _lib is not None:
        return _lib
    path = _build.LIB
    if build_if_missing:
        path = _build.build_lib()
    if not os.path.exists(path):
        raise RuntimeError(f"{path} is missing: build it with `python -m paper_2408_11472_b200.build`; "
                           "there is no CPU fallback")
    L = C.CDLL(path)
    vp, hp = C.c_void_p, C.c_void_p
    L.sim_workspace_bytes.argtypes = [C.POINTER(SimConfig), C.POINTER(C.c_size_t)]
    L.sim_create.argtypes = [C.POINTER(SimConfig), vp, C.c_size_t, vp, C.POINTER(hp)]
    L.sim_accumulate_update.argtypes = [hp, C.POINTER(SimScatterers), C.POINTER(SimSatState), C.c_uint32]
    L.sim_accumulate_update_host.argtypes = L.sim_accumulate_update.argtypes
    L.sim_synthesize_pulses.argtypes = [hp, C.c_int64, vp, C.c_uint32]
    L.sim_synthesize_pulses_host.argtypes = L.sim_synthesize_pulses.argtypes
    L.sim_synchronize.argtypes = [hp]
    L.sim_destroy.argtypes = [hp]
    L.sim_get_spectrum.argtypes = [hp, C.c_int64, vp]
    L.sim_spectrum_offset.argtypes = [hp, C.c_int64, C.POINTER(C.c_size_t)]
    L.sim_debug_indices.argtypes = [hp, C.POINTER(SimScatterers), C.POINTER(SimSatState), vp, vp]
    L.sim_set_option.argtypes = [hp, C.c_int32, C.c_int64]
    L.sim_set_antenna_lut.argtypes = [hp, vp, C.c_int32, C.c_int32, C.c_double, C.c_double, C.c_double, C.c_double]
    L.sim_get_stats.argtypes = [hp, C.POINTER(SimStats)]
    L.sim_read_counters.argtypes = [hp, C.POINTER(C.c_uint32), C.c_int32]
    L.sim_accumulate_static.argtypes = [C.POINTER(SimConfig), C.POINTER(SimScatterers), C.POINTER(SimSatState), vp, vp,
                                        C.c_uint32]
    L.sim_last_error.argtypes = [hp]
    L.sim_last_error.restype = C.c_char_p
    for name in EXPORTS:
        if name != "sim_last_error":
            getattr(L, name).restype = C.c_int
    _lib = L
    return L


def make_config(n_gates, n_doppler, pulses_per_update, wavelength_m, prf_hz, gate_spacing_m,
                antenna_alpha, max_pending_updates=4, weight_mode=W_SQRT, device=0,
                host_stage_scatterers=0, host_stage_pulses=0, doppler_mode=DOPPLER_ANALYTIC) -> SimConfig:
    return SimConfig(C.sizeof(SimConfig), int(n_gates), int(n_doppler), int(pulses_per_update),
                     int(max_pending_updates), int(weight_mode), int(device), int(doppler_mode), float(wavelength_m),
                     float(prf_hz), float(gate_spacing_m), float(antenna_alpha),
                     int(host_stage_scatterers), int(host_stage_pulses))


def make_sat(pos, vel, boresight, range_gate0_m) -> SimSatState:
    s = SimSatState()
    for i in range(3):
        s.pos[i], s.vel[i], s.boresight[i] = float(pos[i]), float(vel[i]), float(boresight[i])
    s.range_gate0_m = float(range_gate0_m)
    return s


def _scat_struct(arrs, cuda: bool) -> SimScatterers:
    names = ("x", "y", "z", "vx", "vy", "vz", "s0dA")
    ts = [arrs[n] for n in names]
    n = ts[0].numel()
    for t in ts:
        if t.dtype != torch.float32 or not t.is_contiguous() or t.numel() != n or t.is_cuda != cuda:
            raise ValueError("scatterer arrays must be contiguous float32 tensors of equal length on the "
                             + ("CUDA device" if cuda else "host"))
    s = SimScatterers()
    for name, t in zip(names, ts):
        setattr(s, name, t.data_ptr() if n else None)
    s.n = n
    return s


class Sim:
    """One simulation stream: sim_create / sim_accumulate_update / sim_synthesize_pulses / sim_destroy."""

    def __init__(self, cfg: SimConfig, stream: "torch.cuda.Stream | None" = None):
        if not torch.cuda.is_available():
            raise RuntimeError("paper_2408_11472_b200.sim needs a CUDA device (B200); there is no CPU fallback")
        self.lib = load_library()
        self.cfg = cfg
        self.device = torch.device("cuda", cfg.device)
        nbytes = C.c_size_t()
        self._check(self.lib.sim_workspace_bytes(C.byref(cfg), C.byref(nbytes)), None)
        with torch.cuda.device(self.device):
            self.workspace = torch.empty(max(nbytes.value, 256), dtype=torch.uint8, device=self.device)
            self.stream = stream if stream is not None else torch.cuda.current_stream(self.device)
        assert self.workspace.data_ptr() % 256 == 0
        h = C.c_void_p()
        self._h = None
        self._check(self.lib.sim_create(C.byref(cfg), self.workspace.data_ptr(), self.workspace.numel(),
                                        self.stream.cuda_stream, C.byref(h)), None)
        self._h = h

    # -- helpers ---------------------------------------------------------------------------------
    def _check(self, rc, h):
        if rc != OK:
            msg = self.lib.sim_last_error(h)
            raise SimError(rc, msg.decode() if msg else "")

    def close(self):
        if getattr(self, "_h", None) is not None:
            self.lib.sim_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # -- the four calls of the path ----------------------------------------------------------------
    def accumulate_update(self, scat: dict, sat: SimSatState, flags: int = 0):
        s = _scat_struct(scat, cuda=True)
        self._check(self.lib.sim_accumulate_update(self._h, C.byref(s), C.byref(sat), flags), self._h)

    def synthesize_pulses(self, n_pulses: int, out: "torch.Tensor | None" = None, flags: int = 0):
        G = self.cfg.n_gates
        if out is None:
            out = torch.empty((n_pulses, G), dtype=torch.complex64, device=self.device)
        if out.dtype != torch.complex64 or not out.is_contiguous() or out.numel() < n_pulses * G or not out.is_cuda:
            raise ValueError("out must be a contiguous CUDA complex64 tensor of at least n_pulses*G elements")
        self._check(self.lib.sim_synthesize_pulses(self._h, n_pulses, out.data_ptr(), flags), self._h)
        return out

    def regular_pulses(self, scat: dict, sat: SimSatState, first_pulse: int, n_pulses: int,
                       out: "torch.Tensor | None" = None, flags: int = 0):
        """Regular mode (sim_regular_pulses): [n_pulses][G] complex64 for pulses first_pulse.. relative to `sat`."""
        G = self.cfg.n_gates
        if out is None:
            out = torch.empty((n_pulses, G), dtype=torch.complex64, device=self.device)
        if out.dtype != torch.complex64 or not out.is_contiguous() or out.numel() < n_pulses * G or not out.is_cuda:
            raise ValueError("out must be a contiguous CUDA complex64 tensor of at least n_pulses*G elements")
        s = _scat_struct(scat, cuda=True)
        self._check(self.lib.sim_regular_pulses(self._h, C.byref(s), C.byref(sat), C.c_int64(first_pulse),
                                                C.c_int64(n_pulses), C.c_void_p(out.data_ptr()), C.c_uint32(flags)),
                    self._h)
        return out

    def burst_beams(self, iq: torch.Tensor, burst: int = 64):
        """Delay-Doppler burst step (sim_burst_beams): [n_pulses][G] -> [n_pulses / burst][burst][G] complex64."""
        G = self.cfg.n_gates
        if iq.dtype != torch.complex64 or not iq.is_contiguous() or not iq.is_cuda or iq.shape[-1] != G:
            raise ValueError("iq must be a contiguous CUDA complex64 tensor [n_pulses][G]")
        n = iq.shape[0]
        out = torch.empty((n // max(burst, 1), burst, G), dtype=torch.complex64, device=self.device)
        self._check(self.lib.sim_burst_beams(self._h, C.c_void_p(iq.data_ptr()), C.c_int64(n), C.c_int32(burst),
                                             C.c_void_p(out.data_ptr()), C.c_uint32(0)), self._h)
        return out

    def accumulate_update_host(self, scat: dict, sat: SimSatState, flags: int = 0):
        s = _scat_struct(scat, cuda=False)
        self._check(self.lib.sim_accumulate_update_host(self._h, C.byref(s), C.byref(sat), flags), self._h)

    def synthesize_pulses_host(self, n_pulses: int, out: torch.Tensor, flags: int = 0):
        G = self.cfg.n_gates
        if out.dtype != torch.complex64 or not out.is_contiguous() or out.numel() < n_pulses * G or out.is_cuda:
            raise ValueError("out must be a contiguous host complex64 tensor of at least n_pulses*G elements")
        self._check(self.lib.sim_synthesize_pulses_host(self._h, n_pulses, out.data_ptr(), flags), self._h)
        return out

    def synchronize(self):
        self._check(self.lib.sim_synchronize(self._h), self._h)

    # -- parity / debug ----------------------------------------------------------------------------
    def get_spectrum(self, update_index: int) -> torch.Tensor:
        out = torch.empty((self.cfg.n_gates, self.cfg.n_doppler), dtype=torch.complex64, device=self.device)
        self._check(self.lib.sim_get_spectrum(self._h, update_index, out.data_ptr()), self._h)
        return out

    def spectrum_view(self, update_index: int) -> torch.Tensor:
        """In-place float32 view [G][N][2] of a spectrum inside the workspace (multi-GPU all-reduce)."""
        off = C.c_size_t()
        self._check(self.lib.sim_spectrum_offset(self._h, update_index, C.byref(off)), self._h)
        nb = self.cfg.n_gates * self.cfg.n_doppler * 8
        return self.workspace[off.value:off.value + nb].view(torch.float32).view(self.cfg.n_gates, self.cfg.n_doppler, 2)

    def debug_indices(self, scat: dict, sat: SimSatState):
        s = _scat_struct({**scat, "s0dA": scat.get("s0dA", scat["x"])}, cuda=True)
        n = int(s.n)
        g0 = torch.empty(n, dtype=torch.int32, device=self.device)
        k = torch.empty(n, dtype=torch.int32, device=self.device)
        self._check(self.lib.sim_debug_indices(self._h, C.byref(s), C.byref(sat), g0.data_ptr() if n else None,
                                               k.data_ptr() if n else None), self._h)
        return g0, k

    def set_antenna_lut(self, table: "torch.Tensor | None", u0: float = 0.0, du: float = 1.0, v0: float = 0.0,
                        dv: float = 1.0):
        """table: complex64 CUDA tensor [n_v][n_u] (kept alive here while it is set), or None for the analytic gain."""
        if table is None:
            self._lut = None
            self._check(self.lib.sim_set_antenna_lut(self._h, None, 0, 0, 0.0, 1.0, 0.0, 1.0), self._h)
            return
        assert table.is_cuda and table.dtype == torch.complex64 and table.dim() == 2 and table.is_contiguous()
        self._lut = table
        self._check(self.lib.sim_set_antenna_lut(self._h, table.data_ptr(), table.shape[1], table.shape[0], float(u0),
                                                 float(du), float(v0), float(dv)), self._h)

    def set_option(self, option: int, value: int):
        self._check(self.lib.sim_set_option(self._h, option, value), self._h)

    def stats(self) -> dict:
        st = SimStats()
        self._check(self.lib.sim_get_stats(self._h, C.byref(st)), self._h)
        return {f: int(getattr(st, f)) for f, _ in SimStats._fields_}

    def read_counters(self, reset: bool = False) -> dict:
        a = (C.c_uint32 * 4)()
        self._check(self.lib.sim_read_counters(self._h, a, int(reset)), self._h)
        return {"escapes": a[1], "index_fallbacks": a[3]}      # [0], [2]: the kernel's own scheduling words, 0 between launches


def accumulate_static(cfg: SimConfig, scat: dict, sat: SimSatState, out: "torch.Tensor | None" = None,
                      stream: "torch.cuda.Stream | None" = None, flags: int = 0) -> torch.Tensor:
    """sim_accumulate_static: the spectrum [G][N] of one update, for callers that cannot provide a device workspace
    (no handle; the kernel's scratch memory is an array built into libsim.so, G * N <= STATIC_MAX_CELLS).  `out` is
    the caller's complex64 CUDA buffer; only when none is given does this wrapper ask torch for one, which a caller
    that cannot allocate would not do.  Calls that overlap on the GPU share the scratch array and race."""
    if not torch.cuda.is_available():
        raise RuntimeError("paper_2408_11472_b200.sim needs a CUDA device (B200); there is no CPU fallback")
    lib = load_library()
    device = torch.device("cuda", cfg.device)
    if out is None:
        out = torch.empty((cfg.n_gates, cfg.n_doppler), dtype=torch.complex64, device=device)
    if out.dtype != torch.complex64 or not out.is_contiguous() or not out.is_cuda or out.numel() < cfg.n_gates * cfg.n_doppler:
        raise ValueError("out must be a contiguous CUDA complex64 tensor of at least G*N elements")
    s = _scat_struct(scat, cuda=True)
    st = stream if stream is not None else torch.cuda.current_stream(device)
    rc = lib.sim_accumulate_static(C.byref(cfg), C.byref(s), C.byref(sat), C.c_void_p(out.data_ptr()),
                                   C.c_void_p(st.cuda_stream), C.c_uint32(flags))
    if rc != OK:
        msg = lib.sim_last_error(None)
        raise SimError(rc, msg.decode() if msg else "")
    return out


def config_for(wl, **kw) -> SimConfig:
    """SimConfig of a workloads.Workload."""
    return make_config(wl.n_gates, wl.n_doppler, wl.pulses_per_update, wl.wavelength_m, wl.prf_hz,
                       wl.gate_spacing_m, wl.antenna_alpha, **kw)


def sat_for(wl, u: int) -> SimSatState:
    from . import workloads
    s = workloads.sat_state(wl, u)
    return make_sat(s["pos"], s["vel"], s["boresight"], s["range_gate0_m"])
