"""Seeded synthetic workloads (BASELINE.json:configs[0..4]; recipe in DESIGN.md "Input recipe").

This module serves BOTH the CUDA path and the test oracle and therefore holds none of the method's
arithmetic: it only draws scatterer arrays (x, y, z, vx, vy, vz, s0dA as fp32 SoA) and states the
scenario constants (satellite orbit, wavelength, PRF, gate spacing, window origin, beamwidth).
The scenes stand in for the paper's SRAL altimetry scenario; the paper's own sea
states, NRCS look-up tables and antenna patterns are not available.
"""
from __future__ import annotations

import math
from dataclasses import dataclass, replace

import torch

WAVELENGTH_M = 0.0221          # 13.575 GHz Ku band (configs)
PRF_HZ = 18000.0               # PAPER.md:17 (reading A15)
GATE_SPACING_M = 0.468         # c / (2 * 320 MHz)
ALTITUDE_M = 814500.0
SAT_SPEED_MPS = 7000.0
THETA_3DB_DEG = 1.35           # SRAL Ku beamwidth; not in the paper (reading A10)
ANTENNA_ALPHA = 4.0 * math.log(2.0) / math.sin(math.radians(THETA_3DB_DEG)) ** 2
SIGMA_Z_M = 0.5                # 2 m SWH = 4 sigma
GRAVITY = 9.81


@dataclass(frozen=True)
class Workload:
    name: str
    n_along: int               # scatterers along track (x, slowest index)
    n_cross: int               # scatterers cross track (y, fastest index)
    n_gates: int               # G
    n_doppler: int             # N
    pulses_per_update: int     # P = n_fast
    n_updates: int             # U
    seed: int
    sea: str = "white"         # "white": iid normal heights/velocities; "pm": Pierson-Moskowitz field
    spacing_m: float = 1.0
    wavelength_m: float = WAVELENGTH_M
    prf_hz: float = PRF_HZ
    gate_spacing_m: float = GATE_SPACING_M
    antenna_alpha: float = ANTENNA_ALPHA

    @property
    def n_scatterers(self) -> int:
        return self.n_along * self.n_cross

    @property
    def n_pulses(self) -> int:
        return self.n_updates * self.pulses_per_update

    @property
    def range_gate0_m(self) -> float:
        """Window "centred on nadir" (configs): gate G/2 sits at the nadir range (reading A9)."""
        return ALTITUDE_M - (self.n_gates // 2) * self.gate_spacing_m

    def scaled(self, **kw) -> "Workload":
        """Same recipe at another size (parity-test cases)."""
        return replace(self, **kw)


WORKLOADS = {
    # BASELINE.json:configs[0]
    "tiny": Workload("tiny", 256, 256, 64, 64, 64, 2, seed=0),
    # configs[1]
    "nadir_patch_16m": Workload("nadir_patch_16m", 4096, 4096, 128, 256, 256, 8, seed=1),
    # configs[2]
    "sar_footprint_268m": Workload("sar_footprint_268m", 16384, 16384, 128, 512, 512, 4, seed=2,
                                   sea="pm"),
    # configs[4] (64 updates over a 16384 (along) x 4096 (cross) strip)
    "track_segment_67m": Workload("track_segment_67m", 16384, 4096, 128, 256, 256, 64, seed=4),
}
# configs[3]: update-interval sweep on the 16.8M patch, P = N in {16..512}, U = 8 (reading in DESIGN.md)
for _p in (16, 32, 64, 128, 256, 512):
    WORKLOADS[f"sweep_p{_p}"] = Workload(f"sweep_p{_p}", 4096, 4096, 128, _p, _p, 8, seed=3)


def get(name: str) -> Workload:
    return WORKLOADS[name]


def sat_state(wl: Workload, u: int) -> dict:
    """Satellite state at update u (pulse u*P): flat Earth, z up, +x along track (reading A12/A13)."""
    t = u * wl.pulses_per_update / wl.prf_hz - wl.n_updates * wl.pulses_per_update / (2.0 * wl.prf_hz)
    return {
        "pos": (SAT_SPEED_MPS * t, 0.0, ALTITUDE_M),
        "vel": (SAT_SPEED_MPS, 0.0, 0.0),
        "boresight": (0.0, 0.0, -1.0),
        "range_gate0_m": wl.range_gate0_m,
    }


def _positions(wl: Workload, device):
    ia = torch.arange(wl.n_along, dtype=torch.float64, device=device)
    ic = torch.arange(wl.n_cross, dtype=torch.float64, device=device)
    xa = ((ia - (wl.n_along - 1) / 2.0) * wl.spacing_m).to(torch.float32)
    yc = ((ic - (wl.n_cross - 1) / 2.0) * wl.spacing_m).to(torch.float32)
    x = xa[:, None].expand(wl.n_along, wl.n_cross).reshape(-1).contiguous()
    y = yc[None, :].expand(wl.n_along, wl.n_cross).reshape(-1).contiguous()
    return x, y


def _pm_field(wl: Workload, gen: torch.Generator, device):
    """Gaussian random sea surface by 2-D FFT synthesis with a Pierson-Moskowitz-shaped wavenumber
    spectrum Psi(k) ~ k^-4 exp(-(5/4)(k_p/k)^2) cos^2(phi), |phi| < pi/2 (waves travel towards +x),
    k_p = 0.0805 rad/m, rescaled to std(z) = 0.5 m; velocities are the linear deep-water orbital
    velocities of the same Fourier components (omega = sqrt(g k))."""
    na, nc = wl.n_along, wl.n_cross
    n = na * nc
    noise = torch.randn(2 * n, generator=gen, dtype=torch.float32)  # CPU draw: same on any device
    noise = torch.complex(noise[:n], noise[n:]).reshape(na, nc).to(device)
    kx = (2.0 * math.pi * torch.fft.fftfreq(na, d=wl.spacing_m, device=device)).to(torch.float32)
    ky = (2.0 * math.pi * torch.fft.fftfreq(nc, d=wl.spacing_m, device=device)).to(torch.float32)
    KX = kx[:, None]
    KY = ky[None, :]
    k2 = KX * KX + KY * KY
    k2c = torch.where(k2 > 0, k2, torch.ones_like(k2))
    kp = 0.0805
    psi = torch.exp(-1.25 * kp * kp / k2c) / (k2c * k2c) * (KX * KX / k2c)
    psi = torch.where((k2 > 0) & (KX > 0), psi, torch.zeros_like(psi))
    spec = noise * torch.sqrt(psi)
    del noise, psi
    kmag = torch.sqrt(k2c)
    omega = torch.sqrt(GRAVITY * kmag)
    z = torch.fft.ifft2(spec).real.contiguous()
    scale = SIGMA_Z_M / float(z.double().std(unbiased=False))
    z = (z * scale).to(torch.float32).reshape(-1)
    vz = (torch.fft.ifft2(spec * (-1j * omega)).real * scale).to(torch.float32).reshape(-1).contiguous()
    vx = (torch.fft.ifft2(spec * (omega * KX / kmag)).real * scale).to(torch.float32).reshape(-1).contiguous()
    vy = (torch.fft.ifft2(spec * (omega * KY / kmag)).real * scale).to(torch.float32).reshape(-1).contiguous()
    return z, vx, vy, vz


def scatterers(wl: Workload, device="cpu") -> dict:
    """fp32 SoA scatterer arrays, flat index i = ia * n_cross + ic.  Random draws always come from a
    CPU generator (draw order z, vx, vy, vz, ln sigma0) so that any device sees the same scene."""
    device = torch.device(device)
    gen = torch.Generator("cpu").manual_seed(wl.seed)
    n = wl.n_scatterers
    x, y = _positions(wl, device)
    if wl.sea == "pm":
        z, vx, vy, vz = _pm_field(wl, gen, device)
    else:
        z = (torch.randn(n, generator=gen, dtype=torch.float32) * SIGMA_Z_M).to(device)
        vx = torch.randn(n, generator=gen, dtype=torch.float32).to(device)
        vy = torch.randn(n, generator=gen, dtype=torch.float32).to(device)
        vz = (torch.randn(n, generator=gen, dtype=torch.float32) * 0.3).to(device)
    ln_s0 = torch.randn(n, generator=gen, dtype=torch.float32) * 0.3 + math.log(10.0)
    s0dA = (torch.exp(ln_s0) * (wl.spacing_m * wl.spacing_m)).to(torch.float32).to(device)
    return {"x": x, "y": y, "z": z, "vx": vx, "vy": vy, "vz": vz, "s0dA": s0dA}


FIELDS = ("x", "y", "z", "vx", "vy", "vz", "s0dA")
