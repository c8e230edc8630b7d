"""The BASELINE.json configurations as plain data (no arithmetic of the method).

Shapes follow the paper's Table 1 and Table 2 (L430-465);
the concrete numbers are the synthetic stand-ins stated in DESIGN.md ("Input
recipe").  Angles are in arcsec, lengths in metres.
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field
from typing import List, Tuple

BASE_SEED = 180607938
INF = float("inf")


@dataclass(frozen=True)
class WFS:
    ax: float            # direction alpha_j, arcsec
    ay: float
    h_gs: float = INF    # guide-star altitude [m]; inf = NGS (L158)
    n_remove: int = 0    # 0, 2 (tip/tilt) or 3 (tip/tilt/focus) removed (L321-329)


@dataclass(frozen=True)
class TomoConfig:
    name: str
    cfg_id: int
    D: float                      # pupil diameter [m]
    n: int                        # subapertures across (d = D/n)
    wfs: Tuple[WFS, ...]          # high-order WFSs (the CG system)
    targets: Tuple[Tuple[float, float], ...]   # beta_i, arcsec
    h: Tuple[float, ...]          # layer altitudes h_k [m]
    frac: Tuple[float, ...]       # Cn2 fractions, sum to 1
    r0: float = 0.15              # Fried parameter at 500 nm [m]
    L0: float = 25.0              # outer scale [m]
    noise_frac: float = 0.05      # sigma^2 as a fraction of the model slope variance
    n_iter: int = 50
    pad: int = 0                  # FFT edge for C_ss (0 = next 5-smooth even >= 2n-1)
    pad_os: int = 0               # FFT edge for C_os (0 = next 5-smooth even >= n'+n-1)
    lo_wfs: Tuple[WFS, ...] = field(default_factory=tuple)  # low-order NGS (geometry only)
    obstruction: float = 0.0
    screen_npx: int = 2048

    @property
    def d(self) -> float:
        return self.D / self.n

    @property
    def n_wfs(self) -> int:
        return len(self.wfs)

    @property
    def n_layers(self) -> int:
        return len(self.h)


def ring(n_gs: int, radius_arcsec: float, h_gs: float, n_remove: int,
         phase_deg: float = 0.0) -> Tuple[WFS, ...]:
    out = []
    for i in range(n_gs):
        a = 2.0 * math.pi * i / n_gs + math.radians(phase_deg)
        out.append(WFS(radius_arcsec * math.cos(a), radius_arcsec * math.sin(a), h_gs, n_remove))
    return tuple(out)


def _exp_profile(n_layers: int, h_max: float, scale: float):
    h = [k * h_max / (n_layers - 1) for k in range(n_layers)]
    w = [math.exp(-hk / scale) for hk in h]
    s = sum(w)
    return tuple(h), tuple(x / s for x in w)


def _cfg1() -> TomoConfig:
    return TomoConfig(
        name="cfg1_tiny_ngs", cfg_id=1, D=4.0, n=8,
        wfs=(WFS(10.0, 0.0), WFS(-10.0, 0.0)),
        targets=((0.0, 0.0),), h=(0.0, 5000.0), frac=(0.7, 0.3),
        noise_frac=0.01, n_iter=20, pad=16, pad_os=16, screen_npx=1024)


def _cfg2() -> TomoConfig:
    h, f = _exp_profile(7, 16000.0, 4000.0)
    return TomoConfig(
        name="cfg2_mid_ltao", cfg_id=2, D=8.0, n=20,
        wfs=ring(4, 30.0, 90e3, 2), targets=((0.0, 0.0),), h=h, frac=f,
        noise_frac=0.05, n_iter=30, pad=40, pad_os=48, screen_npx=1024)


def _cfg3() -> TomoConfig:
    h, f = _exp_profile(35, 25000.0, 5000.0)
    return TomoConfig(
        name="cfg3_elt_ltao", cfg_id=3, D=38.0, n=74,
        wfs=ring(6, 45.0, 90e3, 2), targets=((0.0, 0.0),), h=h, frac=f,
        noise_frac=0.05, n_iter=50, pad=160, pad_os=180)


def _cfg4() -> TomoConfig:
    h, f = _exp_profile(35, 25000.0, 5000.0)
    tg = []
    for t in range(10):
        rad = 110.0 * math.sqrt((t + 0.5) / 10.0)
        tg.append((rad * math.cos(2.39996 * t), rad * math.sin(2.39996 * t)))
    lo = tuple(WFS(90.0 * math.cos(math.radians(a)), 90.0 * math.sin(math.radians(a)))
               for a in (90.0, 210.0, 330.0))
    return TomoConfig(
        name="cfg4_elt_moao", cfg_id=4, D=38.0, n=74,
        wfs=ring(8, 120.0, 90e3, 2), targets=tuple(tg), h=h, frac=f,
        noise_frac=0.05, n_iter=50, pad=160, pad_os=180, lo_wfs=lo)


def sweep_config(n: int) -> TomoConfig:
    """cfg5: complexity sweep, 6 LGS at 90 km, 35 layers, d = 0.5 m."""
    h, f = _exp_profile(35, 25000.0, 5000.0)
    return TomoConfig(
        name=f"cfg5_sweep_n{n}", cfg_id=5, D=n / 2.0, n=n,
        wfs=ring(6, 45.0, 90e3, 2), targets=((0.0, 0.0),), h=h, frac=f,
        noise_frac=0.05, n_iter=50, pad=0, pad_os=0)


SWEEP_N = (16, 32, 64, 96, 128)
CONFIG_NAMES = ("cfg1", "cfg2", "cfg3", "cfg4")


def get_config(name: str) -> TomoConfig:
    table = {"cfg1": _cfg1, "cfg2": _cfg2, "cfg3": _cfg3, "cfg4": _cfg4}
    if name in table:
        return table[name]()
    if name.startswith("cfg5_n"):
        return sweep_config(int(name[len("cfg5_n"):]))
    raise KeyError(name)


def small_lgs_config(n: int = 10, n_gs: int = 3, n_layers: int = 3, n_remove: int = 2,
                     targets=((0.0, 0.0),), D: float = 4.0, radius: float = 30.0,
                     h_max: float = 12000.0, n_iter: int = 20) -> TomoConfig:
    """A reduced LGS case (same structure as cfg2) the dense oracle builds in seconds."""
    h, f = _exp_profile(n_layers, h_max, 4000.0) if n_layers > 1 else ((0.0,), (1.0,))
    return TomoConfig(
        name=f"small_lgs_n{n}_g{n_gs}_k{n_layers}", cfg_id=9, D=D, n=n,
        wfs=ring(n_gs, radius, 90e3, n_remove), targets=tuple(targets), h=h, frac=f,
        noise_frac=0.05, n_iter=n_iter, pad=0, pad_os=0, screen_npx=512)
