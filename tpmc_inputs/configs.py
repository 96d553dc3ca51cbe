"""Run parameters of the five BASELINE.json configs (plain records, no arithmetic of the method).

Readings of the config text:
n = 1e15 m^-3 where not given (cancels in coefficients); config 3 uses config 1's gas;
N is per run (one V, one attitude); the attitude/pitch sweeps rotate V, not the mesh.
"""
from __future__ import annotations

from dataclasses import dataclass, field, replace
from typing import Callable, List, Tuple

import numpy as np

from . import meshes

K_B = 1.380649e-23          # J/K (exact, SI 2019)
AMU = 1.66053906660e-27     # kg


@dataclass
class RunConfig:
    name: str
    mesh_fn: Callable[[], meshes.Mesh]
    n: float = 1.0e15                      # number density, 1/m^3
    T_inf: float = 1000.0                  # K
    T_W: float = 300.0                     # K
    V: Tuple[float, float, float] = (-7500.0, 0.0, 0.0)   # bulk velocity, body frame, m/s
    accommodation: float = 1.0             # sigma: P(diffuse); 1-sigma specular
    m: Tuple[float, ...] = (16.0 * AMU,)   # species masses, kg
    x: Tuple[float, ...] = (1.0,)          # species number fractions
    cv_radius_factor: float = 1.5
    N: int = 100_000
    seed: int = 0
    max_bounces: int = 1024
    x_ref: Tuple[float, float, float] = (0.0, 0.0, 0.0)
    energy_accommodation: float = 1.0      # alpha_E: 1 = re-emission at T_W (the paper's case)
    control_volume: int = 0                # 0 sphere (the paper's scheme), 1 box, 2 box with unweighted inward speed
    A_ref: float = 1.0                     # m^2, for coefficients only
    label: str = ""
    _mesh_cache: list = field(default_factory=list, repr=False, compare=False)

    def mesh(self) -> meshes.Mesh:
        if not self._mesh_cache:
            self._mesh_cache.append(self.mesh_fn())
        return self._mesh_cache[0]

    def with_(self, **kw) -> "RunConfig":
        c = replace(self, **kw)
        c._mesh_cache = self._mesh_cache   # share the generated mesh
        return c

    @property
    def speed(self) -> float:
        return float(np.linalg.norm(self.V))

    @property
    def rho(self) -> float:
        return self.n * float(np.dot(self.x, self.m))

    @property
    def q_inf(self) -> float:
        return 0.5 * self.rho * self.speed ** 2


def fibonacci_directions(k: int) -> np.ndarray:
    """k quasi-uniform unit vectors (attitude sweep directions)."""
    i = np.arange(k) + 0.5
    z = 1.0 - 2.0 * i / k
    r = np.sqrt(np.maximum(0.0, 1.0 - z * z))
    ph = i * np.pi * (3.0 - np.sqrt(5.0))
    return np.stack([r * np.cos(ph), r * np.sin(ph), z], 1)


def _t_inf_for_speed_ratio(S: float, speed: float, m: float) -> float:
    return m * (speed / S) ** 2 / (2.0 * K_B)


def config_names() -> List[str]:
    return ["C1", "C2", "C3", "C4", "C5"]


def config(name: str) -> List[RunConfig]:
    """All runs (sweep points) of one BASELINE.json config, sharing one mesh."""
    mO = 16.0 * AMU
    if name == "C1":
        base = RunConfig("C1", lambda: meshes.plate(30.0), N=100_000, A_ref=1.0, label="plate a=30")
        return [base]
    if name == "C2":
        base = RunConfig("C2", lambda: meshes.geodesic_sphere(32), N=10_000_000, A_ref=float(np.pi))
        return [base.with_(T_inf=_t_inf_for_speed_ratio(S, 7500.0, mO), label=f"sphere S={S:g}")
                for S in (2.0, 5.0, 8.0)]
    if name == "C3":
        base = RunConfig("C3", lambda: meshes.cylinder(0.5, 2.0, 256, 3), N=100_000_000,
                         accommodation=0.8, A_ref=1.0)
        out = []
        for ang in (0.0, 45.0, 90.0):
            a = np.deg2rad(ang)
            # flow direction at angle `ang` to the cylinder axis (z), in the x-z plane
            vhat = np.array([-np.sin(a), 0.0, -np.cos(a)])
            out.append(base.with_(V=tuple(7500.0 * vhat), label=f"cylinder axis@{ang:g}deg"))
        return out
    if name == "C4":
        base = RunConfig("C4", lambda: meshes.satellite(4), N=100_000_000, A_ref=1.0)
        out = []
        for k in range(16):
            a = np.deg2rad(90.0 * k / 15.0)
            # pitch about y: flow from +z (into the pocket) at 0 deg to from +x at 90 deg
            vhat = np.array([-np.sin(a), 0.0, -np.cos(a)])
            out.append(base.with_(V=tuple(7500.0 * vhat), label=f"satellite pitch={np.rad2deg(a):.0f}deg"))
        return out
    if name == "C5":
        base = RunConfig("C5", lambda: meshes.large_body(5, 224), N=1_000_000_000, T_inf=900.0,
                         m=(16.0 * AMU, 4.0 * AMU), x=(0.7, 0.3), A_ref=float(np.pi))
        dirs = fibonacci_directions(64)
        return [base.with_(V=tuple(-7700.0 * d), label=f"large body attitude {k}") for k, d in enumerate(dirs)]
    raise KeyError(name)
