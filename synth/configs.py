"""The five BASELINE.json workloads as seeded synthetic inputs.

``make_config(idx, n_markers=..., nx=...)`` builds equilibrium, mesh, tables and markers; both sizes
may be reduced for tests (the physics recipe is unchanged).  Normalisation (reading G17):
charge = 1, mass = 0.02, B0 = 1  =>  Omega0 = 50, axis gyro-period 2 pi / 50.
"""
from __future__ import annotations

from dataclasses import dataclass, field
from typing import List, Optional

import numpy as np

from .tokamak import CircularTokamak, Perturbation, Harmonic, kink_radial, gaussian_radial
from .mesh import rect_tri_mesh, eq_tables, pert_tables
from .markers import load_markers

# f0 kinds (values mirror include/m3dk.h)
F0_MAXWELLIAN, F0_SLOWING_DOWN, F0_BEAM_PITCH = 0, 1, 2

CHARGE = 1.0
MASS = 0.02
BOX = (1.9, 4.1, -1.1, 1.1)


@dataclass
class F0Params:
    kind: int = F0_MAXWELLIAN
    T: float = 1.0          # Maxwellian temperature (energy units)
    v_c: float = 0.3        # slowing-down critical speed
    Lambda0: float = 0.75   # beam pitch centre, Lambda = mu B_axis / E
    dLambda: float = 0.2
    B_axis: float = 1.0


@dataclass
class Workload:
    name: str
    eq: CircularTokamak
    perts: List[Perturbation]
    node_RZ: np.ndarray
    tri: np.ndarray
    eq_coef: np.ndarray
    pert_coef: np.ndarray
    n_tor: np.ndarray
    omega: np.ndarray
    markers: dict
    charge: float
    mass: float
    f0: F0Params
    dt: float
    nsteps: int
    sort_interval: int
    seed: int
    nx: int

    @property
    def n_markers(self) -> int:
        return int(self.markers["x"].shape[0])

    @property
    def n_elems(self) -> int:
        return int(self.tri.shape[0])

    @property
    def n_modes(self) -> int:
        return int(self.n_tor.shape[0])


CONFIGS = {
    0: dict(name="cfg0-tiny-equilibrium", n=4096, nx=32, dt_gyro=4.0, nsteps=200, sort_interval=0),
    1: dict(name="cfg1-fishbone-n1", n=1 << 20, nx=128, dt_gyro=5.0, nsteps=1000, sort_interval=10),
    2: dict(name="cfg2-tae-n4", n=1 << 22, nx=192, dt_gyro=8.0, nsteps=1000, sort_interval=10),
    3: dict(name="cfg3-rsae-n3", n=1 << 24, nx=256, dt_gyro=8.0, nsteps=500, sort_interval=10),
    4: dict(name="cfg4-scaling", n=1 << 20, nx=256, dt_gyro=4.0, nsteps=200, sort_interval=10),
}

_table_cache = {}


def _equilibrium(idx: int) -> CircularTokamak:
    if idx in (0, 1):
        return CircularTokamak(qkind=0, qc=(1.1, 1.5, 0.0))
    if idx == 2:
        return CircularTokamak(qkind=0, qc=(1.0, 2.0, 0.0))
    return CircularTokamak(qkind=1, qc=(2.0, 3.0, 0.25))


def _perturbations(idx: int, eq: CircularTokamak, amp: float) -> List[Perturbation]:
    if idx == 0:
        return []
    if idx == 1:
        p = Perturbation(eq, n=1, omega=0.01, harmonics=[Harmonic(1, kink_radial(0.4, 0.05))])
    elif idx == 2:
        hs = [Harmonic(4, gaussian_radial(4, 0.25, 0.08)), Harmonic(5, gaussian_radial(5, np.sqrt(0.1875), 0.08))]
        p = Perturbation(eq, n=4, omega=0.5 / (2 * 1.125 * eq.R0), harmonics=hs)
    else:
        p = Perturbation(eq, n=3, omega=0.02, harmonics=[Harmonic(6, gaussian_radial(6, 0.5, 0.05))])
    return [p.normalise(amp * eq.B0)]


def _kappa_fn(eq: CircularTokamak, profile_L: Optional[float]):
    """kappa = d ln f0 / d psi for n(r) = exp(-(r/L)^2):  (d ln n/dr)/(d psi/dr) = -2 q(r) / (L^2 B0)."""
    if profile_L is None:
        return None

    def fn(R, Z):
        r, _ = eq.rtheta(R, Z)
        return -2.0 * eq.q(r) / (profile_L ** 2 * eq.B0)
    return fn


def make_config(idx: int, n_markers: Optional[int] = None, nx: Optional[int] = None, amp: float = 1.0e-4,
                dt_gyro: Optional[float] = None, seed: Optional[int] = None, tables: bool = True) -> Workload:
    """tables = False: mesh, mode structure and markers only (eq_coef / pert_coef are None): for the ranks that receive
    the field image from rank 0 instead of fitting the tables themselves."""
    spec = CONFIGS[idx]
    n = spec["n"] if n_markers is None else int(n_markers)
    nx = spec["nx"] if nx is None else int(nx)
    dtg = spec["dt_gyro"] if dt_gyro is None else float(dt_gyro)
    seed = 1000 + idx if seed is None else int(seed)
    eq = _equilibrium(idx)
    dt = dtg * eq.gyro_period_axis(CHARGE, MASS)
    perts = _perturbations(idx, eq, amp)

    if idx == 0:
        mk = dict(rmin=0.1, rmax=0.8, profile_L=None, speed="mono", pitch="uniform")
        f0 = F0Params(kind=F0_MAXWELLIAN, T=0.5 * MASS)
        L = None
    elif idx == 1:
        mk = dict(rmin=0.02, rmax=0.9, profile_L=0.3, speed="slowing", v_c=0.3, pitch="uniform")
        f0 = F0Params(kind=F0_SLOWING_DOWN, v_c=0.3)
        L = 0.3
    elif idx == 2:
        mk = dict(rmin=0.1, rmax=0.8, profile_L=None, speed="mono", pitch="gauss", lam0=0.5, dlam=0.2)
        f0 = F0Params(kind=F0_BEAM_PITCH, v_c=0.3, Lambda0=0.75, dLambda=0.2, B_axis=eq.B0)
        L = None
    else:
        mk = dict(rmin=0.02, rmax=0.9, profile_L=0.4, speed="slowing", v_c=0.3, pitch="uniform")
        f0 = F0Params(kind=F0_SLOWING_DOWN, v_c=0.3)
        L = 0.4

    key = (idx, nx, amp)
    if not tables:
        node_RZ, tri = rect_tri_mesh(nx, BOX)
        eqc, pc = None, None
        n_tor = np.array([p.n for p in perts], dtype=np.int32)
        omega = np.array([p.omega for p in perts], dtype=np.float64)
    else:
        if key not in _table_cache:
            node_RZ, tri = rect_tri_mesh(nx, BOX)
            eqc = eq_tables(eq, node_RZ, tri, _kappa_fn(eq, L))
            if perts:
                pc, n_tor, omega = pert_tables(perts, node_RZ, tri)
            else:
                pc = np.zeros((0, tri.shape[0], 7, 2, 21))
                n_tor = np.zeros(0, dtype=np.int32)
                omega = np.zeros(0)
            _table_cache.clear()  # keep at most one big table set alive
            _table_cache[key] = (node_RZ, tri, eqc, pc, n_tor, omega)
        node_RZ, tri, eqc, pc, n_tor, omega = _table_cache[key]

    markers = load_markers(eq, n, seed, CHARGE, MASS, dt, **mk)
    return Workload(name=spec["name"], eq=eq, perts=perts, node_RZ=node_RZ, tri=tri, eq_coef=eqc, pert_coef=pc,
                    n_tor=n_tor, omega=omega, markers=markers, charge=CHARGE, mass=MASS, f0=f0, dt=dt,
                    nsteps=spec["nsteps"], sort_interval=spec["sort_interval"], seed=seed, nx=nx)
