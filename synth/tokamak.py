"""Analytic large-aspect-ratio circular tokamak and shear-Alfven-like perturbations.

Inputs only (see synth/__init__.py).  Conventions (readings G4, G18, G19):

* right-handed cylindrical (R, phi, Z);  B0 = grad(psi0) x grad(phi) + F0 grad(phi), i.e.
  B_R = -psi_Z / R,  B_Z = +psi_R / R,  B_phi = F0 / R  with F0 = B0 * R0 constant;
* minor radius r = sqrt((R-R0)^2 + Z^2), poloidal angle theta = atan2(Z, R-R0);
* d psi0 / d r = B0 r / q(r); q is frozen at q(a) for r > a so that every element of the
  rectangular box has smooth fields to fit;
* a perturbation is a sum of poloidal harmonics with complex amplitudes multiplying
  exp(i (n phi - omega t)); physical field = Re[amplitude * exp(i (n phi - omega t))].
"""
from __future__ import annotations

from dataclasses import dataclass, field
from typing import Callable, List, Sequence, Tuple

import numpy as np


@dataclass
class CircularTokamak:
    R0: float = 3.0
    a: float = 1.0
    B0: float = 1.0
    # qkind 0: q = qc[0] + qc[1] u ;  qkind 1: q = qc[0] + qc[1] (u - qc[2])^2 ;  u = (r/a)^2
    qkind: int = 0
    qc: Tuple[float, float, float] = (1.1, 1.5, 0.0)

    # ---- safety factor -------------------------------------------------------------
    def q_of_u(self, u):
        u = np.minimum(np.asarray(u, dtype=np.float64), 1.0)  # frozen outside r = a
        if self.qkind == 0:
            return self.qc[0] + self.qc[1] * u
        return self.qc[0] + self.qc[1] * (u - self.qc[2]) ** 2

    def q(self, r):
        return self.q_of_u((np.asarray(r, dtype=np.float64) / self.a) ** 2)

    def dq_dr(self, r):
        r = np.asarray(r, dtype=np.float64)
        u = (r / self.a) ** 2
        inside = u < 1.0
        if self.qkind == 0:
            dqdu = np.full_like(u, self.qc[1])
        else:
            dqdu = 2.0 * self.qc[1] * (u - self.qc[2])
        return np.where(inside, dqdu * 2.0 * r / self.a ** 2, 0.0)

    @property
    def F0(self) -> float:
        return self.B0 * self.R0

    # ---- poloidal flux -------------------------------------------------------------
    def _psi_inside(self, u):
        B0, a = self.B0, self.a
        if self.qkind == 0:
            q0, q2 = self.qc[0], self.qc[1]
            return B0 * a * a / (2.0 * q2) * np.log1p(q2 * u / q0)
        qa, qb, uc = self.qc
        s = np.sqrt(qb / qa)
        return B0 * a * a / (2.0 * np.sqrt(qa * qb)) * (np.arctan(s * (u - uc)) + np.arctan(s * uc))

    def psi_of_r(self, r):
        r = np.asarray(r, dtype=np.float64)
        u = (r / self.a) ** 2
        inside = self._psi_inside(np.minimum(u, 1.0))
        qa = self.q_of_u(1.0)
        outside = self.B0 * (r * r - self.a ** 2) / (2.0 * qa)
        return inside + np.where(u > 1.0, outside, 0.0)

    def g(self, r):
        """(d psi0 / d r) / r = B0 / q(r); regular on the axis."""
        return self.B0 / self.q(r)

    # ---- fields at (R, Z) ----------------------------------------------------------
    def rtheta(self, R, Z):
        dR = np.asarray(R, dtype=np.float64) - self.R0
        Z = np.asarray(Z, dtype=np.float64)
        return np.hypot(dR, Z), np.arctan2(Z, dR)

    def psi(self, R, Z):
        r, _ = self.rtheta(R, Z)
        return self.psi_of_r(r)

    def grad_psi(self, R, Z):
        r, _ = self.rtheta(R, Z)
        g = self.g(r)
        return g * (np.asarray(R) - self.R0), g * np.asarray(Z)

    def B_cyl(self, R, Z):
        pR, pZ = self.grad_psi(R, Z)
        R = np.asarray(R, dtype=np.float64)
        return -pZ / R, self.F0 / R + 0.0 * pR, pR / R

    def Bmag(self, R, Z):
        bR, bP, bZ = self.B_cyl(R, Z)
        return np.sqrt(bR * bR + bP * bP + bZ * bZ)

    def grad_Bmag(self, R, Z, h: float = 1.0e-5):
        """Central differences of the analytic |B| (inputs only: marker bootstrap)."""
        R = np.asarray(R, dtype=np.float64)
        Z = np.asarray(Z, dtype=np.float64)
        dR = (self.Bmag(R + h, Z) - self.Bmag(R - h, Z)) / (2 * h)
        dZ = (self.Bmag(R, Z + h) - self.Bmag(R, Z - h)) / (2 * h)
        return dR, dZ

    def B_cart(self, x, y, z):
        x = np.asarray(x, dtype=np.float64)
        y = np.asarray(y, dtype=np.float64)
        R = np.hypot(x, y)
        c, s = x / R, y / R
        bR, bP, bZ = self.B_cyl(R, z)
        return bR * c - bP * s, bR * s + bP * c, bZ

    def gyro_period_axis(self, charge: float, mass: float) -> float:
        return 2.0 * np.pi * mass / (abs(charge) * self.B0)


# ---------------------------------------------------------------------------------------
# perturbations (reading G19)
# ---------------------------------------------------------------------------------------

@dataclass
class Harmonic:
    """One poloidal harmonic  P(r) exp(-i m theta)  of the perturbed electrostatic potential.

    ``radial(r)`` returns (P, dP/dr, P/r); all three must be regular at r = 0.
    """
    m: int
    radial: Callable[[np.ndarray], Tuple[np.ndarray, np.ndarray, np.ndarray]]


def kink_radial(r0: float, width: float):
    """P(r) = r xi(r),  xi = 0.5 (1 - tanh((r - r0)/width))  (config 1, m = 1)."""
    def f(r):
        t = np.tanh((r - r0) / width)
        xi = 0.5 * (1.0 - t)
        dxi = -0.5 * (1.0 - t * t) / width
        return r * xi, xi + r * dxi, xi
    return f


def gaussian_radial(m: int, rc: float, width: float):
    """P(r) = (r/rc)^m exp(-((r-rc)/width)^2); the r^m factor keeps it regular on the axis."""
    def f(r):
        e = np.exp(-((r - rc) / width) ** 2)
        pm1 = r ** (m - 1) / rc ** m
        P = pm1 * r * e
        dP = e * (m * pm1 - 2.0 * (r - rc) / width ** 2 * pm1 * r)
        return P, dP, pm1 * e
    return f


# order of the 7 complex amplitude fields in every perturbation table
PERT_FIELDS = ("E_R", "E_phi", "E_Z", "B_R", "B_phi", "B_Z", "B_par")


@dataclass
class Perturbation:
    """Toroidal mode n: delta Phi = Re sum_m P_m(r) e^{i(n phi - m theta - omega t)}.

    Electromagnetic (ideal-MHD-like, E_par ~ 0) when ``electrostatic`` is False:
    delta A = (delta psi / R) phi_hat with  delta psi_m = (n q - m)/(q omega) P_m,
    delta B = grad(delta psi) x grad(phi),  delta E = -grad(delta Phi) - d(delta A)/dt.
    ``scale`` multiplies every amplitude (set by ``normalise``).
    """
    eq: CircularTokamak
    n: int
    omega: float
    harmonics: Sequence[Harmonic]
    electrostatic: bool = False
    scale: float = 1.0

    def potentials(self, R, Z):
        """Complex amplitudes Phi, dPhi/dR, dPhi/dZ, psi1, dpsi1/dR, dpsi1/dZ at (R, Z)."""
        eq = self.eq
        R = np.asarray(R, dtype=np.float64)
        Z = np.asarray(Z, dtype=np.float64)
        r, th = eq.rtheta(R, Z)
        ct, st = np.cos(th), np.sin(th)
        q = eq.q(r)
        dq = eq.dq_dr(r)
        out = [np.zeros(R.shape, dtype=np.complex128) for _ in range(6)]
        for h in self.harmonics:
            P, dP, Por = h.radial(r)
            ph = np.exp(-1j * h.m * th)
            # f(r) e^{-i m theta}: d/dR = (f' cos + i m (f/r) sin) e^{..}, d/dZ = (f' sin - i m (f/r) cos) e^{..}
            out[0] += P * ph
            out[1] += (dP * ct + 1j * h.m * Por * st) * ph
            out[2] += (dP * st - 1j * h.m * Por * ct) * ph
            if not self.electrostatic:
                al = (self.n * q - h.m) / (q * self.omega)
                dal = h.m * dq / (q * q * self.omega)
                f, df, fr = al * P, dal * P + al * dP, al * Por
                out[3] += f * ph
                out[4] += (df * ct + 1j * h.m * fr * st) * ph
                out[5] += (df * st - 1j * h.m * fr * ct) * ph
        return [self.scale * o for o in out]

    def amplitudes(self, R, Z):
        """The 7 complex amplitude fields (PERT_FIELDS order), each shaped like R."""
        eq = self.eq
        R = np.asarray(R, dtype=np.float64)
        Phi, PhiR, PhiZ, ps, psR, psZ = self.potentials(R, Z)
        E_R = -PhiR
        E_Z = -PhiZ
        E_p = -(1j * self.n / R) * Phi + (1j * self.omega / R) * ps
        B_R = -psZ / R
        B_Z = psR / R
        B_p = np.zeros_like(B_R)
        b0R, b0P, b0Z = eq.B_cyl(R, Z)
        Bm = np.sqrt(b0R ** 2 + b0P ** 2 + b0Z ** 2)
        B_par = (b0R * B_R + b0Z * B_Z) / Bm
        return np.stack([E_R, E_p, E_Z, B_R, B_p, B_Z, B_par], axis=-1)

    def normalise(self, target_dB: float, nr: int = 400, nth: int = 64) -> "Perturbation":
        """Rescale so that max |delta B| over the plasma equals ``target_dB`` (electromagnetic)
        or max |delta E| equals it (electrostatic)."""
        eq = self.eq
        r = np.linspace(1e-3, eq.a, nr)[:, None]
        th = np.linspace(0.0, 2 * np.pi, nth, endpoint=False)[None, :]
        R = eq.R0 + r * np.cos(th)
        Z = r * np.sin(th) + 0.0 * R
        self.scale = 1.0
        A = self.amplitudes(R, Z)
        sl = slice(0, 3) if self.electrostatic else slice(3, 6)
        mag = np.sqrt((np.abs(A[..., sl]) ** 2).sum(-1)).max()
        self.scale = target_dB / mag
        return self
