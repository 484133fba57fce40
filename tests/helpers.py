"""Shared helpers for the CPU test-suite (inputs and diagnostics only; no method arithmetic of the CUDA path)."""
import numpy as np

import synth


def gc_start(eq, r, lam, dt, charge, mass, v=1.0, theta=0.0, phi=0.0):
    """One marker state [x,y,z,vx,vy,vz,mu,w] at minor radius r on the slow manifold (reading G20)."""
    R = eq.R0 + r * np.cos(theta)
    x = np.array([R * np.cos(phi)])
    y = np.array([R * np.sin(phi)])
    z = np.array([r * np.sin(theta)])
    Bm = eq.Bmag(np.array([R]), z)
    mu = mass * v * v * (1.0 - lam * lam) / (2.0 * Bm)
    vx, vy, vz = synth.slow_manifold_velocity(eq, x, y, z, np.array([v * lam]), mu, charge, mass, dt)
    return np.array([x[0], y[0], z[0], vx[0], vy[0], vz[0], mu[0], 0.0])


def invariants(orc, an, tr, mu, charge, mass):
    """E_tot = m |v_l|^2 / 2 + mu |B|(x_l) and P_phi = q psi(x_l) + m R v_phi,l (reading G4)."""
    x, y, z, vx, vy, vz = (tr[:, k] for k in range(6))
    R = np.hypot(x, y)
    f, psi = orc.eval_analytic(an, R, np.arctan2(y, x), z)
    E = 0.5 * mass * (vx ** 2 + vy ** 2 + vz ** 2) + mu * f[:, 2]
    vphi = (-vx * y + vy * x) / R
    return E, charge * psi + mass * R * vphi


def trend_and_swing(t, q):
    """(linear-fit slope * total time, peak-to-peak), both relative to |mean|."""
    a = np.polyfit(t, q, 1)[0] * (t[-1] - t[0])
    return abs(a) / abs(q.mean()), (q.max() - q.min()) / abs(q.mean())


def rel_err(a, b, floor=0.0):
    a = np.asarray(a)
    b = np.asarray(b)
    return np.abs(a - b) / np.maximum(np.abs(b), floor if floor > 0 else np.finfo(float).tiny)
