"""Seeded marker loads (inputs only).  Recipe: SURVEY.md 8(d) D1, readings G17, G20.

RNG: numpy Generator(PCG64(seed)); draw order r, theta, phi, speed, pitch, each one full array.
State returned: Cartesian x, y, z, vx, vy, vz (v is v_{1/2}, on the slow manifold to first order),
mu = m v^2 (1 - lambda^2) / (2 |B|0(x)), w = 0.
"""
from __future__ import annotations

import numpy as np


def _sample_radius(rng, n, rmin, rmax, profile_L):
    """pdf proportional to r * n(r) on [rmin, rmax]; n(r) = exp(-(r/L)^2) or 1 (L None).

    (The toroidal Jacobian R/R0 is ignored - stated simplification of the recipe.)
    """
    u = rng.random(n)
    if profile_L is None:
        # "uniform in r" of config 0 is literal: r ~ U[rmin, rmax]
        return rmin + (rmax - rmin) * u
    L2 = profile_L ** 2
    a, b = np.exp(-rmin ** 2 / L2), np.exp(-rmax ** 2 / L2)
    return np.sqrt(-L2 * np.log(a - u * (a - b)))


def _sample_speed(rng, n, kind, v_b, v_c):
    u = rng.random(n)
    if kind == "mono":
        return np.full(n, v_b)
    # slowing-down f0 ~ 1/(v^3 + v_c^3), v < v_b: inverse CDF of v^2 f0
    Lg = np.log1p(v_b ** 3 / v_c ** 3)
    return v_c * np.expm1(u * Lg) ** (1.0 / 3.0)


def _sample_pitch(rng, n, kind, lam0, dlam):
    if kind == "uniform":
        return -1.0 + 2.0 * rng.random(n)
    lam = lam0 + dlam * rng.standard_normal(n)
    return np.clip(lam, -1.0, 1.0)


def slow_manifold_velocity(eq, x, y, z, vpar, mu, charge, mass, dt):
    """v_{1/2} = v_par' b + v_D  with  v_D = b x (mu grad|B| + m v_par^2 (b.grad)b) / (q |B|)   (Eq. 24 form)
    and the half-step mirror kick v_par' = v_par - (dt/2)(mu/m) b.grad|B|  (reading G20).

    (b.grad)b is a central difference of the analytic unit vector along b (Cartesian components).
    """
    x = np.asarray(x, dtype=np.float64)
    y = np.asarray(y, dtype=np.float64)
    z = np.asarray(z, dtype=np.float64)

    def bhat(px, py, pz):
        bx, by, bz = eq.B_cart(px, py, pz)
        B = np.sqrt(bx * bx + by * by + bz * bz)
        return bx / B, by / B, bz / B, B

    bx, by, bz, B = bhat(x, y, z)
    R = np.hypot(x, y)
    c, s = x / R, y / R
    gR, gZ = eq.grad_Bmag(R, z)
    gx, gy, gz = gR * c, gR * s, gZ
    eps = 1.0e-5
    pbx, pby, pbz, _ = bhat(x + eps * bx, y + eps * by, z + eps * bz)
    mbx, mby, mbz, _ = bhat(x - eps * bx, y - eps * by, z - eps * bz)
    kx, ky, kz = (pbx - mbx) / (2 * eps), (pby - mby) / (2 * eps), (pbz - mbz) / (2 * eps)
    fx = mu * gx + mass * vpar ** 2 * kx
    fy = mu * gy + mass * vpar ** 2 * ky
    fz = mu * gz + mass * vpar ** 2 * kz
    dx = (by * fz - bz * fy) / (charge * B)
    dy = (bz * fx - bx * fz) / (charge * B)
    dz = (bx * fy - by * fx) / (charge * B)
    vp = vpar - 0.5 * dt * (mu / mass) * (bx * gx + by * gy + bz * gz)
    return vp * bx + dx, vp * by + dy, vp * bz + dz


def load_markers(eq, n, seed, charge, mass, dt, *, rmin, rmax, profile_L=None,
                 speed="mono", v_b=1.0, v_c=0.3, pitch="uniform", lam0=0.5, dlam=0.2):
    rng = np.random.Generator(np.random.PCG64(seed))
    r = _sample_radius(rng, n, rmin * eq.a, rmax * eq.a, None if profile_L is None else profile_L * eq.a)
    th = 2.0 * np.pi * rng.random(n)
    ph = 2.0 * np.pi * rng.random(n)
    v = _sample_speed(rng, n, speed, v_b, v_c)
    lam = _sample_pitch(rng, n, pitch, lam0, dlam)
    R = eq.R0 + r * np.cos(th)
    Z = r * np.sin(th)
    x, y, z = R * np.cos(ph), R * np.sin(ph), Z
    Bm = eq.Bmag(R, Z)
    mu = mass * v * v * (1.0 - lam * lam) / (2.0 * Bm)
    vx, vy, vz = slow_manifold_velocity(eq, x, y, z, v * lam, mu, charge, mass, dt)
    w = np.zeros(n)
    cont = np.ascontiguousarray
    return dict(x=cont(x), y=cont(y), z=cont(z), vx=cont(vx), vy=cont(vy), vz=cont(vz), mu=cont(mu), w=cont(w))
