"""Pins of the oracle's finite-Larmor-radius mode (Eq. 14; reading G23): mode 2 =
linear delta-f with the perturbed fields replaced by their 4-point gyro-ring averages.  Checked against the geometry the
paper states (four vectors of length |rho_L|, uniform in gyro-angle, perpendicular to b), the paper's own numbers for the
gyro-radius (test E1), the zero-radius limit, exactness for fields that are linear in space, and the
plane-wave reduction factor of the 4-point rule.  CPU only."""
import json
import os

import numpy as np
import pytest

import synth
from synth.configs import CHARGE, MASS

from helpers import gc_start

EQ = synth.CircularTokamak()
TG = EQ.gyro_period_axis(CHARGE, MASS)
GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


def test_f1_ring_geometry(orc):
    """Four points at distance rho = m v_perp / (|q| B), v_perp = sqrt(2 mu B / m), perpendicular to b0, 90 degrees apart,
    summing to zero; the first along the major radius made perpendicular to b0."""
    an = orc.analytic_of(EQ)
    sp = orc.species(CHARGE, MASS)
    rng = np.random.Generator(np.random.PCG64(2))
    for _ in range(20):
        R, Z, phi = rng.uniform(2.4, 3.6), rng.uniform(-0.5, 0.5), rng.uniform(-np.pi, np.pi)
        X = np.array([R * np.cos(phi), R * np.sin(phi), Z])
        mu = rng.uniform(0.001, 0.02)
        pts = orc.gyro_ring(sp, X, mu, an=an)
        BR, BP, BZ = (float(np.asarray(b).reshape(-1)[0]) for b in EQ.B_cyl(np.array([R]), np.array([Z])))
        Bn = np.sqrt(BR ** 2 + BP ** 2 + BZ ** 2)
        b = np.array([BR * np.cos(phi) - BP * np.sin(phi), BR * np.sin(phi) + BP * np.cos(phi), BZ]) / Bn
        rho = MASS * np.sqrt(2 * mu * Bn / MASS) / (abs(CHARGE) * Bn)
        d = pts - X
        assert np.allclose(np.linalg.norm(d, axis=1), rho, rtol=1e-12)
        assert np.abs(d @ b).max() < 1e-12 * rho
        assert np.abs(d.sum(axis=0)).max() < 1e-14
        assert abs(d[0] @ d[1]) < 1e-12 * rho ** 2 and np.allclose(d[2], -d[0]) and np.allclose(d[3], -d[1])
        Rhat = np.array([np.cos(phi), np.sin(phi), 0.0])
        e1 = Rhat - (Rhat @ b) * b
        assert np.allclose(d[0] / rho, e1 / np.linalg.norm(e1), atol=1e-12)
        assert np.allclose(np.cross(b, d[0]) / rho, d[1] / rho, atol=1e-12)      # e2 = b x e1: right-handed


def test_f1b_gyro_radius_of_the_papers_test_particle(orc):
    """deuterium, B = 2 T, v_perp = 2.4e6 m/s (the trapped particle of test E1): rho = m v_perp / (q B) =
    3.3436e-27 * 2.4e6 / (1.6022e-19 * 2) = 2.504e-2 m, from the scenario fixture."""
    with open(os.path.join(GOLDEN, "paper_e1_scenario.json")) as fh:
        sc = json.load(fh)
    m_D, q_e = 3.3435837724e-27, 1.602176634e-19
    vperp = 2.4e6
    eq = synth.CircularTokamak(R0=sc["R0_m"], a=sc["a_m"], B0=sc["B0_T"]) if "R0_m" in sc else synth.CircularTokamak(R0=1.67, a=0.67, B0=2.0)
    an = orc.analytic_of(eq)
    sp = orc.species(q_e, m_D)
    X = np.array([eq.R0, 0.0, 0.0])                                     # on the axis: |B| = B0
    mu = m_D * vperp ** 2 / (2 * eq.B0)
    pts = orc.gyro_ring(sp, X, mu, an=an)
    rho = np.linalg.norm(pts - X, axis=1)
    assert np.allclose(rho, m_D * vperp / (q_e * eq.B0), rtol=1e-12)
    assert abs(rho[0] - 2.504e-2) < 2e-5


def test_f2_zero_magnetic_moment_is_the_linear_mode(orc):
    """rho = 0: the four ring points coincide with X, so the weights must equal the linear mode's up to the rounding of the
    rotation into Cartesian components and back (cos^2 + sin^2 = 1 only to an ulp); the orbits are the same bits."""
    w = synth.make_config(1, n_markers=200, nx=16)
    mk = {k: v.copy() for k, v in w.markers.items()}
    mk["mu"][:] = 0.0
    mesh = orc.Mesh.of(w)
    a, _, _ = orc.push_fe(mesh, orc.species_of(w, mode=0), mk, 30, w.dt)
    b, _, _ = orc.push_fe(mesh, orc.species_of(w, mode=2), mk, 30, w.dt)
    for k in a:
        if k != "w":
            assert np.array_equal(a[k], b[k]), k
    assert np.abs(a["w"]).max() > 0
    assert np.abs(a["w"] - b["w"]).max() < 1e-13 * np.sqrt(np.mean(a["w"] ** 2))


def test_f3_fields_linear_in_space_are_averaged_exactly(orc):
    """The 4-point rule is exact for fields that vary linearly over the ring.  A table whose only perturbed amplitude is
    E_Z = c0 + c1 xi + c2 eta with n = 0 (no toroidal dependence, a Cartesian component): <E_Z> at X equals E_Z(X)
    wherever the ring stays inside the element's neighbours with the same polynomial -- here the SAME linear function in
    every element, written in each element's own frame."""
    w = synth.make_config(1, n_markers=8, nx=16)
    from synth.mesh import element_frames
    cen, se = element_frames(w.node_RZ, w.tri)
    pc = np.zeros_like(w.pert_coef)
    a0, aR, aZ = 0.3, 0.7, -0.4                                          # E_Z = a0 + aR R + aZ Z, globally
    pc[0, :, 2, 0, 0] = a0 + aR * cen[:, 0] + aZ * cen[:, 1]             # constant term in the local frame
    pc[0, :, 2, 0, 1] = aR / se                                          # xi  coefficient
    pc[0, :, 2, 0, 6] = aZ / se                                          # eta coefficient
    mesh = orc.Mesh(w.node_RZ, w.tri, w.eq_coef, pc, np.array([0], dtype=np.int32), np.array([0.0]))
    sp = orc.species_of(w, mode=2)
    rng = np.random.Generator(np.random.PCG64(8))
    for _ in range(20):
        R, Z, phi = rng.uniform(2.5, 3.5), rng.uniform(-0.6, 0.6), rng.uniform(-np.pi, np.pi)
        X = np.array([R * np.cos(phi), R * np.sin(phi), Z])
        out = orc.flr_fields(sp, X, mu=0.01, mesh=mesh)
        assert abs(out[2] - (a0 + aR * R + aZ * Z)) < 1e-5              # R is not linear in Cartesian: O(rho^2 / R) left over
        assert np.abs(np.delete(out, 2)).max() < 1e-14


def test_f4_plane_wave_reduction_factor(orc):
    """Short-wavelength electrostatic wave: locally Phi ~ cos(k . x), and the 4-point rule multiplies the field at X by
    (1/2) [cos(k . e1 rho) + cos(k . e2 rho)] (its approximation of J0(k_perp rho)).  Checked on E1's
    dominant component with the wave vector taken from the analytic phase n phi - m theta."""
    n, m = 0, 14
    p = dict(pA=1e-3, prc=0.3, pwd=0.25, pomega=0.0, pn=n, pm=m)
    an = orc.analytic_of(EQ, kappa=0.0, **p)
    sp = orc.species(CHARGE, MASS, mode=2)
    r0, th0 = 0.3, 0.9
    R, Z = EQ.R0 + r0 * np.cos(th0), r0 * np.sin(th0)
    X = np.array([R, 0.0, Z])
    for mu in (0.002, 0.006):
        pts = orc.gyro_ring(sp, X, mu, an=an)
        d = pts - X
        # wave vector of cos(-m theta) at X: k = -m grad theta = -(m / r) theta-hat  (in the (R, Z) plane)
        k = -(m / r0) * np.array([-np.sin(th0), 0.0, np.cos(th0)])
        factor = 0.5 * (np.cos(k @ d[0]) + np.cos(k @ d[1]))
        f0, _ = orc.eval_analytic(an, np.array([R]), np.array([0.0]), np.array([Z]))
        avg = orc.flr_fields(sp, X, mu, an=an)
        e_theta0 = -f0[0, 7] * np.sin(th0) + f0[0, 9] * np.cos(th0)      # E1 along theta-hat (the direction of k)
        e_theta = -avg[0] * np.sin(th0) + avg[2] * np.cos(th0)
        assert abs(factor) < 0.98                                        # a real reduction at this k rho
        assert abs(e_theta / e_theta0 - factor) < 0.04, (mu, e_theta / e_theta0, factor)


def test_f5_ring_where_b_is_parallel_to_the_major_radius(orc):
    """The construction of reading G23 starts from the major-radius direction made perpendicular to b0; where b0 is
    (anti)parallel to it (a purely radial field: psi0 = A Z, F = 0) it starts from Z-hat instead.  The ring must still be
    four finite points at distance rho, perpendicular to b0, 90 degrees apart."""
    from handmade import HandMade
    from synth.configs import CHARGE, MASS
    A, mu = 0.9, 0.004
    hm = HandMade(eq=dict(psi=(0.0, 0.0, A), Bm=(1.0,), F=(0.0,), kappa=(0.0,)))
    sp = orc.species(CHARGE, MASS)
    X = np.array([3.2 * np.cos(0.4), 3.2 * np.sin(0.4), 0.1])
    pts = orc.gyro_ring(sp, X, mu, mesh=hm.oracle_mesh(orc))
    assert np.isfinite(pts).all()
    bx = -np.array([np.cos(0.4), np.sin(0.4), 0.0])                 # B_R = -A / R: b0 = -R-hat
    rho = np.sqrt(2 * MASS * mu / (A / 3.2)) / abs(CHARGE)
    d = pts - X
    assert np.allclose(np.linalg.norm(d, axis=1), rho, rtol=1e-12)
    assert np.abs(d @ bx).max() < 1e-12 * rho
    assert np.allclose(d[0], -d[2], atol=1e-15) and np.allclose(d[1], -d[3], atol=1e-15)
    assert abs(d[0] @ d[1]) < 1e-12 * rho * rho
    assert np.allclose(np.cross(bx, d[0]), d[1], rtol=1e-12, atol=1e-15)          # e2 = b0 x e1


def check_f6_nonlinear_mode_with_gyro_average(orc):
    """Mode 3 = the non-linear trajectories of mode 1 in the gyro-averaged perturbed fields of mode 2 ("use
    orbit-averaged fields in the above equations").  (a) mu = 0: the ring collapses onto X, mode 3 is mode 1 up to the
    rounding of the rotation to Cartesian components and back.  (b) Amplitudes of the Z components (E_Z, B_Z: Cartesian
    components) that are linear in Z with n = 0 are averaged exactly by the symmetric ring, so the trajectories of modes 3
    and 1 agree to round-off although rho != 0.  (c) On the config-1 kink (a field that is NOT linear over the ring) the two
    modes differ by much more: the average does something; and with amplitude 0 mode 3 is the linear mode bit for bit."""
    from handmade import HandMade
    from synth.configs import CHARGE, MASS
    w = synth.make_config(1, n_markers=300, nx=16, amp=1e-2)
    mesh = orc.Mesh.of(w)
    mk0 = {k: v.copy() for k, v in w.markers.items()}
    mk0["mu"][:] = 0.0
    a, _, _ = orc.push_fe(mesh, orc.species_of(w, mode=1), mk0, 20, w.dt)
    b, _, _ = orc.push_fe(mesh, orc.species_of(w, mode=3), mk0, 20, w.dt)
    for k in ("x", "vx", "vz", "w"):
        scale = np.sqrt(np.mean(a[k] ** 2))
        assert np.abs(a[k] - b[k]).max() < 1e-11 * scale, k
    # (b)
    hm = HandMade(eq=dict(psi=(0.0, 0.0, 0.0, 0.4), Bm=(0.8,), F=(2.4,), kappa=(0.3,)),
                  pert=dict(E_Z=(1e-3, 0.0, -1e-3), B_Z=(2e-3, 0.0, 3e-3)), n_tor=0, omega=0.0)
    hmesh = hm.oracle_mesh(orc)
    rng = np.random.Generator(np.random.PCG64(14))
    n = 50
    R, ph, Z = rng.uniform(2.6, 3.4, n), rng.uniform(-3, 3, n), rng.uniform(-0.5, 0.5, n)
    m2 = dict(x=R * np.cos(ph), y=R * np.sin(ph), z=Z, vx=0.3 * rng.normal(size=n), vy=0.3 * rng.normal(size=n),
              vz=0.3 * rng.normal(size=n), mu=np.full(n, 0.01), w=np.zeros(n))
    sp1, sp3 = orc.species(CHARGE, MASS, 0, T=0.5, mode=1), orc.species(CHARGE, MASS, 0, T=0.5, mode=3)
    a, _, _ = orc.push_fe(hmesh, sp1, m2, 3, 0.01)
    b, _, _ = orc.push_fe(hmesh, sp3, m2, 3, 0.01)
    rho = np.sqrt(2 * MASS * 0.01 / 0.8)
    assert rho > 0.02
    assert np.abs(a["vz"] - b["vz"]).max() < 1e-14 and np.abs(a["x"] - b["x"]).max() < 1e-14
    assert np.abs(a["vz"] - m2["vz"]).max() > 1e-5                     # the fields do act
    # (c)
    a, _, _ = orc.push_fe(mesh, orc.species_of(w, mode=1), w.markers, 20, w.dt)
    b, _, _ = orc.push_fe(mesh, orc.species_of(w, mode=3), w.markers, 20, w.dt)
    assert np.abs(a["w"] - b["w"]).max() > 1e-3 * np.sqrt(np.mean(a["w"] ** 2))
    w0 = synth.make_config(1, n_markers=100, nx=16, amp=0.0)
    a, _, _ = orc.push_fe(orc.Mesh.of(w0), orc.species_of(w0, mode=0), w0.markers, 10, w0.dt)
    b, _, _ = orc.push_fe(orc.Mesh.of(w0), orc.species_of(w0, mode=3), w0.markers, 10, w0.dt)
    for k in a:
        assert np.array_equal(a[k], b[k]), k


def test_f6_nonlinear_mode_with_gyro_average(orc):
    check_f6_nonlinear_mode_with_gyro_average(orc)
