"""Pins of the CPU oracle (oracle/m3dk_oracle.c) against what the paper and the mathematics fix.

None of these compares the oracle with itself or with the CUDA path: each check is a closed form, an
invariant, a textbook property, a library routine on a special case, or brute force (SURVEY.md 8(c) P1-P15,
DESIGN.md section 3).  All run on the CPU (``-m "not gpu"``).
"""
import json
import os

import numpy as np
import pytest
from numpy.polynomial import polynomial as npoly
from scipy.special import ellipk

import synth
from synth.configs import CHARGE, MASS
from synth.mesh import rect_tri_mesh, perturbed_tri_mesh, eq_tables, pert_tables, monomial_exponents
from synth.tokamak import Perturbation, Harmonic, gaussian_radial

from helpers import gc_start, invariants, trend_and_swing

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")
EQ = synth.CircularTokamak()
TG = EQ.gyro_period_axis(CHARGE, MASS)


# ------------------------------------------------------------------------------------------------------------
# P1, P2: Eq. (6) and Eq. (5) in uniform fields (textbook Boris properties, ref. [12])
# ------------------------------------------------------------------------------------------------------------

def test_p1_eq6_conserves_speed_with_E0(orc):
    rng = np.random.default_rng(1)
    for _ in range(200):
        vm, B = rng.normal(size=3), rng.normal(size=3) * 10 ** rng.uniform(-2, 2)
        h = 10 ** rng.uniform(-3, 1)
        vp = orc.eq6(vm, np.zeros(3), B, h)
        # exact in real arithmetic; in fp64 the direct 3x3 solve loses ~(1 + h|B|) ulp (h|B| = Omega dt/2 is the
        # condition number of I - hM): <= 4 ulp for h|B| <= 1, i.e. for dt up to a third of a gyro-period
        ulp = np.spacing(np.linalg.norm(vm))
        assert abs(np.linalg.norm(vp) - np.linalg.norm(vm)) <= 4 * (1 + h * np.linalg.norm(B)) * ulp


def test_p1_eq6_equals_boris_rotation_form(orc):
    """The 3x3 solve of Eq. (6) equals the explicit Boris t/s form of ref. [12] ("can be calculated explicitly")."""
    rng = np.random.default_rng(2)
    for _ in range(200):
        vm, B, E = rng.normal(size=3), rng.normal(size=3), rng.normal(size=3)
        h = 10 ** rng.uniform(-3, 0.5)
        vminus = vm + h * E
        t = h * B
        s = 2 * t / (1 + t @ t)
        vplus = vminus + np.cross(vminus + np.cross(vminus, t), s)
        ref = vplus + h * E
        got = orc.eq6(vm, E, B, h)
        assert np.allclose(got, ref, rtol=0, atol=2e-15 * max(1.0, np.abs(ref).max()))
        # and it satisfies Eq. (6) itself: (v+ - v-)/(2h) = E + (v+ + v-)/2 x B
        res = (got - vm) / (2 * h) - E - np.cross(0.5 * (got + vm), B)
        assert np.abs(res).max() < 1e-13 * max(1.0, np.abs(E).max(), np.abs(np.cross(vm, B)).max() / h)


def test_p2_uniform_B_gyrophase_and_radius(orc):
    q, m, B0, dt, n = 1.3, 0.7, 2.1, 0.37, 500
    Om = q * B0 / m
    x0 = np.array([[0.3, -0.2, 0.1]])
    v0 = np.array([[0.8, 0.5, 0.25]])
    xs, vs = [x0], [v0]
    for _ in range(n):
        x1, v1 = orc.push_uniform(xs[-1], vs[-1], [0, 0, B0], [0, 0, 0], q, m, 1, dt)
        xs.append(x1)
        vs.append(v1)
    v = np.concatenate(vs)
    ang = np.unwrap(np.arctan2(v[:, 1], v[:, 0]))
    dphi = np.diff(ang)
    # rotation per step is exactly -sign(q) 2 atan(Omega dt / 2) about B
    assert np.allclose(dphi, -2 * np.arctan(Om * dt / 2), rtol=0, atol=1e-12)   # (unwrapped angles reach ~600 rad)
    assert np.allclose(np.hypot(v[:, 0], v[:, 1]), np.hypot(*v0[0, :2]), rtol=1e-13)
    assert np.allclose(v[:, 2], v0[0, 2], rtol=0, atol=0)       # parallel velocity untouched
    x = np.concatenate(xs)
    # the positions lie on a circle (constant distance from a fixed centre) and z advances uniformly (Eq. 5)
    A = np.c_[2 * x[:, 0], 2 * x[:, 1], np.ones(len(x))]
    cx, cy, c = np.linalg.lstsq(A, x[:, 0] ** 2 + x[:, 1] ** 2, rcond=None)[0]
    rad = np.hypot(x[:, 0] - cx, x[:, 1] - cy)
    assert rad.std() / rad.mean() < 1e-12
    assert np.allclose(np.diff(x[:, 2]), dt * v0[0, 2], rtol=1e-12)


def test_p2_ExB_drift_exact(orc):
    q, m, dt = 1.0, 0.5, 0.9
    B = np.array([0.0, 0.0, 1.7])
    E = np.array([0.3, -0.2, 0.0])
    vd = np.cross(E, B) / (B @ B)
    # a marker that starts with the drift velocity keeps it exactly; any other one gyrates about it
    x1, v1 = orc.push_uniform(np.zeros((1, 3)), vd[None, :], B, E, q, m, 1000, dt)
    assert np.allclose(v1[0], vd, rtol=0, atol=1e-14)
    assert np.allclose(x1[0], 1000 * dt * vd, rtol=1e-12)
    n = 4000
    x2, v2 = orc.push_uniform(np.zeros((1, 3)), np.array([[0.4, 0.1, 0.0]]), B, E, q, m, n, dt)
    rho = np.linalg.norm(np.array([0.4, 0.1, 0.0]) - vd) * m / (q * 1.7) * 2
    assert np.linalg.norm(x2[0] - n * dt * vd) < 2 * rho          # mean drift = E x B / B^2


# ------------------------------------------------------------------------------------------------------------
# analytic back-end is a consistent equilibrium (readings G4, G18): pins the fields every physics pin rests on
# ------------------------------------------------------------------------------------------------------------

@pytest.mark.parametrize("idx", [0, 2, 3])
def test_analytic_fields_consistent(orc, idx):
    from synth.configs import _equilibrium
    eq = _equilibrium(idx)
    an = orc.analytic_of(eq)
    rng = np.random.default_rng(3)
    r = rng.uniform(0.05, 0.95, 400)
    th = rng.uniform(0, 2 * np.pi, 400)
    R, Z, phi = eq.R0 + r * np.cos(th), r * np.sin(th), rng.uniform(0, 6, 400)
    f, psi = orc.eval_analytic(an, R, phi, Z)
    h = 1e-5
    _, pRp = orc.eval_analytic(an, R + h, phi, Z)
    _, pRm = orc.eval_analytic(an, R - h, phi, Z)
    _, pZp = orc.eval_analytic(an, R, phi, Z + h)
    _, pZm = orc.eval_analytic(an, R, phi, Z - h)
    assert np.allclose(f[:, 0], (pRp - pRm) / (2 * h), rtol=0, atol=2e-9)       # psi_R
    assert np.allclose(f[:, 1], (pZp - pZm) / (2 * h), rtol=0, atol=2e-9)       # psi_Z
    # d psi / d r = B0 r / q(r)  (G18)
    assert np.allclose(np.hypot(f[:, 0], f[:, 1]), eq.B0 * r / eq.q(r), rtol=1e-12)
    # |B| is the norm of B = grad psi x grad phi + F grad phi (G4), and its stored gradient is its gradient
    Bm = np.sqrt(f[:, 0] ** 2 + f[:, 1] ** 2 + f[:, 5] ** 2) / R
    assert np.allclose(f[:, 2], Bm, rtol=1e-14)
    fp, _ = orc.eval_analytic(an, R + h, phi, Z)
    fm, _ = orc.eval_analytic(an, R - h, phi, Z)
    assert np.allclose(f[:, 3], (fp[:, 2] - fm[:, 2]) / (2 * h), rtol=0, atol=3e-9)
    fp, _ = orc.eval_analytic(an, R, phi, Z + h)
    fm, _ = orc.eval_analytic(an, R, phi, Z - h)
    assert np.allclose(f[:, 4], (fp[:, 2] - fm[:, 2]) / (2 * h), rtol=0, atol=3e-9)
    # independent generator (synth) agrees: psi closed form, |B|
    assert np.allclose(psi, eq.psi(R, Z), rtol=1e-13, atol=1e-15)
    assert np.allclose(f[:, 2], eq.Bmag(R, Z), rtol=1e-13)


# ------------------------------------------------------------------------------------------------------------
# P3, P4, P6: invariants of the whole pusher on the analytic back-end (Fig. 1)
# ------------------------------------------------------------------------------------------------------------

def test_p3_mu_bitwise_constant(orc):
    w = synth.make_config(1, n_markers=512, nx=16)
    st, _, _ = orc.push_fe(orc.Mesh.of(w), orc.species_of(w), w.markers, 50, w.dt)
    assert np.array_equal(st["mu"], w.markers["mu"])
    assert not np.array_equal(st["x"], w.markers["x"])


@pytest.mark.parametrize("lam,dtg,nsteps", [(0.8, 0.25, 160000), (0.8, 4.0, 100000), (0.2, 0.25, 160000), (0.2, 4.0, 100000)])
def test_p4_energy_and_pphi_bounded_no_secular_drift(orc, lam, dtg, nsteps):
    an = orc.analytic_of(EQ)
    sp = orc.species(CHARGE, MASS)
    dt = dtg * TG
    s = gc_start(EQ, 0.3, lam, dt, CHARGE, MASS)
    tr, _ = orc.trace(sp, s, nsteps, dt, an=an)
    assert len(tr) == nsteps
    E, P = invariants(orc, an, tr, s[6], CHARGE, MASS)
    for q in (E, P):
        trend, swing = trend_and_swing(tr[:, 7], q)
        assert trend < 0.01 * swing            # no linear trend: the fitted slope x T is << the oscillation
        assert swing < 0.12 * (dtg / 4.0) ** 2 + 1e-3   # oscillation amplitude O(dt^2), percent level at 4 gyro-periods
    # O(dt^2): the swing at 4 gyro-periods is ~256x the swing at 0.25
    if dtg == 4.0:
        s2 = gc_start(EQ, 0.3, lam, 0.25 * TG, CHARGE, MASS)
        tr2, _ = orc.trace(sp, s2, 40000, 0.25 * TG, an=an)
        E2, _ = invariants(orc, an, tr2, s2[6], CHARGE, MASS)
        ratio = trend_and_swing(tr[:, 7], E)[1] / trend_and_swing(tr2[:, 7], E2)[1]
        assert 100 < ratio < 600


def test_p6_paper_e1_scenario_bounded(orc):
    """the paper's own conservation test set-up (values in tests/golden/paper_e1_scenario.json)."""
    g = json.load(open(os.path.join(GOLDEN, "paper_e1_scenario.json")))
    q, m = g["charge_C"], g["mass_kg"]
    # reading G1: the garbled "3.2e-7 s 5/(2 pi/Omega)" means about five deuterium gyro-periods at 2 T
    Tg = 2 * np.pi * m / (q * g["B0_T"])
    assert abs(g["dt_rk4_s"] / Tg - g["gyro_periods_per_rk4_step_stated"]) < 0.2
    assert g["dt_boris_s"] == pytest.approx(g["dt_rk4_s"] / 4)
    eq = synth.CircularTokamak(R0=g["R0_m"], a=g["a_m"], B0=g["B0_T"])
    an = orc.analytic_of(eq)
    sp = orc.species(q, m)
    dt, nsteps = g["dt_boris_s"], 1_000_000
    for kind in ("passing", "trapped"):
        vpar, vperp = g[kind]["v_par"], g[kind]["v_perp"]
        v = np.hypot(vpar, vperp)
        s = gc_start(eq, 0.5 * eq.a, vpar / v, dt, q, m, v=v)
        tr, _ = orc.trace(sp, s, nsteps, dt, an=an, stride=10)
        assert len(tr) == nsteps // 10
        E, P = invariants(orc, an, tr, s[6], q, m)
        # bounded: first and last tenth of the run have the same envelope, and no trend
        k = len(tr) // 10
        for qty in (E, P):
            trend, swing = trend_and_swing(tr[:, 7], qty)
            assert swing < 5e-2
            assert trend < 0.02 * swing
            sw0 = qty[:k].max() - qty[:k].min()
            sw1 = qty[-k:].max() - qty[-k:].min()
            assert 0.8 < sw1 / sw0 < 1.25


# ------------------------------------------------------------------------------------------------------------
# P7: slow-manifold orbit = guiding-centre orbit of the brute-force full orbit
# ------------------------------------------------------------------------------------------------------------

def _orbit_stats(eq, tr, smooth):
    x, y, z, t = tr[:, 0], tr[:, 1], tr[:, 2], tr[:, 7]
    if smooth > 1:
        k = np.ones(smooth) / smooth
        x, y, z, t = (np.convolve(a, k, "valid") for a in (x, y, z, t))
    R = np.hypot(x, y)
    phi = np.unwrap(np.arctan2(y, x))
    r = np.hypot(R - eq.R0, z)
    return (phi[-1] - phi[0]) / (t[-1] - t[0]), r.min(), r.max()


@pytest.mark.parametrize("lam", [0.2, 0.7])
def test_p7_slow_manifold_matches_bruteforce_full_orbit(orc, lam):
    an = orc.analytic_of(EQ)
    sp = orc.species(CHARGE, MASS)
    r0, T = 0.3, 1500.0
    X = np.array([EQ.R0 + r0, 0.0, 0.0])
    b = np.array([c[0] for c in EQ.B_cart(X[0:1], X[1:2], X[2:3])])
    B = np.linalg.norm(b)
    b /= B
    vpar, vperp = lam, np.sqrt(1 - lam * lam)
    mu = MASS * vperp ** 2 / (2 * B)
    dt = TG
    s = gc_start(EQ, r0, lam, dt, CHARGE, MASS)
    trS, _ = orc.trace(sp, s, int(T / dt), dt, an=an)
    # brute force: the same particle as a true full orbit: no mu force (mu = 0), gyrating velocity, dt = T_gyro/200
    e1 = np.cross(b, [0.0, 0.0, 1.0])
    e1 /= np.linalg.norm(e1)
    v = vpar * b + vperp * e1
    rho = MASS / (CHARGE * B) * np.cross(b, v)           # x = X + rho, d rho/dt = v_perp
    sF = np.concatenate([X + rho, v, [0.0, 0.0]])
    dtf = TG / 200
    trF, _ = orc.trace(sp, sF, int(T / dtf), dtf, an=an, stride=4)
    precS, rminS, rmaxS = _orbit_stats(EQ, trS, 1)
    precF, rminF, rmaxF = _orbit_stats(EQ, trF, 50)      # 50 samples x 4 sub-steps = one gyro-period average
    rhoL = MASS * vperp / (CHARGE * B)
    assert abs(precS / precF - 1) < 0.01                # toroidal precession / transit frequency
    assert abs(rmaxS - rmaxF) < 0.5 * rhoL              # banana / drift-surface width to a fraction of rho_L
    assert abs(rminS - rminF) < 0.5 * rhoL
    assert rmaxS - r0 > 3 * rhoL if lam == 0.2 else True  # (the trapped orbit really has a banana to compare)


# ------------------------------------------------------------------------------------------------------------
# P8: bounce / transit frequencies against their closed forms (large aspect ratio, north_star)
# ------------------------------------------------------------------------------------------------------------

@pytest.mark.parametrize("r,lam,tol", [(0.1, 0.8, 0.005), (0.1, 0.5, 0.01), (0.3, 0.8, 0.01), (0.1, 0.1, 0.02),
                                       (0.3, 0.1, 0.10), (0.3, 0.2, 0.08)])
def test_p8_bounce_transit_frequency_closed_form(orc, r, lam, tol):
    mass = 0.002                      # rho* = 0.002: thin orbits, so that the zero-width closed form applies
    an = orc.analytic_of(EQ)
    sp = orc.species(CHARGE, mass)
    dt = 0.5 * 2 * np.pi * mass / CHARGE
    s = gc_start(EQ, r, lam, dt, CHARGE, mass)
    tr, _ = orc.trace(sp, s, int(3000 / dt), dt, an=an)
    x, y, z, t = tr[:, 0], tr[:, 1], tr[:, 2], tr[:, 7]
    th = np.unwrap(np.arctan2(z, np.hypot(x, y) - EQ.R0))
    eps, mu = r / EQ.R0, s[6]
    q_true = EQ.q(r) * EQ.R0 / np.sqrt(EQ.R0 ** 2 - r ** 2)             # G18
    w0 = np.sqrt(eps * mu * EQ.B0 / mass) / (q_true * EQ.R0)
    k2 = mass * lam ** 2 / (4 * eps * mu * EQ.B0)                       # v_par0 = lam at the outboard mid-plane
    if k2 < 1:      # trapped: omega_b = pi omega_0 / (2 K(k))
        ref = np.pi * w0 / (2 * ellipk(k2))                             # scipy ellipk takes the parameter k^2
        c = np.where((th[:-1] < 0) & (th[1:] >= 0))[0]
        tc = t[c] - th[c] / (th[c + 1] - th[c]) * dt
        got = 2 * np.pi / np.mean(np.diff(tc))
    else:           # passing: omega_t = pi kappa omega_0 / K(1/kappa)
        ref = np.pi * np.sqrt(k2) * w0 / ellipk(1 / k2)
        got = abs(th[-1] - th[0]) / (t[-1] - t[0])
    assert abs(got / ref - 1) < tol


# ------------------------------------------------------------------------------------------------------------
# P9, P14: finite-element back-end: polynomial evaluation, frames, element search
# ------------------------------------------------------------------------------------------------------------

def test_p9_fe_evaluation_is_the_g10_polynomial(orc):
    """Random coefficient tables on a jittered mesh: the oracle's value / gradient equal numpy's polyval2d of the
    coefficient matrix c[i, j] (monomials xi^i eta^j, j outer / i inner storage, centroid frame, s = 1/longest edge)."""
    rng = np.random.default_rng(5)
    node, tri = perturbed_tri_mesh(6, seed=11)
    ne = tri.shape[0]
    eqc = rng.normal(size=(ne, 4, 21))
    pc = rng.normal(size=(2, ne, 7, 2, 21))
    n_tor, omega = np.array([3, -2], dtype=np.int32), np.array([0.7, -0.3])
    m = orc.Mesh(node, tri, eqc, pc, n_tor, omega)
    npts = 300
    R, Z = rng.uniform(2.0, 4.0, npts), rng.uniform(-1.0, 1.0, npts)
    phi, t = rng.uniform(-3, 3, npts), 1.9
    elem, out = m.eval(R, phi, Z, t)
    assert (elem >= 0).all()
    ex = monomial_exponents()

    def poly(c21, xi, eta):
        C = np.zeros((6, 6), dtype=c21.dtype)
        C[ex[:, 0], ex[:, 1]] = c21
        v = npoly.polyval2d(xi, eta, C)
        dx = npoly.polyval2d(xi, eta, npoly.polyder(C, axis=0))
        de = npoly.polyval2d(xi, eta, npoly.polyder(C, axis=1))
        return v, dx, de

    for p in range(npts):
        e = elem[p]
        P = node[tri[e]]
        # containment by barycentric coordinates (independent of the edge-function form)
        lam = np.linalg.solve(np.c_[P, np.ones(3)].T, [R[p], Z[p], 1.0])
        assert (lam > -1e-12).all()
        cen = P.mean(axis=0)
        s = 1.0 / max(np.linalg.norm(P[1] - P[0]), np.linalg.norm(P[2] - P[1]), np.linalg.norm(P[0] - P[2]))
        xi, eta = (R[p] - cen[0]) * s, (Z[p] - cen[1]) * s
        _, dx, de = poly(eqc[e, 0], xi, eta)
        v1, dx1, de1 = poly(eqc[e, 1], xi, eta)
        exp = [dx * s, de * s, v1, dx1 * s, de1 * s, poly(eqc[e, 2], xi, eta)[0], poly(eqc[e, 3], xi, eta)[0]]
        assert np.allclose(out[p, :7], exp, rtol=1e-12, atol=1e-12)
        # perturbed part: Re[C exp(i(n phi - omega t))], d/dphi -> i n, d/dt -> -i omega  (G8)
        E1 = np.zeros(3)
        B1 = np.zeros(3)
        g = np.zeros(3)
        dtB = 0.0
        Bp = 0.0
        for k in range(2):
            cc = pc[k, e, :, 0, :] + 1j * pc[k, e, :, 1, :]
            ph = np.exp(1j * (n_tor[k] * phi[p] - omega[k] * t))
            vals = [poly(cc[f], xi, eta) for f in range(7)]
            E1 += [(vals[f][0] * ph).real for f in range(3)]
            B1 += [(vals[3 + f][0] * ph).real for f in range(3)]
            Bp += (vals[6][0] * ph).real
            g += [(vals[6][1] * s * ph).real, (1j * n_tor[k] * vals[6][0] * ph).real / R[p], (vals[6][2] * s * ph).real]
            dtB += (-1j * omega[k] * vals[6][0] * ph).real
        assert np.allclose(out[p, 7:10], E1, rtol=1e-12, atol=1e-12)
        assert np.allclose(out[p, 10:13], B1, rtol=1e-12, atol=1e-12)
        assert np.allclose(out[p, 13:16], g, rtol=1e-12, atol=1e-12)
        assert np.allclose(out[p, 16], dtB, rtol=1e-12, atol=1e-12)
        assert np.allclose(out[p, 17], Bp, rtol=1e-12, atol=1e-12)


def test_p9_fe_tables_reproduce_analytic_fields(orc):
    """LSQ quintic tables on the 32^2 mesh agree with the analytic equilibrium to the fit accuracy, refined mesh better."""
    err = {}
    for nx in (16, 32):
        node, tri = rect_tri_mesh(nx)
        m = orc.Mesh(node, tri, eq_tables(EQ, node, tri))
        rng = np.random.default_rng(6)
        r, th = rng.uniform(0.05, 0.9, 2000), rng.uniform(0, 2 * np.pi, 2000)
        R, Z, phi = EQ.R0 + r * np.cos(th), r * np.sin(th), np.zeros(2000)
        _, fe = m.eval(R, phi, Z)
        an, _ = orc.eval_analytic(orc.analytic_of(EQ), R, phi, Z)
        err[nx] = np.abs(fe[:, :6] - an[:, :6]).max(axis=0)
    assert (err[32] < 2e-7).all()
    assert (err[32][:5] < 0.2 * err[16][:5]).all()


@pytest.mark.parametrize("mesh", ["rect", "jittered"])
def test_p14_grid_search_equals_brute_force(orc, mesh):
    node, tri = rect_tri_mesh(20) if mesh == "rect" else perturbed_tri_mesh(20, seed=3)
    m = orc.Mesh(node, tri, np.zeros((tri.shape[0], 4, 21)))
    rng = np.random.default_rng(7)
    n = 200_000
    R, Z = rng.uniform(1.85, 4.15, n), rng.uniform(-1.15, 1.15, n)
    # include points exactly on nodes, edges and cell corners (the tie-break cases of G11)
    R[:441], Z[:441] = node[:, 0], node[:, 1]
    mid = 0.5 * (node[tri[:, 0]] + node[tri[:, 1]])
    R[441:441 + len(mid)], Z[441:441 + len(mid)] = mid[:, 0], mid[:, 1]
    a, b = m.locate(R, Z), m.locate(R, Z, brute=True)
    assert np.array_equal(a, b)
    inside = (R >= 1.9) & (R <= 4.1) & (Z >= -1.1) & (Z <= 1.1)
    assert ((a >= 0) == inside).all()
    # smallest index wins on shared edges: a node belongs to up to 6 triangles
    for p in range(0, 441, 37):
        owners = np.where((tri == p).any(axis=1))[0]
        assert a[p] == owners.min()


# ------------------------------------------------------------------------------------------------------------
# P5: invariants on the finite-element back-end are bounded up to the fit discontinuities and improve with the mesh
# ------------------------------------------------------------------------------------------------------------

def test_p5_fe_backend_conservation_improves_with_refinement(orc):
    sp = orc.species(CHARGE, MASS)
    an = orc.analytic_of(EQ)
    dt = 0.5 * TG
    dev = {}
    for nx in (16, 32):
        node, tri = rect_tri_mesh(nx)
        m = orc.Mesh(node, tri, eq_tables(EQ, node, tri))
        s = gc_start(EQ, 0.3, 0.2, dt, CHARGE, MASS)
        trA, _ = orc.trace(sp, s, 40000, dt, an=an)
        trF, _ = orc.trace(sp, s, 40000, dt, mesh=m)
        assert len(trF) == 40000
        E, P = invariants(orc, an, trF, s[6], CHARGE, MASS)
        EA, PA = invariants(orc, an, trA, s[6], CHARGE, MASS)
        # the FE orbit carries the analytic orbit's O(dt^2) oscillation plus a random walk from the fit jumps
        dev[nx] = max(abs(np.ptp(E) - np.ptp(EA)) / abs(E.mean()), abs(np.ptp(P) - np.ptp(PA)) / abs(P.mean()))
    assert dev[32] < 1e-5
    assert dev[32] < dev[16]


# ------------------------------------------------------------------------------------------------------------
# P10-P12: the delta-f weight equation
# ------------------------------------------------------------------------------------------------------------

def test_p10_zero_amplitude_gives_zero_weight(orc):
    w = synth.make_config(1, n_markers=256, nx=16, amp=0.0)
    st, _, _ = orc.push_fe(orc.Mesh.of(w), orc.species_of(w), w.markers, 100, w.dt)
    assert (st["w"] == 0.0).all()
    w0 = synth.make_config(0, n_markers=256, nx=16)           # and with no perturbation table at all
    st, _, _ = orc.push_fe(orc.Mesh.of(w0), orc.species_of(w0), w0.markers, 100, w0.dt)
    assert (st["w"] == 0.0).all()


@pytest.mark.parametrize("idx", [1, 2, 3])
def test_p11_weight_is_linear_in_amplitude(orc, idx):
    """Linear mode: trajectories do not see the perturbation and w scales with the amplitude."""
    wa = synth.make_config(idx, n_markers=256, nx=16, amp=1e-4)
    wb = synth.make_config(idx, n_markers=256, nx=16, amp=2e-4)
    sa, _, _ = orc.push_fe(orc.Mesh.of(wa), orc.species_of(wa), wa.markers, 100, wa.dt)
    sb, _, _ = orc.push_fe(orc.Mesh.of(wb), orc.species_of(wb), wb.markers, 100, wb.dt)
    assert np.array_equal(sa["x"], sb["x"]) and np.array_equal(sa["vz"], sb["vz"])
    scale = np.sqrt(np.mean(sa["w"] ** 2))
    assert scale > 0
    assert np.abs(sb["w"] - 2 * sa["w"]).max() < 1e-9 * scale


def _phi_es(eq, p, x, y, z, t):
    pA, prc, pwd, pom, pn, pm = p
    R = np.hypot(x, y)
    dR = R - eq.R0
    r, th = np.hypot(dR, z), np.arctan2(z, dR)
    return pA * np.exp(-((r - prc) / pwd) ** 2) * np.cos(pn * np.arctan2(y, x) - pm * th - pom * t)


@pytest.mark.parametrize("lam", [0.7, 0.2])
def test_p12_static_potential_weight_closed_form(orc, lam):
    """omega = 0, electrostatic, Maxwellian, kappa = 0:  dw/dt = (q/T) v.E1 = -(q/T) d Phi/dt along the orbit, so
    w(t) = -(q/T) [Phi(x(t)) - Phi(x(0))] up to the O(dt^2) error of the staggered quadrature (G9)."""
    p = (1e-3, 0.3, 0.1, 0.0, 2, 3)
    T0 = 0.37
    an = orc.analytic_of(EQ, kappa=0.0, pA=p[0], prc=p[1], pwd=p[2], pomega=p[3], pn=p[4], pm=p[5])
    sp = orc.species(CHARGE, MASS, 0, T=T0)
    errs = []
    for dtg in (1.0, 0.5, 0.25):
        dt = dtg * TG
        s = gc_start(EQ, 0.3, lam, dt, CHARGE, MASS)
        tr, _ = orc.trace(sp, s, int(40 / dt), dt, an=an)
        xm = 0.5 * (tr[:-1, 0:3] + tr[1:, 0:3])            # x_{l+1/2}, where w_{l+1/2} lives
        x0 = s[0:3] - 0.5 * dt * s[3:6]                    # x_{-1/2}
        ref = -(CHARGE / T0) * (_phi_es(EQ, p, xm[:, 0], xm[:, 1], xm[:, 2], 0.0) - _phi_es(EQ, p, x0[0], x0[1], x0[2], 0.0))
        errs.append(np.abs(tr[:-1, 6] - ref).max() / np.abs(ref).max())
    assert errs[0] < 5e-3
    assert 3.0 < errs[0] / errs[1] < 5.0 and 3.0 < errs[1] / errs[2] < 5.0      # second order


@pytest.mark.parametrize("lam", [0.7, 0.2])
def test_p12b_energy_pphi_exchange_identity(orc, lam):
    """A perturbation exp(i(n phi - omega t)) exchanges energy and P_phi in the ratio omega/n.  For an electrostatic
    one Eqs. (10)-(13) give exactly dP_phi/dt = q R E_phi and dE/dt = q v.E1, hence
        int dE/dt - (omega/n) int dP_phi/dt = -q [Phi(x(t), t) - Phi(x(0), 0)].
    The two integrals are read off two oracle runs (Maxwellian with kappa = 0; kappa != 0 with T -> infinity).  Pins the
    signs and factors of Eq. (10), (11), (12) (E x B term), (13) (q E.b term) against each other and against Phi."""
    p = (1e-3, 0.3, 0.1, 0.05, 2, 3)
    T0, k0 = 0.37, 1.7
    errs = []
    for dtg in (1.0, 0.5):
        dt = dtg * TG
        s = gc_start(EQ, 0.3, lam, dt, CHARGE, MASS)
        n = int(40 / dt)
        kw = dict(pA=p[0], prc=p[1], pwd=p[2], pomega=p[3], pn=p[4], pm=p[5])
        trE, _ = orc.trace(orc.species(CHARGE, MASS, 0, T=T0), s, n, dt, an=orc.analytic_of(EQ, kappa=0.0, **kw))
        trP, _ = orc.trace(orc.species(CHARGE, MASS, 0, T=1e300), s, n, dt, an=orc.analytic_of(EQ, kappa=k0, **kw))
        IE, IP = T0 * trE[:-1, 6], -CHARGE * trP[:-1, 6] / k0
        assert np.abs(IE).max() > 3e-4 and np.abs(p[3] / p[4] * IP).max() > 3e-4       # both terms matter
        xm, tm = 0.5 * (trE[:-1, 0:3] + trE[1:, 0:3]), 0.5 * (trE[:-1, 7] + trE[1:, 7])
        x0 = s[0:3] - 0.5 * dt * s[3:6]
        rhs = -CHARGE * (_phi_es(EQ, p, xm[:, 0], xm[:, 1], xm[:, 2], tm) - _phi_es(EQ, p, x0[0], x0[1], x0[2], -0.5 * dt))
        errs.append(np.abs(IE - p[3] / p[4] * IP - rhs).max() / np.abs(rhs).max())
    assert errs[0] < 2e-3
    assert 3.0 < errs[0] / errs[1] < 5.0


def test_p12c_weight_rhs_is_the_vector_form_of_eqs_8_to_13(orc):
    """Eqs. (8)-(13) written with numpy's cross / dot on random inputs (all terms, incl. the magnetic ones that no exact
    orbit identity isolates): catches a wrong component, sign or transposed operand in the scalar C arithmetic."""
    rng = np.random.default_rng(8)
    for trial in range(100):
        f = rng.normal(size=18)
        f[2] = abs(f[2]) + 0.5                      # |B|0
        R, mu = rng.uniform(2, 4), rng.uniform(0.001, 0.02)
        vl = rng.normal(size=3)
        q, m = rng.choice([-1.0, 1.0, 2.0]), rng.uniform(0.01, 0.05)
        kind = trial % 3
        T, vc, L0, dL, Bax = 0.4, 0.3, 0.7, 0.25, 1.1
        sp = orc.species(q, m, kind, T=T, v_c=vc, Lambda0=L0, dLambda=dL, B_axis=Bax)
        psiR, psiZ, Bm, F, kappa = f[0], f[1], f[2], f[5], f[6]
        E1, B1, gB, dtB = f[7:10], f[10:13], f[13:16], f[16]
        B0 = np.array([-psiZ / R, F / R, psiR / R])                   # (R, phi, Z), G4
        gradpsi = np.array([psiR, 0.0, psiZ])
        B0n = np.linalg.norm(B0)
        b0 = B0 / B0n
        vpar = vl @ b0
        dX = np.cross(E1, B0) / B0n ** 2 + vpar * B1 / B0n            # Eq. (12)
        Fpar = q * E1 @ b0 - mu * b0 @ gB                             # Eq. (13) x m   (G5)
        dP = q * dX @ gradpsi + Fpar * F / B0n                        # Eq. (10)       (G5): R B_phi0 = F
        dE = q * vl @ E1 + mu * dtB                                   # Eq. (11)       (G6)
        Ek = 0.5 * m * vl @ vl + mu * Bm
        if kind == 0:
            kE = -1 / T                                               # f0 ~ exp(-E/T)
        else:
            v = np.sqrt(2 * Ek / m)
            h = 1e-6 * Ek                                              # d ln f0/dE of 1/(v^3+vc^3) by finite differences
            lnf = lambda E_: -np.log(np.sqrt(2 * E_ / m) ** 3 + vc ** 3)
            kE = (lnf(Ek + h) - lnf(Ek - h)) / (2 * h)
            if kind == 2:                                              # x exp(-((Lambda - L0)/dL)^2), Lambda = mu B_axis / E
                lng = lambda E_: -((mu * Bax / E_ - L0) / dL) ** 2
                kE += (lng(Ek + h) - lng(Ek - h)) / (2 * h)
        ref = -((kappa / q) * dP + kE * dE)                           # Eqs. (8)-(9), (1 - w) -> 1
        got = orc.weight_rhs(f, sp, R, vl, mu)
        assert got == pytest.approx(ref, rel=2e-7, abs=1e-12)


# ------------------------------------------------------------------------------------------------------------
# P13 (sort oracle) and P15 (bootstrap)
# ------------------------------------------------------------------------------------------------------------

def test_p13_sort_perm_is_a_valid_counting_sort(orc):
    rng = np.random.default_rng(9)
    elem = rng.integers(-1, 50, 5000).astype(np.int32)
    perm = orc.sort_perm(elem, 50)
    assert np.array_equal(np.sort(perm), np.arange(5000))
    key = np.where(elem[perm] < 0, 50, elem[perm])
    assert (np.diff(key) >= 0).all()
    assert (np.diff(perm)[np.diff(key) == 0] > 0).all()      # stable


def test_p15_bad_initialisation_zigzags(orc):
    """PAPER.md:82 (footnote): a marker that does not start on the slow manifold jumps back and forth across it.
    With dt > gyro-period the rotation angle of Eq. (6), 2 atan(Omega dt/2), is close to pi, so a perpendicular velocity
    error flips sign every step and never decays; its step-to-step alternation in Z is ~ dt * |error|."""
    an = orc.analytic_of(EQ)
    sp = orc.species(CHARGE, MASS)
    dt = 4 * TG
    good = gc_start(EQ, 0.3, 0.5, dt, CHARGE, MASS)
    bad = good.copy()
    dv = 0.05
    bad[5] += dv                                               # off the manifold: an extra perpendicular (Z) velocity
    zz = []
    for s in (good, bad):
        tr, _ = orc.trace(sp, s, 200, dt, an=an)
        Z = tr[:, 2]
        d2 = Z[2:] - 2 * Z[1:-1] + Z[:-2]
        zz.append(0.5 * np.abs(np.diff(d2)).mean())             # alternating part of the second difference
    assert zz[1] > 2 * zz[0]
    assert 0.5 * dt * dv < zz[1] - zz[0] < 2 * dt * dv       # the excess alternation is the velocity error times dt
