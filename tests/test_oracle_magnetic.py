"""Pins of the oracle pieces that the electrostatic pins P10-P19 and the analytic-back-end pins G1-G4 cannot see:

  M1  v_par B1 / B0 of Eq. (12)    closed form w(t) = -kappa v_par eps R0 t
  M2  -mu b0 . grad B1par of Eq. (13)    closed form for a marker at rest, per component
  M3  mu dB1par/dt of Eq. (11)    closed form w = (mu/T) [B1par(t) - B1par(0)] (discrete sum)
  N1  B0 + B1 and grad(|B|0 + B1par) in the mode-1 push (reading G21), one step against the explicit
      Boris rotation written with numpy
  Q1  poly_eval2 and the finite-element branch of gc_fields (second derivatives) against numpy's polyder
  Q2  pointwise dE/dt = dP_phi/dt = 0 of Eqs. (1)-(4) on the FINITE-ELEMENT back-end, to the fit error, shrinking with h

All on hand-made tables (tests/handmade.py) whose fields are polynomials known in closed form, through the oracle's
finite-element back-end (search, local frame, naive monomial sums, phase factors, weight equation).  Each check_* function
is also run against mutated copies of the oracle in tests/test_oracle_mutants.py, which shows the mistake it catches.
CPU only.
"""
import numpy as np
import pytest
from numpy.polynomial import polynomial as npoly

import synth
from synth.configs import CHARGE, MASS
from synth.mesh import eq_tables, element_frames, monomial_exponents, rect_tri_mesh

from handmade import HandMade

EQ = synth.CircularTokamak()


def _trace_w(orc, hm, sp, state8, nsteps, dt, t0=0.0):
    tr, s = orc.trace(sp, state8, nsteps, dt, mesh=hm.oracle_mesh(orc), t0=t0)
    assert len(tr) == nsteps
    return tr, s


# ---- M1 --------------------------------------------------------------------------------------------------------------
def check_m1_vpar_B1_over_B0(orc):
    """psi0 = A R, F = 0: B0 = (0, 0, A/R), a purely vertical field.  A marker with mu = 0 and v = (0, 0, vz) moves along it
    in a straight line at constant speed (v x B = 0 exactly), so R = R0, v_par = vz and |B0| = A/R0 are constants.  With the
    static radial perturbation B1_R = eps (n = 0, omega = 0) and nothing else, Eq. (12) gives (dX/dt)_1 = v_par eps/|B0| R-hat,
    Eq. (10) dP_phi/dt = q v_par eps R0, and Eqs. (8)-(9) with T -> infinity  dw/dt = -kappa v_par eps R0:
        w_{l+1/2} = -kappa vz eps R0 (l + 1) dt          (exact: every step adds the same number).
    Physically: the marker follows the perturbed field line outward at v_par B1_R/B0, psi changes at v_par eps R0 and
    delta f / f0 = -kappa delta psi."""
    A, eps, kap, R0, vz, dt, n = 0.37, 2.5e-3, -1.7, 2.9, 0.8, 0.011, 60
    for q in (CHARGE, -2.0):
        hm = HandMade(eq=dict(psi=(0.0, A), Bm=(1.0,), F=(0.0,), kappa=(kap,)), pert=dict(B_R=(eps,)), n_tor=0, omega=0.0)
        sp = orc.species(q, MASS, 0, T=1e300)
        tr, s = _trace_w(orc, hm, sp, [R0, 0.0, -0.3, 0.0, 0.0, vz, 0.0, 0.0], n, dt)
        assert np.array_equal(tr[:, 0], np.full(n, R0)) and np.array_equal(tr[:, 5], np.full(n, vz))   # straight line
        ref = -kap * vz * eps * R0 * dt * np.arange(1, n + 1)
        assert np.abs(tr[:, 6] - ref).max() <= 1e-13 * np.abs(ref).max()


# ---- M2 --------------------------------------------------------------------------------------------------------------
def check_m2_mirror_force_of_B1par(orc):
    """A marker at rest (v = 0) with mu > 0 in a field of constant strength table (|B|0 = const: no mirror force) never
    moves.  psi0 = aR R + aZ Z, F = F0: B0 = (-aZ, F0, aR)/R0, b0 = (-aZ, F0, aR)/S, S = sqrt(aR^2 + aZ^2 + F0^2),
    R B_phi0/|B0| = F0 R0/S.  With only B1par switched on (static), Eq. (13) gives m (dv_par/dt)_1 = -mu b0 . grad B1par,
    Eq. (10) dP_phi/dt = that times F0 R0/S, and with T -> infinity
        dw/dt = +(kappa/q) mu (b0 . grad B1par) F0 R0 / S        (a constant),
    one case per component of grad B1par: d/dR, d/dZ and (1/R) d/dphi (amplitude eps cos(n phi))."""
    aR, aZ, F0, kap, mu, eps, dt, n = 0.31, -0.23, 2.7, 1.3, 0.004, 3.0e-3, 0.05, 25
    R0, phi0, Z0 = 3.3, 0.7, 0.25
    S = np.sqrt(aR * aR + aZ * aZ + F0 * F0)
    b0 = np.array([-aZ, F0, aR]) / S
    ntor = 3
    cases = {"R": (dict(B_par=(0.0, eps, 0.0)), 0, np.array([eps, 0.0, 0.0])),
             "Z": (dict(B_par=(0.0, 0.0, eps)), 0, np.array([0.0, 0.0, eps])),
             "phi": (dict(B_par=(eps,)), ntor, np.array([0.0, -ntor * eps * np.sin(ntor * phi0) / R0, 0.0]))}
    for name, (pert, nt, grad) in cases.items():
        for q in (CHARGE, -1.5):
            hm = HandMade(eq=dict(psi=(0.0, aR, aZ), Bm=(1.1,), F=(F0,), kappa=(kap,)), pert=pert, n_tor=nt, omega=0.0)
            sp = orc.species(q, MASS, 0, T=1e300)
            x0 = [R0 * np.cos(phi0), R0 * np.sin(phi0), Z0]
            tr, s = _trace_w(orc, hm, sp, x0 + [0.0, 0.0, 0.0, mu, 0.0], n, dt)
            assert np.array_equal(tr[:, 0:3], np.tile(x0, (n, 1)))                                   # at rest
            wdot = (kap / q) * mu * (b0 @ grad) * F0 * R0 / S
            ref = wdot * dt * np.arange(1, n + 1)
            assert abs(wdot) > 0
            assert np.abs(tr[:, 6] - ref).max() <= 1e-12 * np.abs(ref).max(), name


# ---- M3 --------------------------------------------------------------------------------------------------------------
def check_m3_mu_dB1par_dt(orc):
    """The same marker at rest in an n = 0 perturbation B1par = eps cos(omega t) (amplitude eps, phase -omega t; reading G8)
    with kappa = 0 and a Maxwellian f0 ~ exp(-E/T): Eq. (11) gives dE/dt = mu dB1par/dt = -mu eps omega sin(omega t) and
    Eqs. (8)-(9) dw/dt = +(1/T) dE/dt, so on the staggered grid (reading G9)
        w_{L+1/2} = -(mu eps omega/T) dt sum_{l=0..L} sin(omega t_l),
    which tends to (mu/T) [B1par(t) - B1par(0)]: the marker's energy mu B follows the field strength."""
    mu, eps, om, T0, dt, n, t0 = 0.006, 4.0e-3, 0.9, 0.013, 0.04, 120, 0.3
    hm = HandMade(eq=dict(psi=(0.0, 0.2, 0.1), Bm=(0.9,), F=(3.0,), kappa=(0.0,)), pert=dict(B_par=(eps,)), n_tor=0, omega=om)
    sp = orc.species(CHARGE, MASS, 0, T=T0)
    tr, s = _trace_w(orc, hm, sp, [3.1, 0.2, -0.4, 0.0, 0.0, 0.0, mu, 0.0], n, dt, t0=t0)
    tl = t0 + dt * np.arange(n)
    ref = -(mu * eps * om / T0) * dt * np.cumsum(np.sin(om * tl))
    assert np.abs(tr[:, 6] - ref).max() <= 1e-12 * np.abs(ref).max()
    cont = (mu / T0) * eps * (np.cos(om * (tl + dt)) - np.cos(om * t0))          # the continuum limit, first order in dt
    assert np.abs(tr[:, 6] - cont).max() < 0.6 * om * dt * np.abs(cont).max()


# ---- N1 --------------------------------------------------------------------------------------------------------------
def _boris_ts(v, E, B, h):
    vminus = v + h * E
    t = h * B
    s = 2.0 * t / (1.0 + t @ t)
    return vminus + np.cross(vminus + np.cross(vminus, t), s) + h * E


def check_n1_mode1_push_uses_total_fields(orc):
    """One step of the non-linear trajectory mode on hand-made tables with every perturbed component switched on
    (amplitudes complex, n = 2, omega != 0, t != 0): the new velocity and position equal the explicit Boris rotation
    (t / s vectors, numpy cross products) in B = B0 + B1 and E-dagger = E1 - (mu/q) grad(|B|0 + B1par), all evaluated here
    from the closed forms of the tables.  A wrong sign or a missing component of B1 or grad B1par changes v+ at first order
    in the amplitude (1e-2 here)."""
    rng = np.random.default_rng(21)
    ntor, om, t = 2, 0.7, 1.9
    eqd = dict(psi=(0.1, 0.33, -0.21), Bm=(0.4, 0.15, -0.05), F=(2.9,), kappa=(0.5,))
    z = lambda: complex(rng.normal(), rng.normal()) * 1e-2
    pert = {k: (z(),) for k in ("E_R", "E_phi", "E_Z", "B_R", "B_phi", "B_Z")}
    pert["B_par"] = (z(), z(), z())
    hm = HandMade(eq=eqd, pert=pert, n_tor=ntor, omega=om)
    mesh = hm.oracle_mesh(orc)
    for q in (CHARGE, -1.0):
        sp = orc.species(q, MASS, 0, T=0.5, mode=1)
        n = 40
        R, phi, Z = rng.uniform(2.1, 3.9, n), rng.uniform(-3, 3, n), rng.uniform(-0.9, 0.9, n)
        v = rng.normal(size=(n, 3))
        mu = rng.uniform(0.0, 0.02, n)
        dt = 0.03
        mk = dict(x=R * np.cos(phi), y=R * np.sin(phi), z=Z, vx=v[:, 0], vy=v[:, 1], vz=v[:, 2], mu=mu, w=np.zeros(n))
        st, e, lost = orc.push_fe(mesh, sp, mk, 1, dt, t0=t)
        assert lost == 0
        ph = np.exp(1j * (ntor * phi - om * t))
        re = lambda name: (hm.amp_at(name, R, Z) * ph).real
        B0 = np.stack([-hm.eq_grad("psi", R, Z)[1] / R, hm.eq_at("F", R, Z) / R, hm.eq_grad("psi", R, Z)[0] / R], -1)
        B1 = np.stack([re("B_R"), re("B_phi"), re("B_Z")], -1)
        E1 = np.stack([re("E_R"), re("E_phi"), re("E_Z")], -1)
        gR, gZ = hm.amp_grad("B_par", R, Z)
        gB1 = np.stack([(gR * ph).real, (1j * ntor * hm.amp_at("B_par", R, Z) * ph).real / R, (gZ * ph).real], -1)
        gB0 = np.stack([hm.eq_grad("Bm", R, Z)[0] + 0 * R, 0 * R, hm.eq_grad("Bm", R, Z)[1] + 0 * R], -1)
        Bc = B0 + B1
        Ec = E1 - (mu / q)[:, None] * (gB0 + gB1)
        c, s = np.cos(phi), np.sin(phi)
        cart = lambda a: np.stack([a[:, 0] * c - a[:, 1] * s, a[:, 0] * s + a[:, 1] * c, a[:, 2]], -1)
        Bx, Ex = cart(Bc), cart(Ec)
        h = q * dt / (2 * MASS)
        for p in range(n):
            vp = _boris_ts(v[p], Ex[p], Bx[p], h)
            got_v = np.array([st["vx"][p], st["vy"][p], st["vz"][p]])
            got_x = np.array([st["x"][p], st["y"][p], st["z"][p]])
            assert np.abs(got_v - vp).max() <= 1e-12 * np.abs(vp).max()
            assert np.abs(got_x - (np.array([mk["x"][p], mk["y"][p], mk["z"][p]]) + dt * vp)).max() <= 1e-12 * 4.0


# ---- Q1 --------------------------------------------------------------------------------------------------------------
def check_q1_second_derivatives_against_numpy_polyder(orc):
    """Random coefficient tables on a jitter-free 5 x 5 box: psi_RR, psi_RZ, psi_ZZ (poly_eval2), psi_R, psi_Z, F, F_R, F_Z,
    |B|, |B|_R, |B|_Z of the finite-element branch of gc_fields against numpy.polynomial (polyder applied once / twice to
    the coefficient matrix, polyval2d), with the chain rule d/dR = s_e d/dxi done here."""
    rng = np.random.default_rng(22)
    node, tri = rect_tri_mesh(5)
    ne = tri.shape[0]
    eqc = rng.normal(size=(ne, 4, 21))
    m = orc.Mesh(node, tri, eqc)
    npts = 300
    R, Z = rng.uniform(1.95, 4.05, npts), rng.uniform(-1.05, 1.05, npts)
    elem, out = orc.gc_fields(R, Z, mesh=m)
    assert (elem >= 0).all() and np.array_equal(elem, m.locate(R, Z))
    cen, s = element_frames(node, tri)
    ex = monomial_exponents()

    def mat(c21):
        Cm = np.zeros((6, 6))
        Cm[ex[:, 0], ex[:, 1]] = c21
        return Cm
    for p in range(npts):
        e = elem[p]
        xi, eta, se = (R[p] - cen[e, 0]) * s[e], (Z[p] - cen[e, 1]) * s[e], s[e]
        d = lambda Cm, i, j: npoly.polyval2d(xi, eta, npoly.polyder(npoly.polyder(Cm, i, axis=0), j, axis=1) if (i or j) else Cm)
        P, Bm, F = mat(eqc[e, 0]), mat(eqc[e, 1]), mat(eqc[e, 2])
        exp = [d(P, 1, 0) * se, d(P, 0, 1) * se, d(P, 2, 0) * se * se, d(P, 1, 1) * se * se, d(P, 0, 2) * se * se,
               d(F, 0, 0), d(F, 1, 0) * se, d(F, 0, 1) * se, d(Bm, 0, 0), d(Bm, 1, 0) * se, d(Bm, 0, 1) * se]
        scale = np.abs(eqc[e]).max() * se * se
        assert np.abs(out[p] - exp).max() <= 1e-12 * max(1.0, scale), (p, out[p], exp)


# ---- Q2 --------------------------------------------------------------------------------------------------------------
def _g1_residuals(orc, nx, n=400, seed=23):
    """Largest relative dE/dt and dP_phi/dt of the oracle's guiding-centre right-hand side on the finite-element tables of
    the analytic equilibrium (nx x nx mesh); grad|B| and grad(R b_phi) from the ANALYTIC equilibrium by central differences."""
    node, tri = rect_tri_mesh(nx)
    m = orc.Mesh(node, tri, eq_tables(EQ, node, tri))
    sp = orc.species(CHARGE, MASS)
    rng = np.random.Generator(np.random.PCG64(seed))
    R, Z = rng.uniform(2.3, 3.7, n), rng.uniform(-0.6, 0.6, n)
    vpar, mu = rng.uniform(-1.0, 1.0, n), rng.uniform(0.0, 0.01, n)
    out = orc.gc_rhs(sp, R, Z, vpar, mu, mesh=m)
    dR, dZ, dv = out[:, 0], out[:, 2], out[:, 3]
    h = 1e-5
    Bm = lambda r, z: np.sqrt(sum(b ** 2 for b in EQ.B_cyl(r, z)))
    bphiR = lambda r, z: r * EQ.B_cyl(r, z)[1] / Bm(r, z)
    gBR, gBZ = (Bm(R + h, Z) - Bm(R - h, Z)) / (2 * h), (Bm(R, Z + h) - Bm(R, Z - h)) / (2 * h)
    dE = MASS * vpar * dv + mu * (gBR * dR + gBZ * dZ)
    sE = np.abs(MASS * vpar * dv) + np.abs(mu * gBR * dR) + np.abs(mu * gBZ * dZ) + 1e-12
    pR, pZ = EQ.grad_psi(R, Z)
    gR, gZ = (bphiR(R + h, Z) - bphiR(R - h, Z)) / (2 * h), (bphiR(R, Z + h) - bphiR(R, Z - h)) / (2 * h)
    dP = CHARGE * (pR * dR + pZ * dZ) + MASS * dv * bphiR(R, Z) + MASS * vpar * (gR * dR + gZ * dZ)
    sP = np.abs(CHARGE * pR * dR) + np.abs(CHARGE * pZ * dZ) + np.abs(MASS * dv * bphiR(R, Z)) + 1e-12
    return (np.abs(dE) / sE).max(), (np.abs(dP) / sP).max()


def check_q2_fe_backend_rhs_conserves_invariants(orc):
    """Pin G1 on the finite-element back-end (poly_eval2 and the FE branch of gc_fields inside gc_rhs): the residuals are
    the fit error of the quintic tables (second derivatives: O(h^4)) and shrink with the mesh."""
    e32, p32 = _g1_residuals(orc, 32)
    e64, p64 = _g1_residuals(orc, 64)
    assert e32 < 2e-6 and p32 < 5e-6, (e32, p32)          # measured 6.4e-7, 1.4e-6 (16^2: 1.2e-5, 2.2e-5)
    assert e64 < 0.1 * e32 and p64 < 0.1 * p32, (e32, e64, p32, p64)   # measured 9.0e-9, 5.1e-8


CHECKS = {"m1": check_m1_vpar_B1_over_B0, "m2": check_m2_mirror_force_of_B1par, "m3": check_m3_mu_dB1par_dt,
          "n1": check_n1_mode1_push_uses_total_fields, "q1": check_q1_second_derivatives_against_numpy_polyder,
          "q2": check_q2_fe_backend_rhs_conserves_invariants}


@pytest.mark.parametrize("name", sorted(CHECKS))
def test_pin(orc, name):
    CHECKS[name](orc)
