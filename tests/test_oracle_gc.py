"""Pins of the oracle's RK4 guiding-centre pusher (Eqs. 1-4; reading G24).  Against the
exact invariants of the continuous equations (which involve curl b), the order of the integrator, the paper's qualitative
claim of Fig. 1 (RK4 errors accumulate, slow-manifold Boris errors stay bounded) and the slow-manifold orbit itself.  CPU."""
import numpy as np
import pytest

import synth
from synth.configs import CHARGE, MASS

from helpers import gc_start, invariants, trend_and_swing

EQ = synth.CircularTokamak()
TG = EQ.gyro_period_axis(CHARGE, MASS)


def _bphi_R(R, Z):
    BR, BP, BZ = EQ.B_cyl(R, Z)
    return R * BP / np.sqrt(BR ** 2 + BP ** 2 + BZ ** 2)


def test_g1_rhs_conserves_energy_and_pphi_pointwise(orc):
    """dE/dt = m v_par dv_par/dt + mu grad|B| . dX/dt = 0 and dP_phi/dt = q grad psi . dX/dt + m d(v_par R b_phi)/dt = 0 hold
    identically for Eqs. (1)-(4) in an axisymmetric field -- the second only if curl b is right.  grad|B| and grad(R b_phi)
    are taken from the ANALYTIC equilibrium by central differences, independently of the oracle's own derivatives."""
    an = orc.analytic_of(EQ)
    sp = orc.species(CHARGE, MASS)
    rng = np.random.Generator(np.random.PCG64(5))
    n = 200
    R, Z = rng.uniform(2.3, 3.7, n), rng.uniform(-0.6, 0.6, n)
    vpar, mu = rng.uniform(-1.0, 1.0, n), rng.uniform(0.0, 0.01, n)
    out = orc.gc_rhs(sp, R, Z, vpar, mu, an=an)
    dR, dZ, dv = out[:, 0], out[:, 2], out[:, 3]
    h = 1e-5
    Bm = lambda r, z: np.sqrt(sum(b ** 2 for b in EQ.B_cyl(r, z)))
    gBR, gBZ = (Bm(R + h, Z) - Bm(R - h, Z)) / (2 * h), (Bm(R, Z + h) - Bm(R, Z - h)) / (2 * h)
    dE = MASS * vpar * dv + mu * (gBR * dR + gBZ * dZ)
    scaleE = np.abs(MASS * vpar * dv) + np.abs(mu * gBR * dR) + np.abs(mu * gBZ * dZ) + 1e-12
    assert (np.abs(dE) / scaleE).max() < 1e-7
    pR, pZ = EQ.grad_psi(R, Z)
    gR = (_bphi_R(R + h, Z) - _bphi_R(R - h, Z)) / (2 * h)
    gZ = (_bphi_R(R, Z + h) - _bphi_R(R, Z - h)) / (2 * h)
    dP = CHARGE * (pR * dR + pZ * dZ) + MASS * dv * _bphi_R(R, Z) + MASS * vpar * (gR * dR + gZ * dZ)
    scaleP = np.abs(CHARGE * pR * dR) + np.abs(CHARGE * pZ * dZ) + np.abs(MASS * dv * _bphi_R(R, Z)) + 1e-12
    assert (np.abs(dP) / scaleP).max() < 1e-6
    # and the leading behaviour: parallel streaming along B plus a vertical grad-B / curvature drift of order rho* v
    BR, BP, BZ = EQ.B_cyl(R, Z)
    assert np.allclose(out[:, 1], vpar * BP / Bm(R, Z), rtol=0.05, atol=2e-3)


def test_g2_fourth_order_convergence(orc):
    an = orc.analytic_of(EQ)
    sp = orc.species(CHARGE, MASS)
    s = gc_start(EQ, 0.3, 0.6, 0.0, CHARGE, MASS)
    R0 = np.hypot(s[0], s[1])
    Bm = float(np.sqrt(sum(np.asarray(b) ** 2 for b in EQ.B_cyl(np.array([R0]), np.array([s[2]])))).reshape(-1)[0])
    vpar0, mu = 0.6, MASS * (1 - 0.36) / (2 * Bm)
    T = 60.0

    def err(dt):
        n = int(round(T / dt))
        x, y, z, vp, e, lost = orc.gc_push(sp, [s[0]], [s[1]], [s[2]], [vpar0], [mu], n, T / n, an=an)
        R = np.hypot(x, y)
        B = np.sqrt(sum(np.asarray(b) ** 2 for b in EQ.B_cyl(R, z)))
        return abs(0.5 * MASS * vp[0] ** 2 + mu * B[0] - (0.5 * MASS * vpar0 ** 2 + mu * Bm))
    e1, e2, e3 = err(1.0), err(0.5), err(0.25)
    assert 10.0 < e1 / e2 < 24.0 and 10.0 < e2 / e3 < 24.0, (e1, e2, e3)


@pytest.mark.parametrize("lam", [0.8, 0.2])
def test_g3_rk4_errors_accumulate_while_boris_errors_stay_bounded(orc, lam):
    """PAPER.md:84, :92 (Fig. 1): with dt of several gyro-periods the energy error of the RK4 guiding-centre orbit
    accumulates (a secular trend that dominates its oscillation), that of the slow-manifold Boris orbit at a quarter of the
    step stays bounded (trend far below the oscillation)."""
    an = orc.analytic_of(EQ)
    sp = orc.species(CHARGE, MASS)
    dt = 5.0 * TG
    s = gc_start(EQ, 0.3, lam, dt / 4, CHARGE, MASS)
    R0 = np.hypot(s[0], s[1])
    Bm = float(np.sqrt(sum(np.asarray(b) ** 2 for b in EQ.B_cyl(np.array([R0]), np.array([s[2]])))).reshape(-1)[0])
    mu = MASS * (1 - lam ** 2) / (2 * Bm)
    nblk, per = 60, 200
    x, y, z, vp = np.array([s[0]]), np.array([s[1]]), np.array([s[2]]), np.array([lam])
    E = []
    for _ in range(nblk):
        x, y, z, vp, _, lost = orc.gc_push(sp, x, y, z, vp, [mu], per, dt, an=an)
        assert lost == 0
        B = np.sqrt(sum(np.asarray(b) ** 2 for b in EQ.B_cyl(np.hypot(x, y), z)))
        E.append(0.5 * MASS * vp[0] ** 2 + mu * B[0])
    E = np.array(E)
    t = np.arange(nblk) * per * dt
    drift = abs(E[-1] - E[0]) / abs(E[0])
    trend, swing = trend_and_swing(t, E)
    assert trend > 0.5 * swing and drift > 1e-8, (trend, swing, drift)          # RK4: the error is a trend
    tr, _ = orc.trace(sp, s, 4 * nblk * per, dt / 4, an=an, stride=4 * per)
    Eb, _ = invariants(orc, an, tr, s[6], CHARGE, MASS)
    trend_b, swing_b = trend_and_swing(tr[:, 7], Eb)
    assert trend_b < 0.2 * swing_b, (trend_b, swing_b)                           # Boris: bounded
    assert trend / swing > 3.0 * trend_b / swing_b


def test_g4_guiding_centre_orbit_lies_on_the_slow_manifold_orbit(orc):
    """The slow-manifold Boris marker follows the guiding-centre orbit: same radial excursion (banana /
    drift-surface shift) and the same poloidal transit time to a few per cent at rho* = 0.02."""
    an = orc.analytic_of(EQ)
    sp = orc.species(CHARGE, MASS)
    lam = 0.75
    dt = 0.5 * TG
    s = gc_start(EQ, 0.3, lam, dt, CHARGE, MASS)
    n = int(260 / dt)
    tr, _ = orc.trace(sp, s, n, dt, an=an, stride=8)
    rb = np.hypot(np.hypot(tr[:, 0], tr[:, 1]) - EQ.R0, tr[:, 2])
    thb = np.unwrap(np.arctan2(tr[:, 2], np.hypot(tr[:, 0], tr[:, 1]) - EQ.R0))
    R0 = np.hypot(s[0], s[1])
    Bm = float(np.sqrt(sum(np.asarray(b) ** 2 for b in EQ.B_cyl(np.array([R0]), np.array([s[2]])))).reshape(-1)[0])
    mu = s[6]
    BR, BP, BZ = (float(np.asarray(b).reshape(-1)[0]) for b in EQ.B_cyl(np.array([R0]), np.array([s[2]])))
    vpar0 = (s[3] * BR + s[4] * BP + s[5] * BZ) / Bm                              # phi = 0 at the start: (vx, vy, vz) = (vR, vphi, vZ)
    x, y, z, vp = np.array([s[0]]), np.array([s[1]]), np.array([s[2]]), np.array([vpar0])
    rg, thg = [], []
    for _ in range(len(tr)):
        rg.append(np.hypot(np.hypot(x[0], y[0]) - EQ.R0, z[0])); thg.append(np.arctan2(z[0], np.hypot(x[0], y[0]) - EQ.R0))
        x, y, z, vp, _, _ = orc.gc_push(sp, x, y, z, vp, [mu], 8, dt, an=an)
    rg, thg = np.array(rg), np.unwrap(np.array(thg))
    assert abs((rg.max() - rg.min()) - (rb.max() - rb.min())) < 0.1 * (rb.max() - rb.min()) + 2e-3
    assert abs(thg[-1] - thb[-1]) < 0.05 * abs(thb[-1])


def check_g5_phase_space_volume(orc):
    """Liouville's theorem of Eqs. (1)-(4) (the B*par of Eq. 4 is the phase-space Jacobian):
        (1/R) d(R B*par dR/dt)/dR + d(B*par dZ/dt)/dZ + d(B*par dv_par/dt)/dv_par = 0      (axisymmetric).
    B*par = |B| + (m v_par/q) b . curl b is computed HERE from the analytic equilibrium (curl b by central differences of
    b), the divergence by central differences of the oracle's right-hand side.  The conservation pins G1 cannot see B*par
    (it divides both equations alike, and (curl b)_phi enters nothing else); this one fails when any component of curl b or
    the form of B*par in the oracle is wrong."""
    an = orc.analytic_of(EQ)
    sp = orc.species(CHARGE, MASS)
    rng = np.random.Generator(np.random.PCG64(11))
    n = 120
    R, Z = rng.uniform(2.4, 3.6, n), rng.uniform(-0.5, 0.5, n)
    vpar, mu = rng.uniform(-1.0, 1.0, n), rng.uniform(0.001, 0.01, n)
    h = 2e-4

    def bhat(r, z):
        B = np.array(EQ.B_cyl(r, z))
        return B / np.sqrt((B ** 2).sum(axis=0))

    def Bspar(r, z, vp):
        b = bhat(r, z)
        dbR, dbZ = (bhat(r + h, z) - bhat(r - h, z)) / (2 * h), (bhat(r, z + h) - bhat(r, z - h)) / (2 * h)
        curl = np.array([-dbZ[1], dbZ[0] - dbR[2], b[1] / r + dbR[1]])       # axisymmetric curl in (R, phi, Z)
        Bm = np.sqrt(sum(c ** 2 for c in EQ.B_cyl(r, z)))
        return Bm + (MASS * vp / CHARGE) * (b * curl).sum(axis=0)

    def flux(r, z, vp):
        o = orc.gc_rhs(sp, r, z, vp, mu, an=an)
        J = Bspar(r, z, vp)
        return r * J * o[:, 0], J * o[:, 2], J * o[:, 3]
    d = 1e-3
    fR = (flux(R + d, Z, vpar)[0] - flux(R - d, Z, vpar)[0]) / (2 * d) / R
    fZ = (flux(R, Z + d, vpar)[1] - flux(R, Z - d, vpar)[1]) / (2 * d)
    fv = (flux(R, Z, vpar + d)[2] - flux(R, Z, vpar - d)[2]) / (2 * d)
    div = fR + fZ + fv
    scale = np.abs(fR) + np.abs(fZ) + np.abs(fv)
    assert (np.abs(div) / scale).max() < 2e-5, (np.abs(div) / scale).max()


def test_g5_phase_space_volume(orc):
    check_g5_phase_space_volume(orc)


def _zigzag(orc, sp, an, s, dt, n=200):
    tr, _ = orc.trace(sp, s, n, dt, an=an)
    Z = tr[:, 2]
    d2 = Z[2:] - 2 * Z[1:-1] + Z[:-2]
    return 0.5 * np.abs(np.diff(d2)).mean()                    # alternating part of the second difference (pin P15)


def check_g6_bootstrap(orc):
    """one RK4 guiding-centre step x_0 -> x_1 and v_{1/2} = (x_1 - x_0)/dt give the staggered state
    (x_1, v_{1/2}) of the slow manifold: a marker started that way shows none of the step-to-step zig-zag (pin P15's
    measure: the alternating part of the second difference of Z) that a marker started with v_par b alone shows, at
    dt of 4 gyro-periods and of 1 (measured: 300 times less; the drift-formula start of reading G20, whose velocity has the
    direction of b at x_0 instead of the chord's, zig-zags as much as v_par b).  The bootstrap velocity is v_par b plus
    drifts: within |v| dt kappa of v_par b(x_0), so a reversed difference (x_0 - x_1)/dt fails by 2 |v_par|."""
    an = orc.analytic_of(EQ)
    sp = orc.species(CHARGE, MASS)
    for dtg in (4.0, 1.0):
        for lam in (0.8, 0.3):
            dt = dtg * TG
            s0 = gc_start(EQ, 0.3, lam, dt, CHARGE, MASS)
            x0, mu = s0[0:3], s0[6]
            B = np.array(EQ.B_cart(np.array([x0[0]]), np.array([x0[1]]), np.array([x0[2]]))).ravel()
            vb = lam * B / np.linalg.norm(B)
            x1, y1, z1, vx, vy, vz, ok = orc.gc_bootstrap(sp, [x0[0]], [x0[1]], [x0[2]], [lam], [mu], dt, an=an)
            assert ok.all()
            s_boot = s0.copy()
            s_boot[0:3] = [x1[0], y1[0], z1[0]]
            s_boot[3:6] = [vx[0], vy[0], vz[0]]
            s_bare = s0.copy()
            s_bare[3:6] = vb
            zb, z0 = _zigzag(orc, sp, an, s_boot, dt), _zigzag(orc, sp, an, s_bare, dt)
            assert zb < 0.02 * z0, (dtg, lam, zb, z0)
            assert np.linalg.norm(s_boot[3:6] - vb) < 0.15 * dt / TG * 0.1 + 0.02, (s_boot[3:6], vb)
            assert np.allclose(np.array([x1[0], y1[0], z1[0]]) - x0, dt * s_boot[3:6], rtol=0, atol=1e-15)


def test_g6_bootstrap_puts_the_marker_on_the_slow_manifold(orc):
    check_g6_bootstrap(orc)


def check_g7_perturbed_guiding_centre_rhs(orc):
    """Eqs. (1)-(2) with the perturbed fields (sp.mode = 1; reading G26).
    (a) Closed forms on hand-made tables: psi0 = A R^2/2, F = 0, |B|0 = A is a uniform vertical field (b0 = Z-hat,
    curl b0 = 0), so B* = B0 + B1 and B*par = A + B1_Z; with one perturbed component at a time
        B1_R = eps:        dR/dt = v_par eps / A                      (v_par B1/B0 of Eq. 12)
        E1_phi = eps:      dR/dt = eps / A                            (E x B / B^2:  phi-hat x Z-hat = R-hat)
        E1_R = eps:        R dphi/dt = -eps / A                       (R-hat x Z-hat = -phi-hat)
        E1_Z = eps:        dv_par/dt = (q/m) eps                      (Eq. 2)
        B1par = eps Z:     dv_par/dt = -(mu/m) eps                    (mirror force of the perturbed field strength)
        B1par = eps R:     R dphi/dt = -(mu/q) eps / A                (grad-B drift: b x grad B / B = Z-hat x R-hat = +phi-hat, sign of -b x (-(mu/q) grad B))
    (b) An invariant: with a static electrostatic perturbation on the analytic back-end, H = m v_par^2/2 + mu |B| + q Phi is
    conserved pointwise by Eqs. (1)-(2): m v_par dv_par/dt + (mu grad|B| + q grad Phi) . dX/dt = 0 (gradients by central
    differences of the analytic fields)."""
    from handmade import HandMade
    A, eps = 0.8, 1e-3
    q, m = CHARGE, MASS
    R, Z, phi = np.array([3.1]), np.array([0.2]), np.array([0.6])
    vpar, mu = np.array([0.7]), np.array([0.004])
    eqd = dict(psi=(0.0, 0.0, 0.0, 0.5 * A), Bm=(A,), F=(0.0,), kappa=(0.0,))
    sp = orc.species(q, m, mode=1)

    def rhs(pert):
        hm = HandMade(eq=eqd, pert=pert, n_tor=0)
        return orc.gc_rhs(sp, R, Z, vpar, mu, mesh=hm.oracle_mesh(orc), phi=phi)[0]
    base = rhs(dict(B_R=(0.0,)))
    assert np.allclose(base, [0.0, 0.0, vpar[0], 0.0], atol=1e-15)           # streaming along the uniform field
    assert np.allclose(rhs(dict(B_R=(eps,))) - base, [vpar[0] * eps / A, 0, 0, 0], rtol=1e-12, atol=1e-18)
    assert np.allclose(rhs(dict(E_phi=(eps,))) - base, [eps / A, 0, 0, 0], rtol=1e-12, atol=1e-18)
    assert np.allclose(rhs(dict(E_R=(eps,))) - base, [0, -eps / A, 0, 0], rtol=1e-12, atol=1e-18)
    assert np.allclose(rhs(dict(E_Z=(eps,))) - base, [0, 0, 0, q / m * eps], rtol=1e-12, atol=1e-18)
    assert np.allclose(rhs(dict(B_par=(0.0, 0.0, eps))) - base, [0, 0, 0, -mu[0] / m * eps], rtol=1e-12, atol=1e-18)
    assert np.allclose(rhs(dict(B_par=(0.0, eps, 0.0))) - base, [0, mu[0] / q * eps / A, 0, 0], rtol=1e-12, atol=1e-18)
    # B1_Z changes the Jacobian B*par = A + eps but not the streaming velocity: v_par (A + eps) / (A + eps)
    assert np.allclose(rhs(dict(B_Z=(eps,))), base, rtol=1e-12, atol=1e-15)
    # (b)
    p = (2e-3, 0.3, 0.1, 0.0, 2, 3)
    an = orc.analytic_of(EQ, pA=p[0], prc=p[1], pwd=p[2], pomega=p[3], pn=p[4], pm=p[5])
    rng = np.random.Generator(np.random.PCG64(13))
    n = 150
    Rr, Zz, ph = rng.uniform(2.5, 3.5, n), rng.uniform(-0.45, 0.45, n), rng.uniform(-3, 3, n)
    vp, mm = rng.uniform(-1, 1, n), rng.uniform(0.001, 0.01, n)
    out = orc.gc_rhs(sp, Rr, Zz, vp, mm, an=an, phi=ph)
    h = 1e-5
    Bm = lambda r, z: np.sqrt(sum(b ** 2 for b in EQ.B_cyl(r, z)))

    def Phi(r, f, z):
        dR = r - EQ.R0
        rr, th = np.hypot(dR, z), np.arctan2(z, dR)
        return p[0] * np.exp(-((rr - p[1]) / p[2]) ** 2) * np.cos(p[4] * f - p[5] * th)
    gB = [(Bm(Rr + h, Zz) - Bm(Rr - h, Zz)) / (2 * h), 0 * Rr, (Bm(Rr, Zz + h) - Bm(Rr, Zz - h)) / (2 * h)]
    gP = [(Phi(Rr + h, ph, Zz) - Phi(Rr - h, ph, Zz)) / (2 * h), (Phi(Rr, ph + h, Zz) - Phi(Rr, ph - h, Zz)) / (2 * h) / Rr,
          (Phi(Rr, ph, Zz + h) - Phi(Rr, ph, Zz - h)) / (2 * h)]
    dH = m * vp * out[:, 3] + sum((mm * gB[k] + q * gP[k]) * out[:, k] for k in range(3))
    scale = np.abs(m * vp * out[:, 3]) + sum(np.abs((mm * gB[k] + q * gP[k]) * out[:, k]) for k in range(3)) + 1e-12
    assert (np.abs(dH) / scale).max() < 1e-6, (np.abs(dH) / scale).max()
    assert np.abs(q * gP[1] * out[:, 1]).max() > 1e-5                        # the potential does take part


def test_g7_perturbed_guiding_centre_rhs(orc):
    check_g7_perturbed_guiding_centre_rhs(orc)
