"""Pins of the oracle's non-linear trajectory mode (reading G21).

Mode 1: the marker is pushed in the TOTAL fields, B = B0 + B1 and E-dagger = E1 - (mu/q) grad(|B|0 + B1par), and the factor
(1 - w) of Eq. (8) is kept.  None of these checks compares the oracle with itself: an invariant of the equations of motion,
a closed form of the weight ODE, and the two limits (zero and small amplitude) in which the mode must reduce to the pinned
linear mode.  CPU only."""
import numpy as np
import pytest

import synth
from synth.configs import CHARGE, MASS

from helpers import gc_start, invariants

EQ = synth.CircularTokamak()
TG = EQ.gyro_period_axis(CHARGE, MASS)


def _phi_es(eq, p, x, y, z, t):
    pA, prc, pwd, pom, pn, pm = p
    R = np.hypot(x, y)
    dR = R - eq.R0
    r, th = np.hypot(dR, z), np.arctan2(z, dR)
    return pA * np.exp(-((r - prc) / pwd) ** 2) * np.cos(pn * np.arctan2(y, x) - pm * th - pom * t)


def test_p16_zero_amplitude_is_the_linear_mode_bit_for_bit(orc):
    """No perturbation: total fields = equilibrium fields and w stays 0, so both modes must give the same bits."""
    w = synth.make_config(1, n_markers=256, nx=16, amp=0.0)
    mesh = orc.Mesh.of(w)
    a, _, _ = orc.push_fe(mesh, orc.species_of(w, mode=0), w.markers, 50, w.dt)
    b, _, _ = orc.push_fe(mesh, orc.species_of(w, mode=1), w.markers, 50, w.dt)
    for k in a:
        assert np.array_equal(a[k], b[k]), k
    assert (b["w"] == 0.0).all()


@pytest.mark.parametrize("lam", [0.7, 0.2])
def test_p17_static_potential_total_energy_is_conserved(orc, lam):
    """omega = 0, electrostatic perturbation: the non-linear trajectory is the motion in the static Hamiltonian
    H = m v^2 / 2 + mu |B0| + q Phi, which the slow-manifold Boris scheme keeps bounded like the unperturbed energy
    (PAPER.md:84, :92).  So the swing of H must stay at the level of the unperturbed run, far below the swing of q Phi
    itself; in the LINEAR mode the trajectory does not feel Phi and H wanders by the full q Phi."""
    p = (2.0e-3, 0.3, 0.1, 0.0, 2, 3)
    dt = 0.5 * TG
    s0 = gc_start(EQ, 0.3, lam, dt, CHARGE, MASS)
    n = int(400 / dt)
    swing = {}
    for name, pA, mode in (("free", 0.0, 1), ("nl", p[0], 1), ("lin", p[0], 0)):
        an = orc.analytic_of(EQ, kappa=0.0, pA=pA, prc=p[1], pwd=p[2], pomega=0.0, pn=p[4], pm=p[5])
        tr, _ = orc.trace(orc.species(CHARGE, MASS, 0, T=0.4, mode=mode), s0, n, dt, an=orc.analytic_of(EQ) if pA == 0 else an)
        E0, _ = invariants(orc, orc.analytic_of(EQ), tr, s0[6], CHARGE, MASS)
        H = E0 + CHARGE * _phi_es(EQ, (pA,) + p[1:], tr[:, 0], tr[:, 1], tr[:, 2], 0.0)
        swing[name] = (H.max() - H.min()) / abs(H.mean())
        if name == "nl":
            qphi = CHARGE * _phi_es(EQ, p, tr[:, 0], tr[:, 1], tr[:, 2], 0.0)
            swing["qphi"] = (qphi.max() - qphi.min()) / abs(H.mean())
            t = tr[:, 7]
            slope = np.polyfit(t, H, 1)[0] * (t[-1] - t[0]) / abs(H.mean())
            assert abs(slope) < 0.1 * swing["nl"] + 1e-9                # no secular drift
    assert swing["qphi"] > 20 * swing["free"]                           # the test can see the difference
    assert swing["nl"] < 3 * swing["free"] + 0.02 * swing["qphi"]       # H conserved as well as without Phi
    assert swing["lin"] > 0.5 * swing["qphi"]                           # the linear trajectory ignores Phi


@pytest.mark.parametrize("lam", [0.7, 0.2])
def test_p18_one_minus_w_closed_form(orc, lam):
    """Maxwellian, kappa = 0, static Phi: (1/f0) df0/dt = (q/T) dPhi/dt along the orbit, so Eq. (8) with (1 - w) kept is
    d ln(1 - w)/dt = (q/T) dPhi/dt and 1 - w(t) = exp((q/T) [Phi(x(t)) - Phi(x(0))]) along the PERTURBED orbit.  The
    explicit staggered update converges at first order in dt."""
    p = (2.0e-4, 0.3, 0.1, 0.0, 2, 3)                       # E1 ~ 2e-3 v B: a small push on the orbit ...
    T0 = 1.0e-3                                             # ... but q Phi / T ~ 0.2: a large weight
    an = orc.analytic_of(EQ, kappa=0.0, pA=p[0], prc=p[1], pwd=p[2], pomega=0.0, pn=p[4], pm=p[5])
    sp = orc.species(CHARGE, MASS, 0, T=T0, mode=1)
    errs, size = [], 0.0
    for dtg in (0.5, 0.25, 0.125):
        dt = dtg * TG
        s = gc_start(EQ, 0.3, lam, dt, CHARGE, MASS)
        tr, _ = orc.trace(sp, s, int(40 / dt), dt, an=an)
        xm = 0.5 * (tr[:-1, 0:3] + tr[1:, 0:3])            # x_{l+1/2}, where w_{l+1/2} lives
        x0 = s[0:3] - 0.5 * dt * s[3:6]
        dphi = _phi_es(EQ, p, xm[:, 0], xm[:, 1], xm[:, 2], 0.0) - _phi_es(EQ, p, x0[0], x0[1], x0[2], 0.0)
        ref = 1.0 - np.exp((CHARGE / T0) * dphi)
        errs.append(np.abs(tr[:-1, 6] - ref).max())
        size = np.abs(ref).max()
    assert size > 0.05                                      # a genuinely non-linear weight, not the small-w limit
    lin = np.abs(-(CHARGE / T0) * dphi - ref).max()         # what the linear formula would give
    assert errs[2] < 0.1 * lin                              # the (1 - w) factor is there
    assert 1.6 < errs[0] / errs[1] < 2.6 and 1.6 < errs[1] / errs[2] < 2.6      # first order


@pytest.mark.parametrize("idx", [1, 3])
def test_p19_small_amplitude_limit_is_the_linear_mode(orc, idx):
    """FE back-end, the synthetic electromagnetic perturbations: as the amplitude A -> 0 the non-linear result must
    approach the linear one, the difference of the weights scaling like A^2 (trajectory change O(A) times field O(A),
    and w^2 = O(A^2)) and the difference of the orbits like A."""
    d = {}
    for amp in (1e-4, 2e-4):
        w = synth.make_config(idx, n_markers=200, nx=16, amp=amp)
        mesh = orc.Mesh.of(w)
        a, ea, _ = orc.push_fe(mesh, orc.species_of(w, mode=0), w.markers, 60, w.dt)
        b, eb, _ = orc.push_fe(mesh, orc.species_of(w, mode=1), w.markers, 60, w.dt)
        ok = (ea >= 0) & (eb >= 0)
        d[amp] = (np.abs(b["w"] - a["w"])[ok], np.sqrt((b["x"] - a["x"]) ** 2 + (b["y"] - a["y"]) ** 2 + (b["z"] - a["z"]) ** 2)[ok],
                  np.sqrt(np.mean(a["w"][ok] ** 2)), ok)
    ok = d[1e-4][3] & d[2e-4][3]
    dw1, dx1, wr1, _ = d[1e-4]
    dw2, dx2, wr2, _ = d[2e-4]
    assert np.median(dw1) < 0.05 * wr1                      # close to the linear weights at this amplitude
    assert dx1.max() > 0                                    # but the orbits do feel the perturbation
    rw = np.sqrt(np.mean(dw2 ** 2)) / np.sqrt(np.mean(dw1 ** 2))
    rx = np.sqrt(np.mean(dx2 ** 2)) / np.sqrt(np.mean(dx1 ** 2))
    assert 3.0 < rw < 5.0, rw                               # ~ A^2
    assert 1.6 < rx < 2.5, rx                               # ~ A
