"""Pins of the oracle's moment deposition (Eqs. 17-18 with a delta-function shape;
readings G10, G22).  Checked against what the mathematics fixes, never against itself: sums that must equal totals
computed from the ANALYTIC equilibrium, the closed-form integrals of monomials over a triangle (Monte Carlo limit),
the orthogonality of the toroidal harmonics, linearity.  CPU only."""
from math import factorial

import numpy as np
import pytest

import synth
from synth.mesh import element_frames, monomial_exponents


@pytest.fixture(scope="module")
def wl():
    return synth.make_config(1, n_markers=20000, nx=16)


def _weights(w, seed=3):
    rng = np.random.Generator(np.random.PCG64(seed))
    mk = {k: v.copy() for k, v in w.markers.items()}
    mk["w"] = rng.normal(size=w.n_markers) * 1e-3
    return mk


def test_d1_unit_test_function_sums_to_the_analytic_totals(orc, wl):
    """nu_0 = 1, T_0 = 1: summing the k = 0, h = 0 entries over the elements must give sum_p w m v_par^2 and
    sum_p w mu |B|, here with v_par and |B| from the ANALYTIC equilibrium (the tables are quintic fits of it: agreement to
    the fit error pins b0, |B|0, the element assignment and the indexing of the two moments)."""
    mk = _weights(wl)
    rhs, lost = orc.deposit(orc.Mesh.of(wl), orc.species_of(wl), mk)
    assert lost == 0 and rhs.shape == (wl.n_elems, 2, 3, 21)
    eq = wl.eq
    R = np.hypot(mk["x"], mk["y"])
    BR, BP, BZ = eq.B_cyl(R, mk["z"])
    Bn = np.sqrt(BR ** 2 + BP ** 2 + BZ ** 2)
    c, s = mk["x"] / R, mk["y"] / R
    vpar = ((mk["vx"] * c + mk["vy"] * s) * BR + (-mk["vx"] * s + mk["vy"] * c) * BP + mk["vz"] * BZ) / Bn
    par, perp = mk["w"] * wl.mass * vpar ** 2, mk["w"] * mk["mu"] * Bn
    for mom, a in ((0, par), (1, perp)):
        tot, ref = rhs[:, mom, 0, 0].sum(), a.sum()
        assert abs(tot - ref) < 2e-5 * np.abs(a).sum(), (mom, tot, ref)
    # per element, and the first moments: sum_p a_p xi_p = s_e (sum_p a_p R_p - R_c sum_p a_p) (frame of reading G10)
    mesh = orc.Mesh.of(wl)
    elem = mesh.locate(R, mk["z"])
    cen, se = element_frames(wl.node_RZ, wl.tri)
    for mom, a in ((0, par), (1, perp)):
        s0 = np.bincount(elem, weights=a, minlength=wl.n_elems)
        sR = np.bincount(elem, weights=a * R, minlength=wl.n_elems)
        sZ = np.bincount(elem, weights=a * mk["z"], minlength=wl.n_elems)
        scale = np.abs(s0).max()
        assert np.abs(rhs[:, mom, 0, 0] - s0).max() < 2e-5 * scale
        assert np.abs(rhs[:, mom, 0, 1] - se * (sR - cen[:, 0] * s0)).max() < 2e-5 * scale       # k = 1: xi
        assert np.abs(rhs[:, mom, 0, 6] - se * (sZ - cen[:, 1] * s0)).max() < 2e-5 * scale       # k = 6: eta


def test_d2_monte_carlo_limit_is_the_integral_of_the_monomials_over_the_triangle(orc):
    """Markers uniform in ONE triangle, identical w mu |B| up to the slow variation of |B|: rhs_perp[k] / rhs_perp[0] ->
    (1/A) int_T xi^i eta^j dA, which has the closed form 2A a! b! c! / (a + b + c + 2)! in barycentric monomials; here the
    expectation is computed exactly by expanding xi^i eta^j in the vertices' local coordinates."""
    w = synth.make_config(1, n_markers=8, nx=8)
    e = 70
    P = w.node_RZ[w.tri[e]]
    rng = np.random.Generator(np.random.PCG64(12))
    N = 400000
    u = rng.random((N, 2))
    flip = u.sum(1) > 1
    u[flip] = 1 - u[flip]
    lam = np.stack([1 - u[:, 0] - u[:, 1], u[:, 0], u[:, 1]], 1)
    RZ = lam @ P
    phi = rng.uniform(0, 2 * np.pi, N)
    eqB = np.sqrt(sum(b ** 2 for b in w.eq.B_cyl(RZ[:, 0], RZ[:, 1])))
    mk = dict(x=RZ[:, 0] * np.cos(phi), y=RZ[:, 0] * np.sin(phi), z=RZ[:, 1], vx=np.zeros(N), vy=np.zeros(N), vz=np.zeros(N),
              mu=1.0 / eqB, w=np.ones(N))                   # w mu |B| = 1 for every marker (up to the fit error)
    rhs, lost = orc.deposit(orc.Mesh.of(w), orc.species_of(w), mk)
    assert lost == 0
    got = rhs[e, 1, 0] / N
    assert np.abs(rhs[np.arange(w.n_elems) != e]).max() == 0.0          # nothing leaks into other elements
    cen, se = element_frames(w.node_RZ, w.tri)
    V = (P - cen[e]) * se[e]                                            # vertices in the local frame: xi = sum_v lam_v V_v0

    def bary_integral(a, b, c):                                         # (1/A) int lam1^a lam2^b lam3^c dA
        return 2.0 * factorial(a) * factorial(b) * factorial(c) / factorial(a + b + c + 2)

    from itertools import product
    loc = (RZ - cen[e]) * se[e]                                          # the samples in the local frame (for the error bar only)
    for k, (i, j) in enumerate(monomial_exponents()):
        # expand (sum_v lam_v x_v)^i (sum_v lam_v y_v)^j by brute-force multinomial enumeration
        exp = 0.0
        for pick in product(range(3), repeat=int(i + j)):
            coef = np.prod([V[v, 0] for v in pick[:i]]) * np.prod([V[v, 1] for v in pick[i:]])
            exp += coef * bary_integral(pick.count(0), pick.count(1), pick.count(2))
        sigma = np.std(loc[:, 0] ** i * loc[:, 1] ** j) / np.sqrt(N)       # Monte Carlo standard error of this mean
        assert abs(got[k] - exp) < 6.0 * sigma + 3e-6 * max(abs(exp), 1e-3), (k, i, j, got[k], exp, sigma)


def test_d3_toroidal_harmonics_are_orthogonal_projections(orc):
    """Markers at ONE poloidal point, evenly spaced in phi, weights w = A + B cos(n phi) + C sin(n phi) (n the mode of the
    field set): T_0 picks N A, the cos harmonic N B / 2, the sin harmonic N C / 2 (discrete orthogonality)."""
    w = synth.make_config(3, n_markers=8, nx=8)             # n = 3
    n = int(w.n_tor[0])
    N = 360
    phi = 2 * np.pi * np.arange(N) / N
    R0, Z0 = 3.37, 0.21
    A, Bc, Cs = 0.7, -0.4, 0.25
    Bm = np.sqrt(sum(b ** 2 for b in w.eq.B_cyl(np.array([R0]), np.array([Z0]))))[0]
    mk = dict(x=R0 * np.cos(phi), y=R0 * np.sin(phi), z=np.full(N, Z0), vx=np.zeros(N), vy=np.zeros(N), vz=np.zeros(N),
              mu=np.full(N, 1.0 / Bm), w=A + Bc * np.cos(n * phi) + Cs * np.sin(n * phi))
    rhs, _ = orc.deposit(orc.Mesh.of(w), orc.species_of(w), mk)
    e = int(orc.Mesh.of(w).locate(np.array([R0]), np.array([Z0]))[0])
    got = rhs[e, 1, :, 0]
    assert np.allclose(got, [N * A, N * Bc / 2, N * Cs / 2], rtol=2e-5, atol=1e-9), got
    assert np.abs(rhs[e, 0]).max() == 0.0                   # v = 0: no parallel pressure


def test_d4_linear_in_w_and_independent_of_marker_order(orc, wl):
    mk = _weights(wl)
    mesh, sp = orc.Mesh.of(wl), orc.species_of(wl)
    a, _ = orc.deposit(mesh, sp, mk)
    mk2 = dict(mk)
    mk2["w"] = 3.0 * mk["w"]
    b, _ = orc.deposit(mesh, sp, mk2)
    assert np.abs(b - 3.0 * a).max() <= 1e-13 * np.abs(a).max()
    perm = np.random.Generator(np.random.PCG64(1)).permutation(wl.n_markers)
    c, _ = orc.deposit(mesh, sp, {k: v[perm] for k, v in mk.items()})
    assert np.abs(c - a).max() <= 1e-12 * np.abs(a).max()


def test_d5_b1par_term_of_eq16(orc):
    """flags bit 0: with w = 0 the perpendicular moment is sum_p mu_p B1par(x_p, t) (Eq. 16); B1par here from the ANALYTIC
    perturbation of the workload (the tables are quintic fits of it), at a time t != 0 so that the phase counts; the
    parallel moment and the w-terms are untouched."""
    w = synth.make_config(3, n_markers=20000, nx=32)
    mk = {k: v.copy() for k, v in w.markers.items()}
    mk["w"][:] = 0.0
    t = 7.3
    mesh, sp = orc.Mesh.of(w), orc.species_of(w)
    rhs, _ = orc.deposit(mesh, sp, mk, flags=1, t=t)
    off, _ = orc.deposit(mesh, sp, mk, flags=0, t=t)
    assert np.abs(off).max() == 0.0 and np.abs(rhs[:, 0]).max() == 0.0
    R, phi = np.hypot(mk["x"], mk["y"]), np.arctan2(mk["y"], mk["x"])
    pert = w.perts[0]
    amp = pert.amplitudes(R, mk["z"])                        # complex amplitudes in the table order, B_par last
    Bpar = amp[6] if isinstance(amp, (list, tuple)) else amp[..., 6]
    b1 = np.real(Bpar * np.exp(1j * (pert.n * phi - pert.omega * t)))
    ref = (mk["mu"] * b1).sum()
    got = rhs[:, 1, 0, 0].sum()
    assert abs(got - ref) < 2e-3 * np.abs(mk["mu"] * b1).sum(), (got, ref)
    # linear superposition with the w-term
    mk2 = dict(mk)
    mk2["w"] = np.full(w.n_markers, 0.25)
    both, _ = orc.deposit(mesh, sp, mk2, flags=1, t=t)
    wonly, _ = orc.deposit(mesh, sp, mk2, flags=0, t=t)
    assert np.abs(both[:, 1] - wonly[:, 1] - rhs[:, 1]).max() < 1e-12 * np.abs(both[:, 1]).max()


def test_d6_four_point_flr_deposition(orc):
    """flags bit 1: each marker deposits a quarter of its amplitude at each of its four gyro-ring points.
    One marker with a gyro-radius of a few elements: exactly the four elements that contain the ring points (ring from the
    pinned gyro_ring, elements from the pinned search) receive a quarter each; over many markers the total of the unit test
    function is unchanged and so is the total first moment in z (the ring is centred on the marker and z is linear)."""
    from synth.mesh import element_frames
    w = synth.make_config(1, n_markers=4000, nx=32)
    mesh, sp = orc.Mesh.of(w), orc.species_of(w)
    X = np.array([3.31, 0.0, 0.12])
    BR, BP, BZ = (float(np.asarray(b).reshape(-1)[0]) for b in w.eq.B_cyl(np.array([X[0]]), np.array([X[2]])))
    Bn = np.sqrt(BR ** 2 + BP ** 2 + BZ ** 2)
    mu = 0.02 * 4.0                                         # rho = sqrt(2 m mu / B) / q ~ 0.1: several elements of size 0.07
    one = dict(x=X[:1], y=X[1:2], z=X[2:], vx=np.zeros(1), vy=np.zeros(1), vz=np.zeros(1), mu=np.array([mu]), w=np.array([2.0]))
    rhs, _ = orc.deposit(mesh, sp, one, flags=2)
    pts = orc.gyro_ring(sp, X, mu, mesh=mesh)
    el = mesh.locate(np.hypot(pts[:, 0], pts[:, 1]), pts[:, 2])
    assert len(set(el.tolist())) == 4 and (el >= 0).all()
    a_perp = 2.0 * mu * Bn
    hit = np.flatnonzero(np.abs(rhs[:, 1, 0, 0]) > 0)
    assert sorted(hit.tolist()) == sorted(el.tolist())
    assert np.allclose(rhs[el, 1, 0, 0], 0.25 * a_perp, rtol=1e-5)
    # many markers: totals and the z-moment are those of the plain deposition
    rng = np.random.Generator(np.random.PCG64(3))
    mk = {k: v.copy() for k, v in w.markers.items()}
    mk["w"] = rng.normal(size=w.n_markers)
    plain, _ = orc.deposit(mesh, sp, mk, flags=0)
    flr, _ = orc.deposit(mesh, sp, mk, flags=2)
    cen, se = element_frames(w.node_RZ, w.tri)
    for mom in (0, 1):
        scale = np.abs(plain[:, mom, 0, 0]).sum()
        assert abs(flr[:, mom, 0, 0].sum() - plain[:, mom, 0, 0].sum()) < 1e-11 * scale
        zmom = lambda r: (r[:, mom, 0, 6] / se + cen[:, 1] * r[:, mom, 0, 0]).sum()
        assert abs(zmom(flr) - zmom(plain)) < 1e-10 * scale
    assert np.abs(flr[:, 1, 0, 0] - plain[:, 1, 0, 0]).max() > 1e-3 * np.abs(plain[:, 1, 0, 0]).max()   # but it is spread out


# ---- D7: d = w + B1*/B* replaces w (reading G25) ----------------------------------------------------------
def check_d7_jacobian_substitution(orc):
    """flags bit 2.  (a) Zero amplitude: the tables of pin D1 with the perturbation switched off give exactly the flags = 0
    result.  (b) Closed form on hand-made tables: psi0 = A R^2 / 2, F = 0, |B|0 = A is a uniform vertical field (curl b = 0,
    B*par = |B| = A) and B1par = eps A a uniform compression: d = w + eps, so the unit test function sums to
    sum_p (w_p + eps) m v_par^2 and sum_p (w_p + eps) mu A.  (c) With curl b: the quintic tables of the analytic equilibrium,
    B*par = |B| + (m v_par/q) b . curl b computed HERE from the analytic field by central differences; the extra deposit
    sum_p mu |B| B1par / B*par agrees to the fit error, and fails when the curl b term is dropped (it is 0.1 % of |B|)."""
    from handmade import HandMade
    from synth.configs import CHARGE, MASS
    rng = np.random.Generator(np.random.PCG64(12))
    # (a)
    w0 = synth.make_config(1, n_markers=3000, nx=16, amp=0.0)
    mk = _weights(w0)
    r0, _ = orc.deposit(orc.Mesh.of(w0), orc.species_of(w0), mk, 0)
    r4, _ = orc.deposit(orc.Mesh.of(w0), orc.species_of(w0), mk, 4)
    assert np.array_equal(r0, r4)
    # (b)
    A, eps, n = 0.8, 3.0e-3, 4000
    hm = HandMade(eq=dict(psi=(0.0, 0.0, 0.0, 0.5 * A), Bm=(A,), F=(0.0,), kappa=(0.0,)), pert=dict(B_par=(eps * A,)), n_tor=0)
    R, phi, Z = rng.uniform(2.0, 4.0, n), rng.uniform(-3, 3, n), rng.uniform(-1.0, 1.0, n)
    m2 = dict(x=R * np.cos(phi), y=R * np.sin(phi), z=Z, vx=rng.normal(size=n), vy=rng.normal(size=n), vz=rng.normal(size=n),
              mu=rng.uniform(0, 0.02, n), w=rng.normal(size=n) * 1e-3)
    sp = orc.species(CHARGE, MASS)
    rhs, lost = orc.deposit(hm.oracle_mesh(orc), sp, m2, 4)
    assert lost == 0
    par = ((m2["w"] + eps) * MASS * m2["vz"] ** 2).sum()           # b0 = +Z: v_par = vz
    perp = ((m2["w"] + eps) * m2["mu"] * A).sum()
    assert abs(rhs[:, 0, 0, 0].sum() - par) <= 1e-12 * np.abs((np.abs(m2["w"]) + eps) * MASS * m2["vz"] ** 2).sum()
    assert abs(rhs[:, 1, 0, 0].sum() - perp) <= 1e-12 * ((np.abs(m2["w"]) + eps) * m2["mu"] * A).sum()
    # (c)
    w1 = synth.make_config(3, n_markers=12000, nx=32, amp=1e-2)
    mesh, sp1 = orc.Mesh.of(w1), orc.species_of(w1)
    t = 0.4
    eq = w1.eq
    h = 2e-4

    def bhat(r, z):
        B = np.array(eq.B_cyl(r, z))
        return B / np.sqrt((B ** 2).sum(axis=0))

    def analytic(mk):
        R = np.hypot(mk["x"], mk["y"])
        _, fe = mesh.eval(R, np.arctan2(mk["y"], mk["x"]), mk["z"], t)
        b = bhat(R, mk["z"])
        dbR, dbZ = (bhat(R + h, mk["z"]) - bhat(R - h, mk["z"])) / (2 * h), (bhat(R, mk["z"] + h) - bhat(R, mk["z"] - h)) / (2 * h)
        curl = np.array([-dbZ[1], dbZ[0] - dbR[2], b[1] / R + dbR[1]])
        c, s = mk["x"] / R, mk["y"] / R
        vpar = (mk["vx"] * c + mk["vy"] * s) * b[0] + (-mk["vx"] * s + mk["vy"] * c) * b[1] + mk["vz"] * b[2]
        Babs = np.sqrt(sum(x ** 2 for x in eq.B_cyl(R, mk["z"])))
        return fe[:, 17], fe[:, 2], vpar, Babs, Babs + (w1.mass * vpar / w1.charge) * (b * curl).sum(axis=0)
    B1p, _, vpar, _, _ = analytic(w1.markers)
    # the markers on which the curl b correction (proportional to v_par) has one sign, so that it does not cancel in a sum
    keep = (B1p * vpar > 0) & (np.abs(vpar) > 0.3)
    mk = {k: v[keep].copy() for k, v in w1.markers.items()}        # w = 0: only the B1par / B*par part deposits
    B1p, Bm, vpar, Babs, Bstar = analytic(mk)
    rhs, _ = orc.deposit(mesh, sp1, mk, 4, t)
    for mom, amp in ((0, w1.mass * vpar ** 2), (1, mk["mu"] * Bm)):
        want, without_curl = (amp * B1p / Bstar).sum(), (amp * B1p / Babs).sum()
        got = rhs[:, mom, 0, 0].sum()
        assert abs(got - want) < 1e-5 * abs(want), (mom, got, want)
        assert abs(without_curl - want) > 1e-4 * abs(want), (mom, without_curl, want)      # the pin tells the two apart


def test_d7_jacobian_substitution(orc):
    check_d7_jacobian_substitution(orc)
