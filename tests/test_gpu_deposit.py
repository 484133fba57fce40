"""GPU parity of m3dk_deposit (Eqs. 17-18 with a delta-function shape) against the oracle's deposition
(pinned by tests/test_oracle_deposit.py), through the C ABI.  The GPU accumulates with fp64 atomics, so the order of
addition is free: entries are compared within 1e-12 of the sum of the ABSOLUTE contributions to that element and moment
(the monomials and toroidal factors are bounded by 1 in the element's frame)."""
import dataclasses

import numpy as np
import pytest

import oracle
import synth
from gpu_helpers import KEYS, make_pusher, oracle_of
from test_gpu_ordered import _unstructured

pytestmark = pytest.mark.gpu


def _check(w, markers, p, flags=0, t=0.0):
    mesh, sp = oracle_of(w)
    ref, lost = oracle.deposit(mesh, sp, markers, flags=flags, t=t)
    absw = dict(markers)
    absw["w"] = np.abs(markers["w"])
    scale, _ = oracle.deposit(mesh, sp, absw)
    S = scale[:, :, 0, 0][:, :, None, None]                     # sum of |a_p| per element and moment
    if flags & 1:                                               # + sum of |mu_p B1par| bounded by mu_p * max|B1par|
        zero = dict(markers)
        zero["w"] = np.zeros_like(markers["w"])
        b1, _ = oracle.deposit(mesh, sp, zero, flags=1, t=t)
        S = S + np.abs(b1).max() * 64.0 + np.abs(b1[:, :, 0, 0])[:, :, None, None] * 64.0
    got = p.deposit(flags=flags, t=t)
    assert got.shape == ref.shape
    err = np.abs(got - ref)
    assert (err <= 1e-12 * S + 1e-300).all(), float((err / (S + 1e-300)).max())
    assert np.abs(ref).max() > 0
    return got, ref, lost


@pytest.mark.parametrize("si", [0, 1])
def test_deposit_matches_oracle_after_a_push(si):
    """Weights produced by the push itself (config 3 shape), arrays in caller order (si = 0) and element order (si = 1)."""
    w = synth.make_config(3, n_markers=1 << 16, nx=32)
    p = make_pusher(w, verify=False, sort_interval=si)
    p.push(12, w.dt)
    raw, elem, ids = p.state(by_id=False)                       # exactly the arrays the library deposits from
    got, ref, lost = _check(w, raw, p)
    assert lost == int((elem < 0).sum())
    # order independence: the same markers deposited from id order give the same table within the tolerance
    by_id, _, _ = p.state()
    ref2, _ = oracle.deposit(*oracle_of(w), by_id)
    assert np.abs(ref2 - ref).max() <= 1e-12 * np.abs(ref).max() * 50


def test_deposit_two_modes_unstructured_mesh_with_lost_markers():
    w0 = _unstructured(two_modes=True)
    rng = np.random.Generator(np.random.PCG64(4))
    mk = {k: v.copy() for k, v in w0.markers.items()}
    mk["w"] = rng.normal(size=w0.n_markers)
    mk["x"][:11] = 40.0                                         # outside the mesh: must deposit nothing
    w = dataclasses.replace(w0, markers=mk)
    p = make_pusher(w, verify=True)
    got, ref, lost = _check(w, mk, p)
    assert lost == 11 and got.shape[2] == 5                     # harmonics 1, cos / sin of both modes
    # the rows of the lost markers' would-be elements are not polluted: total of the unit test function
    live = np.ones(w.n_markers, dtype=bool)
    live[:11] = False
    assert abs(got[:, 1, 0, 0].sum() - ref[:, 1, 0, 0].sum()) <= 1e-9 * np.abs(mk["w"][live]).sum()


def test_deposit_equilibrium_only_and_empty():
    w = synth.make_config(0, n_markers=4096, nx=32)             # no modes: a single harmonic
    mk = {k: v.copy() for k, v in w.markers.items()}
    mk["w"] = np.linspace(-1.0, 1.0, w.n_markers)
    p = make_pusher(dataclasses.replace(w, markers=mk), verify=False)
    got, ref, _ = _check(w, mk, p)
    assert got.shape == (w.n_elems, 2, 1, 21)
    empty = {k: np.zeros(0) for k in KEYS}
    p2 = make_pusher(dataclasses.replace(w, markers=empty), verify=False)
    assert np.abs(p2.deposit()).max() == 0.0


def test_deposit_with_b1par_term_of_eq16():
    """flags = M3DK_DEPOSIT_B1PAR at t != 0, one and two modes: the perpendicular moment gains mu B1par(x, t)."""
    for two in (False, True):
        w = _unstructured(two_modes=two)
        rng = np.random.Generator(np.random.PCG64(9))
        mk = {k: v.copy() for k, v in w.markers.items()}
        mk["w"] = rng.normal(size=w.n_markers) * 1e-4
        p = make_pusher(dataclasses.replace(w, markers=mk), verify=True)
        got, ref, _ = _check(w, mk, p, flags=1, t=5.7)
        off = p.deposit(flags=0, t=5.7)
        assert np.abs(got[:, 1] - off[:, 1]).max() > 1e-3 * np.abs(off[:, 1]).max()      # the term is there
        assert np.abs(got[:, 0] - off[:, 0]).max() <= 1e-12 * np.abs(off[:, 0]).max()     # parallel moment untouched


def test_deposit_flr_four_point():
    """flags = M3DK_DEPOSIT_FLR (with and without the B1par term): a quarter of every amplitude at each gyro-ring point."""
    w = _unstructured(two_modes=True)
    rng = np.random.Generator(np.random.PCG64(10))
    mk = {k: v.copy() for k, v in w.markers.items()}
    mk["w"] = rng.normal(size=w.n_markers) * 1e-4
    mk["mu"] = mk["mu"] * 4.0                                   # rings of a few elements; near the edge some points fall outside
    p = make_pusher(dataclasses.replace(w, markers=mk), verify=True)
    mesh, sp = oracle_of(w)
    for ring_stream in (False, True):               # every lane loops over its ring's elements / ordered ring items
        if ring_stream:
            p.set_flr_workspace()
        for flags in (2, 3, 7):
            ref, _ = oracle.deposit(mesh, sp, mk, flags=flags, t=2.1)
            got = p.deposit(flags=flags, t=2.1)
            S = np.abs(ref).max()
            assert np.abs(got - ref).max() <= 1e-11 * S, (ring_stream, flags, float(np.abs(got - ref).max() / S))
    plain = p.deposit(flags=0)
    assert np.abs(got[:, 1, 0, 0] - plain[:, 1, 0, 0]).max() > 1e-3 * np.abs(plain[:, 1, 0, 0]).max()


def test_deposit_without_sort_workspace_uses_the_callers_arrays():
    """No sort workspace registered: plain and FLR deposition fall back to the any-order kernels; same tables."""
    import paper_2107_13663_b200 as m3dk
    w = _unstructured(two_modes=False)
    rng = np.random.Generator(np.random.PCG64(11))
    mk = {k: v.copy() for k, v in w.markers.items()}
    mk["w"] = rng.normal(size=w.n_markers)
    p = m3dk.Pusher(device=0, verify=True)
    p.fields_create(w.node_RZ, w.tri, w.eq_coef, w.n_tor, w.omega, w.pert_coef)
    p.particles_init(mk, w.charge, w.mass, w.f0, with_sort_workspace=False)
    mesh, sp = oracle_of(w)
    for flags in (0, 1, 2):
        ref, _ = oracle.deposit(mesh, sp, mk, flags=flags, t=1.3)
        got = p.deposit(flags=flags, t=1.3)
        assert np.abs(got - ref).max() <= 1e-11 * np.abs(ref).max(), flags


@pytest.mark.parametrize("flags", [4, 5, 6, 7])
@pytest.mark.parametrize("si", [0, 1])
def test_deposit_with_the_jacobian_substitution(flags, si):
    """flags bit 2 (M3DK_DEPOSIT_BSTAR): d = w + B1par/B*par replaces w, alone and together with the B1par
    term of Eq. (16) and the 4-point FLR deposition; element-ordered (items kernel) and caller order."""
    w = synth.make_config(3, n_markers=30000 + 11, nx=32, amp=1e-2)
    rng = np.random.Generator(np.random.PCG64(9))
    mk = {k: v.copy() for k, v in w.markers.items()}
    mk["w"] = rng.normal(size=w.n_markers) * 1e-2
    w = dataclasses.replace(w, markers=mk)
    p = make_pusher(w, verify=True, sort_interval=si)
    if si:
        p.sort()
    raw, elem, ids = p.state(by_id=False)
    mesh, sp = oracle_of(w)
    t = 0.7
    ref, lost = oracle.deposit(mesh, sp, raw, flags=flags, t=t)
    absw = dict(raw)
    absw["w"] = np.abs(raw["w"]) + 2e-2                        # |w| + a bound of |B1par / B*par| (amplitude 1e-2 B0)
    scale, _ = oracle.deposit(mesh, sp, absw, flags=flags & 2)
    S = np.abs(scale[:, :, 0, 0])[:, :, None, None] + np.abs(scale).max() * 1e-3
    got = p.deposit(flags=flags, t=t)
    err = np.abs(got - ref)
    assert (err <= 1e-11 * S).all(), float((err / S).max())
    base, _ = oracle.deposit(mesh, sp, raw, flags=flags & 3, t=t)
    assert np.abs(ref - base).max() > 1e-4 * np.abs(base).max()          # the substitution does change the table


@pytest.mark.parametrize("flags", [0, 1, 5, 3, 7])
def test_full_size_deposit_on_sampled_elements(flags):
    """BASELINE.json configs[3] at full size (2^24 markers, 256 x 256 mesh) in the launch configuration
    `bench.py --deposit --deposit-flags F` times (sort workspace, FLR workspace for the 4-point deposition, timing build).
    The oracle computes the rows of a sample of elements: it deposits only the markers that can reach a sampled element
    (position inside the element's bounding box, widened by more than the largest gyro-radius when the ring is
    deposited), chosen from the INPUT positions; the rows of the sampled elements are then complete and are compared."""
    from synth.configs import CHARGE, MASS
    w = synth.make_config(3)
    assert w.n_markers == 1 << 24 and w.n_elems == 131072
    rng = np.random.Generator(np.random.PCG64(2024))
    mk = {k: v.copy() for k, v in w.markers.items()}
    mk["w"] = rng.normal(size=w.n_markers) * 1e-3
    R, Z = np.hypot(mk["x"], mk["y"]), mk["z"]
    flr = bool(flags & 2)
    margin = 0.0
    if flr:
        # textbook gyro-radius m v_perp / (|q| B) with v_perp^2 = 2 mu B / m: only to size the margin generously
        B = w.eq.Bmag(R, Z)
        rho = np.sqrt(2.0 * mk["mu"] * B / MASS) * MASS / (abs(CHARGE) * B)
        margin = 1.5 * float(rho.max()) + 1e-3
        assert margin < 0.1
    n_sample = 24 if flr else 192
    elems = np.linspace(1000, w.n_elems - 1000, n_sample).astype(np.int64)
    # keep the sampled elements that hold markers at all (the mesh box is larger than the plasma)
    tri = w.node_RZ[w.tri[elems]]                                # [n_sample][3][2]
    lo, hi = tri.min(axis=1) - margin, tri.max(axis=1) + margin
    sel = np.zeros(w.n_markers, dtype=bool)
    for k in range(n_sample):
        sel |= (R >= lo[k, 0]) & (R <= hi[k, 0]) & (Z >= lo[k, 1]) & (Z <= hi[k, 1])
    sub = {k: np.ascontiguousarray(v[sel]) for k, v in mk.items()}
    assert 10_000 < sub["x"].size < 4_000_000
    mesh, sp = oracle_of(w)
    t = 0.9
    ref, _ = oracle.deposit(mesh, sp, sub, flags=flags, t=t)
    absw = dict(sub)
    absw["w"] = np.abs(sub["w"]) + (1e-3 if flags & 4 else 0.0)  # + a bound of |B1par / B*par| (amplitude 1e-4 B0)
    scale, _ = oracle.deposit(mesh, sp, absw, flags=flags & 2)
    S = np.abs(scale[:, :, 0, 0])[:, :, None, None] + np.abs(scale).max() * 1e-3
    p = make_pusher(dataclasses.replace(w, markers=mk), verify=False, sort_interval=1)
    if flr:
        p.set_flr_workspace()
    got = p.deposit(flags=flags, t=t)
    assert got.shape == (w.n_elems, 2, 3, 21)
    err = np.abs(got[elems] - ref[elems])
    assert (err <= 1e-11 * S[elems]).all(), float((err / S[elems]).max())
    assert (np.abs(ref[elems]).max(axis=(1, 2, 3)) > 0).sum() > n_sample // 3       # the sample does hold markers
    # nothing is lost or duplicated on the way through the ordering: the unit test function sums to sum(d)
    if flags == 0:
        tot = got[:, 1, 0, 0].sum()
        refsum = float(np.sum(mk["w"] * mk["mu"] * w.eq.Bmag(R, Z)))
        assert abs(tot - refsum) <= 1e-5 * float(np.sum(np.abs(mk["w"]) * mk["mu"] * w.eq.Bmag(R, Z)))
