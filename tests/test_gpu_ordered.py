"""GPU tests of the ordered pipeline (work items, record gather, fused histogram), of the element search on an
unstructured mesh and on adversarial points, of several toroidal modes, and of the full-size bench configuration on
sampled markers.  All comparisons are against the CPU oracle on the same seeded inputs, through the C ABI."""
import dataclasses

import numpy as np
import pytest

import synth
from synth import configs as sc
from synth.mesh import eq_tables, pert_tables, perturbed_tri_mesh
from gpu_helpers import KEYS, g16_errors, make_pusher, oracle_of, oracle_push, take

pytestmark = pytest.mark.gpu

TOL_STEP = 1.0e-12


def _unstructured(idx=1, nx=24, n_markers=5000 + 11, two_modes=False):
    """Config idx's physics on a jittered, randomly triangulated, shuffled mesh (a generic unstructured input)."""
    w = synth.make_config(idx, n_markers=n_markers, nx=nx)
    node_RZ, tri = perturbed_tri_mesh(nx, sc.BOX, jitter=0.3, seed=11)
    L = {1: 0.3, 3: 0.4}.get(idx)
    eqc = eq_tables(w.eq, node_RZ, tri, sc._kappa_fn(w.eq, L))
    perts = list(w.perts)
    if two_modes:   # a second toroidal mode with NEGATIVE n and another frequency
        p2 = synth.Perturbation(w.eq, n=-2, omega=0.013, harmonics=[synth.Harmonic(3, sc.gaussian_radial(3, 0.45, 0.1))])
        perts.append(p2.normalise(0.7e-4 * w.eq.B0))
    pc, n_tor, omega = pert_tables(perts, node_RZ, tri)
    return dataclasses.replace(w, node_RZ=node_RZ, tri=tri, eq_coef=eqc, pert_coef=pc, n_tor=n_tor, omega=omega, perts=perts)


def test_element_search_on_unstructured_mesh_and_adversarial_points():
    """The fp32 fast search + exact fallback must return the oracle's element (rule G11) everywhere: random points,
    points ON nodes and edges, points one ulp to either side of them, points outside the mesh."""
    w = _unstructured()
    mesh, _ = oracle_of(w)
    rng = np.random.Generator(np.random.PCG64(5))
    P = w.node_RZ[w.tri]                                    # [ne, 3, 2]
    nodes = w.node_RZ
    mid = 0.5 * (P[:, [0, 1, 2]] + P[:, [1, 2, 0]]).reshape(-1, 2)
    third = (P[:, [0, 1, 2]] * (1.0 / 3.0) + P[:, [1, 2, 0]] * (2.0 / 3.0)).reshape(-1, 2)
    cen = P.mean(axis=1)
    pts = np.concatenate([nodes, mid, third, cen, np.stack([rng.uniform(1.85, 4.15, 30000), rng.uniform(-1.15, 1.15, 30000)], 1)])
    pts = np.concatenate([pts, np.nextafter(pts, np.inf), np.nextafter(pts, -np.inf),
                          np.stack([np.nextafter(pts[:, 0], np.inf), np.nextafter(pts[:, 1], -np.inf)], 1)])
    R, Z = np.ascontiguousarray(pts[:, 0]), np.ascontiguousarray(pts[:, 1])
    e_ref = mesh.locate(R, Z)
    p = make_pusher(w, verify=False)
    e_gpu, _ = p.eval_fields(R, np.zeros_like(R), Z, 0.0)
    assert np.array_equal(e_gpu, e_ref), int((e_gpu != e_ref).sum())
    assert (e_ref < 0).sum() > 100 and (e_ref >= 0).sum() > 0.9 * R.size


@pytest.mark.parametrize("two_modes", [False, True])
def test_ordered_pipeline_parity_on_unstructured_mesh(two_modes):
    """Several steps of the element-ordered path (sort_interval = 1: work items, record gather, fused histogram,
    re-ordering every step) on an unstructured mesh, one and two toroidal modes (one with n < 0), against the oracle;
    and the same bits as the SoA path (sort_interval = 0) and as sort_interval = 3."""
    w = _unstructured(two_modes=two_modes)
    mesh, sp = oracle_of(w)
    nsteps = 6
    ref, e_ref, _ = oracle_push(mesh, sp, w.markers, nsteps, w.dt)
    _, e_next, _ = oracle_push(mesh, sp, w.markers, nsteps + 1, w.dt)     # element of x_nsteps is what step nsteps+1 finds
    res = {}
    for si in (0, 1, 3):
        p = make_pusher(w, verify=True, sort_interval=si)
        p.push(nsteps, w.dt)
        got, elem, ids = p.state()
        assert np.array_equal(np.sort(ids), np.arange(w.n_markers))
        res[si] = got
        live = e_ref >= 0
        wrms = np.sqrt(np.mean(ref["w"][live] ** 2))
        ex, ev, ew = g16_errors(take(got, live), take(ref, live), w_floor=wrms)
        assert max(ex.max(), ev.max(), ew.max()) <= 6 * TOL_STEP, (si, ex.max(), ev.max(), ew.max())
        assert np.array_equal(elem < 0, e_next < 0)
        assert np.array_equal(got["mu"], w.markers["mu"])
        if si:
            st = p.stats()
            assert st["n_sorts"] >= nsteps // si and st["steps_done"] == nsteps
    for si in (1, 3):
        for k in KEYS:
            assert np.array_equal(res[si][k], res[0][k]), (si, k)


@pytest.mark.parametrize("n", [1, 31, 32, 33, 64, 65, 129, 1000])
def test_ragged_item_sizes(n):
    """Work items of every fill: fewer markers than a warp, exactly one / two slots per lane, one past, a lone marker."""
    w = synth.make_config(3, n_markers=n, nx=16)
    mesh, sp = oracle_of(w)
    ref, e_ref, _ = oracle_push(mesh, sp, w.markers, 3, w.dt)
    p = make_pusher(w, verify=True, sort_interval=1)
    p.push(3, w.dt)
    got, _, ids = p.state()
    assert np.array_equal(np.sort(ids), np.arange(n))
    live = e_ref >= 0
    if live.any():
        wrms = np.sqrt(np.mean(ref["w"][live] ** 2))
        ex, ev, ew = g16_errors(take(got, live), take(ref, live), w_floor=wrms)
        assert max(ex.max(), ev.max(), ew.max()) <= 3 * TOL_STEP


def test_all_markers_in_one_element_and_all_lost():
    """Degenerate orderings: every marker in the same element (one long run of work items), and every marker lost."""
    w = synth.make_config(1, n_markers=700, nx=16)
    mk = {k: np.repeat(v[:1], 700) for k, v in w.markers.items()}
    mk["vx"] = mk["vx"] * np.linspace(0.5, 1.5, 700)             # same start point, different velocities
    w1 = dataclasses.replace(w, markers=mk)
    mesh, sp = oracle_of(w1)
    ref, e_ref, _ = oracle_push(mesh, sp, mk, 2, w.dt)
    p = make_pusher(w1, verify=True, sort_interval=1)
    p.push(2, w.dt)
    got, _, _ = p.state()
    ex, ev, ew = g16_errors(got, ref, w_floor=max(np.sqrt(np.mean(ref["w"] ** 2)), 1e-300))
    assert max(ex.max(), ev.max(), ew.max()) <= 2 * TOL_STEP
    lost = {k: v.copy() for k, v in w.markers.items()}
    lost["x"][:] = 50.0
    w2 = dataclasses.replace(w, markers=lost)
    p = make_pusher(w2, verify=False, sort_interval=1)
    p.push(4, w.dt)
    got, elem, ids = p.state()
    assert p.stats()["n_lost"] == 700 and (elem < 0).all()
    for k in KEYS:
        assert np.array_equal(got[k], lost[k])                   # frozen bit for bit (G12)


@pytest.mark.parametrize("mode", [0, 1, 2, 3])
def test_full_size_bench_configuration_on_sampled_markers(mode):
    """BASELINE.json configs[3] at full size (2^24 markers, 256 x 256 mesh) in the launch configuration bench.py times
    (sort_interval = 1, timing build; `--mode` 0 = the headline, 1 non-linear, 2 FLR through the ordered ring stream,
    3 non-linear + FLR): 3 steps, then every 8192-th marker against the oracle (markers are independent, so
    the oracle can compute the sample alone); ids are a permutation and mu is untouched."""
    w = synth.make_config(3)
    assert w.n_markers == 1 << 24 and w.n_elems == 131072
    nsteps = 3
    idx = np.arange(0, w.n_markers, 8192)
    sample = take(w.markers, idx)
    mesh, sp = oracle_of(w, mode=mode)
    ref, e_ref, _ = oracle_push(mesh, sp, sample, nsteps, w.dt)
    p = make_pusher(w, verify=False, sort_interval=1, mode=mode)
    p.push(nsteps, w.dt)
    got, elem, ids = p.state()
    assert np.array_equal(np.bincount(ids, minlength=w.n_markers), np.ones(w.n_markers, dtype=np.int64))
    assert np.array_equal(got["mu"], w.markers["mu"])
    live = e_ref >= 0
    gs = take(got, idx)
    wrms = np.sqrt(np.mean(ref["w"][live] ** 2))
    ex, ev, ew = g16_errors(take(gs, live), take(ref, live), w_floor=wrms)
    assert live.mean() > 0.99
    assert max(ex.max(), ev.max(), ew.max()) <= 3 * TOL_STEP, (ex.max(), ev.max(), ew.max())
    st = p.stats()
    assert st["steps_done"] == nsteps and st["n_markers"] == w.n_markers


def test_four_modes_including_axisymmetric_and_negative_n():
    """M3DK_MAX_MODES toroidal modes at once (n = 1, -2, 0, 5): the largest tile (11.5 KB, staged by TMA), the n = 0 phase
    (no complex power at all) and a negative n, linear and non-linear mode, ordered and SoA path, against the oracle."""
    w0 = synth.make_config(1, n_markers=3000 + 5, nx=24)
    eq = w0.eq
    perts = list(w0.perts)
    for n, m, rc, om in ((-2, 3, 0.45, 0.013), (0, 2, 0.35, 0.004), (5, 6, 0.3, 0.021)):
        p = synth.Perturbation(eq, n=n, omega=om, harmonics=[synth.Harmonic(m, sc.gaussian_radial(m, rc, 0.1))])
        perts.append(p.normalise(0.6e-4 * eq.B0))
    pc, n_tor, omega = pert_tables(perts, w0.node_RZ, w0.tri)
    w = dataclasses.replace(w0, pert_coef=pc, n_tor=n_tor, omega=omega, perts=perts)
    assert w.n_modes == 4 and 0 in list(n_tor) and min(n_tor) < 0
    for mode in (0, 1):
        mesh, sp = oracle_of(w, mode=mode)
        ref, e_ref, _ = oracle_push(mesh, sp, w.markers, 4, w.dt, t0=0.3)
        out = {}
        for si in (0, 1):
            p = make_pusher(w, verify=True, sort_interval=si, t0=0.3, mode=mode)
            p.push(4, w.dt)
            out[si], _, _ = p.state()
            live = e_ref >= 0
            wrms = np.sqrt(np.mean(ref["w"][live] ** 2))
            ex, ev, ew = g16_errors(take(out[si], live), take(ref, live), w_floor=wrms)
            assert max(ex.max(), ev.max(), ew.max()) <= 4 * TOL_STEP, (mode, si, ex.max(), ev.max(), ew.max())
        for k in KEYS:
            assert np.array_equal(out[0][k], out[1][k]), (mode, k)


@pytest.mark.parametrize("mode", [0, 1])
def test_async_push_variant_gives_the_same_bits(mode):
    """m3dk_set_push_variant(1): the asynchronously staged kernel (records, order entries, descriptors and search records
    requested one item ahead with cp.async; histogram without returned values, slots drawn by the re-ordering) must
    produce exactly the bits of the default kernel, lost markers and ragged items included, and the oracle's numbers."""
    w = _unstructured(n_markers=7000 + 3)
    mk = {k: v.copy() for k, v in w.markers.items()}
    mk["x"][:5] = 10.0                                      # lost from the start
    mk["vx"][5:40] = 30.0                                   # leave the mesh within a step or two
    w = dataclasses.replace(w, markers=mk)
    mesh, sp = oracle_of(w, mode=mode)
    nsteps = 7
    ref, e_ref, _ = oracle_push(mesh, sp, mk, nsteps, w.dt)
    out = {}
    for variant in (0, 1):
        p = make_pusher(w, verify=True, sort_interval=1, mode=mode)
        p.set_push_variant(variant)
        p.push(nsteps, w.dt)
        out[variant], elem, ids = p.state()
        assert np.array_equal(np.sort(ids), np.arange(w.n_markers))
        assert p.stats()["n_sorts"] >= nsteps
    for k in KEYS:
        assert np.array_equal(out[0][k], out[1][k]), k
    live = e_ref >= 0
    wrms = np.sqrt(np.mean(ref["w"][live] ** 2))
    ex, ev, ew = g16_errors(take(out[1], live), take(ref, live), w_floor=wrms)
    assert max(ex.max(), ev.max(), ew.max()) <= nsteps * TOL_STEP
