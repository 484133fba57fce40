"""GPU parity on BASELINE.json configs[4] (the scaling sweep: config-3 equilibrium and perturbation, dt in {1, 4, 16}
gyro-periods, sort interval in {1, 10, never}, up to 2^26 markers) and the long run of the element-ordered kernel.

dt = 16 gyro-periods moves a marker two length units per step (about 18 elements at 256^2): many markers
leave the mesh, the fp32 fast search falls back to the exact one more often; dt = 1 keeps most markers near their element.
Every comparison is against the CPU oracle on the same seeded inputs, through the C ABI; tolerances are BASELINE.json's.
"""
import dataclasses

import numpy as np
import pytest

import synth
from gpu_helpers import KEYS, g16_errors, make_pusher, oracle_of, oracle_push, take

pytestmark = pytest.mark.gpu

TOL_STEP = 1.0e-12
TOL_1000 = 1.0e-8
DTS = (1.0, 4.0, 16.0)
SORT_INTERVALS = (1, 10, 0)


@pytest.fixture(scope="module")
def small4():
    cache = {}

    def get(dtg):
        if dtg not in cache:
            cache[dtg] = synth.make_config(4, n_markers=6000 + 37, nx=64, dt_gyro=dtg)
        return cache[dtg]
    return get


@pytest.mark.parametrize("si", SORT_INTERVALS)
@pytest.mark.parametrize("dtg", DTS)
def test_config4_per_step_parity(small4, dtg, si):
    """Reading G16: restart the GPU from the oracle's state at steps 0, 1, 10, one step, <= 1e-12 in x, v, w; the cached
    element of the new position and n_lost are the oracle's (what its next step finds)."""
    w = small4(dtg)
    mesh, sp = oracle_of(w)
    p = make_pusher(w, verify=True, sort_interval=si)
    state = {k: w.markers[k].copy() for k in KEYS}
    done = 0
    for s in (0, 1, 10):
        if s > done:
            state, _, _ = oracle_push(mesh, sp, state, s - done, w.dt, t0=0.0, step0=done)
            done = s
        ref, e_ref, _ = oracle_push(mesh, sp, state, 1, w.dt, t0=0.0, step0=s)
        _, e_next, lost_next = oracle_push(mesh, sp, state, 2, w.dt, t0=0.0, step0=s)
        p.set_state(state)
        p.set_options(sort_interval=si, t0=s * w.dt)
        p.push(1, w.dt)
        got, e_gpu, ids = p.state()
        assert np.array_equal(np.sort(ids), np.arange(w.n_markers))
        live = e_ref >= 0
        assert np.array_equal(got["mu"], state["mu"])
        for k in KEYS:                                                    # lost markers are frozen bit for bit (G12)
            assert np.array_equal(got[k][~live], state[k][~live])
        wrms = np.sqrt(np.mean(ref["w"][live] ** 2))
        ex, ev, ew = g16_errors(take(got, live), take(ref, live), w_floor=wrms)
        assert max(ex.max(), ev.max(), ew.max()) <= TOL_STEP, (dtg, si, s, ex.max(), ev.max(), ew.max())
        assert np.array_equal(e_gpu < 0, e_next < 0)
        assert p.stats()["n_lost"] == lost_next


@pytest.mark.parametrize("si", SORT_INTERVALS)
def test_config4_markers_leaving_the_mesh_at_dt16(small4, si):
    """The loss regime of the sweep: markers loaded at the edge of the mesh (0.9 a < r < 1.09 a; the box ends at 1.1 a) with
    dt = 16 gyro-periods; after 11 chained steps about 9 % are outside.  Which markers are lost, and when, must be the
    oracle's: a lost marker keeps the state of its last live step (G12), so every marker is compared."""
    from synth.configs import CHARGE, MASS
    w0 = small4(16.0)
    mk = synth.load_markers(w0.eq, 3000 + 19, 4242, CHARGE, MASS, w0.dt, rmin=0.9, rmax=1.09, profile_L=None,
                            speed="slowing", v_c=0.3, pitch="uniform")
    w = dataclasses.replace(w0, markers=mk)
    mesh, sp = oracle_of(w)
    nsteps = 11
    ref, e_ref, lost = oracle_push(mesh, sp, mk, nsteps, w.dt)
    _, e_next, lost_next = oracle_push(mesh, sp, mk, nsteps + 1, w.dt)
    assert lost > 200
    p = make_pusher(w, verify=True, sort_interval=si)
    p.push(nsteps, w.dt)
    got, e_gpu, ids = p.state()
    assert np.array_equal(np.sort(ids), np.arange(w.n_markers))
    assert np.array_equal(e_gpu < 0, e_next < 0) and p.stats()["n_lost"] == lost_next
    wrms = np.sqrt(np.mean(ref["w"][e_ref >= 0] ** 2))
    ex, ev, ew = g16_errors(got, ref, w_floor=wrms)
    assert max(ex.max(), ev.max(), ew.max()) <= nsteps * TOL_STEP, (si, ex.max(), ev.max(), ew.max())


@pytest.mark.parametrize("dtg", DTS)
def test_config4_bitwise_independent_of_sort_interval(small4, dtg):
    """12 chained steps at every dt of the sweep: sort intervals 1 (element-ordered kernel every step), 10 (ordered kernel
    after each ordering, record kernel in between) and never (SoA kernel) give the same bits for every marker."""
    w = small4(dtg)
    res = {}
    for si in SORT_INTERVALS:
        p = make_pusher(w, verify=False, sort_interval=si)
        p.push(12, w.dt)
        res[si], elem, ids = p.state()
        assert np.array_equal(np.sort(ids), np.arange(w.n_markers))
    for si in (1, 10):
        for k in KEYS:
            assert np.array_equal(res[si][k], res[0][k]), (dtg, si, k)


@pytest.mark.parametrize("idx", [1, 3])
def test_1000_steps_through_the_element_ordered_kernel(idx):
    """The 1e-8 bar after 1000 steps on the non-chaotic orbits (readings G15, G16), linear delta-f, with sort_interval = 1:
    every one of the 1000 steps runs push_items_kernel (work items, staged tiles, fused histogram, re-ordering)."""
    w = synth.make_config(idx, n_markers=1024 + 13, nx={1: 32, 3: 64}[idx])
    mesh, sp = oracle_of(w)
    nsteps = 1000
    a, ea, _ = oracle_push(mesh, sp, w.markers, nsteps, w.dt)
    twin = {k: w.markers[k].copy() for k in KEYS}
    for k in ("x", "y", "z"):
        twin[k] *= (1.0 + 1.0e-13)
    b, eb, _ = oracle_push(mesh, sp, twin, nsteps, w.dt)
    ex, ev, _ = g16_errors(b, a)
    keep = (ex < 1e-9) & (ev < 1e-9) & (ea == eb) & (ea >= 0)
    assert keep.mean() > 0.5, keep.mean()
    p = make_pusher(w, verify=True, sort_interval=1)
    p.push(nsteps, w.dt)
    got, _, ids = p.state()
    assert np.array_equal(np.sort(ids), np.arange(w.n_markers))
    st = p.stats()
    assert st["steps_done"] == nsteps and st["n_sorts"] >= nsteps
    wrms = np.sqrt(np.mean(a["w"][keep] ** 2))
    ex, ev, ew = g16_errors(take(got, keep), take(a, keep), w_floor=wrms)
    assert max(ex.max(), ev.max(), ew.max()) <= TOL_1000, (ex.max(), ev.max(), ew.max(), keep.mean())


def test_config4_full_size_2p26_markers_on_sampled_markers():
    """The largest point of the sweep in the launch configuration bench.py --sweep times: 2^26 markers (4.3 GB of state),
    256 x 256 mesh, dt = 16 gyro-periods, sort_interval = 1, timing build; 3 steps, then every 32 768-th marker against the
    oracle (markers are independent).  ids are a permutation, mu is untouched, and the number of lost
    markers on the sample equals the oracle's."""
    n = 1 << 26
    w = synth.make_config(4, n_markers=n, dt_gyro=16.0)
    assert w.n_markers == n and w.n_elems == 131072
    nsteps = 3
    idx = np.arange(0, n, 32768)
    sample = take(w.markers, idx)
    mesh, sp = oracle_of(w)
    ref, e_ref, _ = oracle_push(mesh, sp, sample, nsteps, w.dt)
    _, e_next, lost_next = oracle_push(mesh, sp, sample, nsteps + 1, w.dt)
    p = make_pusher(w, verify=False, sort_interval=1)
    mu0 = w.markers["mu"]
    p.push(nsteps, w.dt)
    st = p.stats()
    assert st["steps_done"] == nsteps and st["n_markers"] == n
    ids = p.id_t.cpu().numpy()
    assert np.array_equal(np.bincount(ids, minlength=n), np.ones(n, dtype=np.int64))
    inv = np.empty_like(ids)
    inv[ids] = np.arange(n, dtype=ids.dtype)
    slot = inv[idx]                                                      # where the sampled markers sit now
    got = {k: p.state_t[k].cpu().numpy()[slot] for k in KEYS}
    elem = p.elem_t.cpu().numpy()[slot]
    assert np.array_equal(p.state_t["mu"].cpu().numpy(), mu0[ids])
    live = e_ref >= 0
    wrms = np.sqrt(np.mean(ref["w"][live] ** 2))
    # every sampled marker, the lost ones included: they hold the state of their last live step on both sides (G12)
    ex, ev, ew = g16_errors(got, ref, w_floor=wrms)
    assert max(ex.max(), ev.max(), ew.max()) <= 3 * TOL_STEP, (ex.max(), ev.max(), ew.max())
    assert np.array_equal(elem < 0, e_next < 0) and int((elem < 0).sum()) == lost_next
    assert live.mean() > 0.9
