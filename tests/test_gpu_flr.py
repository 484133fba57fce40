"""GPU parity of the finite-Larmor-radius mode (m3dk_set_options mode = 2, Eq. 14,
reading G23) against the oracle's mode 2 (pinned by tests/test_oracle_flr.py), through the C ABI."""
import dataclasses

import numpy as np
import pytest

import synth
from gpu_helpers import KEYS, g16_errors, make_pusher, oracle_of, oracle_push, take
from test_gpu_ordered import _unstructured

pytestmark = pytest.mark.gpu

TOL_STEP = 1.0e-12
SMALL = {1: dict(n_markers=5000 + 37, nx=32), 2: dict(n_markers=5000 + 37, nx=48), 3: dict(n_markers=5000 + 37, nx=64)}


@pytest.mark.parametrize("verify", [True, False])
@pytest.mark.parametrize("idx", [1, 2, 3])
def test_per_step_parity_flr(idx, verify):
    w = synth.make_config(idx, **SMALL[idx])
    mesh, sp = oracle_of(w, mode=2)
    p = make_pusher(w, verify=verify, mode=2)
    state = {k: w.markers[k].copy() for k in KEYS}
    done, worst = 0, np.zeros(3)
    for s in (0, 1, 10, 40):
        if s > done:
            state, _, _ = oracle_push(mesh, sp, state, s - done, w.dt, t0=0.0, step0=done)
            done = s
        ref, e_ref, _ = oracle_push(mesh, sp, state, 1, w.dt, t0=0.0, step0=s)
        p.set_state(state)
        p.set_options(sort_interval=0, mode=2, t0=s * w.dt)
        p.push(1, w.dt)
        got, _, _ = p.state()
        live = e_ref >= 0
        assert live.sum() > 0.9 * live.size
        wrms = np.sqrt(np.mean(ref["w"][live] ** 2))
        ex, ev, ew = g16_errors(take(got, live), take(ref, live), w_floor=wrms)
        worst = np.maximum(worst, [ex.max(), ev.max(), ew.max()])
    assert worst.max() <= TOL_STEP, worst
    # the averaging does something: the weights differ from the linear mode's on the same orbits
    lin, _, _ = oracle_push(oracle_of(w)[0], oracle_of(w)[1], w.markers, 20, w.dt)
    flr, _, _ = oracle_push(mesh, sp, w.markers, 20, w.dt)
    assert np.array_equal(lin["x"], flr["x"])
    assert np.abs(lin["w"] - flr["w"]).max() > 1e-3 * np.sqrt(np.mean(lin["w"] ** 2))


@pytest.mark.parametrize("two_modes", [False, True])
def test_flr_ordered_pipeline_and_bitwise_order_independence(two_modes):
    """Mode 2 through the element-ordered path on an unstructured mesh (ring points land in other, arbitrary elements and
    some fall outside the mesh), against the oracle, and the same bits for sort_interval 0, 1 and 3."""
    w = _unstructured(two_modes=two_modes)
    mesh, sp = oracle_of(w, mode=2)
    nsteps = 5
    ref, e_ref, _ = oracle_push(mesh, sp, w.markers, nsteps, w.dt)
    res = {}
    for si in (0, 1, 3, -1):                       # -1: ordered pipeline WITHOUT the FLR workspace (every lane gathers)
        p = make_pusher(w, verify=True, sort_interval=abs(si), mode=2, flr_ws=si > 0)
        p.push(nsteps, w.dt)
        got, elem, ids = p.state()
        assert np.array_equal(np.sort(ids), np.arange(w.n_markers))
        res[si] = got
        live = e_ref >= 0
        wrms = np.sqrt(np.mean(ref["w"][live] ** 2))
        ex, ev, ew = g16_errors(take(got, live), take(ref, live), w_floor=wrms)
        assert max(ex.max(), ev.max(), ew.max()) <= 5 * TOL_STEP, (si, ex.max(), ev.max(), ew.max())
    for si in (1, 3, -1):
        for k in KEYS:
            assert np.array_equal(res[si][k], res[0][k]), (si, k)


@pytest.mark.parametrize("verify", [True, False])
def test_flr_ring_stream_per_step_parity_with_lost_markers(verify):
    """The ordered FLR path (ring points emitted, ordered by their element, evaluated with staged tiles, summed back):
    one step restarted from the oracle at steps 0 and 7, config 3 shape, with markers outside the mesh from the start and
    ring points that fall outside it (markers at the edge of the box)."""
    import dataclasses
    w0 = synth.make_config(3, n_markers=9000 + 5, nx=64)
    mk = {k: v.copy() for k, v in w0.markers.items()}
    mk["x"][:9] = 20.0                                      # lost from the start: no ring
    mk["z"][9:60] = 1.0995                                  # at the upper edge: part of the ring is outside the mesh
    w = dataclasses.replace(w0, markers=mk)
    mesh, sp = oracle_of(w, mode=2)
    p = make_pusher(w, verify=verify, sort_interval=1, mode=2)
    state = {k: mk[k].copy() for k in KEYS}
    done = 0
    for s in (0, 7):
        if s > done:
            state, _, _ = oracle_push(mesh, sp, state, s - done, w.dt, t0=0.0, step0=done)
            done = s
        ref, e_ref, _ = oracle_push(mesh, sp, state, 1, w.dt, t0=0.0, step0=s)
        p.set_state(state)
        p.set_options(sort_interval=1, mode=2, t0=s * w.dt)
        p.push(1, w.dt)
        got, _, ids = p.state()
        assert np.array_equal(np.sort(ids), np.arange(w.n_markers))
        live = e_ref >= 0
        for k in KEYS:
            assert np.array_equal(got[k][~live], state[k][~live])
        wrms = np.sqrt(np.mean(ref["w"][live] ** 2))
        ex, ev, ew = g16_errors(take(got, live), take(ref, live), w_floor=wrms)
        assert max(ex.max(), ev.max(), ew.max()) <= TOL_STEP, (s, ex.max(), ev.max(), ew.max())


def test_flr_where_b_is_parallel_to_the_major_radius():
    """the ring basis must not divide by zero where b0 is parallel to the major-radius direction.  Hand-made
    tables with a nearly radial field (psi0 = A Z, a weak F): push (mode 2) and 4-point deposition against the oracle."""
    import dataclasses
    import oracle
    from handmade import HandMade
    w0 = synth.make_config(1, n_markers=2000 + 3, nx=12)
    hm = HandMade(eq=dict(psi=(0.0, 0.0, 0.9), Bm=(1.0, 0.0, 0.0), F=(0.0,), kappa=(0.3,)),
                  pert=dict(E_R=(1e-3,), E_Z=(2e-3 + 1e-3j,), B_Z=(1e-3j,), B_par=(1e-3, 2e-3, -1e-3)), n_tor=2, omega=0.05, nx=12)
    w = dataclasses.replace(w0, node_RZ=hm.node, tri=hm.tri, eq_coef=hm.eq_coef, pert_coef=hm.pert_coef,
                            n_tor=hm.n_tor_a, omega=hm.omega_a)
    mesh, sp = oracle_of(w, mode=2)
    ref, e_ref, _ = oracle_push(mesh, sp, w.markers, 2, 0.01)
    p = make_pusher(w, verify=True, sort_interval=1, mode=2)
    p.push(2, 0.01)
    got, _, _ = p.state()
    live = e_ref >= 0
    assert live.mean() > 0.9 and np.isfinite(got["w"]).all()
    wrms = np.sqrt(np.mean(ref["w"][live] ** 2))
    ex, ev, ew = g16_errors(take(got, live), take(ref, live), w_floor=wrms)
    assert max(ex.max(), ev.max(), ew.max()) <= 3 * TOL_STEP, (ex.max(), ev.max(), ew.max())
    raw, _, _ = p.state(by_id=False)
    want, _ = oracle.deposit(mesh, sp, raw, 2, 0.0)
    rhs = p.deposit(flags=2, t=0.0)
    assert np.isfinite(rhs).all()
    assert np.abs(rhs - want).max() <= 1e-10 * max(np.abs(want).max(), 1e-300)


@pytest.mark.parametrize("verify", [True, False])
def test_nonlinear_mode_with_gyro_average(verify):
    """Mode 3 (non-linear trajectories in the gyro-averaged perturbed fields; oracle pin F6): one step restarted from the
    oracle at steps 0 and 9, amplitude 1e-2 so that the perturbation moves the orbits; then the same bits for the SoA path and
    the ordered pipeline over 6 chained steps."""
    w = synth.make_config(3, n_markers=5000 + 11, nx=64, amp=1e-2)
    mesh, sp = oracle_of(w, mode=3)
    p = make_pusher(w, verify=verify, mode=3)
    state = {k: w.markers[k].copy() for k in KEYS}
    done = 0
    for s in (0, 9):
        if s > done:
            state, _, _ = oracle_push(mesh, sp, state, s - done, w.dt, t0=0.0, step0=done)
            done = s
        ref, e_ref, _ = oracle_push(mesh, sp, state, 1, w.dt, t0=0.0, step0=s)
        p.set_state(state)
        p.set_options(sort_interval=0, mode=3, t0=s * w.dt)
        p.push(1, w.dt)
        got, _, _ = p.state()
        live = e_ref >= 0
        wrms = np.sqrt(np.mean(ref["w"][live] ** 2))
        ex, ev, ew = g16_errors(take(got, live), take(ref, live), w_floor=wrms)
        assert max(ex.max(), ev.max(), ew.max()) <= TOL_STEP, (s, ex.max(), ev.max(), ew.max())
    lin, _, _ = oracle_push(*oracle_of(w, mode=1), w.markers, 6, w.dt)
    res = {}
    # SoA kernel; ordered pipeline with per-lane ring gathers; ordered pipeline through the ring stream (two passes per step)
    for name, si, ws in (("soa", 0, False), ("gather", 1, False), ("stream", 1, True)):
        q = make_pusher(w, verify=verify, sort_interval=si, mode=3, flr_ws=ws)
        q.push(6, w.dt)
        res[name], _, ids = q.state()
        assert np.array_equal(np.sort(ids), np.arange(w.n_markers))
    for name in ("gather", "stream"):
        for k in KEYS:
            assert np.array_equal(res["soa"][k], res[name][k]), (name, k)
    assert np.abs(res["soa"]["vx"] - lin["vx"]).max() > 1e-7          # the average changes the orbit itself


def test_nonlinear_gyro_average_ring_stream_with_lost_markers_and_ring_points_outside():
    """Mode 3 through the ring stream on markers loaded at the edge of the mesh with large gyro-radii: ring points fall
    outside the mesh (zero contribution), markers are lost on the way (their slots carry no ring) and the ordering changes
    every step; chained steps against the oracle, and bit for bit against the per-lane gathers."""
    from synth.configs import CHARGE, MASS
    w0 = synth.make_config(3, n_markers=4000 + 9, nx=48, dt_gyro=16.0)
    mk = synth.load_markers(w0.eq, 4000 + 9, 99, CHARGE, MASS, w0.dt, rmin=0.85, rmax=1.09, profile_L=None,
                            speed="slowing", v_c=0.3, pitch="uniform")
    mk["mu"] = mk["mu"] * 3.0
    w = dataclasses.replace(w0, markers=mk)
    mesh, sp = oracle_of(w, mode=3)
    nsteps = 7
    ref, e_ref, lost = oracle_push(mesh, sp, mk, nsteps, w.dt)
    assert lost > 100
    res = {}
    for name, ws in (("gather", False), ("stream", True)):
        q = make_pusher(w, verify=True, sort_interval=1, mode=3, flr_ws=ws)
        q.push(nsteps, w.dt)
        res[name], _, ids = q.state()
        assert np.array_equal(np.sort(ids), np.arange(w.n_markers))
    for k in KEYS:
        assert np.array_equal(res["gather"][k], res["stream"][k]), k
    wrms = np.sqrt(np.mean(ref["w"][e_ref >= 0] ** 2))
    ex, ev, ew = g16_errors(res["stream"], ref, w_floor=wrms)
    assert max(ex.max(), ev.max(), ew.max()) <= nsteps * TOL_STEP, (ex.max(), ev.max(), ew.max())
