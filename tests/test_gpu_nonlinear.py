"""GPU parity of the non-linear trajectory mode (m3dk_set_options mode = 1, reading
G21) against the oracle's mode 1 (itself pinned by tests/test_oracle_nonlinear.py), through the C ABI."""
import dataclasses

import numpy as np
import pytest

import synth
from gpu_helpers import KEYS, g16_errors, make_pusher, oracle_of, oracle_push, take
from test_gpu_ordered import _unstructured

pytestmark = pytest.mark.gpu

TOL_STEP = 1.0e-12
SMALL = {1: dict(n_markers=6000 + 37, nx=32), 2: dict(n_markers=6000 + 37, nx=48), 3: dict(n_markers=6000 + 37, nx=64)}


def _amp(idx):
    # a perturbation strong enough that the orbit change and the (1 - w) factor are far above the tolerance
    return synth.make_config(idx, amp=5.0e-3, **SMALL[idx])


@pytest.mark.parametrize("verify", [True, False])
@pytest.mark.parametrize("idx", [1, 2, 3])
def test_per_step_parity_nonlinear(idx, verify):
    """Reading G16: restart the GPU from the oracle's state at steps 0, 1, 10, 50, one step, compare."""
    w = _amp(idx)
    mesh, sp = oracle_of(w, mode=1)
    p = make_pusher(w, verify=verify, mode=1)
    state = {k: w.markers[k].copy() for k in KEYS}
    done, worst = 0, np.zeros(3)
    for s in (0, 1, 10, 50):
        if s > done:
            state, _, _ = oracle_push(mesh, sp, state, s - done, w.dt, t0=0.0, step0=done)
            done = s
        ref, e_ref, _ = oracle_push(mesh, sp, state, 1, w.dt, t0=0.0, step0=s)
        p.set_state(state)
        p.set_options(sort_interval=0, mode=1, t0=s * w.dt)
        p.push(1, w.dt)
        got, _, _ = p.state()
        live = e_ref >= 0
        assert live.sum() > 0.9 * live.size
        assert np.array_equal(got["mu"], state["mu"])
        wrms = np.sqrt(np.mean(ref["w"][live] ** 2))
        ex, ev, ew = g16_errors(take(got, live), take(ref, live), w_floor=wrms)
        worst = np.maximum(worst, [ex.max(), ev.max(), ew.max()])
    assert worst.max() <= TOL_STEP, worst
    # the mode does something: the linear mode gives a different orbit from the same start
    lin, _, _ = oracle_push(oracle_of(w)[0], oracle_of(w)[1], w.markers, 5, w.dt)
    nl, _, _ = oracle_push(mesh, sp, w.markers, 5, w.dt)
    assert np.abs(lin["x"] - nl["x"]).max() > 1e-7


@pytest.mark.parametrize("two_modes", [False, True])
def test_nonlinear_ordered_pipeline_and_bitwise_order_independence(two_modes):
    """Several steps of mode 1 through the element-ordered path on an unstructured mesh (one and two toroidal modes, one
    with n < 0) against the oracle, and the same bits for sort_interval 0, 1 and 3."""
    w0 = _unstructured(two_modes=two_modes)
    w = dataclasses.replace(w0, pert_coef=w0.pert_coef * 30.0)          # 3e-3 B0: a visibly non-linear case
    mesh, sp = oracle_of(w, mode=1)
    nsteps = 6
    ref, e_ref, _ = oracle_push(mesh, sp, w.markers, nsteps, w.dt)
    res = {}
    for si in (0, 1, 3):
        p = make_pusher(w, verify=True, sort_interval=si, mode=1)
        p.push(nsteps, w.dt)
        got, elem, ids = p.state()
        assert np.array_equal(np.sort(ids), np.arange(w.n_markers))
        res[si] = got
        live = e_ref >= 0
        wrms = np.sqrt(np.mean(ref["w"][live] ** 2))
        ex, ev, ew = g16_errors(take(got, live), take(ref, live), w_floor=wrms)
        assert max(ex.max(), ev.max(), ew.max()) <= 6 * TOL_STEP, (si, ex.max(), ev.max(), ew.max())
    for si in (1, 3):
        for k in KEYS:
            assert np.array_equal(res[si][k], res[0][k]), (si, k)


def test_nonlinear_zero_amplitude_equals_linear_mode_on_gpu():
    """Without a perturbation the two modes are the same map; with the weights at zero the GPU must agree bit for bit in
    x and v (the arithmetic of the velocity update is written once for both modes up to the vanishing terms)."""
    w = synth.make_config(1, n_markers=3000, nx=32, amp=0.0)
    out = {}
    for mode in (0, 1):
        p = make_pusher(w, verify=True, sort_interval=1, mode=mode)
        p.push(7, w.dt)
        out[mode], _, _ = p.state()
    assert (out[1]["w"] == 0.0).all() and (out[0]["w"] == 0.0).all()
    for k in ("x", "y", "z", "vx", "vy", "vz"):
        d = np.abs(out[1][k] - out[0][k]).max()
        assert d <= 1e-13, (k, d)


@pytest.mark.parametrize("mode", [1, 2])
def test_300_step_parity_on_non_chaotic_orbits(mode):
    """The long-run bar of BASELINE.json (<= 1e-8 on non-chaotic orbits, filter of reading G15 from the oracle alone) for the
    non-linear and the FLR mode, through the ordered pipeline."""
    w0 = synth.make_config(3, n_markers=600 + 7, nx=48)
    w = dataclasses.replace(w0, pert_coef=w0.pert_coef * (20.0 if mode == 1 else 1.0))
    mesh, sp = oracle_of(w, mode=mode)
    nsteps = 300
    a, ea, _ = oracle_push(mesh, sp, w.markers, nsteps, w.dt)
    twin = {k: w.markers[k].copy() for k in KEYS}
    for k in ("x", "y", "z"):
        twin[k] *= (1.0 + 1.0e-13)
    b, eb, _ = oracle_push(mesh, sp, twin, nsteps, w.dt)
    ex, ev, _ = g16_errors(b, a)
    keep = (ex < 1e-9) & (ev < 1e-9) & (ea == eb) & (ea >= 0)
    assert keep.mean() > 0.5
    p = make_pusher(w, verify=True, sort_interval=1, mode=mode)
    p.push(nsteps, w.dt)
    got, _, _ = p.state()
    wrms = np.sqrt(np.mean(a["w"][keep] ** 2))
    ex, ev, ew = g16_errors(take(got, keep), take(a, keep), w_floor=wrms)
    assert max(ex.max(), ev.max(), ew.max()) <= 1.0e-8, (ex.max(), ev.max(), ew.max(), keep.mean())


@pytest.mark.parametrize("mode", [1, 2])
def test_modes_without_any_perturbation_table(mode):
    """n_modes = 0 (config 0): both modes reduce to the equilibrium push, w is never written, parity with the oracle."""
    w = synth.make_config(0, n_markers=2000 + 3, nx=32)
    mesh, sp = oracle_of(w, mode=mode)
    ref, e_ref, _ = oracle_push(mesh, sp, w.markers, 5, w.dt)
    for si in (0, 1):
        p = make_pusher(w, verify=True, sort_interval=si, mode=mode)
        p.push(5, w.dt)
        got, _, _ = p.state()
        live = e_ref >= 0
        ex, ev, _ = g16_errors(take(got, live), take(ref, live), w_floor=1.0)
        assert max(ex.max(), ev.max()) <= 5 * TOL_STEP
        assert np.array_equal(got["w"], w.markers["w"])
