"""GPU parity of m3dk_gc_push (RK4 guiding-centre pusher, Eqs. 1-4, reading G24) against the oracle's
gc_push on the same finite-element tables (pinned by tests/test_oracle_gc.py), through the C ABI."""
import dataclasses

import numpy as np
import pytest

import oracle
import synth
from gpu_helpers import make_pusher

pytestmark = pytest.mark.gpu


def _vpar(w):
    """v . b0 of the workload's markers from the analytic equilibrium (an input, not method arithmetic)."""
    mk = w.markers
    R = np.hypot(mk["x"], mk["y"])
    BR, BP, BZ = w.eq.B_cyl(R, mk["z"])
    Bn = np.sqrt(BR ** 2 + BP ** 2 + BZ ** 2)
    c, s = mk["x"] / R, mk["y"] / R
    return ((mk["vx"] * c + mk["vy"] * s) * BR + (-mk["vx"] * s + mk["vy"] * c) * BP + mk["vz"] * BZ) / Bn


def _err(got, ref, live):
    gx, gy, gz, gv = got
    rx, ry, rz, rv = ref
    dx = np.sqrt((gx - rx) ** 2 + (gy - ry) ** 2 + (gz - rz) ** 2) / np.sqrt(rx ** 2 + ry ** 2 + rz ** 2)
    dv = np.abs(gv - rv) / np.maximum(np.abs(rv), np.sqrt(np.mean(rv[live] ** 2)))
    return float(dx[live].max()), float(dv[live].max())


@pytest.mark.parametrize("verify", [True, False])
@pytest.mark.parametrize("idx,nx", [(0, 32), (3, 64)])
def test_gc_push_matches_oracle(idx, nx, verify):
    w = synth.make_config(idx, n_markers=5000 + 13, nx=nx)
    mesh, sp = oracle.Mesh.of(w), oracle.species_of(w)
    mk, vp0 = w.markers, _vpar(w)
    dt = 2.0 * w.dt
    for nsteps, tol in ((1, 1e-12), (40, 1e-9)):
        rx, ry, rz, rv, e_ref, lost = oracle.gc_push(sp, mk["x"], mk["y"], mk["z"], vp0, mk["mu"], nsteps, dt, mesh=mesh)
        p = make_pusher(w, verify=verify)
        gx, gy, gz, gv, e_gpu = p.gc_push(nsteps, dt, vp0)
        live = e_ref >= 0
        assert live.mean() > 0.9
        assert np.array_equal(e_gpu < 0, e_ref < 0)
        assert np.array_equal(e_gpu, e_ref)                # element of the CURRENT position, step after step
        ex, ev = _err((gx, gy, gz, gv), (rx, ry, rz, rv), live)
        assert max(ex, ev) <= tol, (nsteps, ex, ev)
        st, _, _ = p.state(by_id=False)
        assert np.array_equal(st["mu"], mk["mu"]) and np.array_equal(st["vx"], mk["vx"])      # untouched arrays


def test_gc_lost_guiding_centres_are_frozen():
    w = synth.make_config(0, n_markers=400, nx=16)
    mk = {k: v.copy() for k, v in w.markers.items()}
    vp = _vpar(w)
    mk["x"][:5] = 60.0                                  # outside from the start
    mk["z"][5:25] = 1.0995                              # next to the upper edge: drift / streaming takes some of them out
    w2 = dataclasses.replace(w, markers=mk)
    mesh, sp = oracle.Mesh.of(w2), oracle.species_of(w2)
    rx, ry, rz, rv, e_ref, lost = oracle.gc_push(sp, mk["x"], mk["y"], mk["z"], vp, mk["mu"], 30, 4.0 * w.dt, mesh=mesh)
    p = make_pusher(w2, verify=True)
    gx, gy, gz, gv, e_gpu = p.gc_push(30, 4.0 * w.dt, vp)
    assert lost >= 6 and np.array_equal(e_gpu < 0, e_ref < 0)
    assert np.array_equal(gx[:5], mk["x"][:5]) and np.array_equal(gv[:5], vp[:5])
    dead = e_ref < 0
    # a lost guiding centre keeps the state it had before the step that left the mesh: same as the oracle's
    assert np.allclose(gx[dead], rx[dead], rtol=1e-9) and np.allclose(gz[dead], rz[dead], rtol=1e-9, atol=1e-12)
    ex, ev = _err((gx, gy, gz, gv), (rx, ry, rz, rv), ~dead)
    assert max(ex, ev) <= 1e-9


def test_gc_bootstrap_then_push_then_deposit_matches_the_oracle_chain():
    """PAPER.md:80 on the device: m3dk_gc_bootstrap writes (x_1, (x_1 - x_0)/dt) and the element of x_1; a following
    m3dk_push and m3dk_deposit trust that element (it used to be one step stale).  The same chain through the
    oracle: gc_bootstrap -> push_fe -> deposit."""
    w = synth.make_config(3, n_markers=6000 + 7, nx=64)
    mesh, sp = oracle.Mesh.of(w), oracle.species_of(w)
    mk, vp0 = w.markers, _vpar(w)
    x1, y1, z1, vx, vy, vz, ok = oracle.gc_bootstrap(sp, mk["x"], mk["y"], mk["z"], vp0, mk["mu"], w.dt, mesh=mesh)
    assert ok.mean() > 0.99
    start = {k: v.copy() for k, v in mk.items()}
    for k, a in (("x", x1), ("y", y1), ("z", z1)):
        start[k] = a
    for k, a in (("vx", vx), ("vy", vy), ("vz", vz)):
        start[k] = np.where(ok, a, mk[k])
    nsteps = 3
    ref, e_ref, _ = oracle.push_fe(mesh, sp, start, nsteps, w.dt, t0=w.dt)
    p = make_pusher(w, verify=True, sort_interval=1, t0=w.dt)
    p.gc_bootstrap(w.dt, vp0)
    got0, e0, _ = p.state()
    assert np.array_equal(e0 >= 0, ok)
    for k in ("x", "y", "z", "vx", "vy", "vz"):
        assert np.allclose(got0[k][ok], start[k][ok], rtol=1e-12, atol=1e-13), k
    R1 = np.hypot(start["x"], start["y"])
    assert np.array_equal(e0[ok], mesh.locate(R1, start["z"])[ok])          # element of x_1, not of x_0
    p.push(nsteps, w.dt)
    got, e_gpu, _ = p.state()
    live = (e_ref >= 0) & ok
    from gpu_helpers import g16_errors, take
    wrms = np.sqrt(np.mean(ref["w"][live] ** 2))
    ex, ev, ew = g16_errors(take(got, live), take(ref, live), w_floor=wrms)
    assert max(ex.max(), ev.max(), ew.max()) <= 1e-11, (ex.max(), ev.max(), ew.max())
    # deposit after a guiding-centre push: bins by the element gc_push left behind
    q = make_pusher(w, verify=True, sort_interval=1)
    gx, gy, gz, gv, e_gc = q.gc_push(2, w.dt, vp0)
    rhs = q.deposit(flags=0, t=0.0)
    mk2 = {k: v.copy() for k, v in mk.items()}
    rx, ry, rz, rv, e_or, _ = oracle.gc_push(sp, mk["x"], mk["y"], mk["z"], vp0, mk["mu"], 2, w.dt, mesh=mesh)
    mk2["x"], mk2["y"], mk2["z"] = rx, ry, rz
    want, _ = oracle.deposit(mesh, sp, mk2, 0, 0.0)
    scale = np.abs(want).max()
    assert np.abs(rhs - want).max() <= 1e-9 * scale


@pytest.mark.parametrize("verify", [True, False])
def test_gc_push_in_the_total_fields_matches_oracle(verify):
    """Mode 1: Eqs. (1)-(2) with E1, B1 and grad B1par (reading G26) at the context's time; the clock advances."""
    w = synth.make_config(3, n_markers=4000 + 7, nx=64, amp=1e-2)
    mesh, sp = oracle.Mesh.of(w), oracle.species_of(w, mode=1)
    mk, vp0 = w.markers, _vpar(w)
    dt, t0, nsteps = 2.0 * w.dt, 0.9, 6
    rx, ry, rz, rv, e_ref, lost = oracle.gc_push(sp, mk["x"], mk["y"], mk["z"], vp0, mk["mu"], nsteps, dt, mesh=mesh, t0=t0)
    p = make_pusher(w, verify=verify, mode=1, t0=t0)
    gx, gy, gz, gv, e_gpu = p.gc_push(nsteps, dt, vp0)
    live = e_ref >= 0
    assert live.mean() > 0.9 and np.array_equal(e_gpu, e_ref)
    ex, ev = _err((gx, gy, gz, gv), (rx, ry, rz, rv), live)
    assert max(ex, ev) <= 1e-10, (ex, ev)
    st = p.stats()
    assert st["steps_done"] == nsteps and abs(st["t"] - (t0 + nsteps * dt)) < 1e-12
    # the perturbation matters at this amplitude: the equilibrium-only orbit differs by far more than the tolerance
    qx, qy, qz, qv, _, _ = oracle.gc_push(oracle.species_of(w), mk["x"], mk["y"], mk["z"], vp0, mk["mu"], nsteps, dt, mesh=mesh)
    assert np.abs(qv - rv)[live].max() > 1e-5
