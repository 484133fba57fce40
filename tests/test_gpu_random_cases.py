"""Seeded random combinations of the knobs of the push and of the deposition, against the oracle through the C ABI: marker
counts around the work-item boundaries (1, 2, 31..33, 63..65, 97 markers: items of one lane, ragged tails, a single small
item), coarse and fine meshes, dt of 1..16 gyro-periods, the four modes, every ordering interval, both builds, and the
chunk-pipelined host path (bitwise equal to m3dk_push).  The fixed cases of the other files pick their sizes by hand; this
file exists to hit the combinations nobody thought of."""
import dataclasses

import numpy as np
import pytest
import torch

import oracle
import synth
from gpu_helpers import KEYS, g16_errors, make_pusher, oracle_of, oracle_push, take

pytestmark = pytest.mark.gpu

_cache = {}


def _workload(rng, idx, nx, dtg, n, amp=1.0e-4):
    key = (idx, nx, dtg, amp)
    if key not in _cache:
        _cache[key] = synth.make_config(idx, n_markers=4096, nx=nx, dt_gyro=dtg, amp=amp)
    w = _cache[key]
    sel = rng.choice(4096, size=n, replace=False)
    return dataclasses.replace(w, markers={k: np.ascontiguousarray(v[sel]) for k, v in w.markers.items()})


def test_random_push_cases_against_the_oracle():
    rng = np.random.default_rng(2025)
    for _ in range(24):
        idx = int(rng.choice([1, 2, 3]))
        nx = int(rng.choice([8, 16, 40]))
        dtg = float(rng.choice([1.0, 8.0, 16.0]))
        n = int(rng.choice([1, 2, 31, 32, 33, 63, 64, 65, 97, 500, 4096]))
        mode = int(rng.choice([0, 1, 2, 3]))
        si = int(rng.choice([0, 1, 10]))
        nsteps = int(rng.choice([1, 2, 5]))
        verify = bool(rng.integers(2))
        case = dict(idx=idx, nx=nx, dtg=dtg, n=n, mode=mode, si=si, nsteps=nsteps, verify=verify)
        w = _workload(rng, idx, nx, dtg, n)
        mesh, sp = oracle_of(w, mode=mode)
        ref, e_ref, _ = oracle_push(mesh, sp, w.markers, nsteps, w.dt)
        _, _, lost_next = oracle_push(mesh, sp, w.markers, nsteps + 1, w.dt)
        p = make_pusher(w, verify=verify, sort_interval=si, mode=mode)
        p.push(nsteps, w.dt)
        got, _, ids = p.state()
        assert np.array_equal(np.sort(ids), np.arange(n)), case
        assert p.stats()["n_lost"] == lost_next, case
        live = e_ref >= 0
        if live.any():
            wrms = max(float(np.sqrt(np.mean(ref["w"][live] ** 2))), 1e-30)
            ex, ev, ew = g16_errors(take(got, live), take(ref, live), w_floor=wrms)
            assert max(ex.max(), ev.max(), ew.max()) <= nsteps * 1.0e-12, (case, ex.max(), ev.max(), ew.max())
        # the host path gives the same bits, whatever the number of chunks
        host = {k: torch.from_numpy(w.markers[k].copy()).pin_memory() for k in KEYS}
        hid = torch.empty(n, dtype=torch.int32).pin_memory()
        q = make_pusher(w, verify=verify, sort_interval=si, mode=mode)
        q.push_host(host, nsteps, w.dt, n_chunks=int(rng.choice([1, 2, 5, 9])), host_id=hid)
        for k in KEYS:
            r = np.empty(n)
            r[hid.numpy()] = host[k].numpy()
            assert np.array_equal(r, got[k]), (case, k)


def test_random_deposit_cases_against_the_oracle():
    rng = np.random.default_rng(77)
    for _ in range(24):
        idx = int(rng.choice([1, 3]))
        nx = int(rng.choice([8, 24, 40]))
        n = int(rng.choice([1, 2, 31, 33, 64, 65, 129, 1000, 4096]))
        flags = int(rng.integers(0, 8))
        si = int(rng.choice([0, 1]))
        t = float(rng.uniform(0.0, 3.0))
        w = _workload(rng, idx, nx, 8.0, n, amp=1.0e-2)
        mk = {k: v.copy() for k, v in w.markers.items()}
        mk["w"] = rng.normal(size=n) * 1.0e-2
        if rng.integers(2):
            mk["mu"] = mk["mu"] * 3.0                                       # larger rings: more points outside the mesh
        w = dataclasses.replace(w, markers=mk)
        case = dict(idx=idx, nx=nx, n=n, flags=flags, si=si)
        mesh, sp = oracle_of(w)
        ref, _ = oracle.deposit(mesh, sp, mk, flags=flags, t=t)
        absw = dict(mk)
        absw["w"] = np.abs(mk["w"]) + 3.0e-2                                # |w| + a bound of |B1par / B*par|
        scale, _ = oracle.deposit(mesh, sp, absw, flags=flags & 2)
        S = np.abs(scale[:, :, 0, 0])[:, :, None, None] + np.abs(scale).max() * 1.0e-3 + 1.0e-300
        p = make_pusher(w, verify=bool(rng.integers(2)), sort_interval=si)
        if (flags & 2) and rng.integers(2):
            p.set_flr_workspace(nonlinear=bool(rng.integers(2)))           # ordered ring stream of the 4-point deposition
        got = p.deposit(flags=flags, t=t)
        assert (np.abs(got - ref) <= 1.0e-11 * S).all(), (case, float((np.abs(got - ref) / S).max()))
        rhs = torch.full((p.deposit_bytes() // 8,), float("nan"), dtype=torch.float64, device=p.device)
        p.deposit_noalloc_into(rhs, flags, t)
        p.stats()
        got2 = rhs.cpu().numpy().reshape(ref.shape)
        assert (np.abs(got2 - ref) <= 1.0e-11 * S).all(), (case, "noalloc", float((np.abs(got2 - ref) / S).max()))
