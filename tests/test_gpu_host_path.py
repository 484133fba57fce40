"""GPU tests of the host-buffer path: m3dk_particles_upload / _download and the chunk-pipelined m3dk_push_host, against the
CPU oracle on the same seeded inputs (through the C ABI)."""
import numpy as np
import pytest
import torch

import synth
from gpu_helpers import KEYS, g16_errors, make_pusher, oracle_of, oracle_push, take

pytestmark = pytest.mark.gpu

TOL_STEP = 1.0e-12


def _pinned(markers):
    return {k: torch.from_numpy(np.ascontiguousarray(markers[k]).copy()).pin_memory() for k in KEYS}


@pytest.mark.parametrize("si", [1, 0])
@pytest.mark.parametrize("n_chunks", [0, 1, 3, 7])      # 0: the library chooses
def test_push_host_matches_the_oracle(n_chunks, si):
    """m3dk_push_host in place on pinned host buffers: ids are a permutation of the caller's indices (global across the
    chunks), every marker carries its own mu, and the state is the oracle's after nsteps steps from t0; the context's
    clock advances once, so a following m3dk_push continues at the right phase."""
    w = synth.make_config(3, n_markers=9000 + 41, nx=48)
    mesh, sp = oracle_of(w)
    nsteps, t0 = 5, 0.37
    ref, e_ref, _ = oracle_push(mesh, sp, w.markers, nsteps, w.dt, t0=t0)
    p = make_pusher(w, verify=True, sort_interval=si, t0=t0)
    host = _pinned(w.markers)
    ids = torch.empty(w.n_markers, dtype=torch.int32).pin_memory()
    elem = torch.empty(w.n_markers, dtype=torch.int32).pin_memory()
    p.push_host(host, nsteps, w.dt, n_chunks=n_chunks, host_id=ids, host_elem=elem)
    ids = ids.numpy()
    assert np.array_equal(np.sort(ids), np.arange(w.n_markers))
    got = {k: np.empty(w.n_markers) for k in KEYS}
    for k in KEYS:
        got[k][ids] = host[k].numpy()
    assert np.array_equal(got["mu"], w.markers["mu"])
    live = e_ref >= 0
    wrms = np.sqrt(np.mean(ref["w"][live] ** 2))
    ex, ev, ew = g16_errors(take(got, live), take(ref, live), w_floor=wrms)
    assert max(ex.max(), ev.max(), ew.max()) <= nsteps * TOL_STEP, (ex.max(), ev.max(), ew.max())
    st = p.stats()
    assert st["steps_done"] == nsteps and abs(st["t"] - (t0 + nsteps * w.dt)) < 1e-12
    # the device arrays hold the same state (chunk by chunk); two more steps through m3dk_push continue from it
    ref2, e2, _ = oracle_push(mesh, sp, ref, 2, w.dt, t0=t0, step0=nsteps, elem=e_ref)
    p.push(2, w.dt)
    got2, _, _ = p.state()
    # ids on the device are global too, so state() orders by the caller's index
    live2 = e2 >= 0
    ex, ev, ew = g16_errors(take(got2, live2), take(ref2, live2), w_floor=wrms)
    assert max(ex.max(), ev.max(), ew.max()) <= (nsteps + 2) * TOL_STEP


def test_push_host_is_bitwise_the_upload_push_download_path():
    w = synth.make_config(1, n_markers=5000 + 3, nx=32)
    out = {}
    for chunks in (0, 1, 4):
        p = make_pusher(w, verify=False, sort_interval=1)
        host = _pinned(w.markers)
        ids = torch.empty(w.n_markers, dtype=torch.int32).pin_memory()
        if chunks == 0:
            p.upload(host)
            p.set_options(sort_interval=1, t0=0.0)
            p.push(6, w.dt)
            p.download(host, host_id=ids)
        else:
            p.push_host(host, 6, w.dt, n_chunks=chunks, host_id=ids)
        r = {k: np.empty(w.n_markers) for k in KEYS}
        for k in KEYS:
            r[k][ids.numpy()] = host[k].numpy()
        out[chunks] = r
    for chunks in (1, 4):
        for k in KEYS:
            assert np.array_equal(out[chunks][k], out[0][k]), (chunks, k)


def test_sort_workspace_is_recarved_on_reinit_with_a_larger_n():
    """an oversized sort workspace must be carved again when m3dk_particles_init comes with another n."""
    import ctypes as C
    w_small = synth.make_config(1, n_markers=2000, nx=32)
    w_big = synth.make_config(1, n_markers=6000 + 5, nx=32)
    p = make_pusher(w_small, verify=False, sort_interval=1)
    # a workspace large enough for the bigger marker set, bound while the small one is registered
    p.n = w_big.n_markers
    big_bytes = p.sort_workspace_bytes()
    p.n = w_small.n_markers
    ws = p._empty(big_bytes)
    p._ck(p.L.m3dk_set_sort_workspace(p.h, p._p(ws), ws.numel()))
    p._keep["sort_ws"] = ws
    p.push(2, w_small.dt)
    # re-init with the bigger set WITHOUT giving a new workspace: the library must re-carve the one it has
    p.particles_init(w_big.markers, w_big.charge, w_big.mass, w_big.f0, with_sort_workspace=False)
    p.set_options(sort_interval=1, t0=0.0)
    p.push(4, w_big.dt)
    got, _, ids = p.state()
    q = make_pusher(w_big, verify=False, sort_interval=0)
    q.push(4, w_big.dt)
    want, _, _ = q.state()
    assert np.array_equal(np.sort(ids), np.arange(w_big.n_markers))
    for k in KEYS:
        assert np.array_equal(got[k], want[k]), k


def test_fields_attach_binds_a_copy_of_the_workspace():
    """m3dk_fields_attach on a byte-for-byte copy of another context's fields workspace (what the NCCL broadcast of
    bench.py --gpus N delivers): no host tables, same search and field evaluation, same pushed bits."""
    import paper_2107_13663_b200 as m3dk
    w = synth.make_config(3, n_markers=4000 + 9, nx=48)
    a = make_pusher(w, verify=False, sort_interval=1)
    copy = a.fields_workspace().clone()
    b = m3dk.Pusher(device=0, verify=False)
    b.fields_attach(copy, w.n_elems, w.n_modes)
    b.particles_init(w.markers, w.charge, w.mass, w.f0)
    b.set_options(sort_interval=1, t0=0.0)
    a.push(5, w.dt)
    b.push(5, w.dt)
    ra, ea, _ = a.state()
    rb, eb, _ = b.state()
    assert np.array_equal(ea, eb)
    for k in KEYS:
        assert np.array_equal(ra[k], rb[k]), k
    garbage = torch.zeros(4096, dtype=torch.uint8, device="cuda")
    with pytest.raises(m3dk.M3DKError):
        m3dk.Pusher(device=0, verify=False).fields_attach(garbage, 1, 0)


@pytest.mark.parametrize("mode", [1, 2, 3])
def test_push_host_two_chunks_in_flight_in_the_other_modes(mode):
    """The chunk pipeline keeps two chunks in flight on two compute streams, each with its own carving of the sort and
    FLR workspaces: non-linear mode and the FLR ring streams (modes 2 and 3) against the oracle, 5 chunks (odd: the slots alternate
    unevenly), and bitwise against the one-chunk call."""
    w = synth.make_config(3, n_markers=7000 + 13, nx=48)
    mesh, sp = oracle_of(w, mode=mode)
    nsteps = 4
    ref, e_ref, _ = oracle_push(mesh, sp, w.markers, nsteps, w.dt)
    out = {}
    for chunks in (1, 5):
        p = make_pusher(w, verify=True, sort_interval=1, mode=mode)
        host = _pinned(w.markers)
        ids = torch.empty(w.n_markers, dtype=torch.int32).pin_memory()
        p.push_host(host, nsteps, w.dt, n_chunks=chunks, host_id=ids)
        assert np.array_equal(np.sort(ids.numpy()), np.arange(w.n_markers))
        r = {k: np.empty(w.n_markers) for k in KEYS}
        for k in KEYS:
            r[k][ids.numpy()] = host[k].numpy()
        out[chunks] = r
    live = e_ref >= 0
    wrms = np.sqrt(np.mean(ref["w"][live] ** 2))
    ex, ev, ew = g16_errors(take(out[5], live), take(ref, live), w_floor=wrms)
    assert max(ex.max(), ev.max(), ew.max()) <= nsteps * TOL_STEP, (ex.max(), ev.max(), ew.max())
    for k in KEYS:
        assert np.array_equal(out[5][k], out[1][k]), k
