"""GPU test of m3dk_deposit_noalloc (include/m3dk.h): the element-ordered deposition with its ordering scratch in the
library's static device array, for callers that cannot allocate device memory.  Collected last on purpose (the file name
sorts after every other test file): the suite runs with pytest -x.

The output is compared with the existing path, m3dk_deposit with a caller-lent sort workspace, on two calls in a row (the
second on other marker data and other flags: the static array keeps the first call's contents).  The sums are accumulated
with fp64 atomics in both paths, so the comparison carries the tolerance of tests/test_gpu_deposit.py: 1e-12 of the sum
of the absolute contributions to an element and moment (from the oracle, as there), and both paths are also held to the
oracle itself."""
import dataclasses

import numpy as np
import pytest
import torch

import oracle
import synth
from gpu_helpers import make_pusher, oracle_of

pytestmark = pytest.mark.gpu


def _abs_scale(w, markers, bound_b1=0.0):
    mesh, sp = oracle_of(w)
    absw = dict(markers)
    absw["w"] = np.abs(markers["w"]) + bound_b1
    scale, _ = oracle.deposit(mesh, sp, absw)
    return np.abs(scale[:, :, 0, 0])[:, :, None, None] + np.abs(scale).max() * 1e-3


def _both_paths(p, w, flags, t):
    rhs = torch.full((p.deposit_bytes() // 8,), float("nan"), dtype=torch.float64, device=p.device)
    p.deposit_noalloc_into(rhs, flags, t)
    p.stats()                                                   # synchronise, surface asynchronous errors
    got = rhs.cpu().numpy().reshape(w.n_elems, 2, 1 + 2 * w.n_modes, 21)
    ref = p.deposit(flags=flags, t=t)                           # existing path: the caller's sort workspace
    return got, ref


def test_noalloc_deposit_matches_the_workspace_path_on_two_calls_in_a_row():
    w0 = synth.make_config(3, n_markers=30000 + 7, nx=32, amp=1e-2)
    rng = np.random.Generator(np.random.PCG64(77))
    mk = {k: v.copy() for k, v in w0.markers.items()}
    mk["w"] = rng.normal(size=w0.n_markers) * 1e-2
    w = dataclasses.replace(w0, markers=mk)
    p = make_pusher(w, verify=True, sort_interval=1)
    assert p.noalloc_scratch_bytes() == 8 << 20
    mesh, sp = oracle_of(w)

    # call 1: plain deposition of the loaded markers
    got1, ref1 = _both_paths(p, w, 0, 0.0)
    S1 = _abs_scale(w, mk)
    assert np.isfinite(got1).all() and np.abs(ref1).max() > 0
    assert (np.abs(got1 - ref1) <= 1e-12 * S1).all(), float((np.abs(got1 - ref1) / S1).max())
    orc1, _ = oracle.deposit(mesh, sp, mk, flags=0, t=0.0)
    assert (np.abs(got1 - orc1) <= 1e-12 * S1).all()

    # call 2, straight after: the markers have moved (other elements, other counts per element, some lost) and the
    # deposition carries the B1par term and the Jacobian substitution; the array still holds call 1's ordering
    p.push(7, w.dt)
    raw, elem, _ = p.state(by_id=False)
    got2, ref2 = _both_paths(p, w, 5, 0.7)
    S2 = _abs_scale(w, raw, bound_b1=2e-2)
    assert (np.abs(got2 - ref2) <= 1e-11 * S2).all(), float((np.abs(got2 - ref2) / S2).max())
    orc2, lost = oracle.deposit(mesh, sp, raw, flags=5, t=0.7)
    assert lost == int((elem < 0).sum())
    assert (np.abs(got2 - orc2) <= 1e-11 * S2).all()
    assert np.abs(got2 - got1).max() > 1e-3 * np.abs(got1).max()            # the two calls did differ

    # call 3: the 4-point deposition on the ordered records, and the first result again (nothing leaked between calls)
    got3, ref3 = _both_paths(p, w, 3, 0.7)
    assert np.abs(got3 - ref3).max() <= 1e-11 * np.abs(ref3).max()
    p.set_state(mk)
    got4, _ = _both_paths(p, w, 0, 0.0)
    assert (np.abs(got4 - got1) <= 1e-12 * S1).all()


def test_noalloc_deposit_needs_no_workspace_and_rejects_sizes_beyond_the_array():
    """A context WITHOUT any sort workspace still gets the ordered deposition; a marker count whose ordering scratch
    exceeds the static array is refused with a clear error and nothing is enqueued."""
    import paper_2107_13663_b200 as m3dk
    w = synth.make_config(1, n_markers=12000 + 5, nx=32)
    rng = np.random.Generator(np.random.PCG64(78))
    mk = {k: v.copy() for k, v in w.markers.items()}
    mk["w"] = rng.normal(size=w.n_markers)
    p = m3dk.Pusher(device=0, verify=False)
    p.fields_create(w.node_RZ, w.tri, w.eq_coef, w.n_tor, w.omega, w.pert_coef)
    p.particles_init(mk, w.charge, w.mass, w.f0, with_sort_workspace=False)
    rhs = torch.empty(p.deposit_bytes() // 8, dtype=torch.float64, device=p.device)
    p.deposit_noalloc_into(rhs, 1, 1.3)
    p.stats()
    got = rhs.cpu().numpy().reshape(w.n_elems, 2, 1 + 2 * w.n_modes, 21)
    ref, _ = oracle.deposit(*oracle_of(w), mk, flags=1, t=1.3)
    assert np.abs(got - ref).max() <= 1e-11 * np.abs(ref).max()

    big = synth.make_config(1, n_markers=80000, nx=32)
    q = m3dk.Pusher(device=0, verify=False)
    q.fields_create(big.node_RZ, big.tri, big.eq_coef, big.n_tor, big.omega, big.pert_coef)
    q.particles_init(big.markers, big.charge, big.mass, big.f0, with_sort_workspace=False)
    rhs2 = torch.full((q.deposit_bytes() // 8,), 7.0, dtype=torch.float64, device=q.device)
    with pytest.raises(m3dk.M3DKError) as ei:
        q.deposit_noalloc_into(rhs2, 0, 0.0)
    assert "M3DK_NOALLOC_SCRATCH_BYTES" in str(ei.value) and "80000 markers" in str(ei.value)
    q.stats()
    assert bool((rhs2 == 7.0).all())                                        # untouched: nothing was enqueued
