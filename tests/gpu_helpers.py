"""Helpers of the GPU parity tests: error norms of reading G16 and oracle/GPU drivers on the same seeded inputs.

Nothing here contains arithmetic of the method: it only calls oracle/ (CPU) and the libm3dk binding (CUDA).
"""
import numpy as np

import oracle
import paper_2107_13663_b200 as m3dk

KEYS = m3dk.STATE_KEYS


def g16_errors(got: dict, ref: dict, w_floor=None):
    """Per-marker relative errors (reading G16): |dx|_2/|x|_2, |dv|_2/|v|_2, |dw|/max(|w|, w_rms of the ensemble)."""
    dx = np.sqrt(sum((got[k] - ref[k]) ** 2 for k in ("x", "y", "z")))
    nx = np.sqrt(sum(ref[k] ** 2 for k in ("x", "y", "z")))
    dv = np.sqrt(sum((got[k] - ref[k]) ** 2 for k in ("vx", "vy", "vz")))
    nv = np.sqrt(sum(ref[k] ** 2 for k in ("vx", "vy", "vz")))
    wrms = float(np.sqrt(np.mean(ref["w"] ** 2))) if w_floor is None else float(w_floor)
    den = np.maximum(np.abs(ref["w"]), wrms)
    dw = np.abs(got["w"] - ref["w"])
    ew = np.where(den > 0, dw / np.where(den > 0, den, 1.0), dw)
    return dx / nx, dv / nv, ew


def take(markers: dict, idx):
    return {k: np.ascontiguousarray(markers[k][idx]) for k in KEYS}


def make_pusher(w, verify=True, markers=None, sort_interval=0, t0=0.0, mode=0, flr_ws=True):
    """flr_ws: in mode 2 with the ordered pipeline, also lend the FLR workspace (ring stream); False = every lane gathers."""
    p = m3dk.Pusher(device=0, verify=verify)
    p.fields_create(w.node_RZ, w.tri, w.eq_coef, w.n_tor if w.n_modes else None, w.omega if w.n_modes else None,
                    w.pert_coef if w.n_modes else None)
    p.particles_init(w.markers if markers is None else markers, w.charge, w.mass, w.f0)
    p.set_options(sort_interval=sort_interval, mode=mode, t0=t0)
    if mode in (2, 3) and sort_interval > 0 and flr_ws:
        p.set_flr_workspace(nonlinear=(mode == 3))
    return p


def oracle_of(w, mode=0):
    return oracle.Mesh.of(w), oracle.species_of(w, mode=mode)


def oracle_push(mesh, sp, markers, nsteps, dt, t0=0.0, step0=0, elem=None):
    st, e, lost = oracle.push_fe(mesh, sp, markers, nsteps, dt, t0=t0, step0=step0, elem=elem)
    return st, e, lost
