"""ctypes binding of libm3dk: same names as include/m3dk.h, argument marshalling only."""
from __future__ import annotations

import ctypes as C
import os
import re
from typing import Dict, Optional

import numpy as np

from . import _build

F0_MAXWELLIAN, F0_SLOWING_DOWN, F0_BEAM_PITCH = 0, 1, 2
STATE_KEYS = ("x", "y", "z", "vx", "vy", "vz", "mu", "w")

_c_dp = C.POINTER(C.c_double)
_c_ip = C.POINTER(C.c_int)
_libs: Dict[bool, C.CDLL] = {}


class M3DKError(RuntimeError):
    def __init__(self, code: int, msg: str):
        super().__init__(f"libm3dk error {code}: {msg}")
        self.code = code


class _F0(C.Structure):
    _fields_ = [("kind", C.c_int), ("T", C.c_double), ("v_c", C.c_double), ("Lambda0", C.c_double),
                ("dLambda", C.c_double), ("B_axis", C.c_double)]


class _Stats(C.Structure):
    _fields_ = [("n_markers", C.c_long), ("n_lost", C.c_long), ("steps_done", C.c_long), ("n_sorts", C.c_long),
                ("t", C.c_double)]


class _Timing(C.Structure):
    _fields_ = [("push_ms", C.c_double), ("sort_ms", C.c_double), ("push_launches", C.c_long),
                ("sort_launches", C.c_long), ("kernel_launches", C.c_long)]


def lib_path(verify: bool = False) -> str:
    return _build.lib_path(verify)


def exported_symbols():
    """Function names include/m3dk.h declares (parsed from the header itself)."""
    hdr = os.path.join(os.path.dirname(os.path.dirname(os.path.abspath(__file__))), "include", "m3dk.h")
    with open(hdr) as fh:
        text = fh.read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(m3dk_[a-z0-9_]+)\s*\(", text)))


def lib(verify: bool = False) -> C.CDLL:
    """Load libm3dk.so (timing build) or libm3dk_verify.so (no FMA contraction).  Fails loudly if it is missing."""
    if verify in _libs:
        return _libs[verify]
    path = lib_path(verify)
    if not os.path.exists(path):
        raise M3DKError(-4, f"{path} is not built: run `python -m paper_2107_13663_b200._build` (no CPU fallback exists)")
    L = C.CDLL(path)
    vp, sz, dbl, lng, i = C.c_void_p, C.c_size_t, C.c_double, C.c_long, C.c_int
    sig = {
        "m3dk_version": ([], i),
        "m3dk_create": ([C.POINTER(vp), i, vp], i),
        "m3dk_destroy": ([vp], i),
        "m3dk_last_error": ([vp], C.c_char_p),
        "m3dk_fields_workspace_bytes": ([i, i, i, C.POINTER(sz)], i),
        "m3dk_fields_create": ([vp, i, _c_dp, i, _c_ip, _c_dp, i, _c_ip, _c_dp, _c_dp, vp, sz], i),
        "m3dk_fields_attach": ([vp, vp, sz], i),
        "m3dk_particles_init": ([vp, lng] + [vp] * 10 + [dbl, dbl, C.POINTER(_F0)], i),
        "m3dk_set_options": ([vp, i, i, dbl], i),
        "m3dk_set_push_variant": ([vp, i], i),
        "m3dk_sort_workspace_bytes": ([lng, i, C.POINTER(sz)], i),
        "m3dk_set_sort_workspace": ([vp, vp, sz], i),
        "m3dk_flr_workspace_bytes": ([lng, i, C.POINTER(sz)], i),
        "m3dk_flr_workspace_bytes_nl": ([lng, i, C.POINTER(sz)], i),
        "m3dk_set_flr_workspace": ([vp, vp, sz], i),
        "m3dk_push": ([vp, i, dbl], i),
        "m3dk_sort": ([vp, vp, sz], i),
        "m3dk_stats": ([vp, C.POINTER(_Stats)], i),
        "m3dk_particles_upload": ([vp] + [vp] * 8, i),
        "m3dk_particles_download": ([vp] + [vp] * 10, i),
        "m3dk_push_host": ([vp] + [vp] * 10 + [i, dbl, i], i),
        "m3dk_eval_fields": ([vp, lng, vp, vp, vp, dbl, vp, vp], i),
        "m3dk_gc_push": ([vp, i, dbl, vp], i),
        "m3dk_gc_bootstrap": ([vp, dbl, vp], i),
        "m3dk_deposit_bytes": ([vp, C.POINTER(sz)], i),
        "m3dk_deposit": ([vp, vp, i, dbl], i),
        "m3dk_noalloc_scratch_bytes": ([C.POINTER(sz)], i),
        "m3dk_deposit_noalloc": ([vp, vp, i, dbl], i),
        "m3dk_fp64_peak_tflops": ([vp, _c_dp], i),
        "m3dk_set_profiling": ([vp, i], i),
        "m3dk_timing": ([vp, C.POINTER(_Timing)], i),
    }
    for name, (args, res) in sig.items():
        fn = getattr(L, name)  # AttributeError if the library does not export what the header declares
        fn.argtypes, fn.restype = args, res
    _libs[verify] = L
    return L


def _np_d(a):
    return np.ascontiguousarray(a, dtype=np.float64)


class Pusher:
    """One libm3dk context on one CUDA device / stream, with the torch tensors it borrows kept alive.

    >>> p = Pusher(device=0)
    >>> p.fields_create(node_RZ, tri, eq_coef, n_tor, omega, pert_coef)
    >>> p.particles_init(markers, charge, mass, f0)          # numpy dict -> device tensors
    >>> p.set_options(sort_interval=10, t0=0.0)
    >>> p.push(nsteps, dt)
    >>> out = p.state()                                        # dict of numpy arrays ordered by marker id
    """

    def __init__(self, device: int = 0, verify: bool = False, stream=None):
        import torch  # device memory and streams only

        if not torch.cuda.is_available():
            raise M3DKError(-4, "no CUDA device: libm3dk has no CPU fallback")
        self.torch = torch
        self.L = lib(verify)
        self.verify = verify
        self.device = torch.device("cuda", device)
        torch.cuda.set_device(self.device)
        self.stream = stream if stream is not None else torch.cuda.current_stream(self.device)
        h = C.c_void_p()
        rc = self.L.m3dk_create(C.byref(h), device, C.c_void_p(self.stream.cuda_stream))
        if rc != 0:
            raise M3DKError(rc, (self.L.m3dk_last_error(None) or b"").decode())
        self.h = h
        self.n = 0
        self.n_elems = 0
        self.n_modes = 0
        self._keep = {}

    # ---- plumbing -------------------------------------------------------------------------------------------
    def _ck(self, rc: int):
        if rc != 0:
            raise M3DKError(rc, (self.L.m3dk_last_error(self.h) or b"").decode())

    def close(self):
        if getattr(self, "h", None):
            self.L.m3dk_destroy(self.h)
            self.h = None
            self._keep.clear()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _empty(self, nbytes: int):
        return self.torch.empty(max(int(nbytes), 256), dtype=self.torch.uint8, device=self.device)

    @staticmethod
    def _p(t):
        return C.c_void_p(t.data_ptr())

    # ---- m3dk_fields_create ---------------------------------------------------------------------------------
    def fields_create(self, node_RZ, tri, eq_coef, n_tor=None, omega=None, pert_coef=None):
        node_RZ = _np_d(node_RZ)
        tri = np.ascontiguousarray(tri, dtype=np.int32)
        eq_coef = _np_d(eq_coef)
        n_modes = 0 if n_tor is None else int(len(n_tor))
        n_nodes, n_elems = node_RZ.shape[0], tri.shape[0]
        assert eq_coef.shape == (n_elems, 4, 21)
        if n_modes:
            n_tor = np.ascontiguousarray(n_tor, dtype=np.int32)
            omega = _np_d(omega)
            pert_coef = _np_d(pert_coef)
            assert pert_coef.shape == (n_modes, n_elems, 7, 2, 21)
        need = C.c_size_t()
        self._ck(self.L.m3dk_fields_workspace_bytes(n_nodes, n_elems, n_modes, C.byref(need)))
        ws = self._empty(need.value)
        self._ck(self.L.m3dk_fields_create(
            self.h, n_nodes, node_RZ.ctypes.data_as(_c_dp), n_elems, tri.ctypes.data_as(_c_ip),
            eq_coef.ctypes.data_as(_c_dp), n_modes,
            n_tor.ctypes.data_as(_c_ip) if n_modes else None, omega.ctypes.data_as(_c_dp) if n_modes else None,
            pert_coef.ctypes.data_as(_c_dp) if n_modes else None, self._p(ws), ws.numel()))
        self._keep["fields_ws"] = ws
        self.n_elems, self.n_modes = n_elems, n_modes
        self.fields_bytes = need.value

    def fields_workspace(self):
        """The device tensor (uint8) that holds the fields image: what a broadcast to the other ranks sends."""
        return self._keep["fields_ws"]

    def fields_attach(self, ws, n_elems: int, n_modes: int):
        """m3dk_fields_attach: bind a byte-for-byte copy of another context's fields workspace (a uint8 device tensor)."""
        self._ck(self.L.m3dk_fields_attach(self.h, self._p(ws), ws.numel()))
        self._keep["fields_ws"] = ws
        self.n_elems, self.n_modes = int(n_elems), int(n_modes)
        self.fields_bytes = ws.numel()

    # ---- m3dk_particles_init --------------------------------------------------------------------------------
    def _f0(self, f0) -> _F0:
        s = _F0()
        if f0 is None:
            s.kind, s.T, s.v_c, s.Lambda0, s.dLambda, s.B_axis = 0, 1.0, 0.3, 0.75, 0.2, 1.0
        else:
            s.kind, s.T, s.v_c = int(f0.kind), float(f0.T), float(f0.v_c)
            s.Lambda0, s.dLambda, s.B_axis = float(f0.Lambda0), float(f0.dLambda), float(f0.B_axis)
        return s

    def particles_alloc(self, n: int, charge: float, mass: float, f0=None, with_sort_workspace: bool = True):
        """Allocate the device arrays for n markers (uninitialised) and register them; fill with upload()."""
        t = self.torch
        self.n = int(n)
        self.state_t = {k: t.empty(self.n, dtype=t.float64, device=self.device) for k in STATE_KEYS}
        self.elem_t = t.empty(self.n, dtype=t.int32, device=self.device)
        self.id_t = t.empty(self.n, dtype=t.int32, device=self.device)
        self._species = (float(charge), float(mass), self._f0(f0))
        self._register(locate=False)
        if with_sort_workspace:
            self.set_sort_workspace()

    def _register(self, locate=True):
        q, m, f0 = self._species
        if not locate:
            # arrays are uninitialised: give the locate kernel finite positions
            for k in ("x", "y", "z"):
                self.state_t[k].fill_(1.0)
        self._ck(self.L.m3dk_particles_init(
            self.h, self.n, *[self._p(self.state_t[k]) for k in STATE_KEYS], self._p(self.elem_t), self._p(self.id_t),
            q, m, C.byref(f0)))

    def particles_init(self, markers: dict, charge: float, mass: float, f0=None, with_sort_workspace: bool = True):
        """Device arrays from a dict of numpy arrays (x, y, z, vx, vy, vz, mu, w) and m3dk_particles_init."""
        t = self.torch
        self.n = int(np.asarray(markers["x"]).shape[0])
        self.state_t = {k: t.from_numpy(_np_d(markers[k]).copy()).to(self.device) for k in STATE_KEYS}
        self.elem_t = t.empty(self.n, dtype=t.int32, device=self.device)
        self.id_t = t.empty(self.n, dtype=t.int32, device=self.device)
        self._species = (float(charge), float(mass), self._f0(f0))
        self._register()
        if with_sort_workspace:
            self.set_sort_workspace()

    def set_state(self, markers: dict):
        """Overwrite the device arrays (slot i <- marker i) and re-register (re-locates, id = 0..n-1)."""
        t = self.torch
        for k in STATE_KEYS:
            self.state_t[k].copy_(t.from_numpy(_np_d(markers[k])))
        self._register()

    # ---- options, sort ----------------------------------------------------------------------------------------
    def set_options(self, sort_interval: int = 0, mode: int = 0, t0: float = 0.0):
        self._ck(self.L.m3dk_set_options(self.h, int(sort_interval), int(mode), float(t0)))

    def set_push_variant(self, variant: int):
        self._ck(self.L.m3dk_set_push_variant(self.h, int(variant)))

    def sort_workspace_bytes(self) -> int:
        need = C.c_size_t()
        self._ck(self.L.m3dk_sort_workspace_bytes(self.n, self.n_elems, C.byref(need)))
        return int(need.value)

    def set_sort_workspace(self):
        ws = self._empty(self.sort_workspace_bytes())
        self._ck(self.L.m3dk_set_sort_workspace(self.h, self._p(ws), ws.numel()))
        self._keep["sort_ws"] = ws

    def set_flr_workspace(self, nonlinear: bool = False):
        """Allocate and lend the FLR workspace (ring stream of the ordered mode 2 and of the FLR deposition; nonlinear:
        the larger one that also carries the ring stream of mode 3)."""
        need = C.c_size_t()
        fn = self.L.m3dk_flr_workspace_bytes_nl if nonlinear else self.L.m3dk_flr_workspace_bytes
        self._ck(fn(self.n, self.n_elems, C.byref(need)))
        ws = self._empty(need.value)
        self._ck(self.L.m3dk_set_flr_workspace(self.h, self._p(ws), ws.numel()))
        self._keep["flr_ws"] = ws

    def push(self, nsteps: int, dt: float):
        self._ck(self.L.m3dk_push(self.h, int(nsteps), float(dt)))

    def sort(self):
        self._ck(self.L.m3dk_sort(self.h, None, 0))

    def stats(self) -> dict:
        s = _Stats()
        self._ck(self.L.m3dk_stats(self.h, C.byref(s)))
        return {k: getattr(s, k) for k, _ in _Stats._fields_}

    def set_profiling(self, on: bool):
        self._ck(self.L.m3dk_set_profiling(self.h, int(bool(on))))

    def timing(self) -> dict:
        s = _Timing()
        self._ck(self.L.m3dk_timing(self.h, C.byref(s)))
        return {k: getattr(s, k) for k, _ in _Timing._fields_}

    # ---- host-buffer path -------------------------------------------------------------------------------------
    def upload(self, host: dict):
        """host: dict of (pinned) torch CPU tensors or numpy arrays, fp64, length n."""
        ptrs = []
        for k in STATE_KEYS:
            a = host[k]
            ptrs.append(C.c_void_p(a.data_ptr() if hasattr(a, "data_ptr") else a.ctypes.data))
        self._ck(self.L.m3dk_particles_upload(self.h, *ptrs))

    def download(self, host: dict, host_id=None, host_elem=None):
        ptrs = []
        for k in STATE_KEYS:
            a = host[k]
            ptrs.append(C.c_void_p(a.data_ptr() if hasattr(a, "data_ptr") else a.ctypes.data))
        for a in (host_id, host_elem):
            ptrs.append(None if a is None else C.c_void_p(a.data_ptr() if hasattr(a, "data_ptr") else a.ctypes.data))
        self._ck(self.L.m3dk_particles_download(self.h, *ptrs))

    def push_host(self, host: dict, nsteps: int, dt: float, n_chunks: int = 1, host_id=None, host_elem=None):
        """m3dk_push_host: upload, nsteps steps and download pipelined by marker chunk, in place on the (pinned) host
        buffers of ``host`` (dict of torch CPU tensors or numpy arrays, fp64, length n).  Synchronises."""
        ptrs = []
        for k in STATE_KEYS:
            a = host[k]
            ptrs.append(C.c_void_p(a.data_ptr() if hasattr(a, "data_ptr") else a.ctypes.data))
        for a in (host_id, host_elem):
            ptrs.append(None if a is None else C.c_void_p(a.data_ptr() if hasattr(a, "data_ptr") else a.ctypes.data))
        self._ck(self.L.m3dk_push_host(self.h, *ptrs, int(nsteps), float(dt), int(n_chunks)))

    # ---- results ------------------------------------------------------------------------------------------------
    def state(self, by_id: bool = True):
        """Synchronise and return (dict of numpy arrays, elem, id).  by_id: rows reordered so row k is marker id k."""
        self.stats()
        out = {k: self.state_t[k].cpu().numpy() for k in STATE_KEYS}
        elem = self.elem_t.cpu().numpy()
        ids = self.id_t.cpu().numpy()
        if by_id:
            inv = np.empty_like(ids)
            inv[ids] = np.arange(ids.shape[0], dtype=ids.dtype)
            out = {k: v[inv] for k, v in out.items()}
            elem = elem[inv]
        return out, elem, ids

    # ---- diagnostics ----------------------------------------------------------------------------------------------
    def eval_fields(self, R, phi, Z, t: float = 0.0):
        tt = self.torch
        R_t = tt.from_numpy(_np_d(R)).to(self.device)
        p_t = tt.from_numpy(_np_d(phi)).to(self.device)
        Z_t = tt.from_numpy(_np_d(Z)).to(self.device)
        n = R_t.numel()
        elem = tt.empty(n, dtype=tt.int32, device=self.device)
        out = tt.full((n, 18), float("nan"), dtype=tt.float64, device=self.device)
        self._ck(self.L.m3dk_eval_fields(self.h, n, self._p(R_t), self._p(p_t), self._p(Z_t), float(t), self._p(elem),
                                         self._p(out)))
        self.stats()
        return elem.cpu().numpy(), out.cpu().numpy()

    def gc_push(self, nsteps: int, dt: float, vpar):
        """m3dk_gc_push: RK4 guiding-centre steps; vpar is a numpy array (copied to the device and back).  Returns
        (x, y, z, vpar, elem) as numpy arrays in slot order (synchronises)."""
        t = self.torch
        vp = t.from_numpy(_np_d(vpar).copy()).to(self.device)
        self._ck(self.L.m3dk_gc_push(self.h, int(nsteps), float(dt), self._p(vp)))
        self.stats()
        self._keep["vpar"] = vp
        return (self.state_t["x"].cpu().numpy(), self.state_t["y"].cpu().numpy(), self.state_t["z"].cpu().numpy(),
                vp.cpu().numpy(), self.elem_t.cpu().numpy())

    def gc_bootstrap(self, dt: float, vpar):
        """m3dk_gc_bootstrap: (x, v) <- (x_1, (x_1 - x_0)/dt) from one RK4 guiding-centre step; vpar is a numpy array."""
        vp = self.torch.from_numpy(_np_d(vpar).copy()).to(self.device)
        self._keep["vpar_boot"] = vp
        self._ck(self.L.m3dk_gc_bootstrap(self.h, float(dt), self._p(vp)))

    def gc_push_into(self, nsteps: int, dt: float, vpar_t):
        """m3dk_gc_push on a caller's device tensor vpar [n] (asynchronous)."""
        self._ck(self.L.m3dk_gc_push(self.h, int(nsteps), float(dt), self._p(vpar_t)))

    def deposit_bytes(self) -> int:
        need = C.c_size_t()
        self._ck(self.L.m3dk_deposit_bytes(self.h, C.byref(need)))
        return int(need.value)

    def deposit_into(self, rhs, flags: int = 0, t: float = 0.0):
        """m3dk_deposit into a caller's device tensor of deposit_bytes() bytes (asynchronous)."""
        self._ck(self.L.m3dk_deposit(self.h, self._p(rhs), int(flags), float(t)))

    def deposit(self, flags: int = 0, t: float = 0.0):
        """m3dk_deposit into a fresh device tensor; returns it as numpy [n_elems][2][1 + 2 n_modes][21] (synchronises)."""
        need = C.c_size_t()
        self._ck(self.L.m3dk_deposit_bytes(self.h, C.byref(need)))
        rhs = self.torch.empty(need.value // 8, dtype=self.torch.float64, device=self.device)
        self._ck(self.L.m3dk_deposit(self.h, self._p(rhs), int(flags), float(t)))
        self.stats()
        self._keep["rhs"] = rhs
        return rhs.cpu().numpy().reshape(self.n_elems, 2, 1 + 2 * self.n_modes, 21)

    def noalloc_scratch_bytes(self) -> int:
        need = C.c_size_t()
        self._ck(self.L.m3dk_noalloc_scratch_bytes(C.byref(need)))
        return int(need.value)

    def deposit_noalloc_into(self, rhs, flags: int = 0, t: float = 0.0):
        """m3dk_deposit_noalloc into a caller's device tensor of deposit_bytes() bytes (asynchronous): the ordered
        deposition with its scratch in the library's static device array; raises M3DKError beyond its size limit."""
        self._ck(self.L.m3dk_deposit_noalloc(self.h, self._p(rhs), int(flags), float(t)))

    def fp64_peak_tflops(self) -> float:
        v = C.c_double()
        self._ck(self.L.m3dk_fp64_peak_tflops(self.h, C.byref(v)))
        return float(v.value)
