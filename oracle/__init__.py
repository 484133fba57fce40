"""ctypes binding of the CPU fp64 oracle (oracle/m3dk_oracle.c).

TEST INFRASTRUCTURE ONLY: imported by tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
``--impl reference`` legs.  Never imported by paper_2107_13663_b200 (the product path), and it imports
nothing from it.  ``build()`` compiles the C file in-tree with gcc -O2 -ffp-contract=off -fopenmp.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from typing import Optional

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "m3dk_oracle.c")
_SO = os.path.join(_HERE, "libm3dk_oracle.so")
_lib = None

c_dp = C.POINTER(C.c_double)
c_ip = C.POINTER(C.c_int)
c_lp = C.POINTER(C.c_long)


class Analytic(C.Structure):
    _fields_ = [("R0", C.c_double), ("a", C.c_double), ("B0", C.c_double), ("qkind", C.c_int),
                ("qc", C.c_double * 3), ("kappa", C.c_double), ("pA", C.c_double), ("prc", C.c_double),
                ("pwd", C.c_double), ("pomega", C.c_double), ("pn", C.c_int), ("pm", C.c_int)]


class Species(C.Structure):
    _fields_ = [("charge", C.c_double), ("mass", C.c_double), ("f0kind", C.c_int), ("f0par", C.c_double * 5),
                ("mode", C.c_int)]


def build(force: bool = False) -> str:
    if force or not os.path.exists(_SO) or os.path.getmtime(_SO) < os.path.getmtime(_SRC):
        cmd = ["gcc", "-O2", "-ffp-contract=off", "-fopenmp", "-fPIC", "-shared", "-Wall", "-o", _SO, _SRC, "-lm"]
        subprocess.run(cmd, check=True)
    return _SO


def _configure(L):
    """Declare the argument / result types of every exported oracle function on the loaded library L."""
    L.orc_mesh_create.restype = C.c_void_p
    L.orc_mesh_create.argtypes = [C.c_int, c_dp, C.c_int, c_ip, c_dp, C.c_int, c_ip, c_dp, c_dp]
    L.orc_mesh_free.argtypes = [C.c_void_p]
    L.orc_locate.argtypes = [C.c_void_p, C.c_long, c_dp, c_dp, c_ip, C.c_int]
    L.orc_eval_fe.argtypes = [C.c_void_p, C.c_long, c_dp, c_dp, c_dp, C.c_double, c_ip, c_dp]
    L.orc_eval_analytic.argtypes = [C.POINTER(Analytic), C.c_long, c_dp, c_dp, c_dp, C.c_double, c_dp, c_dp]
    L.orc_push_fe.restype = C.c_long
    L.orc_push_fe.argtypes = [C.c_void_p, C.POINTER(Species), C.c_long] + [c_dp] * 8 + [c_ip, C.c_int, C.c_double,
                              C.c_double, C.c_long, C.c_int, C.c_int]
    L.orc_push_analytic.restype = C.c_long
    L.orc_push_analytic.argtypes = [C.POINTER(Analytic), C.POINTER(Species), C.c_long] + [c_dp] * 8 + [
        C.c_int, C.c_double, C.c_double, C.c_long, C.c_int]
    L.orc_gyro_ring.argtypes = [C.c_void_p, C.POINTER(Analytic), C.POINTER(Species), c_dp, C.c_double, c_dp]
    L.orc_flr_fields.argtypes = [C.c_void_p, C.POINTER(Analytic), C.POINTER(Species), c_dp, C.c_double, C.c_double, c_dp]
    L.orc_gc_push.restype = C.c_long
    L.orc_gc_push.argtypes = [C.c_void_p, C.POINTER(Analytic), C.POINTER(Species), C.c_long] + [c_dp] * 5 + [c_ip, C.c_int,
                              C.c_double, C.c_double, C.c_int]
    L.orc_gc_rhs.argtypes = [C.c_void_p, C.POINTER(Analytic), C.POINTER(Species), C.c_long] + [c_dp] * 5 + [C.c_double, c_dp]
    L.orc_gc_bootstrap.argtypes = [C.c_void_p, C.POINTER(Analytic), C.POINTER(Species), C.c_long] + [c_dp] * 5 + [C.c_double] + [c_dp] * 3 + [c_ip]
    L.orc_gc_fields.argtypes = [C.c_void_p, C.POINTER(Analytic), C.c_long, c_dp, c_dp, c_ip, c_dp]
    L.orc_deposit.restype = C.c_long
    L.orc_deposit.argtypes = [C.c_void_p, C.POINTER(Species), C.c_long] + [c_dp] * 8 + [c_dp, C.c_int, C.c_double]
    L.orc_trace.restype = C.c_long
    L.orc_trace.argtypes = [C.c_void_p, C.POINTER(Analytic), C.POINTER(Species), c_dp, C.c_long, C.c_double,
                            C.c_double, C.c_long, c_dp]
    L.orc_push_uniform.argtypes = [C.c_long] + [c_dp] * 6 + [c_dp, c_dp, C.c_double, C.c_double, C.c_long, C.c_double]
    L.orc_eq6.argtypes = [c_dp, c_dp, c_dp, C.c_double, c_dp]
    L.orc_weight_rhs.restype = C.c_double
    L.orc_weight_rhs.argtypes = [c_dp, C.POINTER(Species), C.c_double, c_dp, C.c_double]
    L.orc_sort_perm.argtypes = [C.c_long, c_ip, C.c_int, c_lp]
    L.orc_max_threads.restype = C.c_int
    return L


def lib():
    global _lib
    if _lib is None:
        _lib = _configure(C.CDLL(build()))
    return _lib


class variant:
    """Context manager for the mutation checks of the pins (tests/test_oracle_mutants.py): compile a COPY of the oracle
    source with one textual substitution into ``workdir`` and route every call of this module to it while the block runs.
    The oracle itself is never edited; a substitution that does not apply exactly once is an error."""

    def __init__(self, old: str, new: str, workdir: str, tag: str):
        with open(_SRC) as fh:
            src = fh.read()
        if src.count(old) != 1:
            raise ValueError(f"mutation {tag!r}: pattern occurs {src.count(old)} times in the oracle source, expected 1")
        c_path = os.path.join(workdir, f"m3dk_oracle_{tag}.c")
        self.so = os.path.join(workdir, f"libm3dk_oracle_{tag}.so")
        with open(c_path, "w") as fh:
            fh.write(src.replace(old, new))
        subprocess.run(["gcc", "-O2", "-ffp-contract=off", "-fopenmp", "-fPIC", "-shared", "-o", self.so, c_path, "-lm"],
                       check=True)

    def __enter__(self):
        global _lib
        lib()
        self._saved = _lib
        _lib = _configure(C.CDLL(self.so))
        return self

    def __exit__(self, *exc):
        global _lib
        _lib = self._saved
        return False


def _d(a):
    a = np.ascontiguousarray(a, dtype=np.float64)
    return a, a.ctypes.data_as(c_dp)


def _i(a):
    a = np.ascontiguousarray(a, dtype=np.int32)
    return a, a.ctypes.data_as(c_ip)


def species(charge, mass, f0kind=0, T=1.0, v_c=0.3, Lambda0=0.75, dLambda=0.2, B_axis=1.0, mode=0) -> Species:
    """mode 0: linear delta-f; 1: non-linear trajectories with (1 - w) kept (reading G21); 2: linear delta-f with the
    4-point gyro-average of the perturbed fields (reading G23)."""
    s = Species()
    s.charge, s.mass, s.f0kind, s.mode = float(charge), float(mass), int(f0kind), int(mode)
    for k, v in enumerate((T, v_c, Lambda0, dLambda, B_axis)):
        s.f0par[k] = float(v)
    return s


def species_of(workload, mode=0) -> Species:
    f = workload.f0
    return species(workload.charge, workload.mass, f.kind, f.T, f.v_c, f.Lambda0, f.dLambda, f.B_axis, mode=mode)


def analytic_of(eq, kappa=0.0, pA=0.0, prc=0.5, pwd=0.1, pomega=0.0, pn=0, pm=0) -> Analytic:
    a = Analytic()
    a.R0, a.a, a.B0, a.qkind = eq.R0, eq.a, eq.B0, eq.qkind
    for k in range(3):
        a.qc[k] = eq.qc[k]
    a.kappa, a.pA, a.prc, a.pwd, a.pomega, a.pn, a.pm = kappa, pA, prc, pwd, pomega, pn, pm
    return a


class Mesh:
    """Finite-element tables in the layouts include/m3dk.h documents; arrays are kept alive here."""

    def __init__(self, node_RZ, tri, eq_coef, pert_coef=None, n_tor=None, omega=None):
        self.node_RZ, p_nodes = _d(node_RZ)
        self.tri, p_tri = _i(tri)
        self.eq_coef, p_eq = _d(eq_coef)
        self.n_elems = self.tri.shape[0]
        n_modes = 0 if n_tor is None else len(n_tor)
        self.n_modes = n_modes
        self.pert_coef, p_pc = _d(pert_coef if n_modes else np.zeros(1))
        self.n_tor, p_nt = _i(n_tor if n_modes else np.zeros(1, dtype=np.int32))
        self.omega, p_om = _d(omega if n_modes else np.zeros(1))
        assert self.eq_coef.shape == (self.n_elems, 4, 21)
        if n_modes:
            assert self.pert_coef.shape == (n_modes, self.n_elems, 7, 2, 21)
        self.h = lib().orc_mesh_create(self.node_RZ.shape[0], p_nodes, self.n_elems, p_tri, p_eq, n_modes, p_nt, p_om, p_pc)

    @classmethod
    def of(cls, w):
        return cls(w.node_RZ, w.tri, w.eq_coef, w.pert_coef, w.n_tor, w.omega)

    def __del__(self):
        if getattr(self, "h", None) and _lib is not None:
            _lib.orc_mesh_free(self.h)
            self.h = None

    def locate(self, R, Z, brute=False):
        R, pR = _d(R)
        Z, pZ = _d(Z)
        out = np.empty(R.shape[0], dtype=np.int32)
        lib().orc_locate(self.h, R.shape[0], pR, pZ, out.ctypes.data_as(c_ip), int(brute))
        return out

    def eval(self, R, phi, Z, t=0.0):
        R, pR = _d(R)
        phi, pP = _d(phi)
        Z, pZ = _d(Z)
        n = R.shape[0]
        elem = np.empty(n, dtype=np.int32)
        out = np.full((n, 18), np.nan)
        lib().orc_eval_fe(self.h, n, pR, pP, pZ, float(t), elem.ctypes.data_as(c_ip), out.ctypes.data_as(c_dp))
        return elem, out


FIELD_COLS = ("psi_R", "psi_Z", "Bm", "Bm_R", "Bm_Z", "F", "kappa", "E1_R", "E1_phi", "E1_Z", "B1_R", "B1_phi",
              "B1_Z", "gB1p_R", "gB1p_phi", "gB1p_Z", "dtB1p", "B1p")


def eval_analytic(an: Analytic, R, phi, Z, t=0.0):
    R, pR = _d(R)
    phi, pP = _d(phi)
    Z, pZ = _d(Z)
    n = R.shape[0]
    out = np.empty((n, 18))
    psi = np.empty(n)
    lib().orc_eval_analytic(C.byref(an), n, pR, pP, pZ, float(t), out.ctypes.data_as(c_dp), psi.ctypes.data_as(c_dp))
    return out, psi


def _state(m):
    keys = ("x", "y", "z", "vx", "vy", "vz", "mu", "w")
    arrs = [np.array(m[k], dtype=np.float64, copy=True, order="C") for k in keys]
    return dict(zip(keys, arrs)), [a.ctypes.data_as(c_dp) for a in arrs]


def push_fe(mesh: Mesh, sp: Species, markers: dict, nsteps: int, dt: float, t0: float = 0.0, step0: int = 0,
            brute: bool = False, nthreads: int = 0, elem: Optional[np.ndarray] = None):
    """Returns (new marker dict, elem, n_lost).  Input arrays are not modified."""
    st, ptrs = _state(markers)
    n = st["x"].shape[0]
    e = np.full(n, -2, dtype=np.int32) if elem is None else np.array(elem, dtype=np.int32, copy=True)
    lost = lib().orc_push_fe(mesh.h, C.byref(sp), n, *ptrs, e.ctypes.data_as(c_ip), int(nsteps), float(dt), float(t0),
                             int(step0), int(brute), int(nthreads))
    return st, e, int(lost)


def push_analytic(an: Analytic, sp: Species, markers: dict, nsteps: int, dt: float, t0: float = 0.0, step0: int = 0,
                  nthreads: int = 0):
    st, ptrs = _state(markers)
    n = st["x"].shape[0]
    lib().orc_push_analytic(C.byref(an), C.byref(sp), n, *ptrs, int(nsteps), float(dt), float(t0), int(step0), int(nthreads))
    return st


def gc_push(sp: Species, x, y, z, vpar, mu, nsteps: int, dt: float, *, mesh=None, an=None, nthreads: int = 0, t0: float = 0.0):
    """RK4 on the guiding-centre equations (Eqs. 1-4; equilibrium fields, reading G24; sp.mode == 1: total fields, reading
    G26, from time t0).  Returns (x, y, z, vpar, elem, lost)."""
    arrs = [np.array(a, dtype=np.float64, copy=True, order="C") for a in (x, y, z, vpar)]
    mu = np.ascontiguousarray(mu, dtype=np.float64)
    n = arrs[0].shape[0]
    e = np.zeros(n, dtype=np.int32)
    lost = lib().orc_gc_push(mesh.h if mesh is not None else None, C.byref(an) if an is not None else None, C.byref(sp), n,
                             *[a.ctypes.data_as(c_dp) for a in arrs], mu.ctypes.data_as(c_dp), e.ctypes.data_as(c_ip),
                             int(nsteps), float(dt), float(t0), int(nthreads))
    return arrs[0], arrs[1], arrs[2], arrs[3], e, int(lost)


def gc_bootstrap(sp: Species, x, y, z, vpar, mu, dt: float, *, mesh=None, an=None):
    """one RK4 guiding-centre step x_0 -> x_1 and v_{1/2} = (x_1 - x_0)/dt.
    Returns (x1, y1, z1, vx, vy, vz, ok); rows with ok False keep x_0 and have v = 0."""
    pos = [np.array(a, dtype=np.float64, copy=True, order="C") for a in (x, y, z)]
    vpar, mu = (np.ascontiguousarray(a, dtype=np.float64) for a in (vpar, mu))
    n = pos[0].shape[0]
    v = [np.zeros(n) for _ in range(3)]
    ok = np.zeros(n, dtype=np.int32)
    lib().orc_gc_bootstrap(mesh.h if mesh is not None else None, C.byref(an) if an is not None else None, C.byref(sp), n,
                           *[a.ctypes.data_as(c_dp) for a in pos], vpar.ctypes.data_as(c_dp), mu.ctypes.data_as(c_dp),
                           float(dt), *[a.ctypes.data_as(c_dp) for a in v], ok.ctypes.data_as(c_ip))
    return pos[0], pos[1], pos[2], v[0], v[1], v[2], ok.astype(bool)


def gc_rhs(sp: Species, R, Z, vpar, mu, *, mesh=None, an=None, phi=None, t: float = 0.0):
    """Right-hand sides of Eqs. (1)-(2): rows (dR/dt, R dphi/dt, dZ/dt, dv_par/dt); phi and t matter with sp.mode == 1."""
    R, Z, vpar, mu = (np.ascontiguousarray(a, dtype=np.float64) for a in (R, Z, vpar, mu))
    phi = np.zeros_like(R) if phi is None else np.ascontiguousarray(phi, dtype=np.float64)
    out = np.zeros((R.shape[0], 4))
    lib().orc_gc_rhs(mesh.h if mesh is not None else None, C.byref(an) if an is not None else None, C.byref(sp), R.shape[0],
                     R.ctypes.data_as(c_dp), phi.ctypes.data_as(c_dp), Z.ctypes.data_as(c_dp), vpar.ctypes.data_as(c_dp),
                     mu.ctypes.data_as(c_dp), float(t), out.ctypes.data_as(c_dp))
    return out


def gc_fields(R, Z, *, mesh=None, an=None):
    """The field values the guiding-centre right-hand side works from: (elem, out[n][11]) with columns GC_FIELD_COLS."""
    R, Z = (np.ascontiguousarray(a, dtype=np.float64) for a in (R, Z))
    n = R.shape[0]
    elem = np.empty(n, dtype=np.int32)
    out = np.full((n, 11), np.nan)
    lib().orc_gc_fields(mesh.h if mesh is not None else None, C.byref(an) if an is not None else None, n,
                        R.ctypes.data_as(c_dp), Z.ctypes.data_as(c_dp), elem.ctypes.data_as(c_ip), out.ctypes.data_as(c_dp))
    return elem, out


GC_FIELD_COLS = ("psi_R", "psi_Z", "psi_RR", "psi_RZ", "psi_ZZ", "F", "F_R", "F_Z", "Bm", "Bm_R", "Bm_Z")


def gyro_ring(sp: Species, X, mu: float, *, mesh=None, an=None):
    """The four gyro-ring points X + rho_L,j of reading G23 (Cartesian, shape (4, 3)); None when X is outside the mesh."""
    X = np.ascontiguousarray(X, dtype=np.float64)
    pts = np.empty((4, 3))
    ok = lib().orc_gyro_ring(mesh.h if mesh is not None else None, C.byref(an) if an is not None else None, C.byref(sp),
                             X.ctypes.data_as(c_dp), float(mu), pts.ctypes.data_as(c_dp))
    return pts if ok else None


def flr_fields(sp: Species, X, mu: float, t: float = 0.0, *, mesh=None, an=None):
    """Gyro-averaged perturbed fields of Eq. (14) at X in the marker's cylindrical frame: <E1>, <B1>, <grad B1par>, <dB1par/dt>."""
    X = np.ascontiguousarray(X, dtype=np.float64)
    out = np.empty(10)
    ok = lib().orc_flr_fields(mesh.h if mesh is not None else None, C.byref(an) if an is not None else None, C.byref(sp),
                              X.ctypes.data_as(c_dp), float(mu), float(t), out.ctypes.data_as(c_dp))
    return out if ok else None


def deposit(mesh: "Mesh", sp: Species, markers: dict, flags: int = 0, t: float = 0.0):
    """Right-hand sides of Eqs. (17)-(18) with a delta-function shape: rhs[n_elems][2][1 + 2 n_modes][21], n_lost.
    flags bit 0: add the mu B1par term of Eq. (16) to the perpendicular moment (B1par at time t)."""
    st, ptrs = _state(markers)
    n = st["x"].shape[0]
    H = 1 + 2 * mesh.n_modes
    rhs = np.zeros((mesh.n_elems, 2, H, 21), dtype=np.float64)
    lost = lib().orc_deposit(mesh.h, C.byref(sp), n, *ptrs, rhs.ctypes.data_as(c_dp), int(flags), float(t))
    return rhs, int(lost)


def trace(sp: Species, state8, nsteps: int, dt: float, *, mesh: Optional[Mesh] = None, an: Optional[Analytic] = None,
          t0: float = 0.0, stride: int = 1):
    """Trajectory of one marker: rows (x_l[3], v_l[3], w_{l+1/2}, t_l) every ``stride`` steps."""
    s = np.array(state8, dtype=np.float64, copy=True)
    nout = (nsteps + stride - 1) // stride
    out = np.empty((nout, 8))
    k = lib().orc_trace(mesh.h if mesh is not None else None, C.byref(an) if an is not None else None, C.byref(sp),
                        s.ctypes.data_as(c_dp), int(nsteps), float(dt), float(t0), int(stride), out.ctypes.data_as(c_dp))
    return out[:k], s


def push_uniform(x, v, B, E, charge, mass, nsteps, dt):
    xs = [np.array(x[..., k], dtype=np.float64, copy=True, order="C").ravel() for k in range(3)]
    vs = [np.array(v[..., k], dtype=np.float64, copy=True, order="C").ravel() for k in range(3)]
    B, pB = _d(B)
    E, pE = _d(E)
    lib().orc_push_uniform(xs[0].shape[0], *[a.ctypes.data_as(c_dp) for a in xs + vs], pB, pE, float(charge), float(mass),
                           int(nsteps), float(dt))
    return np.stack(xs, -1), np.stack(vs, -1)


def eq6(vm, E, B, h):
    vm, p1 = _d(vm)
    E, p2 = _d(E)
    B, p3 = _d(B)
    out = np.empty(3)
    lib().orc_eq6(p1, p2, p3, float(h), out.ctypes.data_as(c_dp))
    return out


def weight_rhs(fields18, sp: Species, R, vl_cyl, mu):
    f, p1 = _d(fields18)
    v, p2 = _d(vl_cyl)
    return float(lib().orc_weight_rhs(p1, C.byref(sp), float(R), p2, float(mu)))


def sort_perm(elem, n_elems):
    e, pe = _i(elem)
    perm = np.empty(e.shape[0], dtype=np.int64)
    lib().orc_sort_perm(e.shape[0], pe, int(n_elems), perm.ctypes.data_as(c_lp))
    return perm


def max_threads() -> int:
    return int(lib().orc_max_threads())
