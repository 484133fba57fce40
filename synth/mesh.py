"""Triangulated poloidal meshes and per-element least-squares quintic tables (inputs only).

Readings G10 (monomial basis, element-local frame) and G14 (36 interior lattice points):

* monomials xi^i eta^j, i + j <= 5, ordered j outer 0..5, i inner 0..5-j  (21 terms);
* xi = (R - R_c) * s_e, eta = (Z - Z_c) * s_e, (R_c, Z_c) the centroid, s_e = 1/(longest edge);
* fit points: the interior nodes (i, j, k)/10, i, j, k >= 1, i + j + k = 10 of the order-10
  barycentric lattice (36 points); least squares by QR in fp64.

The table layouts are the ones ``include/m3dk.h`` documents for m3dk_fields_create:
``eq_coef[n_elems][4][21]`` (psi0, |B|0, F0, kappa) and
``pert_coef[n_modes][n_elems][7][2][21]`` (re, im of the PERT_FIELDS amplitudes).
"""
from __future__ import annotations

from typing import Callable, Sequence, Tuple

import numpy as np

NCOEF = 21
DEGREE = 5


def monomial_exponents() -> np.ndarray:
    """(21, 2) int array of (i, j) in table order."""
    return np.array([(i, j) for j in range(DEGREE + 1) for i in range(DEGREE + 1 - j)], dtype=np.int64)


def rect_tri_mesh(nx: int, box: Tuple[float, float, float, float] = (1.9, 4.1, -1.1, 1.1), nz: int | None = None):
    """nx x nz cells on [Rmin,Rmax] x [Zmin,Zmax], each split by the lower-left -> upper-right diagonal.

    Nodes row-major (index iz*(nx+1)+ix); element 2*(iz*nx+ix)+t, t=0: (LL, LR, UR), t=1: (LL, UR, UL);
    both counter-clockwise.  Returns node_RZ float64 [n_nodes, 2], tri int32 [n_elems, 3].
    """
    nz = nx if nz is None else nz
    Rmin, Rmax, Zmin, Zmax = box
    Rn = np.linspace(Rmin, Rmax, nx + 1)
    Zn = np.linspace(Zmin, Zmax, nz + 1)
    RR, ZZ = np.meshgrid(Rn, Zn, indexing="xy")  # [nz+1, nx+1]
    node_RZ = np.stack([RR.ravel(), ZZ.ravel()], axis=1).astype(np.float64)
    ix, iz = np.meshgrid(np.arange(nx), np.arange(nz), indexing="xy")
    ll = (iz * (nx + 1) + ix).ravel()
    lr = ll + 1
    ul = ll + (nx + 1)
    ur = ul + 1
    tri = np.empty((2 * nx * nz, 3), dtype=np.int32)
    tri[0::2] = np.stack([ll, lr, ur], axis=1)
    tri[1::2] = np.stack([ll, ur, ul], axis=1)
    return np.ascontiguousarray(node_RZ), np.ascontiguousarray(tri)


def perturbed_tri_mesh(nx: int, box=(1.9, 4.1, -1.1, 1.1), jitter: float = 0.25, seed: int = 7, flip: bool = True):
    """An *unstructured-looking* mesh for tests: interior nodes jittered, random diagonals,
    element order shuffled.  Still a valid CCW triangulation of the box."""
    node_RZ, _ = rect_tri_mesh(nx, box)
    rng = np.random.Generator(np.random.PCG64(seed))
    hx = (box[1] - box[0]) / nx
    hz = (box[3] - box[2]) / nx
    n1 = nx + 1
    interior = np.ones((n1, n1), dtype=bool)
    interior[0, :] = interior[-1, :] = interior[:, 0] = interior[:, -1] = False
    d = (rng.random((n1 * n1, 2)) - 0.5) * 2.0 * jitter
    node_RZ = node_RZ + d * np.array([hx, hz]) * interior.ravel()[:, None]
    tris = []
    flips = rng.random(nx * nx) < 0.5 if flip else np.zeros(nx * nx, dtype=bool)
    for iz in range(nx):
        for ix in range(nx):
            ll = iz * n1 + ix
            lr, ul, ur = ll + 1, ll + n1, ll + n1 + 1
            if flips[iz * nx + ix]:
                tris += [(ll, lr, ul), (lr, ur, ul)]
            else:
                tris += [(ll, lr, ur), (ll, ur, ul)]
    tri = np.array(tris, dtype=np.int32)
    tri = tri[rng.permutation(len(tri))]
    return np.ascontiguousarray(node_RZ), np.ascontiguousarray(tri)


def lattice_points() -> np.ndarray:
    """(36, 3) barycentric coordinates of the interior order-10 lattice nodes (G14)."""
    pts = [(i / 10.0, j / 10.0, (10 - i - j) / 10.0) for i in range(1, 9) for j in range(1, 10 - i)]
    return np.array(pts, dtype=np.float64)


def element_frames(node_RZ: np.ndarray, tri: np.ndarray):
    """Centroid (R_c, Z_c) and scale s_e = 1/(longest edge) of every element (G10)."""
    P = node_RZ[tri]  # [ne, 3, 2]
    c = P.mean(axis=1)
    e = np.stack([P[:, 1] - P[:, 0], P[:, 2] - P[:, 1], P[:, 0] - P[:, 2]], axis=1)
    L = np.sqrt((e ** 2).sum(-1)).max(axis=1)
    return c, 1.0 / L


def fit_tables(node_RZ: np.ndarray, tri: np.ndarray, fn: Callable[[np.ndarray, np.ndarray], np.ndarray],
               chunk: int = 16384, return_residual: bool = False):
    """Least-squares quintic of ``fn`` on every element.

    ``fn(R, Z)`` takes arrays [ne, 36] and returns [ne, 36, nf] (real or complex).  Returns coefficients
    [ne, nf, 21] in table order (complex if fn is complex), and optionally the max |residual| per field.
    """
    ne = tri.shape[0]
    lam = lattice_points()  # [36, 3]
    ex = monomial_exponents()
    cen, s = element_frames(node_RZ, tri)
    out = None
    resid = None
    for a in range(0, ne, chunk):
        b = min(ne, a + chunk)
        P = node_RZ[tri[a:b]]  # [n, 3, 2]
        pts = np.einsum("pk,nkd->npd", lam, P)  # [n, 36, 2]
        xi = (pts[..., 0] - cen[a:b, None, 0]) * s[a:b, None]
        eta = (pts[..., 1] - cen[a:b, None, 1]) * s[a:b, None]
        xp = [np.ones_like(xi)]
        ep = [np.ones_like(eta)]
        for _ in range(DEGREE):
            xp.append(xp[-1] * xi)
            ep.append(ep[-1] * eta)
        A = np.stack([xp[i] * ep[j] for i, j in ex], axis=-1)  # [n, 36, 21]
        f = np.asarray(fn(pts[..., 0], pts[..., 1]))  # [n, 36, nf]
        Q, Rm = np.linalg.qr(A)  # Q [n,36,21], R [n,21,21]
        rhs = np.matmul(np.swapaxes(Q, 1, 2), f)
        coef = np.linalg.solve(Rm.astype(rhs.dtype), rhs)  # [n, 21, nf]
        if out is None:
            out = np.empty((ne, f.shape[-1], NCOEF), dtype=coef.dtype)
            resid = np.zeros(f.shape[-1])
        out[a:b] = np.swapaxes(coef, 1, 2)
        if return_residual:
            r = np.abs(np.matmul(A, coef) - f).max(axis=(0, 1))
            resid = np.maximum(resid, r)
    if return_residual:
        return out, resid
    return out


def eq_tables(eq, node_RZ, tri, kappa_fn=None):
    """eq_coef[n_elems][4][21]: psi0, |B|0, F0 = R B_phi, kappa = d ln f0 / d psi."""
    def fn(R, Z):
        k = np.zeros_like(R) if kappa_fn is None else kappa_fn(R, Z)
        return np.stack([eq.psi(R, Z), eq.Bmag(R, Z), np.full_like(R, eq.F0), k], axis=-1)
    return np.ascontiguousarray(fit_tables(node_RZ, tri, fn))


def pert_tables(perts: Sequence, node_RZ, tri):
    """pert_coef[n_modes][n_elems][7][2][21] (re, im) plus n_tor[n_modes], omega[n_modes]."""
    ne = tri.shape[0]
    out = np.zeros((len(perts), ne, 7, 2, NCOEF), dtype=np.float64)
    for k, p in enumerate(perts):
        c = fit_tables(node_RZ, tri, p.amplitudes)  # [ne, 7, 21] complex
        out[k, :, :, 0, :] = c.real
        out[k, :, :, 1, :] = c.imag
    n_tor = np.array([p.n for p in perts], dtype=np.int32)
    omega = np.array([p.omega for p in perts], dtype=np.float64)
    return np.ascontiguousarray(out), n_tor, omega
