"""Hand-made finite-element tables whose fields are known in closed form (inputs of the pins M1-M3, N1, Q1).

Every field is a low-order polynomial of (R, Z), so its per-element quintic in the local frame of reading G10
(xi = (R - R_c) s_e, eta = (Z - Z_c) s_e) is exact: no fit, no fit error.  Only table construction lives here -- no
arithmetic of the method.
"""
import numpy as np

from synth.mesh import element_frames, rect_tri_mesh

# table order of the monomials xi^i eta^j (j outer, i inner): (0,0) -> 0, (1,0) -> 1, (2,0) -> 2, (0,1) -> 6
K_1, K_XI, K_XI2, K_ETA = 0, 1, 2, 6


def poly_coef(cen, s, c0=0.0, cR=0.0, cZ=0.0, cRR=0.0):
    """Coefficients [n_elems][21] of f(R, Z) = c0 + cR R + cZ Z + cRR R^2 in every element's local frame.
    c0..cRR may be complex (perturbed amplitudes)."""
    ne = cen.shape[0]
    out = np.zeros((ne, 21), dtype=np.result_type(c0, cR, cZ, cRR, np.float64))
    Rc, Zc = cen[:, 0], cen[:, 1]
    out[:, K_1] = c0 + cR * Rc + cZ * Zc + cRR * Rc * Rc
    out[:, K_XI] = (cR + 2.0 * cRR * Rc) / s
    out[:, K_ETA] = cZ / s
    out[:, K_XI2] = cRR / (s * s)
    return out


class HandMade:
    """A rectangular triangulated box with polynomial equilibrium tables and one toroidal mode with polynomial amplitudes.

    eq: dict name -> (c0, cR, cZ, cRR) for 'psi', 'Bm', 'F', 'kappa' (missing = 0).
    pert: dict name -> (c0, cR, cZ) complex for 'E_R', 'E_phi', 'E_Z', 'B_R', 'B_phi', 'B_Z', 'B_par' (missing = 0).
    """
    PERT = ("E_R", "E_phi", "E_Z", "B_R", "B_phi", "B_Z", "B_par")

    def __init__(self, eq, pert=None, n_tor=0, omega=0.0, nx=6, box=(1.9, 4.1, -1.1, 1.1)):
        self.node, self.tri = rect_tri_mesh(nx, box)
        cen, s = element_frames(self.node, self.tri)
        ne = self.tri.shape[0]
        self.eq_coef = np.zeros((ne, 4, 21))
        for k, name in enumerate(("psi", "Bm", "F", "kappa")):
            self.eq_coef[:, k, :] = poly_coef(cen, s, *eq.get(name, (0.0,)))
        self.eq, self.pert = dict(eq), dict(pert or {})
        self.n_tor, self.omega = int(n_tor), float(omega)
        if pert is None:
            self.pert_coef, self.n_tor_a, self.omega_a = None, None, None
        else:
            self.pert_coef = np.zeros((1, ne, 7, 2, 21))
            for k, name in enumerate(self.PERT):
                c = poly_coef(cen, s, *[complex(v) for v in pert.get(name, (0.0,))])
                self.pert_coef[0, :, k, 0, :] = c.real
                self.pert_coef[0, :, k, 1, :] = c.imag
            self.n_tor_a = np.array([n_tor], dtype=np.int32)
            self.omega_a = np.array([omega], dtype=np.float64)

    def oracle_mesh(self, orc):
        return orc.Mesh(self.node, self.tri, self.eq_coef, self.pert_coef, self.n_tor_a, self.omega_a)

    # closed forms of the same fields (numpy), for the expected values of the pins
    @staticmethod
    def _lin(c, R, Z):
        c = tuple(c) + (0.0,) * (4 - len(c))
        return c[0] + c[1] * R + c[2] * Z + c[3] * R * R

    def eq_at(self, name, R, Z):
        return self._lin(self.eq.get(name, (0.0,)), R, Z)

    def eq_grad(self, name, R, Z):
        c = tuple(self.eq.get(name, (0.0,))) + (0.0,) * 4
        return c[1] + 2.0 * c[3] * R, c[2] + 0.0 * Z

    def amp_at(self, name, R, Z):
        return self._lin([complex(v) for v in self.pert.get(name, (0.0,))], R, Z)

    def amp_grad(self, name, R, Z):
        c = [complex(v) for v in self.pert.get(name, (0.0,))] + [0.0] * 3
        return c[1], c[2]
