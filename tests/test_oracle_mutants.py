"""Mutation checks of the pins M1-M3, N1, Q1, Q2 (tests/test_oracle_magnetic.py), G5, G6, G7 (tests/test_oracle_gc.py) D7
(tests/test_oracle_deposit.py) and F6 (tests/test_oracle_flr.py).

Each case compiles a COPY of oracle/m3dk_oracle.c with one plausible mistake (a flipped sign, a dropped factor, a wrong
index) into a temporary directory, routes the oracle binding to that copy and asserts that the named pin FAILS -- the
evidence that the pin would catch that mistake.  The oracle itself is never modified (oracle.variant).  CPU only.
"""
import pytest

from test_oracle_gc import check_g5_phase_space_volume, check_g6_bootstrap, check_g7_perturbed_guiding_centre_rhs
from test_oracle_deposit import check_d7_jacobian_substitution
from test_oracle_flr import check_f6_nonlinear_mode_with_gyro_average
from test_oracle_magnetic import CHECKS as _MAGNETIC

CHECKS = dict(_MAGNETIC, g5=check_g5_phase_space_volume, g6=check_g6_bootstrap, g7=check_g7_perturbed_guiding_centre_rhs,
              d7=check_d7_jacobian_substitution, f6=check_f6_nonlinear_mode_with_gyro_average)

#        pin   tag                      text in the oracle source                         mutated text
MUTANTS = [
    ("m1", "eq12_sign", "+ vpar * B1[k] / B0n;", "- vpar * B1[k] / B0n;"),
    ("m1", "eq12_factor", "+ vpar * B1[k] / B0n;", "+ vpar * B1[k] / (B0n * B0n);"),
    ("m1", "eq12_dropped", "+ vpar * B1[k] / B0n;", ";"),
    ("m2", "eq13_sign", "- mu * (b0[0] * f->gB1p[0] + b0[1] * f->gB1p[1] + b0[2] * f->gB1p[2]);",
     "+ mu * (b0[0] * f->gB1p[0] + b0[1] * f->gB1p[1] + b0[2] * f->gB1p[2]);"),
    ("m2", "eq13_component", "- mu * (b0[0] * f->gB1p[0] + b0[1] * f->gB1p[1] + b0[2] * f->gB1p[2]);",
     "- mu * (b0[0] * f->gB1p[0] + b0[2] * f->gB1p[1] + b0[1] * f->gB1p[2]);"),
    ("m2", "eq10_factor", "+ Fpar * f->F / B0n;", "+ Fpar * f->F / (B0n * R);"),
    ("m2", "dphi_sign", "f->gB1p[1] += -n * qd / R;", "f->gB1p[1] += n * qd / R;"),
    ("m3", "eq11_sign", "+ mu * f->dtB1p;", "- mu * f->dtB1p;"),
    ("m3", "eq11_dropped", "+ mu * f->dtB1p;", ";"),
    ("m3", "dt_sign", "f->dtB1p += om * qd;", "f->dtB1p += -om * qd;"),
    ("n1", "B1R_sign", "BR += f.B1[0];", "BR -= f.B1[0];"),
    ("n1", "B1phi_dropped", "BP += f.B1[1];", ""),
    ("n1", "B1Z_sign", "BZ += f.B1[2];", "BZ -= f.B1[2];"),
    ("n1", "gradB1par_R_sign", "(f.Bm_R + f.gB1p[0])", "(f.Bm_R - f.gB1p[0])"),
    ("n1", "gradB1par_phi_sign", "EP = f.E1[1] - (mu / q) * f.gB1p[1];", "EP = f.E1[1] + (mu / q) * f.gB1p[1];"),
    ("n1", "gradB1par_Z_dropped", "(f.Bm_Z + f.gB1p[2])", "(f.Bm_Z)"),
    ("q1", "dxe_factor", "(double)(i * j) *", "(double)(i + j) *"),
    ("q1", "dxx_index", "(xp[i - 2] * ep[j])", "(xp[i - 1] * ep[j])"),
    ("q1", "psi_RZ_scale", "g->psi_RZ = b * s * s;", "g->psi_RZ = b * s;"),
    ("q2", "curlb_R_sign", "double curlb[3] = {-bP_Z,", "double curlb[3] = {bP_Z,"),
    ("q2", "curlb_Z_term", "b[1] / R + bP_R};", "bP_R};"),
    ("g5", "curlb_phi_sign", "double curlb[3] = {-bP_Z, bR_Z - bZ_R,", "double curlb[3] = {-bP_Z, bZ_R - bR_Z,"),
    ("g5", "Bstar_par", "Bspar += Bs[k] * b[k]; }", "Bspar += B[k] * b[k]; }"),
    ("d7", "jacobian_sign", "dd += f.B1p / bstar(&g, sp, R, vpar, Bs, bb);", "dd -= f.B1p / bstar(&g, sp, R, vpar, Bs, bb);"),
    ("d7", "jacobian_without_curl_b", "dd += f.B1p / bstar(&g, sp, R, vpar, Bs, bb);", "dd += f.B1p / g.Bm;"),
    ("g7", "ExB_sign", "dX[k] = (vpar * Bs[k] - bxE[k]) / Bspar;", "dX[k] = (vpar * Bs[k] + bxE[k]) / Bspar;"),
    ("g7", "B1_dropped_from_Bstar", "Bs[k] += f.B1[k]; Bspar += Bs[k] * b[k];", "Bspar += Bs[k] * b[k];"),
    ("g7", "mirror_of_B1par_dropped", "gB[k] += f.gB1p[k]; E[k] = f.E1[k]; }", "E[k] = f.E1[k]; }"),
    ("g7", "parallel_E_sign", "*dvpar = (q / m) * (Bs[0] * Ee[0] + Bs[1] * Ee[1] + Bs[2] * Ee[2]) / Bspar;",
     "*dvpar = -(q / m) * (Bs[0] * Ee[0] + Bs[1] * Ee[1] + Bs[2] * Ee[2]) / Bspar;"),
    ("f6", "mode3_without_average", "flr = sp->mode == 2 || sp->mode == 3;", "flr = sp->mode == 2;"),
    ("f6", "mode3_linear_trajectory", "nonlinear = sp->mode == 1 || sp->mode == 3,", "nonlinear = sp->mode == 1,"),
    ("g6", "bootstrap_sign", "vx[i] = (s[0] - x[i]) / dt;", "vx[i] = (x[i] - s[0]) / dt;"),
    ("g6", "bootstrap_keeps_x0", "x[i] = s[0]; y[i] = s[1]; z[i] = s[2];\n    }\n}", "\n    }\n}"),
    ("q1", "psi_ZZ_dropped", "g->psi_ZZ = d * s * s;", "g->psi_ZZ = 0.0 * d;"),
]


@pytest.mark.parametrize("pin,tag,old,new", MUTANTS, ids=[f"{m[0]}-{m[1]}" for m in MUTANTS])
def test_pin_fails_on_mutated_oracle(orc, tmp_path, pin, tag, old, new):
    CHECKS[pin](orc)                                   # green on the oracle as it stands
    with orc.variant(old, new, str(tmp_path), tag):
        with pytest.raises(AssertionError):
            CHECKS[pin](orc)
    CHECKS[pin](orc)                                   # and the binding is back on the real oracle
