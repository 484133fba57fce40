/*
 * m3dk_oracle.c -- CPU fp64 ORACLE for the M3D-C1-K energetic-particle push.
 *
 * TEST INFRASTRUCTURE ONLY.  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * --impl reference legs may build, load or call this file.  It shares no code with the CUDA path
 * (paper_2107_13663_b200/csrc) and neither includes the other.  Compile: gcc -O2 -ffp-contract=off -fopenmp.
 *
 * What it is: the method of PAPER.md sections 2-3 written out step by step, one marker at a time,
 * scalar loops, in the paper's order and notation (the method is a time integrator, so the oracle is
 * the algorithm itself):
 *
 *   per marker, per step l, state (x_l, v_{l-1/2}, mu, w_{l-1/2}), time t_l = t0 + l*dt
 *    1. (R, phi, Z) from Cartesian x                          [tokamak geometry; reading G3]
 *    2. element containing (R, Z)                              [whole mesh visible; reading G11]
 *    3. fields = per-element polynomials, first derivatives    [PAPER.md:86; readings G4, G10]
 *       |B| is its own scalar field, grad|B| from its first derivatives [PAPER.md:86]
 *    4. perturbed fields Re[C(R,Z) exp(i(n phi - omega t))]    [PAPER.md:130; reading G8]
 *    5. E-dagger = E - (mu/q) grad|B|  (linear mode: E = 0, B = B0)    [PAPER.md:78, :108; reading G2]
 *    6. Eq. (6) solved for v_{l+1/2} as a 3x3 linear system    [PAPER.md:75-78]
 *    7. v_l = (v_{l-1/2}+v_{l+1/2})/2, weight RHS Eqs. (8)-(13) with (1-w) -> 1   [PAPER.md:106-130, :140; G5-G7, G9]
 *    8. Eq. (5): x_{l+1} = x_l + dt v_{l+1/2}                  [PAPER.md:73]
 *   mu is never modified [PAPER.md:114].
 *
 * Deliberately different routes from the CUDA path where the mathematics allows (so that agreement means
 * something): naive monomial sums instead of Horner, libm atan2/cos/sin instead of complex powers,
 * Gaussian elimination of the 3x3 system instead of the Boris t/s vectors, brute-force / full-list element
 * search instead of the prioritised bucket search.
 *
 * Mode 1 (non-linear trajectories; reading G21): step 5 uses the total fields,
 * B = B0 + B1 and E-dagger = E1 - (mu/q) grad(|B|0 + B1par), and step 7 keeps the factor (1 - w) of Eq. (8).
 *
 * Mode 2 (finite Larmor radius; Eq. 14; reading G23): step 7 uses the quarter sum of the
 * perturbed fields over the four gyro-ring points (gyro_ring, flr_average); pins F1-F4.
 *
 * orc_gc_push: RK4 on the guiding-centre equations (1)-(4), equilibrium fields (reading G24); pins G1-G5.
 * orc_gc_bootstrap: v_{1/2} = (x_1 - x_0)/dt from one such step; pin G6.
 *
 * orc_deposit: right-hand sides of Eqs. (17)-(18) with a delta-function shape (readings G10, G22).
 *
 * Pins (tests/test_oracle_*.py, run with -m "not gpu"): P1-P15 of SURVEY.md 8(c), P16-P19 for mode 1, M1-M3 for the
 * magnetic terms of Eqs. (11)-(13), N1 for the total fields of the mode-1 push, Q1-Q2 for poly_eval2 and the finite-element
 * branch of gc_fields, F1-F4 (FLR), G1-G5 (guiding centre), D1-D6 (deposition); mutation checks of M1-M3, N1, Q1, Q2, G5 in
 * tests/test_oracle_mutants.py (they compile mutated COPIES of this file); see DESIGN.md section 4.
 * Unpinned by the paper (fixed by DESIGN.md readings, parity unpinned): the kappa_E model (G7),
 * the construction of the synthetic perturbations (G19), rho* (G17).
 */
#include <math.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define NCOEF 21
#define DEG 5
#define N_EQ 4
#define N_PERT 7

/* ------------------------------------------------------------------------------------------------ */
/* field values at one point, cylindrical components (R, phi, Z)                                      */
typedef struct {
    double psi_R, psi_Z;   /* d psi0/dR, d psi0/dZ                    */
    double Bm, Bm_R, Bm_Z; /* |B|0 (its own scalar field) and gradient */
    double F;              /* R B_phi0                                 */
    double kappa;          /* d ln f0 / d psi                          */
    double E1[3], B1[3];   /* perturbed E, B                           */
    double gB1p[3];        /* grad B1par (phi component = (1/R) d/dphi) */
    double dtB1p;          /* d B1par / dt                             */
    double B1p;            /* B1par itself (diagnostic)                */
} orc_fields;

typedef struct {
    int n_nodes, n_elems, n_modes;
    const double *node_RZ; /* [n_nodes][2]                    */
    const int *tri;        /* [n_elems][3] CCW                */
    const double *eq_coef; /* [n_elems][4][21]                */
    const double *pert_coef; /* [n_modes][n_elems][7][2][21]  */
    const int *n_tor;
    const double *omega;
    /* background grid for the assisted search (own construction, bbox lists, ascending ids) */
    int gx, gz;
    double Rmin, Rmax, Zmin, Zmax, hx, hz;
    int *start; /* [gx*gz+1] */
    int *cand;
} orc_mesh;

/* analytic large-aspect-ratio circular tokamak (reading G18) + optional electrostatic harmonic */
typedef struct {
    double R0, a, B0;
    int qkind;          /* 0: q = qc0 + qc1 u ; 1: q = qc0 + qc1 (u-qc2)^2 ; u=(r/a)^2, frozen for u>1 */
    double qc[3];
    double kappa;       /* constant d ln f0 / d psi used by the analytic back-end */
    /* electrostatic perturbation Phi = A exp(-((r-rc)/wd)^2) cos(n phi - m theta - omega t); A = 0: none */
    double pA, prc, pwd, pomega;
    int pn, pm;
} orc_analytic;

typedef struct {
    double charge, mass;
    int f0kind;        /* 0 Maxwellian, 1 slowing-down, 2 beam pitch (reading G7) */
    double f0par[5];   /* T, v_c, Lambda0, dLambda, B_axis */
    int mode;          /* 0: linear delta-f; 1: non-linear trajectories, (1 - w) kept (reading G21);
                          2: linear delta-f with 4-point gyro-averaged perturbed fields (Eq. 14; reading G23);
                          3: non-linear trajectories in the gyro-averaged perturbed fields (modes 1 and 2 together) */
} orc_species;

/* ------------------------------------------------------------------------------------------------ */
/* 2. element search (reading G11): smallest element index whose three edge functions
 *    (x_b-x_a)(Z-z_a) - (z_b-z_a)(R-r_a), evaluated in exactly this order without FMA, are all >= 0.     */
static int tri_contains(const orc_mesh *m, int e, double R, double Z)
{
    const int *t = m->tri + 3 * e;
    for (int k = 0; k < 3; ++k) {
        const double *pa = m->node_RZ + 2 * t[k];
        const double *pb = m->node_RZ + 2 * t[(k + 1) % 3];
        double ra = pa[0], za = pa[1], rb = pb[0], zb = pb[1];
        double ef = (rb - ra) * (Z - za) - (zb - za) * (R - ra);
        if (!(ef >= 0.0)) return 0;
    }
    return 1;
}

static int locate_brute(const orc_mesh *m, double R, double Z)
{
    for (int e = 0; e < m->n_elems; ++e)
        if (tri_contains(m, e, R, Z)) return e;
    return -1;
}

static int locate_grid(const orc_mesh *m, double R, double Z)
{
    if (!(R >= m->Rmin && R <= m->Rmax && Z >= m->Zmin && Z <= m->Zmax)) return -1;
    int ix = (int)floor((R - m->Rmin) / m->hx);
    int iz = (int)floor((Z - m->Zmin) / m->hz);
    if (ix < 0) ix = 0;
    if (ix >= m->gx) ix = m->gx - 1;
    if (iz < 0) iz = 0;
    if (iz >= m->gz) iz = m->gz - 1;
    int b = iz * m->gx + ix;
    for (int k = m->start[b]; k < m->start[b + 1]; ++k) /* ascending ids: first hit = smallest index */
        if (tri_contains(m, m->cand[k], R, Z)) return m->cand[k];
    return -1;
}

static void build_grid(orc_mesh *m)
{
    double Rmin = 1e300, Rmax = -1e300, Zmin = 1e300, Zmax = -1e300;
    for (int i = 0; i < m->n_nodes; ++i) {
        double r = m->node_RZ[2 * i], z = m->node_RZ[2 * i + 1];
        if (r < Rmin) Rmin = r;
        if (r > Rmax) Rmax = r;
        if (z < Zmin) Zmin = z;
        if (z > Zmax) Zmax = z;
    }
    int g = (int)floor(sqrt(0.5 * (double)m->n_elems));
    if (g < 1) g = 1;
    m->gx = m->gz = g;
    m->Rmin = Rmin; m->Rmax = Rmax; m->Zmin = Zmin; m->Zmax = Zmax;
    m->hx = (Rmax - Rmin) / g;
    m->hz = (Zmax - Zmin) / g;
    const double infl = 1e-6; /* buckets, inflated: conservative against rounding of the bucket index */
    int nb = g * g;
    m->start = (int *)calloc((size_t)nb + 1, sizeof(int));
    for (int pass = 0; pass < 2; ++pass) {
        int *fill = NULL;
        if (pass == 1) {
            int acc = 0;
            for (int b = 0; b < nb; ++b) { int c = m->start[b]; m->start[b] = acc; acc += c; }
            m->start[nb] = acc;
            m->cand = (int *)malloc(sizeof(int) * (size_t)(acc > 0 ? acc : 1));
            fill = (int *)malloc(sizeof(int) * (size_t)nb);
            memcpy(fill, m->start, sizeof(int) * (size_t)nb);
        }
        for (int e = 0; e < m->n_elems; ++e) {
            const int *t = m->tri + 3 * e;
            double r0 = 1e300, r1 = -1e300, z0 = 1e300, z1 = -1e300;
            for (int k = 0; k < 3; ++k) {
                double r = m->node_RZ[2 * t[k]], z = m->node_RZ[2 * t[k] + 1];
                if (r < r0) r0 = r;
                if (r > r1) r1 = r;
                if (z < z0) z0 = z;
                if (z > z1) z1 = z;
            }
            int ix0 = (int)floor((r0 - Rmin) / m->hx - infl), ix1 = (int)floor((r1 - Rmin) / m->hx + infl);
            int iz0 = (int)floor((z0 - Zmin) / m->hz - infl), iz1 = (int)floor((z1 - Zmin) / m->hz + infl);
            if (ix0 < 0) ix0 = 0;
            if (iz0 < 0) iz0 = 0;
            if (ix1 >= g) ix1 = g - 1;
            if (iz1 >= g) iz1 = g - 1;
            for (int iz = iz0; iz <= iz1; ++iz)
                for (int ix = ix0; ix <= ix1; ++ix) {
                    int b = iz * g + ix;
                    if (pass == 0) m->start[b]++;
                    else m->cand[fill[b]++] = e;
                }
        }
        if (fill) free(fill);
    }
}

/* ------------------------------------------------------------------------------------------------ */
/* 3. naive polynomial evaluation (reading G10): sum_k c_k xi^i eta^j, k <-> (i,j), j outer, i inner     */
static void poly_eval(const double *c, double xi, double eta, double *val, double *dxi, double *deta)
{
    double xp[DEG + 1], ep[DEG + 1];
    xp[0] = 1.0; ep[0] = 1.0;
    for (int p = 1; p <= DEG; ++p) { xp[p] = xp[p - 1] * xi; ep[p] = ep[p - 1] * eta; }
    double v = 0.0, dx = 0.0, de = 0.0;
    int k = 0;
    for (int j = 0; j <= DEG; ++j)
        for (int i = 0; i <= DEG - j; ++i, ++k) {
            v += c[k] * (xp[i] * ep[j]);
            if (i > 0) dx += c[k] * ((double)i * (xp[i - 1] * ep[j]));
            if (j > 0) de += c[k] * ((double)j * (xp[i] * ep[j - 1]));
        }
    *val = v; *dxi = dx; *deta = de;
}

static void elem_frame(const orc_mesh *m, int e, double *Rc, double *Zc, double *s)
{
    const int *t = m->tri + 3 * e;
    const double *a = m->node_RZ + 2 * t[0], *b = m->node_RZ + 2 * t[1], *c = m->node_RZ + 2 * t[2];
    *Rc = (a[0] + b[0] + c[0]) / 3.0;
    *Zc = (a[1] + b[1] + c[1]) / 3.0;
    double l0 = sqrt((b[0] - a[0]) * (b[0] - a[0]) + (b[1] - a[1]) * (b[1] - a[1]));
    double l1 = sqrt((c[0] - b[0]) * (c[0] - b[0]) + (c[1] - b[1]) * (c[1] - b[1]));
    double l2 = sqrt((a[0] - c[0]) * (a[0] - c[0]) + (a[1] - c[1]) * (a[1] - c[1]));
    double L = l0 > l1 ? l0 : l1;
    if (l2 > L) L = l2;
    *s = 1.0 / L;
}

/* steps 3-4 on the finite-element tables */
static void fe_fields(const orc_mesh *m, int e, double R, double phi, double Z, double t, orc_fields *f)
{
    double Rc, Zc, s;
    elem_frame(m, e, &Rc, &Zc, &s);
    double xi = (R - Rc) * s, eta = (Z - Zc) * s;
    const double *ce = m->eq_coef + (size_t)e * N_EQ * NCOEF;
    double v, dx, de;
    poly_eval(ce + 0 * NCOEF, xi, eta, &v, &dx, &de);
    f->psi_R = dx * s; f->psi_Z = de * s;
    poly_eval(ce + 1 * NCOEF, xi, eta, &v, &dx, &de);
    f->Bm = v; f->Bm_R = dx * s; f->Bm_Z = de * s;
    poly_eval(ce + 2 * NCOEF, xi, eta, &v, &dx, &de);
    f->F = v;
    poly_eval(ce + 3 * NCOEF, xi, eta, &v, &dx, &de);
    f->kappa = v;
    for (int k = 0; k < 3; ++k) { f->E1[k] = 0.0; f->B1[k] = 0.0; f->gB1p[k] = 0.0; }
    f->dtB1p = 0.0; f->B1p = 0.0;
    for (int md = 0; md < m->n_modes; ++md) {
        const double *cp = m->pert_coef + ((size_t)md * m->n_elems + e) * (N_PERT * 2 * NCOEF);
        double n = (double)m->n_tor[md], om = m->omega[md];
        double th = n * phi - om * t;
        double cth = cos(th), sth = sin(th);
        double re[N_PERT], im[N_PERT], reR = 0, imR = 0, reZ = 0, imZ = 0;
        for (int q = 0; q < N_PERT; ++q) {
            double a, b, c2, d;
            poly_eval(cp + (2 * q + 0) * NCOEF, xi, eta, &re[q], &a, &b);
            poly_eval(cp + (2 * q + 1) * NCOEF, xi, eta, &im[q], &c2, &d);
            if (q == 6) { reR = a * s; reZ = b * s; imR = c2 * s; imZ = d * s; }
        }
        /* Re[C e^{i th}] = Cr cos - Ci sin ; d/dphi -> Re[i n C e^{i th}] = -n (Cr sin + Ci cos) ;
           d/dt -> Re[-i om C e^{i th}] = om (Cr sin + Ci cos)                                       */
        for (int k = 0; k < 3; ++k) {
            f->E1[k] += re[k] * cth - im[k] * sth;
            f->B1[k] += re[3 + k] * cth - im[3 + k] * sth;
        }
        double qd = re[6] * sth + im[6] * cth;
        f->B1p += re[6] * cth - im[6] * sth;
        f->gB1p[0] += reR * cth - imR * sth;
        f->gB1p[1] += -n * qd / R;
        f->gB1p[2] += reZ * cth - imZ * sth;
        f->dtB1p += om * qd;
    }
}

/* analytic back-end: the same quantities from closed forms */
static double an_q(const orc_analytic *a, double u, double *dqdu)
{
    if (u > 1.0) { u = 1.0; if (dqdu) *dqdu = 0.0; dqdu = NULL; }
    if (a->qkind == 0) { if (dqdu) *dqdu = a->qc[1]; return a->qc[0] + a->qc[1] * u; }
    if (dqdu) *dqdu = 2.0 * a->qc[1] * (u - a->qc[2]);
    return a->qc[0] + a->qc[1] * (u - a->qc[2]) * (u - a->qc[2]);
}

static double an_psi(const orc_analytic *a, double r)
{
    double u = (r / a->a) * (r / a->a), ui = u > 1.0 ? 1.0 : u, p;
    if (a->qkind == 0) p = a->B0 * a->a * a->a / (2.0 * a->qc[1]) * log1p(a->qc[1] * ui / a->qc[0]);
    else {
        double s = sqrt(a->qc[1] / a->qc[0]);
        p = a->B0 * a->a * a->a / (2.0 * sqrt(a->qc[0] * a->qc[1])) * (atan(s * (ui - a->qc[2])) + atan(s * a->qc[2]));
    }
    if (u > 1.0) p += a->B0 * (r * r - a->a * a->a) / (2.0 * an_q(a, 1.0, NULL));
    return p;
}

static void an_fields(const orc_analytic *a, double R, double phi, double Z, double t, orc_fields *f)
{
    double dR = R - a->R0, r2 = dR * dR + Z * Z, u = r2 / (a->a * a->a);
    double dqdu, q = an_q(a, u, &dqdu);
    double g = a->B0 / q;                                  /* (dpsi/dr)/r                    */
    double gp_over_r = -a->B0 / (q * q) * dqdu * 2.0 / (a->a * a->a); /* (dg/dr)/r          */
    double F = a->B0 * a->R0;
    f->psi_R = g * dR; f->psi_Z = g * Z; f->F = F; f->kappa = a->kappa;
    double S = g * g * r2 + F * F, sq = sqrt(S);           /* |B| = sqrt(S)/R                */
    double Sr_over_r = 2.0 * g * gp_over_r * r2 + 2.0 * g * g;
    f->Bm = sq / R;
    f->Bm_R = Sr_over_r * dR / (2.0 * sq * R) - sq / (R * R);
    f->Bm_Z = Sr_over_r * Z / (2.0 * sq * R);
    for (int k = 0; k < 3; ++k) { f->E1[k] = 0.0; f->B1[k] = 0.0; f->gB1p[k] = 0.0; }
    f->dtB1p = 0.0; f->B1p = 0.0;
    if (a->pA != 0.0) {
        double r = sqrt(r2), th = atan2(Z, dR);
        double arg = (r - a->prc) / a->pwd, G = a->pA * exp(-arg * arg), dG = -2.0 * arg / a->pwd * G;
        double ang = a->pn * phi - a->pm * th - a->pomega * t, ca = cos(ang), sa = sin(ang);
        double ct = dR / r, st = Z / r;
        /* Phi = G cos(ang); dang/dR = +m sin(th)/r, dang/dZ = -m cos(th)/r ; E = -grad Phi */
        double PhiR = dG * ct * ca - G * sa * (a->pm * st / r);
        double PhiZ = dG * st * ca - G * sa * (-a->pm * ct / r);
        f->E1[0] = -PhiR;
        f->E1[1] = (double)a->pn * G * sa / R;
        f->E1[2] = -PhiZ;
    }
}

/* ------------------------------------------------------------------------------------------------ */
/* 6. Eq. (6): (m/q)(v+ - v-)/dt = E + (v+ + v-)/2 x B.  With h = q dt/(2m) and (v x B) = M v,
 *    (I - h M) v+ = (I + h M) v- + 2 h E : solved by Gaussian elimination with partial pivoting.          */
static void eq6_solve(const double vm[3], const double E[3], const double B[3], double h, double vp[3])
{
    double M[3][3] = {{0.0, B[2], -B[1]}, {-B[2], 0.0, B[0]}, {B[1], -B[0], 0.0}};
    double A[3][4];
    for (int i = 0; i < 3; ++i) {
        double Mv = M[i][0] * vm[0] + M[i][1] * vm[1] + M[i][2] * vm[2];
        for (int j = 0; j < 3; ++j) A[i][j] = (i == j ? 1.0 : 0.0) - h * M[i][j];
        A[i][3] = vm[i] + h * Mv + 2.0 * h * E[i];
    }
    for (int c = 0; c < 3; ++c) {
        int p = c;
        for (int i = c + 1; i < 3; ++i)
            if (fabs(A[i][c]) > fabs(A[p][c])) p = i;
        if (p != c)
            for (int j = 0; j < 4; ++j) { double tmp = A[c][j]; A[c][j] = A[p][j]; A[p][j] = tmp; }
        for (int i = c + 1; i < 3; ++i) {
            double l = A[i][c] / A[c][c];
            for (int j = c; j < 4; ++j) A[i][j] -= l * A[c][j];
        }
    }
    for (int i = 2; i >= 0; --i) {
        double sacc = A[i][3];
        for (int j = i + 1; j < 3; ++j) sacc -= A[i][j] * vp[j];
        vp[i] = sacc / A[i][i];
    }
}

/* 7. weight RHS, Eqs. (8)-(13) in linear form (readings G5, G6, G7); all vectors cylindrical        */
static double weight_rhs(const orc_fields *f, const orc_species *sp, double R, const double vl[3], double mu)
{
    double q = sp->charge, m = sp->mass;
    double B0[3] = {-f->psi_Z / R, f->F / R, f->psi_R / R};            /* reading G4 */
    double B0n = sqrt(B0[0] * B0[0] + B0[1] * B0[1] + B0[2] * B0[2]);
    double b0[3] = {B0[0] / B0n, B0[1] / B0n, B0[2] / B0n};
    double vpar = vl[0] * b0[0] + vl[1] * b0[1] + vl[2] * b0[2];
    const double *E1 = f->E1, *B1 = f->B1;
    /* Eq. (12): (dX/dt)_1 = E1 x B0 / B0^2 + vpar B1 / B0 */
    double ExB[3] = {E1[1] * B0[2] - E1[2] * B0[1], E1[2] * B0[0] - E1[0] * B0[2], E1[0] * B0[1] - E1[1] * B0[0]};
    double dX[3];
    for (int k = 0; k < 3; ++k) dX[k] = ExB[k] / (B0n * B0n) + vpar * B1[k] / B0n;
    /* Eq. (13) (G5): m (dvpar/dt)_1 = q E1.b0 - mu b0.grad B1par */
    double Fpar = q * (E1[0] * b0[0] + E1[1] * b0[1] + E1[2] * b0[2])
                - mu * (b0[0] * f->gB1p[0] + b0[1] * f->gB1p[1] + b0[2] * f->gB1p[2]);
    /* Eq. (10) (G5): dPphi/dt = q (dX/dt)_1 . grad psi0 + m (dvpar/dt)_1 R Bphi0 / B0 */
    double dPphi = q * (dX[0] * f->psi_R + dX[2] * f->psi_Z) + Fpar * f->F / B0n;
    /* Eq. (11) (G6): dE/dt = q v_l . E1 + mu dB1par/dt */
    double dE = q * (vl[0] * E1[0] + vl[1] * E1[1] + vl[2] * E1[2]) + mu * f->dtB1p;
    /* d ln f0 / dE at fixed (Pphi, mu) (G7) */
    double v2 = vl[0] * vl[0] + vl[1] * vl[1] + vl[2] * vl[2];
    double Ekin = 0.5 * m * v2 + mu * f->Bm;
    double kE;
    if (sp->f0kind == 0) kE = -1.0 / sp->f0par[0];
    else {
        double v = sqrt(2.0 * Ekin / m), vc = sp->f0par[1];
        kE = -3.0 * v / (m * (v * v * v + vc * vc * vc));
        if (sp->f0kind == 2) {
            if (Ekin > 0.0) {                          /* a marker with v = 0 and mu = 0 has no pitch: the term is dropped */
                double Lam = mu * sp->f0par[4] / Ekin, L0 = sp->f0par[2], dL = sp->f0par[3];
                kE += 2.0 * (Lam - L0) * Lam / (dL * dL * Ekin);
            }
        }
    }
    /* Eqs. (8)-(9), (1-w) -> 1:  dw/dt = -[ (kappa/q) dPphi/dt + kE dE/dt ] */
    return -((f->kappa / q) * dPphi + kE * dE);
}

typedef struct {
    int kind;               /* 0: FE tables, 1: analytic */
    const orc_mesh *mesh;
    const orc_analytic *an;
    int brute;
} provider;

/* fields of either back-end at (R, phi, Z); returns 0 when the point is outside the mesh (FE back-end) */
static int provider_fields(const provider *pv, double R, double phi, double Z, double t, orc_fields *f)
{
    if (pv->kind == 0) {
        int e = pv->brute ? locate_brute(pv->mesh, R, Z) : locate_grid(pv->mesh, R, Z);
        if (e < 0) return 0;
        fe_fields(pv->mesh, e, R, phi, Z, t, f);
    } else {
        an_fields(pv->an, R, phi, Z, t, f);
    }
    return 1;
}

/* Finite Larmor radius (Eq. 14; reading G23): the four gyro-ring points
 * X + rho_L,j, |rho_L| = m v_perp / (|q| B) with v_perp = sqrt(2 mu B / m) "calculated from mu", uniformly spaced in
 * the gyro-angle in the plane perpendicular to b0: +-rho e1, +-rho e2 with e1 = the major-radius direction made
 * perpendicular to b0 and e2 = b0 x e1.  B0c = equilibrium field at X in cylindrical components, (c, sn) = cos / sin of
 * the marker's phi.  pts[4][3] Cartesian.                                                                          */
static void gyro_ring(const double X[3], const double B0c[3], double c, double sn, double mu, double q, double m,
                      double pts[4][3])
{
    double Bn = sqrt(B0c[0] * B0c[0] + B0c[1] * B0c[1] + B0c[2] * B0c[2]);
    double b[3] = {B0c[0] / Bn, B0c[1] / Bn, B0c[2] / Bn};
    double rho = sqrt(2.0 * m * mu / Bn) / fabs(q);
    double e1[3] = {1.0 - b[0] * b[0], -b[0] * b[1], -b[0] * b[2]};      /* R-hat - (R-hat . b) b, cylindrical */
    if (b[0] * b[0] > 0.999999) {                                        /* b (anti)parallel to R-hat: start from Z-hat */
        e1[0] = -b[2] * b[0]; e1[1] = -b[2] * b[1]; e1[2] = 1.0 - b[2] * b[2];
    }
    double n1 = sqrt(e1[0] * e1[0] + e1[1] * e1[1] + e1[2] * e1[2]);
    for (int k = 0; k < 3; ++k) e1[k] /= n1;
    double e2[3] = {b[1] * e1[2] - b[2] * e1[1], b[2] * e1[0] - b[0] * e1[2], b[0] * e1[1] - b[1] * e1[0]};
    /* cylindrical (R, phi, Z) components at the marker -> Cartesian */
    double e1c[3] = {e1[0] * c - e1[1] * sn, e1[0] * sn + e1[1] * c, e1[2]};
    double e2c[3] = {e2[0] * c - e2[1] * sn, e2[0] * sn + e2[1] * c, e2[2]};
    for (int k = 0; k < 3; ++k) {
        pts[0][k] = X[k] + rho * e1c[k]; pts[1][k] = X[k] + rho * e2c[k];
        pts[2][k] = X[k] - rho * e1c[k]; pts[3][k] = X[k] - rho * e2c[k];
    }
}

/* Eq. (14): <E1>, <B1>, <grad B1par>, <dB1par/dt> = quarter of the sum over the four ring points, vectors averaged in
 * Cartesian components and returned in the marker's cylindrical frame.  A ring point outside the mesh contributes zero. */
static void flr_average(const provider *pv, const double pts[4][3], double c, double sn, double t, orc_fields *f)
{
    double E[3] = {0, 0, 0}, B[3] = {0, 0, 0}, G[3] = {0, 0, 0}, dT = 0.0, Bp = 0.0;
    for (int j = 0; j < 4; ++j) {
        double x = pts[j][0], y = pts[j][1], z = pts[j][2];
        double R = sqrt(x * x + y * y), phi = atan2(y, x);
        orc_fields fj;
        if (!provider_fields(pv, R, phi, z, t, &fj)) continue;
        double cj = x / R, sj = y / R;
        const double *src[3] = {fj.E1, fj.B1, fj.gB1p};
        double *dst[3] = {E, B, G};
        for (int v = 0; v < 3; ++v) {
            dst[v][0] += src[v][0] * cj - src[v][1] * sj;
            dst[v][1] += src[v][0] * sj + src[v][1] * cj;
            dst[v][2] += src[v][2];
        }
        dT += fj.dtB1p; Bp += fj.B1p;
    }
    double *dst[3] = {f->E1, f->B1, f->gB1p};
    const double *src[3] = {E, B, G};
    for (int v = 0; v < 3; ++v) {
        dst[v][0] = 0.25 * (src[v][0] * c + src[v][1] * sn);
        dst[v][1] = 0.25 * (-src[v][0] * sn + src[v][1] * c);
        dst[v][2] = 0.25 * src[v][2];
    }
    f->dtB1p = 0.25 * dT; f->B1p = 0.25 * Bp;
}

/* one full step of one marker.  s = {x,y,z,vx,vy,vz,mu,w}.  Returns element (FE), 0 (analytic) or -1 = lost
 * (reading G12: a lost marker is frozen).  vl_out (optional) receives the Cartesian v_l.                  */
static int step_marker(const provider *pv, const orc_species *sp, double *s, double t, double dt, double *vl_out)
{
    double x = s[0], y = s[1], z = s[2];
    /* 1 */
    double R = sqrt(x * x + y * y), phi = atan2(y, x), Z = z;
    double c = x / R, sn = y / R;
    orc_fields f;
    int e = 0;
    if (pv->kind == 0) {
        /* 2 */
        e = pv->brute ? locate_brute(pv->mesh, R, Z) : locate_grid(pv->mesh, R, Z);
        if (e < 0) return -1;
        /* 3, 4 */
        fe_fields(pv->mesh, e, R, phi, Z, t, &f);
    } else {
        an_fields(pv->an, R, phi, Z, t, &f);
    }
    /* 5: linear mode: trajectory in the equilibrium field only.  Non-linear mode (reading G21):
     *    "the particle trajectories are calculated using the total fields": B = B0 + B1,
     *    E-dagger = E1 - (mu/q) grad(|B|0 + B1par), the mirror force of the total field strength.   */
    double mu = s[6], q = sp->charge, m = sp->mass;
    double BR = -f.psi_Z / R, BP = f.F / R, BZ = f.psi_R / R;
    double ER = -(mu / q) * f.Bm_R, EP = 0.0, EZ = -(mu / q) * f.Bm_Z;
    const int nonlinear = sp->mode == 1 || sp->mode == 3, flr = sp->mode == 2 || sp->mode == 3;
    if (flr) {   /* 4-point gyro-average of the perturbed fields (Eq. 14, reading G23): "one can use orbit-averaged fields <E1>,
                    <B1> in the above equations" -- in the weight equation (mode 2) and, in the non-linear
                    mode (mode 3), in the trajectory as well.  The ring is built on the EQUILIBRIUM field at x_l.            */
        double X[3] = {x, y, z}, B0c[3] = {BR, BP, BZ}, pts[4][3];
        gyro_ring(X, B0c, c, sn, mu, q, m, pts);
        flr_average(pv, pts, c, sn, t, &f);
    }
    if (nonlinear) {
        BR += f.B1[0]; BP += f.B1[1]; BZ += f.B1[2];
        ER = f.E1[0] - (mu / q) * (f.Bm_R + f.gB1p[0]);
        EP = f.E1[1] - (mu / q) * f.gB1p[1];
        EZ = f.E1[2] - (mu / q) * (f.Bm_Z + f.gB1p[2]);
    }
    double B[3] = {BR * c - BP * sn, BR * sn + BP * c, BZ};
    double E[3] = {ER * c - EP * sn, ER * sn + EP * c, EZ};
    /* 6 */
    double vm[3] = {s[3], s[4], s[5]}, vp[3];
    double h = q * dt / (2.0 * m);
    eq6_solve(vm, E, B, h, vp);
    /* 7 */
    double vl[3] = {0.5 * (vm[0] + vp[0]), 0.5 * (vm[1] + vp[1]), 0.5 * (vm[2] + vp[2])};
    double vlc[3] = {vl[0] * c + vl[1] * sn, -vl[0] * sn + vl[1] * c, vl[2]};
    double wdot = weight_rhs(&f, sp, R, vlc, mu);
    /* Eq. (8): dw/dt = -(1 - w) (1/f0) df0/dt; the linear mode takes (1 - w) -> 1, the non-linear mode
     * keeps the factor, explicit in w on the staggered grid (readings G9, G21)                                    */
    if (nonlinear) wdot *= (1.0 - s[7]);
    s[7] = s[7] + dt * wdot;
    /* 8 */
    s[0] = x + dt * vp[0]; s[1] = y + dt * vp[1]; s[2] = z + dt * vp[2];
    s[3] = vp[0]; s[4] = vp[1]; s[5] = vp[2];
    if (vl_out) { vl_out[0] = vl[0]; vl_out[1] = vl[1]; vl_out[2] = vl[2]; }
    return e;
}

/* ================================================================================================ */
/* exported entry points (ctypes)                                                                    */

orc_mesh *orc_mesh_create(int n_nodes, const double *node_RZ, int n_elems, const int *tri, const double *eq_coef,
                          int n_modes, const int *n_tor, const double *omega, const double *pert_coef)
{
    orc_mesh *m = (orc_mesh *)calloc(1, sizeof(orc_mesh));
    m->n_nodes = n_nodes; m->node_RZ = node_RZ; m->n_elems = n_elems; m->tri = tri; m->eq_coef = eq_coef;
    m->n_modes = n_modes; m->n_tor = n_tor; m->omega = omega; m->pert_coef = pert_coef;
    build_grid(m);
    return m;
}

void orc_mesh_free(orc_mesh *m)
{
    if (!m) return;
    free(m->start); free(m->cand); free(m);
}

void orc_locate(const orc_mesh *m, long n, const double *R, const double *Z, int *elem, int brute)
{
#pragma omp parallel for schedule(dynamic, 256)
    for (long i = 0; i < n; ++i) elem[i] = brute ? locate_brute(m, R[i], Z[i]) : locate_grid(m, R[i], Z[i]);
}

/* out[i][0..17] = psi_R psi_Z Bm Bm_R Bm_Z F kappa E1(3) B1(3) gB1p(3) dtB1p B1p ; elem[i] = -1: row untouched */
void orc_eval_fe(const orc_mesh *m, long n, const double *R, const double *phi, const double *Z, double t,
                 int *elem, double *out)
{
    for (long i = 0; i < n; ++i) {
        int e = locate_grid(m, R[i], Z[i]);
        elem[i] = e;
        if (e < 0) continue;
        orc_fields f;
        fe_fields(m, e, R[i], phi[i], Z[i], t, &f);
        double *o = out + 18 * i;
        o[0] = f.psi_R; o[1] = f.psi_Z; o[2] = f.Bm; o[3] = f.Bm_R; o[4] = f.Bm_Z; o[5] = f.F; o[6] = f.kappa;
        for (int k = 0; k < 3; ++k) { o[7 + k] = f.E1[k]; o[10 + k] = f.B1[k]; o[13 + k] = f.gB1p[k]; }
        o[16] = f.dtB1p; o[17] = f.B1p;
    }
}

void orc_eval_analytic(const orc_analytic *a, long n, const double *R, const double *phi, const double *Z, double t,
                       double *out, double *psi)
{
    for (long i = 0; i < n; ++i) {
        orc_fields f;
        an_fields(a, R[i], phi[i], Z[i], t, &f);
        double *o = out + 18 * i;
        o[0] = f.psi_R; o[1] = f.psi_Z; o[2] = f.Bm; o[3] = f.Bm_R; o[4] = f.Bm_Z; o[5] = f.F; o[6] = f.kappa;
        for (int k = 0; k < 3; ++k) { o[7 + k] = f.E1[k]; o[10 + k] = f.B1[k]; o[13 + k] = f.gB1p[k]; }
        o[16] = f.dtB1p; o[17] = f.B1p;
        double dR = R[i] - a->R0;
        if (psi) psi[i] = an_psi(a, sqrt(dR * dR + Z[i] * Z[i]));
    }
}

static void set_threads(int nthreads)
{
#ifdef _OPENMP
    if (nthreads > 0) omp_set_num_threads(nthreads);
#else
    (void)nthreads;
#endif
}

int orc_max_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/* push n markers nsteps steps; step counter starts at step0 (t_l = t0 + (step0+l) dt).
 * elem (optional, in/out): -1 on input = lost in an earlier call (stays frozen; pass -2 for "unknown");
 * on return the element of the last evaluated position x_l of the final step, or -1 if lost.
 * Returns the number of lost markers.                                                                  */
static long push_generic(const provider *pv, const orc_species *sp, long n, double *x, double *y, double *z,
                         double *vx, double *vy, double *vz, const double *mu, double *w, int *elem,
                         int nsteps, double dt, double t0, long step0, int nthreads)
{
    long lost = 0;
    set_threads(nthreads);
#pragma omp parallel for schedule(dynamic, 64) reduction(+ : lost)
    for (long i = 0; i < n; ++i) {
        double s[8] = {x[i], y[i], z[i], vx[i], vy[i], vz[i], mu[i], w[i]};
        int e = 0, dead = (elem && elem[i] == -1) ? 1 : 0; /* -1 on input: lost earlier, stays frozen */
        for (int l = 0; l < nsteps && !dead; ++l) {
            double t = t0 + (double)(step0 + l) * dt;
            e = step_marker(pv, sp, s, t, dt, NULL);
            if (e < 0) dead = 1;
        }
        if (dead) { lost++; e = -1; }
        x[i] = s[0]; y[i] = s[1]; z[i] = s[2]; vx[i] = s[3]; vy[i] = s[4]; vz[i] = s[5]; w[i] = s[7];
        if (elem) elem[i] = e;
    }
    return lost;
}

long orc_push_fe(const orc_mesh *m, const orc_species *sp, long n, double *x, double *y, double *z, double *vx,
                 double *vy, double *vz, const double *mu, double *w, int *elem, int nsteps, double dt, double t0,
                 long step0, int brute, int nthreads)
{
    provider pv = {0, m, NULL, brute};
    return push_generic(&pv, sp, n, x, y, z, vx, vy, vz, mu, w, elem, nsteps, dt, t0, step0, nthreads);
}

long orc_push_analytic(const orc_analytic *a, const orc_species *sp, long n, double *x, double *y, double *z,
                       double *vx, double *vy, double *vz, const double *mu, double *w, int nsteps, double dt,
                       double t0, long step0, int nthreads)
{
    provider pv = {1, NULL, a, 0};
    return push_generic(&pv, sp, n, x, y, z, vx, vy, vz, mu, w, NULL, nsteps, dt, t0, step0, nthreads);
}

/* trajectory of ONE marker: every `stride` steps store (x_l, v_l, w_{l+1/2}, t_l) -> out[k][8].
 * s[8] is updated in place.  mesh == NULL: analytic back-end.  Returns samples written.                  */
long orc_trace(const orc_mesh *m, const orc_analytic *a, const orc_species *sp, double *s, long nsteps, double dt,
               double t0, long stride, double *out)
{
    provider pv = {m ? 0 : 1, m, a, 0};
    long k = 0;
    for (long l = 0; l < nsteps; ++l) {
        double t = t0 + (double)l * dt, xl[3] = {s[0], s[1], s[2]}, vl[3];
        int e = step_marker(&pv, sp, s, t, dt, vl);
        if (e < 0) break;
        if (l % stride == 0) {
            double *o = out + 8 * k++;
            o[0] = xl[0]; o[1] = xl[1]; o[2] = xl[2]; o[3] = vl[0]; o[4] = vl[1]; o[5] = vl[2]; o[6] = s[7]; o[7] = t;
        }
    }
    return k;
}

/* Eq. (5)-(6) in uniform Cartesian fields (pins P1, P2) */
void orc_push_uniform(long n, double *x, double *y, double *z, double *vx, double *vy, double *vz, const double *B,
                      const double *E, double charge, double mass, long nsteps, double dt)
{
    double h = charge * dt / (2.0 * mass);
    for (long i = 0; i < n; ++i)
        for (long l = 0; l < nsteps; ++l) {
            double vm[3] = {vx[i], vy[i], vz[i]}, vp[3];
            eq6_solve(vm, E, B, h, vp);
            x[i] += dt * vp[0]; y[i] += dt * vp[1]; z[i] += dt * vp[2];
            vx[i] = vp[0]; vy[i] = vp[1]; vz[i] = vp[2];
        }
}

/* gyro ring of one marker at Cartesian X with magnetic moment mu (pins of reading G23); analytic back-end when m == NULL */
int orc_gyro_ring(const orc_mesh *m, const orc_analytic *a, const orc_species *sp, const double *X, double mu, double *pts12)
{
    provider pv = {m ? 0 : 1, m, a, 0};
    double R = sqrt(X[0] * X[0] + X[1] * X[1]), phi = atan2(X[1], X[0]);
    orc_fields f;
    if (!provider_fields(&pv, R, phi, X[2], 0.0, &f)) return 0;
    double B0c[3] = {-f.psi_Z / R, f.F / R, f.psi_R / R}, pts[4][3];
    gyro_ring(X, B0c, X[0] / R, X[1] / R, mu, sp->charge, sp->mass, pts);
    memcpy(pts12, pts, sizeof(pts));
    return 1;
}

/* gyro-averaged perturbed fields at X (marker frame): out10 = <E1>(3), <B1>(3), <grad B1par>(3), <dB1par/dt> */
int orc_flr_fields(const orc_mesh *m, const orc_analytic *a, const orc_species *sp, const double *X, double mu, double t,
                   double *out10)
{
    provider pv = {m ? 0 : 1, m, a, 0};
    double R = sqrt(X[0] * X[0] + X[1] * X[1]), phi = atan2(X[1], X[0]);
    orc_fields f;
    if (!provider_fields(&pv, R, phi, X[2], t, &f)) return 0;
    double B0c[3] = {-f.psi_Z / R, f.F / R, f.psi_R / R}, pts[4][3];
    gyro_ring(X, B0c, X[0] / R, X[1] / R, mu, sp->charge, sp->mass, pts);
    flr_average(&pv, pts, X[0] / R, X[1] / R, t, &f);
    for (int k = 0; k < 3; ++k) { out10[k] = f.E1[k]; out10[3 + k] = f.B1[k]; out10[6 + k] = f.gB1p[k]; }
    out10[9] = f.dtB1p;
    return 1;
}

void orc_eq6(const double *vm, const double *E, const double *B, double h, double *vp) { eq6_solve(vm, E, B, h, vp); }

double orc_weight_rhs(const double *fields18, const orc_species *sp, double R, const double *vl_cyl, double mu)
{
    orc_fields f;
    const double *o = fields18;
    f.psi_R = o[0]; f.psi_Z = o[1]; f.Bm = o[2]; f.Bm_R = o[3]; f.Bm_Z = o[4]; f.F = o[5]; f.kappa = o[6];
    for (int k = 0; k < 3; ++k) { f.E1[k] = o[7 + k]; f.B1[k] = o[10 + k]; f.gB1p[k] = o[13 + k]; }
    f.dtB1p = o[16]; f.B1p = o[17];
    return weight_rhs(&f, sp, R, vl_cyl, mu);
}

/* ================================================================================================ */
/* Guiding-centre equations with RK4 (Eqs. 1-4: the comparator pusher of Fig. 1 and the
 * "(dX/dt)_0 using only the equilibrium fields" of PAPER.md:130), equilibrium fields only (E = 0; reading G24):
 *     dX/dt      = (1/B*par) [ v_par B* + (mu/q) b x grad|B| ]            Eq. (1) with E = 0
 *     m dv_par/dt = -(mu/B*par) B* . grad|B|                               Eq. (2) with E = 0
 *     B* = B + (m v_par/q) curl b,   B*par = B* . b                        Eqs. (3), (4)
 * b = B/|B| with B = grad psi x grad phi + F grad phi (G4); grad|B| from the |B| table; curl b needs the
 * second derivatives of psi and the first of F -- the cost the paper's profile points at.
 * Axisymmetric: (curl b)_R = -d b_phi/dZ, (curl b)_phi = d b_R/dZ - d b_Z/dR, (curl b)_Z = (1/R) d(R b_phi)/dR.   */
typedef struct {
    double psi_R, psi_Z, psi_RR, psi_RZ, psi_ZZ, F, F_R, F_Z, Bm, Bm_R, Bm_Z;
} orc_gcf;

static void poly_eval2(const double *c, double xi, double eta, double *dxx, double *dxe, double *dee)
{
    double xp[DEG + 1], ep[DEG + 1];
    xp[0] = 1.0; ep[0] = 1.0;
    for (int p = 1; p <= DEG; ++p) { xp[p] = xp[p - 1] * xi; ep[p] = ep[p - 1] * eta; }
    double a = 0.0, b = 0.0, d = 0.0;
    int k = 0;
    for (int j = 0; j <= DEG; ++j)
        for (int i = 0; i <= DEG - j; ++i, ++k) {
            if (i > 1) a += c[k] * ((double)(i * (i - 1)) * (xp[i - 2] * ep[j]));
            if (i > 0 && j > 0) b += c[k] * ((double)(i * j) * (xp[i - 1] * ep[j - 1]));
            if (j > 1) d += c[k] * ((double)(j * (j - 1)) * (xp[i] * ep[j - 2]));
        }
    *dxx = a; *dxe = b; *dee = d;
}

static int gc_fields(const provider *pv, double R, double Z, orc_gcf *g)
{
    if (pv->kind == 0) {
        const orc_mesh *m = pv->mesh;
        int e = pv->brute ? locate_brute(m, R, Z) : locate_grid(m, R, Z);
        if (e < 0) return -1;
        double Rc, Zc, s;
        elem_frame(m, e, &Rc, &Zc, &s);
        double xi = (R - Rc) * s, eta = (Z - Zc) * s;
        const double *ce = m->eq_coef + (size_t)e * N_EQ * NCOEF;
        double v, dx, de, a, b, d;
        poly_eval(ce, xi, eta, &v, &dx, &de);
        poly_eval2(ce, xi, eta, &a, &b, &d);
        g->psi_R = dx * s; g->psi_Z = de * s; g->psi_RR = a * s * s; g->psi_RZ = b * s * s; g->psi_ZZ = d * s * s;
        poly_eval(ce + NCOEF, xi, eta, &v, &dx, &de);
        g->Bm = v; g->Bm_R = dx * s; g->Bm_Z = de * s;
        poly_eval(ce + 2 * NCOEF, xi, eta, &v, &dx, &de);
        g->F = v; g->F_R = dx * s; g->F_Z = de * s;
        return e;
    }
    const orc_analytic *a = pv->an;
    double dR = R - a->R0, r2 = dR * dR + Z * Z, u = r2 / (a->a * a->a);
    double dqdu, q = an_q(a, u, &dqdu);
    double gq = a->B0 / q, gp_over_r = -a->B0 / (q * q) * dqdu * 2.0 / (a->a * a->a);
    orc_fields f;
    an_fields(a, R, 0.0, Z, 0.0, &f);
    g->psi_R = f.psi_R; g->psi_Z = f.psi_Z; g->F = f.F; g->F_R = 0.0; g->F_Z = 0.0;
    g->Bm = f.Bm; g->Bm_R = f.Bm_R; g->Bm_Z = f.Bm_Z;
    g->psi_RR = gq + gp_over_r * dR * dR; g->psi_RZ = gp_over_r * dR * Z; g->psi_ZZ = gq + gp_over_r * Z * Z;
    return 0;
}

/* Eqs. (3)-(4) at (R, Z, v_par) from the field values g: b = B/|B| with |B| from its own table, curl b by the quotient rule
 * (axisymmetric), B* = B + (m v_par/q) curl b and the phase-space Jacobian B*par = B* . b.                              */
static double bstar(const orc_gcf *g, const orc_species *sp, double R, double vpar, double Bs[3], double b[3])
{
    double q = sp->charge, m = sp->mass;
    double B[3] = {-g->psi_Z / R, g->F / R, g->psi_R / R};
    double BR_R = -g->psi_RZ / R + g->psi_Z / (R * R), BR_Z = -g->psi_ZZ / R;
    double BP_R = g->F_R / R - g->F / (R * R), BP_Z = g->F_Z / R;
    double BZ_R = g->psi_RR / R - g->psi_R / (R * R), BZ_Z = g->psi_RZ / R;
    double Bm = g->Bm;
    for (int k = 0; k < 3; ++k) b[k] = B[k] / Bm;
    double bR_Z = (BR_Z - b[0] * g->Bm_Z) / Bm;
    double bP_R = (BP_R - b[1] * g->Bm_R) / Bm, bP_Z = (BP_Z - b[1] * g->Bm_Z) / Bm;
    double bZ_R = (BZ_R - b[2] * g->Bm_R) / Bm;
    (void)BR_R; (void)BZ_Z;
    double curlb[3] = {-bP_Z, bR_Z - bZ_R, b[1] / R + bP_R};
    double Bspar = 0.0;
    for (int k = 0; k < 3; ++k) { Bs[k] = B[k] + (m * vpar / q) * curlb[k]; Bspar += Bs[k] * b[k]; }
    return Bspar;
}

/* right-hand side of Eqs. (1)-(2) at (R, phi, Z, v_par, t): dX/dt in cylindrical components, dv_par/dt.  Returns -1 outside.
 *     dX/dt       = (1/B*par) [ v_par B* - b x (E - (mu/q) grad B) ]          Eq. (1)
 *     m dv_par/dt = (1/B*par) B* . (q E - mu grad B)                          Eq. (2)
 * sp->mode != 1: equilibrium fields only, E = 0 (reading G24).  sp->mode == 1 (reading G26): the guiding centre moves in
 * the total fields to first order in the perturbation: E = E1, B = B0 + B1 in B*, grad B = grad(|B|0 + B1par) as in the
 * mode-1 push (G21), while b, curl b and B*par = B* . b keep the equilibrium unit vector b0 (the perturbed part of b
 * needs derivatives of B1 that the field tables do not carry).  Linearised in the amplitude and at lowest order in rho*
 * the difference to the equilibrium right-hand side is Eq. (12): E1 x B0/B0^2 + v_par B1/B0.                          */
static int gc_rhs(const provider *pv, const orc_species *sp, double R, double phi, double Z, double vpar, double mu, double t,
                  double dX[3], double *dvpar)
{
    orc_gcf g;
    int e = gc_fields(pv, R, Z, &g);
    if (e < 0) return -1;
    double q = sp->charge, m = sp->mass;
    double Bs[3], b[3];
    double Bspar = bstar(&g, sp, R, vpar, Bs, b);
    double gB[3] = {g.Bm_R, 0.0, g.Bm_Z};
    double E[3] = {0.0, 0.0, 0.0};
    if (sp->mode == 1) {
        orc_fields f;
        if (pv->kind == 0) fe_fields(pv->mesh, e, R, phi, Z, t, &f);
        else an_fields(pv->an, R, phi, Z, t, &f);
        Bspar = 0.0;
        for (int k = 0; k < 3; ++k) { Bs[k] += f.B1[k]; Bspar += Bs[k] * b[k]; gB[k] += f.gB1p[k]; E[k] = f.E1[k]; }
    }
    double Ee[3];                                       /* E - (mu/q) grad B */
    for (int k = 0; k < 3; ++k) Ee[k] = E[k] - (mu / q) * gB[k];
    double bxE[3] = {b[1] * Ee[2] - b[2] * Ee[1], b[2] * Ee[0] - b[0] * Ee[2], b[0] * Ee[1] - b[1] * Ee[0]};
    for (int k = 0; k < 3; ++k) dX[k] = (vpar * Bs[k] - bxE[k]) / Bspar;
    *dvpar = (q / m) * (Bs[0] * Ee[0] + Bs[1] * Ee[1] + Bs[2] * Ee[2]) / Bspar;
    return e;
}

/* RK4 on y = (x, y, z, v_par) in Cartesian position.  Returns -1 when one of the four stages lies outside the mesh (the
 * caller keeps the state of the step before: lost), otherwise the element of the NEW position (FE back-end; 0 for the
 * analytic one), which is -1 as well when the step itself ends outside: then the new state is kept and the guiding centre
 * is lost from there.  *stage_lost tells the two cases apart.                                                          */
static int gc_step(const provider *pv, const orc_species *sp, double y[4], double mu, double t, double dt, int *stage_lost)
{
    double k[4][4], yy[4];
    static const double cs[4] = {0.0, 0.5, 0.5, 1.0};
    *stage_lost = 0;
    for (int st = 0; st < 4; ++st) {
        for (int i = 0; i < 4; ++i) yy[i] = y[i] + (st ? cs[st] * dt * k[st - 1][i] : 0.0);
        double R = sqrt(yy[0] * yy[0] + yy[1] * yy[1]), c = yy[0] / R, sn = yy[1] / R;
        double dX[3], dv;
        int e = gc_rhs(pv, sp, R, atan2(yy[1], yy[0]), yy[2], yy[3], mu, t + cs[st] * dt, dX, &dv);
        if (e < 0) { *stage_lost = 1; return -1; }
        k[st][0] = dX[0] * c - dX[1] * sn; k[st][1] = dX[0] * sn + dX[1] * c; k[st][2] = dX[2]; k[st][3] = dv;
    }
    for (int i = 0; i < 4; ++i) y[i] += dt / 6.0 * (k[0][i] + 2.0 * k[1][i] + 2.0 * k[2][i] + k[3][i]);
    if (pv->kind != 0) return 0;
    double Rn = sqrt(y[0] * y[0] + y[1] * y[1]);
    return pv->brute ? locate_brute(pv->mesh, Rn, y[2]) : locate_grid(pv->mesh, Rn, y[2]);
}

/* n guiding centres nsteps RK4 steps; elem (optional out): element of the CURRENT position, -1 = lost (frozen): either a
 * stage of a step left the mesh (state of the step before) or a step ended outside (state after that step)             */
long orc_gc_push(const orc_mesh *m, const orc_analytic *a, const orc_species *sp, long n, double *x, double *y, double *z,
                 double *vpar, const double *mu, int *elem, int nsteps, double dt, double t0, int nthreads)
{
    provider pv = {m ? 0 : 1, m, a, 0};
    long lost = 0;
    set_threads(nthreads);
#pragma omp parallel for schedule(dynamic, 64) reduction(+ : lost)
    for (long i = 0; i < n; ++i) {
        double s[4] = {x[i], y[i], z[i], vpar[i]};
        int e = 0, dead = 0;
        if (m) {                                           /* element of the starting position */
            e = locate_grid(m, sqrt(s[0] * s[0] + s[1] * s[1]), s[2]);
            if (e < 0) dead = 1;
        }
        for (int l = 0; l < nsteps && !dead; ++l) {
            double keep[4] = {s[0], s[1], s[2], s[3]};
            int stage_lost;
            e = gc_step(&pv, sp, s, mu[i], t0 + (double)l * dt, dt, &stage_lost);
            if (e < 0) { dead = 1; if (stage_lost) for (int q = 0; q < 4; ++q) s[q] = keep[q]; }
        }
        if (dead) { lost++; e = -1; }
        x[i] = s[0]; y[i] = s[1]; z[i] = s[2]; vpar[i] = s[3];
        if (elem) elem[i] = e;
    }
    return lost;
}

/* Bootstrap of the slow-manifold Boris scheme: "we use RK4 to advance the guiding center equations of motion
 * (Eqs. (1-4)) from x_0 to x_1, and then use (x_1 - x_0)/dt as v_{1/2}".  One RK4 guiding-centre step of size dt from
 * (x_0, v_par) with the equilibrium fields; on return the position is x_1 and v[3] = (x_1 - x_0)/dt: the pair
 * (x_1, v_{1/2}) is the staggered state the Boris step takes (velocity half a step behind the position).  ok[i] = 0 when
 * the step left the mesh (nothing is written for that marker).                                                        */
void orc_gc_bootstrap(const orc_mesh *m, const orc_analytic *a, const orc_species *sp, long n, double *x, double *y, double *z,
                      const double *vpar, const double *mu, double dt, double *vx, double *vy, double *vz, int *ok)
{
    provider pv = {m ? 0 : 1, m, a, 0};
    orc_species eq = *sp;
    eq.mode = 0;                                         /* the bootstrap uses the equilibrium fields */
    for (long i = 0; i < n; ++i) {
        double s[4] = {x[i], y[i], z[i], vpar[i]};
        int stage_lost;
        int e = gc_step(&pv, &eq, s, mu[i], 0.0, dt, &stage_lost);
        ok[i] = e >= 0;
        if (e < 0) continue;
        vx[i] = (s[0] - x[i]) / dt; vy[i] = (s[1] - y[i]) / dt; vz[i] = (s[2] - z[i]) / dt;
        x[i] = s[0]; y[i] = s[1]; z[i] = s[2];
    }
}

/* the field values gc_rhs works from, at given points, for the pins of poly_eval2 and of the finite-element branch of
 * gc_fields: out[n][11] = psi_R psi_Z psi_RR psi_RZ psi_ZZ F F_R F_Z Bm Bm_R Bm_Z; elem[i] = -1: row untouched          */
void orc_gc_fields(const orc_mesh *m, const orc_analytic *a, long n, const double *R, const double *Z, int *elem, double *out)
{
    provider pv = {m ? 0 : 1, m, a, 0};
    for (long i = 0; i < n; ++i) {
        orc_gcf g;
        elem[i] = gc_fields(&pv, R[i], Z[i], &g);
        if (elem[i] < 0) continue;
        double *o = out + 11 * i;
        o[0] = g.psi_R; o[1] = g.psi_Z; o[2] = g.psi_RR; o[3] = g.psi_RZ; o[4] = g.psi_ZZ;
        o[5] = g.F; o[6] = g.F_R; o[7] = g.F_Z; o[8] = g.Bm; o[9] = g.Bm_R; o[10] = g.Bm_Z;
    }
}

/* right-hand side at given points, for the pins: out[n][4] = dX/dt (R, phi, Z components), dv_par/dt */
void orc_gc_rhs(const orc_mesh *m, const orc_analytic *a, const orc_species *sp, long n, const double *R, const double *phi,
                const double *Z, const double *vpar, const double *mu, double t, double *out)
{
    provider pv = {m ? 0 : 1, m, a, 0};
    for (long i = 0; i < n; ++i) {
        double dX[3] = {0, 0, 0}, dv = 0.0;
        gc_rhs(&pv, sp, R[i], phi[i], Z[i], vpar[i], mu[i], t, dX, &dv);
        out[4 * i] = dX[0]; out[4 * i + 1] = dX[1]; out[4 * i + 2] = dX[2]; out[4 * i + 3] = dv;
    }
}

/* ================================================================================================ */
/* Moment deposition: right-hand sides of the Galerkin projection of the pressure moments with a
 * delta-function particle shape, Eqs. (17)-(18):
 *     rhs_par [e][h][k] = sum over markers p in element e of  w_p m v_par,p^2    nu_k(x_p) T_h(phi_p)
 *     rhs_perp[e][h][k] = sum over markers p in element e of  w_p mu_p |B|0(x_p) nu_k(x_p) T_h(phi_p)
 * nu_k = xi^i eta^j: the element's own polynomial basis (reading G10); T_0 = 1, T_{2m+1} = cos(n_m phi),
 * T_{2m+2} = sin(n_m phi) for the toroidal modes of the field set (reading G22: the delta function is normalised in
 * physical volume, so the Jacobian J of Eq. (17) is absorbed by it; v_par = v . B0/|B0| with the marker's v as stored).
 * rhs[n_elems][2][1 + 2 n_modes][21], zero-filled here.  Lost markers (outside every triangle) deposit nothing.
 * Plain loops, one marker at a time, in marker order.                                                             */
/* flags bit 0: the perpendicular moment carries the term of Eq. (16), mu |B|0 (w + B1par/|B|0) = w mu |B|0 + mu B1par,
 * with B1par = Re[C e^{i(n phi - omega t)}] at time t ("the change of perpendicular pressure due to the variation of
 * B_par"); without it Eq. (18) as printed.  flags bit 1: 4-point FLR deposition.  flags bit 2:
 * d = w + B1par/B*par replaces w in both moments (reading G25).                                           */
long orc_deposit(const orc_mesh *m, const orc_species *sp, long n, const double *x, const double *y, const double *z,
                 const double *vx, const double *vy, const double *vz, const double *mu, const double *w, double *rhs,
                 int flags, double t)
{
    const int H = 1 + 2 * m->n_modes;
    long lost = 0;
    memset(rhs, 0, (size_t)m->n_elems * 2 * H * NCOEF * sizeof(double));
    for (long p = 0; p < n; ++p) {
        double R = sqrt(x[p] * x[p] + y[p] * y[p]), phi = atan2(y[p], x[p]), Z = z[p];
        int e = locate_grid(m, R, Z);
        if (e < 0) { lost++; continue; }
        orc_fields f;
        fe_fields(m, e, R, phi, Z, t, &f);
        double B0[3] = {-f.psi_Z / R, f.F / R, f.psi_R / R};
        double B0n = sqrt(B0[0] * B0[0] + B0[1] * B0[1] + B0[2] * B0[2]);
        double c = x[p] / R, sn = y[p] / R;
        double vc[3] = {vx[p] * c + vy[p] * sn, -vx[p] * sn + vy[p] * c, vz[p]};
        double vpar = (vc[0] * B0[0] + vc[1] * B0[1] + vc[2] * B0[2]) / B0n;
        /* flags bit 2: "use d = w + (1 - w) B1* / B* to replace w in the summation in Eqs. (15) and (16) ... For a
         * linear simulation, the definition of d is d = w + B1* / B*": the change of the phase-space Jacobian B* = B*par of
         * Eq. (4).  B1* is taken as B1par (reading G25: the (m v_par/q)(b . curl b)_1 part of B1* needs curl B1, which the
         * field tables do not carry, and is smaller by rho*); B*par from the equilibrium with this marker's v_par.        */
        double dd = w[p];
        if (flags & 4) {
            provider pv = {0, m, NULL, 0};
            orc_gcf g;
            gc_fields(&pv, R, Z, &g);
            double Bs[3], bb[3];
            dd += f.B1p / bstar(&g, sp, R, vpar, Bs, bb);
        }
        double a[2] = {dd * sp->mass * vpar * vpar, dd * mu[p] * f.Bm};
        if (flags & 1) a[1] += mu[p] * f.B1p;
        /* deposition points: the marker itself, or (flags bit 1) the four gyro-ring points of reading G23
         * with a quarter of the amplitude each; a ring point outside the mesh deposits nothing                         */
        double pts[4][3], wgt = 1.0;
        int npts = 1;
        pts[0][0] = x[p]; pts[0][1] = y[p]; pts[0][2] = z[p];
        if (flags & 2) {
            double X[3] = {x[p], y[p], z[p]};
            gyro_ring(X, B0, c, sn, mu[p], sp->charge, sp->mass, pts);
            npts = 4; wgt = 0.25;
        }
        for (int jp = 0; jp < npts; ++jp) {
            double Rj = sqrt(pts[jp][0] * pts[jp][0] + pts[jp][1] * pts[jp][1]), phij = atan2(pts[jp][1], pts[jp][0]);
            double Zj = pts[jp][2];
            int ej = (flags & 2) ? locate_grid(m, Rj, Zj) : e;
            if (ej < 0) continue;
            double Rc, Zc, s;
            elem_frame(m, ej, &Rc, &Zc, &s);
            double xi = (Rj - Rc) * s, eta = (Zj - Zc) * s;
            double xp[DEG + 1], ep[DEG + 1];
            xp[0] = 1.0; ep[0] = 1.0;
            for (int q = 1; q <= DEG; ++q) { xp[q] = xp[q - 1] * xi; ep[q] = ep[q - 1] * eta; }
            for (int mom = 0; mom < 2; ++mom)
                for (int h = 0; h < H; ++h) {
                    double T = 1.0;
                    if (h > 0) {
                        double nn = (double)m->n_tor[(h - 1) / 2];
                        T = ((h - 1) % 2 == 0) ? cos(nn * phij) : sin(nn * phij);
                    }
                    double *out = rhs + (((size_t)ej * 2 + mom) * H + h) * NCOEF;
                    int k = 0;
                    for (int j = 0; j <= DEG; ++j)
                        for (int i = 0; i <= DEG - j; ++i, ++k) out[k] += wgt * a[mom] * T * (xp[i] * ep[j]);
                }
        }
    }
    return lost;
}

/* reference counting sort by element key (lost markers, key -1, last): returns a permutation.  Any
 * permutation with non-decreasing keys is valid (SURVEY.md 8(c) "Sort oracle"); this one is stable.   */
void orc_sort_perm(long n, const int *elem, int n_elems, long *perm)
{
    long *count = (long *)calloc((size_t)n_elems + 2, sizeof(long));
    for (long i = 0; i < n; ++i) count[(elem[i] < 0 ? n_elems : elem[i]) + 1]++;
    for (int k = 0; k <= n_elems; ++k) count[k + 1] += count[k];
    for (long i = 0; i < n; ++i) perm[count[elem[i] < 0 ? n_elems : elem[i]]++] = i;
    free(count);
}
