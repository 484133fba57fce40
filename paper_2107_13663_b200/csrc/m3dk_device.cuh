// m3dk_device.cuh -- device code of the hot path: element search, Horner field evaluation, Boris step, weight.
// Product path (libm3dk).  Shares nothing with oracle/.  Citations are PAPER.md lines; G# are DESIGN.md readings.
#pragma once

#include "m3dk_internal.h"

namespace m3dk {

// Verification build (-fmad=false -DM3DK_NO_FMA): no fused multiply-add anywhere, explicit or contracted.
#ifdef M3DK_NO_FMA
#define M3DK_FMA(a, b, c) __dadd_rn(__dmul_rn((a), (b)), (c))
#else
#define M3DK_FMA(a, b, c) fma((a), (b), (c))
#endif

struct Fields {
    double psi_R, psi_Z;        // d psi0/dR, d psi0/dZ
    double Bm, Bm_R, Bm_Z;      // |B|0 as its own scalar field and its gradient
    double F, kappa;            // R B_phi0, d ln f0 / d psi
    double E1[3], B1[3];        // perturbed fields, (R, phi, Z)
    double gB[3];               // grad B1par, phi component = (1/R) d/dphi
    double dtB, B1p;            // d B1par/dt, B1par
};

__device__ __forceinline__ double2 ldc(const double2 *p) { return __ldg(p); }

// ---- polynomial pairs (G10: monomials xi^i eta^j, j outer, i inner; row j starts at kRow[j], has 6 - j terms) -----
// c[k] = (a_k, b_k): two quintics evaluated together, Horner in xi inside a row, Horner in eta across rows.
// value only: 15 + 5 FMA per polynomial.
__device__ __forceinline__ void pair_v(const double2 *__restrict__ c, double xi, double eta, double &va, double &vb) {
    constexpr int kRow[6] = {0, 6, 11, 15, 18, 20};
    double a = 0.0, b = 0.0;
#pragma unroll
    for (int j = 5; j >= 0; --j) {
        const int L = 6 - j;
        double2 t = ldc(c + kRow[j] + L - 1);
        double pa = t.x, pb = t.y;
#pragma unroll
        for (int i = L - 2; i >= 0; --i) {
            t = ldc(c + kRow[j] + i);
            pa = M3DK_FMA(pa, xi, t.x);
            pb = M3DK_FMA(pb, xi, t.y);
        }
        if (j == 5) { a = pa; b = pb; }
        else { a = M3DK_FMA(a, eta, pa); b = M3DK_FMA(b, eta, pb); }
    }
    va = a; vb = b;
}

// value, d/dxi, d/deta: 38 FMA per polynomial.
__device__ __forceinline__ void pair_vd(const double2 *__restrict__ c, double xi, double eta, double &va, double &dxa,
                                        double &dea, double &vb, double &dxb, double &deb) {
    constexpr int kRow[6] = {0, 6, 11, 15, 18, 20};
    double a = 0.0, b = 0.0, ax = 0.0, bx = 0.0, ae = 0.0, be = 0.0;
#pragma unroll
    for (int j = 5; j >= 0; --j) {
        const int L = 6 - j;
        double2 t = ldc(c + kRow[j] + L - 1);
        double pa = t.x, pb = t.y, da = 0.0, db = 0.0;
#pragma unroll
        for (int i = L - 2; i >= 0; --i) {
            if (i == L - 2) { da = pa; db = pb; }
            else { da = M3DK_FMA(da, xi, pa); db = M3DK_FMA(db, xi, pb); }
            t = ldc(c + kRow[j] + i);
            pa = M3DK_FMA(pa, xi, t.x);
            pb = M3DK_FMA(pb, xi, t.y);
        }
        if (j == 5) { a = pa; b = pb; }
        else {
            if (j == 4) { ae = a; be = b; ax = da; bx = db; }
            else {
                ae = M3DK_FMA(ae, eta, a); be = M3DK_FMA(be, eta, b);
                ax = M3DK_FMA(ax, eta, da); bx = M3DK_FMA(bx, eta, db);
            }
            a = M3DK_FMA(a, eta, pa); b = M3DK_FMA(b, eta, pb);
        }
    }
    va = a; vb = b; dxa = ax; dxb = bx; dea = ae; deb = be;
}

// ---- element search (G11) ------------------------------------------------------------------------------------------
// Edge functions (x_b - x_a)(Z - z_a) - (z_b - z_a)(R - r_a), each operation rounded separately (never contracted, in
// either build), so that the GPU and the oracle agree bit for bit on which side of an edge a marker is.
__device__ __forceinline__ void edge_fn(const double *__restrict__ rec, double R, double Z, double &e0, double &e1,
                                        double &e2) {
    const double2 *r2 = reinterpret_cast<const double2 *>(rec);
    double2 a0 = ldc(r2 + 0), d0 = ldc(r2 + 1), a1 = ldc(r2 + 2), d1 = ldc(r2 + 3), a2 = ldc(r2 + 4), d2 = ldc(r2 + 5);
    e0 = __dsub_rn(__dmul_rn(d0.x, __dsub_rn(Z, a0.y)), __dmul_rn(d0.y, __dsub_rn(R, a0.x)));
    e1 = __dsub_rn(__dmul_rn(d1.x, __dsub_rn(Z, a1.y)), __dmul_rn(d1.y, __dsub_rn(R, a1.x)));
    e2 = __dsub_rn(__dmul_rn(d2.x, __dsub_rn(Z, a2.y)), __dmul_rn(d2.y, __dsub_rn(R, a2.x)));
}

// Element containing (R, Z): the smallest index among the elements whose three edge functions are all >= 0, or -1.
// Two phases over the bucket's candidate list (a superset of every element touching the bucket, priority order):
// a candidate that contains the point strictly (all edge functions above its tolerance) is the only one that can
// contain it, so it is returned at once; otherwise (the point is within rounding of an edge) take the minimum index.
__device__ __forceinline__ int locate(const GridParams &g, double R, double Z) {
    if (!(R >= g.Rmin && R <= g.Rmax && Z >= g.Zmin && Z <= g.Zmax)) return -1;
    int ix = (int)((R - g.Rmin) * g.inv_hx), iz = (int)((Z - g.Zmin) * g.inv_hz);
    ix = min(max(ix, 0), g.gx - 1);
    iz = min(max(iz, 0), g.gz - 1);
    const int b = iz * g.gx + ix;
    const int k0 = __ldg(g.bstart + b), k1 = __ldg(g.bstart + b + 1);
    int best = 0x7fffffff;
    for (int k = k0; k < k1; ++k) {
        const int e = __ldg(g.bcand + k);
        const double *rec = g.edges + (size_t)e * kEdgeRec;
        double e0, e1, e2;
        edge_fn(rec, R, Z, e0, e1, e2);
        const double tol = __ldg(rec + 12);
        if (e0 > tol && e1 > tol && e2 > tol) return e;
        if (e0 >= 0.0 && e1 >= 0.0 && e2 >= 0.0) best = min(best, e);
    }
    return best == 0x7fffffff ? -1 : best;
}

// ---- fields at (R, phi, Z) in element e -----------------------------------------------------
// cph, sph = cos phi, sin phi; rinv = 1/R; cwt/swt = cos / sin(omega_k t).  NM: number of toroidal modes to evaluate.
__device__ __forceinline__ void eval_fields(const FieldParams &f, int e, double R, double Z, double cph, double sph,
                                            double rinv, const double *cwt, const double *swt, Fields &o) {
    const double *tile = f.tiles + (size_t)e * f.tile_stride;
    const double2 *t2 = reinterpret_cast<const double2 *>(tile);
    const double2 h0 = ldc(t2), h1 = ldc(t2 + 1);
    const double Rc = h0.x, Zc = h0.y, se = h1.x;
    const double xi = (R - Rc) * se, eta = (Z - Zc) * se;
    double v0, dx0, de0, v1, dx1, de1;
    pair_vd(t2 + kTileHeader / 2, xi, eta, v0, dx0, de0, v1, dx1, de1);
    o.psi_R = dx0 * se; o.psi_Z = de0 * se;
    o.Bm = v1; o.Bm_R = dx1 * se; o.Bm_Z = de1 * se;
    pair_v(t2 + (kTileHeader + kPair) / 2, xi, eta, o.F, o.kappa);
#pragma unroll
    for (int k = 0; k < 3; ++k) { o.E1[k] = 0.0; o.B1[k] = 0.0; o.gB[k] = 0.0; }
    o.dtB = 0.0; o.B1p = 0.0;
    for (int md = 0; md < f.n_modes; ++md) {
        // exp(i n phi) by complex powers of (cos phi + i sin phi); exp(-i omega t) from the host
        const int n = f.n_tor[md];
        double cn = 1.0, sn = 0.0;
        for (int k = 0; k < abs(n); ++k) {
            const double c2 = cn * cph - sn * sph;
            sn = cn * sph + sn * cph;
            cn = c2;
        }
        if (n < 0) sn = -sn;
        const double cth = cn * cwt[md] + sn * swt[md];      // cos(n phi - omega t)
        const double sth = sn * cwt[md] - cn * swt[md];      // sin(n phi - omega t)
        const double2 *pm = t2 + (kTileHeader + kTileEq + kTileMode * md) / 2;
        // Re[C e^{i th}] = Cr cos th - Ci sin th
#pragma unroll
        for (int q = 0; q < 3; ++q) {
            double re, im;
            pair_v(pm + q * M3DK_NCOEF, xi, eta, re, im);
            o.E1[q] += re * cth - im * sth;
        }
#pragma unroll
        for (int q = 0; q < 3; ++q) {
            double re, im;
            pair_v(pm + (3 + q) * M3DK_NCOEF, xi, eta, re, im);
            o.B1[q] += re * cth - im * sth;
        }
        double re, reX, reE, im, imX, imE;
        pair_vd(pm + 6 * M3DK_NCOEF, xi, eta, re, reX, reE, im, imX, imE);
        const double qd = re * sth + im * cth;               // -Im-part combination: d/dphi -> -n qd, d/dt -> omega qd
        o.B1p += re * cth - im * sth;
        o.gB[0] += (reX * se) * cth - (imX * se) * sth;
        o.gB[1] += -(double)n * qd * rinv;
        o.gB[2] += (reE * se) * cth - (imE * se) * sth;
        o.dtB += f.omega[md] * qd;
    }
}

// d ln f0 / dE at fixed (P_phi, mu) (G7)
__device__ __forceinline__ double kappa_E(const PushParams &P, double Ekin, double mu) {
    if (P.f0kind == M3DK_F0_MAXWELLIAN) return -P.f0T_inv;
    const double v = sqrt(2.0 * Ekin / P.m);
    double kE = -3.0 * v / (P.m * (v * v * v + P.f0vc3));
    if (P.f0kind == M3DK_F0_BEAM_PITCH) {
        const double Lam = mu * P.f0Bax / Ekin;
        kE += 2.0 * (Lam - P.f0L0) * Lam * P.f0dL2_inv / Ekin;
    }
    return kE;
}

// ---- one step of one marker (PAPER.md:73-78 Eqs. 5-6; :106-130 Eqs. 8-13; :140) -----------------------------------
// state in: (x_l, v_{l-1/2}, mu, w_{l-1/2}) with e = element of x_l;  out: (x_{l+1}, v_{l+1/2}, w_{l+1/2}).
struct Marker { double x, y, z, vx, vy, vz, mu, w; };

__device__ __forceinline__ void step_marker(const PushParams &P, int e, Marker &s) {
    // cylindrical map (G3)
    const double R = sqrt(s.x * s.x + s.y * s.y);
    const double rinv = 1.0 / R;
    const double cph = s.x * rinv, sph = s.y * rinv;
    Fields f;
    eval_fields(P.f, e, R, s.z, cph, sph, rinv, P.cwt, P.swt, f);
    // B0 = grad psi0 x grad phi + F0 grad phi (G4); E-dagger = -(mu/q) grad|B|0 (G2)
    const double BR = -f.psi_Z * rinv, BP = f.F * rinv, BZ = f.psi_R * rinv;
    const double muq = s.mu * P.inv_q;
    const double ER = -muq * f.Bm_R, EZ = -muq * f.Bm_Z;
    const double Bx = BR * cph - BP * sph, By = BR * sph + BP * cph, Bz = BZ;
    const double Ex = ER * cph, Ey = ER * sph, Ez = EZ;
    // Eq. (6) in the explicit Boris form: half kick, rotation t = h B, s = 2 t / (1 + t^2), half kick
    const double h = P.h;
    const double ux = s.vx + h * Ex, uy = s.vy + h * Ey, uz = s.vz + h * Ez;
    const double tx = h * Bx, ty = h * By, tz = h * Bz;
    const double sc = 2.0 / (1.0 + (tx * tx + ty * ty + tz * tz));
    const double px = ux + (uy * tz - uz * ty), py = uy + (uz * tx - ux * tz), pz = uz + (ux * ty - uy * tx);
    const double wx = ux + sc * (py * tz - pz * ty), wy = uy + sc * (pz * tx - px * tz), wz = uz + sc * (px * ty - py * tx);
    const double nvx = wx + h * Ex, nvy = wy + h * Ey, nvz = wz + h * Ez;
    // weight, Eqs. (8)-(13) at (x_l, v_l), v_l = (v_{l-1/2} + v_{l+1/2}) / 2; skipped without modes
    if (P.f.n_modes > 0) {
        const double vlx = 0.5 * (s.vx + nvx), vly = 0.5 * (s.vy + nvy), vlz = 0.5 * (s.vz + nvz);
        const double vR = vlx * cph + vly * sph, vP = vly * cph - vlx * sph, vZ = vlz;
        const double B2 = BR * BR + BP * BP + BZ * BZ;
        const double binv = 1.0 / sqrt(B2);
        const double bR = BR * binv, bP = BP * binv, bZ = BZ * binv;
        const double vpar = vR * bR + vP * bP + vZ * bZ;
        // Eq. (12): (dX/dt)_1 = E1 x B0 / B0^2 + v_par B1 / B0 ; only its (R, Z) components meet grad psi0
        const double cR = f.E1[1] * BZ - f.E1[2] * BP, cZ = f.E1[0] * BP - f.E1[1] * BR;
        const double b2inv = binv * binv;
        const double dXR = cR * b2inv + vpar * f.B1[0] * binv, dXZ = cZ * b2inv + vpar * f.B1[2] * binv;
        // Eq. (13) x m (G5)
        const double Fpar = P.q * (f.E1[0] * bR + f.E1[1] * bP + f.E1[2] * bZ) - s.mu * (bR * f.gB[0] + bP * f.gB[1] + bZ * f.gB[2]);
        // Eq. (10) (G5), Eq. (11) (G6)
        const double dP = P.q * (dXR * f.psi_R + dXZ * f.psi_Z) + Fpar * f.F * binv;
        const double dE = P.q * (vR * f.E1[0] + vP * f.E1[1] + vZ * f.E1[2]) + s.mu * f.dtB;
        const double Ekin = 0.5 * P.m * (vlx * vlx + vly * vly + vlz * vlz) + s.mu * f.Bm;
        const double kE = kappa_E(P, Ekin, s.mu);
        // Eqs. (8)-(9) with (1 - w) -> 1; explicit midpoint on the staggered grid (G9)
        const double wdot = -((f.kappa * P.inv_q) * dP + kE * dE);
        s.w = s.w + P.dt * wdot;
    }
    // Eq. (5)
    s.x = s.x + P.dt * nvx; s.y = s.y + P.dt * nvy; s.z = s.z + P.dt * nvz;
    s.vx = nvx; s.vy = nvy; s.vz = nvz;
}

__device__ __forceinline__ int locate_xyz(const GridParams &g, double x, double y, double z) {
    return locate(g, sqrt(x * x + y * y), z);
}

}  // namespace m3dk
