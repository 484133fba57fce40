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

// One 32-byte read-only load (LDG.E.256.CONSTANT, sm_100): four interleaved coefficients.  Not volatile: the tables
// are immutable for the lifetime of a kernel, so the compiler may hoist and reorder these freely.
struct Quad { double a, b, c, d; };
__device__ __forceinline__ Quad ldq(const double *p) {
    Quad q;
    asm("ld.global.nc.v4.f64 {%0, %1, %2, %3}, [%4];" : "=d"(q.a), "=d"(q.b), "=d"(q.c), "=d"(q.d) : "l"(p));
    return q;
}

// ---- polynomial quads (G10: monomials xi^i eta^j, j outer, i inner; row j starts at kRow[j], has 6 - j terms) -----
// c[4 k + s]: coefficient k of slot s.  Horner in xi inside a row, Horner in eta across rows; value, d/dxi, d/deta of
// all four slots: 38 FMA per slot.  Callers ignore the outputs they do not need; after full unrolling the unused
// chains are dead code and disappear (value only: 20 FMA per slot).
__device__ __forceinline__ void quad_vd(const double *__restrict__ c, double xi, double eta, double (&v)[4],
                                        double (&dx)[4], double (&de)[4]) {
    constexpr int kRow[6] = {0, 6, 11, 15, 18, 20};
    double a[4], ax[4], ae[4];
#pragma unroll
    for (int j = 5; j >= 0; --j) {
        const int L = 6 - j;
        const Quad t = ldq(c + 4 * (kRow[j] + L - 1));
        double p[4] = {t.a, t.b, t.c, t.d}, d[4] = {0.0, 0.0, 0.0, 0.0};
#pragma unroll
        for (int i = L - 2; i >= 0; --i) {
            const Quad u = ldq(c + 4 * (kRow[j] + i));
            const double uu[4] = {u.a, u.b, u.c, u.d};
#pragma unroll
            for (int s = 0; s < 4; ++s) {
                d[s] = (i == L - 2) ? p[s] : M3DK_FMA(d[s], xi, p[s]);
                p[s] = M3DK_FMA(p[s], xi, uu[s]);
            }
        }
#pragma unroll
        for (int s = 0; s < 4; ++s) {
            if (j == 5) { a[s] = p[s]; ax[s] = 0.0; ae[s] = 0.0; }
            else {
                if (j == 4) { ae[s] = a[s]; ax[s] = d[s]; }
                else { ae[s] = M3DK_FMA(ae[s], eta, a[s]); ax[s] = M3DK_FMA(ax[s], eta, d[s]); }
                a[s] = M3DK_FMA(a[s], eta, p[s]);
            }
        }
    }
#pragma unroll
    for (int s = 0; s < 4; ++s) { v[s] = a[s]; dx[s] = ax[s]; de[s] = ae[s]; }
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

// ---- fast element search: fp32 edge functions in bucket-local coordinates, conservative ---------------------------
// Returns the element when the point is strictly inside a candidate by more than the fp32 error bound (then rule G11
// yields the same element), otherwise -2: the caller falls back to the exact search `locate`.
__device__ __forceinline__ FastRec ldrec(const FastRec *p) {
    unsigned r[8];
    asm("ld.global.nc.v8.b32 {%0, %1, %2, %3, %4, %5, %6, %7}, [%8];"
        : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]) : "l"(p));
    FastRec q;
    q.x0 = __uint_as_float(r[0]); q.y0 = __uint_as_float(r[1]); q.x1 = __uint_as_float(r[2]);
    q.y1 = __uint_as_float(r[3]); q.x2 = __uint_as_float(r[4]); q.y2 = __uint_as_float(r[5]);
    q.id = (int)r[6]; q.next = (int)r[7];
    return q;
}

// The asm loads are not volatile, so the compiler may hoist them above the range checks: every address is therefore
// clamped into its table first and the checks only decide whether the loaded record is used.
__device__ __forceinline__ int locate_fast(const FastGrid &g, double R, double Z) {
    const double fx = (R - g.Rmin) * g.inv_hx, fz = (Z - g.Zmin) * g.inv_hz;
    const bool inside = fx >= 0.0 && fx < (double)g.gx && fz >= 0.0 && fz < (double)g.gz;
    const int ix = inside ? (int)fx : 0, iz = inside ? (int)fz : 0;
    const float u = (float)(fx - (double)ix), v = (float)(fz - (double)iz);
    FastRec r = ldrec(g.first + (size_t)(iz * g.gx + ix));
    int found = -2;
    bool open = inside;
#pragma unroll 1
    for (int it = 0; it < 4 && open; ++it) {
        const float e0 = __fmul_rn(r.x1 - r.x0, v - r.y0) - __fmul_rn(r.y1 - r.y0, u - r.x0);
        const float e1 = __fmul_rn(r.x2 - r.x1, v - r.y1) - __fmul_rn(r.y2 - r.y1, u - r.x1);
        const float e2 = __fmul_rn(r.x0 - r.x2, v - r.y2) - __fmul_rn(r.y0 - r.y2, u - r.x2);
        if (r.id >= 0 && e0 > kFastMargin && e1 > kFastMargin && e2 > kFastMargin) { found = r.id; open = false; }
        else if (r.id < 0 || r.next < 0) open = false;
        else r = ldrec(g.ovf + max(r.next, 0));
    }
    return found;
}

__device__ __forceinline__ int locate_any(const FieldParams &f, double R, double Z) {
    const int e = locate_fast(f.fast, R, Z);
    return e != -2 ? e : locate(f.grid, R, Z);
}

// ---- fields at (R, phi, Z) in element e -----------------------------------------------------
// cph, sph = cos phi, sin phi; rinv = 1/R; cwt/swt = cos / sin(omega_k t).  When all lanes of a warp pass the same e
// every load below is a one-wavefront broadcast.
__device__ __forceinline__ void eval_fields(const FieldParams &f, int e, double R, double Z, double cph, double sph,
                                            double rinv, const double *cwt, const double *swt, Fields &o) {
    const double *tile = f.tiles + (size_t)max(e, 0) * f.tile_stride;   // clamped: the loads may be speculated
    const Quad h = ldq(tile);
    const double Rc = h.a, Zc = h.b, se = h.c;
    const double xi = (R - Rc) * se, eta = (Z - Zc) * se;
    double v[4], dx[4], de[4];
    quad_vd(tile + kTileHeader, xi, eta, v, dx, de);          // (psi0, |B|0, F0, kappa)
    o.psi_R = dx[0] * se; o.psi_Z = de[0] * se;
    o.Bm = v[1]; o.Bm_R = dx[1] * se; o.Bm_Z = de[1] * se;
    o.F = v[2]; o.kappa = v[3];
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
        const double *pm = tile + kTileHeader + kTileEq + kTileMode * md;
        // Re[C e^{i th}] = Cr cos th - Ci sin th
        quad_vd(pm, xi, eta, v, dx, de);                      // E_R, E_phi
        o.E1[0] += v[0] * cth - v[1] * sth;
        o.E1[1] += v[2] * cth - v[3] * sth;
        quad_vd(pm + kQuad, xi, eta, v, dx, de);              // E_Z, B_R
        o.E1[2] += v[0] * cth - v[1] * sth;
        o.B1[0] += v[2] * cth - v[3] * sth;
        quad_vd(pm + 2 * kQuad, xi, eta, v, dx, de);          // B_phi, B_Z
        o.B1[1] += v[0] * cth - v[1] * sth;
        o.B1[2] += v[2] * cth - v[3] * sth;
        quad_vd(pm + 3 * kQuad, xi, eta, v, dx, de);          // B_par with gradient (slots 2, 3 are padding)
        const double re = v[0], im = v[1];
        const double qd = re * sth + im * cth;               // -Im-part combination: d/dphi -> -n qd, d/dt -> omega qd
        o.B1p += re * cth - im * sth;
        o.gB[0] += (dx[0] * se) * cth - (dx[1] * se) * sth;
        o.gB[1] += -(double)n * qd * rinv;
        o.gB[2] += (de[0] * se) * cth - (de[1] * se) * sth;
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

struct StepGeom { double R, rinv, cph, sph; };

// cylindrical map (G3)
__device__ __forceinline__ void step_geometry(const Marker &s, StepGeom &g) {
    g.R = sqrt(s.x * s.x + s.y * s.y);
    g.rinv = 1.0 / g.R;
    g.cph = s.x * g.rinv; g.sph = s.y * g.rinv;
}

__device__ __forceinline__ void step_marker(const PushParams &P, const StepGeom &g, const Fields &f, Marker &s) {
    const double rinv = g.rinv, cph = g.cph, sph = g.sph;
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

__device__ __forceinline__ int locate_xyz(const FieldParams &f, double x, double y, double z) {
    return locate_any(f, sqrt(x * x + y * y), z);
}

}  // namespace m3dk
