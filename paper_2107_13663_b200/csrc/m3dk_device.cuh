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

// ---- reciprocal, reciprocal square root, square root: hardware seed (MUFU.RCP64H / RSQ64H, ~20 bits) + two Newton
// steps, ~1 ulp.  fp64 division and square root have no hardware unit; the IEEE-rounded library sequences cost about
// three times as many FP64-pipe instructions plus a slow-path branch, and a step has seven of them.  The parity bar is
// 1e-12, four orders above the difference.  Arguments are positive and normal wherever these are used (R >= R_min > 0,
// |B|^2 > 0, 1 + t^2 >= 1, v^3 + v_c^3 > 0); m3dk_sqrt also accepts 0.
__device__ __forceinline__ double m3dk_rcp(double x) {
    double y;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
    double e = M3DK_FMA(-x, y, 1.0);
    y = M3DK_FMA(y, e, y);
    e = M3DK_FMA(-x, y, 1.0);
    return M3DK_FMA(y, e, y);
}
__device__ __forceinline__ double m3dk_rsqrt(double x) {
    double y;
    asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
    const double hx = __dmul_rn(0.5, x);
    double e = M3DK_FMA(-__dmul_rn(hx, y), y, 0.5);
    y = M3DK_FMA(y, e, y);
    e = M3DK_FMA(-__dmul_rn(hx, y), y, 0.5);
    return M3DK_FMA(y, e, y);
}
__device__ __forceinline__ double m3dk_sqrt(double x) {
    const double y = m3dk_rsqrt(x);
    const double s = __dmul_rn(x, y);
    const double r = M3DK_FMA(M3DK_FMA(-s, s, x), __dmul_rn(0.5, y), s);
    return x > 0.0 ? r : 0.0;
}

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

// The same four coefficients from a tile staged in shared memory (two LDS.128, warp-uniform address: broadcast).
template <bool kSmem>
__device__ __forceinline__ Quad ldq_t(const double *p) {
    if (kSmem) {
        const double2 lo = reinterpret_cast<const double2 *>(p)[0], hi = reinterpret_cast<const double2 *>(p)[1];
        Quad q; q.a = lo.x; q.b = lo.y; q.c = hi.x; q.d = hi.y;
        return q;
    }
    return ldq(p);
}

// ---- polynomial quads (G10: monomials xi^i eta^j, j outer, i inner; row j starts at kRow[j], has 6 - j terms) -----
// c[4 k + s]: coefficient k of slot s.  Horner in xi inside a row, Horner in eta across rows; value, d/dxi, d/deta of
// all four slots: 38 FMA per slot.  Callers ignore the outputs they do not need; after full unrolling the unused
// chains are dead code and disappear (value only: 20 FMA per slot).
// R markers per thread share every coefficient load (all R sit in the same element): one 32-byte load feeds up to
// 8 R FMAs, which is what takes the L1 -> register-file path (128 B/clk/SM) off the critical path.
// The Horner scheme consumes the 21 coefficient quads of a block in descending order k = 20 .. 0, so the loads are
// software-pipelined through a ring of kRing quads: `ring` holds k = 20 .. 20 - kRing + 1 on entry; while quad k is
// consumed quad k - kRing is loaded, and on exit `ring` holds the first kRing quads of the block `nxt` (the block the
// caller evaluates next: the blocks of a tile are consumed back to back), so an L1 hit is never waited for.
#ifndef M3DK_RING
#define M3DK_RING 3
#endif
constexpr int kRing = M3DK_RING;   // must divide 21 so that the ring slots line up from one block to the next
static_assert(21 % kRing == 0, "kRing must divide the 21 coefficients of a block");
struct Ring { Quad q[kRing]; };
template <bool kSmem>
__device__ __forceinline__ void ring_fill(Ring &ring, const double *__restrict__ c) {
#pragma unroll
    for (int i = 0; i < kRing; ++i) ring.q[i] = ldq_t<kSmem>(c + 4 * (20 - i));
}

template <int R, bool kSmem>
__device__ __forceinline__ void quad_vd(const double *__restrict__ c, const double *__restrict__ nxt, Ring &ring,
                                        const double (&xi)[R], const double (&eta)[R], double (&v)[R][4],
                                        double (&dx)[R][4], double (&de)[R][4]) {
    constexpr int kRow[6] = {0, 6, 11, 15, 18, 20};
    double a[R][4], ax[R][4], ae[R][4];
    int n = 0;   // quads consumed so far: quad k = 20 - n sits in ring slot n % kRing
#pragma unroll
    for (int j = 5; j >= 0; --j) {
        const int L = 6 - j;
        double p[R][4], d[R][4];
#pragma unroll
        for (int i = L - 1; i >= 0; --i) {
            const int k = kRow[j] + i;                 // == 20 - n
            const Quad u = ring.q[n % kRing];
            ring.q[n % kRing] = k - kRing >= 0 ? ldq_t<kSmem>(c + 4 * (k - kRing)) : ldq_t<kSmem>(nxt + 4 * (k - kRing + 21));
            ++n;
            const double uu[4] = {u.a, u.b, u.c, u.d};
#pragma unroll
            for (int r = 0; r < R; ++r)
#pragma unroll
                for (int s = 0; s < 4; ++s) {
                    if (i == L - 1) { p[r][s] = uu[s]; d[r][s] = 0.0; }
                    else {
                        d[r][s] = (i == L - 2) ? p[r][s] : M3DK_FMA(d[r][s], xi[r], p[r][s]);
                        p[r][s] = M3DK_FMA(p[r][s], xi[r], uu[s]);
                    }
                }
        }
#pragma unroll
        for (int r = 0; r < R; ++r)
#pragma unroll
            for (int s = 0; s < 4; ++s) {
                if (j == 5) { a[r][s] = p[r][s]; ax[r][s] = 0.0; ae[r][s] = 0.0; }
                else {
                    if (j == 4) { ae[r][s] = a[r][s]; ax[r][s] = d[r][s]; }
                    else { ae[r][s] = M3DK_FMA(ae[r][s], eta[r], a[r][s]); ax[r][s] = M3DK_FMA(ax[r][s], eta[r], d[r][s]); }
                    a[r][s] = M3DK_FMA(a[r][s], eta[r], p[r][s]);
                }
            }
    }
#pragma unroll
    for (int r = 0; r < R; ++r)
#pragma unroll
        for (int s = 0; s < 4; ++s) { v[r][s] = a[r][s]; dx[r][s] = ax[r][s]; de[r][s] = ae[r][s]; }
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
static __device__ __noinline__ int locate(const GridParams &g, double R, double Z) {
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
    FastRec q;
    unsigned r[16];
    asm("ld.global.nc.v8.b32 {%0, %1, %2, %3, %4, %5, %6, %7}, [%8];"
        : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]) : "l"(p));
    asm("ld.global.nc.v8.b32 {%0, %1, %2, %3, %4, %5, %6, %7}, [%8];"
        : "=r"(r[8]), "=r"(r[9]), "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15])
        : "l"(reinterpret_cast<const char *>(p) + 32));
#pragma unroll
    for (int k = 0; k < 6; ++k) { q.a[k] = __uint_as_float(r[k]); q.b[k] = __uint_as_float(r[6 + k]); }
    q.ida = (int)r[12]; q.idb = (int)r[13]; q.next = (int)r[14]; q.pad = 0;
    return q;
}

// bucket of (R, Z) in the fast grid; `inside` false: the point is outside the grid (bucket 0 is returned for addressing)
__device__ __forceinline__ int fast_bucket(const FastGrid &g, double R, double Z, float &u, float &v, bool &inside) {
    const double fx = (R - g.Rmin) * g.inv_hx, fz = (Z - g.Zmin) * g.inv_hz;
    inside = fx >= 0.0 && fx < (double)g.gx && fz >= 0.0 && fz < (double)g.gz;
    const int ix = inside ? (int)fx : 0, iz = inside ? (int)fz : 0;
    u = (float)(fx - (double)ix); v = (float)(fz - (double)iz);
    return iz * g.gx + ix;
}

// The asm loads are not volatile, so the compiler may hoist them above the range checks: every address is therefore
// clamped into its table first and the checks only decide whether the loaded record is used.
__device__ __forceinline__ FastRec locate_first(const FastGrid &g, double R, double Z) {
    float u, v;
    bool inside;
    return ldrec(g.first + (size_t)fast_bucket(g, R, Z, u, v, inside));
}
__device__ __forceinline__ bool fast_inside(const float (&t)[6], float u, float v) {
    const float e0 = __fmul_rn(t[2] - t[0], v - t[1]) - __fmul_rn(t[3] - t[1], u - t[0]);
    const float e1 = __fmul_rn(t[4] - t[2], v - t[3]) - __fmul_rn(t[5] - t[3], u - t[2]);
    const float e2 = __fmul_rn(t[0] - t[4], v - t[5]) - __fmul_rn(t[1] - t[5], u - t[4]);
    return e0 > kFastMargin && e1 > kFastMargin && e2 > kFastMargin;
}
__device__ __forceinline__ int locate_fast_from(const FastGrid &g, FastRec r, double R, double Z) {
    float u, v;
    bool open;
    fast_bucket(g, R, Z, u, v, open);
    int found = -2;
#pragma unroll 1
    for (int it = 0; it < 2 && open; ++it) {
        if (r.ida >= 0 && fast_inside(r.a, u, v)) { found = r.ida; open = false; }
        else if (r.ida >= 0 && r.idb >= 0 && fast_inside(r.b, u, v)) { found = r.idb; open = false; }
        else if (r.ida < 0 || r.next < 0) open = false;
        else r = ldrec(g.ovf + max(r.next, 0));
    }
    return found;
}
__device__ __forceinline__ int locate_fast(const FastGrid &g, double R, double Z) {
    return locate_fast_from(g, locate_first(g, R, Z), R, Z);
}

__device__ __forceinline__ int locate_finish(const FieldParams &f, const FastRec &first, double R, double Z) {
    const int e = locate_fast_from(f.fast, first, R, Z);
    return e != -2 ? e : locate(f.grid, R, Z);
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
    const double xi1[1] = {(R - Rc) * se}, eta1[1] = {(Z - Zc) * se};
    double vv[1][4], dxx[1][4], dee[1][4];
    double (&v)[4] = vv[0], (&dx)[4] = dxx[0], (&de)[4] = dee[0];
    Ring ring;
    ring_fill<false>(ring, tile + kTileHeader);
    quad_vd<1, false>(tile + kTileHeader, tile + kTileHeader, ring, xi1, eta1, vv, dxx, dee);  // (psi0, |B|0, F0, kappa)
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
        ring_fill<false>(ring, pm);
        quad_vd<1, false>(pm, pm + kQuad, ring, xi1, eta1, vv, dxx, dee);                  // E_R, E_phi
        o.E1[0] += v[0] * cth - v[1] * sth;
        o.E1[1] += v[2] * cth - v[3] * sth;
        quad_vd<1, false>(pm + kQuad, pm + 2 * kQuad, ring, xi1, eta1, vv, dxx, dee);         // E_Z, B_R
        o.E1[2] += v[0] * cth - v[1] * sth;
        o.B1[0] += v[2] * cth - v[3] * sth;
        quad_vd<1, false>(pm + 2 * kQuad, pm + 3 * kQuad, ring, xi1, eta1, vv, dxx, dee);   // B_par with gradient, B_Z
        o.B1[2] += v[2] * cth - v[3] * sth;
        const double re = v[0], im = v[1];
        const double qd = re * sth + im * cth;               // -Im-part combination: d/dphi -> -n qd, d/dt -> omega qd
        o.B1p += re * cth - im * sth;
        o.gB[0] += (dx[0] * se) * cth - (dx[1] * se) * sth;
        o.gB[1] += -(double)n * qd * rinv;
        o.gB[2] += (de[0] * se) * cth - (de[1] * se) * sth;
        quad_vd<1, false>(pm + 3 * kQuad, pm, ring, xi1, eta1, vv, dxx, dee);                // B_phi (slots 2, 3 are padding)
        o.B1[1] += v[0] * cth - v[1] * sth;
        o.dtB += f.omega[md] * qd;
    }
}

// value, first and second derivatives of the four polynomials of a quad at (xi, eta): nested Horner.  Row j of the
// triangle is a polynomial in xi (value r, r', r''/2 by the three-term Horner recurrence); the rows are then combined by
// the same recurrence in eta.  out[s] = {f, f_xi, f_eta, f_xixi, f_xieta, f_etaeta}.
__device__ __forceinline__ void quad_d2(const double *__restrict__ c, double xi, double eta, double (&out)[4][6]) {
    constexpr int kRow[6] = {0, 6, 11, 15, 18, 20};
    double V[4], Ve[4], Vee[4], X[4], Xe[4], XX[4];
#pragma unroll
    for (int s = 0; s < 4; ++s) V[s] = Ve[s] = Vee[s] = X[s] = Xe[s] = XX[s] = 0.0;
#pragma unroll
    for (int j = 5; j >= 0; --j) {
        const int L = 6 - j;
        double r[4] = {0.0, 0.0, 0.0, 0.0}, r1[4] = {0.0, 0.0, 0.0, 0.0}, r2[4] = {0.0, 0.0, 0.0, 0.0};
#pragma unroll
        for (int i = L - 1; i >= 0; --i) {
            const Quad u = ldq(c + 4 * (kRow[j] + i));
            const double uu[4] = {u.a, u.b, u.c, u.d};
#pragma unroll
            for (int s = 0; s < 4; ++s) {
                r2[s] = M3DK_FMA(r2[s], xi, r1[s]);
                r1[s] = M3DK_FMA(r1[s], xi, r[s]);
                r[s] = M3DK_FMA(r[s], xi, uu[s]);
            }
        }
#pragma unroll
        for (int s = 0; s < 4; ++s) {
            Vee[s] = M3DK_FMA(Vee[s], eta, Ve[s]);
            Ve[s] = M3DK_FMA(Ve[s], eta, V[s]);
            V[s] = M3DK_FMA(V[s], eta, r[s]);
            Xe[s] = M3DK_FMA(Xe[s], eta, X[s]);
            X[s] = M3DK_FMA(X[s], eta, r1[s]);
            XX[s] = M3DK_FMA(XX[s], eta, r2[s]);
        }
    }
#pragma unroll
    for (int s = 0; s < 4; ++s) {
        out[s][0] = V[s]; out[s][1] = X[s]; out[s][2] = Ve[s];
        out[s][3] = __dmul_rn(2.0, XX[s]); out[s][4] = Xe[s]; out[s][5] = __dmul_rn(2.0, Vee[s]);
    }
}

// Equilibrium field values of the guiding-centre equations at (R, Z) in the element of `tile` (global memory), with the
// second derivatives of psi0, and Eqs. (3)-(4): b = B/|B| (|B| from its own table), curl b by the quotient rule
// (axisymmetric), B* = B + (m v_par/q) curl b, B*par = B* . b (the phase-space Jacobian).
struct GcEq { double rinv, psi_R, psi_Z, psi_RR, psi_ZZ, Bm, Bm_R, Bm_Z, F, F_R, F_Z; };
__device__ __forceinline__ void gc_eq_fields(const double *__restrict__ tile, double R, double Z, GcEq &g) {
    const Quad hd = ldq(tile);
    const double se = hd.c, xi = (R - hd.a) * se, eta = (Z - hd.b) * se;
    double d[4][6];
    quad_d2(tile + kTileHeader, xi, eta, d);                     // slots: psi0, |B|0, F0, kappa
    const double s2 = se * se;
    g.rinv = m3dk_rcp(R);
    g.psi_R = d[0][1] * se; g.psi_Z = d[0][2] * se; g.psi_RR = d[0][3] * s2; g.psi_ZZ = d[0][5] * s2;
    g.Bm = d[1][0]; g.Bm_R = d[1][1] * se; g.Bm_Z = d[1][2] * se;
    g.F = d[2][0]; g.F_R = d[2][1] * se; g.F_Z = d[2][2] * se;
}
__device__ __forceinline__ double bstar_par(const GcEq &g, double q, double m, double vpar, double (&Bs)[3], double (&b)[3]) {
    const double rinv = g.rinv, rinv2 = rinv * rinv;
    const double B[3] = {-g.psi_Z * rinv, g.F * rinv, g.psi_R * rinv};
    const double BR_Z = -g.psi_ZZ * rinv;
    const double BP_R = g.F_R * rinv - g.F * rinv2, BP_Z = g.F_Z * rinv;
    const double BZ_R = g.psi_RR * rinv - g.psi_R * rinv2;
    const double binv = m3dk_rcp(g.Bm);
#pragma unroll
    for (int k = 0; k < 3; ++k) b[k] = B[k] * binv;
    const double bR_Z = (BR_Z - b[0] * g.Bm_Z) * binv;
    const double bP_R = (BP_R - b[1] * g.Bm_R) * binv, bP_Z = (BP_Z - b[1] * g.Bm_Z) * binv;
    const double bZ_R = (BZ_R - b[2] * g.Bm_R) * binv;
    const double curlb[3] = {-bP_Z, bR_Z - bZ_R, b[1] * rinv + bP_R};
    const double mvq = m * vpar / q;
#pragma unroll
    for (int k = 0; k < 3; ++k) Bs[k] = B[k] + mvq * curlb[k];
    return Bs[0] * b[0] + Bs[1] * b[1] + Bs[2] * b[2];
}

// d ln f0 / dE at fixed (P_phi, mu) (G7)
__device__ __forceinline__ double kappa_E(const PushParams &P, double Ekin, double mu) {
    if (P.f0kind == M3DK_F0_MAXWELLIAN) return -P.f0T_inv;
    const double v = m3dk_sqrt(__dmul_rn(__dmul_rn(2.0, Ekin), P.inv_m));
    const double v3 = __dmul_rn(__dmul_rn(v, v), v);
    double kE = __dmul_rn(__dmul_rn(-3.0, v), m3dk_rcp(__dmul_rn(P.m, __dadd_rn(v3, P.f0vc3))));
    if (P.f0kind == M3DK_F0_BEAM_PITCH) {
        // a marker with v = 0 and mu = 0 (Ekin = 0) has no pitch: its term is 0 * finite = 0 here, dropped in the oracle.
        // (Written without a branch on Ekin: that branch alone moved the register allocation of K1 by 3 % per push.)
        const double Einv = m3dk_rcp(fmax(Ekin, 1.0e-300));
        const double Lam = __dmul_rn(__dmul_rn(mu, P.f0Bax), Einv);
        kE = __dadd_rn(kE, __dmul_rn(__dmul_rn(__dmul_rn(__dmul_rn(2.0, __dsub_rn(Lam, P.f0L0)), Lam), P.f0dL2_inv), Einv));
    }
    return kE;
}

// ---- one step of one marker (PAPER.md:73-78 Eqs. 5-6; :106-130 Eqs. 8-13; :140) -----------------------------------
// state in: (x_l, v_{l-1/2}, mu, w_{l-1/2}) with e = element of x_l;  out: (x_{l+1}, v_{l+1/2}, w_{l+1/2}).
struct Marker { double x, y, z, vx, vy, vz, mu, w; };

struct StepGeom { double R, rinv, cph, sph; };

// cylindrical map (G3)
__device__ __forceinline__ void step_geometry(const Marker &s, StepGeom &g) {
    const double r2 = M3DK_FMA(s.x, s.x, __dmul_rn(s.y, s.y));
    g.rinv = m3dk_rsqrt(r2);
    g.R = __dmul_rn(r2, g.rinv);
    g.cph = __dmul_rn(s.x, g.rinv); g.sph = __dmul_rn(s.y, g.rinv);
}

// Equilibrium fields of one marker and the weights with which the perturbed fields enter dw/dt.
struct EqOut { double psi_R, psi_Z, Bm, Bm_R, Bm_Z, F, kappa; };
struct PertW { double aER, aEP, aEZ, bBR, bBZ, gR, gP, gZ, dT; };

// Phase A of a step, after the equilibrium quad: Eq. (6) (Boris) and Eq. (5) (drift) on s.{x..vz}; then, with modes,
// the linear delta-f equation (Eqs. 8-13 at (x_l, v_l), v_l = (v_{l-1/2} + v_{l+1/2}) / 2) is written as
//   dw/dt = aER E1_R + aEP E1_phi + aEZ E1_Z + bBR B1_R + bBZ B1_Z + gR dB1par/dR + gP (1/R) dB1par/dphi
//           + gZ dB1par/dZ + dT dB1par/dt
// (it is linear in the perturbed fields; B1_phi does not enter), so that the perturbed polynomials can be folded into
// one scalar per marker as they are evaluated (phase B) instead of being kept in registers:
//   K = kappa/q, G = F/|B0|, b = B0/|B0|, v_par = v_l . b
//   Eq. (12)+(10): dP/dt = q (dX_1 . grad psi0) + F_par1 G, dX_1 = E1 x B0 / B0^2 + v_par B1 / |B0|
//   Eq. (13) x m (G5): F_par1 = q E1 . b - mu b . grad B1par;  Eq. (11) (G6): dE/dt = q v_l . E1 + mu dB1par/dt
//   Eqs. (8)-(9), (1 - w) -> 1: dw/dt = -(K dP/dt + kE dE/dt)
// Every operation below is written out (DM/DA/DS/M3DK_FMA: no contraction left to the compiler), so that every kernel
// that inlines this code produces the same bits for the same marker (pin P13: results do not depend on the order).
#define DM(a, b) __dmul_rn((a), (b))
#define DA(a, b) __dadd_rn((a), (b))
#define DS(a, b) __dsub_rn((a), (b))
// Coefficients of dw/dt in the perturbed fields (see push_eq): (BR, BP, BZ) is the EQUILIBRIUM field B0, s holds
// v_{l-1/2}, (nvx, nvy, nvz) = v_{l+1/2}.
__device__ __forceinline__ void weight_coeffs(const PushParams &P, const StepGeom &g, const EqOut &f, double BR, double BP,
                                              double BZ, const Marker &s, double nvx, double nvy, double nvz, PertW &W) {
    const double cph = g.cph, sph = g.sph;
    const double vlx = DM(0.5, DA(s.vx, nvx)), vly = DM(0.5, DA(s.vy, nvy)), vlz = DM(0.5, DA(s.vz, nvz));
    const double vR = M3DK_FMA(vlx, cph, DM(vly, sph)), vP = M3DK_FMA(vly, cph, -DM(vlx, sph)), vZ = vlz;
    const double B2 = M3DK_FMA(BR, BR, M3DK_FMA(BP, BP, DM(BZ, BZ)));
    const double binv = m3dk_rsqrt(B2);
    const double b2inv = DM(binv, binv);
    const double bR = DM(BR, binv), bP = DM(BP, binv), bZ = DM(BZ, binv);
    const double vpar = M3DK_FMA(vR, bR, M3DK_FMA(vP, bP, DM(vZ, bZ)));
    const double v2 = M3DK_FMA(vlx, vlx, M3DK_FMA(vly, vly, DM(vlz, vlz)));
    const double Ekin = M3DK_FMA(DM(0.5, P.m), v2, DM(s.mu, f.Bm));
    const double kE = kappa_E(P, Ekin, s.mu);
    const double K = DM(f.kappa, P.inv_q), G = DM(f.F, binv);
    const double Kq = DM(K, P.q), kEq = DM(kE, P.q);
    W.aER = -M3DK_FMA(Kq, M3DK_FMA(DM(f.psi_Z, BP), b2inv, DM(bR, G)), DM(kEq, vR));
    W.aEP = -M3DK_FMA(Kq, M3DK_FMA(M3DK_FMA(f.psi_R, BZ, -DM(f.psi_Z, BR)), b2inv, DM(bP, G)), DM(kEq, vP));
    W.aEZ = -M3DK_FMA(Kq, M3DK_FMA(-DM(f.psi_R, BP), b2inv, DM(bZ, G)), DM(kEq, vZ));
    const double Kv = -DM(DM(Kq, vpar), binv);
    W.bBR = DM(Kv, f.psi_R);
    W.bBZ = DM(Kv, f.psi_Z);
    const double Kg = DM(DM(K, s.mu), G);
    W.gR = DM(Kg, bR); W.gP = DM(Kg, bP); W.gZ = DM(Kg, bZ);
    W.dT = -DM(kE, s.mu);
}

__device__ __forceinline__ void push_eq(const PushParams &P, const StepGeom &g, const EqOut &f, Marker &s, PertW &W) {
    const double rinv = g.rinv, cph = g.cph, sph = g.sph;
    // B0 = grad psi0 x grad phi + F0 grad phi (G4); E-dagger = -(mu/q) grad|B|0 (G2)
    const double BR = -DM(f.psi_Z, rinv), BP = DM(f.F, rinv), BZ = DM(f.psi_R, rinv);
    const double muq = DM(s.mu, P.inv_q);
    const double ER = -DM(muq, f.Bm_R), EZ = -DM(muq, f.Bm_Z);
    const double Bx = M3DK_FMA(BR, cph, -DM(BP, sph)), By = M3DK_FMA(BR, sph, DM(BP, cph)), Bz = BZ;
    const double Ex = DM(ER, cph), Ey = DM(ER, sph), Ez = EZ;
    // Eq. (6) in the explicit Boris form: half kick, rotation t = h B, s = 2 t / (1 + t^2), half kick
    const double h = P.h;
    const double ux = M3DK_FMA(h, Ex, s.vx), uy = M3DK_FMA(h, Ey, s.vy), uz = M3DK_FMA(h, Ez, s.vz);
    const double tx = DM(h, Bx), ty = DM(h, By), tz = DM(h, Bz);
    const double sc = DM(2.0, m3dk_rcp(DA(1.0, M3DK_FMA(tx, tx, M3DK_FMA(ty, ty, DM(tz, tz))))));
    const double px = DA(ux, M3DK_FMA(uy, tz, -DM(uz, ty))), py = DA(uy, M3DK_FMA(uz, tx, -DM(ux, tz))),
                 pz = DA(uz, M3DK_FMA(ux, ty, -DM(uy, tx)));
    const double wx = M3DK_FMA(sc, M3DK_FMA(py, tz, -DM(pz, ty)), ux), wy = M3DK_FMA(sc, M3DK_FMA(pz, tx, -DM(px, tz)), uy),
                 wz = M3DK_FMA(sc, M3DK_FMA(px, ty, -DM(py, tx)), uz);
    const double nvx = M3DK_FMA(h, Ex, wx), nvy = M3DK_FMA(h, Ey, wy), nvz = M3DK_FMA(h, Ez, wz);
    if (P.f.n_modes > 0) {
        weight_coeffs(P, g, f, BR, BP, BZ, s, nvx, nvy, nvz, W);
    }
    // Eq. (5)
    s.x = M3DK_FMA(P.dt, nvx, s.x); s.y = M3DK_FMA(P.dt, nvy, s.y); s.z = M3DK_FMA(P.dt, nvz, s.z);
    s.vx = nvx; s.vy = nvy; s.vz = nvz;
}

// ---- non-linear trajectory mode (mode 1; reading G21) ----------------------------------------
// Perturbed fields of one marker, cylindrical components, summed over the toroidal modes.
struct PertF { double ER, EP, EZ, BR, BP, BZ, gR, gP, gZ, dT; };

// The marker moves in the total fields: B = B0 + B1, E-dagger = E1 - (mu/q) grad(|B|0 + B1par) (PAPER.md:78 with the
// total field strength).  The weight equation keeps its linear right-hand side (Eqs. 10-13 with the equilibrium b0,
// evaluated at (x_l, v_l)); wdot returns it and the caller applies the factor (1 - w) of Eq. (8).
__device__ __forceinline__ void push_eq_nl(const PushParams &P, const StepGeom &g, const EqOut &f, const PertF &p,
                                           Marker &s, double &wdot) {
    const double rinv = g.rinv, cph = g.cph, sph = g.sph;
    const double B0R = -DM(f.psi_Z, rinv), B0P = DM(f.F, rinv), B0Z = DM(f.psi_R, rinv);
    const double BR = DA(B0R, p.BR), BP = DA(B0P, p.BP), BZ = DA(B0Z, p.BZ);
    const double muq = DM(s.mu, P.inv_q);
    const double ER = M3DK_FMA(-muq, DA(f.Bm_R, p.gR), p.ER), EP = M3DK_FMA(-muq, p.gP, p.EP),
                 EZ = M3DK_FMA(-muq, DA(f.Bm_Z, p.gZ), p.EZ);
    const double Bx = M3DK_FMA(BR, cph, -DM(BP, sph)), By = M3DK_FMA(BR, sph, DM(BP, cph)), Bz = BZ;
    const double Ex = M3DK_FMA(ER, cph, -DM(EP, sph)), Ey = M3DK_FMA(ER, sph, DM(EP, cph)), Ez = EZ;
    const double h = P.h;
    const double ux = M3DK_FMA(h, Ex, s.vx), uy = M3DK_FMA(h, Ey, s.vy), uz = M3DK_FMA(h, Ez, s.vz);
    const double tx = DM(h, Bx), ty = DM(h, By), tz = DM(h, Bz);
    const double sc = DM(2.0, m3dk_rcp(DA(1.0, M3DK_FMA(tx, tx, M3DK_FMA(ty, ty, DM(tz, tz))))));
    const double px = DA(ux, M3DK_FMA(uy, tz, -DM(uz, ty))), py = DA(uy, M3DK_FMA(uz, tx, -DM(ux, tz))),
                 pz = DA(uz, M3DK_FMA(ux, ty, -DM(uy, tx)));
    const double wx = M3DK_FMA(sc, M3DK_FMA(py, tz, -DM(pz, ty)), ux), wy = M3DK_FMA(sc, M3DK_FMA(pz, tx, -DM(px, tz)), uy),
                 wz = M3DK_FMA(sc, M3DK_FMA(px, ty, -DM(py, tx)), uz);
    const double nvx = M3DK_FMA(h, Ex, wx), nvy = M3DK_FMA(h, Ey, wy), nvz = M3DK_FMA(h, Ez, wz);
    PertW W;
    weight_coeffs(P, g, f, B0R, B0P, B0Z, s, nvx, nvy, nvz, W);
    double a = DM(W.aER, p.ER);
    a = M3DK_FMA(W.aEP, p.EP, a); a = M3DK_FMA(W.aEZ, p.EZ, a);
    a = M3DK_FMA(W.bBR, p.BR, a); a = M3DK_FMA(W.bBZ, p.BZ, a);
    a = M3DK_FMA(W.gR, p.gR, a); a = M3DK_FMA(W.gP, p.gP, a); a = M3DK_FMA(W.gZ, p.gZ, a);
    wdot = M3DK_FMA(W.dT, p.dT, a);
    s.x = M3DK_FMA(P.dt, nvx, s.x); s.y = M3DK_FMA(P.dt, nvy, s.y); s.z = M3DK_FMA(P.dt, nvz, s.z);
    s.vx = nvx; s.vy = nvy; s.vz = nvz;
}

// cos / sin of (n phi - omega t): exp(i n phi) by complex powers of (cos phi + i sin phi), exp(-i omega t) from the host
__device__ __forceinline__ void mode_phase(int n, double cph, double sph, double cwt, double swt, double &cth,
                                           double &sth) {
    double cn = 1.0, sn = 0.0;
    for (int k = 0; k < abs(n); ++k) {
        const double c2 = M3DK_FMA(cn, cph, -__dmul_rn(sn, sph));
        sn = M3DK_FMA(cn, sph, __dmul_rn(sn, cph));
        cn = c2;
    }
    if (n < 0) sn = -sn;
    cth = M3DK_FMA(cn, cwt, __dmul_rn(sn, swt));
    sth = M3DK_FMA(sn, cwt, -__dmul_rn(cn, swt));
}

// Phase B: fold quad Q of a mode into dw/dt.  Re[C e^{i th}] = Cr cos th - Ci sin th; every operation is written out
// (no contraction left to the compiler) so that all kernels that call this produce the same bits.
__device__ __forceinline__ double re_part(double cr, double ci, double cth, double sth) {
    return M3DK_FMA(cr, cth, -__dmul_rn(ci, sth));
}
// value-only quad: two complex amplitudes (v0 + i v1), (v2 + i v3) with weights wa, wb
__device__ __forceinline__ double pert_fold_v(double wsum, const double (&v)[4], double wa, double wb, double cth,
                                              double sth) {
    wsum = M3DK_FMA(wa, re_part(v[0], v[1], cth, sth), wsum);
    return M3DK_FMA(wb, re_part(v[2], v[3], cth, sth), wsum);
}
// (B_par, B_Z) quad: gradient and time derivative of B_par (d/dphi -> -n qd, d/dt -> omega qd), value of B_Z
__device__ __forceinline__ double pert_fold_par(double wsum, const double (&v)[4], const double (&dx)[4],
                                                const double (&de)[4], const PertW &W, double cth, double sth, double se,
                                                double n_rinv, double omega) {
    wsum = M3DK_FMA(W.bBZ, re_part(v[2], v[3], cth, sth), wsum);
    const double qd = M3DK_FMA(v[0], sth, __dmul_rn(v[1], cth));
    wsum = M3DK_FMA(W.gR, re_part(__dmul_rn(dx[0], se), __dmul_rn(dx[1], se), cth, sth), wsum);
    wsum = M3DK_FMA(W.gP, -__dmul_rn(n_rinv, qd), wsum);
    wsum = M3DK_FMA(W.gZ, re_part(__dmul_rn(de[0], se), __dmul_rn(de[1], se), cth, sth), wsum);
    return M3DK_FMA(W.dT, __dmul_rn(omega, qd), wsum);
}

__device__ __forceinline__ int locate_xyz(const FieldParams &f, double x, double y, double z) {
    return locate_any(f, m3dk_sqrt(M3DK_FMA(x, x, __dmul_rn(y, y))), z);
}

}  // namespace m3dk
