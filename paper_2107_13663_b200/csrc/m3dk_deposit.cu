// m3dk_deposit.cu -- moment deposition: right-hand sides of the Galerkin projection of the pressure
// moments with a delta-function particle shape, Eqs. (17)-(18) (readings G10, G22):
//     rhs[e][0][h][k] = sum over markers p in element e of  w_p m v_par,p^2    nu_k(x_p) T_h(phi_p)
//     rhs[e][1][h][k] = sum over markers p in element e of  w_p mu_p |B|0(x_p) nu_k(x_p) T_h(phi_p)
// nu_k = xi^i eta^j (the element's own basis), T_0 = 1, T_{2m+1} = cos(n_m phi), T_{2m+2} = sin(n_m phi).
// One marker per lane; the lanes of a warp that sit in the same element are reduced with shuffles and their sum enters the
// table with ONE fp64 atomic per entry, so on an element-ordered marker stream (what m3dk_push leaves behind when
// sort_interval >= 1) a warp makes one or two passes and an element's 42 (1 + 2 n_modes) sums receive a few atomics each.
#include <math.h>

#include "m3dk_device.cuh"

namespace m3dk {

constexpr int kDepHarmMax = 1 + 2 * M3DK_MAX_MODES;

// contributions of one marker: amp[0] = w m v_par^2, amp[1] = w mu |B|0; T[h]; xp[i] = xi^i, ep[j] = eta^j
struct DepMarker { double amp[2], T[kDepHarmMax], xp[6], ep[6]; };

// options of one deposition: with_b1par adds mu B1par (Eq. 16) to the perpendicular moment; with_bstar replaces w by
// d = w + B1par / B*par in both moments (reading G25); cwt / swt = cos / sin(omega_k t); q = species charge
struct DepOpts { int with_b1par, with_bstar; double q; double cwt[M3DK_MAX_MODES], swt[M3DK_MAX_MODES]; };

// kF: bit 0 = with_b1par, bit 1 = with_bstar, as compile-time constants (the second-derivative scheme of B*par costs
// 80 registers, which the plain deposition must not pay for)
template <int kF>
__device__ __forceinline__ void dep_marker(const FieldParams &f, const DepOpts &o, int e, const Marker &s, double mass,
                                           DepMarker &d) {
    constexpr bool kB1 = (kF & 1) != 0, kBs = (kF & 2) != 0;
    StepGeom g;
    step_geometry(s, g);
    // equilibrium quad at the marker: B0 = grad psi0 x grad phi + F0 grad phi (G4), |B|0 from its own table
    const double *tile = f.tiles + (size_t)max(e, 0) * f.tile_stride;     // clamped: the loads may be speculated
    const Quad hd = ldq(tile);
    const double se = hd.c;
    const double xi1[1] = {__dmul_rn(__dsub_rn(g.R, hd.a), se)}, eta1[1] = {__dmul_rn(__dsub_rn(s.z, hd.b), se)};
    double v[1][4], dx[1][4], de[1][4];
    Ring ring;
    ring_fill<false>(ring, tile + kTileHeader);
    quad_vd<1, false>(tile + kTileHeader, tile + kTileHeader, ring, xi1, eta1, v, dx, de);
    const double BR = -__dmul_rn(__dmul_rn(de[0][0], se), g.rinv), BP = __dmul_rn(v[0][2], g.rinv),
                 BZ = __dmul_rn(__dmul_rn(dx[0][0], se), g.rinv);
    const double binv = m3dk_rsqrt(M3DK_FMA(BR, BR, M3DK_FMA(BP, BP, __dmul_rn(BZ, BZ))));
    const double vR = M3DK_FMA(s.vx, g.cph, __dmul_rn(s.vy, g.sph)), vP = M3DK_FMA(s.vy, g.cph, -__dmul_rn(s.vx, g.sph));
    const double vpar = __dmul_rn(M3DK_FMA(vR, BR, M3DK_FMA(vP, BP, __dmul_rn(s.vz, BZ))), binv);
    double b1p = 0.0;     // B1par = Re[C e^{i(n phi - omega t)}] from quad 2 of every mode
    if (kB1 || kBs) {
        const double Bm0 = v[0][1];
        for (int md = 0; md < f.n_modes; ++md) {
            double cth, sth;
            mode_phase(f.n_tor[md], g.cph, g.sph, o.cwt[md], o.swt[md], cth, sth);
            const double *pm = tile + kTileHeader + kTileEq + kTileMode * md + 2 * kQuad;
            ring_fill<false>(ring, pm);
            quad_vd<1, false>(pm, pm, ring, xi1, eta1, v, dx, de);
            b1p = __dadd_rn(b1p, re_part(v[0][0], v[0][1], cth, sth));
        }
        v[0][1] = Bm0;
    }
    double dd = s.w;
    if (kBs) {   // d = w + B1* / B* with B1* -> B1par and B* = B*par of Eq. (4) at this marker's v_par
        GcEq ge;
        gc_eq_fields(tile, g.R, s.z, ge);
        double Bs[3], bb[3];
        dd = __dadd_rn(dd, __dmul_rn(b1p, m3dk_rcp(bstar_par(ge, o.q, mass, vpar, Bs, bb))));
    }
    d.amp[0] = __dmul_rn(__dmul_rn(dd, mass), __dmul_rn(vpar, vpar));
    d.amp[1] = __dmul_rn(__dmul_rn(dd, s.mu), v[0][1]);
    if (kB1) d.amp[1] = M3DK_FMA(s.mu, b1p, d.amp[1]);   // Eq. (16): mu |B|0 (w + B1par/|B|0)
    d.T[0] = 1.0;     // toroidal factors by complex powers of (cos phi + i sin phi)
#pragma unroll
    for (int md = 0; md < M3DK_MAX_MODES; ++md)
        if (md < f.n_modes) mode_phase(f.n_tor[md], g.cph, g.sph, 1.0, 0.0, d.T[1 + 2 * md], d.T[2 + 2 * md]);
    d.xp[0] = 1.0; d.ep[0] = 1.0;
#pragma unroll
    for (int q = 1; q < 6; ++q) { d.xp[q] = __dmul_rn(d.xp[q - 1], xi1[0]); d.ep[q] = __dmul_rn(d.ep[q - 1], eta1[0]); }
}


// Sums over the warp of N values per lane by a transposing butterfly: every exchange halves the number of values a lane
// holds (N/2 + N/4 + .. + 1 shuffles, then one per remaining lane bit), instead of five shuffles per value.  On return
// lane L holds the total of value (L >> log2(32 / N)) & (N - 1); lanes that share those bits hold the same total.
template <int N>
__device__ __forceinline__ double warp_sum_columns(double (&v)[N], int lane) {
    static_assert(N == 8 || N == 16 || N == 32, "N values per lane, a power of two");
    int s = 16;
#pragma unroll
    for (int cnt = N; cnt > 1; cnt >>= 1, s >>= 1) {
        const bool up = (lane & s) != 0;
#pragma unroll
        for (int i = 0; i < cnt / 2; ++i) {
            const double send = up ? v[i] : v[i + cnt / 2];
            const double keep = up ? v[i + cnt / 2] : v[i];
            v[i] = keep + __shfl_xor_sync(0xffffffffu, send, s);
        }
    }
    double t = v[0];
#pragma unroll
    for (; s > 0; s >>= 1) t += __shfl_xor_sync(0xffffffffu, t, s);
    return t;
}

// One row (moment, harmonic) of an item's table update: the 21 entries k = (i, j) of o[] each receive the sum over the
// warp's markers of val(i, j).  Entries 0..15 and 16..20 (padded to 8) are reduced by warp_sum_columns (16 + 9 shuffles of
// a double for the row against 105 for a butterfly per entry); the totals end up one per lane, so the table is updated by
// two atomic instructions per row (16 and 5 active lanes).
template <class F>
__device__ __forceinline__ void dep_row_add(double *__restrict__ o, int lane, F val) {
    double va[16], vb[8];
    int k = 0;
#pragma unroll
    for (int j = 0; j < 6; ++j)
#pragma unroll
        for (int ii = 0; ii < 6 - j; ++ii, ++k) {
            const double x = val(ii, j);
            if (k < 16) va[k] = x; else vb[k - 16] = x;
        }
    vb[5] = 0.0; vb[6] = 0.0; vb[7] = 0.0;
    const double ta = warp_sum_columns<16>(va, lane);       // lane L: entry L >> 1
    const double tb = warp_sum_columns<8>(vb, lane);        // lane L: entry 16 + (L >> 2)
    if ((lane & 1) == 0) atomicAdd(o + (lane >> 1), ta);
    if ((lane & 3) == 0 && (lane >> 2) < 5) atomicAdd(o + 16 + (lane >> 2), tb);
}

// any marker order: one marker per lane, the warp loops over its distinct elements
template <int kF>
__global__ void __launch_bounds__(128) deposit_kernel(const __grid_constant__ FieldParams f, const __grid_constant__ DepOpts o,
                                                      MarkerArrays a, long n, double mass, double *__restrict__ rhs) {
    const long i = (long)blockIdx.x * blockDim.x + threadIdx.x;
    const int lane = threadIdx.x & 31;
    const bool valid = i < n;
    const int e = valid ? a.elem[i] : -1;
    const bool active = e >= 0;                      // lost markers deposit nothing
    const int H = 1 + 2 * f.n_modes;
    Marker s;
    if (active) {
        s.x = a.x[i]; s.y = a.y[i]; s.z = a.z[i]; s.vx = a.vx[i]; s.vy = a.vy[i]; s.vz = a.vz[i]; s.mu = a.mu[i]; s.w = a.w[i];
    } else {
        s.x = 1.0; s.y = 0.0; s.z = 0.0; s.vx = s.vy = s.vz = 0.0; s.mu = 0.0; s.w = 0.0;
    }
    DepMarker d;
    dep_marker<kF>(f, o, e, s, mass, d);
    const size_t stride_e = (size_t)2 * H * M3DK_NCOEF;
    unsigned todo = __ballot_sync(0xffffffffu, active);
    while (todo) {
        const int ke = __shfl_sync(0xffffffffu, e, __ffs(todo) - 1);
        const bool mine = active && e == ke;
        double *out = rhs + (size_t)ke * stride_e;
        for (int mom = 0; mom < 2; ++mom)
#pragma unroll
            for (int h = 0; h < kDepHarmMax; ++h) {
                if (h >= H) break;
                const double ah = mine ? __dmul_rn(d.amp[mom], d.T[h]) : 0.0;
                double *o = out + ((size_t)mom * H + h) * M3DK_NCOEF;
                int k = 0;
#pragma unroll
                for (int j = 0; j < 6; ++j)
#pragma unroll
                    for (int ii = 0; ii < 6 - j; ++ii, ++k) {
                        double val = __dmul_rn(ah, __dmul_rn(d.xp[ii], d.ep[j]));
#pragma unroll
                        for (int sft = 16; sft > 0; sft >>= 1) val += __shfl_xor_sync(0xffffffffu, val, sft);
                        if (lane == 0) atomicAdd(o + k, val);
                    }
            }
        todo &= ~__ballot_sync(0xffffffffu, mine);
    }
}

// 4-point FLR deposition (flags bit 1): a marker deposits a quarter of its amplitudes at each of its four
// gyro-ring points (the ring of reading G23, as in the FLR push).  One marker per lane; for each of the four points the lane
// finds the point's element and the warp loops over its distinct elements exactly as deposit_kernel does.
// kRec: the markers are read from the element-ordered records of the sort workspace (a warp's 32 markers then share an
// element and their rings touch a handful of elements), else from the caller's arrays in whatever order they are.
template <bool kRec, int kF>
__global__ void __launch_bounds__(128) deposit_flr_kernel(const __grid_constant__ FieldParams f, const __grid_constant__ DepOpts o,
                                                          MarkerArrays a, const double *__restrict__ rec,
                                                          const int *__restrict__ key, long n, double q, double mass,
                                                          double *__restrict__ rhs) {
    const long i = (long)blockIdx.x * blockDim.x + threadIdx.x;
    const int lane = threadIdx.x & 31;
    const bool valid = i < n;
    int e = -1;
    if (valid) { e = kRec ? key[i] : a.elem[i]; if (kRec && e >= f.n_elems) e = -1; }
    const bool active = e >= 0;
    const int H = 1 + 2 * f.n_modes;
    Marker s;
    if (active && kRec) {
        const double *p = rec + (size_t)kRecDoubles * i;
        s.x = p[0]; s.y = p[1]; s.z = p[2]; s.w = p[3]; s.vx = p[4]; s.vy = p[5]; s.vz = p[6]; s.mu = p[7];
    } else if (active) {
        s.x = a.x[i]; s.y = a.y[i]; s.z = a.z[i]; s.vx = a.vx[i]; s.vy = a.vy[i]; s.vz = a.vz[i]; s.mu = a.mu[i]; s.w = a.w[i];
    } else {
        s.x = 1.0; s.y = 0.0; s.z = 0.0; s.vx = s.vy = s.vz = 0.0; s.mu = 0.0; s.w = 0.0;
    }
    DepMarker d;
    dep_marker<kF>(f, o, e, s, mass, d);          // amplitudes at the marker itself
    // the ring: same construction as flr_wdot of the push (reading G23)
    StepGeom g;
    step_geometry(s, g);
    const double *tile = f.tiles + (size_t)max(e, 0) * f.tile_stride;
    const Quad hd = ldq(tile);
    const double se0 = hd.c;
    const double xi1[1] = {__dmul_rn(__dsub_rn(g.R, hd.a), se0)}, eta1[1] = {__dmul_rn(__dsub_rn(s.z, hd.b), se0)};
    double v[1][4], dx[1][4], de[1][4];
    Ring ring;
    ring_fill<false>(ring, tile + kTileHeader);
    quad_vd<1, false>(tile + kTileHeader, tile + kTileHeader, ring, xi1, eta1, v, dx, de);
    const double BR = -__dmul_rn(__dmul_rn(de[0][0], se0), g.rinv), BP = __dmul_rn(v[0][2], g.rinv),
                 BZ = __dmul_rn(__dmul_rn(dx[0][0], se0), g.rinv);
    const double binv = m3dk_rsqrt(M3DK_FMA(BR, BR, M3DK_FMA(BP, BP, __dmul_rn(BZ, BZ))));
    const double bR = __dmul_rn(BR, binv), bP = __dmul_rn(BP, binv), bZ = __dmul_rn(BZ, binv);
    const double rho = __dmul_rn(m3dk_sqrt(__dmul_rn(__dmul_rn(__dmul_rn(2.0, mass), s.mu), binv)), fabs(1.0 / q));
    double e1R = M3DK_FMA(-bR, bR, 1.0), e1P = -__dmul_rn(bR, bP), e1Z = -__dmul_rn(bR, bZ);
    if (__dmul_rn(bR, bR) > 0.999999) {   // b (anti)parallel to R-hat: start from Z-hat instead (same rule as the oracle)
        e1R = -__dmul_rn(bZ, bR); e1P = -__dmul_rn(bZ, bP); e1Z = M3DK_FMA(-bZ, bZ, 1.0);
    }
    const double n1 = m3dk_rsqrt(M3DK_FMA(e1R, e1R, M3DK_FMA(e1P, e1P, __dmul_rn(e1Z, e1Z))));
    e1R = __dmul_rn(e1R, n1); e1P = __dmul_rn(e1P, n1); e1Z = __dmul_rn(e1Z, n1);
    const double e2R = M3DK_FMA(bP, e1Z, -__dmul_rn(bZ, e1P)), e2P = M3DK_FMA(bZ, e1R, -__dmul_rn(bR, e1Z)),
                 e2Z = M3DK_FMA(bR, e1P, -__dmul_rn(bP, e1R));
    const double c = g.cph, sn = g.sph;
    const double ex[2] = {M3DK_FMA(e1R, c, -__dmul_rn(e1P, sn)), M3DK_FMA(e2R, c, -__dmul_rn(e2P, sn))};
    const double ey[2] = {M3DK_FMA(e1R, sn, __dmul_rn(e1P, c)), M3DK_FMA(e2R, sn, __dmul_rn(e2P, c))};
    const double ez[2] = {e1Z, e2Z};
    const double X = __dmul_rn(g.R, c), Y = __dmul_rn(g.R, sn);
    const size_t stride_e = (size_t)2 * H * M3DK_NCOEF;
#pragma unroll 1
    for (int j = 0; j < 4; ++j) {
        const double sg = j < 2 ? rho : -rho;
        Marker sp;
        sp.x = M3DK_FMA(sg, ex[j & 1], X); sp.y = M3DK_FMA(sg, ey[j & 1], Y); sp.z = M3DK_FMA(sg, ez[j & 1], s.z);
        StepGeom gj;
        step_geometry(sp, gj);
        const int ej = active ? locate_any(f, gj.R, sp.z) : -1;
        const bool on = ej >= 0;
        const double *tj = f.tiles + (size_t)max(ej, 0) * f.tile_stride;
        const Quad hj = ldq(tj);
        const double xi = __dmul_rn(__dsub_rn(gj.R, hj.a), hj.c), eta = __dmul_rn(__dsub_rn(sp.z, hj.b), hj.c);
        double xp[6], ep[6], T[kDepHarmMax];
        xp[0] = 1.0; ep[0] = 1.0;
#pragma unroll
        for (int p = 1; p < 6; ++p) { xp[p] = __dmul_rn(xp[p - 1], xi); ep[p] = __dmul_rn(ep[p - 1], eta); }
        T[0] = 1.0;
#pragma unroll
        for (int md = 0; md < M3DK_MAX_MODES; ++md)
            if (md < f.n_modes) mode_phase(f.n_tor[md], gj.cph, gj.sph, 1.0, 0.0, T[1 + 2 * md], T[2 + 2 * md]);
        unsigned todo = __ballot_sync(0xffffffffu, on);
        while (todo) {
            const int ke = __shfl_sync(0xffffffffu, ej, __ffs(todo) - 1);
            const bool mine = on && ej == ke;
            double *out = rhs + (size_t)ke * stride_e;
            for (int mom = 0; mom < 2; ++mom)
#pragma unroll
                for (int h = 0; h < kDepHarmMax; ++h) {
                    if (h >= H) break;
                    const double ah = mine ? __dmul_rn(__dmul_rn(0.25, d.amp[mom]), T[h]) : 0.0;
                    double *op = out + ((size_t)mom * H + h) * M3DK_NCOEF;
                    int k = 0;
#pragma unroll
                    for (int jj = 0; jj < 6; ++jj)
#pragma unroll
                        for (int ii = 0; ii < 6 - jj; ++ii, ++k) {
                            double val = __dmul_rn(ah, __dmul_rn(xp[ii], ep[jj]));
#pragma unroll
                            for (int sft = 16; sft > 0; sft >>= 1) val += __shfl_xor_sync(0xffffffffu, val, sft);
                            if (lane == 0) atomicAdd(op + k, val);
                        }
                }
            todo &= ~__ballot_sync(0xffffffffu, mine);
        }
    }
}

// element-ordered records cut into work items (the ordering kernels of m3dk_sort.cu): a warp takes an item (<= 64
// markers of ONE element), every lane two of them, one reduction and one atomic per table entry and item
template <int kF>
__global__ void __launch_bounds__(128) deposit_items_kernel(const __grid_constant__ FieldParams f, const __grid_constant__ DepOpts o,
                                                            const double *__restrict__ rec,
                                                            const int4 *__restrict__ items, const int *__restrict__ n_items,
                                                            double mass, double *__restrict__ rhs) {
    const int lane = threadIdx.x & 31;
    const int it = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
    if (it >= *n_items) return;
    const int4 w = __ldg(items + it);
    const int e = w.x, start = w.y, count = w.z;
    if (e >= f.n_elems) return;                      // the pseudo-element of the lost markers
    const int H = 1 + 2 * f.n_modes;
    DepMarker d[kItemR];
#pragma unroll
    for (int r = 0; r < kItemR; ++r) {
        const bool on = 32 * r + lane < count;
        Marker s;
        s.x = 1.0; s.y = 0.0; s.z = 0.0; s.vx = s.vy = s.vz = 0.0; s.mu = 0.0; s.w = 0.0;
        if (on) {
            const double *p = rec + (size_t)kRecDoubles * (start + 32 * r + lane);
            s.x = p[0]; s.y = p[1]; s.z = p[2]; s.w = p[3]; s.vx = p[4]; s.vy = p[5]; s.vz = p[6]; s.mu = p[7];
        }
        dep_marker<kF>(f, o, e, s, mass, d[r]);
        if (!on) { d[r].amp[0] = 0.0; d[r].amp[1] = 0.0; }
    }
    double *out = rhs + (size_t)e * 2 * H * M3DK_NCOEF;
    for (int mom = 0; mom < 2; ++mom)
#pragma unroll
        for (int h = 0; h < kDepHarmMax; ++h) {
            if (h >= H) break;
            double ah[kItemR];
#pragma unroll
            for (int r = 0; r < kItemR; ++r) ah[r] = __dmul_rn(d[r].amp[mom], d[r].T[h]);
            dep_row_add(out + ((size_t)mom * H + h) * M3DK_NCOEF, lane, [&](int ii, int j) {
                double val = 0.0;
#pragma unroll
                for (int r = 0; r < kItemR; ++r) val = M3DK_FMA(ah[r], __dmul_rn(d[r].xp[ii], d[r].ep[j]), val);
                return val;
            });
        }
}

// ---- 4-point FLR deposition through the ordered ring stream (FLR workspace set) ---------------------------------------
// The ring points of all markers are emitted (position + the marker's two amplitudes), ordered by THEIR element with the
// ring-ordering kernels of the FLR push (ring_key_kernel, scan, work-item cut, placement), and a warp deposits a ring item
// (up to 64 ring points of one element) with shuffle reductions and one atomic per table entry.
template <int kF>
__global__ void __launch_bounds__(128) deposit_flr_emit_kernel(const __grid_constant__ FieldParams f, const __grid_constant__ DepOpts o,
                                                               const double *__restrict__ rec, const int *__restrict__ key, long n,
                                                               double q, double mass, double *__restrict__ ring,
                                                               double *__restrict__ wts) {
    const long i = (long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    int e = key[i];
    if (e >= f.n_elems) e = -1;
    if (e < 0) {                                     // lost markers deposit nothing: no ring
        for (int j = 0; j < 4; ++j) {
            double *r = ring + 4 * (4 * i + j);
            r[0] = 0.0; r[1] = 0.0; r[2] = 0.0; r[3] = -1.0;
        }
        return;
    }
    const double *p = rec + (size_t)kRecDoubles * i;
    Marker s;
    s.x = p[0]; s.y = p[1]; s.z = p[2]; s.w = p[3]; s.vx = p[4]; s.vy = p[5]; s.vz = p[6]; s.mu = p[7];
    DepMarker d;
    dep_marker<kF>(f, o, e, s, mass, d);          // amplitudes at the marker itself
    wts[10 * i] = d.amp[0]; wts[10 * i + 1] = d.amp[1];
    // the ring: same construction as the FLR push (reading G23)
    StepGeom g;
    step_geometry(s, g);
    const double *tile = f.tiles + (size_t)e * f.tile_stride;
    const Quad hd = ldq(tile);
    const double se0 = hd.c;
    const double xi1[1] = {__dmul_rn(__dsub_rn(g.R, hd.a), se0)}, eta1[1] = {__dmul_rn(__dsub_rn(s.z, hd.b), se0)};
    double v[1][4], dx[1][4], de[1][4];
    Ring rg;
    ring_fill<false>(rg, tile + kTileHeader);
    quad_vd<1, false>(tile + kTileHeader, tile + kTileHeader, rg, xi1, eta1, v, dx, de);
    const double BR = -__dmul_rn(__dmul_rn(de[0][0], se0), g.rinv), BP = __dmul_rn(v[0][2], g.rinv),
                 BZ = __dmul_rn(__dmul_rn(dx[0][0], se0), g.rinv);
    const double binv = m3dk_rsqrt(M3DK_FMA(BR, BR, M3DK_FMA(BP, BP, __dmul_rn(BZ, BZ))));
    const double bR = __dmul_rn(BR, binv), bP = __dmul_rn(BP, binv), bZ = __dmul_rn(BZ, binv);
    const double rho = __dmul_rn(m3dk_sqrt(__dmul_rn(__dmul_rn(__dmul_rn(2.0, mass), s.mu), binv)), fabs(1.0 / q));
    double e1R = M3DK_FMA(-bR, bR, 1.0), e1P = -__dmul_rn(bR, bP), e1Z = -__dmul_rn(bR, bZ);
    if (__dmul_rn(bR, bR) > 0.999999) {   // b (anti)parallel to R-hat: start from Z-hat instead (same rule as the oracle)
        e1R = -__dmul_rn(bZ, bR); e1P = -__dmul_rn(bZ, bP); e1Z = M3DK_FMA(-bZ, bZ, 1.0);
    }
    const double n1 = m3dk_rsqrt(M3DK_FMA(e1R, e1R, M3DK_FMA(e1P, e1P, __dmul_rn(e1Z, e1Z))));
    e1R = __dmul_rn(e1R, n1); e1P = __dmul_rn(e1P, n1); e1Z = __dmul_rn(e1Z, n1);
    const double e2R = M3DK_FMA(bP, e1Z, -__dmul_rn(bZ, e1P)), e2P = M3DK_FMA(bZ, e1R, -__dmul_rn(bR, e1Z)),
                 e2Z = M3DK_FMA(bR, e1P, -__dmul_rn(bP, e1R));
    const double c = g.cph, sn = g.sph;
    const double ex[2] = {M3DK_FMA(e1R, c, -__dmul_rn(e1P, sn)), M3DK_FMA(e2R, c, -__dmul_rn(e2P, sn))};
    const double ey[2] = {M3DK_FMA(e1R, sn, __dmul_rn(e1P, c)), M3DK_FMA(e2R, sn, __dmul_rn(e2P, c))};
    const double ez[2] = {e1Z, e2Z};
    const double X = __dmul_rn(g.R, c), Y = __dmul_rn(g.R, sn);
#pragma unroll
    for (int j = 0; j < 4; ++j) {
        const double sg = j < 2 ? rho : -rho;
        double *r = ring + 4 * (4 * i + j);
        r[0] = M3DK_FMA(sg, ex[j & 1], X); r[1] = M3DK_FMA(sg, ey[j & 1], Y); r[2] = M3DK_FMA(sg, ez[j & 1], s.z); r[3] = 1.0;
    }
}

template <int kR>
__global__ void __launch_bounds__(128) deposit_ring_items_kernel(const __grid_constant__ FieldParams f, const double *__restrict__ ring,
                                                                 const double *__restrict__ wts, const int *__restrict__ rorder,
                                                                 const int4 *__restrict__ items, const int *__restrict__ n_items,
                                                                 double *__restrict__ rhs) {
    const int lane = threadIdx.x & 31;
    const int it = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
    if (it >= *n_items) return;
    const int4 w = __ldg(items + it);
    const int e = w.x, start = w.y, count = w.z;
    if (e >= f.n_elems) return;                      // ring points outside the mesh deposit nothing
    const int H = 1 + 2 * f.n_modes;
    const Quad hd = ldq(f.tiles + (size_t)e * f.tile_stride);
    double amp[kR][2], T[kR][kDepHarmMax], xp[kR][6], ep[kR][6];
#pragma unroll
    for (int r = 0; r < kR; ++r) {
        const bool on = 32 * r + lane < count;
        Marker sp;
        sp.x = 1.0; sp.y = 0.0; sp.z = 0.0;
        amp[r][0] = 0.0; amp[r][1] = 0.0;
        if (on) {
            const long idx = rorder[start + 32 * r + lane];
            const double *p = ring + 4 * idx;
            sp.x = p[0]; sp.y = p[1]; sp.z = p[2];
            amp[r][0] = __dmul_rn(0.25, wts[10 * (idx >> 2)]); amp[r][1] = __dmul_rn(0.25, wts[10 * (idx >> 2) + 1]);
        }
        StepGeom gj;
        step_geometry(sp, gj);
        const double xi = __dmul_rn(__dsub_rn(gj.R, hd.a), hd.c), eta = __dmul_rn(__dsub_rn(sp.z, hd.b), hd.c);
        xp[r][0] = 1.0; ep[r][0] = 1.0;
#pragma unroll
        for (int q = 1; q < 6; ++q) { xp[r][q] = __dmul_rn(xp[r][q - 1], xi); ep[r][q] = __dmul_rn(ep[r][q - 1], eta); }
        T[r][0] = 1.0;
#pragma unroll
        for (int md = 0; md < M3DK_MAX_MODES; ++md)
            if (md < f.n_modes) mode_phase(f.n_tor[md], gj.cph, gj.sph, 1.0, 0.0, T[r][1 + 2 * md], T[r][2 + 2 * md]);
    }
    double *out = rhs + (size_t)e * 2 * H * M3DK_NCOEF;
    for (int mom = 0; mom < 2; ++mom)
#pragma unroll
        for (int h = 0; h < kDepHarmMax; ++h) {
            if (h >= H) break;
            double ah[kR];
#pragma unroll
            for (int r = 0; r < kR; ++r) ah[r] = __dmul_rn(amp[r][mom], T[r][h]);
            dep_row_add(out + ((size_t)mom * H + h) * M3DK_NCOEF, lane, [&](int ii, int j) {
                double val = 0.0;
#pragma unroll
                for (int r = 0; r < kR; ++r) val = M3DK_FMA(ah[r], __dmul_rn(xp[r][ii], ep[r][j]), val);
                return val;
            });
        }
}

// the four instantiations of a kernel template whose LAST parameter is kF (0 .. 3)
#define M3DK_DEP_PICK(kf, ...) ((kf) == 0 ? __VA_ARGS__ 0> : (kf) == 1 ? __VA_ARGS__ 1> : (kf) == 2 ? __VA_ARGS__ 2> : __VA_ARGS__ 3>)

cudaError_t launch_deposit(m3dk_ctx *c, long n, double *rhs, int flags, double t) {
    DepOpts o{};
    o.with_b1par = (flags & 1) && c->f.n_modes > 0;
    o.with_bstar = (flags & 4) && c->f.n_modes > 0;
    o.q = c->q;
    const int kf = (o.with_b1par ? 1 : 0) | (o.with_bstar ? 2 : 0);
    for (int k = 0; k < c->f.n_modes; ++k) { o.cwt[k] = cos(c->f.omega[k] * t); o.swt[k] = sin(c->f.omega[k] * t); }
    const size_t bytes = (size_t)c->f.n_elems * 2 * (1 + 2 * c->f.n_modes) * M3DK_NCOEF * sizeof(double);
    cudaError_t e = cudaMemsetAsync(rhs, 0, bytes, c->stream);
    if (e != cudaSuccess || n == 0) return e;
    if (flags & 2) {   // 4-point FLR deposition: the ring points leave the marker's element, one marker per lane
        if (c->have_sortws && c->have_flrws) {
            // ordered ring stream: markers into element order, ring points emitted, ordered by their own element, deposited
            // item by item
            e = launch_pack_sorted(c, n);
            if (e != cudaSuccess) return e;
            e = cudaMemsetAsync(c->fb.a.rhist, 0, (size_t)(c->f.n_elems + 1) * sizeof(int), c->stream);
            if (e != cudaSuccess) return e;
            c->kernel_launches += 3;
            M3DK_DEP_PICK(kf, deposit_flr_emit_kernel<)<<<(unsigned)((n + 127) / 128), 128, 0, c->stream>>>(
                c->f, o, c->sb.rec[c->cur], c->sb.key, n, c->q, c->m, c->fb.a.ring, c->fb.a.wts);
            e = launch_flr_ring_keys(c, n);
            if (e != cudaSuccess) return e;
            e = launch_flr_ring_stage(c, n);
            if (e != cudaSuccess) return e;
            const long max_items = 4 * n / kItemMarkers + c->f.n_elems + 2, max_small = c->f.n_elems + 2;
            deposit_ring_items_kernel<2><<<(unsigned)((max_items + 3) / 4), 128, 0, c->stream>>>(
                c->f, c->fb.a.ring, c->fb.a.wts, c->fb.a.rorder, c->fb.ritems, c->fb.rioffs + c->f.n_elems + 1, rhs);
            deposit_ring_items_kernel<1><<<(unsigned)((max_small + 3) / 4), 128, 0, c->stream>>>(
                c->f, c->fb.a.ring, c->fb.a.wts, c->fb.a.rorder, c->fb.ritems_small,
                reinterpret_cast<const int *>(c->fb.rstate + 1), rhs);
        } else if (c->have_sortws) {
            e = launch_pack_sorted(c, n);
            if (e != cudaSuccess) return e;
            c->kernel_launches += 1;
            M3DK_DEP_PICK(kf, deposit_flr_kernel<true,)<<<(unsigned)((n + 127) / 128), 128, 0, c->stream>>>(
                c->f, o, c->user, c->sb.rec[c->cur], c->sb.key, n, c->q, c->m, rhs);
        } else {
            c->kernel_launches += 1;
            M3DK_DEP_PICK(kf, deposit_flr_kernel<false,)<<<(unsigned)((n + 127) / 128), 128, 0, c->stream>>>(
                c->f, o, c->user, nullptr, nullptr, n, c->q, c->m, rhs);
        }
        return cudaGetLastError();
    }
    if (c->have_sortws) {
        // order the markers by the element of their CURRENT position first (after a push the arrays are in the order of
        // the previous positions): records in element order + work items, then one warp per item
        e = launch_pack_sorted(c, n);
        if (e != cudaSuccess) return e;
        const long max_items = n / kItemMarkers + c->f.n_elems + 2, max_small = c->f.n_elems + 2;
        c->kernel_launches += 2;
        M3DK_DEP_PICK(kf, deposit_items_kernel<)<<<(unsigned)((max_items + 3) / 4), 128, 0, c->stream>>>(
            c->f, o, c->sb.rec[c->cur], c->sb.items, c->sb.ioffs + c->f.n_elems + 1, c->m, rhs);
        M3DK_DEP_PICK(kf, deposit_items_kernel<)<<<(unsigned)((max_small + 3) / 4), 128, 0, c->stream>>>(          // the small items
            c->f, o, c->sb.rec[c->cur], c->sb.items_small, reinterpret_cast<const int *>(c->sb.scan_state + 1), c->m, rhs);
        return cudaGetLastError();
    }
    c->kernel_launches += 1;
    M3DK_DEP_PICK(kf, deposit_kernel<)<<<(unsigned)((n + 127) / 128), 128, 0, c->stream>>>(c->f, o, c->user, n, c->m, rhs);
    return cudaGetLastError();
}

}  // namespace m3dk
