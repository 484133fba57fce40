// m3dk_push.cu -- kernels of the fused push and their launchers.
#include <math.h>

#include "m3dk_device.cuh"

namespace m3dk {

// CTA shape of the element-ordered kernel: 128 threads x 3 CTAs per SM (168 registers); measured alternatives in
// profiles/r1_development_notes.md
#ifndef M3DK_PUSH_THREADS
#define M3DK_PUSH_THREADS 128
#endif
#ifndef M3DK_PUSH_MINBLOCKS
#define M3DK_PUSH_MINBLOCKS 3
#endif
constexpr int kPushThreads = M3DK_PUSH_THREADS;

// ---- element of every marker (particles_init / upload) ------------------------------------------------------------
__global__ void __launch_bounds__(256) locate_kernel(const __grid_constant__ FieldParams f, MarkerArrays a, long n,
                                                     int fill_id, int id_base) {
    const long i = (long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    a.elem[i] = locate_xyz(f, a.x[i], a.y[i], a.z[i]);
    if (fill_id) a.id[i] = id_base + (int)i;
}

// Warp-aggregated histogram with returned ranks for R keys per lane (lanes with the same key elect a leader that does
// one atomic), in two halves: the atomics are issued as soon as the new keys exist, the returned
// values are consumed (rank_finish) only after the next block of arithmetic, so their round trip to L2 is never waited for.
template <int R>
__device__ __forceinline__ void hist_issue(int *hist, const int (&key)[R], const bool (&on)[R], unsigned (&peers)[R],
                                           int (&base)[R]) {
    const int lane = threadIdx.x & 31;
#pragma unroll
    for (int r = 0; r < R; ++r) {
        const unsigned live = __ballot_sync(0xffffffffu, on[r]);
        peers[r] = 0u; base[r] = 0;
        if (on[r]) {
            peers[r] = __match_any_sync(live, key[r]);
            if (lane == __ffs(peers[r]) - 1) base[r] = atomicAdd(hist + key[r], __popc(peers[r]));
        }
    }
}
template <int R>
__device__ __forceinline__ void rank_finish(int *rank, const long (&m)[R], const bool (&on)[R], const unsigned (&peers)[R],
                                            const int (&base)[R]) {
    const int lane = threadIdx.x & 31;
#pragma unroll
    for (int r = 0; r < R; ++r)
        if (on[r]) {
            const int b = __shfl_sync(peers[r], base[r], __ffs(peers[r]) - 1);
            rank[m[r]] = b + __popc(peers[r] & ((1u << lane) - 1u));
        }
}

// ---- marker state access: the caller's SoA arrays (any order, in place) or 64-byte records (ordered pipeline) -------
__device__ __forceinline__ void ldrec256(const double *p, double &a, double &b, double &c, double &d) {
    // not volatile, no memory clobber: a thread only ever writes a record after it has read it, and every value it
    // stores depends on the values loaded here, so the data dependences already order the accesses
    asm("ld.global.v4.f64 {%0, %1, %2, %3}, [%4];" : "=d"(a), "=d"(b), "=d"(c), "=d"(d) : "l"(p));
}
__device__ __forceinline__ void strec256(double *p, double a, double b, double c, double d) {
    asm volatile("st.global.v4.f64 [%0], {%1, %2, %3, %4};" ::"l"(p), "d"(a), "d"(b), "d"(c), "d"(d));
}

struct SoAIO {
    MarkerArrays a;
    int n_elems;
    __device__ __forceinline__ void load_pos(long i, double &x, double &y, double &z, double &w) const {
        x = a.x[i]; y = a.y[i]; z = a.z[i]; w = a.w[i];
    }
    __device__ __forceinline__ void load_vel(long i, double &vx, double &vy, double &vz, double &mu) const {
        vx = a.vx[i]; vy = a.vy[i]; vz = a.vz[i]; mu = a.mu[i];
    }
    __device__ __forceinline__ void store_pos(long o, double x, double y, double z, double) const {
        a.x[o] = x; a.y[o] = y; a.z[o] = z;
    }
    __device__ __forceinline__ void store_vel(long o, double vx, double vy, double vz, double) const {
        a.vx[o] = vx; a.vy[o] = vy; a.vz[o] = vz;          // mu is never written
    }
    __device__ __forceinline__ void store_w(long o, double w) const { a.w[o] = w; }
    __device__ __forceinline__ void store_key(long o, int ne) const { a.elem[o] = ne; }
};

struct RecIO {   // record = (x, y, z, w | vx, vy, vz, mu): two 32-byte sectors, each moved by one 256-bit access
    const double *in;
    double *out;
    int *key;
    int n_elems;
    __device__ __forceinline__ void load_pos(long i, double &x, double &y, double &z, double &w) const {
        ldrec256(in + kRecDoubles * i, x, y, z, w);
    }
    __device__ __forceinline__ void load_vel(long i, double &vx, double &vy, double &vz, double &mu) const {
        ldrec256(in + kRecDoubles * i + 4, vx, vy, vz, mu);
    }
    __device__ __forceinline__ void store_pos(long o, double x, double y, double z, double w_old) const {
        strec256(out + kRecDoubles * o, x, y, z, w_old);      // w is patched by store_w once phase B has it
    }
    __device__ __forceinline__ void store_vel(long o, double vx, double vy, double vz, double mu) const {
        strec256(out + kRecDoubles * o + 4, vx, vy, vz, mu);
    }
    __device__ __forceinline__ void store_w(long o, double w) const { out[kRecDoubles * o + 3] = w; }
    __device__ __forceinline__ void store_key(long o, int ne) const { key[o] = ne < 0 ? n_elems : ne; }
};

// ---- one step of R markers of one thread that sit in the same element (rows a1-a10) ------------------------------
// mi[r] / mo[r]: input / output slot of marker r, on[r]: marker r exists.  Phase A: a1 load, a2 cylindrical map, a4-a5
// equilibrium quad (every coefficient load shared by the R markers), a7 assemble, a8 Boris, a10 drift + store.
// Phase B: a6 perturbed quads folded into dw/dt as they are evaluated, a9 weight update.  Then a3 for the NEW position
// (cached for the next step; it is the sort key) and, with kHist, the sort histogram of the new keys.
// tile: the element's coefficient tile, in global memory (kSmem = false) or staged in shared memory (kSmem = true).
__device__ __forceinline__ double flr_wdot(const PushParams &P, const EqOut &f, const StepGeom &g, double zl, double mu,
                                           const PertW &W);
__device__ __forceinline__ void flr_emit(const PushParams &P, const EqOut &f, const StepGeom &g, double zl, double mu,
                                         const PertW &W, long slot);
struct PertF;

// kFlr (mode 2): phase B is replaced by the 4-point gyro-average of the perturbed fields.  kFlr = 1: every lane evaluates
// its four ring points itself, each on its own element's tile read from global memory (flr_wdot).  kFlr = 2: the lane only
// EMITS the ring points (position, element, weights of the perturbed fields in dw/dt) into the ring stream (flr_emit);
// they are ordered by THEIR element, evaluated by ring_items_kernel with staged tiles and summed back by flr_reduce_kernel.
// kPost (asynchronously staged kernel): the step ends with the new (R, Z) in Rn, Zn; search, key, histogram and rank are
// the caller's (it runs them one item later, on data that was fetched in the meantime); io.stage_next() is called once
// all of this lane's input has been consumed.
template <int R, bool kHist, bool kSmem, class IO, int kFlr = 0, bool kPost = false>
__device__ __forceinline__ void step_R(const PushParams &P, const IO &io, const double *__restrict__ tile,
                                       const long (&mi)[R], const long (&mo)[R], const bool (&on)[R], double (&Rn)[R],
                                       double (&Zn)[R]) {
    Marker s[R];
    StepGeom g[R];
#pragma unroll
    for (int r = 0; r < R; ++r) {
        if (on[r]) io.load_pos(mi[r], s[r].x, s[r].y, s[r].z, s[r].w);
        else { s[r].x = 1.0; s[r].y = 0.0; s[r].z = 0.0; s[r].w = 0.0; }
    }
    const Quad hd = ldq_t<kSmem>(tile);
    const double Rc = hd.a, Zc = hd.b, se = hd.c;
    double xi[R], eta[R];
#pragma unroll
    for (int r = 0; r < R; ++r) {
        step_geometry(s[r], g[r]);
        xi[r] = __dmul_rn(__dsub_rn(g[r].R, Rc), se); eta[r] = __dmul_rn(__dsub_rn(s[r].z, Zc), se);
    }
    double v[R][4], dx[R][4], de[R][4];
    Ring ring;
    ring_fill<kSmem>(ring, tile + kTileHeader);
    quad_vd<R, kSmem>(tile + kTileHeader, tile + kTileHeader, ring, xi, eta, v, dx, de);   // (psi0, |B|0, F0, kappa)
    PertW W[R];
    FastRec rec[kPost ? 1 : R];
    // three separate loops (loads, arithmetic, stores): the arithmetic of the R markers sits in one block with no
    // memory operation in between, so that the scheduler interleaves the R dependent chains (DFMA latency 8 cycles)
#pragma unroll
    for (int r = 0; r < R; ++r) {
        if (on[r]) io.load_vel(mi[r], s[r].vx, s[r].vy, s[r].vz, s[r].mu);
        else { s[r].vx = s[r].vy = s[r].vz = 0.0; s[r].mu = 0.0; }
    }
    EqOut fe[kFlr ? R : 1];   // kept for the gyro ring (mode 2)
    double zl[kFlr ? R : 1];
#pragma unroll
    for (int r = 0; r < R; ++r) {
        EqOut f;
        f.psi_R = __dmul_rn(dx[r][0], se); f.psi_Z = __dmul_rn(de[r][0], se);
        f.Bm = v[r][1]; f.Bm_R = __dmul_rn(dx[r][1], se); f.Bm_Z = __dmul_rn(de[r][1], se);
        f.F = v[r][2]; f.kappa = v[r][3];
        if (kFlr) { fe[r] = f; zl[r] = s[r].z; }
        push_eq(P, g[r], f, s[r], W[r]);
        Rn[r] = m3dk_sqrt(M3DK_FMA(s[r].x, s[r].x, __dmul_rn(s[r].y, s[r].y)));
        Zn[r] = s[r].z;
    }
#pragma unroll
    for (int r = 0; r < R; ++r) {
        if (on[r]) {
            io.store_pos(mo[r], s[r].x, s[r].y, s[r].z, s[r].w);
            io.store_vel(mo[r], s[r].vx, s[r].vy, s[r].vz, s[r].mu);
        }
        // the element search of the new position runs after phase B (loading its first record here, or searching
        // between the quads, costs registers in the hottest part of the kernel and measured slower; an L1 prefetch of
        // the record measured no gain)
    }
    if constexpr (kPost) io.stage_next();
    // a3 for the NEW position (the key of the next sort) and, with kHist, the sort histogram of the new keys with each
    // marker's rank inside its key (the sort then needs no pass over the keys)
    unsigned peers[R];
    int base[R];
    auto locate_and_count = [&]() {
        if constexpr (!kPost) {
#pragma unroll
            for (int r = 0; r < R; ++r) rec[r] = locate_first(P.f.fast, Rn[r], Zn[r]);   // all first records in flight together
            int key[R];
#pragma unroll
            for (int r = 0; r < R; ++r) {
                int ne = -1;
                if (on[r]) {
                    ne = locate_finish(P.f, rec[r], Rn[r], Zn[r]);
                    io.store_key(mo[r], ne);
                }
                key[r] = ne < 0 ? P.f.n_elems : ne;
            }
            if (kHist) hist_issue<R>(P.hist, key, on, peers, base);
        }
    };
    if (kFlr && P.f.n_modes > 0) {
#pragma unroll
        for (int r = 0; r < R; ++r) {
            if constexpr (kFlr == 2) {
                if (on[r]) flr_emit(P, fe[kFlr ? r : 0], g[r], zl[kFlr ? r : 0], s[r].mu, W[r], mo[r]);
            } else {
                const double wdot = flr_wdot(P, fe[kFlr ? r : 0], g[r], zl[kFlr ? r : 0], s[r].mu, W[r]);
                if (on[r]) io.store_w(mo[r], M3DK_FMA(P.dt, wdot, s[r].w));
            }
        }
        locate_and_count();
    } else if (P.f.n_modes > 0) {
        double wsum[R];
#pragma unroll
        for (int r = 0; r < R; ++r) wsum[r] = 0.0;
        for (int md = 0; md < P.f.n_modes; ++md) {
            const int n = P.f.n_tor[md];
            const double om = P.f.omega[md];
            double cth[R], sth[R], nri[R];
#pragma unroll
            for (int r = 0; r < R; ++r) {
                mode_phase(n, g[r].cph, g[r].sph, P.cwt[md], P.swt[md], cth[r], sth[r]);
                nri[r] = __dmul_rn((double)n, g[r].rinv);
            }
            const double *pm = tile + kTileHeader + kTileEq + kTileMode * md;
            ring_fill<kSmem>(ring, pm);
            // the two value-only quads share one copy of the Horner code (rolled: the kernel must fit the 32 KB
            // instruction cache); the weights of quad q are picked by selects
#pragma unroll 1
            for (int q = 0; q < 2; ++q) {
                quad_vd<R, kSmem>(pm + q * kQuad, pm + (q + 1) * kQuad, ring, xi, eta, v, dx, de);
#pragma unroll
                for (int r = 0; r < R; ++r) {
                    const double wa = q == 0 ? W[r].aER : W[r].aEZ;
                    const double wb = q == 0 ? W[r].aEP : W[r].bBR;
                    wsum[r] = pert_fold_v(wsum[r], v[r], wa, wb, cth[r], sth[r]);
                }
            }
            quad_vd<R, kSmem>(pm + 2 * kQuad, pm, ring, xi, eta, v, dx, de);   // (B_par, B_Z); quad 3 (B_phi) is not needed
#pragma unroll
            for (int r = 0; r < R; ++r) wsum[r] = pert_fold_par(wsum[r], v[r], dx[r], de[r], W[r], cth[r], sth[r], se, nri[r], om);
        }
        // Eqs. (8)-(9): explicit midpoint on the staggered grid (G9)
#pragma unroll
        for (int r = 0; r < R; ++r)
            if (on[r]) io.store_w(mo[r], M3DK_FMA(P.dt, wsum[r], s[r].w));
        locate_and_count();
    } else {
        locate_and_count();
    }
    if (kHist && !kPost) rank_finish<R>(P.rank, mo, on, peers, base);
}

// Perturbed fields of R markers of one element, summed over the toroidal modes, in each marker's own cylindrical frame
// (all four quads of every mode: E_R E_phi | E_Z B_R | B_par with gradient, B_Z | B_phi).  pf must be zeroed by the caller.
template <int R, bool kSmem>
__device__ __forceinline__ void pert_fields(const PushParams &P, const double *__restrict__ tile, const double (&xi)[R],
                                            const double (&eta)[R], const StepGeom (&g)[R], double se, PertF (&pf)[R]) {
    double v[R][4], dx[R][4], de[R][4];
    Ring ring;
    for (int md = 0; md < P.f.n_modes; ++md) {
        const int n = P.f.n_tor[md];
        const double om = P.f.omega[md];
        double cth[R], sth[R], nri[R];
#pragma unroll
        for (int r = 0; r < R; ++r) {
            mode_phase(n, g[r].cph, g[r].sph, P.cwt[md], P.swt[md], cth[r], sth[r]);
            nri[r] = __dmul_rn((double)n, g[r].rinv);
        }
        const double *pm = tile + kTileHeader + kTileEq + kTileMode * md;
        ring_fill<kSmem>(ring, pm);
        quad_vd<R, kSmem>(pm, pm + kQuad, ring, xi, eta, v, dx, de);                          // E_R, E_phi
#pragma unroll
        for (int r = 0; r < R; ++r) {
            pf[r].ER = __dadd_rn(pf[r].ER, re_part(v[r][0], v[r][1], cth[r], sth[r]));
            pf[r].EP = __dadd_rn(pf[r].EP, re_part(v[r][2], v[r][3], cth[r], sth[r]));
        }
        quad_vd<R, kSmem>(pm + kQuad, pm + 2 * kQuad, ring, xi, eta, v, dx, de);             // E_Z, B_R
#pragma unroll
        for (int r = 0; r < R; ++r) {
            pf[r].EZ = __dadd_rn(pf[r].EZ, re_part(v[r][0], v[r][1], cth[r], sth[r]));
            pf[r].BR = __dadd_rn(pf[r].BR, re_part(v[r][2], v[r][3], cth[r], sth[r]));
        }
        quad_vd<R, kSmem>(pm + 2 * kQuad, pm + 3 * kQuad, ring, xi, eta, v, dx, de);         // B_par (+ gradient), B_Z
#pragma unroll
        for (int r = 0; r < R; ++r) {
            pf[r].BZ = __dadd_rn(pf[r].BZ, re_part(v[r][2], v[r][3], cth[r], sth[r]));
            const double qd = M3DK_FMA(v[r][0], sth[r], __dmul_rn(v[r][1], cth[r]));   // d/dphi -> -n qd, d/dt -> omega qd
            pf[r].gR = __dadd_rn(pf[r].gR, re_part(__dmul_rn(dx[r][0], se), __dmul_rn(dx[r][1], se), cth[r], sth[r]));
            pf[r].gP = __dsub_rn(pf[r].gP, __dmul_rn(nri[r], qd));
            pf[r].gZ = __dadd_rn(pf[r].gZ, re_part(__dmul_rn(de[r][0], se), __dmul_rn(de[r][1], se), cth[r], sth[r]));
            pf[r].dT = M3DK_FMA(om, qd, pf[r].dT);
        }
        quad_vd<R, kSmem>(pm + 3 * kQuad, pm, ring, xi, eta, v, dx, de);                      // B_phi
#pragma unroll
        for (int r = 0; r < R; ++r) pf[r].BP = __dadd_rn(pf[r].BP, re_part(v[r][0], v[r][1], cth[r], sth[r]));
    }
}

// ---- finite Larmor radius (mode 2; Eq. 14; reading G23) ------------------------------------------
// dw/dt of one marker with the perturbed fields replaced by the quarter sum over the four gyro-ring points
// X +- rho e1, X +- rho e2 (rho = m v_perp / (|q| B), v_perp = sqrt(2 mu B / m); e1 = the major-radius direction made
// perpendicular to b0, e2 = b0 x e1).  dw/dt is linear in the perturbed fields, so the quarter sum is taken of the four
// scalar contributions c_j = (weights) . (fields at ring point j): the nine weights of PertW are rotated once to Cartesian
// components (FlrW), the fields of a ring point are rotated from that point's cylindrical frame, and
//     dw/dt = 0.25 (((c_0 + c_1) + c_2) + c_3),      c_j = 0 for a ring point outside the mesh.
// Every kernel takes the same route through flr_ring_point / flr_fold, so the bits do not depend on who evaluates a point.
struct FlrRing { double X, Y, rho, ex[2], ey[2], ez[2]; };
struct FlrW { double aEx, aEy, aEz, bBx, bBy, bBz, gGx, gGy, gGz, dT; };

__device__ __forceinline__ void flr_ring(const PushParams &P, const EqOut &f, const StepGeom &g, double mu, FlrRing &rg) {
    const double BR = -__dmul_rn(f.psi_Z, g.rinv), BP = __dmul_rn(f.F, g.rinv), BZ = __dmul_rn(f.psi_R, g.rinv);
    const double binv = m3dk_rsqrt(M3DK_FMA(BR, BR, M3DK_FMA(BP, BP, __dmul_rn(BZ, BZ))));
    const double bR = __dmul_rn(BR, binv), bP = __dmul_rn(BP, binv), bZ = __dmul_rn(BZ, binv);
    rg.rho = __dmul_rn(m3dk_sqrt(__dmul_rn(__dmul_rn(__dmul_rn(2.0, P.m), mu), binv)), fabs(P.inv_q));
    // e1 = R-hat - (R-hat . b) b, normalised; e2 = b x e1 (cylindrical components at the marker)
    double e1R = M3DK_FMA(-bR, bR, 1.0), e1P = -__dmul_rn(bR, bP), e1Z = -__dmul_rn(bR, bZ);
    if (__dmul_rn(bR, bR) > 0.999999) {   // b (anti)parallel to R-hat: start from Z-hat instead (same rule as the oracle)
        e1R = -__dmul_rn(bZ, bR); e1P = -__dmul_rn(bZ, bP); e1Z = M3DK_FMA(-bZ, bZ, 1.0);
    }
    const double n1 = m3dk_rsqrt(M3DK_FMA(e1R, e1R, M3DK_FMA(e1P, e1P, __dmul_rn(e1Z, e1Z))));
    e1R = __dmul_rn(e1R, n1); e1P = __dmul_rn(e1P, n1); e1Z = __dmul_rn(e1Z, n1);
    const double e2R = M3DK_FMA(bP, e1Z, -__dmul_rn(bZ, e1P)), e2P = M3DK_FMA(bZ, e1R, -__dmul_rn(bR, e1Z)),
                 e2Z = M3DK_FMA(bR, e1P, -__dmul_rn(bP, e1R));
    const double c = g.cph, sn = g.sph;
    rg.ex[0] = M3DK_FMA(e1R, c, -__dmul_rn(e1P, sn)); rg.ex[1] = M3DK_FMA(e2R, c, -__dmul_rn(e2P, sn));
    rg.ey[0] = M3DK_FMA(e1R, sn, __dmul_rn(e1P, c)); rg.ey[1] = M3DK_FMA(e2R, sn, __dmul_rn(e2P, c));
    rg.ez[0] = e1Z; rg.ez[1] = e2Z;
    rg.X = __dmul_rn(g.R, c); rg.Y = __dmul_rn(g.R, sn);
}
__device__ __forceinline__ void flr_ring_point(const FlrRing &rg, double zl, int j, double &x, double &y, double &z) {
    const double sg = j < 2 ? rg.rho : -rg.rho;
    x = M3DK_FMA(sg, rg.ex[j & 1], rg.X); y = M3DK_FMA(sg, rg.ey[j & 1], rg.Y); z = M3DK_FMA(sg, rg.ez[j & 1], zl);
}
// the weights of PertW (marker's cylindrical frame; B1_phi does not enter) as Cartesian vectors
__device__ __forceinline__ void flr_cart_weights(const PertW &W, double c, double sn, FlrW &cw) {
    cw.aEx = M3DK_FMA(W.aER, c, -__dmul_rn(W.aEP, sn)); cw.aEy = M3DK_FMA(W.aER, sn, __dmul_rn(W.aEP, c)); cw.aEz = W.aEZ;
    cw.bBx = __dmul_rn(W.bBR, c); cw.bBy = __dmul_rn(W.bBR, sn); cw.bBz = W.bBZ;
    cw.gGx = M3DK_FMA(W.gR, c, -__dmul_rn(W.gP, sn)); cw.gGy = M3DK_FMA(W.gR, sn, __dmul_rn(W.gP, c)); cw.gGz = W.gZ;
    cw.dT = W.dT;
}
// c_j: the fields pf of a ring point (its own cylindrical frame, cos / sin of its phi = cj, sj) against the weights
__device__ __forceinline__ double flr_fold(const PertF &pf, double cj, double sj, const FlrW &cw) {
    const double Ex = M3DK_FMA(pf.ER, cj, -__dmul_rn(pf.EP, sj)), Ey = M3DK_FMA(pf.ER, sj, __dmul_rn(pf.EP, cj));
    const double Bx = M3DK_FMA(pf.BR, cj, -__dmul_rn(pf.BP, sj)), By = M3DK_FMA(pf.BR, sj, __dmul_rn(pf.BP, cj));
    const double Gx = M3DK_FMA(pf.gR, cj, -__dmul_rn(pf.gP, sj)), Gy = M3DK_FMA(pf.gR, sj, __dmul_rn(pf.gP, cj));
    double a = __dmul_rn(cw.aEx, Ex);
    a = M3DK_FMA(cw.aEy, Ey, a); a = M3DK_FMA(cw.aEz, pf.EZ, a);
    a = M3DK_FMA(cw.bBx, Bx, a); a = M3DK_FMA(cw.bBy, By, a); a = M3DK_FMA(cw.bBz, pf.BZ, a);
    a = M3DK_FMA(cw.gGx, Gx, a); a = M3DK_FMA(cw.gGy, Gy, a); a = M3DK_FMA(cw.gGz, pf.gZ, a);
    return M3DK_FMA(cw.dT, pf.dT, a);
}

// kFlr = 1: the lane evaluates its four ring points itself, each searched and evaluated on its own element's tile (global
// memory: the ring leaves the marker's element).  (g, zl) = cylindrical map and z of x_l.
__device__ __forceinline__ double flr_wdot(const PushParams &P, const EqOut &f, const StepGeom &g, double zl, double mu,
                                           const PertW &W) {
    FlrRing rg;
    flr_ring(P, f, g, mu, rg);
    FlrW cw;
    flr_cart_weights(W, g.cph, g.sph, cw);
    double sum = 0.0;
#pragma unroll 1
    for (int j = 0; j < 4; ++j) {
        Marker sp;
        flr_ring_point(rg, zl, j, sp.x, sp.y, sp.z);
        StepGeom gj[1];
        step_geometry(sp, gj[0]);
        const int ej = locate_any(P.f, gj[0].R, sp.z);
        double cj = 0.0;
        if (ej >= 0) {
            const double *tile = P.f.tiles + (size_t)ej * P.f.tile_stride;
            const Quad hd = ldq(tile);
            const double se = hd.c;
            const double xi[1] = {__dmul_rn(__dsub_rn(gj[0].R, hd.a), se)}, eta[1] = {__dmul_rn(__dsub_rn(sp.z, hd.b), se)};
            PertF pf[1];
            pf[0].ER = pf[0].EP = pf[0].EZ = pf[0].BR = pf[0].BP = pf[0].BZ = pf[0].gR = pf[0].gP = pf[0].gZ = pf[0].dT = 0.0;
            pert_fields<1, false>(P, tile, xi, eta, gj, se, pf);
            cj = flr_fold(pf[0], gj[0].cph, gj[0].sph, cw);
        }
        sum = j == 0 ? cj : __dadd_rn(sum, cj);
    }
    return __dmul_rn(0.25, sum);
}

// The perturbed fields of a ring point (its own cylindrical frame, cos / sin of its phi = cj, sj) as ten Cartesian
// components (E, B1, grad B1par, dB1par/dt), and the quarter sums of those rotated into the marker's frame (Eq. 14).
__device__ __forceinline__ void flr_cart_fields(const PertF &pf, double cj, double sj, double (&c)[10]) {
    c[0] = M3DK_FMA(pf.ER, cj, -__dmul_rn(pf.EP, sj)); c[1] = M3DK_FMA(pf.ER, sj, __dmul_rn(pf.EP, cj)); c[2] = pf.EZ;
    c[3] = M3DK_FMA(pf.BR, cj, -__dmul_rn(pf.BP, sj)); c[4] = M3DK_FMA(pf.BR, sj, __dmul_rn(pf.BP, cj)); c[5] = pf.BZ;
    c[6] = M3DK_FMA(pf.gR, cj, -__dmul_rn(pf.gP, sj)); c[7] = M3DK_FMA(pf.gR, sj, __dmul_rn(pf.gP, cj)); c[8] = pf.gZ;
    c[9] = pf.dT;
}
__device__ __forceinline__ void flr_avg_finish(const double (&t)[10], double c, double sn, PertF &out) {
    out.ER = __dmul_rn(0.25, M3DK_FMA(t[0], c, __dmul_rn(t[1], sn))); out.EP = __dmul_rn(0.25, M3DK_FMA(t[1], c, -__dmul_rn(t[0], sn)));
    out.EZ = __dmul_rn(0.25, t[2]);
    out.BR = __dmul_rn(0.25, M3DK_FMA(t[3], c, __dmul_rn(t[4], sn))); out.BP = __dmul_rn(0.25, M3DK_FMA(t[4], c, -__dmul_rn(t[3], sn)));
    out.BZ = __dmul_rn(0.25, t[5]);
    out.gR = __dmul_rn(0.25, M3DK_FMA(t[6], c, __dmul_rn(t[7], sn))); out.gP = __dmul_rn(0.25, M3DK_FMA(t[7], c, -__dmul_rn(t[6], sn)));
    out.gZ = __dmul_rn(0.25, t[8]);
    out.dT = __dmul_rn(0.25, t[9]);
}

// Gyro-averaged perturbed fields of one marker in its own cylindrical frame (mode 3: non-linear trajectories in the
// averaged fields): quarter sum over the ring points of the vectors in Cartesian components (Eq. 14), each
// point searched and evaluated on its own element's tile (global memory); a point outside the mesh contributes zero.
__device__ __forceinline__ void flr_avg_fields(const PushParams &P, const EqOut &f, const StepGeom &g, double zl, double mu,
                                               PertF &out) {
    FlrRing rg;
    flr_ring(P, f, g, mu, rg);
    double Ex = 0.0, Ey = 0.0, Ez = 0.0, Bx = 0.0, By = 0.0, Bz = 0.0, Gx = 0.0, Gy = 0.0, Gz = 0.0, dT = 0.0;
#pragma unroll 1
    for (int j = 0; j < 4; ++j) {
        Marker sp;
        flr_ring_point(rg, zl, j, sp.x, sp.y, sp.z);
        StepGeom gj[1];
        step_geometry(sp, gj[0]);
        const int ej = locate_any(P.f, gj[0].R, sp.z);
        if (ej < 0) continue;
        const double *tile = P.f.tiles + (size_t)ej * P.f.tile_stride;
        const Quad hd = ldq(tile);
        const double se = hd.c;
        const double xi[1] = {__dmul_rn(__dsub_rn(gj[0].R, hd.a), se)}, eta[1] = {__dmul_rn(__dsub_rn(sp.z, hd.b), se)};
        PertF pf[1];
        pf[0].ER = pf[0].EP = pf[0].EZ = pf[0].BR = pf[0].BP = pf[0].BZ = pf[0].gR = pf[0].gP = pf[0].gZ = pf[0].dT = 0.0;
        pert_fields<1, false>(P, tile, xi, eta, gj, se, pf);
        double c10[10];
        flr_cart_fields(pf[0], gj[0].cph, gj[0].sph, c10);
        Ex = __dadd_rn(Ex, c10[0]); Ey = __dadd_rn(Ey, c10[1]); Ez = __dadd_rn(Ez, c10[2]);
        Bx = __dadd_rn(Bx, c10[3]); By = __dadd_rn(By, c10[4]); Bz = __dadd_rn(Bz, c10[5]);
        Gx = __dadd_rn(Gx, c10[6]); Gy = __dadd_rn(Gy, c10[7]); Gz = __dadd_rn(Gz, c10[8]);
        dT = __dadd_rn(dT, c10[9]);
    }
    const double sum10[10] = {Ex, Ey, Ez, Bx, By, Bz, Gx, Gy, Gz, dT};
    flr_avg_finish(sum10, g.cph, g.sph, out);
}

// Mode 3 through the ring stream: the same average from the ten Cartesian components that ring_items_kernel<.., true> has
// stored for the four ring points of the marker in slot `slot` (zeros for a point outside the mesh), summed in the same
// order as flr_avg_fields.
__device__ __forceinline__ void flr_avg_from_stream(const PushParams &P, const StepGeom &g, long slot, PertF &out) {
    double sum10[10];
#pragma unroll
    for (int k = 0; k < 10; ++k) sum10[k] = 0.0;
#pragma unroll
    for (int j = 0; j < 4; ++j) {
        const double *a = P.fl.avg + kAvgDoubles * (4 * slot + j);
        double c[12];
        ldrec256(a, c[0], c[1], c[2], c[3]); ldrec256(a + 4, c[4], c[5], c[6], c[7]); ldrec256(a + 8, c[8], c[9], c[10], c[11]);
#pragma unroll
        for (int k = 0; k < 10; ++k) sum10[k] = __dadd_rn(sum10[k], c[k]);
    }
    flr_avg_finish(sum10, g.cph, g.sph, out);
}

// kFlr = 2: emit the four ring points of the marker in output slot `slot` into the ring stream (positions, flagged live)
// and the marker's weights.  Their elements are found by ring_key_kernel, one thread per ring point: four searches and
// four returned atomics in a row inside the push would serialise eight L2 round trips per marker.
__device__ __forceinline__ void flr_emit(const PushParams &P, const EqOut &f, const StepGeom &g, double zl, double mu,
                                         const PertW &W, long slot) {
    FlrRing rg;
    flr_ring(P, f, g, mu, rg);
    FlrW cw;
    flr_cart_weights(W, g.cph, g.sph, cw);
    double *wt = P.fl.wts + 10 * slot;
    wt[0] = cw.aEx; wt[1] = cw.aEy; wt[2] = cw.aEz; wt[3] = cw.bBx; wt[4] = cw.bBy; wt[5] = cw.bBz;
    wt[6] = cw.gGx; wt[7] = cw.gGy; wt[8] = cw.gGz; wt[9] = cw.dT;
#pragma unroll
    for (int j = 0; j < 4; ++j) {
        double x, y, z;
        flr_ring_point(rg, zl, j, x, y, z);
        strec256(P.fl.ring + 4 * (4 * slot + j), x, y, z, 1.0);
    }
}

// element of every ring point (the key of the ring ordering; n_elems = outside the mesh, -1 = the slot of a lost marker)
// and its rank inside the key, from the ring histogram (warp-aggregated atomics)
__global__ void __launch_bounds__(256, 6) ring_key_kernel(const __grid_constant__ FieldParams f, long n4,
                                                       const double *__restrict__ ring, int *__restrict__ rkey,
                                                       int *__restrict__ rrank, int *__restrict__ rhist, unsigned cstride) {
    // ring points are in the order of the markers' elements, so neighbouring blocks would hit the same few histogram bins
    // at the same time: block b takes chunk (b * cstride) mod gridDim.x (cstride coprime with the grid)
    const long i = (long)(((unsigned long long)blockIdx.x * cstride) % gridDim.x) * blockDim.x + threadIdx.x;
    bool on = i < n4;
    int key = 0;
    if (on) {
        Marker sp;
        double live;
        ldrec256(ring + 4 * i, sp.x, sp.y, sp.z, live);
        if (live < 0.0) { rkey[i] = -1; on = false; }
        else {
            StepGeom gj;
            step_geometry(sp, gj);                        // the same R as the evaluation will see
            const int ej = locate_any(f, gj.R, sp.z);
            key = ej < 0 ? f.n_elems : ej;
            rkey[i] = key;
        }
    }
    const unsigned live_mask = __ballot_sync(0xffffffffu, on);
    if (on) {
        const unsigned peers = __match_any_sync(live_mask, key);
        const int lane = threadIdx.x & 31, leader = __ffs(peers) - 1;
        int base = 0;
        if (lane == leader) base = atomicAdd(rhist + key, __popc(peers));
        base = __shfl_sync(peers, base, leader);
        rrank[i] = base + __popc(peers & ((1u << lane) - 1u));
    }
}

// ---- the same step in the non-linear trajectory mode (mode 1: PAPER.md:108, :130; reading G21) ------------------------
// All perturbed fields are needed BEFORE the velocity update (the marker moves in the total fields), so they are
// accumulated per marker (10 values) and the folding trick of the linear mode does not apply; B1_phi (quad 3) enters.
// kFlr: 0 fields at the marker; 1 every lane gathers its four ring points (flr_avg_fields); 2 the averages come from the
// ring stream (flr_avg_from_stream: ring points emitted by flr_emit_nl, evaluated by ring_items_kernel<.., true>)
template <int R, bool kHist, bool kSmem, class IO, bool kPost = false, int kFlr = 0>
__device__ __forceinline__ void step_R_nl(const PushParams &P, const IO &io, const double *__restrict__ tile,
                                          const long (&mi)[R], const long (&mo)[R], const bool (&on)[R], double (&Rn)[R],
                                          double (&Zn)[R]) {
    Marker s[R];
    StepGeom g[R];
#pragma unroll
    for (int r = 0; r < R; ++r) {
        if (on[r]) { io.load_pos(mi[r], s[r].x, s[r].y, s[r].z, s[r].w); io.load_vel(mi[r], s[r].vx, s[r].vy, s[r].vz, s[r].mu); }
        else { s[r].x = 1.0; s[r].y = 0.0; s[r].z = 0.0; s[r].w = 0.0; s[r].vx = s[r].vy = s[r].vz = 0.0; s[r].mu = 0.0; }
    }
    const Quad hd = ldq_t<kSmem>(tile);
    const double Rc = hd.a, Zc = hd.b, se = hd.c;
    double xi[R], eta[R];
#pragma unroll
    for (int r = 0; r < R; ++r) {
        step_geometry(s[r], g[r]);
        xi[r] = __dmul_rn(__dsub_rn(g[r].R, Rc), se); eta[r] = __dmul_rn(__dsub_rn(s[r].z, Zc), se);
    }
    double v[R][4], dx[R][4], de[R][4];
    Ring ring;
    ring_fill<kSmem>(ring, tile + kTileHeader);
    quad_vd<R, kSmem>(tile + kTileHeader, tile + kTileHeader, ring, xi, eta, v, dx, de);   // (psi0, |B|0, F0, kappa)
    EqOut f[R];
    PertF pf[R];
#pragma unroll
    for (int r = 0; r < R; ++r) {
        f[r].psi_R = __dmul_rn(dx[r][0], se); f[r].psi_Z = __dmul_rn(de[r][0], se);
        f[r].Bm = v[r][1]; f[r].Bm_R = __dmul_rn(dx[r][1], se); f[r].Bm_Z = __dmul_rn(de[r][1], se);
        f[r].F = v[r][2]; f[r].kappa = v[r][3];
        pf[r].ER = pf[r].EP = pf[r].EZ = pf[r].BR = pf[r].BP = pf[r].BZ = pf[r].gR = pf[r].gP = pf[r].gZ = pf[r].dT = 0.0;
    }
    if constexpr (kFlr == 2) {      // mode 3, ordered with a ring stream
#pragma unroll
        for (int r = 0; r < R; ++r)
            if (on[r]) flr_avg_from_stream(P, g[r], mo[r], pf[r]);
    } else if constexpr (kFlr == 1) {   // mode 3: the gyro-averaged perturbed fields replace the fields at the marker
#pragma unroll
        for (int r = 0; r < R; ++r)
            if (P.f.n_modes > 0) flr_avg_fields(P, f[r], g[r], s[r].z, s[r].mu, pf[r]);
    } else {
        pert_fields<R, kSmem>(P, tile, xi, eta, g, se, pf);
    }
#pragma unroll
    for (int r = 0; r < R; ++r) {
        const double w_old = s[r].w;
        double wdot;
        push_eq_nl(P, g[r], f[r], pf[r], s[r], wdot);
        // Eq. (8) with (1 - w) kept, explicit on the staggered grid (readings G9, G21)
        if (P.f.n_modes > 0) s[r].w = M3DK_FMA(P.dt, __dmul_rn(__dsub_rn(1.0, w_old), wdot), w_old);
        Rn[r] = m3dk_sqrt(M3DK_FMA(s[r].x, s[r].x, __dmul_rn(s[r].y, s[r].y)));
        Zn[r] = s[r].z;
    }
    int key[R];
    FastRec rec[kPost ? 1 : R];
    if constexpr (!kPost) {
#pragma unroll
        for (int r = 0; r < R; ++r) rec[r] = locate_first(P.f.fast, Rn[r], Zn[r]);   // all first records in flight together
    }
#pragma unroll
    for (int r = 0; r < R; ++r) {
        int ne = -1;
        if (on[r]) {
            io.store_pos(mo[r], s[r].x, s[r].y, s[r].z, s[r].w);
            io.store_vel(mo[r], s[r].vx, s[r].vy, s[r].vz, s[r].mu);
            if (P.f.n_modes > 0) io.store_w(mo[r], s[r].w);
            if constexpr (!kPost) {
                ne = locate_finish(P.f, rec[r], Rn[r], Zn[r]);
                io.store_key(mo[r], ne);
            }
        }
        key[r] = ne < 0 ? P.f.n_elems : ne;
    }
    if constexpr (kPost) io.stage_next();
    if (kHist && !kPost) {
        unsigned peers[R];
        int base[R];
        hist_issue<R>(P.hist, key, on, peers, base);
        rank_finish<R>(P.rank, mo, on, peers, base);
    }
}

// Mode 3 through the ring stream, first pass: the equilibrium field at x_l and the four ring points of every marker of the
// item into the ring stream (slot = the marker's OUTPUT slot, where the second pass, step_R_nl<.., 2>, reads the averages);
// nothing else is written.
template <int R, bool kSmem, class IO>
__device__ __forceinline__ void flr_emit_nl(const PushParams &P, const IO &io, const double *__restrict__ tile,
                                            const long (&mi)[R], const long (&mo)[R], const bool (&on)[R]) {
    Marker s[R];
    StepGeom g[R];
#pragma unroll
    for (int r = 0; r < R; ++r) {
        if (on[r]) { io.load_pos(mi[r], s[r].x, s[r].y, s[r].z, s[r].w); io.load_vel(mi[r], s[r].vx, s[r].vy, s[r].vz, s[r].mu); }
        else { s[r].x = 1.0; s[r].y = 0.0; s[r].z = 0.0; s[r].w = 0.0; s[r].vx = s[r].vy = s[r].vz = 0.0; s[r].mu = 0.0; }
    }
    const Quad hd = ldq_t<kSmem>(tile);
    const double Rc = hd.a, Zc = hd.b, se = hd.c;
    double xi[R], eta[R];
#pragma unroll
    for (int r = 0; r < R; ++r) {
        step_geometry(s[r], g[r]);
        xi[r] = __dmul_rn(__dsub_rn(g[r].R, Rc), se); eta[r] = __dmul_rn(__dsub_rn(s[r].z, Zc), se);
    }
    double v[R][4], dx[R][4], de[R][4];
    Ring ring;
    ring_fill<kSmem>(ring, tile + kTileHeader);
    quad_vd<R, kSmem>(tile + kTileHeader, tile + kTileHeader, ring, xi, eta, v, dx, de);   // (psi0, |B|0, F0, kappa)
#pragma unroll
    for (int r = 0; r < R; ++r) {
        if (!on[r]) continue;
        EqOut f;
        f.psi_R = __dmul_rn(dx[r][0], se); f.psi_Z = __dmul_rn(de[r][0], se);
        f.Bm = v[r][1]; f.Bm_R = __dmul_rn(dx[r][1], se); f.Bm_Z = __dmul_rn(de[r][1], se);
        f.F = v[r][2]; f.kappa = v[r][3];
        FlrRing rg;
        flr_ring(P, f, g[r], s[r].mu, rg);
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            double x, y, z;
            flr_ring_point(rg, s[r].z, j, x, y, z);
            strec256(P.fl.ring + 4 * (4 * mo[r] + j), x, y, z, 1.0);
        }
    }
}

// ---- generic push: one marker per thread, any marker order (every thread gathers its own element's tile) ------------
// The caller's SoA arrays in place: sort_interval = 0, i.e. no sort workspace.
template <int kMode>
__global__ void __launch_bounds__(128) push_generic_kernel(const __grid_constant__ PushParams P) {
    const long i = (long)blockIdx.x * blockDim.x + threadIdx.x;
    const int e = i < P.n ? P.a.elem[i] : -1;
    const long m[1] = {i};
    const bool on[1] = {e >= 0};             // lost markers are frozen (G12)
    // the tile loads may be speculated above the `on` tests: e is clamped to a valid element for addressing
    const double *tile = P.f.tiles + (size_t)max(e, 0) * P.f.tile_stride;
    if (__any_sync(0xffffffffu, on[0])) {
        double Rn[1], Zn[1];
        const SoAIO io{P.a, P.f.n_elems};
        if (kMode == 1 || kMode == 4) step_R_nl<1, false, false, SoAIO, false, kMode == 4 ? 1 : 0>(P, io, tile, m, m, on, Rn, Zn);
        else step_R<1, false, false, SoAIO, kMode == 2 ? 1 : 0>(P, io, tile, m, m, on, Rn, Zn);
    }
}

// ---- tile staging: one bulk copy (TMA, cp.async.bulk) per item into the warp's double buffer, mbarrier completion --
__device__ __forceinline__ unsigned smem_u32(const void *p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(unsigned bar, unsigned count = 1) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_arrive(unsigned bar, unsigned count = 1) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void tile_copy_issue(unsigned dst, const double *src, unsigned bytes, unsigned bar) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(dst), "l"(src), "r"(bytes), "r"(bar) : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned bar, unsigned parity) {
    asm volatile("{\n .reg .pred p;\n WAIT_%=:\n mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n @!p bra WAIT_%=;\n}"
                 ::"r"(bar), "r"(parity) : "memory");
}

// ---- element-ordered push: the marker stream is sorted by element and cut into work items --------------------------
// A work item is up to kItemMarkers = 32 kItemR consecutive markers of ONE element; a warp takes an item, every lane up to
// kItemR of its markers (slots lane, lane + 32, ...).  The element's coefficient tile is staged in shared memory by one
// bulk copy per item (double-buffered per warp: the next item's tile travels while this one computes), and every
// coefficient read is a broadcast LDS that feeds kItemR markers per lane.  Items are handed out by a ticket counter after
// a warp's first three.  Items of the pseudo-element n_elems hold the lost markers: frozen, they only enter the histogram.
// kR = 2: the items of up to 64 markers; kR = 1: the small items (a remainder of 1..32 markers of an element).
// kMode: 0 linear, 1 non-linear, 2 FLR with per-lane ring gathers, 3 FLR emitting the ring stream, 4 non-linear + FLR with
// per-lane gathers, 5 / 6 the two passes of non-linear + FLR through the ring stream (emit; step with the stream's averages).
template <bool kHist, int kMode, int kR>
__global__ void __launch_bounds__(kPushThreads, kR == 1 ? M3DK_PUSH_MINBLOCKS + 1 : M3DK_PUSH_MINBLOCKS) push_items_kernel(const __grid_constant__ PushParams P) {
    extern __shared__ __align__(128) unsigned char smem_raw[];
    constexpr int kWarps = kPushThreads / 32;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int stride_d = P.f.tile_stride;
    const unsigned tile_bytes = (unsigned)stride_d * 8u;
    double *const tbuf = reinterpret_cast<double *>(smem_raw) + (size_t)warp * 2 * stride_d;
    unsigned long long *const bars = reinterpret_cast<unsigned long long *>(smem_raw + (size_t)kWarps * 2 * tile_bytes) + warp * 2;
    const unsigned bar0 = smem_u32(bars), buf0 = smem_u32(tbuf);
    if (lane == 0) {
        mbar_init(bar0); mbar_init(bar0 + 8);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncwarp();
    const int total = *P.n_items;
    const int stride = gridDim.x * kWarps;
    // Software pipeline over this warp's items:
    //   item descriptors are read two items ahead, the order entries (which record goes to which slot) one item ahead,
    //   and at the start of an item the NEXT item's records are prefetched into L2 and its tile copy is issued,
    // so that an item starts with its tile in shared memory and its records one L2 hit away.
    const int4 none = make_int4(P.f.n_elems, 0, 0, 0);
    // The first three items of a warp are fixed (items it, it + stride, it + 2 stride); every further one is drawn from a
    // ticket counter one item ahead of its descriptor read, so that no warp idles while another still has a queue.
    int it = blockIdx.x * kWarps + warp, it1 = it + stride, it2 = it + 2 * stride;
    int4 w0 = it < total ? __ldg(P.items + it) : none;
    int4 w1 = it1 < total ? __ldg(P.items + it1) : none;
    int src0[kR], src1[kR];
#pragma unroll
    for (int r = 0; r < kR; ++r) {
        src0[r] = 32 * r + lane < w0.z ? P.rc.order[w0.y + 32 * r + lane].x : 0;
        src1[r] = 32 * r + lane < w1.z ? P.rc.order[w1.y + 32 * r + lane].x : 0;
    }
    unsigned b = 0, phase = 0;   // buffer of the current item; bit k of phase: parity to wait for on buffer k
    if (w0.x < P.f.n_elems && lane == 0) tile_copy_issue(buf0, P.f.tiles + (size_t)w0.x * stride_d, tile_bytes, bar0);
    while (it < total) {
        const int e = w0.x, start = w0.y, count = w0.z;   // (element, first slot, count, -)
        const int4 w2 = it2 < total ? __ldg(P.items + it2) : none;
        int ticket = 0;
        if (lane == 0) ticket = atomicAdd(P.ticket, 1);
        __syncwarp();                                  // every lane has finished reading buffer b ^ 1 (previous item)
        if (w1.x < P.f.n_elems && lane == 0)
            tile_copy_issue(buf0 + (b ^ 1) * tile_bytes, P.f.tiles + (size_t)w1.x * stride_d, tile_bytes, bar0 + (b ^ 1) * 8);
        int src2[kR];
#pragma unroll
        for (int r = 0; r < kR; ++r) {
            if (32 * r + lane < w1.z) {
                const double *rp = P.rc.in + (size_t)kRecDoubles * src1[r];
                asm volatile("prefetch.global.L2 [%0];" ::"l"(rp));
            }
            src2[r] = 32 * r + lane < w2.z ? P.rc.order[w2.y + 32 * r + lane].x : 0;
        }
        long mi[kR], mo[kR];
        bool on[kR];
#pragma unroll
        for (int r = 0; r < kR; ++r) { mo[r] = (long)start + 32 * r + lane; on[r] = 32 * r + lane < count; mi[r] = src0[r]; }
        const RecIO io{P.rc.in, P.rc.out, P.rc.key, P.f.n_elems};
        if (kMode == 5 && e >= P.f.n_elems) {          // emit pass of mode 3: the slots of lost markers carry no ring
#pragma unroll
            for (int r = 0; r < kR; ++r)
                if (on[r])
                    for (int j = 0; j < 4; ++j) strec256(P.fl.ring + 4 * (4 * mo[r] + j), 0.0, 0.0, 0.0, -1.0);
        } else if (e >= P.f.n_elems) {                 // lost markers: frozen (G12), moved along and counted for the next sort
            int key[kR];
#pragma unroll
            for (int r = 0; r < kR; ++r) {
                key[r] = P.f.n_elems;
                if (on[r]) {
                    double a0, a1, a2, a3, b0, b1, b2, b3;
                    io.load_pos(mi[r], a0, a1, a2, a3); io.load_vel(mi[r], b0, b1, b2, b3);
                    io.store_pos(mo[r], a0, a1, a2, a3); io.store_vel(mo[r], b0, b1, b2, b3);
                    io.store_key(mo[r], -1);
                    if (kMode == 3)                      // no ring for a lost marker: its slot is skipped by the ring kernels
                        for (int j = 0; j < 4; ++j) strec256(P.fl.ring + 4 * (4 * mo[r] + j), 0.0, 0.0, 0.0, -1.0);
                }
            }
            if (kHist) {
                unsigned peers[kR];
                int base[kR];
                hist_issue<kR>(P.hist, key, on, peers, base);
                rank_finish<kR>(P.rank, mo, on, peers, base);
            }
        } else {
            mbar_wait(bar0 + b * 8, (phase >> b) & 1u);
            phase ^= 1u << b;
            double Rn[kR], Zn[kR];
            if (kMode == 5) flr_emit_nl<kR, true, RecIO>(P, io, tbuf + (size_t)b * stride_d, mi, mo, on);
            else if (kMode == 1 || kMode == 4 || kMode == 6)
                step_R_nl<kR, kHist, true, RecIO, false, kMode == 4 ? 1 : (kMode == 6 ? 2 : 0)>(P, io, tbuf + (size_t)b * stride_d, mi, mo, on, Rn, Zn);
            else step_R<kR, kHist, true, RecIO, kMode == 2 ? 1 : (kMode == 3 ? 2 : 0)>(P, io, tbuf + (size_t)b * stride_d, mi, mo, on, Rn, Zn);
        }
        b ^= 1;
        it = it1; it1 = it2; it2 = 3 * stride + __shfl_sync(0xffffffffu, ticket, 0);
        w0 = w1; w1 = w2;
#pragma unroll
        for (int r = 0; r < kR; ++r) { src0[r] = src1[r]; src1[r] = src2[r]; }
    }
}


// ---- mode 2, ordered: evaluation of the ring stream ---------------------------------------------------------------------
// The ring points emitted by push_items_kernel<.., 3, ..> are ordered by THEIR element (histogram fused into the emit,
// scan + work-item cut + placement: the kernels of the marker ordering) and a warp takes a ring item: up to 64 ring points
// of one element, kR per lane, the element's tile staged in shared memory by a bulk copy (double-buffered, items by
// ticket: the machinery of push_items_kernel).  A lane gathers its points (32 B) and the weights of the markers that own
// them (80 B), evaluates all perturbed polynomials at the points (pert_fields with broadcast coefficient reads shared by
// the lane's points) and stores the scalar contribution c_j of each point.
// kAvg (mode 3): no weights; the ten Cartesian components of the fields at the point are stored (12 doubles per point: three
// full sectors) for the second pass of the push, zeros for a point outside the mesh.
template <int kR, bool kAvg>
__global__ void __launch_bounds__(kPushThreads, kR == 1 ? M3DK_PUSH_MINBLOCKS + 1 : M3DK_PUSH_MINBLOCKS) ring_items_kernel(const __grid_constant__ PushParams P) {
    extern __shared__ __align__(128) unsigned char smem_raw[];
    constexpr int kWarps = kPushThreads / 32;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int stride_d = P.f.tile_stride;
    const unsigned tile_bytes = (unsigned)stride_d * 8u;
    double *const tbuf = reinterpret_cast<double *>(smem_raw) + (size_t)warp * 2 * stride_d;
    unsigned long long *const bars = reinterpret_cast<unsigned long long *>(smem_raw + (size_t)kWarps * 2 * tile_bytes) + warp * 2;
    const unsigned bar0 = smem_u32(bars), buf0 = smem_u32(tbuf);
    if (lane == 0) {
        mbar_init(bar0); mbar_init(bar0 + 8);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncwarp();
    const int total = *P.n_items;
    const int stride = gridDim.x * kWarps;
    const int4 none = make_int4(P.f.n_elems, 0, 0, 0);
    int it = blockIdx.x * kWarps + warp, it1 = it + stride, it2 = it + 2 * stride;
    int4 w0 = it < total ? __ldg(P.items + it) : none;
    int4 w1 = it1 < total ? __ldg(P.items + it1) : none;
    unsigned b = 0, phase = 0;
    if (w0.x < P.f.n_elems && lane == 0) tile_copy_issue(buf0, P.f.tiles + (size_t)w0.x * stride_d, tile_bytes, bar0);
    // the ring points of an item are reached through the order list, and the weights through the point's owner: both
    // indices are read one item ahead and what they point at is prefetched into L2 while the current item computes
    int idx0[kR], idx1[kR];
#pragma unroll
    for (int r = 0; r < kR; ++r) {
        idx0[r] = 32 * r + lane < w0.z ? P.fl.rorder[w0.y + 32 * r + lane] : 0;
        idx1[r] = 32 * r + lane < w1.z ? P.fl.rorder[w1.y + 32 * r + lane] : 0;
    }
    while (it < total) {
        const int e = w0.x, start = w0.y, count = w0.z;
        const int4 w2 = it2 < total ? __ldg(P.items + it2) : none;
        int ticket = 0;
        if (lane == 0) ticket = atomicAdd(P.ticket, 1);
        __syncwarp();                                  // every lane has finished reading buffer b ^ 1 (previous item)
        if (w1.x < P.f.n_elems && lane == 0)
            tile_copy_issue(buf0 + (b ^ 1) * tile_bytes, P.f.tiles + (size_t)w1.x * stride_d, tile_bytes, bar0 + (b ^ 1) * 8);
        long idx[kR];
        bool on[kR];
        Marker sp[kR];
        FlrW cw[kR];
        int idx2[kR];
#pragma unroll
        for (int r = 0; r < kR; ++r) {
            if (32 * r + lane < w1.z) {
                asm volatile("prefetch.global.L2 [%0];" ::"l"(P.fl.ring + 4 * (size_t)idx1[r]));
                if (!kAvg) {
                    const double *wp = P.fl.wts + 10 * (size_t)(idx1[r] >> 2);
                    asm volatile("prefetch.global.L2 [%0];" ::"l"(wp));
                    asm volatile("prefetch.global.L2 [%0];" ::"l"(wp + 9));
                }
            }
            idx2[r] = 32 * r + lane < w2.z ? P.fl.rorder[w2.y + 32 * r + lane] : 0;
        }
#pragma unroll
        for (int r = 0; r < kR; ++r) {
            on[r] = 32 * r + lane < count;
            idx[r] = on[r] ? idx0[r] : 0;
            double pad;
            if (on[r]) ldrec256(P.fl.ring + 4 * idx[r], sp[r].x, sp[r].y, sp[r].z, pad);
            else { sp[r].x = 1.0; sp[r].y = 0.0; sp[r].z = 0.0; }
        }
        if (e < P.f.n_elems) {                          // (ring points outside the mesh contribute zero: written by the placement)
            mbar_wait(bar0 + b * 8, (phase >> b) & 1u);
            phase ^= 1u << b;
            const double *tile = tbuf + (size_t)b * stride_d;
            const Quad hd = ldq_t<true>(tile);
            const double se = hd.c;
            StepGeom g[kR];
            double xi[kR], eta[kR];
            PertF pf[kR];
#pragma unroll
            for (int r = 0; r < kR; ++r) {
                step_geometry(sp[r], g[r]);
                xi[r] = __dmul_rn(__dsub_rn(g[r].R, hd.a), se); eta[r] = __dmul_rn(__dsub_rn(sp[r].z, hd.b), se);
                pf[r].ER = pf[r].EP = pf[r].EZ = pf[r].BR = pf[r].BP = pf[r].BZ = pf[r].gR = pf[r].gP = pf[r].gZ = pf[r].dT = 0.0;
            }
            pert_fields<kR, true>(P, tile, xi, eta, g, se, pf);
#pragma unroll
            for (int r = 0; r < kR; ++r)
                if (kAvg) {
                    if (on[r]) {
                        double c10[10];
                        flr_cart_fields(pf[r], g[r].cph, g[r].sph, c10);
                        double *a = P.fl.avg + kAvgDoubles * idx[r];
                        strec256(a, c10[0], c10[1], c10[2], c10[3]); strec256(a + 4, c10[4], c10[5], c10[6], c10[7]);
                        strec256(a + 8, c10[8], c10[9], 0.0, 0.0);
                    }
                } else if (on[r]) {
                    const double *wt = P.fl.wts + 10 * (idx[r] >> 2);
                    cw[r].aEx = wt[0]; cw[r].aEy = wt[1]; cw[r].aEz = wt[2]; cw[r].bBx = wt[3]; cw[r].bBy = wt[4];
                    cw[r].bBz = wt[5]; cw[r].gGx = wt[6]; cw[r].gGy = wt[7]; cw[r].gGz = wt[8]; cw[r].dT = wt[9];
                    P.fl.contrib[idx[r]] = flr_fold(pf[r], g[r].cph, g[r].sph, cw[r]);
                }
        }
        else if (kAvg) {                                // outside the mesh: the point contributes zero to every average
#pragma unroll
            for (int r = 0; r < kR; ++r)
                if (on[r]) {
                    double *a = P.fl.avg + kAvgDoubles * idx[r];
                    strec256(a, 0.0, 0.0, 0.0, 0.0); strec256(a + 4, 0.0, 0.0, 0.0, 0.0); strec256(a + 8, 0.0, 0.0, 0.0, 0.0);
                }
        }
        b ^= 1;
        it = it1; it1 = it2; it2 = 3 * stride + __shfl_sync(0xffffffffu, ticket, 0);
        w0 = w1; w1 = w2;
#pragma unroll
        for (int r = 0; r < kR; ++r) { idx0[r] = idx1[r]; idx1[r] = idx2[r]; }
    }
}

// ---- element-ordered push with asynchronous staging (modes 0 and 1) ---------------------------------------------------
// The same work decomposition as push_items_kernel (a warp takes a work item of one element, a lane up to kR of its
// markers, tile staged by one bulk copy per item, items drawn from a ticket counter), but no warp ever waits for L2 or HBM
// inside an item: everything an item needs from memory is requested one item ahead and lands in shared memory meanwhile.
//   records   gathered with cp.async (4 x 16 B per marker) into the warp's record box while the previous item computes;
//   search    at the end of item k the lane writes the new (R, Z) of its markers to shared memory and requests the 64-byte
//             record of their search bucket with cp.async; the edge tests, the key store and the histogram atomics of
//             item k run at the end of item k + 1, the returned ranks are stored at the end of item k + 2.
// cp.async groups are committed in the order ... records(k + 1), search(k) ...; both waits allow the most recent group
// to be pending (wait_group 1).
__device__ __forceinline__ void cp_async16(unsigned dst, const void *src) {
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(dst), "l"(src) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N>
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }

// record box of the staged item: [4][32 R] double2 = (x, y), (z, w), (vx, vy), (vz, mu) of the item's slots: every access of
// a warp is conflict-free, and a lane only ever touches the slots of its own markers
template <int R>
struct AsyncIO {
    double2 *box;
    double *out;
    const double *in;
    const int2 *ord_next;   // order entries (src, id) of the NEXT item's slots, src = -1: none (shared memory)
    static constexpr int n = 32 * R;
    __device__ __forceinline__ void load_pos(long i, double &x, double &y, double &z, double &w) const {
        const double2 a = box[i], b = box[n + i];
        x = a.x; y = a.y; z = b.x; w = b.y;
    }
    __device__ __forceinline__ void load_vel(long i, double &vx, double &vy, double &vz, double &mu) const {
        const double2 a = box[2 * n + i], b = box[3 * n + i];
        vx = a.x; vy = a.y; vz = b.x; mu = b.y;
    }
    __device__ __forceinline__ void store_pos(long o, double x, double y, double z, double w_old) const {
        strec256(out + kRecDoubles * o, x, y, z, w_old);
    }
    __device__ __forceinline__ void store_vel(long o, double vx, double vy, double vz, double mu) const {
        strec256(out + kRecDoubles * o + 4, vx, vy, vz, mu);
    }
    __device__ __forceinline__ void store_w(long o, double w) const { out[kRecDoubles * o + 3] = w; }
    // this lane has consumed its records: the next item's may land in the same slots
    __device__ __forceinline__ void stage_next() const {
        const int lane = threadIdx.x & 31;
        const unsigned b0 = smem_u32(box) + lane * 16u;
#pragma unroll
        for (int r = 0; r < R; ++r) {
            const int src = ord_next[32 * r + lane].x;
            if (src >= 0) {
                const double *g = in + (size_t)kRecDoubles * src;
#pragma unroll
                for (int q = 0; q < 4; ++q) cp_async16(b0 + (unsigned)(q * n + 32 * r) * 16u, g + 2 * q);
            }
        }
        cp_async_commit();
    }
};

template <bool kHist, int kMode, int kR>
__global__ void __launch_bounds__(kPushThreads, kR == 1 ? M3DK_PUSH_MINBLOCKS + 1 : M3DK_PUSH_MINBLOCKS) push_async_kernel(const __grid_constant__ PushParams P) {
    extern __shared__ __align__(128) unsigned char smem_raw[];
    constexpr int kWarps = kPushThreads / 32;
    constexpr int kSlots = 32 * kR;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int stride_d = P.f.tile_stride;
    const unsigned tile_bytes = (unsigned)stride_d * 8u;
    // per warp: record box | new (R, Z) | search records | order entries [2] | descriptors [16] | 2 mbarriers | tile[2]
    constexpr unsigned kBoxBytes = 4u * kSlots * 16u, kRzBytes = kSlots * 16u, kFrBytes = 4u * kSlots * 16u;
    constexpr unsigned kOrdBytes = 2u * kSlots * 8u, kDscBytes = 16u * 16u;
    constexpr unsigned kFixed = kBoxBytes + kRzBytes + kFrBytes + kOrdBytes + kDscBytes + 16u;
    const unsigned wblock = 2u * tile_bytes + kFixed;
    // the fixed-size areas come first (constant offsets from the warp's base), the two tile buffers last
    unsigned char *const wbase = smem_raw + (size_t)warp * wblock;
    unsigned char *q = wbase;
    double2 *const box = reinterpret_cast<double2 *>(q); q += kBoxBytes;
    double2 *const rz = reinterpret_cast<double2 *>(q); q += kRzBytes;
    uint4 *const fr = reinterpret_cast<uint4 *>(q); q += kFrBytes;
    int2 *const ord = reinterpret_cast<int2 *>(q); q += kOrdBytes;          // [2][kSlots]: order entries of items k + 1, k + 2
    int4 *const dsc = reinterpret_cast<int4 *>(q); q += kDscBytes;             // ring of 16 item descriptors: items k - 1 .. k + 7
    const unsigned bar0 = smem_u32(q);
    double *const tbuf = reinterpret_cast<double *>(q + 16);
    const unsigned buf0 = smem_u32(tbuf);
    if (lane == 0) {
        mbar_init(bar0); mbar_init(bar0 + 8);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    const int total = *P.n_items;
    const int n_elems = P.f.n_elems;
    const int stride = gridDim.x * kWarps;
    const int4 none = make_int4(n_elems, 0, 0, 0);
    AsyncIO<kR> io{box, P.rc.out, P.rc.in, ord};

    // ---- prologue (blocking loads, once per warp): descriptors of the first four items, order entries of the first two,
    // records and tile of the first.
    // Items 0..3 of a warp are fixed (global warp index + 0, 1, 2, 3 grid strides); every further one comes from the ticket
    // counter, four at a time: a returned atomic is waited for where it is used (a value left pending across an item is
    // spilled by the compiler, i.e. waited for at once), so one wait serves four items
    {
        const int it0 = blockIdx.x * kWarps + warp;
        if (lane < 16) {
            int4 d = none;
            const int it = it0 + lane * stride;
            if (lane < 4 && it < total) d = __ldg(P.items + it);
            dsc[lane] = d;
        }
        __syncwarp();
#pragma unroll
        for (int j = 0; j < 2; ++j) {
            const int4 d = dsc[j];
#pragma unroll
            for (int r = 0; r < kR; ++r) {
                const int i = 32 * r + lane;
                ord[j * kSlots + i] = i < d.z ? P.rc.order[d.y + i] : make_int2(-1, 0);
            }
        }
        const int4 d0 = dsc[0];
        if (d0.x < n_elems && d0.z > 0 && lane == 0) tile_copy_issue(buf0, P.f.tiles + (size_t)d0.x * stride_d, tile_bytes, bar0);
        io.stage_next();                                 // records of the first item (order slot 0)
        cp_async_commit();                               // (stands for the search group of an item before the first)
    }
    unsigned phase = 0;

    // a3 for item k - 1: edge tests on the search records fetched meanwhile, key store, histogram count (no returned value:
    // invert_kernel<true> draws the slots)
    auto search_prev = [&](int k1) {
        if (k1 < 0) return;
        const int4 d = dsc[k1 & 15];
        const int cnt = d.x < n_elems ? d.z : 0;
#pragma unroll
        for (int r = 0; r < kR; ++r) {
            const int i = 32 * r + lane;
            const bool on = i < cnt;
            int key = n_elems;
            if (on) {
                const double2 p = rz[i];
                const uint4 q0 = fr[i], q1 = fr[kSlots + i], q2 = fr[2 * kSlots + i], q3 = fr[3 * kSlots + i];
                FastRec f;
                f.a[0] = __uint_as_float(q0.x); f.a[1] = __uint_as_float(q0.y); f.a[2] = __uint_as_float(q0.z); f.a[3] = __uint_as_float(q0.w);
                f.a[4] = __uint_as_float(q1.x); f.a[5] = __uint_as_float(q1.y); f.b[0] = __uint_as_float(q1.z); f.b[1] = __uint_as_float(q1.w);
                f.b[2] = __uint_as_float(q2.x); f.b[3] = __uint_as_float(q2.y); f.b[4] = __uint_as_float(q2.z); f.b[5] = __uint_as_float(q2.w);
                f.ida = (int)q3.x; f.idb = (int)q3.y; f.next = (int)q3.z; f.pad = 0;
                const int ne = locate_finish(P.f, f, p.x, p.y);
                key = ne < 0 ? n_elems : ne;
                P.rc.key[(long)d.y + i] = key;
            }
            if (kHist && on) atomicAdd(P.hist + key, 1);
        }
    };

    int k = 0;                                           // items this warp has stepped
    for (;; ++k) {
        const unsigned b = k & 1;
        // everything requested up to one item ago has landed: the records of item k, the order entries of item k + 1, the
        // descriptor of item k + 2 (only the search records of item k - 1 may still be under way)
        cp_async_wait<1>();
        __syncwarp();                                  // lane 0's descriptor copies are visible; tile buffer b ^ 1 is free
        const int4 w0 = dsc[k & 15];                   // (element, first slot, count, -)
        if (w0.z == 0) break;                          // tickets only grow: no item left for this warp
        const int e = w0.x, start = w0.y, count = w0.z;
        {
            // requests: tile of item k + 1, order entries of item k + 2, every fourth item the descriptors of items k + 4 .. k + 7
            const int4 w1 = dsc[(k + 1) & 15], w2 = dsc[(k + 2) & 15];
            if (lane == 0 && w1.x < n_elems && w1.z > 0)
                tile_copy_issue(buf0 + (b ^ 1) * tile_bytes, P.f.tiles + (size_t)w1.x * stride_d, tile_bytes, bar0 + (b ^ 1) * 8);
            if ((k & 3) == 0 && lane < 4) {
                int tk = 0;
                if (lane == 0) tk = atomicAdd(P.ticket, 4);
                const int it = 4 * stride + __shfl_sync(0xfu, tk, 0) + lane;
                if (it < total) cp_async16(smem_u32(dsc + ((k + 4 + lane) & 15)), P.items + it);
                else dsc[(k + 4 + lane) & 15] = none;
            }
            int2 *const o2 = ord + ((k + 2) & 1) * kSlots;
#pragma unroll
            for (int r = 0; r < kR; ++r) {
                const int i = 32 * r + lane;
                if (i < w2.z) asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(smem_u32(o2 + i)), "l"(P.rc.order + w2.y + i) : "memory");
                else o2[i] = make_int2(-1, 0);
            }
            cp_async_commit();
        }
        io.ord_next = ord + ((k + 1) & 1) * kSlots;
        long mi[kR], mo[kR];
        bool on[kR];
        double Rn[kR], Zn[kR];
#pragma unroll
        for (int r = 0; r < kR; ++r) { mi[r] = 32 * r + lane; mo[r] = (long)start + 32 * r + lane; on[r] = 32 * r + lane < count; Rn[r] = 1.0; Zn[r] = 0.0; }
        if (e >= n_elems) {                            // lost markers: frozen (G12), moved along and counted for the next sort
            int key[kR];
#pragma unroll
            for (int r = 0; r < kR; ++r) {
                key[r] = n_elems;
                if (on[r]) {
                    double a0, a1, a2, a3, b0, b1, b2, b3;
                    io.load_pos(mi[r], a0, a1, a2, a3); io.load_vel(mi[r], b0, b1, b2, b3);
                    io.store_pos(mo[r], a0, a1, a2, a3); io.store_vel(mo[r], b0, b1, b2, b3);
                    P.rc.key[mo[r]] = n_elems;
                }
            }
            io.stage_next();
            if (kHist) {
                unsigned peers[kR];
                int base[kR];
                hist_issue<kR>(P.hist, key, on, peers, base);
                rank_finish<kR>(P.rank, mo, on, peers, base);
            }
        } else {
            mbar_wait(bar0 + b * 8, (phase >> b) & 1u);
            phase ^= 1u << b;
            if (kMode == 1) step_R_nl<kR, kHist, true, AsyncIO<kR>, true>(P, io, tbuf + (size_t)b * stride_d, mi, mo, on, Rn, Zn);
            else step_R<kR, kHist, true, AsyncIO<kR>, 0, true>(P, io, tbuf + (size_t)b * stride_d, mi, mo, on, Rn, Zn);
        }
        cp_async_wait<2>();                            // the search records of item k - 1 have landed
        search_prev(k - 1);
        // item k: new (R, Z) and the request for the record of their search bucket
        if (e < n_elems) {
#pragma unroll
            for (int r = 0; r < kR; ++r) {
                const int i = 32 * r + lane;
                if (i < count) {
                    rz[i] = make_double2(Rn[r], Zn[r]);
                    float u, v;
                    bool inside;
                    const FastRec *g = P.f.fast.first + (size_t)fast_bucket(P.f.fast, Rn[r], Zn[r], u, v, inside);
                    const unsigned d = smem_u32(fr) + (unsigned)i * 16u;
#pragma unroll
                    for (int c = 0; c < 4; ++c) cp_async16(d + (unsigned)(c * kSlots) * 16u, reinterpret_cast<const char *>(g) + 16 * c);
                }
            }
        }
        cp_async_commit();
    }
    // drain: search and ranks of the last item
    cp_async_wait<0>();
    search_prev(k - 1);
}

static size_t async_smem_bytes(int tile_stride, int kR) {
    const size_t warps = kPushThreads / 32, slots = 32 * (size_t)kR;
    return warps * (2 * (size_t)tile_stride * 8 + slots * (64 + 16 + 64 + 16) + 16 * 16 + 16);
}

// ---- diagnostics ---------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(128) eval_fields_kernel(FieldParams f, long n, const double *R, const double *phi,
                                                          const double *Z, double t, int *elem_out, double *out) {
    const long i = (long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const double r = R[i], z = Z[i];
    const int e = locate_any(f, r, z);
    elem_out[i] = e;
    if (e < 0) return;
    double cwt[M3DK_MAX_MODES], swt[M3DK_MAX_MODES];
    for (int k = 0; k < f.n_modes; ++k) sincos(f.omega[k] * t, &swt[k], &cwt[k]);
    double sp, cp;
    sincos(phi[i], &sp, &cp);
    Fields o;
    eval_fields(f, e, r, z, cp, sp, 1.0 / r, cwt, swt, o);
    double *q = out + 18 * i;
    q[0] = o.psi_R; q[1] = o.psi_Z; q[2] = o.Bm; q[3] = o.Bm_R; q[4] = o.Bm_Z; q[5] = o.F; q[6] = o.kappa;
    for (int k = 0; k < 3; ++k) { q[7 + k] = o.E1[k]; q[10 + k] = o.B1[k]; q[13 + k] = o.gB[k]; }
    q[16] = o.dtB; q[17] = o.B1p;
}

__global__ void count_lost_kernel(const int *elem, long n, int *count) {
    long i = (long)blockIdx.x * blockDim.x + threadIdx.x;
    const long stride = (long)gridDim.x * blockDim.x;
    int c = 0;
    for (; i < n; i += stride) c += elem[i] < 0;
    for (int o = 16; o > 0; o >>= 1) c += __shfl_down_sync(0xffffffffu, c, o);
    if ((threadIdx.x & 31) == 0 && c) atomicAdd(count, c);
}

// ---- FP64 peak probe: 8 independent DFMA chains per thread, register resident -------------------------------------
__global__ void __launch_bounds__(256) dfma_probe_kernel(double *sink, int iters, double a, double b) {
    double r0 = threadIdx.x, r1 = r0 + 1, r2 = r0 + 2, r3 = r0 + 3, r4 = r0 + 4, r5 = r0 + 5, r6 = r0 + 6, r7 = r0 + 7;
    for (int i = 0; i < iters; ++i) {
#pragma unroll
        for (int u = 0; u < 8; ++u) {
            r0 = fma(r0, a, b); r1 = fma(r1, a, b); r2 = fma(r2, a, b); r3 = fma(r3, a, b);
            r4 = fma(r4, a, b); r5 = fma(r5, a, b); r6 = fma(r6, a, b); r7 = fma(r7, a, b);
        }
    }
    const double s = ((r0 + r1) + (r2 + r3)) + ((r4 + r5) + (r6 + r7));
    if (s == 123.456) sink[0] = s;  // never true in practice; keeps the chains alive
}

// ---- launchers -----------------------------------------------------------------------------------------------------
static PushParams make_params(m3dk_ctx *c, const MarkerArrays &a, long n, double dt, double t) {
    PushParams P{};
    P.n = n; P.a = a; P.f = c->f;
    P.dt = dt; P.q = c->q; P.m = c->m; P.inv_q = 1.0 / c->q; P.inv_m = 1.0 / c->m;
    P.h = c->q * dt / (2.0 * c->m);
    P.f0kind = c->f0.kind;
    P.f0T_inv = c->f0.kind == M3DK_F0_MAXWELLIAN ? 1.0 / c->f0.T : 0.0;
    P.f0vc3 = c->f0.v_c * c->f0.v_c * c->f0.v_c;
    P.f0L0 = c->f0.Lambda0;
    P.f0dL2_inv = c->f0.kind == M3DK_F0_BEAM_PITCH ? 1.0 / (c->f0.dLambda * c->f0.dLambda) : 0.0;
    P.f0Bax = c->f0.B_axis;
    for (int k = 0; k < c->f.n_modes; ++k) {
        P.cwt[k] = cos(c->f.omega[k] * t);
        P.swt[k] = sin(c->f.omega[k] * t);
    }
    return P;
}

cudaError_t launch_locate(m3dk_ctx *c, const MarkerArrays &a, long n, bool fill_id, int id_base) {
    if (n == 0) return cudaSuccess;
    const unsigned grid = (unsigned)((n + 255) / 256);
    c->kernel_launches += 1;
    locate_kernel<<<grid, 256, 0, c->stream>>>(c->f, a, n, fill_id ? 1 : 0, id_base);
    return cudaGetLastError();
}

cudaError_t launch_push_soa(m3dk_ctx *c, long n, double dt, double t) {
    if (n == 0) return cudaSuccess;
    PushParams P = make_params(c, c->user, n, dt, t);
    c->kernel_launches += 1;
    if (c->mode == 1) push_generic_kernel<1><<<(unsigned)((n + 127) / 128), 128, 0, c->stream>>>(P);
    else if (c->mode == 2) push_generic_kernel<2><<<(unsigned)((n + 127) / 128), 128, 0, c->stream>>>(P);
    else if (c->mode == 3) push_generic_kernel<4><<<(unsigned)((n + 127) / 128), 128, 0, c->stream>>>(P);
    else push_generic_kernel<0><<<(unsigned)((n + 127) / 128), 128, 0, c->stream>>>(P);
    return cudaGetLastError();
}

// mode 3 runs through the ring stream when the FLR workspace holds the averages array
bool flr_nl_stream(const m3dk_ctx *c) { return c->mode == 3 && c->have_flrws && c->flr_with_avg && c->f.n_modes > 0; }

// Mode 3 through the ring stream, first pass over the current work items: the ring points of every marker into the stream
// (push_items_kernel<false, 5, .>: nothing but the stream is written).  The item tickets are cleared again afterwards: the
// second pass (launch_push_rec) walks the same item lists.
cudaError_t launch_flr_emit_nl(m3dk_ctx *c, long n, double dt, double t) {
    if (n == 0) return cudaSuccess;
    PushParams P = make_params(c, c->user, n, dt, t);
    P.rc.key = c->sb.key; P.rc.order = c->sb.order[c->ocur];
    P.rc.in = c->sb.rec[c->cur]; P.rc.out = c->sb.rec[c->cur ^ 1];
    P.fl = c->fb.a;
    cudaError_t e = cudaMemsetAsync(c->fb.a.rhist, 0, (size_t)(c->f.n_elems + 1) * sizeof(int), c->stream);
    if (e != cudaSuccess) return e;
    const unsigned grid = (unsigned)(c->sm_count * M3DK_PUSH_MINBLOCKS);
    const size_t smem = (size_t)(kPushThreads / 32) * 2 * (c->f.tile_stride * 8 + 8);
    int *const tickets = reinterpret_cast<int *>(c->sb.scan_state + (c->f.n_elems + 1 + 4095) / 4096 + 2);
    for (int small = 0; small < 2; ++small) {
        P.items = small ? c->sb.items_small : c->sb.items;
        P.n_items = small ? reinterpret_cast<const int *>(c->sb.scan_state + 1) : c->sb.ioffs + c->f.n_elems + 1;
        P.ticket = tickets + small;
        void (*kern)(PushParams) = small ? push_items_kernel<false, 5, 1> : push_items_kernel<false, 5, 2>;
        e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
        c->kernel_launches += 1;
        kern<<<small ? grid / M3DK_PUSH_MINBLOCKS * (M3DK_PUSH_MINBLOCKS + 1) : grid, kPushThreads, smem, c->stream>>>(P);
    }
    e = cudaMemsetAsync(tickets, 0, 2 * sizeof(int), c->stream);
    return e != cudaSuccess ? e : cudaGetLastError();
}

// One element-ordered step on the records: sb.rec[cur] gathered through sb.order[ocur] into sb.rec[cur ^ 1], which becomes
// current.  with_hist: also histogram the new keys for the reorder that follows.
cudaError_t launch_push_rec(m3dk_ctx *c, long n, double dt, double t, bool with_hist) {
    if (n == 0) return cudaSuccess;
    PushParams P = make_params(c, c->user, n, dt, t);
    c->kernel_launches += 1;
    P.hist = c->sb.hist; P.rank = c->sb.rank;
    c->ranks_valid = true;
    P.rc.key = c->sb.key; P.rc.order = c->sb.order[c->ocur];
    P.rc.in = c->sb.rec[c->cur];
    if (with_hist) {
        cudaError_t e = cudaMemsetAsync(c->sb.hist, 0, (size_t)(c->f.n_elems + 1) * sizeof(int), c->stream);
        if (e != cudaSuccess) return e;
    }
    const bool flr_stream = c->mode == 2 && c->have_flrws && c->f.n_modes > 0;
    const bool nl_stream = flr_nl_stream(c);     // mode 3: the averages are in the ring stream (launch_flr_emit_nl .. ring eval)
    if (flr_stream) {
        P.fl = c->fb.a;
        cudaError_t e = cudaMemsetAsync(c->fb.a.rhist, 0, (size_t)(c->f.n_elems + 1) * sizeof(int), c->stream);
        if (e != cudaSuccess) return e;
    }
    if (nl_stream) P.fl = c->fb.a;
    {
        P.rc.out = c->sb.rec[c->cur ^ 1];
        P.items = c->sb.items; P.n_items = c->sb.ioffs + c->f.n_elems + 1;
        const unsigned grid = (unsigned)(c->sm_count * M3DK_PUSH_MINBLOCKS);
        const size_t smem = (size_t)(kPushThreads / 32) * 2 * (c->f.tile_stride * 8 + 8);
        // two launches: the items of up to 64 markers (two per lane), then the small items (one per lane)
        for (int small = 0; small < 2; ++small) {
            P.items = small ? c->sb.items_small : c->sb.items;
            P.n_items = small ? reinterpret_cast<const int *>(c->sb.scan_state + 1) : c->sb.ioffs + c->f.n_elems + 1;
            P.ticket = reinterpret_cast<int *>(c->sb.scan_state + (c->f.n_elems + 1 + 4095) / 4096 + 2) + small;
            void (*kern)(PushParams);
            const size_t as_smem = async_smem_bytes(c->f.tile_stride, small ? 1 : 2);
            if (c->push_variant == 1 && (c->mode == 0 || c->mode == 1) && as_smem <= c->smem_optin) {
                if (small)
                    kern = c->mode == 1 ? (with_hist ? push_async_kernel<true, 1, 1> : push_async_kernel<false, 1, 1>)
                                        : (with_hist ? push_async_kernel<true, 0, 1> : push_async_kernel<false, 0, 1>);
                else
                    kern = c->mode == 1 ? (with_hist ? push_async_kernel<true, 1, 2> : push_async_kernel<false, 1, 2>)
                                        : (with_hist ? push_async_kernel<true, 0, 2> : push_async_kernel<false, 0, 2>);
                cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)as_smem);
                if (e != cudaSuccess) return e;
                int per_sm = 0;
                e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kern, kPushThreads, as_smem);
                if (e != cudaSuccess) return e;
                if (per_sm < 1) per_sm = 1;
                if (small) c->kernel_launches += 1;
                kern<<<(unsigned)(c->sm_count * per_sm), kPushThreads, as_smem, c->stream>>>(P);
                c->ranks_valid = false;      // this kernel only counts; invert_kernel draws the slots
                continue;
            }
            // mode 2: with an FLR workspace the push emits the ring stream (kernel mode 3), else every lane gathers its ring
            const int km = c->mode == 2 ? (flr_stream ? 3 : (c->f.n_modes > 0 ? 2 : 0)) : c->mode == 3 ? (nl_stream ? 6 : 4) : c->mode;
            if (small)
                kern = km == 1   ? (with_hist ? push_items_kernel<true, 1, 1> : push_items_kernel<false, 1, 1>)
                       : km == 2 ? (with_hist ? push_items_kernel<true, 2, 1> : push_items_kernel<false, 2, 1>)
                       : km == 3 ? (with_hist ? push_items_kernel<true, 3, 1> : push_items_kernel<false, 3, 1>)
                       : km == 4 ? (with_hist ? push_items_kernel<true, 4, 1> : push_items_kernel<false, 4, 1>)
                       : km == 6 ? (with_hist ? push_items_kernel<true, 6, 1> : push_items_kernel<false, 6, 1>)
                                 : (with_hist ? push_items_kernel<true, 0, 1> : push_items_kernel<false, 0, 1>);
            else
                kern = km == 1   ? (with_hist ? push_items_kernel<true, 1, 2> : push_items_kernel<false, 1, 2>)
                       : km == 2 ? (with_hist ? push_items_kernel<true, 2, 2> : push_items_kernel<false, 2, 2>)
                       : km == 3 ? (with_hist ? push_items_kernel<true, 3, 2> : push_items_kernel<false, 3, 2>)
                       : km == 4 ? (with_hist ? push_items_kernel<true, 4, 2> : push_items_kernel<false, 4, 2>)
                       : km == 6 ? (with_hist ? push_items_kernel<true, 6, 2> : push_items_kernel<false, 6, 2>)
                                 : (with_hist ? push_items_kernel<true, 0, 2> : push_items_kernel<false, 0, 2>);
            cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
            if (e != cudaSuccess) return e;
            if (small) c->kernel_launches += 1;
            kern<<<small ? grid / M3DK_PUSH_MINBLOCKS * (M3DK_PUSH_MINBLOCKS + 1) : grid, kPushThreads, smem, c->stream>>>(P);
        }
        c->cur ^= 1;
    }
    return cudaGetLastError();
}

cudaError_t launch_flr_ring_keys(m3dk_ctx *c, long n) {
    if (n == 0) return cudaSuccess;
    const long n4 = 4 * n;
    c->kernel_launches += 1;
    const unsigned grid = (unsigned)((n4 + 255) / 256);
    static const unsigned primes[] = {1009u, 1013u, 1019u, 1021u, 1031u};
    unsigned cs = 1u;
    for (unsigned p : primes)
        if (grid % p != 0) { cs = p; break; }
    ring_key_kernel<<<grid, 256, 0, c->stream>>>(c->f, n4, c->fb.a.ring, c->fb.a.rkey, c->fb.a.rrank, c->fb.a.rhist, cs);
    return cudaGetLastError();
}

// evaluation of the ordered ring stream (mode 2): the ring items of up to 64 points, then the small ones
cudaError_t launch_flr_ring_eval(m3dk_ctx *c, long n, double dt, double t, bool avg) {
    if (n == 0) return cudaSuccess;
    PushParams P = make_params(c, c->user, n, dt, t);
    P.fl = c->fb.a;
    const size_t smem = (size_t)(kPushThreads / 32) * 2 * (c->f.tile_stride * 8 + 8);
    const unsigned grid = (unsigned)(c->sm_count * M3DK_PUSH_MINBLOCKS);
    for (int small = 0; small < 2; ++small) {
        P.items = small ? c->fb.ritems_small : c->fb.ritems;
        P.n_items = small ? reinterpret_cast<const int *>(c->fb.rstate + 1) : c->fb.rioffs + c->f.n_elems + 1;
        P.ticket = reinterpret_cast<int *>(c->fb.rstate + (c->f.n_elems + 1 + 4095) / 4096 + 2) + small;
        void (*kern)(PushParams) = avg ? (small ? ring_items_kernel<1, true> : ring_items_kernel<2, true>)
                                       : (small ? ring_items_kernel<1, false> : ring_items_kernel<2, false>);
        cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
        c->kernel_launches += 1;
        kern<<<small ? grid / M3DK_PUSH_MINBLOCKS * (M3DK_PUSH_MINBLOCKS + 1) : grid, kPushThreads, smem, c->stream>>>(P);
    }
    return cudaGetLastError();
}

cudaError_t launch_eval_fields(m3dk_ctx *c, long n, const double *R, const double *phi, const double *Z, double t,
                               int *elem_out, double *out) {
    if (n == 0) return cudaSuccess;
    const unsigned grid = (unsigned)((n + 127) / 128);
    c->kernel_launches += 1;
    eval_fields_kernel<<<grid, 128, 0, c->stream>>>(c->f, n, R, phi, Z, t, elem_out, out);
    return cudaGetLastError();
}

cudaError_t launch_count_lost(m3dk_ctx *c, const MarkerArrays &a, long n, int *d_count) {
    cudaError_t e = cudaMemsetAsync(d_count, 0, sizeof(int), c->stream);
    if (e != cudaSuccess || n == 0) return e;
    const unsigned grid = (unsigned)((n + 255) / 256 < 1184 ? (n + 255) / 256 : 1184);
    c->kernel_launches += 1;
    count_lost_kernel<<<grid, 256, 0, c->stream>>>(a.elem, n, d_count);
    return cudaGetLastError();
}

cudaError_t fp64_probe(m3dk_ctx *c, double *tflops) {
    int sms = 0;
    cudaError_t e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, c->device);
    if (e != cudaSuccess) return e;
    const int iters = 4096, blocks = sms * 8, threads = 256;
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0); cudaEventCreate(&e1);
    double best = 0.0;
    for (int rep = 0; rep < 5; ++rep) {
        cudaEventRecord(e0, c->stream);
        dfma_probe_kernel<<<blocks, threads, 0, c->stream>>>(reinterpret_cast<double *>(c->d_count), iters, 0.999999, 1e-9);
        cudaEventRecord(e1, c->stream);
        e = cudaEventSynchronize(e1);
        if (e != cudaSuccess) break;
        float ms = 0.f;
        cudaEventElapsedTime(&ms, e0, e1);
        const double flops = 2.0 * 64.0 * iters * (double)blocks * threads;
        if (rep > 0 && ms > 0.f) best = fmax(best, flops / (ms * 1e-3) * 1e-12);
    }
    cudaEventDestroy(e0); cudaEventDestroy(e1);
    if (e == cudaSuccess) e = cudaGetLastError();
    *tflops = best;
    return e;
}

}  // namespace m3dk
