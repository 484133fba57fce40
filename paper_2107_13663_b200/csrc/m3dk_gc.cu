// m3dk_gc.cu -- RK4 guiding-centre pusher (Eqs. 1-4; reading G24): the paper's comparator
// pusher (Fig. 1) and the "(dX/dt)_0 using only the equilibrium fields" of PAPER.md:130.  Equilibrium fields only (E = 0):
//     dX/dt       = (1/B*par) [ v_par B* + (mu/q) b x grad|B| ]      B* = B + (m v_par/q) curl b,  B*par = B* . b
//     m dv_par/dt = -(mu/B*par) B* . grad|B|
// curl b needs the SECOND derivatives of psi0 and the first of F0 (the cost that made the authors prefer the
// Boris scheme); |B| and its gradient come from the |B| table.  One guiding centre per thread, four stages per step, each
// with its own element search and tile gather (the stages leave the element): the one-marker-per-thread regime.
#include "m3dk_device.cuh"

namespace m3dk {

// right-hand side of Eqs. (1)-(2) at (R, phi, Z, v_par, t): dX/dt in cylindrical components, dv_par/dt; false outside the mesh
//     dX/dt = (1/B*par) [v_par B* - b x (E - (mu/q) grad B)],   m dv_par/dt = (1/B*par) B* . (q E - mu grad B)
// kPert (reading G26): E = E1, B1 added to B*, grad B = grad(|B|0 + B1par); b, curl b and B*par = B* . b keep b0.
template <bool kPert>
__device__ __forceinline__ bool gc_rhs(const FieldParams &f, double q, double m, double R, double Z, double cph, double sph,
                                       double vpar, double mu, double t, double (&dX)[3], double &dv, int &elem) {
    const int e = locate_any(f, R, Z);
    elem = e;
    if (e < 0) return false;
    const double *tile = f.tiles + (size_t)e * f.tile_stride;
    GcEq g;
    gc_eq_fields(tile, R, Z, g);
    double Bs[3], b[3];
    double Bspar = bstar_par(g, q, m, vpar, Bs, b);
    double gB[3] = {g.Bm_R, 0.0, g.Bm_Z}, E[3] = {0.0, 0.0, 0.0};
    if (kPert) {
        double cwt[M3DK_MAX_MODES], swt[M3DK_MAX_MODES];
        for (int k = 0; k < f.n_modes; ++k) sincos(f.omega[k] * t, &swt[k], &cwt[k]);
        Fields o;
        eval_fields(f, e, R, Z, cph, sph, g.rinv, cwt, swt, o);
        Bspar = 0.0;
#pragma unroll
        for (int k = 0; k < 3; ++k) { Bs[k] += o.B1[k]; Bspar += Bs[k] * b[k]; gB[k] += o.gB[k]; E[k] = o.E1[k]; }
    }
    const double bsinv = m3dk_rcp(Bspar);
    const double muq = mu / q;
    const double Ee[3] = {E[0] - muq * gB[0], E[1] - muq * gB[1], E[2] - muq * gB[2]};
    const double bxE[3] = {b[1] * Ee[2] - b[2] * Ee[1], b[2] * Ee[0] - b[0] * Ee[2], b[0] * Ee[1] - b[1] * Ee[0]};
#pragma unroll
    for (int k = 0; k < 3; ++k) dX[k] = (vpar * Bs[k] - bxE[k]) * bsinv;
    dv = (q / m) * (Bs[0] * Ee[0] + Bs[1] * Ee[1] + Bs[2] * Ee[2]) * bsinv;
    return true;
}

// One RK4 step of y = (x, y, z, v_par).  false: one of the four stages lies outside the mesh (y is left untouched).
template <bool kPert>
__device__ __forceinline__ bool gc_rk4_step(const FieldParams &f, double q, double m, double mu, double t, double dt, double (&y)[4]) {
    double k[4][4], yy[4];
    bool ok = true;
#pragma unroll
    for (int st = 0; st < 4; ++st) {
        const double cs = st == 0 ? 0.0 : (st == 3 ? 1.0 : 0.5);
#pragma unroll
        for (int c = 0; c < 4; ++c) yy[c] = st ? y[c] + cs * dt * k[st > 0 ? st - 1 : 0][c] : y[c];
        const double r2 = yy[0] * yy[0] + yy[1] * yy[1];
        const double rinv = m3dk_rsqrt(r2), R = r2 * rinv, c = yy[0] * rinv, sn = yy[1] * rinv;
        double dX[3], dv;
        int es;
        if (ok && !gc_rhs<kPert>(f, q, m, R, yy[2], c, sn, yy[3], mu, t + cs * dt, dX, dv, es)) ok = false;
        if (!ok) { dX[0] = dX[1] = dX[2] = 0.0; dv = 0.0; }
        k[st][0] = dX[0] * c - dX[1] * sn; k[st][1] = dX[0] * sn + dX[1] * c; k[st][2] = dX[2]; k[st][3] = dv;
    }
    if (!ok) return false;
#pragma unroll
    for (int c = 0; c < 4; ++c) y[c] += dt / 6.0 * (k[0][c] + 2.0 * k[1][c] + 2.0 * k[2][c] + k[3][c]);
    return true;
}

// nsteps RK4 steps.  elem is kept at the element of the CURRENT position (every other entry point trusts it).  A guiding
// centre is lost (elem = -1, frozen; reading G12) when a stage of a step leaves the mesh (it keeps the state of the step
// before) or when a step ends outside (it keeps that state).
template <bool kPert>
__global__ void __launch_bounds__(128) gc_push_kernel(const __grid_constant__ FieldParams f, MarkerArrays a, double *vpar,
                                                      long n, double q, double m, double t0, double dt, int nsteps) {
    const long i = (long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    int e = a.elem[i];
    if (e < 0) return;
    double y[4] = {a.x[i], a.y[i], a.z[i], vpar[i]};
    const double mu = a.mu[i];
    for (int l = 0; l < nsteps && e >= 0; ++l) {
        if (!gc_rk4_step<kPert>(f, q, m, mu, t0 + (double)l * dt, dt, y)) { e = -1; break; }
        e = locate_xyz(f, y[0], y[1], y[2]);
    }
    a.x[i] = y[0]; a.y[i] = y[1]; a.z[i] = y[2]; vpar[i] = y[3];
    a.elem[i] = e;
}

// Bootstrap of the slow-manifold Boris scheme: one RK4 guiding-centre step x_0 -> x_1, then
// (x, v) <- (x_1, (x_1 - x_0)/dt): the staggered state (x_l, v_{l-1/2}) m3dk_push starts from.  A marker whose step leaves
// the mesh (a stage or the end point) is lost: elem = -1, state untouched.
__global__ void __launch_bounds__(128) gc_bootstrap_kernel(const __grid_constant__ FieldParams f, MarkerArrays a,
                                                           const double *vpar, long n, double q, double m, double dt) {
    const long i = (long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    if (a.elem[i] < 0) return;
    const double x0 = a.x[i], y0 = a.y[i], z0 = a.z[i];
    double y[4] = {x0, y0, z0, vpar[i]};
    int e = -1;
    if (gc_rk4_step<false>(f, q, m, a.mu[i], 0.0, dt, y)) e = locate_xyz(f, y[0], y[1], y[2]);
    a.elem[i] = e;
    if (e < 0) return;
    const double rdt = 1.0 / dt;
    a.vx[i] = (y[0] - x0) * rdt; a.vy[i] = (y[1] - y0) * rdt; a.vz[i] = (y[2] - z0) * rdt;
    a.x[i] = y[0]; a.y[i] = y[1]; a.z[i] = y[2];
}

cudaError_t launch_gc_push(m3dk_ctx *c, long n, double *vpar, int nsteps, double dt, bool pert, double t0) {
    if (n == 0 || nsteps == 0) return cudaSuccess;
    c->kernel_launches += 1;
    const unsigned grid = (unsigned)((n + 127) / 128);
    if (pert) gc_push_kernel<true><<<grid, 128, 0, c->stream>>>(c->f, c->user, vpar, n, c->q, c->m, t0, dt, nsteps);
    else gc_push_kernel<false><<<grid, 128, 0, c->stream>>>(c->f, c->user, vpar, n, c->q, c->m, t0, dt, nsteps);
    return cudaGetLastError();
}

cudaError_t launch_gc_bootstrap(m3dk_ctx *c, long n, const double *vpar, double dt) {
    if (n == 0) return cudaSuccess;
    c->kernel_launches += 1;
    gc_bootstrap_kernel<<<(unsigned)((n + 127) / 128), 128, 0, c->stream>>>(c->f, c->user, vpar, n, c->q, c->m, dt);
    return cudaGetLastError();
}

}  // namespace m3dk
