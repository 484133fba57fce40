// m3dk_gc.cu -- RK4 guiding-centre pusher (Eqs. 1-4; reading G24): the paper's comparator
// pusher (Fig. 1) and the "(dX/dt)_0 using only the equilibrium fields" of PAPER.md:130.  Equilibrium fields only (E = 0):
//     dX/dt       = (1/B*par) [ v_par B* + (mu/q) b x grad|B| ]      B* = B + (m v_par/q) curl b,  B*par = B* . b
//     m dv_par/dt = -(mu/B*par) B* . grad|B|
// curl b needs the SECOND derivatives of psi0 and the first of F0 (the cost that made the authors prefer the
// Boris scheme); |B| and its gradient come from the |B| table.  One guiding centre per thread, four stages per step, each
// with its own element search and tile gather (the stages leave the element): the one-marker-per-thread regime.
#include "m3dk_device.cuh"

namespace m3dk {

// right-hand side of Eqs. (1)-(2) at (R, Z, v_par): dX/dt in cylindrical components, dv_par/dt; false outside the mesh
__device__ __forceinline__ bool gc_rhs(const FieldParams &f, double q, double m, double R, double Z, double vpar, double mu,
                                       double (&dX)[3], double &dv, int &elem) {
    const int e = locate_any(f, R, Z);
    elem = e;
    if (e < 0) return false;
    const double *tile = f.tiles + (size_t)e * f.tile_stride;
    GcEq g;
    gc_eq_fields(tile, R, Z, g);
    double Bs[3], b[3];
    const double Bspar = bstar_par(g, q, m, vpar, Bs, b);
    const double Bm_R = g.Bm_R, Bm_Z = g.Bm_Z;
    const double bsinv = m3dk_rcp(Bspar);
    const double muq = mu / q;
    const double bxg[3] = {b[1] * Bm_Z, b[2] * Bm_R - b[0] * Bm_Z, -b[1] * Bm_R};     // b x grad|B|, grad|B| = (Bm_R, 0, Bm_Z)
#pragma unroll
    for (int k = 0; k < 3; ++k) dX[k] = (vpar * Bs[k] + muq * bxg[k]) * bsinv;
    dv = -(mu / m) * (Bs[0] * Bm_R + Bs[2] * Bm_Z) * bsinv;
    return true;
}

// One RK4 step of y = (x, y, z, v_par).  false: one of the four stages lies outside the mesh (y is left untouched).
__device__ __forceinline__ bool gc_rk4_step(const FieldParams &f, double q, double m, double mu, double dt, double (&y)[4]) {
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
        if (ok && !gc_rhs(f, q, m, R, yy[2], yy[3], mu, dX, dv, es)) ok = false;
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
__global__ void __launch_bounds__(128) gc_push_kernel(const __grid_constant__ FieldParams f, MarkerArrays a, double *vpar,
                                                      long n, double q, double m, double dt, int nsteps) {
    const long i = (long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    int e = a.elem[i];
    if (e < 0) return;
    double y[4] = {a.x[i], a.y[i], a.z[i], vpar[i]};
    const double mu = a.mu[i];
    for (int l = 0; l < nsteps && e >= 0; ++l) {
        if (!gc_rk4_step(f, q, m, mu, dt, y)) { e = -1; break; }
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
    if (gc_rk4_step(f, q, m, a.mu[i], dt, y)) e = locate_xyz(f, y[0], y[1], y[2]);
    a.elem[i] = e;
    if (e < 0) return;
    const double rdt = 1.0 / dt;
    a.vx[i] = (y[0] - x0) * rdt; a.vy[i] = (y[1] - y0) * rdt; a.vz[i] = (y[2] - z0) * rdt;
    a.x[i] = y[0]; a.y[i] = y[1]; a.z[i] = y[2];
}

cudaError_t launch_gc_push(m3dk_ctx *c, long n, double *vpar, int nsteps, double dt) {
    if (n == 0 || nsteps == 0) return cudaSuccess;
    c->kernel_launches += 1;
    gc_push_kernel<<<(unsigned)((n + 127) / 128), 128, 0, c->stream>>>(c->f, c->user, vpar, n, c->q, c->m, dt, nsteps);
    return cudaGetLastError();
}

cudaError_t launch_gc_bootstrap(m3dk_ctx *c, long n, const double *vpar, double dt) {
    if (n == 0) return cudaSuccess;
    c->kernel_launches += 1;
    gc_bootstrap_kernel<<<(unsigned)((n + 127) / 128), 128, 0, c->stream>>>(c->f, c->user, vpar, n, c->q, c->m, dt);
    return cudaGetLastError();
}

}  // namespace m3dk
