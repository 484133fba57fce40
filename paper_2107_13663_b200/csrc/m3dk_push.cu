// m3dk_push.cu -- kernels of the fused push and their launchers.
#include <math.h>

#include "m3dk_device.cuh"

namespace m3dk {

#ifndef M3DK_PUSH_THREADS
#define M3DK_PUSH_THREADS 128
#endif
#ifndef M3DK_PUSH_MINBLOCKS
#define M3DK_PUSH_MINBLOCKS 4
#endif
constexpr int kPushThreads = M3DK_PUSH_THREADS;

// ---- element of every marker (particles_init / upload) ------------------------------------------------------------
__global__ void __launch_bounds__(256) locate_kernel(const __grid_constant__ FieldParams f, MarkerArrays a, long n,
                                                     int fill_id) {
    const long i = (long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    a.elem[i] = locate_xyz(f, a.x[i], a.y[i], a.z[i]);
    if (fill_id) a.id[i] = (int)i;
}

// Warp-aggregated histogram with returned ranks: lanes with the same key elect a leader that does one atomic.
__device__ __forceinline__ int hist_rank(int *hist, int key, bool on) {
    const unsigned live = __ballot_sync(0xffffffffu, on);
    int r = 0;
    if (on) {
        const unsigned peers = __match_any_sync(live, key);
        const int lane = threadIdx.x & 31;
        const int leader = __ffs(peers) - 1;
        int base = 0;
        if (lane == leader) base = atomicAdd(hist + key, __popc(peers));
        base = __shfl_sync(peers, base, leader);
        r = base + __popc(peers & ((1u << lane) - 1u));
    }
    return r;
}

// Lane l touches line l of the element's tile (27 lines for one mode): the whole tile is in flight with one instruction
// per lane, long before the Horner chains ask for it.
__device__ __forceinline__ void prefetch_tile(const FieldParams &f, int e) {
    const int lane = threadIdx.x & 31;
    const int nlines = f.tile_stride >> 4;
    const double *tile = f.tiles + (size_t)e * f.tile_stride;
    for (int l = lane; l < nlines; l += 32) asm volatile("prefetch.global.L1 [%0];" ::"l"(tile + 16 * l));
}

// ---- one step of R markers of one thread that sit in the same element e (rows a1-a10) -------------------------------
// m[r]: slot of marker r in the SoA arrays, on[r]: marker r exists.  Phase A: a1 load, a2 cylindrical map, a4-a5
// equilibrium quad (every coefficient load shared by the R markers), a7 assemble, a8 Boris, a10 drift + store, a3 for
// the NEW position (cached for the next step; it is the sort key) and, with kHist, the sort histogram of the new keys.
// Phase B: a6 perturbed quads folded into dw/dt as they are evaluated, a9 weight update.
template <int R, bool kHist>
__device__ __forceinline__ void step_R(const PushParams &P, int e, const long (&m)[R], const bool (&on)[R]) {
    // the loads below may be speculated above the `on` tests: e is clamped to a valid element for addressing
    const double *tile = P.f.tiles + (size_t)max(e, 0) * P.f.tile_stride;
    Marker s[R];
    StepGeom g[R];
#pragma unroll
    for (int r = 0; r < R; ++r) {
        if (on[r]) { s[r].x = P.a.x[m[r]]; s[r].y = P.a.y[m[r]]; s[r].z = P.a.z[m[r]]; }
        else { s[r].x = 1.0; s[r].y = 0.0; s[r].z = 0.0; }
    }
    const Quad hd = ldq(tile);
    const double Rc = hd.a, Zc = hd.b, se = hd.c;
    double xi[R], eta[R];
#pragma unroll
    for (int r = 0; r < R; ++r) {
        step_geometry(s[r], g[r]);
        xi[r] = __dmul_rn(__dsub_rn(g[r].R, Rc), se); eta[r] = __dmul_rn(__dsub_rn(s[r].z, Zc), se);
    }
    double v[R][4], dx[R][4], de[R][4];
    quad_vd<R>(tile + kTileHeader, xi, eta, v, dx, de);          // (psi0, |B|0, F0, kappa)
    PertW W[R];
    double Rn[R], Zn[R];
#pragma unroll
    for (int r = 0; r < R; ++r) {
        EqOut f;
        f.psi_R = __dmul_rn(dx[r][0], se); f.psi_Z = __dmul_rn(de[r][0], se);
        f.Bm = v[r][1]; f.Bm_R = __dmul_rn(dx[r][1], se); f.Bm_Z = __dmul_rn(de[r][1], se);
        f.F = v[r][2]; f.kappa = v[r][3];
        if (on[r]) {
            s[r].vx = P.a.vx[m[r]]; s[r].vy = P.a.vy[m[r]]; s[r].vz = P.a.vz[m[r]]; s[r].mu = P.a.mu[m[r]];
        } else { s[r].vx = s[r].vy = s[r].vz = 0.0; s[r].mu = 0.0; }
        push_eq(P, g[r], f, s[r], W[r]);
        if (on[r]) {
            P.a.x[m[r]] = s[r].x; P.a.y[m[r]] = s[r].y; P.a.z[m[r]] = s[r].z;
            P.a.vx[m[r]] = s[r].vx; P.a.vy[m[r]] = s[r].vy; P.a.vz[m[r]] = s[r].vz;
        }
        // the element search of the new position runs after phase B; its first record starts travelling now
        Rn[r] = __dsqrt_rn(M3DK_FMA(s[r].x, s[r].x, __dmul_rn(s[r].y, s[r].y)));
        Zn[r] = s[r].z;
        locate_prefetch(P.f.fast, Rn[r], Zn[r]);
    }
    if (P.f.n_modes > 0) {
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
            // the three value-only quads share one copy of the Horner code (rolled: the kernel must fit the 32 KB
            // instruction cache); the weights of quad q are picked by selects
#pragma unroll 1
            for (int q = 0; q < 3; ++q) {
                quad_vd<R>(pm + q * kQuad, xi, eta, v, dx, de);
#pragma unroll
                for (int r = 0; r < R; ++r) {
                    const double wa = q == 0 ? W[r].aER : (q == 1 ? W[r].aEZ : 0.0);     // B_phi does not enter
                    const double wb = q == 0 ? W[r].aEP : (q == 1 ? W[r].bBR : W[r].bBZ);
                    wsum[r] = pert_fold_v(wsum[r], v[r], wa, wb, cth[r], sth[r]);
                }
            }
            quad_vd<R>(pm + 3 * kQuad, xi, eta, v, dx, de);
#pragma unroll
            for (int r = 0; r < R; ++r) wsum[r] = pert_fold_par(wsum[r], v[r], dx[r], de[r], W[r], cth[r], sth[r], se, nri[r], om);
        }
        // Eqs. (8)-(9): explicit midpoint on the staggered grid (G9)
#pragma unroll
        for (int r = 0; r < R; ++r)
            if (on[r]) P.a.w[m[r]] = M3DK_FMA(P.dt, wsum[r], P.a.w[m[r]]);
    }
    // a3 for the NEW position (the key of the next sort) and, with kHist, the sort histogram of the new keys with each
    // marker's rank inside its key: the sort then needs no pass over the keys
#pragma unroll
    for (int r = 0; r < R; ++r) {
        int ne = -1;
        if (on[r]) {
            ne = locate_any(P.f, Rn[r], Zn[r]);
            P.a.elem[m[r]] = ne;
        }
        if (kHist) {
            const int rk = hist_rank(P.hist, ne < 0 ? P.f.n_elems : ne, on[r]);
            if (on[r]) P.rank[m[r]] = rk;
        }
    }
}

// ---- generic push: one marker per thread, any marker order (every thread gathers its own element's tile) ------------
template <bool kHist>
__global__ void __launch_bounds__(128) push_generic_kernel(const __grid_constant__ PushParams P) {
    const long i = (long)blockIdx.x * blockDim.x + threadIdx.x;
    const bool valid = i < P.n;
    const int e = valid ? P.a.elem[i] : -1;
    const long m[1] = {i};
    const bool on[1] = {e >= 0};             // lost markers are frozen (G12)
    if (__any_sync(0xffffffffu, on[0])) step_R<1, false>(P, e, m, on);
    if (kHist) {
        const int ne = valid ? P.a.elem[i] : -1;
        const int rk = hist_rank(P.hist, ne < 0 ? P.f.n_elems : ne, valid);
        if (valid) P.rank[i] = rk;
    }
}

// ---- element-ordered push: the marker stream is sorted by element and cut into work items --------------------------
// A work item is up to kItemMarkers = 32 kItemR consecutive markers of ONE element; a warp takes an item, every lane up to
// kItemR of its markers (slots lane, lane + 32, ...), so that each 32-byte coefficient load is a one-wavefront broadcast
// that feeds kItemR markers per lane.  Persistent warps draw items from an atomic counter.  Items of the pseudo-element n_elems hold the lost
// markers: they are frozen and only enter the histogram.
template <int R, bool kHist>
__device__ __forceinline__ void item_R(const PushParams &P, int e, int start, int count) {
    const int lane = threadIdx.x & 31;
    long m[R];
    bool on[R];
#pragma unroll
    for (int r = 0; r < R; ++r) { m[r] = (long)start + 32 * r + lane; on[r] = 32 * r + lane < count; }
    step_R<R, kHist>(P, e, m, on);
}

// Lines of the next item's marker state (8 arrays x at most 5 lines of 128 B) and of its coefficient tile, one
// prefetch per lane: they travel while the current item computes.
__device__ __forceinline__ void prefetch_item(const PushParams &P, int e, int start) {
    const int lane = threadIdx.x & 31;
    const double *const arr[8] = {P.a.x, P.a.y, P.a.z, P.a.vx, P.a.vy, P.a.vz, P.a.mu, P.a.w};
    const double *base = arr[lane >> 2] + (start & ~15);
    constexpr int kLines = (kItemMarkers * 8 + 127) / 128 + 1;
#pragma unroll
    for (int j = 0; j < (kLines + 3) / 4; ++j)
        if (4 * j + (lane & 3) < kLines) asm volatile("prefetch.global.L1 [%0];" ::"l"(base + 16 * (4 * j + (lane & 3))));
    if (e < P.f.n_elems) prefetch_tile(P.f, e);
}

template <bool kHist>
__global__ void __launch_bounds__(kPushThreads, M3DK_PUSH_MINBLOCKS) push_items_kernel(const __grid_constant__ PushParams P) {
    const int lane = threadIdx.x & 31;
    const int total = *P.n_items;
    // static assignment: the warps of a CTA take consecutive items (mostly the same element: shared L1 lines)
    constexpr int kWarps = kPushThreads / 32;
    const int stride = gridDim.x * kWarps;
    int it = blockIdx.x * kWarps + (threadIdx.x >> 5);
    int4 w = make_int4(P.f.n_elems, 0, 0, 0);
    if (it < total) { w = __ldg(P.items + it); prefetch_item(P, w.x, w.y); }
    while (it < total) {
        const int e = w.x, start = w.y, count = w.z;   // (element, first slot, count, -)
        it += stride;
        if (it < total) { w = __ldg(P.items + it); prefetch_item(P, w.x, w.y); }
        if (e >= P.f.n_elems) {                        // lost markers: frozen (G12), counted for the next sort
            if (kHist) {
#pragma unroll 1
                for (int k = lane; k < ((count + 31) & ~31); k += 32) {
                    const bool onk = k < count;
                    const int rk = hist_rank(P.hist, P.f.n_elems, onk);
                    if (onk) P.rank[start + k] = rk;
                }
            }
            continue;
        }
        item_R<kItemR, kHist>(P, e, start, count);
    }
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
    P.dt = dt; P.q = c->q; P.m = c->m; P.inv_q = 1.0 / c->q;
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

cudaError_t launch_locate(m3dk_ctx *c, const MarkerArrays &a, long n, bool fill_id) {
    if (n == 0) return cudaSuccess;
    const unsigned grid = (unsigned)((n + 255) / 256);
    c->kernel_launches += 1;
    locate_kernel<<<grid, 256, 0, c->stream>>>(c->f, a, n, fill_id ? 1 : 0);
    return cudaGetLastError();
}

cudaError_t launch_push(m3dk_ctx *c, const MarkerArrays &a, long n, double dt, double t, bool with_hist, bool use_items) {
    if (n == 0) return cudaSuccess;
    PushParams P = make_params(c, a, n, dt, t);
    c->kernel_launches += 1;
    if (with_hist) {
        P.hist = c->sb.hist; P.rank = c->sb.rank;
        cudaError_t e = cudaMemsetAsync(c->sb.hist, 0, (size_t)(c->f.n_elems + 1) * sizeof(int), c->stream);
        if (e != cudaSuccess) return e;
    }
    if (use_items) {
        P.items = c->sb.items; P.n_items = c->sb.ioffs + c->f.n_elems + 1; P.item_counter = c->d_count + 1;
        cudaError_t e = cudaMemsetAsync(c->d_count + 1, 0, sizeof(int), c->stream);
        if (e != cudaSuccess) return e;
        const unsigned grid = (unsigned)(c->sm_count * M3DK_PUSH_MINBLOCKS);
        if (with_hist) push_items_kernel<true><<<grid, kPushThreads, 0, c->stream>>>(P);
        else push_items_kernel<false><<<grid, kPushThreads, 0, c->stream>>>(P);
    } else {
        const unsigned grid = (unsigned)((n + 127) / 128);
        if (with_hist) push_generic_kernel<true><<<grid, 128, 0, c->stream>>>(P);
        else push_generic_kernel<false><<<grid, 128, 0, c->stream>>>(P);
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
