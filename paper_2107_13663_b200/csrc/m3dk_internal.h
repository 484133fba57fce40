// m3dk_internal.h -- host-side context and the parameter blocks handed to the kernels.
// Part of libm3dk (product path).  Shares nothing with oracle/.
#pragma once

#include <cuda_runtime.h>
#include <stddef.h>
#include <stdint.h>

#include <string>
#include <utility>
#include <vector>

#include "../../include/m3dk.h"

namespace m3dk {

// ---- device data layout -------------------------------------------------------------------
// Element tile, `tile_stride` doubles, 128-byte aligned:
//   [0..15]   header: R_c, Z_c, s_e, 13 x pad
//   [16..57]  pair A: (psi0_k, |B|0_k) k = 0..20   interleaved so that one 16-byte load feeds two Horner chains
//   [58..99]  pair B: (F0_k, kappa_k)
//   per mode m: 7 pairs (re_k, im_k) of E_R E_phi E_Z B_R B_phi B_Z B_par, 42 doubles each (294 per mode)
constexpr int kTileHeader = 16;
constexpr int kPair = 2 * M3DK_NCOEF;                 // 42
constexpr int kTileEq = 2 * kPair;                    // 84
constexpr int kTileMode = M3DK_N_PERT * kPair;        // 294
inline int tile_stride_doubles(int n_modes) {
    int n = kTileHeader + kTileEq + kTileMode * n_modes;
    return (n + 15) / 16 * 16;
}
// Edge record of one element for the search, 16 doubles = one 128-byte line:
//   3 x (r_a, z_a, r_b - r_a, z_b - z_a), strict-interior tolerance, 3 x pad
constexpr int kEdgeRec = 16;

struct GridParams {          // bucket grid of the element search
    double Rmin, Rmax, Zmin, Zmax, inv_hx, inv_hz;
    int gx, gz;
    const int *bstart;       // [gx*gz + 1]
    const int *bcand;        // candidate elements, per bucket in priority order
    const double *edges;     // [n_elems][kEdgeRec]
};

struct FieldParams {
    const double *tiles;
    int tile_stride;         // doubles
    int n_elems;
    int n_modes;
    int n_tor[M3DK_MAX_MODES];
    double omega[M3DK_MAX_MODES];
    GridParams grid;
};

struct MarkerArrays {
    double *x, *y, *z, *vx, *vy, *vz, *mu, *w;
    int *elem, *id;
};

struct PushParams {
    long n;
    MarkerArrays a;
    FieldParams f;
    double dt, h;            // h = q dt / (2 m)
    double q, m, inv_q;
    int f0kind;
    double f0T_inv, f0vc3, f0L0, f0dL2_inv, f0Bax;
    double cwt[M3DK_MAX_MODES], swt[M3DK_MAX_MODES];   // cos / sin (omega_k t_l) of this step
};

struct SortBuffers {         // carved from the sort workspace
    MarkerArrays alt;        // second set of marker arrays (ping-pong partner of the caller's)
    int *rank;               // [n]
    int *hist;               // [n_elems + 2]
    int *offs;               // [n_elems + 2]
    size_t bytes;
};

}  // namespace m3dk

struct m3dk_ctx {
    int device = 0;
    cudaStream_t stream = nullptr;
    std::string err;
    // fields
    bool have_fields = false;
    m3dk::FieldParams f{};
    // markers
    bool have_markers = false;
    long n = 0;
    m3dk::MarkerArrays user{};   // caller's arrays
    int cur = 0;                 // 0: state lives in `user`, 1: in sb.alt (only transiently inside push / sort)
    double q = 1.0, m = 1.0;
    m3dk_f0_params f0{};
    // options / clock
    int sort_interval = 0;
    int mode = 0;
    double t0 = 0.0;
    long steps_done = 0;
    long steps_since_sort = 0;
    long n_sorts = 0;
    double last_dt = 0.0;
    // sort workspace
    bool have_sortws = false;
    m3dk::SortBuffers sb{};
    int *d_count = nullptr;      // small device scratch inside the fields workspace (lost counter etc.)
    // profiling (m3dk_set_profiling / m3dk_timing)
    bool profiling = false;
    std::vector<std::pair<cudaEvent_t, cudaEvent_t>> ev_push, ev_sort;
    double push_ms = 0.0, sort_ms = 0.0;
    long push_launches = 0, sort_launches = 0, kernel_launches = 0;
};

namespace m3dk {

// launchers (defined in push.cu / sort.cu); all enqueue on ctx->stream and return cudaGetLastError()
cudaError_t launch_locate(m3dk_ctx *c, const MarkerArrays &a, long n, bool fill_id);
cudaError_t launch_push(m3dk_ctx *c, const MarkerArrays &a, long n, double dt, double t);
cudaError_t launch_eval_fields(m3dk_ctx *c, long n, const double *R, const double *phi, const double *Z, double t,
                               int *elem_out, double *out);
cudaError_t launch_count_lost(m3dk_ctx *c, const MarkerArrays &a, long n, int *d_count);
cudaError_t launch_sort(m3dk_ctx *c, const MarkerArrays &src, const MarkerArrays &dst, long n);
cudaError_t fp64_probe(m3dk_ctx *c, double *tflops);

size_t sort_workspace_bytes(long n, int n_elems);
void carve_sort_workspace(void *ws, long n, int n_elems, SortBuffers *sb);

}  // namespace m3dk
