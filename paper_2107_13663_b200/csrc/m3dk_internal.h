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
// Element tile, `tile_stride` doubles, 128-byte aligned.  Four polynomials are interleaved coefficient by coefficient
// ("quad"), so that one 32-byte load (LDG.E.256) feeds four independent Horner chains:
//   [0..3]    header: R_c, Z_c, s_e, pad
//   [4..87]   quad EQ: (psi0_k, |B|0_k, F0_k, kappa_k), k = 0..20
//   per mode m, 4 quads of 84 doubles (336 per mode), (re, im) parts of the complex amplitudes:
//     quad 0: (E_R re, E_R im, E_phi re, E_phi im)     quad 1: (E_Z re, E_Z im, B_R re, B_R im)
//     quad 2: (B_par re, B_par im, B_Z re, B_Z im)     quad 3: (B_phi re, B_phi im, 0, 0)
//   B_phi does not enter the linear delta-f weight equation: the push never reads quad 3 (m3dk_eval_fields does).
constexpr int kTileHeader = 4;
constexpr int kQuad = 4 * M3DK_NCOEF;                 // 84
constexpr int kTileEq = kQuad;                        // 84
constexpr int kTileMode = 4 * kQuad;                  // 336
inline int tile_stride_doubles(int n_modes) {
    int n = kTileHeader + kTileEq + kTileMode * n_modes;
    return (n + 15) / 16 * 16;
}
// Edge record of one element for the exact search, 16 doubles = one 128-byte line:
//   3 x (r_a, z_a, r_b - r_a, z_b - z_a), strict-interior tolerance, 3 x pad
constexpr int kEdgeRec = 16;

// Fast search grid (fp32, conservative): one 64-byte record per bucket, two candidate triangles each:
//   a[6], b[6]          vertices (x0 y0 x1 y1 x2 y2) of the two candidates in bucket-local units (bucket = [0,1)^2), all
//                       within [-kFastCmax+1, kFastCmax]
//   ida, idb            their element indices; ida = -1: "use the exact search for this bucket"; idb = -1: no second one
//   next                index of a record with two more candidates in the overflow array, -1 = none
// A point whose three fp32 edge functions exceed kFastMargin is strictly inside that triangle in exact arithmetic
// (error bound 720 * 2^-24 = 4.3e-5 for coordinates bounded by kFastCmax), so the exact rule G11 gives the same element.
// Two candidates per record: one 64-byte fetch settles the search for nearly every point (a bucket of the regular mesh
// meets one or two triangles), so the record of the new position can be fetched asynchronously ahead of its use.
constexpr float kFastMargin = 1.0e-4f;
constexpr double kFastCmax = 5.0;
struct FastRec { float a[6], b[6]; int ida, idb, next, pad; };
static_assert(sizeof(FastRec) == 64, "FastRec must be two 32-byte sectors");

struct FastGrid {
    double Rmin, Zmin, inv_hx, inv_hz;
    int gx, gz;
    const FastRec *first;    // [gx*gz]
    const FastRec *ovf;      // overflow records
};

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
    FastGrid fast;
};

struct MarkerArrays {
    double *x, *y, *z, *vx, *vy, *vz, *mu, *w;
    int *elem, *id;
};

// Marker record of the ordered pipeline: 64 bytes = two 32-byte sectors, fields (x, y, z, w | vx, vy, vz, mu).
// Records are gathered / written with 256-bit accesses: a marker is two full sectors wherever it lands, which is what
// makes re-ordering every step affordable (an 8-byte SoA scatter costs a 32-byte sector and an L1 wavefront per field).
constexpr int kRecDoubles = 8;

struct RecArrays {            // ordered pipeline, carved from the sort workspace
    const double *in;        // records of this step's input  [n][8]
    double *out;             // records of this step's output [n][8] (== in for the in-place generic kernel)
    const int2 *order;       // [n] (src, id): output slot d takes the input record src; id = caller's marker index
    int *key;                // [n] element of the NEW position of output slot d (n_elems = lost)
};

// Ring stream of the ordered FLR mode (mode 2 with an FLR workspace): four ring points per marker slot.
constexpr int kAvgDoubles = 12;   // ten components + two of padding: three full 32-byte sectors per ring point
struct FlrArrays {
    double *ring;            // [4 n][4] (x, y, z, -) of ring point 4 slot + j
    double *wts;             // [n][10] the marker's weights of the perturbed fields in dw/dt, Cartesian (FlrW)
    double *contrib;         // [4 n] c_j of every ring point
    int *rkey, *rrank;       // [4 n] element of the ring point (n_elems = outside, -1 = the slot holds a lost marker), rank in it
    int *rorder;             // [4 n] ring points in element order
    int *rhist;              // [n_elems + 2]
    double *avg;             // [4 n][kAvgDoubles] mode 3: Cartesian field components at every ring point (NULL: not carved)
};

struct PushParams {
    long n;
    MarkerArrays a;          // SoA path (sort_interval = 0)
    RecArrays rc;            // record path (sort_interval >= 1)
    FlrArrays fl;            // ring stream (mode 2, ordered)
    FieldParams f;
    double dt, h;            // h = q dt / (2 m)
    double q, m, inv_q, inv_m;
    int f0kind;
    double f0T_inv, f0vc3, f0L0, f0dL2_inv, f0Bax;
    double cwt[M3DK_MAX_MODES], swt[M3DK_MAX_MODES];   // cos / sin (omega_k t_l) of this step
    int *hist, *rank;        // fused sort histogram of the new keys (kHist kernels), else unused
    const int4 *items;       // work items of the element-ordered kernel: (element, first slot, count, -)
    const int *n_items;      // device: number of items
    int *ticket;             // device: next unassigned item beyond the first three rounds (cleared by the cut)
};

#ifndef M3DK_ITEM_R
#define M3DK_ITEM_R 2
#endif
constexpr int kItemR = M3DK_ITEM_R;              // markers per lane in the element-ordered push
constexpr int kItemMarkers = 32 * kItemR;        // markers per work item

struct FlrBuffers {          // carved from the FLR workspace (m3dk_set_flr_workspace)
    FlrArrays a;
    int *roffs, *rioffs;     // [n_elems + 2]
    int4 *ritems;            // [4 n / kItemMarkers + n_elems + 2]
    int4 *ritems_small;      // [n_elems + 2]
    unsigned long long *rstate;   // scan state + item tickets, as SortBuffers::scan_state
    size_t bytes;
};

struct SortBuffers {         // carved from the sort workspace
    double *rec[2];          // [n][8] record ping-pong
    int2 *order[2];          // [n] (src, id) ping-pong: order[k][d].y is also the id of the record in slot d
    int *key;                // [n]
    int *rank;               // [n]
    int *hist;               // [n_elems + 2]
    int *offs;               // [n_elems + 2]
    int *ioffs;              // [n_elems + 2] first work item of each element; ioffs[n_elems + 1] = number of items
    int4 *items;             // [n / kItemMarkers + n_elems + 2]
    int4 *items_small;       // [n_elems + 2] items of 1..32 markers (one marker per lane); their count is scan_state[1]
    unsigned long long *scan_state;   // ticket, small-item counter, per-chunk totals of the single-pass scan, then
                                      // one word holding the two item tickets of the push kernels (big, small)
    size_t bytes;
};

}  // namespace m3dk

struct m3dk_ctx {
    int device = 0;
    int sm_count = 148;
    size_t smem_optin = 0;       // cudaDevAttrMaxSharedMemoryPerBlockOptin
    int push_variant = 0;        // m3dk_set_push_variant: 0 = push_items_kernel (default), 1 = push_async_kernel (measured slower)
    cudaStream_t stream = nullptr;
    std::string err;
    // fields
    bool have_fields = false;
    m3dk::FieldParams f{};
    // markers
    bool have_markers = false;
    long n = 0;
    m3dk::MarkerArrays user{};   // caller's arrays (the state lives here between calls)
    int cur = 0;                 // record buffer that holds the state inside an ordered push / sort
    int ocur = 0;
    bool ranks_valid = true;     // the last push with a histogram also wrote rank[] (else invert_kernel draws the slots)
    unsigned scan_epoch = 0;     // tag of the current scan launch (decoupled look-back without clearing)                // order buffer whose .y are the ids of the records in sb.rec[cur]
    double q = 1.0, m = 1.0;
    m3dk_f0_params f0{};
    // options / clock
    int sort_interval = 0;
    int mode = 0;
    double t0 = 0.0;             // time of the first step after m3dk_set_options
    double t_base = 0.0;         // time at which the current run of equal steps began; t = t_base + steps_at_dt * last_dt
    long steps_at_dt = 0;
    long steps_done = 0;
    long steps_since_sort = 0;
    long n_sorts = 0;
    double last_dt = 0.0;
    // sort workspace
    bool have_sortws = false;
    m3dk::SortBuffers sb{};
    bool have_flrws = false;
    bool flr_with_avg = false;   // the FLR workspace also holds the averages array (mode 3 through the ring stream)
    m3dk::FlrBuffers fb{};
    void *flrws_base = nullptr;
    size_t flrws_bytes = 0;
    int *d_count = nullptr;      // small device scratch inside the fields workspace (lost counter etc.)
    void *sortws_base = nullptr; // the caller's sort workspace as given (re-carved when n or the mesh changes)
    size_t sortws_bytes = 0;
    // m3dk_push_host: copy streams and per-chunk events (created on first use)
    cudaStream_t s_up = nullptr, s_down = nullptr;
    cudaStream_t s_c[4] = {nullptr, nullptr, nullptr, nullptr};   // extra compute streams of the chunk pipeline (s_c[0] unused)
    int host_slots = 2;                                            // chunks in flight (measured: 2 and 4 within 1 %)
    std::vector<cudaEvent_t> ev_chunk;
    // profiling (m3dk_set_profiling / m3dk_timing)
    bool profiling = false;
    std::vector<std::pair<cudaEvent_t, cudaEvent_t>> ev_push, ev_sort;
    double push_ms = 0.0, sort_ms = 0.0;
    long push_launches = 0, sort_launches = 0, kernel_launches = 0;
};

namespace m3dk {

// launchers (defined in push.cu / sort.cu); all enqueue on ctx->stream and return cudaGetLastError()
cudaError_t launch_locate(m3dk_ctx *c, const MarkerArrays &a, long n, bool fill_id, int id_base = 0);
cudaError_t launch_push_soa(m3dk_ctx *c, long n, double dt, double t);                           // caller's arrays, any order
cudaError_t launch_push_rec(m3dk_ctx *c, long n, double dt, double t, bool with_hist);   // records, element-ordered
cudaError_t launch_eval_fields(m3dk_ctx *c, long n, const double *R, const double *phi, const double *Z, double t,
                               int *elem_out, double *out);
cudaError_t launch_count_lost(m3dk_ctx *c, const MarkerArrays &a, long n, int *d_count);
cudaError_t launch_pack_sorted(m3dk_ctx *c, long n);     // caller's arrays -> records in element order, items cut
cudaError_t launch_reorder(m3dk_ctx *c, long n);         // histogram of the last push -> offsets, items, next order
cudaError_t launch_unpack(m3dk_ctx *c, long n);          // records -> caller's arrays (+ elem, id)
cudaError_t launch_deposit(m3dk_ctx *c, long n, double *rhs, int flags, double t);   // Eqs. (17)-(18) right-hand sides from the caller's arrays
cudaError_t launch_gc_push(m3dk_ctx *c, long n, double *vpar, int nsteps, double dt, bool pert, double t0);   // RK4 guiding-centre steps
cudaError_t launch_gc_bootstrap(m3dk_ctx *c, long n, const double *vpar, double dt);     // (x_1, v_{1/2}) from one such step
cudaError_t fp64_probe(m3dk_ctx *c, double *tflops);

cudaError_t launch_flr_ring_keys(m3dk_ctx *c, long n);    // element + rank of every ring point (push.cu)
cudaError_t launch_flr_ring_stage(m3dk_ctx *c, long n);   // ring histogram -> offsets, ring items, ring order
cudaError_t launch_flr_ring_eval(m3dk_ctx *c, long n, double dt, double t, bool avg = false);   // ring_items_kernel (push.cu)
cudaError_t launch_flr_emit_nl(m3dk_ctx *c, long n, double dt, double t);   // mode 3, first pass: ring points of every marker
bool flr_nl_stream(const m3dk_ctx *c);   // mode 3 goes through the ring stream (FLR workspace with the averages array)
cudaError_t launch_flr_reduce(m3dk_ctx *c, long n, double dt);   // w += dt * quarter sum of the contributions
size_t flr_workspace_bytes(long n, int n_elems, bool with_avg = false);   // with_avg: + the averages array of mode 3
void carve_flr_workspace(void *ws, long n, int n_elems, FlrBuffers *fb, bool with_avg = false);
size_t sort_workspace_bytes(long n, int n_elems);
void carve_sort_workspace(void *ws, long n, int n_elems, SortBuffers *sb);

}  // namespace m3dk
