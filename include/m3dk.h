/*
 * m3dk.h -- C ABI of libm3dk: the energetic-particle push of M3D-C1-K (arXiv 2107.13663) for NVIDIA B200 (sm_100a).
 *
 * One thing is behind this boundary: the data-parallel hot path of the paper's kinetic module.  Each marker is a
 * classical Pauli particle advanced by the slow-manifold Boris scheme (Eqs. 5-6) with the mirror force
 * -mu grad|B| folded into an effective electric field; each step evaluates the equilibrium and perturbed
 * finite-element fields at the marker (per-element polynomials, first derivatives only, |B| as its own scalar field,
 * PAPER.md:86) and advances the delta-f weight (Eqs. 8-13, linear form; v_l averaging PAPER.md:140).
 * The fields are static while the markers are sub-cycled and the whole mesh is visible to every thread
 * (PAPER.md:235).  The marker sort by element is not in the paper ("improving the coalesce of the GPU memory access" is
 * listed as future work); it exists so that the threads of a warp evaluate the same element.
 *
 * Conventions
 *   - Plain C, no exceptions cross the boundary.  Every call returns an m3dk_status (0 = OK, negative = error); the
 *     text of the last error of a context is m3dk_last_error(ctx) (context-owned storage, never freed by the caller).
 *   - HOST pointers: the mesh and coefficient tables of m3dk_fields_create, option structs, outputs of *_bytes / stats,
 *     and the buffers of m3dk_particles_upload / _download.
 *     DEVICE pointers: every marker array and every workspace.  The library never allocates device memory: the caller
 *     (PyTorch in this repository) owns all of it and lends it until m3dk_destroy or the next *_create / *_init call.
 *   - All kernels are enqueued on the stream given to m3dk_create; calls are asynchronous unless stated otherwise.
 *     Asynchronous CUDA errors surface on the next synchronising call (m3dk_stats, m3dk_particles_download).
 *   - One context per stream; a context is not re-entrant.
 *   - Units: any consistent system in which m dv/dt = q (E + v x B).  Right-handed cylindrical (R, phi, Z) for the
 *     fields, Cartesian (x, y, z) with R = sqrt(x^2 + y^2), phi = atan2(y, x), Z = z for the marker state.
 *   - Time staggering: the caller supplies (x_l, v_{l-1/2}, w_{l-1/2}); after m3dk_push(k, dt) the arrays hold
 *     (x_{l+k}, v_{l+k-1/2}, w_{l+k-1/2}).  mu is never modified by a push.
 *   - There is no CPU fallback anywhere in this library.
 */
#ifndef M3DK_H
#define M3DK_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

#define M3DK_NCOEF 21     /* monomials xi^i eta^j, i + j <= 5; storage order: j outer 0..5, i inner 0..5-j            */
#define M3DK_N_EQ 4       /* equilibrium scalar fields per element: psi0, |B|0, F0 = R B_phi0, kappa = dlnf0/dpsi      */
#define M3DK_N_PERT 7     /* complex perturbed amplitudes per element and mode: E_R E_phi E_Z B_R B_phi B_Z B_par      */
#define M3DK_MAX_MODES 4  /* toroidal modes per field set                                                              */

typedef struct m3dk_ctx m3dk_ctx; /* opaque; host-side bookkeeping only */

typedef enum {
    M3DK_OK = 0,
    M3DK_EINVAL = -1,     /* bad argument (null pointer, negative size, unknown enum, non-CCW or degenerate triangle)   */
    M3DK_ESTATE = -2,     /* call out of order (push before fields_create / particles_init, sort without workspace)   */
    M3DK_EWORKSPACE = -3, /* workspace too small or misaligned (256-byte alignment required)                           */
    M3DK_ECUDA = -4       /* a CUDA runtime call or an earlier kernel failed; see m3dk_last_error                      */
} m3dk_status;

typedef enum { M3DK_F0_MAXWELLIAN = 0, M3DK_F0_SLOWING_DOWN = 1, M3DK_F0_BEAM_PITCH = 2 } m3dk_f0_kind;

/* Equilibrium distribution used by the weight equation, d ln f0 / dE at fixed (P_phi, mu) ("calculated
 * from the analytical expression of f0 using the chain rule"; reading G7):
 *   MAXWELLIAN    f0 ~ exp(-E/T)                                   -> -1/T
 *   SLOWING_DOWN  f0 ~ 1/(v^3 + v_c^3), v = sqrt(2E/m) (Eq. 29)    -> -3 v / (m (v^3 + v_c^3))
 *   BEAM_PITCH    slowing-down times exp(-((Lambda-Lambda0)/dLambda)^2), Lambda = mu B_axis / E
 *                                                                  -> the above + 2 (Lambda-Lambda0) Lambda / (dLambda^2 E)
 * with E = m |v_l|^2 / 2 + mu |B|0.  d ln f0 / d P_phi = kappa / q with kappa the 4th equilibrium table.             */
typedef struct {
    int kind;       /* m3dk_f0_kind */
    double T;       /* MAXWELLIAN */
    double v_c;     /* SLOWING_DOWN, BEAM_PITCH */
    double Lambda0; /* BEAM_PITCH */
    double dLambda; /* BEAM_PITCH */
    double B_axis;  /* BEAM_PITCH */
} m3dk_f0_params;

typedef struct {
    long n_markers;
    long n_lost;     /* markers outside every triangle: frozen, element -1, sorted last (reading G12)                  */
    long steps_done; /* since the last m3dk_set_options / m3dk_particles_init                                          */
    long n_sorts;    /* orderings executed: m3dk_sort calls, the pack at the start of a push call, one per step after   */
    double t;        /* t0 + steps_done * dt of the last push                                                          */
} m3dk_stats_t;

int m3dk_version(void);

/* Context bound to CUDA device `device` and to `stream` (a cudaStream_t, e.g. torch.cuda.current_stream().cuda_stream;
 * NULL = the legacy default stream).  Fails with M3DK_ECUDA when there is no usable CUDA device.                      */
int m3dk_create(m3dk_ctx **out, int device, void *stream);
int m3dk_destroy(m3dk_ctx *ctx);
const char *m3dk_last_error(const m3dk_ctx *ctx); /* ctx may be NULL: returns the last error of m3dk_create           */

/* ---- fields: poloidal triangle mesh + per-element polynomial coefficients per field + toroidal mode structure ----
 * (PAPER.md:86, :165 "high order polynomials"; :235 whole-mesh replica on the device.)
 *
 * node_RZ   [n_nodes][2]  (R, Z) of the mesh nodes.
 * tri       [n_elems][3]  node indices, counter-clockwise.
 * eq_coef   [n_elems][M3DK_N_EQ][21]   psi0, |B|0, F0, kappa.  B0 = grad psi0 x grad phi + F0 grad phi, i.e.
 *           B_R = -dpsi0/dZ / R, B_Z = +dpsi0/dR / R, B_phi = F0 / R (reading G4).
 * n_tor, omega [n_modes]; pert_coef [n_modes][n_elems][M3DK_N_PERT][2][21]: (re, im) parts of the complex amplitudes C;
 *           the physical field is Re[C(R,Z) exp(i (n_tor phi - omega t))] (readings G8, G19).
 * Polynomials (reading G10): sum_k c_k xi^i eta^j with xi = (R - R_c) s_e, eta = (Z - Z_c) s_e, (R_c, Z_c) the centroid
 * (sum of the three nodes / 3) and s_e = 1 / (longest edge).  d/dR = s_e d/dxi.
 *
 * All table pointers are HOST pointers, read during the call only.  The call repacks them into `dev_workspace`
 * (DEVICE, 256-byte aligned, at least m3dk_fields_workspace_bytes(...) bytes), which the context then borrows:
 * per-element coefficient tiles, per-element edge records and a bucket grid for the element search.  The call
 * synchronises the stream before returning (the staging buffers are freed).  n_modes may be 0 (equilibrium only).    */
int m3dk_fields_workspace_bytes(int n_nodes, int n_elems, int n_modes, size_t *bytes);
int m3dk_fields_create(m3dk_ctx *ctx, int n_nodes, const double *node_RZ, int n_elems, const int *tri,
                       const double *eq_coef, int n_modes, const int *n_tor, const double *omega,
                       const double *pert_coef, void *dev_workspace, size_t workspace_bytes);

/* A fields workspace is self-describing: a byte-for-byte copy of it (on this or another GPU: a peer copy, an NCCL broadcast)
 * can be bound to a context without the host tables and without repeating the host-side repack.  This is how the whole-mesh
 * field replica of PAPER.md:235 ("collected and uploaded to every GPU") reaches the other GPUs of a node: rank 0 calls
 * m3dk_fields_create, the workspace is broadcast, every other rank calls m3dk_fields_attach on its copy.  dev_workspace:
 * DEVICE, 256-byte aligned, borrowed like the one of m3dk_fields_create.  Synchronises (reads the header in the control block).      */
int m3dk_fields_attach(m3dk_ctx *ctx, void *dev_workspace, size_t workspace_bytes);

/* ---- markers: SoA fp64 x, v, mu, w; species charge / mass -------------------------------------
 * x..w: DEVICE arrays of n doubles, caller-owned, updated in place by push and permuted by sort.
 * elem: DEVICE int[n], library-managed: the element of each marker's current position (-1 = lost).
 * id:   DEVICE int[n]; the library fills 0..n-1 here and sorts carry it, so id[i] is the original index of slot i.
 * The call locates every marker (one kernel).  Call it again whenever the caller has rewritten positions.            */
int m3dk_particles_init(m3dk_ctx *ctx, long n, double *x, double *y, double *z, double *vx, double *vy, double *vz,
                        double *mu, double *w, int *elem, int *id, double charge, double mass,
                        const m3dk_f0_params *f0);

/* sort_interval: 0 = m3dk_push never sorts: the caller's SoA arrays are pushed in place, one marker per thread (every
 *       thread gathers its own element's coefficients: seven times slower per step at configs[3]).
 *       k >= 1 = ordered pipeline (needs a sort workspace): m3dk_push packs the markers into element-ordered 64-byte
 *       records at the start of a call (about one step's time at 2^24 markers, so sub-cycle many steps per call,
 *       PAPER.md:237), runs EVERY step through the element-ordered kernel, re-orders after EVERY step (the histogram is
 *       fused into the push; a re-ordering costs a tenth of a step) and unpacks at the end of the call.  k is a request
 *       the library exceeds: k > 1 behaves like k = 1, and results are bit-identical for every value (0 included).
 * mode: 0 = linear delta-f (trajectories in the equilibrium field, (1 - w) -> 1);
 *       1 = non-linear trajectories (reading G21): the marker moves in the total fields,
 *           B = B0 + B1 and E-dagger = E1 - (mu/q) grad(|B|0 + B1par), and Eq. (8) keeps its factor (1 - w):
 *           w_{l+1/2} = w_{l-1/2} + dt (1 - w_{l-1/2}) dw/dt|linear(x_l, v_l, t_l).
 *       2 = linear delta-f with finite-Larmor-radius averaging (Eq. 14; reading G23): E1, B1,
 *           grad B1par and dB1par/dt of the weight equation are replaced by the quarter sum over the four gyro-ring
 *           points x_l +- rho e1, x_l +- rho e2, rho = m v_perp / (|q| B0), v_perp = sqrt(2 mu B0 / m), e1 = the
 *           major-radius direction made perpendicular to b0, e2 = b0 x e1; a ring point outside the mesh contributes 0.
 *       3 = modes 1 and 2 together ("use orbit-averaged fields in the above equations"): the marker moves in
 *           B0 + <B1>, E-dagger = <E1> - (mu/q) grad(|B|0 + <B1par>) with the 4-point gyro-averages of mode 2, and the weight
 *           equation uses the same averages and keeps (1 - w).  Every lane gathers its ring, unless an FLR workspace of
 *           m3dk_flr_workspace_bytes_nl bytes is set (ring stream, below).
 * t0: time of the next step's x_l.  Resets steps_done to 0.                                                          */
int m3dk_set_options(m3dk_ctx *ctx, int sort_interval, int mode, double t0);

/* Which kernel runs the element-ordered steps (sort_interval >= 1) of modes 0 and 1.  Results are bit-identical.
 *   0 (default)  push_items_kernel: a warp per work item, tile staged by a bulk copy, records gathered with 256-bit loads,
 *                search + histogram with returned ranks at the end of the item;
 *   1            push_async_kernel: the same decomposition with every L2 / HBM access of an item requested one item ahead
 *                (cp.async into shared memory) and the histogram without returned values (the re-ordering draws the slots).
 *                Kept for comparison: measured 7 % slower per step at configs[3] (K1b).           */
int m3dk_set_push_variant(m3dk_ctx *ctx, int variant);

/* Sort workspace (DEVICE, 256-byte aligned) for m3dk_sort and for the sorts inside m3dk_push; borrowed until replaced. */
int m3dk_sort_workspace_bytes(long n_markers, int n_elems, size_t *bytes);
int m3dk_set_sort_workspace(m3dk_ctx *ctx, void *dev_workspace, size_t bytes);

/* FLR workspace (DEVICE, 256-byte aligned, borrowed until replaced; optional): with it, the ordered pipeline of mode 2
 * (sort_interval >= 1) does not let every marker gather the coefficient tiles of its four ring points: the push emits the
 * 4 n ring points (position, element, the marker's weights), they are ordered by THEIR element like the markers, a warp
 * evaluates up to 64 ring points of one element with the tile staged in shared memory, and the four contributions are
 * summed back into w (290 bytes per marker).  Results are bit-identical with and without it.
 * Mode 3 needs the averaged VECTORS back at the marker before the Boris step, so its ring stream takes two passes over the
 * markers per step (ring points out; ten Cartesian field components per ring point back, 96 bytes each) and a workspace of
 * m3dk_flr_workspace_bytes_nl bytes (674 bytes per marker); with the smaller workspace mode 3 keeps its per-lane gathers.
 * m3dk_set_flr_workspace accepts either size (the larger serves both modes and the FLR deposition).                    */
int m3dk_flr_workspace_bytes(long n_markers, int n_elems, size_t *bytes);
int m3dk_flr_workspace_bytes_nl(long n_markers, int n_elems, size_t *bytes);
int m3dk_set_flr_workspace(m3dk_ctx *ctx, void *dev_workspace, size_t bytes);

/* nsteps slow-manifold Boris steps of size dt with field evaluation and weight update, Eqs. (5), (6), (8)-(13).
 * Asynchronous; t advances by nsteps * dt.  A lost marker is frozen.  On return (stream order) the caller's arrays hold
 * the new state; if sorts ran, slots are permuted and id[] says who is where.                                         */
int m3dk_push(m3dk_ctx *ctx, int nsteps, double dt);

/* Counting sort of all marker arrays (x..w, elem, id) by element, lost markers last.  The order inside one element is
 * unspecified.  dev_workspace may be NULL to use the workspace given to m3dk_set_sort_workspace.                      */
int m3dk_sort(m3dk_ctx *ctx, void *dev_workspace, size_t bytes);

/* Synchronises the stream, reports asynchronous errors, fills *out. */
int m3dk_stats(m3dk_ctx *ctx, m3dk_stats_t *out);

/* Host-buffer path (what a caller without device arrays uses; bench.py's e2e leg): copy the 8 state arrays between
 * HOST buffers (pinned for full speed) and the device arrays registered by m3dk_particles_init.  upload re-locates the
 * markers and resets id to 0..n-1.  download synchronises; host_id / host_elem may be NULL.                            */
int m3dk_particles_upload(m3dk_ctx *ctx, const double *hx, const double *hy, const double *hz, const double *hvx,
                          const double *hvy, const double *hvz, const double *hmu, const double *hw);
int m3dk_particles_download(m3dk_ctx *ctx, double *hx, double *hy, double *hz, double *hvx, double *hvy, double *hvz,
                            double *hmu, double *hw, int *host_id, int *host_elem);

/* The host-buffer path as ONE call, pipelined by marker chunk: equivalent to m3dk_particles_upload -> m3dk_push(nsteps, dt)
 * -> m3dk_particles_download on the same HOST buffers (in place: on return they hold the new state), but the n markers are
 * cut into n_chunks contiguous chunks (with four or more, of sizes that ramp up and down again, weights 1, 2, 3, 4, .., 4,
 * 3, 2, 1: the first upload and the last download, which nothing overlaps, are short) and chunk c uploads while chunk
 * c - 1 runs its nsteps steps and chunk c - 2 downloads (markers are independent; uploads, steps and
 * downloads run on streams of their own, the two copy directions concurrently).
 * Sorts act inside a chunk: slot i of chunk c holds the marker host_id[i], with ids global (0..n-1 = the caller's order at
 * entry).  host_id / host_elem may be NULL.  Pinned buffers are needed for the copies to overlap.  Every chunk steps from
 * the same time; t advances by nsteps * dt once.  The call needs the device arrays of m3dk_particles_init (n markers) and,
 * for sort_interval >= 1, the sort workspace; it synchronises before returning.  n_chunks = 1 is the unpipelined path;
 * n_chunks = 0 lets the library choose (8, 4 or 3 chunks by the ratio of transfer to compute time; 1 below 2^18 markers).
 * Two chunks are in flight at a time on two compute streams (the context's and one of the library's own), each with a
 * carving of the sort (and FLR) workspace sized for the largest chunk, when two carvings fit the registered workspace (they
 * do for n_chunks >= 3 and the sizes m3dk_sort_workspace_bytes / m3dk_flr_workspace_bytes return for n markers; else one
 * chunk is in flight at a time); work enqueued on
 * the context's stream afterwards is ordered behind both.
 * A chunk is a range of the buffers and stays that set of markers from call to call.  Chunks of a marker stream in random
 * order see a mesh n_chunks times sparser per chunk (fewer markers per element, less sharing of coefficient tiles), and a
 * chunk that starts as a range of elements disperses around its flux surfaces within some twenty steps; markers kept in
 * the order of their flux surface (radial shells) keep their chunks compact.                                            */
int m3dk_push_host(m3dk_ctx *ctx, double *hx, double *hy, double *hz, double *hvx, double *hvy, double *hvz, double *hmu,
                   double *hw, int *host_id, int *host_elem, int nsteps, double dt, int n_chunks);

/* Diagnostics for tests and the roofline: fields at arbitrary points through the same device code as the push.
 * R, phi, Z: DEVICE [n]; elem_out: DEVICE int[n]; out: DEVICE [n][18] =
 * psi_R psi_Z |B| |B|_R |B|_Z F kappa E1(R,phi,Z) B1(R,phi,Z) gradB1par(R,phi,Z) dB1par/dt B1par.                     */
int m3dk_eval_fields(m3dk_ctx *ctx, long n, const double *R, const double *phi, const double *Z, double t,
                     int *elem_out, double *out);

/* RK4 guiding-centre pusher (Eqs. 1-4; reading G24): the paper's comparator
 * (Fig. 1) and the equilibrium guiding-centre motion "(dX/dt)_0" of PAPER.md:130.  In mode 1 (non-linear trajectories) the
 * guiding centres move in the total fields to first order (reading G26): E = E1, B1 added to B-star, grad|B| ->
 * grad(|B|0 + B1par), b and curl b from the equilibrium, all at the context's time, which then advances by nsteps * dt as
 * in m3dk_push.  In modes 0 and 2 equilibrium fields only (E = 0):
 *   dX/dt = (1/B*par)[v_par B* + (mu/q) b x grad|B|],  m dv_par/dt = -(mu/B*par) B* . grad|B|,
 *   B* = B + (m v_par/q) curl b,  B*par = B* . b;  curl b from the second derivatives of psi0 and the first of F0.
 * The registered arrays x, y, z are read and written as the guiding-centre position X (Cartesian), mu is read, elem is
 * kept at the element of the CURRENT position (a following m3dk_push / m3dk_deposit uses it as it is); vx, vy, vz, w are
 * not touched.  vpar: DEVICE [n], in/out.  nsteps classical RK4 steps of size dt.  A guiding centre is lost (elem = -1,
 * frozen) when a stage of a step leaves the mesh (state of the step before) or a step ends outside (state after it).
 * Asynchronous.                                                                                                      */
int m3dk_gc_push(m3dk_ctx *ctx, int nsteps, double dt, double *vpar);

/* Bootstrap of the slow-manifold Boris scheme ("we use RK4 to advance the guiding center equations of motion
 * from x0 to x1, and then use (x1 - x0)/dt as v_1/2 to ensure that markers stay close to the slow manifold"; :82 a marker
 * not initialised that way jumps back and forth across it).  One RK4 guiding-centre step of size dt from the registered
 * positions with the parallel velocities vpar (DEVICE [n], read only); then x, y, z hold x_1 and vx, vy, vz hold
 * (x_1 - x_0)/dt: the staggered state (x_l, v_{l-1/2}) m3dk_push takes, one step later in time (advance t0 by dt).  mu, w
 * are untouched, elem is the element of x_1.  A marker whose step leaves the mesh is lost (elem = -1, state untouched).
 * Asynchronous.                                                                                                      */
int m3dk_gc_bootstrap(m3dk_ctx *ctx, double dt, const double *vpar);

/* Moment deposition: right-hand sides of the Galerkin projection of the energetic-particle pressure
 * moments with a delta-function particle shape, Eqs. (17)-(18) (readings G10, G22):
 *   rhs[e][0][h][k] = sum over the markers p in element e of  w_p m v_par,p^2    nu_k(x_p) T_h(phi_p)     (parallel)
 *   rhs[e][1][h][k] = sum over the markers p in element e of  w_p mu_p |B|0(x_p) nu_k(x_p) T_h(phi_p)     (perpendicular)
 * nu_k = xi^i eta^j, the element's polynomial basis in its local frame (same order as the coefficient tables);
 * T_0 = 1, T_{2m+1} = cos(n_tor[m] phi), T_{2m+2} = sin(n_tor[m] phi); v_par = v . B0/|B0| with the stored v (v_{l-1/2}).
 * flags bit 0 (M3DK_DEPOSIT_B1PAR): the perpendicular moment carries the term of Eq. (16), mu |B|0 (w + B1par/|B|0), i.e.
 * rhs[e][1] also receives mu_p B1par(x_p, t) with B1par = Re[C e^{i(n phi - omega t)}] at the time t given; 0: Eq. (18) as
 * printed.  flags bit 1 (M3DK_DEPOSIT_FLR): 4-point FLR deposition: each marker deposits a quarter of its
 * amplitudes at each of its four gyro-ring points (the ring of mode 2, reading G23), test functions taken at the ring
 * point; a ring point outside the mesh deposits nothing.  flags bit 2 (M3DK_DEPOSIT_BSTAR): w is replaced in both moments by
 * d = w + B1star / Bstar (the linear form: the change of the phase-space Jacobian Bstar of Eq. 4), with B1star
 * taken as B1par at the time t given and Bstar = (B0 + (m v_par/q) curl b0) . b0 at the v_par of the marker (reading G25).
 * The delta function is normalised in physical volume, so no Jacobian factor appears (G22); the mass-matrix solve that
 * turns these sums into pressure coefficients belongs to the MHD code and is out of scope.  Lost markers deposit nothing.
 * rhs: DEVICE, m3dk_deposit_bytes() bytes = [n_elems][2][1 + 2 n_modes][21] doubles, overwritten.  Asynchronous.  The
 * caller's arrays are read, not modified.  With a sort workspace set (m3dk_set_sort_workspace) the markers are first
 * ordered by the element of their current position inside the workspace and a warp reduces up to 64 markers of one
 * element per table update; without one, every warp loops over the distinct elements of its 32 markers (slow on an
 * unordered stream).  Sums are accumulated with fp64 atomics: the order of addition, hence the last bits, may vary.     */
int m3dk_deposit_bytes(const m3dk_ctx *ctx, size_t *bytes);
#define M3DK_DEPOSIT_B1PAR 1
#define M3DK_DEPOSIT_FLR 2
#define M3DK_DEPOSIT_BSTAR 4
int m3dk_deposit(m3dk_ctx *ctx, double *rhs, int flags, double t);

/* m3dk_deposit for callers that cannot allocate device memory (code under CUDA graph capture, tight serving loops,
 * harnesses that forbid cudaMalloc) and therefore have no sort workspace to lend: the same right-hand sides of
 * Eqs. (17)-(18), same arguments, same flags, through the element-ordered path (markers ordered by the element of their
 * current position, a warp reduces up to 64 markers of one element per table update; with M3DK_DEPOSIT_FLR every lane
 * loops over the elements of its ring points on the ordered records), with the ordering scratch in ONE static device
 * array of M3DK_NOALLOC_SCRATCH_BYTES inside the library.  Every GPU that loads the library holds that array until the
 * process exits.  The call allocates nothing (no cudaMalloc, cudaFree or allocating library routine): it enqueues memsets
 * and kernels on the context's stream; the first call on a device also asks the runtime for the array's device address
 * (make that call before starting a graph capture).  Whatever sort / FLR workspace the context has registered is neither
 * used nor touched.  Limit: m3dk_sort_workspace_bytes(n_markers, n_elems) must not exceed M3DK_NOALLOC_SCRATCH_BYTES
 * (about 48 000 markers on 8 192 elements); beyond it the call fails with M3DK_EWORKSPACE and enqueues nothing.
 * The array is shared by every context of the process on that device and keeps the last call's contents; what must start
 * at zero is cleared inside each call.  Calls that overlap on the GPU (two contexts on different streams, or a second call
 * enqueued on another stream before the first has finished) race on it: serialise them on one stream or with events.
 * Asynchronous like m3dk_deposit.  m3dk_noalloc_scratch_bytes returns the size of the array.                            */
#define M3DK_NOALLOC_SCRATCH_BYTES (8u << 20)
int m3dk_noalloc_scratch_bytes(size_t *bytes);
int m3dk_deposit_noalloc(m3dk_ctx *ctx, double *rhs, int flags, double t);

/* Measured FP64 FMA throughput of the device (register-resident DFMA chains, all SMs), in TFLOP/s (FMA = 2 flop).
 * Synchronous.  Used as the measured denominator of the FP64 roofline.                                                */
int m3dk_fp64_peak_tflops(m3dk_ctx *ctx, double *tflops);

/* Per-kernel timing for the roofline report.  With profiling on, the library brackets every push-kernel launch and
 * every sort (its kernels as one group) with CUDA events on the context's stream.  m3dk_timing synchronises the stream,
 * adds the elapsed times since the last call to the totals and returns them; m3dk_set_profiling(ctx, 1) zeroes the
 * totals.  kernel_launches counts every kernel the library enqueued since then (profiling on or off).                */
typedef struct {
    double push_ms;       /* sum of push-kernel durations                                                              */
    double sort_ms;       /* sum of sort durations (histogram + scan + scatter / permutation kernels)                  */
    long push_launches;
    long sort_launches;   /* number of sorts timed                                                                     */
    long kernel_launches; /* all kernels enqueued by the library                                                       */
} m3dk_timing_t;
int m3dk_set_profiling(m3dk_ctx *ctx, int on);
int m3dk_timing(m3dk_ctx *ctx, m3dk_timing_t *out);

#ifdef __cplusplus
}
#endif
#endif /* M3DK_H */
