// m3dk_api.cu -- the C ABI of libm3dk (include/m3dk.h): argument checks, table repacking, launch logic.
// Host code only; the kernels are in m3dk_push.cu and m3dk_sort.cu.
#include <math.h>
#include <stdio.h>
#include <string.h>

#include <algorithm>
#include <vector>

#include "m3dk_internal.h"

using namespace m3dk;

static thread_local std::string g_create_error;

static int fail(m3dk_ctx *c, int code, const std::string &msg) {
    if (c) c->err = msg; else g_create_error = msg;
    return code;
}
static int cuda_fail(m3dk_ctx *c, cudaError_t e, const char *what) {
    return fail(c, M3DK_ECUDA, std::string(what) + ": " + cudaGetErrorName(e) + " (" + cudaGetErrorString(e) + ")");
}
#define CU(call, what)                                        \
    do {                                                      \
        cudaError_t e__ = (call);                             \
        if (e__ != cudaSuccess) return cuda_fail(ctx, e__, what); \
    } while (0)

static inline size_t up256(size_t b) { return (b + 255) / 256 * 256; }

// profiling brackets: a pair of events around a launch group, kept until m3dk_timing collects them
struct EvScope {
    m3dk_ctx *c; std::vector<std::pair<cudaEvent_t, cudaEvent_t>> *v; cudaEvent_t a = nullptr, b = nullptr;
    EvScope(m3dk_ctx *ctx, std::vector<std::pair<cudaEvent_t, cudaEvent_t>> *vec) : c(ctx), v(vec) {
        if (!c->profiling) return;
        if (cudaEventCreate(&a) != cudaSuccess || cudaEventCreate(&b) != cudaSuccess) { a = b = nullptr; return; }
        cudaEventRecord(a, c->stream);
    }
    ~EvScope() {
        if (!a) return;
        cudaEventRecord(b, c->stream);
        v->emplace_back(a, b);
    }
};
static void drop_events(std::vector<std::pair<cudaEvent_t, cudaEvent_t>> &v, double *acc, long *cnt) {
    for (auto &p : v) {
        float ms = 0.f;
        if (acc && cudaEventElapsedTime(&ms, p.first, p.second) == cudaSuccess) { *acc += ms; ++*cnt; }
        cudaEventDestroy(p.first); cudaEventDestroy(p.second);
    }
    v.clear();
}

extern "C" int m3dk_version(void) { return 100; }

extern "C" const char *m3dk_last_error(const m3dk_ctx *ctx) { return ctx ? ctx->err.c_str() : g_create_error.c_str(); }

extern "C" int m3dk_create(m3dk_ctx **out, int device, void *stream) {
    m3dk_ctx *ctx = nullptr;
    if (!out) return fail(nullptr, M3DK_EINVAL, "m3dk_create: out is NULL");
    *out = nullptr;
    int ndev = 0;
    CU(cudaGetDeviceCount(&ndev), "cudaGetDeviceCount (libm3dk has no CPU fallback)");
    if (device < 0 || device >= ndev) return fail(nullptr, M3DK_EINVAL, "m3dk_create: no such CUDA device");
    CU(cudaSetDevice(device), "cudaSetDevice");
    ctx = new m3dk_ctx();
    ctx->device = device;
    ctx->stream = static_cast<cudaStream_t>(stream);
    if (cudaDeviceGetAttribute(&ctx->sm_count, cudaDevAttrMultiProcessorCount, device) != cudaSuccess || ctx->sm_count < 1)
        ctx->sm_count = 148;
    int optin = 0;
    if (cudaDeviceGetAttribute(&optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, device) == cudaSuccess && optin > 0)
        ctx->smem_optin = (size_t)optin;
    *out = ctx;
    return M3DK_OK;
}

extern "C" int m3dk_destroy(m3dk_ctx *ctx) {
    if (!ctx) return M3DK_EINVAL;
    drop_events(ctx->ev_push, nullptr, nullptr);
    drop_events(ctx->ev_sort, nullptr, nullptr);
    for (cudaEvent_t e : ctx->ev_chunk) cudaEventDestroy(e);
    if (ctx->s_up) cudaStreamDestroy(ctx->s_up);
    if (ctx->s_down) cudaStreamDestroy(ctx->s_down);
    for (cudaStream_t st : ctx->s_c) if (st) cudaStreamDestroy(st);
    delete ctx;
    return M3DK_OK;
}

// ---- fields --------------------------------------------------------------------------------------------------------
// workspace: [control block 256 B][tiles][edge records][bstart][bcand (<= kCandPerElem * n_elems)]
//            [fast grid: first records gf*gf][overflow records: at most one per bucket, gf*gf]
static constexpr int kCandPerElem = 24;

// Header of a fields workspace, kept in its control block at byte 32 (bytes 0..31 are device scratch): everything
// m3dk_fields_attach needs to rebuild the context's FieldParams from a byte-for-byte copy of the workspace on another GPU.
struct FieldsHeader {
    unsigned long long magic;
    unsigned long long off_tiles, off_edges, off_bstart, off_bcand, off_ffirst, off_fovf, total_bytes;
    double Rmin, Rmax, Zmin, Zmax, inv_hx, inv_hz, finv_hx, finv_hz;
    double omega[M3DK_MAX_MODES];
    int n_tor[M3DK_MAX_MODES];
    int n_elems, n_modes, tile_stride, g, gf, pad;
};
static_assert(sizeof(FieldsHeader) <= 224, "the header must fit the control block behind the 32 bytes of scratch");
static constexpr unsigned long long kFieldsMagic = 0x4d33444b46313030ull;   // "M3DKF100"

static void bind_fields(m3dk_ctx *ctx, char *base, const FieldsHeader &h) {
    FieldParams &f = ctx->f;
    f = FieldParams{};
    ctx->d_count = reinterpret_cast<int *>(base);
    f.tiles = reinterpret_cast<const double *>(base + h.off_tiles);
    f.tile_stride = h.tile_stride; f.n_elems = h.n_elems; f.n_modes = h.n_modes;
    for (int k = 0; k < h.n_modes; ++k) { f.n_tor[k] = h.n_tor[k]; f.omega[k] = h.omega[k]; }
    f.grid.Rmin = h.Rmin; f.grid.Rmax = h.Rmax; f.grid.Zmin = h.Zmin; f.grid.Zmax = h.Zmax;
    f.grid.inv_hx = h.inv_hx; f.grid.inv_hz = h.inv_hz; f.grid.gx = h.g; f.grid.gz = h.g;
    f.grid.bstart = reinterpret_cast<const int *>(base + h.off_bstart);
    f.grid.bcand = reinterpret_cast<const int *>(base + h.off_bcand);
    f.grid.edges = reinterpret_cast<const double *>(base + h.off_edges);
    f.fast.Rmin = h.Rmin; f.fast.Zmin = h.Zmin; f.fast.inv_hx = h.finv_hx; f.fast.inv_hz = h.finv_hz;
    f.fast.gx = h.gf; f.fast.gz = h.gf;
    f.fast.first = reinterpret_cast<const FastRec *>(base + h.off_ffirst);
    f.fast.ovf = reinterpret_cast<const FastRec *>(base + h.off_fovf);
    ctx->have_fields = true;
    ctx->have_markers = false;   // cached elements refer to the old mesh
}

static int fast_grid_dim(int n_elems) {
    int g = (int)ceil(sqrt(2.0 * (double)n_elems));
    return g < 1 ? 1 : g;
}

static int grid_dim(int n_elems) {
    int g = (int)ceil(sqrt(0.5 * (double)n_elems));
    return g < 1 ? 1 : g;
}

extern "C" int m3dk_fields_workspace_bytes(int n_nodes, int n_elems, int n_modes, size_t *bytes) {
    if (!bytes || n_nodes < 3 || n_elems < 1 || n_modes < 0 || n_modes > M3DK_MAX_MODES) return M3DK_EINVAL;
    const int g = grid_dim(n_elems);
    size_t b = 256;
    b += up256((size_t)n_elems * tile_stride_doubles(n_modes) * sizeof(double));
    b += up256((size_t)n_elems * kEdgeRec * sizeof(double));
    b += up256(((size_t)g * g + 1) * sizeof(int));
    b += up256((size_t)kCandPerElem * n_elems * sizeof(int) + 1024);
    const int gf = fast_grid_dim(n_elems);
    b += up256((size_t)gf * gf * sizeof(FastRec));
    b += up256((size_t)gf * gf * sizeof(FastRec) + 1024);
    *bytes = b;
    return M3DK_OK;
}

extern "C" int m3dk_fields_create(m3dk_ctx *ctx, int n_nodes, const double *node_RZ, int n_elems, const int *tri,
                                  const double *eq_coef, int n_modes, const int *n_tor, const double *omega,
                                  const double *pert_coef, void *dev_workspace, size_t workspace_bytes) {
    if (!ctx) return M3DK_EINVAL;
    size_t need = 0;
    if (m3dk_fields_workspace_bytes(n_nodes, n_elems, n_modes, &need) != M3DK_OK || !node_RZ || !tri || !eq_coef ||
        (n_modes > 0 && (!n_tor || !omega || !pert_coef)))
        return fail(ctx, M3DK_EINVAL, "m3dk_fields_create: bad sizes or NULL table pointer");
    if (!dev_workspace || workspace_bytes < need || ((uintptr_t)dev_workspace & 255))
        return fail(ctx, M3DK_EWORKSPACE, "m3dk_fields_create: workspace NULL, misaligned or smaller than m3dk_fields_workspace_bytes");
    CU(cudaSetDevice(ctx->device), "cudaSetDevice");
    ctx->have_fields = false;

    const int stride = tile_stride_doubles(n_modes);
    std::vector<double> tiles((size_t)n_elems * stride, 0.0), edges((size_t)n_elems * kEdgeRec, 0.0);
    double Rmin = 1e300, Rmax = -1e300, Zmin = 1e300, Zmax = -1e300;
    for (int i = 0; i < n_nodes; ++i) {
        const double r = node_RZ[2 * i], z = node_RZ[2 * i + 1];
        if (!(r == r) || !(z == z)) return fail(ctx, M3DK_EINVAL, "m3dk_fields_create: NaN node coordinate");
        Rmin = std::min(Rmin, r); Rmax = std::max(Rmax, r); Zmin = std::min(Zmin, z); Zmax = std::max(Zmax, z);
    }
    if (!(Rmin > 0.0)) return fail(ctx, M3DK_EINVAL, "m3dk_fields_create: nodes must have R > 0");

    // per-element header, edge records, interleaved coefficient pairs
    for (int e = 0; e < n_elems; ++e) {
        double pr[3], pz[3];
        for (int k = 0; k < 3; ++k) {
            const int nd = tri[3 * e + k];
            if (nd < 0 || nd >= n_nodes) return fail(ctx, M3DK_EINVAL, "m3dk_fields_create: node index out of range");
            pr[k] = node_RZ[2 * nd]; pz[k] = node_RZ[2 * nd + 1];
        }
        const double area2 = (pr[1] - pr[0]) * (pz[2] - pz[0]) - (pz[1] - pz[0]) * (pr[2] - pr[0]);
        if (!(area2 > 0.0)) return fail(ctx, M3DK_EINVAL, "m3dk_fields_create: triangle is degenerate or not counter-clockwise");
        double L = 0.0;
        double *er = &edges[(size_t)e * kEdgeRec];
        for (int k = 0; k < 3; ++k) {
            const int kb = (k + 1) % 3;
            const double dx = pr[kb] - pr[k], dz = pz[kb] - pz[k];
            er[4 * k + 0] = pr[k]; er[4 * k + 1] = pz[k]; er[4 * k + 2] = dx; er[4 * k + 3] = dz;
            L = std::max(L, sqrt(dx * dx + dz * dz));
        }
        er[12] = 1e-9 * L * L;  // strict-interior tolerance: far above the rounding of an edge function, far below its size
        double *t = &tiles[(size_t)e * stride];
        t[0] = (pr[0] + pr[1] + pr[2]) / 3.0;   // centroid and scale exactly as reading G10 defines them
        t[1] = (pz[0] + pz[1] + pz[2]) / 3.0;
        t[2] = 1.0 / L;
        const double *ce = eq_coef + (size_t)e * M3DK_N_EQ * M3DK_NCOEF;
        double *pq = t + kTileHeader;
        for (int k = 0; k < M3DK_NCOEF; ++k)
            for (int q = 0; q < 4; ++q) pq[4 * k + q] = ce[q * M3DK_NCOEF + k];
        for (int md = 0; md < n_modes; ++md) {
            // caller's order: [7 amplitudes][re, im][21], amplitudes E_R E_phi E_Z B_R B_phi B_Z B_par; tile order:
            // quad 0 (E_R, E_phi), quad 1 (E_Z, B_R), quad 2 (B_par, B_Z), quad 3 (B_phi, zero padding)
            static const int kSlotOf[M3DK_N_PERT] = {0, 2, 4, 6, 12, 10, 8};   // first of the amplitude's two slots
            const double *cp = pert_coef + ((size_t)md * n_elems + e) * (M3DK_N_PERT * 2 * M3DK_NCOEF);
            double *pm = t + kTileHeader + kTileEq + (size_t)kTileMode * md;
            for (int a = 0; a < M3DK_N_PERT; ++a)
                for (int part = 0; part < 2; ++part) {
                    const int pl = kSlotOf[a] + part;
                    for (int k = 0; k < M3DK_NCOEF; ++k)
                        pm[(pl / 4) * kQuad + 4 * k + (pl % 4)] = cp[(2 * a + part) * M3DK_NCOEF + k];
                }
        }
    }

    // bucket grid: every element whose triangle touches the (slightly inflated) bucket, best bbox overlap first
    const int g = grid_dim(n_elems);
    const double hx = (Rmax - Rmin) / g, hz = (Zmax - Zmin) / g;
    const double tolx = 1e-7 * hx, tolz = 1e-7 * hz;
    struct Cand { int b, e; double ov; };
    std::vector<Cand> cands;
    cands.reserve((size_t)n_elems * 10);
    for (int e = 0; e < n_elems; ++e) {
        const double *er = &edges[(size_t)e * kEdgeRec];
        double r0 = std::min({er[0], er[4], er[8]}), r1 = std::max({er[0], er[4], er[8]});
        double z0 = std::min({er[1], er[5], er[9]}), z1 = std::max({er[1], er[5], er[9]});
        int ix0 = std::max(0, (int)floor((r0 - tolx - Rmin) / hx)), ix1 = std::min(g - 1, (int)floor((r1 + tolx - Rmin) / hx));
        int iz0 = std::max(0, (int)floor((z0 - tolz - Zmin) / hz)), iz1 = std::min(g - 1, (int)floor((z1 + tolz - Zmin) / hz));
        for (int iz = iz0; iz <= iz1; ++iz)
            for (int ix = ix0; ix <= ix1; ++ix) {
                const double bx0 = Rmin + ix * hx - tolx, bx1 = Rmin + (ix + 1) * hx + tolx;
                const double bz0 = Zmin + iz * hz - tolz, bz1 = Zmin + (iz + 1) * hz + tolz;
                // separating-axis test against the three edge normals (the bbox axes are covered by the loop bounds)
                bool sep = false;
                for (int k = 0; k < 3 && !sep; ++k) {
                    const double ra = er[4 * k], za = er[4 * k + 1], dx = er[4 * k + 2], dz = er[4 * k + 3];
                    const double cx = dz > 0 ? bx0 : bx1;   // corner that maximises dx (Z - za) - dz (R - ra)
                    const double cz = dx > 0 ? bz1 : bz0;
                    if (dx * (cz - za) - dz * (cx - ra) < 0.0) sep = true;
                }
                if (sep) continue;
                const double ox = std::min(r1, bx1) - std::max(r0, bx0), oz = std::min(z1, bz1) - std::max(z0, bz0);
                cands.push_back({iz * g + ix, e, std::max(ox, 0.0) * std::max(oz, 0.0)});
            }
    }
    if (cands.size() > (size_t)kCandPerElem * n_elems)
        return fail(ctx, M3DK_EWORKSPACE, "m3dk_fields_create: search grid needs more candidate slots than the workspace bound");
    std::sort(cands.begin(), cands.end(), [](const Cand &a, const Cand &b) {
        if (a.b != b.b) return a.b < b.b;
        if (a.ov != b.ov) return a.ov > b.ov;
        return a.e < b.e;
    });
    std::vector<int> bstart((size_t)g * g + 1, 0), bcand(cands.size() + 1, 0);
    for (size_t k = 0; k < cands.size(); ++k) { bstart[cands[k].b + 1]++; bcand[k] = cands[k].e; }
    for (int b = 0; b < g * g; ++b) bstart[b + 1] += bstart[b];

    // fast search grid (fp32 records in bucket-local coordinates; see m3dk_internal.h).  Candidates of a bucket: the
    // triangles that touch it, largest overlap area first, at most 4 (the device loop's bound); a bucket with a
    // candidate too large for the fp32 error bound, or with none, sends its points to the exact search (id = -1).
    const int gf = fast_grid_dim(n_elems);
    const double fhx = (Rmax - Rmin) / gf, fhz = (Zmax - Zmin) / gf;
    const double finv_hx = 1.0 / fhx, finv_hz = 1.0 / fhz;
    struct FCand { int b, e; double area; float c[6]; bool big; };
    std::vector<FCand> fc;
    fc.reserve((size_t)n_elems * 10);
    for (int e = 0; e < n_elems; ++e) {
        const double *er = &edges[(size_t)e * kEdgeRec];
        double gx_[3], gz_[3];
        for (int k = 0; k < 3; ++k) { gx_[k] = (er[4 * k] - Rmin) * finv_hx; gz_[k] = (er[4 * k + 1] - Zmin) * finv_hz; }
        const double x0 = std::min({gx_[0], gx_[1], gx_[2]}), x1 = std::max({gx_[0], gx_[1], gx_[2]});
        const double z0 = std::min({gz_[0], gz_[1], gz_[2]}), z1 = std::max({gz_[0], gz_[1], gz_[2]});
        const double ftol = 1e-6;
        const int ix0 = std::max(0, (int)floor(x0 - ftol)), ix1 = std::min(gf - 1, (int)floor(x1 + ftol));
        const int iz0 = std::max(0, (int)floor(z0 - ftol)), iz1 = std::min(gf - 1, (int)floor(z1 + ftol));
        for (int iz = iz0; iz <= iz1; ++iz)
            for (int ix = ix0; ix <= ix1; ++ix) {
                double lx[3], lz[3];
                bool big = false;
                for (int k = 0; k < 3; ++k) {
                    lx[k] = gx_[k] - ix; lz[k] = gz_[k] - iz;
                    if (lx[k] < -(kFastCmax - 1.0) || lx[k] > kFastCmax || lz[k] < -(kFastCmax - 1.0) || lz[k] > kFastCmax) big = true;
                }
                // separating-axis test of the triangle against the inflated unit square
                bool sep = false;
                for (int k = 0; k < 3 && !sep; ++k) {
                    const int kb = (k + 1) % 3;
                    const double dx = lx[kb] - lx[k], dz = lz[kb] - lz[k];
                    const double cx = dz > 0 ? -ftol : 1.0 + ftol, cz = dx > 0 ? 1.0 + ftol : -ftol;
                    if (dx * (cz - lz[k]) - dz * (cx - lx[k]) < 0.0) sep = true;
                }
                if (sep) continue;
                // overlap area: the triangle clipped to the unit square (Sutherland-Hodgman), shoelace formula
                double px[16], pz[16], qx[16], qz[16];
                int np = 3;
                for (int k = 0; k < 3; ++k) { px[k] = lx[k]; pz[k] = lz[k]; }
                for (int side = 0; side < 4 && np > 0; ++side) {
                    int nq = 0;
                    for (int k = 0; k < np; ++k) {
                        const int kb = (k + 1) % np;
                        const double ax = px[k], az = pz[k], bx = px[kb], bz = pz[kb];
                        const double da = side == 0 ? ax : side == 1 ? 1.0 - ax : side == 2 ? az : 1.0 - az;
                        const double db = side == 0 ? bx : side == 1 ? 1.0 - bx : side == 2 ? bz : 1.0 - bz;
                        if (da >= 0.0) { qx[nq] = ax; qz[nq] = az; ++nq; }
                        if ((da >= 0.0) != (db >= 0.0)) {
                            const double tt = da / (da - db);
                            qx[nq] = ax + tt * (bx - ax); qz[nq] = az + tt * (bz - az); ++nq;
                        }
                    }
                    np = nq;
                    for (int k = 0; k < np; ++k) { px[k] = qx[k]; pz[k] = qz[k]; }
                }
                double area = 0.0;
                for (int k = 0; k < np; ++k) { const int kb = (k + 1) % np; area += px[k] * pz[kb] - px[kb] * pz[k]; }
                FCand cnd{iz * gf + ix, e, 0.5 * fabs(area), {(float)lx[0], (float)lz[0], (float)lx[1], (float)lz[1], (float)lx[2], (float)lz[2]}, big};
                fc.push_back(cnd);
            }
    }
    std::sort(fc.begin(), fc.end(), [](const FCand &a, const FCand &b) {
        if (a.b != b.b) return a.b < b.b;
        if (a.area != b.area) return a.area > b.area;
        return a.e < b.e;
    });
    const size_t ovf_cap = (size_t)gf * gf;
    FastRec empty_rec;
    memset(&empty_rec, 0, sizeof(empty_rec));
    empty_rec.ida = empty_rec.idb = empty_rec.next = -1;
    std::vector<FastRec> ffirst((size_t)gf * gf, empty_rec), fovf;
    fovf.reserve(std::min(ovf_cap, fc.size() / 2 + 1));
    for (size_t k = 0; k < fc.size();) {
        size_t k1 = k;
        bool big = false;
        while (k1 < fc.size() && fc[k1].b == fc[k].b) { big = big || fc[k1].big; ++k1; }
        if (!big) {
            // two candidates per record, at most 4 per bucket (the device loop's bound): first record + one overflow record
            FastRec *cur = &ffirst[fc[k].b];
            for (size_t j = k; j < k1 && j < k + 4; ++j) {
                const FCand &cn = fc[j];
                const size_t pos = j - k;
                if (pos == 2) {
                    if (fovf.size() >= ovf_cap) break;
                    cur->next = (int)fovf.size();
                    fovf.push_back(empty_rec);     // reserve() above keeps `cur` valid: no reallocation below capacity
                    cur = &fovf.back();
                }
                if (pos % 2 == 0) { for (int q = 0; q < 6; ++q) cur->a[q] = cn.c[q]; cur->ida = cn.e; }
                else { for (int q = 0; q < 6; ++q) cur->b[q] = cn.c[q]; cur->idb = cn.e; }
            }
        }
        k = k1;
    }
    if (fovf.empty()) fovf.push_back(empty_rec);

    // carve and upload
    char *p = static_cast<char *>(dev_workspace);
    ctx->d_count = reinterpret_cast<int *>(p); p += 256;
    double *d_tiles = reinterpret_cast<double *>(p); p += up256(tiles.size() * sizeof(double));
    double *d_edges = reinterpret_cast<double *>(p); p += up256(edges.size() * sizeof(double));
    int *d_bstart = reinterpret_cast<int *>(p); p += up256(bstart.size() * sizeof(int));
    int *d_bcand = reinterpret_cast<int *>(p); p += up256((size_t)kCandPerElem * n_elems * sizeof(int) + 1024);
    FastRec *d_ffirst = reinterpret_cast<FastRec *>(p); p += up256(ffirst.size() * sizeof(FastRec));
    FastRec *d_fovf = reinterpret_cast<FastRec *>(p);
    FieldsHeader hdr;
    memset(&hdr, 0, sizeof(hdr));
    hdr.magic = kFieldsMagic;
    char *const base = static_cast<char *>(dev_workspace);
    hdr.off_tiles = (unsigned long long)(reinterpret_cast<char *>(d_tiles) - base);
    hdr.off_edges = (unsigned long long)(reinterpret_cast<char *>(d_edges) - base);
    hdr.off_bstart = (unsigned long long)(reinterpret_cast<char *>(d_bstart) - base);
    hdr.off_bcand = (unsigned long long)(reinterpret_cast<char *>(d_bcand) - base);
    hdr.off_ffirst = (unsigned long long)(reinterpret_cast<char *>(d_ffirst) - base);
    hdr.off_fovf = (unsigned long long)(reinterpret_cast<char *>(d_fovf) - base);
    hdr.total_bytes = need;
    hdr.Rmin = Rmin; hdr.Rmax = Rmax; hdr.Zmin = Zmin; hdr.Zmax = Zmax;
    hdr.inv_hx = 1.0 / hx; hdr.inv_hz = 1.0 / hz; hdr.finv_hx = finv_hx; hdr.finv_hz = finv_hz;
    for (int k = 0; k < n_modes; ++k) { hdr.n_tor[k] = n_tor[k]; hdr.omega[k] = omega[k]; }
    hdr.n_elems = n_elems; hdr.n_modes = n_modes; hdr.tile_stride = stride; hdr.g = g; hdr.gf = gf;
    CU(cudaMemsetAsync(ctx->d_count, 0, 256, ctx->stream), "memset control block");
    CU(cudaMemcpyAsync(base + 32, &hdr, sizeof(hdr), cudaMemcpyHostToDevice, ctx->stream), "upload header");
    CU(cudaMemcpyAsync(d_tiles, tiles.data(), tiles.size() * sizeof(double), cudaMemcpyHostToDevice, ctx->stream), "upload tiles");
    CU(cudaMemcpyAsync(d_edges, edges.data(), edges.size() * sizeof(double), cudaMemcpyHostToDevice, ctx->stream), "upload edge records");
    CU(cudaMemcpyAsync(d_bstart, bstart.data(), bstart.size() * sizeof(int), cudaMemcpyHostToDevice, ctx->stream), "upload grid");
    CU(cudaMemcpyAsync(d_bcand, bcand.data(), bcand.size() * sizeof(int), cudaMemcpyHostToDevice, ctx->stream), "upload grid candidates");
    CU(cudaMemcpyAsync(d_ffirst, ffirst.data(), ffirst.size() * sizeof(FastRec), cudaMemcpyHostToDevice, ctx->stream), "upload fast grid");
    CU(cudaMemcpyAsync(d_fovf, fovf.data(), fovf.size() * sizeof(FastRec), cudaMemcpyHostToDevice, ctx->stream), "upload fast grid overflow");
    CU(cudaStreamSynchronize(ctx->stream), "fields upload");
    bind_fields(ctx, base, hdr);
    return M3DK_OK;
}

extern "C" int m3dk_fields_attach(m3dk_ctx *ctx, void *dev_workspace, size_t workspace_bytes) {
    if (!ctx) return M3DK_EINVAL;
    if (!dev_workspace || workspace_bytes < 256 || ((uintptr_t)dev_workspace & 255))
        return fail(ctx, M3DK_EWORKSPACE, "m3dk_fields_attach: workspace NULL, misaligned or shorter than its control block");
    CU(cudaSetDevice(ctx->device), "cudaSetDevice");
    FieldsHeader hdr;
    char *const base = static_cast<char *>(dev_workspace);
    CU(cudaMemcpyAsync(&hdr, base + 32, sizeof(hdr), cudaMemcpyDeviceToHost, ctx->stream), "read header");
    CU(cudaStreamSynchronize(ctx->stream), "read header");
    if (hdr.magic != kFieldsMagic || hdr.total_bytes > workspace_bytes || hdr.n_elems < 1 || hdr.n_modes < 0 ||
        hdr.n_modes > M3DK_MAX_MODES || hdr.tile_stride != tile_stride_doubles(hdr.n_modes))
        return fail(ctx, M3DK_EINVAL, "m3dk_fields_attach: the workspace does not hold a fields image of this library version");
    ctx->have_fields = false;
    bind_fields(ctx, base, hdr);
    return M3DK_OK;
}

// ---- markers -------------------------------------------------------------------------------------------------------
extern "C" int m3dk_particles_init(m3dk_ctx *ctx, long n, double *x, double *y, double *z, double *vx, double *vy,
                                   double *vz, double *mu, double *w, int *elem, int *id, double charge, double mass,
                                   const m3dk_f0_params *f0) {
    if (!ctx) return M3DK_EINVAL;
    if (!ctx->have_fields) return fail(ctx, M3DK_ESTATE, "m3dk_particles_init: call m3dk_fields_create first");
    if (n < 0 || n > 0x7fffffffL || (n > 0 && (!x || !y || !z || !vx || !vy || !vz || !mu || !w || !elem || !id)) || !f0)
        return fail(ctx, M3DK_EINVAL, "m3dk_particles_init: bad n or NULL array");
    if (!(charge != 0.0) || !(mass > 0.0)) return fail(ctx, M3DK_EINVAL, "m3dk_particles_init: charge must be non-zero and mass positive");
    if (f0->kind < 0 || f0->kind > 2 || (f0->kind == M3DK_F0_MAXWELLIAN && !(f0->T > 0.0)) ||
        (f0->kind != M3DK_F0_MAXWELLIAN && !(f0->v_c > 0.0)) || (f0->kind == M3DK_F0_BEAM_PITCH && !(f0->dLambda > 0.0)))
        return fail(ctx, M3DK_EINVAL, "m3dk_particles_init: bad f0 parameters");
    CU(cudaSetDevice(ctx->device), "cudaSetDevice");
    ctx->n = n;
    ctx->user = MarkerArrays{x, y, z, vx, vy, vz, mu, w, elem, id};
    ctx->q = charge; ctx->m = mass; ctx->f0 = *f0;
    ctx->steps_done = 0; ctx->n_sorts = 0;
    ctx->t_base = ctx->t0; ctx->steps_at_dt = 0;
    ctx->steps_since_sort = ctx->sort_interval;   // the first push sorts first when sorting is on
    ctx->have_markers = true;
    // the sort workspace was carved for the previous n / mesh: carve it again, or drop it if it has become too small
    ctx->have_sortws = false;
    if (ctx->sortws_base && sort_workspace_bytes(n, ctx->f.n_elems) <= ctx->sortws_bytes) {
        carve_sort_workspace(ctx->sortws_base, n, ctx->f.n_elems, &ctx->sb);
        ctx->sb.bytes = ctx->sortws_bytes;
        ctx->have_sortws = true;
    }
    ctx->have_flrws = false;
    ctx->flr_with_avg = false;
    if (ctx->flrws_base && flr_workspace_bytes(n, ctx->f.n_elems) <= ctx->flrws_bytes) {
        ctx->flr_with_avg = flr_workspace_bytes(n, ctx->f.n_elems, true) <= ctx->flrws_bytes;
        carve_flr_workspace(ctx->flrws_base, n, ctx->f.n_elems, &ctx->fb, ctx->flr_with_avg);
        ctx->have_flrws = true;
    }
    CU(launch_locate(ctx, ctx->user, n, true), "locate kernel");
    return M3DK_OK;
}

extern "C" int m3dk_set_options(m3dk_ctx *ctx, int sort_interval, int mode, double t0) {
    if (!ctx) return M3DK_EINVAL;
    if (sort_interval < 0) return fail(ctx, M3DK_EINVAL, "m3dk_set_options: sort_interval < 0");
    if (mode < 0 || mode > 3)
        return fail(ctx, M3DK_EINVAL, "m3dk_set_options: mode must be 0 (linear delta-f), 1 (non-linear trajectories), 2 (linear + FLR) or 3 (non-linear + FLR)");
    ctx->sort_interval = sort_interval; ctx->mode = mode; ctx->t0 = t0;
    ctx->t_base = t0; ctx->steps_at_dt = 0;
    ctx->steps_done = 0;
    ctx->steps_since_sort = sort_interval;
    return M3DK_OK;
}

extern "C" int m3dk_set_push_variant(m3dk_ctx *ctx, int variant) {
    if (!ctx) return M3DK_EINVAL;
    if (variant < 0 || variant > 1) return fail(ctx, M3DK_EINVAL, "m3dk_set_push_variant: variant must be 0 or 1");
    ctx->push_variant = variant;
    return M3DK_OK;
}

extern "C" int m3dk_sort_workspace_bytes(long n_markers, int n_elems, size_t *bytes) {
    if (!bytes || n_markers < 0 || n_elems < 1) return M3DK_EINVAL;
    *bytes = sort_workspace_bytes(n_markers, n_elems);
    return M3DK_OK;
}

static int bind_sort_ws(m3dk_ctx *ctx, void *ws, size_t bytes, const char *who) {
    if (!ctx->have_markers) return fail(ctx, M3DK_ESTATE, std::string(who) + ": call m3dk_particles_init first");
    if (!ws || ((uintptr_t)ws & 255) || bytes < sort_workspace_bytes(ctx->n, ctx->f.n_elems))
        return fail(ctx, M3DK_EWORKSPACE, std::string(who) + ": workspace NULL, misaligned or smaller than m3dk_sort_workspace_bytes");
    carve_sort_workspace(ws, ctx->n, ctx->f.n_elems, &ctx->sb);
    ctx->sb.bytes = bytes;
    ctx->sortws_base = ws; ctx->sortws_bytes = bytes;
    ctx->have_sortws = true;
    return M3DK_OK;
}

extern "C" int m3dk_set_sort_workspace(m3dk_ctx *ctx, void *dev_workspace, size_t bytes) {
    if (!ctx) return M3DK_EINVAL;
    return bind_sort_ws(ctx, dev_workspace, bytes, "m3dk_set_sort_workspace");
}

extern "C" int m3dk_flr_workspace_bytes(long n_markers, int n_elems, size_t *bytes) {
    if (!bytes || n_markers < 0 || n_elems < 1) return M3DK_EINVAL;
    *bytes = flr_workspace_bytes(n_markers, n_elems);
    return M3DK_OK;
}

extern "C" int m3dk_flr_workspace_bytes_nl(long n_markers, int n_elems, size_t *bytes) {
    if (!bytes || n_markers < 0 || n_elems < 1) return M3DK_EINVAL;
    *bytes = flr_workspace_bytes(n_markers, n_elems, true);
    return M3DK_OK;
}

extern "C" int m3dk_set_flr_workspace(m3dk_ctx *ctx, void *dev_workspace, size_t bytes) {
    if (!ctx) return M3DK_EINVAL;
    if (!ctx->have_markers) return fail(ctx, M3DK_ESTATE, "m3dk_set_flr_workspace: call m3dk_particles_init first");
    if (!dev_workspace || ((uintptr_t)dev_workspace & 255) || bytes < flr_workspace_bytes(ctx->n, ctx->f.n_elems))
        return fail(ctx, M3DK_EWORKSPACE, "m3dk_set_flr_workspace: workspace NULL, misaligned or smaller than m3dk_flr_workspace_bytes");
    ctx->flr_with_avg = bytes >= flr_workspace_bytes(ctx->n, ctx->f.n_elems, true);
    carve_flr_workspace(dev_workspace, ctx->n, ctx->f.n_elems, &ctx->fb, ctx->flr_with_avg);
    ctx->flrws_base = dev_workspace; ctx->flrws_bytes = bytes;
    ctx->have_flrws = true;
    return M3DK_OK;
}

// ---- sort and push ---------------------------------------------------------------------------------------------------
// sort_interval = 0: the caller's SoA arrays are pushed in place, in whatever order they are (one marker per thread,
// every thread gathers its own element's coefficients).
// sort_interval = k >= 1: ordered pipeline.  At the start of the call the markers are packed into 64-byte records in
// element order (a sort); EVERY step runs the element-ordered kernel and is followed by a re-ordering (histogram fused
// into the push, scan, work-item cut, order list); at the end of the call the records are unpacked into the caller's
// arrays (permuted; id[] says who is where).  k > 1 is accepted and served as k = 1 (results are bit-identical).
extern "C" int m3dk_sort(m3dk_ctx *ctx, void *dev_workspace, size_t bytes) {
    if (!ctx) return M3DK_EINVAL;
    if (!ctx->have_markers) return fail(ctx, M3DK_ESTATE, "m3dk_sort: call m3dk_particles_init first");
    if (dev_workspace) {
        int rc = bind_sort_ws(ctx, dev_workspace, bytes, "m3dk_sort");
        if (rc != M3DK_OK) return rc;
    } else if (!ctx->have_sortws) {
        return fail(ctx, M3DK_ESTATE, "m3dk_sort: no workspace (pass one or call m3dk_set_sort_workspace)");
    }
    CU(cudaSetDevice(ctx->device), "cudaSetDevice");
    if (ctx->n == 0) return M3DK_OK;
    {
        EvScope ev(ctx, &ctx->ev_sort);
        CU(launch_pack_sorted(ctx, ctx->n), "sort kernels (pack)");
        CU(launch_unpack(ctx, ctx->n), "sort kernels (unpack)");
    }
    ctx->n_sorts++;
    ctx->steps_since_sort = 0;
    return M3DK_OK;
}

// time of the next step's x_l: t_base + (steps taken at the current dt) * dt; a changed dt starts a new run of equal steps
static double step_time(m3dk_ctx *ctx, double dt) {
    if (dt != ctx->last_dt) {
        ctx->t_base += (double)ctx->steps_at_dt * ctx->last_dt;
        ctx->steps_at_dt = 0;
        ctx->last_dt = dt;
    }
    return ctx->t_base + (double)ctx->steps_at_dt * dt;
}

// nsteps steps of the markers currently bound to the context (ctx->n, ctx->user, ctx->sb)
static int run_steps(m3dk_ctx *ctx, int nsteps, double dt) {
    if (ctx->sort_interval == 0 || ctx->n == 0 || nsteps == 0) {
        for (int l = 0; l < nsteps; ++l) {
            const double t = step_time(ctx, dt);            // t_l of this step's x_l
            EvScope ev(ctx, &ctx->ev_push);
            CU(launch_push_soa(ctx, ctx->n, dt, t), "push kernel");
            ctx->steps_done++; ctx->steps_at_dt++;
        }
        return M3DK_OK;
    }
    {
        EvScope ev(ctx, &ctx->ev_sort);
        CU(launch_pack_sorted(ctx, ctx->n), "sort kernels (pack)");
    }
    ctx->n_sorts++;
    ctx->steps_since_sort = 0;
    // Every step runs the element-ordered kernel and is followed by a re-ordering, whatever k >= 1 asks for: the ordering
    // is fused into the push (histogram) and costs a tenth of a step, while a step on a stale order costs seven times one
    // on a fresh order (markers cross 2-18 elements per step; measured in BASELINE.md section 4).
    for (int l = 0; l < nsteps; ++l) {
        const double t = step_time(ctx, dt);
        const bool reorder_after = l + 1 < nsteps;
        {
            EvScope ev(ctx, &ctx->ev_push);
            if (flr_nl_stream(ctx)) {
                // mode 3: ring points of every marker, ordered by their element, fields at the points; the push proper then
                // reads the four sets of field components of each marker
                CU(launch_flr_emit_nl(ctx, ctx->n, dt, t), "ring emit kernel");
                CU(launch_flr_ring_keys(ctx, ctx->n), "ring key kernel");
                CU(launch_flr_ring_stage(ctx, ctx->n), "ring ordering kernels");
                CU(launch_flr_ring_eval(ctx, ctx->n, dt, t, true), "ring evaluation kernel");
            }
            CU(launch_push_rec(ctx, ctx->n, dt, t, reorder_after), "push kernel");
            if (ctx->mode == 2 && ctx->have_flrws && ctx->f.n_modes > 0) {
                // the push has emitted the ring stream: order it by the ring points' elements, evaluate, sum back into w
                CU(launch_flr_ring_keys(ctx, ctx->n), "ring key kernel");
                CU(launch_flr_ring_stage(ctx, ctx->n), "ring ordering kernels");
                CU(launch_flr_ring_eval(ctx, ctx->n, dt, t), "ring evaluation kernel");
                CU(launch_flr_reduce(ctx, ctx->n, dt), "ring reduction kernel");
            }
        }
        ctx->steps_done++; ctx->steps_at_dt++;
        ctx->steps_since_sort = 1;
        if (reorder_after) {
            EvScope ev(ctx, &ctx->ev_sort);
            CU(launch_reorder(ctx, ctx->n), "sort kernels (reorder)");
            ctx->n_sorts++;
            ctx->steps_since_sort = 0;
        }
    }
    {
        EvScope ev(ctx, &ctx->ev_sort);
        CU(launch_unpack(ctx, ctx->n), "sort kernels (unpack)");
    }
    return M3DK_OK;
}

extern "C" int m3dk_push(m3dk_ctx *ctx, int nsteps, double dt) {
    if (!ctx) return M3DK_EINVAL;
    if (!ctx->have_fields || !ctx->have_markers) return fail(ctx, M3DK_ESTATE, "m3dk_push: fields and markers must be set first");
    if (nsteps < 0 || !(dt == dt)) return fail(ctx, M3DK_EINVAL, "m3dk_push: nsteps < 0 or dt is NaN");
    if (ctx->sort_interval > 0 && !ctx->have_sortws)
        return fail(ctx, M3DK_ESTATE, "m3dk_push: sort_interval > 0 needs m3dk_set_sort_workspace");
    CU(cudaSetDevice(ctx->device), "cudaSetDevice");
    return run_steps(ctx, nsteps, dt);
}

extern "C" int m3dk_stats(m3dk_ctx *ctx, m3dk_stats_t *out) {
    if (!ctx || !out) return M3DK_EINVAL;
    memset(out, 0, sizeof(*out));
    CU(cudaSetDevice(ctx->device), "cudaSetDevice");
    int lost = 0;
    if (ctx->have_markers) {
        CU(launch_count_lost(ctx, ctx->user, ctx->n, ctx->d_count), "count kernel");
        CU(cudaMemcpyAsync(&lost, ctx->d_count, sizeof(int), cudaMemcpyDeviceToHost, ctx->stream), "read counter");
    }
    CU(cudaStreamSynchronize(ctx->stream), "stream synchronize (an earlier kernel may have failed)");
    out->n_markers = ctx->have_markers ? ctx->n : 0;
    out->n_lost = lost;
    out->steps_done = ctx->steps_done;
    out->n_sorts = ctx->n_sorts;
    out->t = ctx->t_base + (double)ctx->steps_at_dt * ctx->last_dt;
    return M3DK_OK;
}

extern "C" int m3dk_particles_upload(m3dk_ctx *ctx, const double *hx, const double *hy, const double *hz,
                                     const double *hvx, const double *hvy, const double *hvz, const double *hmu,
                                     const double *hw) {
    if (!ctx) return M3DK_EINVAL;
    if (!ctx->have_markers) return fail(ctx, M3DK_ESTATE, "m3dk_particles_upload: call m3dk_particles_init first");
    if (!hx || !hy || !hz || !hvx || !hvy || !hvz || !hmu || !hw) return fail(ctx, M3DK_EINVAL, "m3dk_particles_upload: NULL buffer");
    CU(cudaSetDevice(ctx->device), "cudaSetDevice");
    const MarkerArrays &d = ctx->user;
    const size_t nd = (size_t)ctx->n * sizeof(double);
    const double *const hs[8] = {hx, hy, hz, hvx, hvy, hvz, hmu, hw};
    double *const dd[8] = {d.x, d.y, d.z, d.vx, d.vy, d.vz, d.mu, d.w};
    for (int k = 0; k < 8; ++k) CU(cudaMemcpyAsync(dd[k], hs[k], nd, cudaMemcpyHostToDevice, ctx->stream), "upload markers");
    ctx->steps_since_sort = ctx->sort_interval;
    CU(launch_locate(ctx, ctx->user, ctx->n, true), "locate kernel");
    return M3DK_OK;
}

extern "C" int m3dk_particles_download(m3dk_ctx *ctx, double *hx, double *hy, double *hz, double *hvx, double *hvy,
                                       double *hvz, double *hmu, double *hw, int *host_id, int *host_elem) {
    if (!ctx) return M3DK_EINVAL;
    if (!ctx->have_markers) return fail(ctx, M3DK_ESTATE, "m3dk_particles_download: call m3dk_particles_init first");
    if (!hx || !hy || !hz || !hvx || !hvy || !hvz || !hmu || !hw) return fail(ctx, M3DK_EINVAL, "m3dk_particles_download: NULL buffer");
    CU(cudaSetDevice(ctx->device), "cudaSetDevice");
    const MarkerArrays &d = ctx->user;
    const size_t nd = (size_t)ctx->n * sizeof(double), ni = (size_t)ctx->n * sizeof(int);
    double *const hs[8] = {hx, hy, hz, hvx, hvy, hvz, hmu, hw};
    const double *const dd[8] = {d.x, d.y, d.z, d.vx, d.vy, d.vz, d.mu, d.w};
    for (int k = 0; k < 8; ++k) CU(cudaMemcpyAsync(hs[k], dd[k], nd, cudaMemcpyDeviceToHost, ctx->stream), "download markers");
    if (host_id) CU(cudaMemcpyAsync(host_id, d.id, ni, cudaMemcpyDeviceToHost, ctx->stream), "download id");
    if (host_elem) CU(cudaMemcpyAsync(host_elem, d.elem, ni, cudaMemcpyDeviceToHost, ctx->stream), "download elem");
    CU(cudaStreamSynchronize(ctx->stream), "stream synchronize (an earlier kernel may have failed)");
    return M3DK_OK;
}

// Host-buffer push, pipelined by marker chunk (markers are independent): chunk c is uploaded on the upload
// stream while chunk c - 1 runs its nsteps steps on the context's stream and chunk c - 2 is downloaded on the download
// stream (the two copy directions run concurrently).  Every chunk goes through the same code as m3dk_push on its
// sub-range of the registered device arrays; the sort workspace is re-carved for the chunk size and used by one chunk at
// a time (the steps of all chunks are in stream order).
extern "C" int m3dk_push_host(m3dk_ctx *ctx, double *hx, double *hy, double *hz, double *hvx, double *hvy, double *hvz,
                              double *hmu, double *hw, int *host_id, int *host_elem, int nsteps, double dt, int n_chunks) {
    if (!ctx) return M3DK_EINVAL;
    if (!ctx->have_fields || !ctx->have_markers) return fail(ctx, M3DK_ESTATE, "m3dk_push_host: fields and markers must be set first");
    if (!hx || !hy || !hz || !hvx || !hvy || !hvz || !hmu || !hw) return fail(ctx, M3DK_EINVAL, "m3dk_push_host: NULL buffer");
    if (nsteps < 0 || !(dt == dt) || n_chunks < 0) return fail(ctx, M3DK_EINVAL, "m3dk_push_host: nsteps < 0, dt is NaN or n_chunks < 0");
    if (ctx->sort_interval > 0 && !ctx->have_sortws)
        return fail(ctx, M3DK_ESTATE, "m3dk_push_host: sort_interval > 0 needs m3dk_set_sort_workspace");
    CU(cudaSetDevice(ctx->device), "cudaSetDevice");
    const long n = ctx->n;
    if (n == 0) return M3DK_OK;
    if (n_chunks == 0) {
        // automatic: many chunks hide the transfers, few chunks keep the work items full and the fixed cost of a chunk-step
        // low.  What decides is the ratio of transfer time (64 B per marker and direction at about 50 GB/s) to compute time
        // (about 80 / 100 / 400 / 420 ps per marker-step in modes 0 .. 3 on a B200); measured at 2^24 markers, mode 0:
        // 20 steps (ratio 0.8) best with 8 chunks, 50 steps (0.3) with 4, 200 steps (0.08) with 3.
        static const double kStepCost[4] = {80e-12, 100e-12, 400e-12, 420e-12};
        const double ratio = nsteps > 0 ? (64.0 / 50e9) / ((double)nsteps * kStepCost[ctx->mode & 3]) : 1.0;
        n_chunks = n < (1L << 18) ? 1 : ratio >= 0.6 ? 8 : ratio >= 0.15 ? 4 : 3;
    }
    if ((long)n_chunks > n) n_chunks = (int)n;
    if (!ctx->s_up) {
        CU(cudaStreamCreateWithFlags(&ctx->s_up, cudaStreamNonBlocking), "create upload stream");
        CU(cudaStreamCreateWithFlags(&ctx->s_down, cudaStreamNonBlocking), "create download stream");
    }
    while (ctx->ev_chunk.size() < (size_t)2 * n_chunks + 1) {
        cudaEvent_t e;
        CU(cudaEventCreateWithFlags(&e, cudaEventDisableTiming), "create chunk event");
        ctx->ev_chunk.push_back(e);
    }
    // the copy streams start after everything already enqueued on the context's stream (the arrays may be in use)
    cudaEvent_t ev_start = ctx->ev_chunk[2 * n_chunks];
    CU(cudaEventRecord(ev_start, ctx->stream), "record start");
    CU(cudaStreamWaitEvent(ctx->s_up, ev_start, 0), "upload stream wait");
    CU(cudaStreamWaitEvent(ctx->s_down, ev_start, 0), "download stream wait");

    const MarkerArrays all = ctx->user;
    const long steps0 = ctx->steps_done, at0 = ctx->steps_at_dt;
    const double tb0 = ctx->t_base, ldt0 = ctx->last_dt;
    double *const hs[8] = {hx, hy, hz, hvx, hvy, hvz, hmu, hw};
    double *const dd[8] = {all.x, all.y, all.z, all.vx, all.vy, all.vz, all.mu, all.w};
    // Chunk boundaries: with four chunks or more the sizes ramp up and down again (weights 1, 2, .., 2, 1 capped at 4), so
    // that the first upload and the last download, which nothing overlaps, are short; fewer chunks are equal.
    std::vector<long> cut(n_chunks + 1, 0);
    {
        std::vector<long> wgt(n_chunks, 1);
        long tot = 0;
        for (int c = 0; c < n_chunks; ++c) {
            if (n_chunks >= 4) wgt[c] = std::min<long>(4, 1 + std::min(c, n_chunks - 1 - c));
            tot += wgt[c];
        }
        long acc = 0;
        for (int c = 0; c < n_chunks; ++c) {
            acc += wgt[c];
            cut[c + 1] = std::max(cut[c], std::min(n, (n * acc + tot - 1) / tot));
        }
        cut[n_chunks] = n;
    }
    long per = 0;                                   // the largest chunk: what a slot of the workspaces must hold
    for (int c = 0; c < n_chunks; ++c) per = std::max(per, cut[c + 1] - cut[c]);
    // Up to host_slots chunks are in flight at a time, each on its own compute stream with its own ordering workspace
    // (chunk-sized carvings of the caller's workspace): the launch gaps, the small ordering kernels and the tail of the
    // persistent push kernels of one chunk are filled by the other.
    const size_t sort_slot = ctx->have_sortws ? sort_workspace_bytes(per, ctx->f.n_elems) : 0;
    const size_t flr_slot = ctx->have_flrws ? flr_workspace_bytes(per, ctx->f.n_elems, ctx->flr_with_avg) : 0;
    int slots = std::min(n_chunks, ctx->host_slots);
    while (slots > 1 && ((ctx->have_sortws && slots * sort_slot > ctx->sortws_bytes) ||
                         (ctx->have_flrws && slots * flr_slot > ctx->flrws_bytes)))
        --slots;
    cudaStream_t const main_stream = ctx->stream;
    for (int k = 1; k < slots; ++k) {
        if (!ctx->s_c[k]) CU(cudaStreamCreateWithFlags(&ctx->s_c[k], cudaStreamNonBlocking), "create compute stream");
        CU(cudaStreamWaitEvent(ctx->s_c[k], ev_start, 0), "compute stream wait");
    }
    // whatever happens below, the context leaves this call bound to all markers, its own stream and the whole workspace
    struct Restore {
        m3dk_ctx *c; long n; MarkerArrays all; cudaStream_t st;
        ~Restore() {
            c->n = n; c->user = all; c->stream = st;
            if (c->have_sortws) { carve_sort_workspace(c->sortws_base, n, c->f.n_elems, &c->sb); c->sb.bytes = c->sortws_bytes; }
            if (c->have_flrws) carve_flr_workspace(c->flrws_base, n, c->f.n_elems, &c->fb, c->flr_with_avg);
        }
    } restore{ctx, n, all, main_stream};
    for (int c = 0; c < n_chunks; ++c) {
        const long o = cut[c], nc = cut[c + 1] - o;
        if (nc <= 0) continue;
        const int slot = c % slots;
        const size_t nb = (size_t)nc * sizeof(double);
        for (int k = 0; k < 8; ++k)
            CU(cudaMemcpyAsync(dd[k] + o, hs[k] + o, nb, cudaMemcpyHostToDevice, ctx->s_up), "upload chunk");
        CU(cudaEventRecord(ctx->ev_chunk[2 * c], ctx->s_up), "record upload");
        ctx->stream = slot ? ctx->s_c[slot] : main_stream;
        CU(cudaStreamWaitEvent(ctx->stream, ctx->ev_chunk[2 * c], 0), "compute waits for upload");
        // bind the chunk: same time and step counter for every chunk
        ctx->n = nc;
        ctx->user = MarkerArrays{all.x + o, all.y + o, all.z + o, all.vx + o, all.vy + o, all.vz + o, all.mu + o, all.w + o,
                                 all.elem + o, all.id + o};
        if (ctx->have_sortws)
            carve_sort_workspace(static_cast<char *>(ctx->sortws_base) + slot * sort_slot, nc, ctx->f.n_elems, &ctx->sb);
        if (ctx->have_flrws)
            carve_flr_workspace(static_cast<char *>(ctx->flrws_base) + slot * flr_slot, nc, ctx->f.n_elems, &ctx->fb, ctx->flr_with_avg);
        ctx->steps_done = steps0; ctx->steps_at_dt = at0; ctx->t_base = tb0; ctx->last_dt = ldt0;
        CU(launch_locate(ctx, ctx->user, nc, true, (int)o), "locate kernel");
        const int rc = run_steps(ctx, nsteps, dt);
        if (rc != M3DK_OK) return rc;
        CU(cudaEventRecord(ctx->ev_chunk[2 * c + 1], ctx->stream), "record compute");
        CU(cudaStreamWaitEvent(ctx->s_down, ctx->ev_chunk[2 * c + 1], 0), "download waits for compute");
        for (int k = 0; k < 8; ++k)                     // mu included: it travels with its marker through the sorts
            CU(cudaMemcpyAsync(hs[k] + o, dd[k] + o, nb, cudaMemcpyDeviceToHost, ctx->s_down), "download chunk");
        if (host_id) CU(cudaMemcpyAsync(host_id + o, all.id + o, (size_t)nc * sizeof(int), cudaMemcpyDeviceToHost, ctx->s_down), "download id");
        if (host_elem) CU(cudaMemcpyAsync(host_elem + o, all.elem + o, (size_t)nc * sizeof(int), cudaMemcpyDeviceToHost, ctx->s_down), "download elem");
    }
    ctx->stream = main_stream;
    for (int k = 1; k < slots; ++k) {      // work enqueued on the context's stream after this call sees every stream finished
        CU(cudaEventRecord(ev_start, ctx->s_c[k]), "record compute stream");
        CU(cudaStreamWaitEvent(main_stream, ev_start, 0), "join compute stream");
    }
    CU(cudaStreamSynchronize(ctx->s_down), "download stream synchronize (an earlier kernel may have failed)");
    CU(cudaStreamSynchronize(ctx->stream), "stream synchronize");
    return M3DK_OK;
}

extern "C" int m3dk_eval_fields(m3dk_ctx *ctx, long n, const double *R, const double *phi, const double *Z, double t,
                                int *elem_out, double *out) {
    if (!ctx) return M3DK_EINVAL;
    if (!ctx->have_fields) return fail(ctx, M3DK_ESTATE, "m3dk_eval_fields: call m3dk_fields_create first");
    if (n < 0 || (n > 0 && (!R || !phi || !Z || !elem_out || !out))) return fail(ctx, M3DK_EINVAL, "m3dk_eval_fields: bad argument");
    CU(cudaSetDevice(ctx->device), "cudaSetDevice");
    CU(launch_eval_fields(ctx, n, R, phi, Z, t, elem_out, out), "eval kernel");
    return M3DK_OK;
}

extern "C" int m3dk_gc_push(m3dk_ctx *ctx, int nsteps, double dt, double *vpar) {
    if (!ctx) return M3DK_EINVAL;
    if (!ctx->have_fields || !ctx->have_markers) return fail(ctx, M3DK_ESTATE, "m3dk_gc_push: fields and markers must be set first");
    if (nsteps < 0 || !(dt == dt) || (ctx->n > 0 && !vpar)) return fail(ctx, M3DK_EINVAL, "m3dk_gc_push: nsteps < 0, dt is NaN or vpar is NULL");
    CU(cudaSetDevice(ctx->device), "cudaSetDevice");
    // mode 1 (non-linear trajectories): the guiding centres move in the total fields at the context's time, which advances
    const bool pert = (ctx->mode == 1 || ctx->mode == 3) && ctx->f.n_modes > 0;
    const double t0 = pert ? step_time(ctx, dt) : 0.0;
    CU(launch_gc_push(ctx, ctx->n, vpar, nsteps, dt, pert, t0), "guiding-centre kernel");
    if (pert) { ctx->steps_done += nsteps; ctx->steps_at_dt += nsteps; }
    return M3DK_OK;
}

extern "C" int m3dk_gc_bootstrap(m3dk_ctx *ctx, double dt, const double *vpar) {
    if (!ctx) return M3DK_EINVAL;
    if (!ctx->have_fields || !ctx->have_markers) return fail(ctx, M3DK_ESTATE, "m3dk_gc_bootstrap: fields and markers must be set first");
    if (!(dt == dt) || dt == 0.0 || (ctx->n > 0 && !vpar)) return fail(ctx, M3DK_EINVAL, "m3dk_gc_bootstrap: dt is NaN or 0, or vpar is NULL");
    CU(cudaSetDevice(ctx->device), "cudaSetDevice");
    CU(launch_gc_bootstrap(ctx, ctx->n, vpar, dt), "guiding-centre bootstrap kernel");
    return M3DK_OK;
}

extern "C" int m3dk_deposit_bytes(const m3dk_ctx *ctx, size_t *bytes) {
    if (!ctx || !bytes) return M3DK_EINVAL;
    if (!ctx->have_fields) return M3DK_ESTATE;
    *bytes = (size_t)ctx->f.n_elems * 2 * (1 + 2 * ctx->f.n_modes) * M3DK_NCOEF * sizeof(double);
    return M3DK_OK;
}

extern "C" int m3dk_deposit(m3dk_ctx *ctx, double *rhs, int flags, double t) {
    if (!ctx) return M3DK_EINVAL;
    if (!ctx->have_fields || !ctx->have_markers) return fail(ctx, M3DK_ESTATE, "m3dk_deposit: fields and markers must be set first");
    if (!rhs || flags < 0 || flags > 7 || !(t == t)) return fail(ctx, M3DK_EINVAL, "m3dk_deposit: rhs is NULL, unknown flag or t is NaN");
    CU(cudaSetDevice(ctx->device), "cudaSetDevice");
    CU(launch_deposit(ctx, ctx->n, rhs, flags, t), "deposit kernel");
    return M3DK_OK;
}

extern "C" int m3dk_fp64_peak_tflops(m3dk_ctx *ctx, double *tflops) {
    if (!ctx || !tflops) return M3DK_EINVAL;
    if (!ctx->have_fields) return fail(ctx, M3DK_ESTATE, "m3dk_fp64_peak_tflops: call m3dk_fields_create first (uses its control block)");
    CU(cudaSetDevice(ctx->device), "cudaSetDevice");
    CU(fp64_probe(ctx, tflops), "fp64 probe");
    return M3DK_OK;
}

extern "C" int m3dk_set_profiling(m3dk_ctx *ctx, int on) {
    if (!ctx) return M3DK_EINVAL;
    CU(cudaSetDevice(ctx->device), "cudaSetDevice");
    CU(cudaStreamSynchronize(ctx->stream), "stream synchronize");
    drop_events(ctx->ev_push, nullptr, nullptr);
    drop_events(ctx->ev_sort, nullptr, nullptr);
    ctx->profiling = on != 0;
    ctx->push_ms = ctx->sort_ms = 0.0;
    ctx->push_launches = ctx->sort_launches = ctx->kernel_launches = 0;
    return M3DK_OK;
}

extern "C" int m3dk_timing(m3dk_ctx *ctx, m3dk_timing_t *out) {
    if (!ctx || !out) return M3DK_EINVAL;
    CU(cudaSetDevice(ctx->device), "cudaSetDevice");
    CU(cudaStreamSynchronize(ctx->stream), "stream synchronize (an earlier kernel may have failed)");
    drop_events(ctx->ev_push, &ctx->push_ms, &ctx->push_launches);
    drop_events(ctx->ev_sort, &ctx->sort_ms, &ctx->sort_launches);
    out->push_ms = ctx->push_ms; out->sort_ms = ctx->sort_ms;
    out->push_launches = ctx->push_launches; out->sort_launches = ctx->sort_launches;
    out->kernel_launches = ctx->kernel_launches;
    return M3DK_OK;
}
