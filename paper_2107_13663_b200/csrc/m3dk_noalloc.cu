// m3dk_noalloc.cu -- m3dk_deposit_noalloc (include/m3dk.h): the element-ordered moment deposition for callers that can
// neither allocate device memory nor lend a sort workspace.  The ordering scratch (records, order list, keys, ranks,
// histogram, offsets, work items, scan state: the layout of carve_sort_workspace) lives in ONE file-scope device array of
// M3DK_NOALLOC_SCRATCH_BYTES, which every GPU that loads the library holds until the process exits.
//
// The array's name is a host-side stand-in in host code, not a device address: the address a kernel can use is asked for
// once per device with cudaGetSymbolAddress (that device current) and cached here.  This entry point calls no cudaMalloc,
// cudaFree or allocating library routine: cudaSetDevice, cudaGetSymbolAddress (first call on a device only),
// cudaMemsetAsync and kernel launches.
#include <mutex>

#include "m3dk_internal.h"

using namespace m3dk;

static __device__ __align__(256) unsigned char g_noalloc_scratch[M3DK_NOALLOC_SCRATCH_BYTES];

static constexpr int kMaxDevices = 64;
static std::mutex g_scratch_mutex;
static void *g_scratch_addr[kMaxDevices] = {};      // device address of g_noalloc_scratch on device k (0 = not asked yet)

// device address of the scratch array on `device`, which must be the current device
static cudaError_t scratch_address(int device, void **out) {
    std::lock_guard<std::mutex> lock(g_scratch_mutex);
    if (!g_scratch_addr[device]) {
        void *p = nullptr;
        const cudaError_t e = cudaGetSymbolAddress(&p, g_noalloc_scratch);
        if (e != cudaSuccess) return e;
        g_scratch_addr[device] = p;
    }
    *out = g_scratch_addr[device];
    return cudaSuccess;
}

static int fail_na(m3dk_ctx *c, int code, const std::string &msg) {
    c->err = msg;
    return code;
}

extern "C" int m3dk_noalloc_scratch_bytes(size_t *bytes) {
    if (!bytes) return M3DK_EINVAL;
    *bytes = (size_t)M3DK_NOALLOC_SCRATCH_BYTES;
    return M3DK_OK;
}

extern "C" int m3dk_deposit_noalloc(m3dk_ctx *ctx, double *rhs, int flags, double t) {
    if (!ctx) return M3DK_EINVAL;
    if (!ctx->have_fields || !ctx->have_markers)
        return fail_na(ctx, M3DK_ESTATE, "m3dk_deposit_noalloc: fields and markers must be set first");
    if (!rhs || flags < 0 || flags > 7 || !(t == t))
        return fail_na(ctx, M3DK_EINVAL, "m3dk_deposit_noalloc: rhs is NULL, unknown flag or t is NaN");
    if (ctx->device < 0 || ctx->device >= kMaxDevices)
        return fail_na(ctx, M3DK_EINVAL, "m3dk_deposit_noalloc: device index beyond the 64 this entry point keeps an address for");
    const size_t need = sort_workspace_bytes(ctx->n, ctx->f.n_elems);
    if (need > (size_t)M3DK_NOALLOC_SCRATCH_BYTES)
        return fail_na(ctx, M3DK_EWORKSPACE,
                       "m3dk_deposit_noalloc: " + std::to_string(ctx->n) + " markers on " + std::to_string(ctx->f.n_elems) +
                           " elements need " + std::to_string(need) + " bytes of ordering scratch, the static array holds " +
                           std::to_string((size_t)M3DK_NOALLOC_SCRATCH_BYTES) +
                           " (M3DK_NOALLOC_SCRATCH_BYTES); use m3dk_deposit with a sort workspace");
    cudaError_t e = cudaSetDevice(ctx->device);
    void *scratch = nullptr;
    if (e == cudaSuccess) e = scratch_address(ctx->device, &scratch);
    if (e != cudaSuccess)
        return fail_na(ctx, M3DK_ECUDA, std::string("m3dk_deposit_noalloc: ") + cudaGetErrorName(e) + " (" + cudaGetErrorString(e) + ")");

    // bind the ordering buffers to the static array for this call only: launch_deposit then takes the element-ordered
    // path (the 4-point deposition without the ring stream, which would need the FLR workspace as well); the context
    // leaves with the caller's own workspaces bound as before
    struct Rebind {
        m3dk_ctx *c; SortBuffers sb; bool sortws, flrws;
        ~Rebind() { c->sb = sb; c->have_sortws = sortws; c->have_flrws = flrws; }
    } rebind{ctx, ctx->sb, ctx->have_sortws, ctx->have_flrws};
    carve_sort_workspace(scratch, ctx->n, ctx->f.n_elems, &ctx->sb);
    ctx->have_sortws = true;
    ctx->have_flrws = false;
    // what must start at zero (histogram, scan state, item counters) is cleared by the ordering launchers themselves on
    // every call; everything else in the array is written before it is read
    e = launch_deposit(ctx, ctx->n, rhs, flags, t);
    if (e != cudaSuccess)
        return fail_na(ctx, M3DK_ECUDA, std::string("m3dk_deposit_noalloc: deposit kernel: ") + cudaGetErrorName(e) + " (" +
                                            cudaGetErrorString(e) + ")");
    return M3DK_OK;
}
