// m3dk_sort.cu -- ordering of the markers by element and the record pipeline around it.
// key = element of the marker's current position (cached by the push), lost markers (-1) get key n_elems (last).
// Counting sort: histogram with returned ranks (one warp-aggregated atomic per marker; normally fused into the push
// kernel that produced the keys) -> exclusive scan (+ work-item cut) -> placement.  The placement never moves SoA
// pieces: markers travel as 64-byte records (two full sectors), and inside a push the records are not moved by a sort
// pass at all -- the next push gathers them through the (src, id) order list written here.
#include "m3dk_internal.h"

namespace m3dk {

static inline size_t up256(size_t b) { return (b + 255) / 256 * 256; }

size_t sort_workspace_bytes(long n, int n_elems) {
    const size_t nr = up256((size_t)n * kRecDoubles * sizeof(double)), no = up256((size_t)n * sizeof(int2));
    const size_t ni = up256((size_t)n * sizeof(int)), nh = up256((size_t)(n_elems + 2) * sizeof(int));
    const size_t nit = up256(((size_t)n / kItemMarkers + n_elems + 2) * sizeof(int4));
    const size_t nst = up256(((size_t)(n_elems + 1) / 4096 + 6) * sizeof(unsigned long long));
    const size_t nsm = up256((size_t)(n_elems + 2) * sizeof(int4));
    return 2 * nr + 2 * no + 2 * ni + 3 * nh + nit + nst + nsm;
}

void carve_sort_workspace(void *ws, long n, int n_elems, SortBuffers *sb) {
    char *p = static_cast<char *>(ws);
    const size_t nr = up256((size_t)n * kRecDoubles * sizeof(double)), no = up256((size_t)n * sizeof(int2));
    const size_t ni = up256((size_t)n * sizeof(int)), nh = up256((size_t)(n_elems + 2) * sizeof(int));
    for (int k = 0; k < 2; ++k) { sb->rec[k] = reinterpret_cast<double *>(p); p += nr; }
    for (int k = 0; k < 2; ++k) { sb->order[k] = reinterpret_cast<int2 *>(p); p += no; }
    sb->key = reinterpret_cast<int *>(p); p += ni;
    sb->rank = reinterpret_cast<int *>(p); p += ni;
    sb->hist = reinterpret_cast<int *>(p); p += nh;
    sb->offs = reinterpret_cast<int *>(p); p += nh;
    sb->ioffs = reinterpret_cast<int *>(p); p += nh;
    sb->items = reinterpret_cast<int4 *>(p); p += up256(((size_t)n / kItemMarkers + n_elems + 2) * sizeof(int4));
    sb->scan_state = reinterpret_cast<unsigned long long *>(p); p += up256(((size_t)(n_elems + 1) / 4096 + 6) * sizeof(unsigned long long));
    sb->items_small = reinterpret_cast<int4 *>(p); p += up256((size_t)(n_elems + 2) * sizeof(int4));
    sb->bytes = (size_t)(p - static_cast<char *>(ws));
}

__global__ void __launch_bounds__(256) hist_rank_kernel(const int *__restrict__ elem, long n, int n_elems,
                                                        int *__restrict__ hist, int *__restrict__ rank) {
    const long i = (long)blockIdx.x * blockDim.x + threadIdx.x;
    const unsigned live = __ballot_sync(0xffffffffu, i < n);
    if (i >= n) return;
    const int e = elem[i];
    const int key = e < 0 ? n_elems : e;
    // warp-aggregated: lanes with the same key elect a leader that does one atomic for the group
    const unsigned peers = __match_any_sync(live, key);
    const int lane = threadIdx.x & 31;
    const int leader = __ffs(peers) - 1;
    int base = 0;
    if (lane == leader) base = atomicAdd(hist + key, __popc(peers));
    base = __shfl_sync(peers, base, leader);
    rank[i] = base + __popc(peers & ((1u << lane) - 1u));
}

// exclusive scan of hist[0..m) into offs[0..m] (offs[m] = total) and, in the same sweep, of the work-item counts
// ceil(hist[k] / kItemMarkers) into ioffs[0..m].  Single pass, decoupled look-back: a CTA takes a chunk of 4096 bins by
// ticket, publishes the chunk's totals at once, then sums the totals of the chunks before it (which were taken earlier,
// so they are running: no deadlock) while it scans its own bins.  state[0] = ticket counter, state[2 + c] = totals of
// chunk c with a ready tag in the upper bits; the launcher clears the state (a few hundred bytes) before each launch.
// word = tag << 56 | items << 31 | markers   (markers < 2^31, items < 2^25)
// Cut of an element's run of c markers: full items of kItemMarkers, a remainder of more than 32 markers is one more item
// of the same kind (both slots of a lane in use), a remainder of 1..32 markers becomes a SMALL item (one marker per lane),
// pushed by the one-slot instance of the kernel: no arithmetic is issued for an empty second slot.
__host__ __device__ inline int n_big_items(int c) { return c / kItemMarkers + ((c % kItemMarkers) > 32 ? 1 : 0); }

constexpr int kScanChunk = 4096;
__global__ void __launch_bounds__(1024) scan_kernel(int *__restrict__ hist, int m, int *__restrict__ offs,
                                                    int *__restrict__ ioffs, unsigned long long *state,
                                                    unsigned epoch) {
    __shared__ int2 wsum[32];
    __shared__ int2 prefix_s;
    __shared__ int chunk_s;
    const int t = threadIdx.x, lane = t & 31, wid = t >> 5;
    if (t == 0) chunk_s = (int)atomicAdd(state, 1ull);
    __syncthreads();
    const int chunk = chunk_s;
    const int nchunks = (m + kScanChunk - 1) / kScanChunk;
    if (chunk >= nchunks) return;
    const int k = chunk * kScanChunk + 4 * t;
    int v[4], it[4];
#pragma unroll
    for (int q = 0; q < 4; ++q) {
        v[q] = k + q < m ? hist[k + q] : 0;
        it[q] = n_big_items(v[q]);
        if (k + q < m) hist[k + q] = 0;       // the counts are consumed: the array serves invert_kernel<true> as slot cursors
    }
    const int2 mine = make_int2(v[0] + v[1] + v[2] + v[3], it[0] + it[1] + it[2] + it[3]);
    int2 inc = mine;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const int ux = __shfl_up_sync(0xffffffffu, inc.x, o), uy = __shfl_up_sync(0xffffffffu, inc.y, o);
        if (lane >= o) { inc.x += ux; inc.y += uy; }
    }
    if (lane == 31) wsum[wid] = inc;
    __syncthreads();
    if (wid == 0) {
        int2 w = wsum[lane];
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const int ux = __shfl_up_sync(0xffffffffu, w.x, o), uy = __shfl_up_sync(0xffffffffu, w.y, o);
            if (lane >= o) { w.x += ux; w.y += uy; }
        }
        wsum[lane] = w;      // inclusive over warps; lane 31 holds the chunk's totals
        const unsigned long long tag = (unsigned long long)(epoch & 0xffu) << 56;
        if (lane == 31) {
            const unsigned long long word = tag | ((unsigned long long)(unsigned)w.y << 31) | (unsigned long long)(unsigned)w.x;
            atomicExch(state + 2 + chunk, word);
        }
        // look back over the chunks before this one, 32 at a time
        long long px = 0, py = 0;
        for (int c0 = chunk - 1; c0 >= 0; c0 -= 32) {
            const int c = c0 - lane;
            unsigned long long word = 0ull;
            if (c >= 0) {
                do { word = *reinterpret_cast<volatile unsigned long long *>(state + 2 + c); } while ((word >> 56) != (tag >> 56));
                px += (long long)(word & 0x7fffffffull);
                py += (long long)((word >> 31) & 0x1ffffffull);
            }
        }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) { px += __shfl_xor_sync(0xffffffffu, px, o); py += __shfl_xor_sync(0xffffffffu, py, o); }
        if (lane == 0) prefix_s = make_int2((int)px, (int)py);
    }
    __syncthreads();
    const int2 carry = prefix_s;
    const int2 wprev = wid ? wsum[wid - 1] : make_int2(0, 0);
    int run = carry.x + wprev.x + inc.x - mine.x, irun = carry.y + wprev.y + inc.y - mine.y;
#pragma unroll
    for (int q = 0; q < 4; ++q) {
        if (k + q < m) { offs[k + q] = run; ioffs[k + q] = irun; }
        run += v[q]; irun += it[q];
    }
    if (chunk == nchunks - 1 && t == 1023) { offs[m] = carry.x + wsum[31].x; ioffs[m] = carry.y + wsum[31].y; }
}

// work items of the element-ordered push: element k's sorted segment [offs[k], offs[k+1]) cut as n_big_items() says;
// k = n_elems is the pseudo-element of the lost markers.  Small items are appended to their own list through a counter
// (their order does not matter: every item is independent).
__global__ void __launch_bounds__(256) items_kernel(const int *__restrict__ offs, const int *__restrict__ ioffs, int m,
                                                    int4 *__restrict__ items, int4 *__restrict__ items_small,
                                                    int *__restrict__ n_small) {
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= m) return;
    const int b = offs[k], cnt = offs[k + 1] - b;
    int j = ioffs[k], c = 0;
    for (; cnt - c > 32; c += kItemMarkers, ++j) items[j] = make_int4(k, b + c, min(kItemMarkers, cnt - c), 0);
    if (cnt - c > 0) items_small[atomicAdd(n_small, 1)] = make_int4(k, b + c, cnt - c, 0);
}

__device__ __forceinline__ void st256(double *p, double a, double b, double c, double d) {
    asm volatile("st.global.v4.f64 [%0], {%1, %2, %3, %4};" ::"l"(p), "d"(a), "d"(b), "d"(c), "d"(d) : "memory");
}
__device__ __forceinline__ void ld256(const double *p, double &a, double &b, double &c, double &d) {
    asm volatile("ld.global.v4.f64 {%0, %1, %2, %3}, [%4];" : "=d"(a), "=d"(b), "=d"(c), "=d"(d) : "l"(p) : "memory");
}

// caller's SoA arrays -> records in element order: slot d = offs[key] + rank; order[d] = (d, id): the first push of the
// call reads its records in place
__global__ void __launch_bounds__(256) pack_kernel(MarkerArrays a, long n, int n_elems, const int *__restrict__ offs,
                                                   const int *__restrict__ rank, double *__restrict__ rec,
                                                   int2 *__restrict__ order, int *__restrict__ key) {
    const long i = (long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const int e = a.elem[i];
    const int k = e < 0 ? n_elems : e;
    const long d = (long)offs[k] + rank[i];
    st256(rec + kRecDoubles * d, a.x[i], a.y[i], a.z[i], a.w[i]);
    st256(rec + kRecDoubles * d + 4, a.vx[i], a.vy[i], a.vz[i], a.mu[i]);
    order[d] = make_int2((int)d, a.id[i]);
    key[d] = k;
}

// next order list: the record in slot j goes to slot d = offs[key[j]] + rank[j] of the next element-ordered push.
// kDraw = false: rank[] was written by the push kernel (returned histogram atomics).  kDraw = true: the push kernel only
// counted (atomics without a returned value: nothing pending in its registers); the rank inside the key is drawn here from
// cursor[] (the histogram array, zeroed by the scan) with one warp-aggregated atomic per distinct key of a warp.  Slots
// are in the order of the OLD elements, so neighbouring warps would hit the same few cursors at the same time: block b
// takes the chunk (b * cstride) mod gridDim.x (cstride coprime with the grid, chosen by the launcher).
template <bool kDraw>
__global__ void __launch_bounds__(256) invert_kernel(long n, const int *__restrict__ key, const int *__restrict__ offs,
                                                     const int *__restrict__ rank, int *__restrict__ cursor,
                                                     const int2 *__restrict__ order_cur, int2 *__restrict__ order_next,
                                                     unsigned cstride) {
    const unsigned blk = kDraw ? (unsigned)(((unsigned long long)blockIdx.x * cstride) % gridDim.x) : blockIdx.x;
    const long j = (long)blk * blockDim.x + threadIdx.x;
    const bool on = j < n;
    if (!kDraw) {
        if (on) order_next[(long)offs[key[j]] + rank[j]] = make_int2((int)j, order_cur[j].y);
        return;
    }
    const unsigned live = __ballot_sync(0xffffffffu, on);
    if (!on) return;
    const int k = key[j];
    const unsigned peers = __match_any_sync(live, k);
    const int lane = threadIdx.x & 31, leader = __ffs(peers) - 1;
    int base = 0;
    if (lane == leader) base = atomicAdd(cursor + k, __popc(peers));
    base = __shfl_sync(peers, base, leader);
    const long d = (long)offs[k] + base + __popc(peers & ((1u << lane) - 1u));
    order_next[d] = make_int2((int)j, order_cur[j].y);
}

// records -> caller's SoA arrays, slot by slot (the caller's arrays end up in the record order; id says who is where)
__global__ void __launch_bounds__(256) unpack_kernel(MarkerArrays a, long n, int n_elems, const double *__restrict__ rec,
                                                     const int2 *__restrict__ order, const int *__restrict__ key) {
    const long j = (long)blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= n) return;
    double x, y, z, w, vx, vy, vz, mu;
    ld256(rec + kRecDoubles * j, x, y, z, w);
    ld256(rec + kRecDoubles * j + 4, vx, vy, vz, mu);
    a.x[j] = x; a.y[j] = y; a.z[j] = z; a.w[j] = w;
    a.vx[j] = vx; a.vy[j] = vy; a.vz[j] = vz; a.mu[j] = mu;
    a.id[j] = order[j].y;
    const int k = key[j];
    a.elem[j] = k >= n_elems ? -1 : k;
}

// scan of a histogram of m = n_elems + 1 bins into segment offsets, work-item cut (shared by the marker ordering and the
// ring ordering of the FLR mode)
static cudaError_t scan_and_cut_arrays(m3dk_ctx *c, int *hist, int *offs, int *ioffs, int4 *items, int4 *items_small,
                                       unsigned long long *state) {
    const int m = c->f.n_elems + 1;
    c->kernel_launches += 2;
    const int nchunks = (m + kScanChunk - 1) / kScanChunk;
    // ticket and per-chunk words cleared together (a few hundred bytes): a word is ready when its tag is set
    cudaError_t e = cudaMemsetAsync(state, 0, (size_t)(nchunks + 3) * sizeof(unsigned long long), c->stream);
    if (e != cudaSuccess) return e;
    scan_kernel<<<nchunks, 1024, 0, c->stream>>>(hist, m, offs, ioffs, state, 1u);
    items_kernel<<<(m + 255) / 256, 256, 0, c->stream>>>(offs, ioffs, m, items, items_small, reinterpret_cast<int *>(state + 1));
    return cudaGetLastError();
}
static cudaError_t scan_and_cut(m3dk_ctx *c) {
    return scan_and_cut_arrays(c, c->sb.hist, c->sb.offs, c->sb.ioffs, c->sb.items, c->sb.items_small, c->sb.scan_state);
}

// ---- ring stream of the ordered FLR mode ----------------------------------------------------------------------------------
size_t flr_workspace_bytes(long n, int n_elems, bool with_avg) {
    const size_t n4 = 4 * (size_t)n;
    const size_t nh = up256((size_t)(n_elems + 2) * sizeof(int));
    return up256(n4 * 4 * sizeof(double)) + up256((size_t)n * 10 * sizeof(double)) + up256(n4 * sizeof(double)) +
           3 * up256(n4 * sizeof(int)) + 3 * nh + up256((n4 / kItemMarkers + n_elems + 2) * sizeof(int4)) +
           up256((size_t)(n_elems + 2) * sizeof(int4)) + up256(((size_t)(n_elems + 1) / 4096 + 6) * sizeof(unsigned long long)) +
           (with_avg ? up256(n4 * kAvgDoubles * sizeof(double)) : 0);
}

void carve_flr_workspace(void *ws, long n, int n_elems, FlrBuffers *fb, bool with_avg) {
    char *p = static_cast<char *>(ws);
    const size_t n4 = 4 * (size_t)n;
    const size_t nh = up256((size_t)(n_elems + 2) * sizeof(int));
    fb->a.ring = reinterpret_cast<double *>(p); p += up256(n4 * 4 * sizeof(double));
    fb->a.wts = reinterpret_cast<double *>(p); p += up256((size_t)n * 10 * sizeof(double));
    fb->a.contrib = reinterpret_cast<double *>(p); p += up256(n4 * sizeof(double));
    fb->a.rkey = reinterpret_cast<int *>(p); p += up256(n4 * sizeof(int));
    fb->a.rrank = reinterpret_cast<int *>(p); p += up256(n4 * sizeof(int));
    fb->a.rorder = reinterpret_cast<int *>(p); p += up256(n4 * sizeof(int));
    fb->a.rhist = reinterpret_cast<int *>(p); p += nh;
    fb->roffs = reinterpret_cast<int *>(p); p += nh;
    fb->rioffs = reinterpret_cast<int *>(p); p += nh;
    fb->ritems = reinterpret_cast<int4 *>(p); p += up256((n4 / kItemMarkers + n_elems + 2) * sizeof(int4));
    fb->ritems_small = reinterpret_cast<int4 *>(p); p += up256((size_t)(n_elems + 2) * sizeof(int4));
    fb->rstate = reinterpret_cast<unsigned long long *>(p); p += up256(((size_t)(n_elems + 1) / 4096 + 6) * sizeof(unsigned long long));
    fb->a.avg = nullptr;
    if (with_avg) { fb->a.avg = reinterpret_cast<double *>(p); p += up256(n4 * kAvgDoubles * sizeof(double)); }
    fb->bytes = (size_t)(p - static_cast<char *>(ws));
}

// ring point i goes to position offs[key] + rank of the element-ordered ring list; a point outside the mesh contributes
// zero; points of a lost marker's slot (key -1) are not in the list
__global__ void __launch_bounds__(256) ring_place_kernel(long n4, int n_elems, const int *__restrict__ rkey,
                                                         const int *__restrict__ rrank, const int *__restrict__ roffs,
                                                         int *__restrict__ rorder, double *__restrict__ contrib) {
    const long i = (long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n4) return;
    const int k = rkey[i];
    if (k < 0) return;
    rorder[(long)roffs[k] + rrank[i]] = (int)i;
    if (k >= n_elems) contrib[i] = 0.0;
}

// Eq. (14) and the weight update (readings G9, G23): w_{l+1/2} = w_{l-1/2} + dt * 0.25 (((c_0 + c_1) + c_2) + c_3) on the
// records the push has just written (their w is still the old one)
__global__ void __launch_bounds__(256) flr_reduce_kernel(long n, double dt, const int *__restrict__ rkey,
                                                         const double *__restrict__ contrib, double *__restrict__ rec) {
    const long d = (long)blockIdx.x * blockDim.x + threadIdx.x;
    if (d >= n) return;
    if (rkey[4 * d] < 0) return;                       // the slot holds a marker that was lost before this step
    const double4 c = *reinterpret_cast<const double4 *>(contrib + 4 * d);
    const double sum = __dadd_rn(__dadd_rn(__dadd_rn(c.x, c.y), c.z), c.w);
    double *w = rec + kRecDoubles * d + 3;
#ifdef M3DK_NO_FMA
    *w = __dadd_rn(__dmul_rn(dt, __dmul_rn(0.25, sum)), *w);
#else
    *w = fma(dt, __dmul_rn(0.25, sum), *w);
#endif
}

cudaError_t launch_flr_ring_stage(m3dk_ctx *c, long n) {
    if (n == 0) return cudaSuccess;
    FlrBuffers &fb = c->fb;
    cudaError_t e = scan_and_cut_arrays(c, fb.a.rhist, fb.roffs, fb.rioffs, fb.ritems, fb.ritems_small, fb.rstate);
    if (e != cudaSuccess) return e;
    c->kernel_launches += 1;
    const long n4 = 4 * n;
    ring_place_kernel<<<(unsigned)((n4 + 255) / 256), 256, 0, c->stream>>>(n4, c->f.n_elems, fb.a.rkey, fb.a.rrank, fb.roffs,
                                                                          fb.a.rorder, fb.a.contrib);
    return cudaGetLastError();
}

cudaError_t launch_flr_reduce(m3dk_ctx *c, long n, double dt) {
    if (n == 0) return cudaSuccess;
    c->kernel_launches += 1;
    flr_reduce_kernel<<<(unsigned)((n + 255) / 256), 256, 0, c->stream>>>(n, dt, c->fb.a.rkey, c->fb.a.contrib, c->sb.rec[c->cur]);
    return cudaGetLastError();
}

cudaError_t launch_pack_sorted(m3dk_ctx *c, long n) {
    if (n == 0) return cudaSuccess;
    const int m = c->f.n_elems + 1;
    const unsigned grid = (unsigned)((n + 255) / 256);
    cudaError_t e = cudaMemsetAsync(c->sb.hist, 0, (size_t)m * sizeof(int), c->stream);
    if (e != cudaSuccess) return e;
    c->kernel_launches += 2;
    hist_rank_kernel<<<grid, 256, 0, c->stream>>>(c->user.elem, n, c->f.n_elems, c->sb.hist, c->sb.rank);
    e = scan_and_cut(c);
    if (e != cudaSuccess) return e;
    c->cur = 0; c->ocur = 0;
    pack_kernel<<<grid, 256, 0, c->stream>>>(c->user, n, c->f.n_elems, c->sb.offs, c->sb.rank, c->sb.rec[0], c->sb.order[0],
                                            c->sb.key);
    return cudaGetLastError();
}

cudaError_t launch_reorder(m3dk_ctx *c, long n) {
    if (n == 0) return cudaSuccess;
    cudaError_t e = scan_and_cut(c);
    if (e != cudaSuccess) return e;
    c->kernel_launches += 1;
    const unsigned grid = (unsigned)((n + 255) / 256);
    if (c->ranks_valid) {
        invert_kernel<false><<<grid, 256, 0, c->stream>>>(n, c->sb.key, c->sb.offs, c->sb.rank, c->sb.hist,
                                                         c->sb.order[c->ocur], c->sb.order[c->ocur ^ 1], 1u);
    } else {
        static const unsigned primes[] = {1009u, 1013u, 1019u, 1021u, 1031u};
        unsigned cs = 1u;
        for (unsigned p : primes)
            if (grid % p != 0) { cs = p; break; }
        invert_kernel<true><<<grid, 256, 0, c->stream>>>(n, c->sb.key, c->sb.offs, c->sb.rank, c->sb.hist,
                                                        c->sb.order[c->ocur], c->sb.order[c->ocur ^ 1], cs);
    }
    c->ocur ^= 1;
    return cudaGetLastError();
}

cudaError_t launch_unpack(m3dk_ctx *c, long n) {
    if (n == 0) return cudaSuccess;
    c->kernel_launches += 1;
    unpack_kernel<<<(unsigned)((n + 255) / 256), 256, 0, c->stream>>>(c->user, n, c->f.n_elems, c->sb.rec[c->cur],
                                                                       c->sb.order[c->ocur], c->sb.key);
    return cudaGetLastError();
}

}  // namespace m3dk
