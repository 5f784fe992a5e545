// ingest.cu -- a0-a3: window/sensor filter, per-pixel histogram, exclusive scan + active
// list + size-classed work list, deterministic (input-order) scatter into CSR.
//
// "For each window, events are moved to the GPU, sorted by pixel index";
// pixels with fewer than n_min events are discarded (L137).  Readings R19 (half-open
// window, bad coordinates dropped and counted) and R20 (input order inside a row).
//
// HBM-bound: 16 B read per event twice (histogram, scatter) + 8 B written and read once
// (unsorted pairs, normally L2-resident) + 4 B written (csr_ev).  The scatter takes a slot
// with an atomic per pixel, which gives an arbitrary order inside a row; k_rowsort then
// ranks every element of a row by its input index, which restores input order exactly, so
// csr_ev is bit-reproducible.
#include "ddhf_internal.cuh"

namespace ddhf {

namespace {

constexpr int kEvThreads = 256;
constexpr int kEvUnroll = 4;
constexpr int kRowPix = 128;       // pixels per k_rowsort_short block
constexpr int kRowCap = 4096;      // pairs staged in shared memory per block
constexpr int kShortMax = 64;      // rows up to this length are ranked by counting
constexpr int kLongBlocks = 148 * 6;

struct Ev {
    int32_t pix;       // -1 if dropped
    uint32_t val;      // (t - t0) << 1 | (p > 0)
};

__device__ __forceinline__ Ev decode_event(const ddhf_event *ev, int64_t i, int64_t t0, int64_t t1,
                                           int32_t width, int32_t height)
{
    const int4 w = __ldg(reinterpret_cast<const int4 *>(ev) + i);
    const uint32_t x = static_cast<uint32_t>(w.x) & 0xffffu;
    const uint32_t y = static_cast<uint32_t>(w.x) >> 16;
    const int32_t p = static_cast<int16_t>(static_cast<uint32_t>(w.y) & 0xffffu);
    const int64_t t = static_cast<int64_t>((static_cast<uint64_t>(static_cast<uint32_t>(w.w)) << 32) |
                                           static_cast<uint32_t>(w.z));
    Ev e;
    const bool ok = (t >= t0) && (t < t1) && (x < static_cast<uint32_t>(width)) &&
                    (y < static_cast<uint32_t>(height));
    e.pix = ok ? static_cast<int32_t>(y * static_cast<uint32_t>(width) + x) : -1;
    e.val = (static_cast<uint32_t>(t - t0) << 1) | (p > 0 ? 1u : 0u);
    return e;
}

__device__ __forceinline__ int size_class(int n)
{
    // 0: n < 8, 1: 8..15, 2: 16..31, ... , 11: n >= 8192
    const int bl = 32 - __clz(n);
    return min(kNumClasses - 1, max(0, bl - 3));
}

// ---- k_init: per-pixel maps for inactive pixels, zeroed histogram and counters ---------
__global__ void k_init(IngestParams p)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < p.np) {
        p.cnt[i] = 0;
        p.sf[i] = __int_as_float(0x7fc00000);   // NaN: pixel not active
        p.score[i] = 0.f;
        p.f0_idx[i] = -1;
        p.mask[i] = 0;
    }
    if (blockIdx.x == 0) {
        if (threadIdx.x < DDHF_N_COUNTERS) p.counters[threadIdx.x] = 0;
        if (threadIdx.x < kNumClasses) {
            p.class_cnt[threadIdx.x] = 0;
            p.class_cur[threadIdx.x] = 0;
        }
        if (threadIdx.x == 0) { *p.work_cursor = 0ull; *p.n_long = 0; }
    }
}

// ---- k_hist: counts[pix] += 1 (a1), dropped-event counter -----------------------------
__global__ void __launch_bounds__(kEvThreads) k_hist(IngestParams p)
{
    __shared__ int s_drop;
    if (threadIdx.x == 0) s_drop = 0;
    __syncthreads();
    const int64_t base = static_cast<int64_t>(blockIdx.x) * (kEvThreads * kEvUnroll) + threadIdx.x;
    Ev e[kEvUnroll];
#pragma unroll
    for (int u = 0; u < kEvUnroll; ++u) {
        const int64_t i = base + u * kEvThreads;
        e[u].pix = -2;
        if (i < p.n) e[u] = decode_event(p.events, i, p.t0, p.t1, p.width, p.height);
    }
    int drop = 0;
#pragma unroll
    for (int u = 0; u < kEvUnroll; ++u) {
        if (e[u].pix >= 0) atomicAdd(&p.cnt[e[u].pix], 1);
        drop += (e[u].pix == -1);
    }
    drop = __reduce_add_sync(0xffffffffu, drop);
    if ((threadIdx.x & 31) == 0 && drop) atomicAdd(&s_drop, drop);
    __syncthreads();
    if (threadIdx.x == 0 && s_drop) atomicAdd(&p.counters[DDHF_CNT_N_DROPPED], s_drop);
}

// ---- block-wide exclusive scan of two ints (1024 threads) -----------------------------
__device__ __forceinline__ void block_scan2(int &a, int &b, int &tot_a, int &tot_b, int *s_a, int *s_b)
{
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    int ia = a, ib = b;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const int ta = __shfl_up_sync(0xffffffffu, ia, o);
        const int tb = __shfl_up_sync(0xffffffffu, ib, o);
        if (lane >= o) { ia += ta; ib += tb; }
    }
    if (lane == 31) { s_a[wid] = ia; s_b[wid] = ib; }
    __syncthreads();
    if (wid == 0) {
        int wa = s_a[lane], wb = s_b[lane];
        const int nw = blockDim.x >> 5;
        if (lane >= nw) { wa = 0; wb = 0; }
        int xa = wa, xb = wb;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const int ta = __shfl_up_sync(0xffffffffu, xa, o);
            const int tb = __shfl_up_sync(0xffffffffu, xb, o);
            if (lane >= o) { xa += ta; xb += tb; }
        }
        s_a[lane] = xa - wa;          // exclusive warp offsets
        s_b[lane] = xb - wb;
        if (lane == 31) { s_a[32] = xa; s_b[32] = xb; }
    }
    __syncthreads();
    a = ia - a + s_a[wid];            // exclusive prefix of this thread
    b = ib - b + s_b[wid];
    tot_a = s_a[32];
    tot_b = s_b[32];
    __syncthreads();
}

__device__ __forceinline__ void load4(const int32_t *src, int base, int np, int (&v)[4])
{
    if (base + 3 < np) {
        const int4 q = *reinterpret_cast<const int4 *>(src + base);
        v[0] = q.x; v[1] = q.y; v[2] = q.z; v[3] = q.w;
    } else {
#pragma unroll
        for (int j = 0; j < 4; ++j) v[j] = (base + j < np) ? src[base + j] : 0;
    }
}

// ---- k_scan_reduce: per-tile totals of counts and active flags, class histogram --------
__global__ void __launch_bounds__(1024) k_scan_reduce(IngestParams p)
{
    __shared__ int s_a[33], s_b[33];
    __shared__ int s_cls[kNumClasses];
    if (threadIdx.x < kNumClasses) s_cls[threadIdx.x] = 0;
    __syncthreads();
    const int base = blockIdx.x * kScanTile + threadIdx.x * 4;
    int v[4];
    load4(p.cnt, base, p.np, v);
    int sum = 0, act = 0;
    const int nmin = max(p.n_min, 1);
#pragma unroll
    for (int j = 0; j < 4; ++j) {
        sum += v[j];
        if (v[j] >= nmin) {
            ++act;
            atomicAdd(&s_cls[size_class(v[j])], 1);
        }
    }
    int ta, tb;
    block_scan2(sum, act, ta, tb, s_a, s_b);
    if (threadIdx.x == 0) {
        p.tile_sum[blockIdx.x] = ta;
        p.tile_act[blockIdx.x] = tb;
    }
    if (threadIdx.x < kNumClasses && s_cls[threadIdx.x])
        atomicAdd(&p.class_cnt[threadIdx.x], s_cls[threadIdx.x]);
}

// ---- k_scan_tiles: one block scans the tile totals; class bases (largest rows first) ---
__global__ void __launch_bounds__(1024) k_scan_tiles(IngestParams p, int n_tiles)
{
    __shared__ int s_a[33], s_b[33];
    int a = (threadIdx.x < n_tiles) ? p.tile_sum[threadIdx.x] : 0;
    int b = (threadIdx.x < n_tiles) ? p.tile_act[threadIdx.x] : 0;
    int ta, tb;
    block_scan2(a, b, ta, tb, s_a, s_b);
    if (threadIdx.x < n_tiles) {
        p.tile_off[threadIdx.x] = a;
        p.tile_aoff[threadIdx.x] = b;
    }
    if (threadIdx.x == 0) {
        p.row_ptr[p.np] = ta;
        p.counters[DDHF_CNT_N_IN] = ta;
        p.counters[DDHF_CNT_N_ACTIVE] = tb;
        if (tb > p.max_active) atomicOr(&p.counters[DDHF_CNT_OVERFLOW], 1);
        int run = 0;
        for (int c = kNumClasses - 1; c >= 0; --c) {     // descending cost
            const int n = p.class_cnt[c];
            p.class_cnt[c] = run;                         // becomes the class base
            run += n;
        }
    }
}

// ---- k_scan_apply: row_ptr, active_idx, work list; re-zero the histogram ---------------
__global__ void __launch_bounds__(1024) k_scan_apply(IngestParams p)
{
    __shared__ int s_a[33], s_b[33];
    __shared__ int s_cls[kNumClasses], s_base[kNumClasses];
    __shared__ int s_nlong, s_longbase;
    if (threadIdx.x < kNumClasses) s_cls[threadIdx.x] = 0;
    if (threadIdx.x == 0) s_nlong = 0;
    __syncthreads();
    const int base = blockIdx.x * kScanTile + threadIdx.x * 4;
    int v[4];
    load4(p.cnt, base, p.np, v);
    const int nmin = max(p.n_min, 1);
    int sum = 0, act = 0;
    int lrank[4], llong[4];
#pragma unroll
    for (int j = 0; j < 4; ++j) {
        sum += v[j];
        lrank[j] = -1;
        llong[j] = -1;
        if (v[j] >= nmin) {
            ++act;
            lrank[j] = atomicAdd(&s_cls[size_class(v[j])], 1);
        }
        if (v[j] > kShortMax) llong[j] = atomicAdd(&s_nlong, 1);
    }
    int ta, tb;
    block_scan2(sum, act, ta, tb, s_a, s_b);       // contains __syncthreads: s_cls, s_nlong are final
    if (threadIdx.x < kNumClasses) {
        const int n = s_cls[threadIdx.x];
        s_base[threadIdx.x] = p.class_cnt[threadIdx.x] + (n ? atomicAdd(&p.class_cur[threadIdx.x], n) : 0);
    }
    if (threadIdx.x == 32) s_longbase = s_nlong ? atomicAdd(p.n_long, s_nlong) : 0;
    __syncthreads();
    int off = p.tile_off[blockIdx.x] + sum;
    int aoff = p.tile_aoff[blockIdx.x] + act;
#pragma unroll
    for (int j = 0; j < 4; ++j) {
        const int pix = base + j;
        if (pix < p.np) {
            p.row_ptr[pix] = off;
            p.cnt[pix] = 0;
            if (llong[j] >= 0) p.long_rows[s_longbase + llong[j]] = pix;
            if (lrank[j] >= 0) {
                if (aoff < p.max_active) p.active_idx[aoff] = pix;
                WorkItem it;
                it.row_begin = off;
                it.n = v[j];
                it.pix = pix;
                it.arow = aoff;
                p.work[s_base[size_class(v[j])] + lrank[j]] = it;
                ++aoff;
            }
            off += v[j];
        }
    }
}

// ---- k_scatter: pairs[row_ptr[pix] + slot] = (input index, value) ----------------------
__global__ void __launch_bounds__(kEvThreads) k_scatter(IngestParams p)
{
    const int64_t base = static_cast<int64_t>(blockIdx.x) * (kEvThreads * kEvUnroll) + threadIdx.x;
    Ev e[kEvUnroll];
#pragma unroll
    for (int u = 0; u < kEvUnroll; ++u) {
        const int64_t i = base + u * kEvThreads;
        e[u].pix = -2;
        if (i < p.n) e[u] = decode_event(p.events, i, p.t0, p.t1, p.width, p.height);
    }
#pragma unroll
    for (int u = 0; u < kEvUnroll; ++u) {
        if (e[u].pix >= 0) {
            const int64_t i = base + u * kEvThreads;
            const int slot = __ldg(&p.row_ptr[e[u].pix]) + atomicAdd(&p.cnt[e[u].pix], 1);
            p.pairs[slot] = (static_cast<uint64_t>(i) << 32) | e[u].val;
        }
    }
}

// ---- row sort: restore input order inside every row (a3, R20) ---------------------------
// Short rows (<= kShortMax events): a block owns kRowPix consecutive pixels, i.e. one
// contiguous span of slots; every element finds its row by binary search over the block's
// row starts and its rank inside the row by counting the elements of the row with a smaller
// input index.  Long rows are listed by k_scan_apply and sorted one per block (bitonic sort
// in shared memory) by k_rowsort_long.
__global__ void __launch_bounds__(256) k_rowsort_short(IngestParams p)
{
    __shared__ int s_rp[kRowPix + 1];
    __shared__ uint64_t s_pair[kRowCap];
    const int p0 = blockIdx.x * kRowPix;
    const int npx = min(kRowPix, p.np - p0);
    for (int i = threadIdx.x; i <= npx; i += blockDim.x) s_rp[i] = p.row_ptr[p0 + i];
    __syncthreads();
    const int beg = s_rp[0], tot = s_rp[npx] - beg;
    if (tot == 0) return;
    const bool staged = tot <= kRowCap;
    if (staged) {
        for (int i = threadIdx.x; i < tot; i += blockDim.x) s_pair[i] = p.pairs[beg + i];
        __syncthreads();
    }
    for (int s = threadIdx.x; s < tot; s += blockDim.x) {
        int lo = 0, hi = npx;                              // row = last r with s_rp[r] - beg <= s
        while (hi - lo > 1) {
            const int mid = (lo + hi) >> 1;
            if (s_rp[mid] - beg <= s) lo = mid; else hi = mid;
        }
        const int rb = s_rp[lo] - beg, re = s_rp[lo + 1] - beg;
        if (re - rb > kShortMax) continue;                 // k_rowsort_long's
        int rank = 0;
        uint64_t mine;
        if (staged) {
            mine = s_pair[s];
            for (int j = rb; j < re; ++j) rank += (s_pair[j] < mine);
        } else {
            mine = p.pairs[beg + s];
            for (int j = rb; j < re; ++j) rank += (p.pairs[beg + j] < mine);
        }
        p.csr_ev[beg + rb + rank] = static_cast<uint32_t>(mine);
    }
}

__global__ void __launch_bounds__(256) k_rowsort_long(IngestParams p)
{
    __shared__ uint64_t s_key[kRowCap];
    const int n_long = *p.n_long;
    for (int r = blockIdx.x; r < n_long; r += gridDim.x) {
        const int pix = p.long_rows[r];
        const int beg = p.row_ptr[pix], n = p.row_ptr[pix + 1] - beg;
        if (n <= kRowCap) {
            int np2 = 1;
            while (np2 < n) np2 <<= 1;
            for (int i = threadIdx.x; i < np2; i += blockDim.x)
                s_key[i] = (i < n) ? p.pairs[beg + i] : ~0ull;
            __syncthreads();
            for (int k = 2; k <= np2; k <<= 1) {
                for (int j = k >> 1; j > 0; j >>= 1) {
                    for (int t = threadIdx.x; t < (np2 >> 1); t += blockDim.x) {
                        const int lo = ((t & ~(j - 1)) << 1) | (t & (j - 1));    // index with bit j clear
                        const int hi = lo | j;
                        const bool asc = (lo & k) == 0;
                        const uint64_t a = s_key[lo], b = s_key[hi];
                        if ((a > b) == asc) { s_key[lo] = b; s_key[hi] = a; }
                    }
                    __syncthreads();
                }
            }
            for (int i = threadIdx.x; i < n; i += blockDim.x)
                p.csr_ev[beg + i] = static_cast<uint32_t>(s_key[i]);
            __syncthreads();
        } else {
            // very long row (thousands of events on one pixel): rank by counting from global memory
            for (int s = threadIdx.x; s < n; s += blockDim.x) {
                const uint64_t mine = p.pairs[beg + s];
                int rank = 0;
                for (int j = 0; j < n; ++j) rank += (p.pairs[beg + j] < mine);
                p.csr_ev[beg + rank] = static_cast<uint32_t>(mine);
            }
        }
    }
}

}  // namespace

int launch_ingest(const IngestParams &p, cudaStream_t st)
{
    const int n_tiles = (p.np + kScanTile - 1) / kScanTile;
    const int ev_blocks = static_cast<int>((p.n + kEvThreads * kEvUnroll - 1) / (kEvThreads * kEvUnroll));
    int launches = 0;
    k_init<<<(p.np + 255) / 256, 256, 0, st>>>(p); ++launches;
    if (ev_blocks > 0) { k_hist<<<ev_blocks, kEvThreads, 0, st>>>(p); ++launches; }
    k_scan_reduce<<<n_tiles, 1024, 0, st>>>(p); ++launches;
    k_scan_tiles<<<1, 1024, 0, st>>>(p, n_tiles); ++launches;
    k_scan_apply<<<n_tiles, 1024, 0, st>>>(p); ++launches;
    if (ev_blocks > 0) {
        k_scatter<<<ev_blocks, kEvThreads, 0, st>>>(p); ++launches;
        k_rowsort_short<<<(p.np + kRowPix - 1) / kRowPix, 256, 0, st>>>(p); ++launches;
        k_rowsort_long<<<kLongBlocks, 256, 0, st>>>(p); ++launches;
    }
    return launches;
}

}  // namespace ddhf
