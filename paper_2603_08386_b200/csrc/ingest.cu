// ingest.cu -- a0-a3: window/sensor filter, per-pixel histogram, exclusive scan + active
// list + size-classed work list, and a STABLE bucketing of the events into CSR form.
//
// "For each window, events are moved to the GPU, sorted by pixel index";
// pixels with fewer than n_min events are discarded (L137).  Readings R19 (half-open
// window, bad coordinates dropped and counted) and R20 (input order inside a row).
//
// The bucketing is a stable two-level sort on the pixel index, pixel = bucket << bL | low,
// at most 1023 buckets, that reads the 16-byte events exactly once:
//
//   k_tile_sort    one CTA per tile of 8192 events: decode, filter, and sort the tile by bucket
//                  in shared memory; the tile goes back to HBM in that order as 4-byte
//                  (low << vb | value) or 8-byte items, with the start of every bucket's run
//                  inside the tile (u16 [tile][bucket]).  Bucket totals by integer atomics; the
//                  last CTA turns them into bucket bases.
//   k_bucket_sort  one CTA per bucket: gathers the bucket's runs from all tiles in tile order
//                  (= input order), sorts them by the low digit in shared memory and writes
//                  csr_ev and the per-pixel counts.  Buckets larger than the CTA's capacity go
//                  through in chunks (two loops over the chunks: count, then place).
//
// Both sorts are least-significant-digit counting sorts of at most 5 bits per sub-pass with
// THREAD-PRIVATE counters: thread t owns K consecutive items and its own column of the
// counter matrix [digit][thread], so counting needs no atomics, no ballots and no match
// instructions, and the rank of an item is a plain exclusive scan of that matrix in
// (digit, thread) order -- input order inside a digit by construction.  No atomic decides any
// position, so csr_ev is bit-reproducible (R20).  The ballot-ranking partition this replaces
// spent 160-185 warp instructions per 32 events and per digit (profiles/r2_ingest_primitives.md);
// a 5-bit sub-pass here costs about 25.
//
// HBM traffic per event: 16 B read, 4 B (8 B when the value does not fit beside the low digit)
// written and read, 4 B written; the run table adds 2 B x buckets per 8192 events.
#include "ddhf_internal.cuh"

namespace ddhf {

namespace {

constexpr int kNT = 512;                       // threads per CTA of both sort kernels
constexpr int kTile = 8192;                    // events per tile of k_tile_sort (16 per thread)
constexpr int kCntStride = kNT + kNT / 32 + 16; // words per counter row: one pad word per 32, and a multiple of 32
                                               // (the bank of a counter depends on the thread only, never on the digit)
constexpr int kCntWords = 16 * kCntStride;     // 32 digits, two 16-bit counters per word
constexpr unsigned kFullMask = 0xffffffffu;

// a bucket with more events than kGiantMin is sorted by several CTAs (see "giant buckets" below)
struct __align__(16) GiantBucket {
    int32_t bucket, tiles_per_chunk, n_chunks, row0;      // row0: first of n_chunks consecutive chunk rows
    int32_t chunk0;                                       // first of the bucket's chunks in the flat numbering
    int32_t done;                                         // chunks sorted so far
    int32_t _pad[2];
};
constexpr int kGiantMin = 4 * 16384;
constexpr int kGiantHelpers = 74;      // extra CTAs of k_bucket_sort (and half as many of k_worklist) for their chunks


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

// A row longer than kSplitMin becomes n_seg work items of seg_len events (the last one shorter); seg_len <= kSegEvents
// unless the row is longer than kMaxSegs * kSegEvents.
__device__ __forceinline__ int row_segments(int n, int &seg_len)
{
    // at most kMaxSegs segments per row: one round of the segment pass on a B200 (148 SMs x 12 warps)
    const int n_seg = (n > kSplitMin) ? min((n + kSegEvents - 1) / kSegEvents, kMaxSegs) : 1;
    seg_len = (n + n_seg - 1) / n_seg;
    return n_seg;
}

// Items a row of n_seg segments adds to the size-classed work list: its segments, unless they go to the
// segment list of their own (lean NDFT kernel followed by the segment pass)
// (nor a long unsplit row that goes to the hot list of the NUFFT path)
__device__ __forceinline__ bool is_hot(const IngestParams &p, int n, int n_seg) { return p.hot_work && n_seg == 1 && n >= p.hot_min; }
__device__ __forceinline__ int class_items(const IngestParams &p, int n, int n_seg)
{
    return ((p.seg_work && n_seg > 1) || is_hot(p, n, n_seg)) ? 0 : n_seg;
}

// ---- k_init: per-pixel maps for inactive pixels, zeroed totals and counters ---------------
__global__ void k_init(IngestParams p)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < p.np) {
        p.sf[i] = __int_as_float(0x7fc00000);   // NaN: pixel not active
        p.score[i] = 0.f;
        p.f0_idx[i] = -1;
        p.mask[i] = 0;
        p.ccl_parent[i] = 0x7fffffff;           // no parent yet
    }
    if (i <= p.nb + 1) {
        p.bkt_total[i] = 0; p.bkt_base[i] = 0; p.bkt_order[i] = i;      // identity order: no tile ran
        p.bkt_maxrun[i] = 64; p.giant_of[i] = -1;
    }
    if (i <= 1024) p.ccl_tile_state[i] = 0;
    if (blockIdx.x == 0) {
        if (threadIdx.x < DDHF_N_COUNTERS) p.counters[threadIdx.x] = 0;
        if (threadIdx.x < kNumClasses) {
            p.class_cnt[threadIdx.x] = 0;
            p.class_cur[threadIdx.x] = 0;
        }
        if (threadIdx.x < 16) p.sync[threadIdx.x] = 0;
        if (threadIdx.x == 0) {
            *p.work_cursor = 0ull;
            if (p.work_cursor2) *p.work_cursor2 = 0ull;
            if (p.hot_cursor) *p.hot_cursor = 0;
        }
    }
}

// ---- the counting-sort sub-pass --------------------------------------------------------------
// Shared-memory positions are padded so that both access patterns are conflict-free: "blocked"
// (thread t reads its K consecutive items) and "striped" (consecutive threads, consecutive items).
template <typename T> __device__ __forceinline__ int pad_pos(int e);
template <> __device__ __forceinline__ int pad_pos<uint32_t>(int e) { return e + (e >> 5); }
template <> __device__ __forceinline__ int pad_pos<uint64_t>(int e) { return e + (e >> 4); }

template <typename T> __device__ __forceinline__ uint32_t digit_of(T it, int shift, uint32_t mask);
template <> __device__ __forceinline__ uint32_t digit_of<uint32_t>(uint32_t it, int shift, uint32_t mask)
{
    return (it >> shift) & mask;
}
template <> __device__ __forceinline__ uint32_t digit_of<uint64_t>(uint64_t it, int shift, uint32_t mask)
{
    return (static_cast<uint32_t>(it >> 32) >> (shift - 32)) & mask;      // every digit sits in the high word
}

// Items it[0..K) of thread t are elements K t .. K t + K - 1 of the current order.  On return
// buf[pad_pos(r)] holds the element of rank r of the order stably sorted by the digit
// (it >> shift) & (2^width - 1), 1 <= width <= 5; the caller synchronises before reading buf.
// cnt: kCntWords words; word (r, t) holds the counters of digits r (low half) and r + R (high half),
// R = 2^(width-1): a packed add scans both halves at once (totals stay below 2^16).
// WC = 5: the width is the compile-time constant 5 (the common case); WC = 0: `width` at run time.
template <int K, typename T, int WC>
__device__ __forceinline__ void sort_subpass(const T (&it)[K], uint32_t *cnt, T *buf, uint32_t *s_warp,
                                             int shift, int width_rt)
{
    const int t = threadIdx.x, lane = t & 31, wid = t >> 5;
    const int width = WC ? WC : width_rt;
    const uint32_t mask = (1u << width) - 1u;
    const int R = 1 << (width - 1);
    const uint32_t rmask = static_cast<uint32_t>(R - 1);
    {
        uint4 *c4 = reinterpret_cast<uint4 *>(cnt);
        const int n4 = R * kCntStride / 4;
        for (int w = t; w < n4; w += kNT) c4[w] = make_uint4(0u, 0u, 0u, 0u);
    }
    __syncthreads();
    // byte offset of the thread's column inside a counter row
    const uint32_t tb4 = static_cast<uint32_t>(t + (t >> 5)) * 4u;
    char *cb = reinterpret_cast<char *>(cnt);
    // two items per round: both counters are read before either is written, so the two shared-memory
    // round trips overlap; when both items hit the same counter the second sees the first's update
#pragma unroll
    for (int i = 0; i < K; i += 2) {
        const uint32_t d0 = digit_of<T>(it[i], shift, mask), d1 = digit_of<T>(it[i + 1], shift, mask);
        uint32_t *c0 = reinterpret_cast<uint32_t *>(cb + (d0 & rmask) * (kCntStride * 4u) + tb4);
        uint32_t *c1 = reinterpret_cast<uint32_t *>(cb + (d1 & rmask) * (kCntStride * 4u) + tb4);
        const uint32_t v0 = *c0, v1 = *c1;
        const uint32_t n0 = v0 + ((d0 >> (width - 1)) * 0xffffu) + 1u;     // +1 in the low or the high half
        *c0 = n0;                                                          // the thread's own column: no other
        *c1 = ((c0 == c1) ? n0 : v1) + ((d1 >> (width - 1)) * 0xffffu) + 1u;   // thread touches it
    }
    __syncthreads();
    // exclusive scan of the matrix in (digit, thread) order: thread j rakes words [R j, R j + R)
    {
        const int w0 = R * t;
        uint32_t *cp = cnt + w0 + (w0 >> 5) + 16 * (w0 >> 9);   // R <= 16: the R words share one pad offset
        uint32_t run = 0;
#pragma unroll
        for (int i = 0; i < 16; ++i)
            if (i < R) run += cp[i];
        uint32_t inc = run;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const uint32_t x = __shfl_up_sync(kFullMask, inc, o);
            if (lane >= o) inc += x;
        }
        if (lane == 31) s_warp[wid] = inc;
        __syncthreads();
        uint32_t ws = (lane < kNT / 32) ? s_warp[lane] : 0u;
#pragma unroll
        for (int o = 1; o < kNT / 32; o <<= 1) {
            const uint32_t x = __shfl_up_sync(kFullMask, ws, o);
            if (lane >= o) ws += x;
        }
        const uint32_t grand = __shfl_sync(kFullMask, ws, kNT / 32 - 1);
        uint32_t wex = __shfl_sync(kFullMask, ws, (wid + 31) & 31);
        if (wid == 0) wex = 0u;
        // every high-half digit ranks after all low-half digits
        uint32_t ex = inc - run + wex + (grand << 16);
#pragma unroll
        for (int i = 0; i < 16; ++i)
            if (i < R) { const uint32_t c = cp[i]; cp[i] = ex; ex += c; }
    }
    __syncthreads();
#pragma unroll
    for (int i = 0; i < K; i += 2) {
        const uint32_t d0 = digit_of<T>(it[i], shift, mask), d1 = digit_of<T>(it[i + 1], shift, mask);
        const uint32_t h0 = d0 >> (width - 1), h1 = d1 >> (width - 1);
        uint32_t *c0 = reinterpret_cast<uint32_t *>(cb + (d0 & rmask) * (kCntStride * 4u) + tb4);
        uint32_t *c1 = reinterpret_cast<uint32_t *>(cb + (d1 & rmask) * (kCntStride * 4u) + tb4);
        const uint32_t v0 = *c0, v1 = *c1;
        const uint32_t n0 = v0 + (h0 * 0xffffu) + 1u;
        const uint32_t o1 = (c0 == c1) ? n0 : v1;
        *c0 = n0;
        *c1 = o1 + (h1 * 0xffffu) + 1u;
        buf[pad_pos<T>(static_cast<int>((v0 >> (h0 * 16u)) & 0xffffu))] = it[i];
        buf[pad_pos<T>(static_cast<int>((o1 >> (h1 * 16u)) & 0xffffu))] = it[i + 1];
    }
}

// sub-passes of a `bits`-bit digit: 5 bits each, the remainder last
__device__ __forceinline__ int subpass_count(int bits) { return (bits + 4) / 5; }

// Sort the K x kNT items of buf (blocked, padded) by the `bits`-bit digit at `shift`; on return
// it[] holds the thread's K items of the sorted order and buf the whole sorted order.
template <int K, typename T>
__device__ __forceinline__ void sort_items(T (&it)[K], uint32_t *cnt, T *buf, uint32_t *s_warp, int shift, int bits)
{
    const int t = threadIdx.x;
    int sh = shift, left = bits;
    while (left > 0) {
        if (left >= 5) sort_subpass<K, T, 5>(it, cnt, buf, s_warp, sh, 5);
        else sort_subpass<K, T, 0>(it, cnt, buf, s_warp, sh, left);
        sh += 5;
        left -= 5;
        __syncthreads();
#pragma unroll
        for (int i = 0; i < K; ++i) it[i] = buf[pad_pos<T>(K * t + i)];
    }
}

// ---- block-wide helpers (kNT threads) --------------------------------------------------------------
// exclusive prefix sum of one value per thread; `total` = sum over the block.  Two barriers.
__device__ __forceinline__ int block_excl_sum(int v, int &total, uint32_t *s_warp)
{
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    int inc = v;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const int x = __shfl_up_sync(kFullMask, inc, o);
        if (lane >= o) inc += x;
    }
    __syncthreads();                                   // earlier readers of s_warp are done
    if (lane == 31) s_warp[wid] = static_cast<uint32_t>(inc);
    __syncthreads();
    int ws = (lane < kNT / 32) ? static_cast<int>(s_warp[lane]) : 0;
#pragma unroll
    for (int o = 1; o < kNT / 32; o <<= 1) {
        const int x = __shfl_up_sync(kFullMask, ws, o);
        if (lane >= o) ws += x;
    }
    total = __shfl_sync(kFullMask, ws, kNT / 32 - 1);
    int wex = __shfl_sync(kFullMask, ws, (wid + 31) & 31);
    if (wid == 0) wex = 0;
    return inc - v + wex;
}

// r[0 .. n) holds the first position of every digit that occurs and 0xffffffff elsewhere; on return
// r[d] = first position of the first digit >= d that occurs, `end` if there is none (the start of every
// digit's run, empty runs included).  Thread t owns PER consecutive entries; n <= PER * kNT.
template <int PER>
__device__ __forceinline__ void fill_run_starts(uint32_t *r, int n, uint32_t end, uint32_t *s_warp)
{
    const int t = threadIdx.x, lane = t & 31, wid = t >> 5;
    uint32_t v[PER];
    uint32_t m = 0xffffffffu;
#pragma unroll
    for (int k = 0; k < PER; ++k) {
        const int i = t * PER + k;
        v[k] = (i < n) ? r[i] : 0xffffffffu;
        m = min(m, v[k]);
    }
    // suffix minimum over the threads after this one
    uint32_t suf = m;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const uint32_t x = __shfl_down_sync(kFullMask, suf, o);
        if (lane + o < 32) suf = min(suf, x);
    }
    __syncthreads();
    if (lane == 0) s_warp[wid] = suf;                  // minimum of the whole warp
    __syncthreads();
    uint32_t carry = end;
    for (int w = wid + 1; w < kNT / 32; ++w) carry = min(carry, s_warp[w]);
    const uint32_t nxt = __shfl_down_sync(kFullMask, suf, 1);
    if (lane < 31) carry = min(carry, nxt);            // threads after this one in the warp
#pragma unroll
    for (int k = PER - 1; k >= 0; --k) {
        const int i = t * PER + k;
        carry = min(carry, v[k]);
        if (i < n) r[i] = carry;
    }
    __syncthreads();
}

// ---- the last CTA of k_tile_sort: bucket bases, event counts, bucket order -----------------------------
// order[] lists the buckets by descending size class (32 classes of the largest total), so that
// k_bucket_sort, whose CTAs start in index order, takes the expensive buckets first.
__device__ __forceinline__ void finish_buckets(const IngestParams &p, uint32_t *cnt, uint32_t *buf32, uint32_t *s_warp)
{
    const int t = threadIdx.x, lane = t & 31;
    const uint32_t nb = static_cast<uint32_t>(p.nb);
    const uint32_t b0 = 2u * t;                                    // nb + 1 <= 1024 = 2 kNT
    const int v0 = (b0 < nb) ? __ldcg(p.bkt_total + b0) : 0;
    const int v1 = (b0 + 1 < nb) ? __ldcg(p.bkt_total + b0 + 1) : 0;
    int grand;
    const int ex = block_excl_sum(v0 + v1, grand, s_warp);
    if (b0 <= nb) p.bkt_base[b0] = ex;
    if (b0 + 1 <= nb) p.bkt_base[b0 + 1] = ex + v0;
    if (t == 0) {
        p.counters[DDHF_CNT_N_IN] = grand;
        p.counters[DDHF_CNT_N_DROPPED] = static_cast<int32_t>(p.n - grand);
    }
    // giant buckets: cut into chunks of whole tiles that fit one chunk each (not on the sliding-window path,
    // whose slab is small; a bucket that finds no room in the giant rows stays on the one-CTA path)
    if (!p.prev_csr) {
        GiantBucket *tab = reinterpret_cast<GiantBucket *>(p.giant_tab);
        const int n_tiles = static_cast<int>((p.n + kTile - 1) / kTile);
        const int cap = p.compact ? 16384 : 8192;
#pragma unroll
        for (int q = 0; q < 2; ++q) {
            const uint32_t b = b0 + q;
            const int m = q ? v1 : v0;
            if (b < nb && m > kGiantMin) {
                const int tr = max(1, cap / max(__ldcg(p.bkt_maxrun + b), 1));
                const int n_chunks = (n_tiles + tr - 1) / tr;
                const int row0 = atomicAdd(p.sync + 14, n_chunks);
                if (row0 + n_chunks <= p.giant_rows) {
                    const int g = atomicAdd(p.sync + 10, 1);
                    GiantBucket gb;
                    gb.bucket = static_cast<int32_t>(b); gb.tiles_per_chunk = tr; gb.n_chunks = n_chunks;
                    gb.row0 = p.giant_row0 + row0; gb.chunk0 = atomicAdd(p.sync + 11, n_chunks); gb.done = 0;
                    gb._pad[0] = 0; gb._pad[1] = 0;
                    tab[g] = gb;
                    p.giant_of[b] = g;
                }
            }
        }
    }
    int mx = __reduce_max_sync(kFullMask, max(v0, v1));
    __syncthreads();
    if (lane == 0) s_warp[t >> 5] = static_cast<uint32_t>(mx);
    __syncthreads();
    mx = 0;
    for (int w = 0; w < kNT / 32; ++w) mx = max(mx, static_cast<int>(s_warp[w]));
    const int shift = max(0, 27 - __clz(mx | 1));                 // mx >> shift < 32
    uint32_t it[2];
    it[0] = ((31u - (static_cast<uint32_t>(v0) >> shift)) << 16) | b0;
    it[1] = ((31u - (static_cast<uint32_t>(v1) >> shift)) << 16) | (b0 + 1u);
    __syncthreads();
    sort_subpass<2, uint32_t, 5>(it, cnt, buf32, s_warp, 16, 5);
    __syncthreads();
    if (t == 0) p.counters[DDHF_CNT_N_GIANT] = *reinterpret_cast<volatile int32_t *>(p.sync + 10);
    // (the list entries of giant buckets are marked: their CTAs of k_bucket_sort leave at once)
    for (uint32_t r = t; r < nb; r += kNT) {
        const uint32_t b = buf32[pad_pos<uint32_t>(static_cast<int>(r))] & 0xffffu;
        p.bkt_order[r] = static_cast<int32_t>(b | (__ldcg(p.giant_of + b) >= 0 ? 0x80000000u : 0u));
    }
}

// ---- k_tile_sort: decode + filter one tile, sort it by bucket, publish its runs -----------------
// Only a 32-bit key (bucket << 13 | position in the tile) goes through the sort; dropped events and
// the padding of the last tile carry the sentinel bucket nb and sort to the end of the tile.  The
// payloads stay where the decode put them and are fetched by position at the end.  A tile goes back to HBM
// with every bucket's run starting on a 16-byte boundary (k_bucket_sort gathers with 128-bit loads);
// run table entry = first item of the run inside the tile's slot | length << 16.
template <bool COMPACT> struct BucketItem { typedef uint32_t type; };
template <> struct BucketItem<false> { typedef uint64_t type; };

template <bool COMPACT> struct TileOut {
    static constexpr int kAlign = COMPACT ? 4 : 2;                      // items per 16 bytes
    static constexpr int kStride = kTile + (COMPACT ? 3 : 1) * 1024;     // items per tile slot (padding included)
};

// Decode one event: sort key = bucket << 13 | position in the tile (the sentinel bucket nb for dropped
// events and for the padding of the last tile); payload = the item k_bucket_sort will read.
template <bool FULL, bool COMPACT, bool PACKED>
__device__ __forceinline__ uint32_t load_event(const IngestParams &p, int64_t idx, uint32_t e, uint32_t nb, uint32_t lmask,
                                               uint32_t window, typename BucketItem<COMPACT>::type &pay)
{
    typedef typename BucketItem<COMPACT>::type TO;
    uint32_t bucket = nb;
    pay = 0;
    if (FULL || idx < p.n) {
        uint32_t x, y, pos;
        uint64_t dt;                                                       // t - t0; window < 2^31: in range iff dt < window
        if (PACKED) {
            const uint2 w = __ldg(reinterpret_cast<const uint2 *>(p.events) + idx);
            x = w.x & 0xffffu;
            y = (w.x >> 16) & 0x7fffu;
            pos = w.x >> 31;
            dt = static_cast<uint64_t>(p.t_base - p.t0) + w.y;
        } else {
            const int4 w = __ldg(reinterpret_cast<const int4 *>(p.events) + idx);
            x = static_cast<uint32_t>(w.x) & 0xffffu;
            y = static_cast<uint32_t>(w.x) >> 16;
            const uint64_t t = (static_cast<uint64_t>(static_cast<uint32_t>(w.w)) << 32) | static_cast<uint32_t>(w.z);
            dt = t - static_cast<uint64_t>(p.t0);
            pos = (static_cast<int32_t>(static_cast<uint32_t>(w.y) << 16) > 0) ? 1u : 0u;    // int16 p > 0
        }
        const bool ok = (dt < window) && (x < static_cast<uint32_t>(p.width)) && (y < static_cast<uint32_t>(p.height));
        const uint32_t px = y * static_cast<uint32_t>(p.width) + x;
        const uint32_t val = (static_cast<uint32_t>(dt) << 1) | pos;
        if (ok) bucket = px >> p.bl;
        if (COMPACT) pay = static_cast<TO>(((px & lmask) << p.vb) | val);
        else pay = static_cast<TO>((static_cast<uint64_t>(px & lmask) << 32) | val);
    }
    return (bucket << 13) | e;
}

template <bool COMPACT, bool PACKED>
__global__ void __launch_bounds__(kNT, 2) k_tile_sort(IngestParams p)
{
    typedef typename BucketItem<COMPACT>::type TO;
    extern __shared__ __align__(16) uint32_t s_raw[];
    __shared__ uint32_t s_warp[kNT / 32];
    __shared__ bool s_last;
    constexpr int K = kTile / kNT;
    // only the 32-bit keys go through the sort; the payloads stay where the decode put them
    uint32_t *keys = s_raw;                                                      // pad_pos(kTile) keys
    uint32_t *cnt = s_raw + (kTile + kTile / 32);
    uint32_t *rstart = cnt + kCntWords;                                          // [1032]
    TO *pay = reinterpret_cast<TO *>(rstart + 1032);                             // [kTile]
    const int t = threadIdx.x;
    const int tile = blockIdx.x;
    const int64_t tile_beg = static_cast<int64_t>(tile) * kTile;
    const uint32_t nb = static_cast<uint32_t>(p.nb);
    const uint32_t lmask = (1u << p.bl) - 1u;
    const uint32_t window = static_cast<uint32_t>(p.t1 - p.t0);

    // coalesced load and decode
    if (tile_beg + kTile <= p.n) {
#pragma unroll 8
        for (int i = 0; i < K; ++i) {
            const uint32_t e = static_cast<uint32_t>(t + kNT * i);
            TO py;
            keys[pad_pos<uint32_t>(e)] = load_event<true, COMPACT, PACKED>(p, tile_beg + e, e, nb, lmask, window, py);
            pay[e] = py;
        }
    } else {
#pragma unroll 4
        for (int i = 0; i < K; ++i) {
            const uint32_t e = static_cast<uint32_t>(t + kNT * i);
            TO py;
            keys[pad_pos<uint32_t>(e)] = load_event<false, COMPACT, PACKED>(p, tile_beg + e, e, nb, lmask, window, py);
            pay[e] = py;
        }
    }
    for (int b = t; b < 1026; b += kNT) rstart[b] = 0xffffffffu;
    __syncthreads();
    uint32_t it[K];                                    // thread t owns 16 consecutive events
#pragma unroll
    for (int i = 0; i < K; ++i) it[i] = keys[pad_pos<uint32_t>(K * t + i)];
    sort_items<K, uint32_t>(it, cnt, keys, s_warp, 13, p.hbits);

    // start of every bucket's run inside the sorted tile
    {
        uint32_t prev = 0xffffffffu;
        if (t > 0) prev = keys[pad_pos<uint32_t>(K * t - 1)] >> 13;
#pragma unroll
        for (int i = 0; i < K; ++i) {
            const uint32_t d = it[i] >> 13;
            if (d != prev) rstart[d] = static_cast<uint32_t>(K * t + i);
            prev = d;
        }
    }
    __syncthreads();
    fill_run_starts<2>(rstart, static_cast<int>(nb) + 1, kTile, s_warp);        // rstart[0 .. nb]; nb = the sentinel's run
    // run lengths, aligned starts in the tile's output slot, bucket totals
    uint32_t *delta = cnt;                                                       // [nb] output position - sorted position
    {
        const uint32_t b0 = 2u * t;
        uint32_t len[2], alen[2];
#pragma unroll
        for (int q = 0; q < 2; ++q) {
            const uint32_t b = b0 + q;
            len[q] = (b < nb) ? rstart[b + 1] - rstart[b] : 0u;
            alen[q] = (len[q] + TileOut<COMPACT>::kAlign - 1) & ~static_cast<uint32_t>(TileOut<COMPACT>::kAlign - 1);
        }
        int tot;
        uint32_t a = static_cast<uint32_t>(block_excl_sum(static_cast<int>(alen[0] + alen[1]), tot, s_warp));
        uint32_t *row = p.run_tab + static_cast<size_t>(tile) * nb;
#pragma unroll
        for (int q = 0; q < 2; ++q) {
            const uint32_t b = b0 + q;
            if (b < nb) {
                row[b] = a | (len[q] << 16);
                delta[b] = a - rstart[b];
                if (len[q]) {
                    atomicAdd(&p.bkt_total[b], static_cast<int>(len[q]));
                    if (len[q] > 64) atomicMax(&p.bkt_maxrun[b], static_cast<int>(len[q]));      // only giant buckets need it
                }
                a += alen[q];
            }
        }
    }
    __syncthreads();
    const int kept = static_cast<int>(rstart[nb]);
    {
        TO *out = reinterpret_cast<TO *>(p.items) + static_cast<size_t>(tile) * TileOut<COMPACT>::kStride;
#pragma unroll
        for (int i = 0; i < K; ++i) {
            const int r = t + kNT * i;
            if (r < kept) {
                const uint32_t key = keys[pad_pos<uint32_t>(r)];
                out[static_cast<uint32_t>(r) + delta[key >> 13]] = pay[key & 8191u];
            }
        }
    }
    // the last CTA to finish turns the bucket totals into bases, publishes the event counts and
    // orders the buckets by descending size class (k_bucket_sort takes them in that order)
    __threadfence();
    __syncthreads();
    if (t == 0) s_last = (atomicAdd(p.sync + 0, 1) == static_cast<int>(gridDim.x) - 1);
    __syncthreads();
    if (!s_last) return;
    __threadfence();
    finish_buckets(p, cnt, keys, s_warp);
}

// ---- k_bucket_sort: gather one bucket from all tiles, sort it by the low digit, write the rows -------
// Items: COMPACT  uint32  low << vb | value   (value < 2^vb, vb = 32 - bL)
//        else     uint64  low << 32 | value
// The padding of a partly filled chunk is all ones: it sorts behind every real item in every sub-pass
// (it also comes last in input order), so positions [0, fill) of the sorted chunk are the real items.

template <bool COMPACT>
struct BucketCfg {
    typedef typename BucketItem<COMPACT>::type T;
    static constexpr int kMaxK = COMPACT ? 32 : 16;
    static constexpr int kCap = kMaxK * kNT;                       // items per chunk
    static constexpr int kBufWords = COMPACT ? (kCap + kCap / 32) : 2 * (kCap + kCap / 16);
    // words: buf | cnt | rstart [2^bL + 1] | pixtot [2^bL]
    static size_t smem_bytes(int bl) { return 4u * (static_cast<size_t>(kBufWords) + kCntWords + 2u * (1u << bl) + 8u); }
    __device__ static __forceinline__ uint32_t low_of(T it, int vb)
    {
        if (COMPACT) return static_cast<uint32_t>(it) >> vb;
        return static_cast<uint32_t>(static_cast<uint64_t>(it) >> 32);
    }
    __device__ static __forceinline__ uint32_t val_of(T it, int vb)
    {
        if (COMPACT) return static_cast<uint32_t>(it) & ((1u << vb) - 1u);
        return static_cast<uint32_t>(it);
    }
};

// Sort the first `fill` items of buf (input order, padded positions) by the low digit; returns with
// rstart[l] = first sorted position of pixel l of the bucket (l = 0 .. 2^bL, rstart[2^bL] = fill) and
// buf = the sorted chunk.
template <int K, bool COMPACT>
__device__ __noinline__ void sort_chunk(typename BucketItem<COMPACT>::type *buf, uint32_t *cnt, uint32_t *rstart,
                                        uint32_t *s_warp, int fill, int bl, int vb)
{
    typedef typename BucketItem<COMPACT>::type T;
    const int t = threadIdx.x;
    const int nl = 1 << bl;
    for (int l = t; l <= nl; l += kNT) rstart[l] = 0xffffffffu;
    T it[K];
#pragma unroll
    for (int i = 0; i < K; ++i) {
        const int e = K * t + i;
        it[i] = (e < fill) ? buf[pad_pos<T>(e)] : static_cast<T>(~static_cast<T>(0));
    }
    sort_items<K, T>(it, cnt, buf, s_warp, COMPACT ? vb : 32, bl);
    uint32_t prev = 0xffffffffu;
    if (t > 0) prev = BucketCfg<COMPACT>::low_of(buf[pad_pos<T>(K * t - 1)], vb);
#pragma unroll
    for (int i = 0; i < K; ++i) {
        const uint32_t d = BucketCfg<COMPACT>::low_of(it[i], vb);
        if (K * t + i < fill && d != prev) rstart[d] = static_cast<uint32_t>(K * t + i);
        prev = d;
    }
    __syncthreads();
    if (nl <= kNT) fill_run_starts<1>(rstart, nl, static_cast<uint32_t>(fill), s_warp);
    else if (nl <= 2 * kNT) fill_run_starts<2>(rstart, nl, static_cast<uint32_t>(fill), s_warp);
    else fill_run_starts<8>(rstart, nl, static_cast<uint32_t>(fill), s_warp);
    if (t == 0) rstart[nl] = static_cast<uint32_t>(fill);
    __syncthreads();
}

template <bool COMPACT>
__device__ __forceinline__ void sort_chunk_any(typename BucketItem<COMPACT>::type *buf, uint32_t *cnt, uint32_t *rstart,
                                               uint32_t *s_warp, int fill, int bl, int vb)
{
    const int k = (fill + kNT - 1) / kNT;                      // items per thread needed
    if (k <= 8) sort_chunk<8, COMPACT>(buf, cnt, rstart, s_warp, fill, bl, vb);
    else if (k <= 12) sort_chunk<12, COMPACT>(buf, cnt, rstart, s_warp, fill, bl, vb);
    else if (!COMPACT || k <= 16) sort_chunk<16, COMPACT>(buf, cnt, rstart, s_warp, fill, bl, vb);
    else if (k <= 20) sort_chunk<COMPACT ? 20 : 16, COMPACT>(buf, cnt, rstart, s_warp, fill, bl, vb);
    else if (k <= 24) sort_chunk<COMPACT ? 24 : 16, COMPACT>(buf, cnt, rstart, s_warp, fill, bl, vb);
    else if (k <= 28) sort_chunk<COMPACT ? 28 : 16, COMPACT>(buf, cnt, rstart, s_warp, fill, bl, vb);
    else sort_chunk<BucketCfg<COMPACT>::kMaxK, COMPACT>(buf, cnt, rstart, s_warp, fill, bl, vb);
}

// One row of the chunk table of a bucket that does not fit one chunk: header {previous row of the
// bucket (-1: none), offset of the chunk inside the bucket, items, 0} followed by 2^bL per-pixel words
// delta[l] = (events of pixel l in earlier chunks) - (first sorted position of pixel l in this chunk).
constexpr int kRowHdr = 4;
constexpr int kLongRun = 256;      // runs longer than this are gathered by the whole CTA

// Bucket b, tiles [tile_lo, tile_hi).  giant_row < 0: the whole bucket (every tile), as described above.
// giant_row >= 0: one chunk of a giant bucket (a tile range that fits one chunk by construction; giant_off = the
// bucket's events in earlier tiles): sort it, leave the sorted chunk in the workspace and its per-pixel counts in
// chunk row giant_row; giant_finish() and the placement CTAs of k_worklist do the rest.
template <bool COMPACT>
__device__ __forceinline__ void bucket_body(const IngestParams &p, uint32_t *s_raw, int b, int tile_lo, int tile_hi,
                                            int giant_row, int giant_off)
{
    typedef BucketCfg<COMPACT> C;
    typedef typename C::T T;
    __shared__ uint32_t s_warp[kNT / 32];
    __shared__ int s_cut, s_row;
    T *buf = reinterpret_cast<T *>(s_raw);
    uint32_t *cnt = s_raw + C::kBufWords;
    uint32_t *rstart = cnt + kCntWords;                       // [nl + 1]
    const int bl = p.bl, vb = p.vb, nl = 1 << bl;
    uint32_t *pixtot = rstart + nl + 4;                        // [nl]
    const int t = threadIdx.x;
    const bool giant = giant_row >= 0;
    const int m = p.bkt_total[b];
    const int gbase = p.bkt_base[b];
    const int pix0 = b << bl;
    __shared__ int s_act, s_class[kNumClasses];           // active pixels / work items per class of this bucket
    __syncthreads();                                      // (a helper CTA comes back here chunk after chunk)
    if (t == 0) { s_act = 0; if (!giant) p.bkt_act[b] = 0; }
    if (t < kNumClasses) s_class[t] = 0;
    if (m == 0) {
        for (int l = t; l < nl; l += kNT)
            if (pix0 + l < p.np) {
                p.cnt[pix0 + l] = 0;
                if (p.slab_row_ptr) p.slab_row_ptr[pix0 + l] = gbase;
            }
        return;
    }
    // (not on the sliding-window path: its counts are completed later and go through the scan kernels)
    const int nmin = p.prev_csr ? 0x7fffffff : max(p.n_min, 1);
    // a pixel's row length is known: count it for the active list and the work-list classes (k_worklist)
    auto tally = [&](int n) {
        if (n >= nmin) {
            int seg_len;
            const int n_seg = row_segments(n, seg_len);
            atomicAdd(&s_act, 1);
            if (class_items(p, n, n_seg)) atomicAdd(&s_class[size_class(seg_len)], class_items(p, n, n_seg));
        }
    };
    auto publish_tally = [&]() {
        __syncthreads();
        if (t == 0) p.bkt_act[b] = s_act;
        if (t < kNumClasses && s_class[t]) atomicAdd(&p.class_cnt[t], s_class[t]);
    };
    const bool single = !giant && m <= C::kCap;
    if (!single)
        for (int l = t; l < nl; l += kNT) pixtot[l] = 0u;
    const uint4 *items = reinterpret_cast<const uint4 *>(p.items);         // runs start on 16-byte boundaries
    constexpr int kPer16 = TileOut<COMPACT>::kAlign;                        // items per 128-bit load
    T *scratch = reinterpret_cast<T *>(p.scratch);
    const int row_words = kRowHdr + 2 * nl;
    int fill = 0;            // items gathered for the chunk being formed
    int chunk_off = giant ? giant_off : 0;       // offset of that chunk inside the bucket
    int last_row = -1;

    // Emit the chunk in buf[0, fill): the only chunk of the bucket -> csr_ev and counts; else loop 1.
    auto flush = [&]() {
        __syncthreads();
        sort_chunk_any<COMPACT>(buf, cnt, rstart, s_warp, fill, bl, vb);
        if (single) {
            for (int l = t; l < nl; l += kNT)
                if (pix0 + l < p.np) {
                    p.cnt[pix0 + l] = static_cast<int32_t>(rstart[l + 1] - rstart[l]);
                    if (p.slab_row_ptr) p.slab_row_ptr[pix0 + l] = gbase + static_cast<int32_t>(rstart[l]);
                    tally(static_cast<int>(rstart[l + 1] - rstart[l]));
                }
            for (int r = t; r < fill; r += kNT) p.csr_ev[gbase + r] = C::val_of(buf[pad_pos<T>(r)], vb);
        } else if (giant) {
            int32_t *rw = p.chunk_rows + static_cast<size_t>(giant_row) * row_words;
            if (t == 0) { rw[0] = -1; rw[1] = chunk_off; rw[2] = fill; rw[3] = 0; }
            for (int l = t; l < nl; l += kNT) rw[kRowHdr + l] = static_cast<int32_t>(rstart[l + 1] - rstart[l]);
            for (int r = t; r < fill; r += kNT) scratch[static_cast<size_t>(gbase) + chunk_off + r] = buf[pad_pos<T>(r)];
        } else {
            if (t == 0) s_row = atomicAdd(p.sync + 1, 1);
            __syncthreads();
            const int row = s_row;
            int32_t *rw = p.chunk_rows + static_cast<size_t>(row) * row_words;
            if (t == 0) { rw[0] = last_row; rw[1] = chunk_off; rw[2] = fill; rw[3] = 0; }
            for (int l = t; l < nl; l += kNT) {
                const uint32_t before = pixtot[l];
                rw[kRowHdr + l] = static_cast<int32_t>(before) - static_cast<int32_t>(rstart[l]);
                pixtot[l] = before + (rstart[l + 1] - rstart[l]);
            }
            for (int r = t; r < fill; r += kNT) scratch[static_cast<size_t>(gbase) + chunk_off + r] = buf[pad_pos<T>(r)];
            last_row = row;
        }
        __syncthreads();
        chunk_off += fill;
        fill = 0;
    };

    // runs of this bucket, 2 kNT tiles at a time, in tile order = input order
    for (int tb = tile_lo; tb < tile_hi; tb += 2 * kNT) {
        int src[2], len[2];
#pragma unroll
        for (int q = 0; q < 2; ++q) {
            const int j = tb + 2 * t + q;
            src[q] = 0; len[q] = 0;
            if (j < tile_hi) {
                const uint32_t e = __ldg(p.run_tab + static_cast<size_t>(j) * p.nb + b);
                src[q] = static_cast<int>(e & 0xffffu); len[q] = static_cast<int>(e >> 16);
            }
        }
        int total;
        int off[2];
        off[0] = block_excl_sum(len[0] + len[1], total, s_warp);
        off[1] = off[0] + len[0];
        int base_off = 0;                                  // runs before this offset are already emitted
        while (true) {
            // cut: the first run that does not fit the chunk any more
            const int room = C::kCap - fill;
            int cut = total;
            if (total - base_off > room) {
                __syncthreads();
                if (t == 0) s_cut = total;
                __syncthreads();
                int cand = total;
#pragma unroll
                for (int q = 1; q >= 0; --q)
                    if (len[q] > 0 && off[q] >= base_off && off[q] + len[q] - base_off > room) cand = off[q];
                if (cand < total) atomicMin(&s_cut, cand);
                __syncthreads();
                cut = s_cut;
            }
            // short runs: one thread each; long runs (a hot pixel fills most of a tile) are queued in the
            // counter array, idle during the gather, and copied by the whole CTA
            uint32_t *lq = cnt;                                   // [0] = queued runs, then {src / 16 B, dst, len}
            if (t == 0) lq[0] = 0u;
            __syncthreads();
#pragma unroll
            for (int q = 0; q < 2; ++q) {
                if (len[q] > 0 && off[q] >= base_off && off[q] < cut) {
                    const int j = tb + 2 * t + q;
                    const size_t s16 = (static_cast<size_t>(j) * TileOut<COMPACT>::kStride + src[q]) / kPer16;
                    const int dst = fill + off[q] - base_off;
                    if (len[q] > kLongRun) {
                        const uint32_t e = atomicAdd(&lq[0], 1u);
                        lq[1 + 4 * e] = static_cast<uint32_t>(s16);
                        lq[2 + 4 * e] = static_cast<uint32_t>(s16 >> 32);
                        lq[3 + 4 * e] = static_cast<uint32_t>(dst);
                        lq[4 + 4 * e] = static_cast<uint32_t>(len[q]);
                        continue;
                    }
                    const uint4 *s = items + s16;
                    for (int i = 0; i < len[q]; i += 2 * kPer16) {     // two independent 128-bit loads per round
                        const uint4 v0 = __ldg(s + i / kPer16);
                        uint4 v1 = make_uint4(0u, 0u, 0u, 0u);
                        if (i + kPer16 < len[q]) v1 = __ldg(s + i / kPer16 + 1);
                        if (COMPACT) {
                            const uint32_t w[8] = {v0.x, v0.y, v0.z, v0.w, v1.x, v1.y, v1.z, v1.w};
#pragma unroll
                            for (int u = 0; u < 8; ++u)
                                if (i + u < len[q]) buf[pad_pos<T>(dst + i + u)] = static_cast<T>(w[u]);
                        } else {
                            const uint64_t w[4] = {(static_cast<uint64_t>(v0.y) << 32) | v0.x, (static_cast<uint64_t>(v0.w) << 32) | v0.z,
                                                   (static_cast<uint64_t>(v1.y) << 32) | v1.x, (static_cast<uint64_t>(v1.w) << 32) | v1.z};
#pragma unroll
                            for (int u = 0; u < 4; ++u)
                                if (i + u < len[q]) buf[pad_pos<T>(dst + i + u)] = static_cast<T>(w[u]);
                        }
                    }
                }
            }
            __syncthreads();
            {
                const int n_long = static_cast<int>(lq[0]);
                const T *items_t = reinterpret_cast<const T *>(p.items);
                for (int e = 0; e < n_long; ++e) {
                    const size_t s16 = (static_cast<size_t>(lq[2 + 4 * e]) << 32) | lq[1 + 4 * e];
                    const int dst = static_cast<int>(lq[3 + 4 * e]), ln = static_cast<int>(lq[4 + 4 * e]);
                    const T *s = items_t + s16 * kPer16;
                    for (int i = t; i < ln; i += kNT) buf[pad_pos<T>(dst + i)] = __ldg(s + i);
                }
            }
            fill += cut - base_off;
            if (cut == total) break;
            flush();
            base_off = cut;
        }
    }
    flush();
    if (single) { publish_tally(); return; }
    if (giant) return;

    // loop 2: row starts of the bucket's pixels, then every chunk goes to its place
    {
        const int per = (nl + kNT - 1) / kNT;                // <= 8 (bL <= 12)
        uint32_t v[8];
        uint32_t sum = 0;
#pragma unroll
        for (int k = 0; k < 8; ++k) {
            const int l = t * per + k;
            v[k] = (k < per && l < nl) ? pixtot[l] : 0u;
            sum += v[k];
        }
        int tot;
        uint32_t ex = static_cast<uint32_t>(block_excl_sum(static_cast<int>(sum), tot, s_warp));
#pragma unroll
        for (int k = 0; k < 8; ++k) {
            const int l = t * per + k;
            if (k < per && l < nl) {
                if (pix0 + l < p.np) {
                    p.cnt[pix0 + l] = static_cast<int32_t>(v[k]);
                    if (p.slab_row_ptr) p.slab_row_ptr[pix0 + l] = gbase + static_cast<int32_t>(ex);
                    tally(static_cast<int>(v[k]));
                }
                rstart[l] = ex;                              // row start of pixel l inside the bucket
                ex += v[k];
            }
        }
        __syncthreads();
    }
    int32_t *delta = reinterpret_cast<int32_t *>(pixtot);    // the chunk's delta row, staged
    for (int row = last_row; row >= 0;) {
        const int32_t *rw = p.chunk_rows + static_cast<size_t>(row) * row_words;
        const int prev_row = rw[0], coff = rw[1], cfill = rw[2];
        __syncthreads();
        for (int l = t; l < nl; l += kNT) delta[l] = rw[kRowHdr + l] + static_cast<int32_t>(rstart[l]);
        __syncthreads();
        for (int r = t; r < cfill; r += kNT) {
            const T item = scratch[static_cast<size_t>(gbase) + coff + r];
            const uint32_t l = C::low_of(item, vb);
            p.csr_ev[gbase + delta[l] + r] = C::val_of(item, vb);
        }
        row = prev_row;
    }
    publish_tally();
}

// ---- giant buckets ------------------------------------------------------------------------------------------
// A bucket of more than kGiantMin events (a stuck pixel puts all of its events into one bucket) would keep one CTA
// busy chunk after chunk.  The last CTA of k_tile_sort lists such buckets (giant_tab) and cuts each into chunks of
// TR consecutive tiles, TR = capacity / (the bucket's longest run in a tile), so that every chunk fits; helper CTAs of
// k_bucket_sort sort the chunks (bucket_body in giant mode), the helper that finishes a bucket's last chunk turns the
// per-chunk counts into row starts and per-chunk bases (giant_finish), and helper CTAs of k_worklist move the sorted
// chunks to their places.  Everything is a function of the data alone: same bits as the one-CTA path.
// chunk row of a giant bucket: header {-, offset in the bucket, items, -}, counts [nl], then bases [nl] (giant_finish)
template <bool COMPACT>
__device__ __forceinline__ void giant_finish(const IngestParams &p, uint32_t *s_raw, const GiantBucket &gb)
{
    typedef BucketCfg<COMPACT> C;
    __shared__ uint32_t s_w[kNT / 32];
    __shared__ int s_act2, s_class2[kNumClasses];
    uint32_t *rowstart = s_raw;                            // [nl] (the sort buffers are idle)
    const int t = threadIdx.x, nl = 1 << p.bl, b = gb.bucket, pix0 = b << p.bl, gbase = p.bkt_base[b];
    const int row_words = kRowHdr + 2 * nl;
    const int per = (nl + kNT - 1) / kNT;                  // <= 8
    if (t == 0) s_act2 = 0;
    if (t < kNumClasses) s_class2[t] = 0;
    __syncthreads();
    // per pixel: events in earlier chunks (prefix over the chunk rows), total
    uint32_t v[8];
    uint32_t sum = 0;
#pragma unroll
    for (int k = 0; k < 8; ++k) {
        const int l = t * per + k;
        v[k] = 0;
        if (k < per && l < nl) {
            uint32_t run = 0;
            for (int c = 0; c < gb.n_chunks; ++c) {
                int32_t *rw = p.chunk_rows + static_cast<size_t>(gb.row0 + c) * row_words;
                const uint32_t n = static_cast<uint32_t>(__ldcg(rw + kRowHdr + l));
                rw[kRowHdr + nl + l] = static_cast<int32_t>(run);
                run += n;
            }
            v[k] = run;
        }
        sum += v[k];
    }
    int tot;
    uint32_t ex = static_cast<uint32_t>(block_excl_sum(static_cast<int>(sum), tot, s_w));
    const int nmin = p.prev_csr ? 0x7fffffff : max(p.n_min, 1);
#pragma unroll
    for (int k = 0; k < 8; ++k) {
        const int l = t * per + k;
        if (k < per && l < nl) {
            rowstart[l] = ex;
            if (pix0 + l < p.np) {
                p.cnt[pix0 + l] = static_cast<int32_t>(v[k]);
                if (p.slab_row_ptr) p.slab_row_ptr[pix0 + l] = gbase + static_cast<int32_t>(ex);
                if (static_cast<int>(v[k]) >= nmin) {
                    int seg_len;
                    const int n_seg = row_segments(static_cast<int>(v[k]), seg_len);
                    atomicAdd(&s_act2, 1);
                    if (class_items(p, static_cast<int>(v[k]), n_seg)) atomicAdd(&s_class2[size_class(seg_len)], class_items(p, static_cast<int>(v[k]), n_seg));
                }
            }
            ex += v[k];
        }
    }
    __syncthreads();
    // bases: row start of the pixel + its events in earlier chunks
    for (int c = 0; c < gb.n_chunks; ++c) {
        int32_t *rw = p.chunk_rows + static_cast<size_t>(gb.row0 + c) * row_words;
        for (int l = t; l < nl; l += kNT) rw[kRowHdr + nl + l] += static_cast<int32_t>(rowstart[l]);
    }
    if (t == 0) p.bkt_act[b] = s_act2;
    if (t < kNumClasses && s_class2[t]) atomicAdd(&p.class_cnt[t], s_class2[t]);
    __syncthreads();
}

template <bool COMPACT>
__global__ void __launch_bounds__(kNT, 2) k_bucket_sort(IngestParams p)
{
    extern __shared__ __align__(16) uint32_t s_raw[];
    __shared__ int s_ticket, s_g;
    __shared__ bool s_lastc;
    const int t = threadIdx.x;
    const int n_tiles = static_cast<int>((p.n + kTile - 1) / kTile);
    if (static_cast<int>(blockIdx.x) < p.nb) {
        const int b = p.bkt_order[blockIdx.x];                 // largest buckets first
        if (b < 0) return;                                     // a giant bucket: its chunks go to the helper CTAs
        bucket_body<COMPACT>(p, s_raw, b, 0, n_tiles, -1, 0);
        return;
    }
    // helper CTAs: chunks of giant buckets
    GiantBucket *tab = reinterpret_cast<GiantBucket *>(p.giant_tab);
    const int n_giant = p.sync[10], n_chunks_all = p.sync[11];
    while (true) {
        __syncthreads();
        if (t == 0) {
            const int ch = atomicAdd(p.sync + 12, 1);
            s_ticket = ch;
            int g = 0;
            if (ch < n_chunks_all)
                while (g + 1 < n_giant && !(ch >= tab[g].chunk0 && ch < tab[g].chunk0 + tab[g].n_chunks)) ++g;
            s_g = g;
        }
        __syncthreads();
        const int ch = s_ticket;
        if (ch >= n_chunks_all) return;
        GiantBucket &gb = tab[s_g];
        const int c = ch - gb.chunk0, b = gb.bucket;
        const int tile_lo = c * gb.tiles_per_chunk, tile_hi = min(n_tiles, tile_lo + gb.tiles_per_chunk);
        // the bucket's events in earlier tiles
        int off = 0;
        for (int j = t; j < tile_lo; j += kNT) off += static_cast<int>(__ldg(p.run_tab + static_cast<size_t>(j) * p.nb + b) >> 16);
        __shared__ uint32_t s_w2[kNT / 32];
        int total_before;
        block_excl_sum(off, total_before, s_w2);
        bucket_body<COMPACT>(p, s_raw, b, tile_lo, tile_hi, gb.row0 + c, total_before);
        __threadfence();
        __syncthreads();
        if (t == 0) s_lastc = (atomicAdd(&gb.done, 1) == gb.n_chunks - 1);
        __syncthreads();
        if (s_lastc) {
            __threadfence();
            giant_finish<COMPACT>(p, s_raw, gb);
        }
    }
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

// placement of one sorted chunk of a giant bucket (helper CTAs of k_worklist, 1024 threads)
template <bool COMPACT>
__device__ __forceinline__ void giant_place(const IngestParams &p, const GiantBucket &gb, int c, int *s_delta, int *s_a, int *s_b)
{
    typedef BucketCfg<COMPACT> C;
    typedef typename C::T T;
    const int t = threadIdx.x, nl = 1 << p.bl, gbase = p.bkt_base[gb.bucket];
    const int row_words = kRowHdr + 2 * nl;
    const int32_t *rw = p.chunk_rows + static_cast<size_t>(gb.row0 + c) * row_words;
    const int coff = rw[1], cfill = rw[2];
    // run start of every pixel inside the sorted chunk = exclusive scan of the chunk's counts (nl <= 4096: 4 per thread)
    int v[4], sum = 0, dummy = 0;
#pragma unroll
    for (int k = 0; k < 4; ++k) {
        const int l = t * 4 + k;
        v[k] = (l < nl) ? rw[kRowHdr + l] : 0;
        sum += v[k];
    }
    int ta, tb;
    block_scan2(sum, dummy, ta, tb, s_a, s_b);              // sum -> exclusive prefix
#pragma unroll
    for (int k = 0; k < 4; ++k) {
        const int l = t * 4 + k;
        if (l < nl) { s_delta[l] = rw[kRowHdr + nl + l] - sum; sum += v[k]; }
    }
    __syncthreads();
    const T *scratch = reinterpret_cast<const T *>(p.scratch);
    for (int r = t; r < cfill; r += 1024) {
        const T item = scratch[static_cast<size_t>(gbase) + coff + r];
        p.csr_ev[gbase + s_delta[C::low_of(item, p.vb)] + r] = C::val_of(item, p.vb);
    }
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

// Work item(s) of one active row: the row itself, or one item per segment of a split row (ndft.cu)
__device__ __forceinline__ void emit_work(const IngestParams &p, WorkItem *dst, int pix, int off, int n, int aoff,
                                          int n_seg, int seg_len)
{
    WorkItem it;
    if (n_seg == 1) {
        if (is_hot(p, n, n_seg)) dst = p.hot_work + atomicAdd(p.sync + 15, 1);
        it.row_begin = off;
        it.n = n;
        it.pix = pix;
        it.arow = aoff;
        *dst = it;
        return;
    }
    // split row: the row's identity goes to the split table, its segments to the segment list if there is one
    if (p.seg_work) dst = p.seg_work + atomicAdd(p.sync + 9, n_seg);
    const int sid = atomicAdd(p.sync + 5, 1);
    SplitRow sr;
    const int nodes = split_nodes(n_seg);
    sr.pix = pix; sr.arow = aoff; sr.n_seg = n_seg;
    sr.seg_base = atomicAdd(p.sync + 6, split_slots(n_seg));
    sr.cnt_base = atomicAdd(p.sync + 7, nodes);
    sr._pad[0] = 0; sr._pad[1] = 0; sr._pad[2] = 0;
    p.split_tab[sid] = sr;
    for (int q = 0; q < nodes; ++q) p.split_cnt[sr.cnt_base + q] = 0;
    for (int sg = 0; sg < n_seg; ++sg) {
        it.row_begin = off + sg * seg_len;
        it.n = min(seg_len, n - sg * seg_len);
        it.pix = static_cast<int32_t>(0x80000000u | static_cast<uint32_t>(sid));
        it.arow = sg;
        dst[sg] = it;
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
            int seg_len;
            const int n_seg = row_segments(v[j], seg_len);
            if (class_items(p, v[j], n_seg)) atomicAdd(&s_cls[size_class(seg_len)], class_items(p, v[j], n_seg));
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
        if (p.prev_csr && ta > p.csr_cap) atomicOr(&p.counters[DDHF_CNT_OVERFLOW], 4);   // sliding window outgrew max_events
        int run = 0;
        for (int c = kNumClasses - 1; c >= 0; --c) {     // descending cost
            const int n = p.class_cnt[c];
            p.class_cnt[c] = run;                         // becomes the class base
            run += n;
        }
        p.sync[4] = run;                                  // work items (a split row counts once per segment)
    }
}

// ---- k_scan_apply: row_ptr, active_idx, size-classed work list --------------------------
__global__ void __launch_bounds__(1024) k_scan_apply(IngestParams p)
{
    __shared__ int s_a[33], s_b[33];
    __shared__ int s_cls[kNumClasses], s_base[kNumClasses];
    if (threadIdx.x < kNumClasses) s_cls[threadIdx.x] = 0;
    __syncthreads();
    const int base = blockIdx.x * kScanTile + threadIdx.x * 4;
    int v[4];
    load4(p.cnt, base, p.np, v);
    const int nmin = max(p.n_min, 1);
    int sum = 0, act = 0;
    int lrank[4];
#pragma unroll
    for (int j = 0; j < 4; ++j) {
        sum += v[j];
        lrank[j] = -1;
        if (v[j] >= nmin) {
            ++act;
            int seg_len;
            const int n_seg = row_segments(v[j], seg_len);
            lrank[j] = atomicAdd(&s_cls[size_class(seg_len)], class_items(p, v[j], n_seg));
        }
    }
    int ta, tb;
    block_scan2(sum, act, ta, tb, s_a, s_b);       // contains __syncthreads: s_cls is final
    if (threadIdx.x < kNumClasses) {
        const int n = s_cls[threadIdx.x];
        s_base[threadIdx.x] = p.class_cnt[threadIdx.x] + (n ? atomicAdd(&p.class_cur[threadIdx.x], n) : 0);
    }
    __syncthreads();
    int off = p.tile_off[blockIdx.x] + sum;
    int aoff = p.tile_aoff[blockIdx.x] + act;
#pragma unroll
    for (int j = 0; j < 4; ++j) {
        const int pix = base + j;
        if (pix < p.np) {
            p.row_ptr[pix] = off;
            if (lrank[j] >= 0) {
                if (aoff < p.max_active) p.active_idx[aoff] = pix;
                int seg_len;
                const int n_seg = row_segments(v[j], seg_len);
                WorkItem *dst = p.work + s_base[size_class(seg_len)] + lrank[j];
                emit_work(p, dst, pix, off, v[j], aoff, n_seg, seg_len);
                ++aoff;
            }
            off += v[j];
        }
    }
}




// ---- k_worklist: active list and size-classed work list, one CTA per bucket ---------------------------
// The from-scratch path: k_bucket_sort has written cnt and row_ptr of every pixel, the active pixels of
// every bucket (bkt_act) and the class totals (class_cnt), so the three scan kernels above (still used by
// the sliding-window path, where the counts come from two sources) collapse into this one.
__global__ void __launch_bounds__(1024) k_worklist(IngestParams p)
{
    __shared__ int s_a[33], s_b[33];
    __shared__ int s_cls[kNumClasses], s_base[kNumClasses], s_tot[kNumClasses];
    const int t = threadIdx.x;
    const int n_list_ctas = (p.np + kScanTile - 1) / kScanTile;
    if (static_cast<int>(blockIdx.x) >= n_list_ctas) {
        // helper CTAs: the sorted chunks of giant buckets go to their places in csr_ev
        __shared__ int s_delta[4096], s_ticket, s_g;
        const GiantBucket *tab = reinterpret_cast<const GiantBucket *>(p.giant_tab);
        const int n_giant = p.sync[10], n_chunks_all = p.sync[11];
        while (true) {
            __syncthreads();
            if (t == 0) {
                const int ch = atomicAdd(p.sync + 13, 1);
                s_ticket = ch;
                int g = 0;
                if (ch < n_chunks_all)
                    while (g + 1 < n_giant && !(ch >= tab[g].chunk0 && ch < tab[g].chunk0 + tab[g].n_chunks)) ++g;
                s_g = g;
            }
            __syncthreads();
            const int ch = s_ticket;
            if (ch >= n_chunks_all) return;
            const GiantBucket &gb = tab[s_g];
            if (p.compact) giant_place<true>(p, gb, ch - gb.chunk0, s_delta, s_a, s_b);
            else giant_place<false>(p, gb, ch - gb.chunk0, s_delta, s_a, s_b);
        }
    }
    if (t < kNumClasses) { s_cls[t] = 0; s_tot[t] = p.class_cnt[t]; }
    // a tile of kScanTile pixels holds whole buckets (2^bL divides it): active pixels in the buckets before it
    const int nl = 1 << p.bl;
    const int first_bucket = (blockIdx.x * kScanTile) >> p.bl;
    int a = (t < p.nb) ? p.bkt_act[t] : 0;                // nb <= 1023: one value per thread
    int before = (t < first_bucket) ? a : 0;
    int ta, tb;
    block_scan2(a, before, ta, tb, s_a, s_b);             // ta = all active pixels, tb = those before this tile
    const int n_active = ta, aoff0 = tb;
    if (t == 0) {
        // class bases: descending cost (every CTA derives the same values from the totals)
        int run = 0;
        for (int c = kNumClasses - 1; c >= 0; --c) { s_base[c] = run; run += s_tot[c]; }
        if (blockIdx.x == 0) {
            p.row_ptr[p.np] = p.bkt_base[p.nb];
            p.counters[DDHF_CNT_N_ACTIVE] = n_active;
            if (n_active > p.max_active) atomicOr(&p.counters[DDHF_CNT_OVERFLOW], 1);
            p.sync[4] = run;                              // work items (a split row counts once per segment)
        }
    }
    __syncthreads();
    (void)nl;
    const int base = blockIdx.x * kScanTile + t * 4;
    const int nmin = max(p.n_min, 1);
    int v[4], lrank[4], act = 0, dummy = 0;
    load4(p.cnt, base, p.np, v);
#pragma unroll
    for (int j = 0; j < 4; ++j) {
        lrank[j] = -1;
        if (v[j] >= nmin) {
            ++act;
            int seg_len;
            const int n_seg = row_segments(v[j], seg_len);
            lrank[j] = atomicAdd(&s_cls[size_class(seg_len)], class_items(p, v[j], n_seg));
        }
    }
    int t1, t2;
    block_scan2(act, dummy, t1, t2, s_a, s_b);            // contains __syncthreads: s_cls is final
    if (t < kNumClasses) {
        const int n = s_cls[t];
        s_base[t] += (n ? atomicAdd(&p.class_cur[t], n) : 0);
    }
    __syncthreads();
    int aoff = aoff0 + act;
#pragma unroll
    for (int j = 0; j < 4; ++j) {
        if (lrank[j] >= 0) {
            const int pix = base + j;
            if (aoff < p.max_active) p.active_idx[aoff] = pix;
            int seg_len;
            const int n_seg = row_segments(v[j], seg_len);
            emit_work(p, p.work + s_base[size_class(seg_len)] + lrank[j], pix, p.row_ptr[pix], v[j], aoff, n_seg, seg_len);
            ++aoff;
        }
    }
}

// ---- sliding windows: the previous window's CSR advanced by one hop --------------------
// Row of a pixel in the new window = the previous row's events that are still inside it (value >= 2 shift,
// shift = t0 - previous t0; re-based to the new t0) followed by the pixel's events of the new slab, which
// has just been bucketed on its own (k_tile_sort / k_bucket_sort: cnt = slab counts, slab_row_ptr, slab_csr).
// That is the input order of the window's slice of the stream, so row_ptr / csr_ev equal a bucketing from
// scratch bit for bit (R20).  One thread per pixel: rows hold a few events.
__global__ void k_slide_count(IngestParams p)
{
    const int pix = blockIdx.x * blockDim.x + threadIdx.x;
    if (pix >= p.np) return;
    const int r0 = p.prev_row_ptr[pix], r1 = p.prev_row_ptr[pix + 1];
    int kept = 0;
    for (int k = r0; k < r1; ++k) kept += (p.prev_csr[k] >= p.shift2) ? 1 : 0;
    p.cnt[pix] += kept;
}

__global__ void k_slide_merge(IngestParams p)
{
    const int pix = blockIdx.x * blockDim.x + threadIdx.x;
    if (pix > p.np) return;
    const int dst0 = p.row_ptr[pix];
    p.next_row_ptr[pix] = dst0;                           // the state of the next call
    if (pix == p.np) return;
    const int total = p.row_ptr[pix + 1] - dst0;
    const int r0 = p.prev_row_ptr[pix], r1 = p.prev_row_ptr[pix + 1];
    int k = 0;
    for (int q = r0; q < r1; ++q) {
        const uint32_t v = p.prev_csr[q];
        if (v >= p.shift2) {
            const uint32_t w = v - p.shift2;
            if (dst0 + k < p.csr_cap) {
                p.csr_ev[dst0 + k] = w;
                p.next_csr[dst0 + k] = w;
            }
            ++k;
        }
    }
    const uint32_t *src = p.slab_csr + p.slab_row_ptr[pix];
    for (int q = 0; k < total; ++q, ++k) {
        const uint32_t w = src[q];
        if (dst0 + k < p.csr_cap) {
            p.csr_ev[dst0 + k] = w;
            p.next_csr[dst0 + k] = w;
        }
    }
}

// first call of a sliding sequence: the window was bucketed from scratch; keep a copy as the state
__global__ void k_slide_save(IngestParams p)
{
    const int n_in = p.row_ptr[p.np];
    for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < n_in; i += gridDim.x * blockDim.x) p.next_csr[i] = p.csr_ev[i];
    for (int i = blockIdx.x * blockDim.x + threadIdx.x; i <= p.np; i += gridDim.x * blockDim.x) p.next_row_ptr[i] = p.row_ptr[i];
}

}  // namespace

namespace {
template <bool COMPACT>
cudaError_t configure_sort_kernels()
{
    cudaError_t e = cudaFuncSetAttribute(k_tile_sort<COMPACT, false>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                         static_cast<int>(ingest_tile_smem(COMPACT)));
    if (e != cudaSuccess) return e;
    e = cudaFuncSetAttribute(k_tile_sort<COMPACT, true>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                             static_cast<int>(ingest_tile_smem(COMPACT)));
    if (e != cudaSuccess) return e;
    return cudaFuncSetAttribute(k_bucket_sort<COMPACT>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                static_cast<int>(BucketCfg<COMPACT>::smem_bytes(12)));
}
}  // namespace

size_t ingest_tile_smem(bool compact) { return 4u * ((kTile + kTile / 32) + kCntWords + 1032u + (compact ? 1u : 2u) * kTile); }

cudaError_t ingest_configure()
{
    const cudaError_t e = configure_sort_kernels<true>();
    if (e != cudaSuccess) return e;
    return configure_sort_kernels<false>();
}

int ingest_tile_events() { return kTile; }
int ingest_tile_stride(bool compact) { return compact ? TileOut<true>::kStride : TileOut<false>::kStride; }

void ingest_plan(int np, int *bl, int *nb, int *hbits)
{
    // pixel = bucket << bL | low with at most 1023 buckets (the sort digit of a tile also holds the
    // sentinel bucket of dropped events); small sensors keep 32 pixels per bucket
    int bits = 1;
    while ((1ll << bits) < np) ++bits;
    int l = bits > 15 ? bits - 10 : 5;
    while (((np + (1 << l) - 1) >> l) > 1023) ++l;
    *bl = l;
    *nb = (np + (1 << l) - 1) >> l;
    int hb = 1;
    while ((1 << hb) < *nb + 1) ++hb;
    *hbits = hb;
}

namespace {
int launch_sort(const IngestParams &p, cudaStream_t st)
{
    const int ev_tiles = static_cast<int>((p.n + kTile - 1) / kTile);
    int launches = 0;
    if (p.compact) {
        if (ev_tiles > 0) {
            if (p.packed) k_tile_sort<true, true><<<ev_tiles, kNT, ingest_tile_smem(true), st>>>(p);
            else k_tile_sort<true, false><<<ev_tiles, kNT, ingest_tile_smem(true), st>>>(p);
            ++launches;
        }
        k_bucket_sort<true><<<p.nb + kGiantHelpers, kNT, BucketCfg<true>::smem_bytes(p.bl), st>>>(p); ++launches;
    } else {
        if (ev_tiles > 0) {
            if (p.packed) k_tile_sort<false, true><<<ev_tiles, kNT, ingest_tile_smem(false), st>>>(p);
            else k_tile_sort<false, false><<<ev_tiles, kNT, ingest_tile_smem(false), st>>>(p);
            ++launches;
        }
        k_bucket_sort<false><<<p.nb + kGiantHelpers, kNT, BucketCfg<false>::smem_bytes(p.bl), st>>>(p); ++launches;
    }
    return launches;
}

int launch_scans(const IngestParams &p, cudaStream_t st)
{
    const int n_tiles = (p.np + kScanTile - 1) / kScanTile;
    k_scan_reduce<<<n_tiles, 1024, 0, st>>>(p);
    k_scan_tiles<<<1, 1024, 0, st>>>(p, n_tiles);
    k_scan_apply<<<n_tiles, 1024, 0, st>>>(p);
    return 3;
}
}  // namespace

int launch_ingest(const IngestParams &p, cudaStream_t st)
{
    int launches = 0;
    const int init_items = max(max(p.np, p.nb + 2), 1025);      // pixels, buckets, CCL tile states
    k_init<<<(init_items + 255) / 256, 256, 0, st>>>(p); ++launches;
    IngestParams q = p;                      // k_bucket_sort writes row_ptr itself
    q.slab_row_ptr = p.row_ptr;
    launches += launch_sort(q, st);
    k_worklist<<<(p.np + kScanTile - 1) / kScanTile + kGiantHelpers / 2, 1024, 0, st>>>(p); ++launches;
    if (p.next_csr) { k_slide_save<<<592, 256, 0, st>>>(p); ++launches; }      // first window of a sliding sequence
    return launches;
}

// p.events / p.n: the new slab only; the previous window is in prev_row_ptr / prev_csr
int launch_ingest_slide(const IngestParams &p, cudaStream_t st)
{
    int launches = 0;
    const int init_items = max(max(p.np, p.nb + 2), 1025);      // pixels, buckets, CCL tile states
    k_init<<<(init_items + 255) / 256, 256, 0, st>>>(p); ++launches;
    IngestParams q = p;                      // the slab is bucketed into its own CSR
    q.csr_ev = p.slab_csr;
    launches += launch_sort(q, st);
    k_slide_count<<<(p.np + 255) / 256, 256, 0, st>>>(p); ++launches;
    launches += launch_scans(p, st);
    k_slide_merge<<<(p.np + 256) / 256, 256, 0, st>>>(p); ++launches;
    return launches;
}

}  // namespace ddhf
