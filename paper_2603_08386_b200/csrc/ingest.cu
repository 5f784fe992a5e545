// ingest.cu -- a0-a3: window/sensor filter, per-pixel histogram, exclusive scan + active
// list + size-classed work list, and a STABLE bucketing of the events into CSR form.
//
// "For each window, events are moved to the GPU, sorted by pixel index";
// pixels with fewer than n_min events are discarded (L137).  Readings R19 (half-open
// window, bad coordinates dropped and counted) and R20 (input order inside a row).
//
// The bucketing is a two-pass least-significant-digit radix partition on the pixel index
// (digits of ceil(bits/2) and floor(bits/2) bits, at most 2048 bins), each pass stable, so
// that events of one pixel keep their input order and csr_ev is bit-reproducible with no
// atomics deciding any position:
//
//   pass 1   k_dhist<1>   one CTA per tile of 8192 events: per-pixel histogram (global
//                         atomics, order-free), per-tile digit histogram M[tile][bin]
//            k_binscan<1> bin-major exclusive scan of the tile histograms (per 8-tile chunk)
//            k_part<1>    re-reads the tile, ranks every event inside its (tile, bin) group in
//                         input order (warp match + per-warp counters + cross-warp scan) and
//                         writes (value, pixel) pairs at base + rank
//   pass 2   the same three kernels on the pairs with the high digit; the output is csr_ev.
//
// HBM traffic per event: 16 B read twice (histogram, partition 1), 8 B written and read twice,
// 4 B written; the tile histograms add 4 B x bins per 8192 events.
#include "ddhf_internal.cuh"

namespace ddhf {

namespace {

#ifndef DDHF_TILE_THREADS
#define DDHF_TILE_THREADS 512
#endif
constexpr int kTileThreads = DDHF_TILE_THREADS;
constexpr int kTileWarps = kTileThreads / 32;
#ifndef DDHF_TILE_EV
#define DDHF_TILE_EV 16
#endif
constexpr int kTileEv = DDHF_TILE_EV;                // events per thread
constexpr int kTile = kTileThreads * kTileEv;        // 8192 events per tile
constexpr int kWarpSpan = 32 * kTileEv;              // consecutive events owned by one warp
constexpr int kChunkTiles = 8;                       // tiles per scan chunk
constexpr unsigned kFullMask = 0xffffffffu;

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

// ---- k_init: per-pixel maps for inactive pixels, zeroed histograms and counters ---------
__global__ void k_init(IngestParams p)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < p.np) {
        p.cnt[i] = 0;
        p.sf[i] = __int_as_float(0x7fc00000);   // NaN: pixel not active
        p.score[i] = 0.f;
        p.f0_idx[i] = -1;
        p.mask[i] = 0;
        p.ccl_parent[i] = 0x7fffffff;           // no parent yet
    }
    for (int k = i; k < p.chunk_words; k += gridDim.x * blockDim.x) p.chunk1[k] = 0;   // chunk1, chunk2
    if (blockIdx.x == 0) {
        if (threadIdx.x < DDHF_N_COUNTERS) p.counters[threadIdx.x] = 0;
        if (threadIdx.x < kNumClasses) {
            p.class_cnt[threadIdx.x] = 0;
            p.class_cur[threadIdx.x] = 0;
        }
        if (threadIdx.x == 0) { *p.work_cursor = 0ull; p.scan_done[0] = 0; p.scan_done[1] = 0; p.scan_done[2] = 0; p.scan_done[3] = 0; }
    }
}

// ---- k_dhist: digit histogram of one tile; pass 2 also counts[pix] += n (a1) ---------------
// The per-pixel histogram is taken in pass 2: its input is sorted by the low digit, so a tile
// holds very few distinct low digits and the counts of (low digit, high digit) = pixel can be
// pre-aggregated in shared memory; only the non-zero sums go to global memory as atomics.
constexpr int kLoSpan = 4;     // distinct low digits per tile that are aggregated in shared memory

template <int PASS>
__global__ void __launch_bounds__(kTileThreads) k_dhist(IngestParams p)
{
    extern __shared__ uint32_t s_hist[];            // [bins] (+ [kLoSpan][bins] in pass 2)
    __shared__ int s_drop;
    const int bits = (PASS == 1) ? p.bits1 : p.bits2;
    const int bins = 1 << bits;
    const int64_t n_src = (PASS == 1) ? p.n : static_cast<int64_t>(p.counters[DDHF_CNT_N_IN]);
    const int64_t tile_beg = static_cast<int64_t>(blockIdx.x) * kTile;
    if (tile_beg >= n_src) return;
    const int words = (PASS == 1) ? bins : (1 + kLoSpan) * bins;
    for (int b = threadIdx.x; b < words; b += kTileThreads) s_hist[b] = 0;
    if (threadIdx.x == 0) s_drop = 0;
    __syncthreads();
    if (PASS == 1) {
        int32_t px[kTileEv];
#pragma unroll
        for (int u = 0; u < kTileEv; ++u) {
            const int64_t i = tile_beg + u * kTileThreads + threadIdx.x;
            px[u] = -2;
            if (i < n_src) px[u] = decode_event(p.events, i, p.t0, p.t1, p.width, p.height).pix;
        }
        const uint32_t dmask = static_cast<uint32_t>(bins - 1);
        int drop = 0;
#pragma unroll
        for (int u = 0; u < kTileEv; ++u) {
            if (px[u] >= 0) atomicAdd(&s_hist[static_cast<uint32_t>(px[u]) & dmask], 1u);
            drop += (px[u] == -1);
        }
        drop = __reduce_add_sync(kFullMask, drop);
        if ((threadIdx.x & 31) == 0 && drop) atomicAdd(&s_drop, drop);
    } else {
        uint32_t *s_pix = s_hist + bins;            // [kLoSpan][bins]
        const uint32_t lmask = (1u << p.bits1) - 1u;
        const uint32_t lo_first = __ldg(reinterpret_cast<const uint32_t *>(p.pairs + tile_beg) + 1) & lmask;
        uint32_t px[kTileEv];
#pragma unroll
        for (int u = 0; u < kTileEv; ++u) {
            const int64_t i = tile_beg + u * kTileThreads + threadIdx.x;
            px[u] = 0xffffffffu;
            if (i < n_src) px[u] = __ldg(reinterpret_cast<const uint32_t *>(p.pairs + i) + 1);
        }
#pragma unroll
        for (int u = 0; u < kTileEv; ++u) {
            if (px[u] != 0xffffffffu) {
                const uint32_t hi = px[u] >> p.bits1, dl = (px[u] & lmask) - lo_first;
                if (dl < static_cast<uint32_t>(kLoSpan)) {
                    atomicAdd(&s_pix[dl * bins + hi], 1u);
                } else {
                    atomicAdd(&s_hist[hi], 1u);
                    atomicAdd(&p.cnt[px[u]], 1);
                }
            }
        }
        __syncthreads();
        for (int b = threadIdx.x; b < bins; b += kTileThreads) {
            uint32_t tot = 0;
#pragma unroll
            for (int l = 0; l < kLoSpan; ++l) {
                const uint32_t c = s_pix[l * bins + b];
                if (c) atomicAdd(&p.cnt[(static_cast<uint32_t>(b) << p.bits1) | (lo_first + l)], static_cast<int>(c));
                tot += c;
            }
            s_hist[b] += tot;                       // same thread reads it below
        }
    }
    __syncthreads();
    int32_t *row = p.tile_hist + static_cast<size_t>(blockIdx.x) * bins;
    int32_t *chunk = ((PASS == 1) ? p.chunk1 : p.chunk2) + static_cast<size_t>(blockIdx.x / kChunkTiles) * bins;
    for (int b = threadIdx.x; b < bins; b += kTileThreads) {
        const int c = static_cast<int>(s_hist[b]);
        row[b] = c;
        if (c) atomicAdd(&chunk[b], c);
    }
    if (PASS == 1 && threadIdx.x == 0 && s_drop) atomicAdd(&p.counters[DDHF_CNT_N_DROPPED], s_drop);
}

// ---- k_binscan: bin-major exclusive scan of the chunk totals ------------------------------
// chunk[c][b] becomes the number of events of bin b in chunks before c; bin_base[b] the number
// of events in bins before b.  One CTA per 32 bins; warp g of a CTA owns a contiguous range
// of chunks, lane l the bin.  The last CTA to finish scans the bin totals.
// Pass 1 also publishes the number of kept events.
template <int PASS>
__global__ void __launch_bounds__(1024) k_binscan(IngestParams p)
{
    __shared__ int s_grp[32][33];
    __shared__ int s_w[33];
    __shared__ bool s_last;
    const int bits = (PASS == 1) ? p.bits1 : p.bits2;
    const int bins = 1 << bits;
    const int64_t n_src = (PASS == 1) ? p.n : static_cast<int64_t>(p.counters[DDHF_CNT_N_IN]);
    const int n_tiles = static_cast<int>((n_src + kTile - 1) / kTile);
    const int n_chunks = (n_tiles + kChunkTiles - 1) / kChunkTiles;
    int32_t *chunk = (PASS == 1) ? p.chunk1 : p.chunk2;
    int32_t *bin_base = (PASS == 1) ? p.bin_base1 : p.bin_base2;
    int32_t *bin_tot = p.bin_tot;
    const int lane = threadIdx.x & 31, g = threadIdx.x >> 5;
    const int b = blockIdx.x * 32 + lane;
    const bool live = b < bins;
    const int per_g = (n_chunks + 31) / 32;
    const int c_beg = min(g * per_g, n_chunks), c_end = min(c_beg + per_g, n_chunks);
    int sum = 0;
    if (live)
        for (int c = c_beg; c < c_end; ++c) sum += chunk[static_cast<size_t>(c) * bins + b];
    s_grp[g][lane] = sum;
    __syncthreads();
    int pre = 0, tot = 0;
    for (int q = 0; q < 32; ++q) {
        const int a = s_grp[q][lane];
        if (q < g) pre += a;
        tot += a;
    }
    if (live)
        for (int c = c_beg; c < c_end; ++c) {
            int32_t *q = chunk + static_cast<size_t>(c) * bins + b;
            const int v = *q;
            *q = pre;
            pre += v;
        }
    if (g == 0 && live) bin_tot[b] = tot;
    // last CTA: exclusive scan of the bin totals
    __threadfence();
    __syncthreads();
    if (threadIdx.x == 0) s_last = (atomicAdd(p.scan_done + (PASS - 1), 1) == static_cast<int>(gridDim.x) - 1);
    __syncthreads();
    if (!s_last) return;
    __threadfence();
    // thread t owns bins 2t and 2t+1 (bins <= 2048)
    const int b0 = 2 * threadIdx.x;
    const int run0 = (b0 < bins) ? *reinterpret_cast<volatile int32_t *>(bin_tot + b0) : 0;
    const int run1 = (b0 + 1 < bins) ? *reinterpret_cast<volatile int32_t *>(bin_tot + b0 + 1) : 0;
    const int wid = g;
    const int mine = run0 + run1;
    int inc = mine;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const int t = __shfl_up_sync(kFullMask, inc, o);
        if (lane >= o) inc += t;
    }
    if (lane == 31) s_w[wid] = inc;
    __syncthreads();
    if (wid == 0) {
        const int w = s_w[lane];
        int x = w;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const int t = __shfl_up_sync(kFullMask, x, o);
            if (lane >= o) x += t;
        }
        s_w[lane] = x - w;
        if (lane == 31) s_w[32] = x;
    }
    __syncthreads();
    const int excl = inc - mine + s_w[wid];
    if (b0 < bins) bin_base[b0] = excl;
    if (b0 + 1 < bins) bin_base[b0 + 1] = excl + run0;
    if (PASS == 1 && threadIdx.x == 0) p.counters[DDHF_CNT_N_IN] = s_w[32];
}

// ---- k_part: stable partition of one tile by the pass's digit ----------------------------
// Warp w of the CTA owns the tile's events [512 w, 512 w + 512) and walks them in 16 steps of
// 32 consecutive events.  Inside a step, lanes with the same digit find each other with
// a ballot per digit bit; the lowest lane of a group advances the warp's counter of that digit, so an
// event's rank inside (tile, digit) follows input order exactly.  The tile is then laid out in
// shared memory in output order (bin-major) and written with consecutive threads on
// consecutive elements, so that every run of a bin is a coalesced store.
// Slow path of the ranking step (two lanes of the warp share a digit): lanes with the same digit
// find each other by one ballot per digit bit (MATCH.ANY is far slower on sm_100); the lowest lane
// of a group writes the group's count.  Kept out of line so that the common conflict-free step
// does not pay for it.
__device__ __noinline__ uint32_t rank_by_ballots(bool ok, uint32_t d, uint32_t c, int lane, unsigned short *my_cnt, int nbits)
{
    const uint32_t lt = (1u << lane) - 1u;
    uint32_t peers = __ballot_sync(kFullMask, ok);
#pragma unroll
    for (int k = 0; k < 11; ++k) {
        if (k < nbits) {                                   // warp-uniform: only the digit's own bits are voted on
            int m;                                         // 0 or -1: bit k of the digit, sign-extended
            asm("bfe.s32 %0, %1, %2, 1;" : "=r"(m) : "r"(d), "r"(k));
            const uint32_t bal = __ballot_sync(kFullMask, m != 0);
            peers &= ~(bal ^ static_cast<uint32_t>(m));    // lanes whose bit k equals mine
        }
    }
    if (ok && (peers & lt) == 0u) my_cnt[d] = static_cast<unsigned short>(c + __popc(peers));
    __syncwarp();
    return c + __popc(peers & lt);
}

template <int PASS>
struct PartSmem {
    // words: base[bins] | binoff[bins] | wcnt[kTileWarps][bins] (u16) | stage
    static constexpr int kStageWords = (PASS == 1) ? 2 * kTile : kTile + kTile / 2;
    static size_t bytes(int bins) { return static_cast<size_t>(bins) * (8 + 2 * kTileWarps) + 4u * kStageWords; }
};

#ifndef DDHF_PART_BLOCKS
#define DDHF_PART_BLOCKS (kTileThreads >= 512 ? 2 : 4)
#endif
template <int PASS>
__global__ void __launch_bounds__(kTileThreads, DDHF_PART_BLOCKS) k_part(IngestParams p)
{
    extern __shared__ uint32_t s_raw[];
    __shared__ int s_ntile;
    const int bits = (PASS == 1) ? p.bits1 : p.bits2;
    const int bins = 1 << bits;
    int32_t *s_base = reinterpret_cast<int32_t *>(s_raw);                              // [bins] global base - tile offset
    uint32_t *s_binoff = s_raw + bins;                                                 // [bins] tile-local offset of the bin
    unsigned short *s_wcnt = reinterpret_cast<unsigned short *>(s_raw + 2 * bins);     // [kTileWarps][bins]
    uint32_t *s_stage = s_raw + 2 * bins + kTileWarps * bins / 2;
    const int64_t n_src = (PASS == 1) ? p.n : static_cast<int64_t>(p.counters[DDHF_CNT_N_IN]);
    const int tile = blockIdx.x;
    const int64_t tile_beg = static_cast<int64_t>(tile) * kTile;
    if (tile_beg >= n_src) return;
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;

    for (int k = threadIdx.x; k < kTileWarps * bins / 2; k += kTileThreads)
        reinterpret_cast<uint32_t *>(s_wcnt)[k] = 0u;
    // global position of the first event of every bin of this tile
    {
        const int32_t *chunk = ((PASS == 1) ? p.chunk1 : p.chunk2) + static_cast<size_t>(tile / kChunkTiles) * bins;
        const int32_t *bin_base = (PASS == 1) ? p.bin_base1 : p.bin_base2;
        const int32_t *rows = p.tile_hist + static_cast<size_t>(tile / kChunkTiles) * kChunkTiles * bins;
        const int n_before = tile % kChunkTiles;
        for (int b = threadIdx.x; b < bins; b += kTileThreads) {
            int acc = bin_base[b] + chunk[b];
#pragma unroll
            for (int t = 0; t < kChunkTiles - 1; ++t)
                if (t < n_before) acc += rows[static_cast<size_t>(t) * bins + b];
            s_base[b] = acc;
        }
    }
    uint32_t val[kTileEv], pix[kTileEv];
    const int64_t warp_beg = tile_beg + wid * kWarpSpan + lane;
#pragma unroll
    for (int s = 0; s < kTileEv; ++s) {
        const int64_t i = warp_beg + s * 32;
        pix[s] = 0xffffffffu;
        val[s] = 0u;
        if (i < n_src) {
            if (PASS == 1) {
                const Ev e = decode_event(p.events, i, p.t0, p.t1, p.width, p.height);
                pix[s] = static_cast<uint32_t>(e.pix);          // -1 -> 0xffffffff
                val[s] = e.val;
            } else {
                const uint2 q = __ldg(reinterpret_cast<const uint2 *>(p.pairs) + i);
                val[s] = q.x;
                pix[s] = q.y;
            }
        }
    }
    __syncthreads();

    // rank inside (warp, digit) in input order
    unsigned short *my_cnt = s_wcnt + wid * bins;
    const uint32_t dmask = static_cast<uint32_t>(bins - 1);
    const uint32_t lt = (1u << lane) - 1u;
    uint32_t key[kTileEv];                    // digit | rank << 16
#pragma unroll
    for (int s = 0; s < kTileEv; ++s) {
        const bool ok = pix[s] != 0xffffffffu;
        const uint32_t d = (PASS == 1) ? (pix[s] & dmask) : ((pix[s] >> p.bits1) & dmask);
        // Optimistic step: every lane bumps its digit's counter and tags it with its lane id
        // (counts are <= 512, the tag sits above bit 11).  If every lane reads its own tag back,
        // no two lanes shared a digit and the ranks are simply the old counts.
        const uint32_t c = ok ? (my_cnt[d] & 0x7ffu) : 0u;
        __syncwarp();
        if (ok) my_cnt[d] = static_cast<unsigned short>((c + 1u) | (static_cast<uint32_t>(lane) << 11));
        __syncwarp();
        const bool lost = ok && (static_cast<uint32_t>(my_cnt[d]) >> 11) != static_cast<uint32_t>(lane);
        uint32_t rank = c;
        if (__any_sync(kFullMask, lost)) rank = rank_by_ballots(ok, d, c, lane, my_cnt, bits);
        key[s] = ok ? (d | (rank << 16)) : 0xffffffffu;
    }
    __syncthreads();
    // per bin: exclusive scan of the per-warp counters over the warps, then of the bin totals
    // over the bins (thread t owns `per` consecutive bins)
    {
        __shared__ uint32_t s_ws[kTileWarps + 1];
        const int per = (bins + kTileThreads - 1) / kTileThreads;
        const int bb = threadIdx.x * per;
        uint32_t tot[8];                                       // per <= 8 (bins <= 2048, >= 256 threads)
        uint32_t sum = 0;
#pragma unroll
        for (int j = 0; j < 8; ++j) {
            tot[j] = 0;
            const int b = bb + j;
            if (j < per && b < bins) {
                uint32_t run = 0;
#pragma unroll
                for (int w = 0; w < kTileWarps; ++w) {
                    const uint32_t t = s_wcnt[w * bins + b] & 0x7ffu;
                    s_wcnt[w * bins + b] = static_cast<unsigned short>(run);
                    run += t;
                }
                tot[j] = run;
                sum += run;
            }
        }
        uint32_t inc = sum;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const uint32_t t = __shfl_up_sync(kFullMask, inc, o);
            if (lane >= o) inc += t;
        }
        if (lane == 31) s_ws[wid] = inc;
        __syncthreads();
        if (wid == 0) {
            const uint32_t w = (lane < kTileWarps) ? s_ws[lane] : 0u;
            uint32_t x = w;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                const uint32_t t = __shfl_up_sync(kFullMask, x, o);
                if (lane >= o) x += t;
            }
            if (lane < kTileWarps) s_ws[lane] = x - w;
        }
        __syncthreads();
        uint32_t off = inc - sum + s_ws[wid];
#pragma unroll
        for (int j = 0; j < 8; ++j) {
            const int b = bb + j;
            if (j < per && b < bins) {
                s_binoff[b] = off;
                s_base[b] -= static_cast<int32_t>(off);
                off += tot[j];
            }
        }
        if (bb < bins && bb + per >= bins) s_ntile = static_cast<int>(off);
    }
    __syncthreads();
    // lay the tile out in output order
    unsigned short *s_sbin = reinterpret_cast<unsigned short *>(s_stage + kTile);      // pass 2: bin of every staged element
#pragma unroll
    for (int s = 0; s < kTileEv; ++s) {
        if (key[s] != 0xffffffffu) {
            const uint32_t d = key[s] & 0xffffu;
            const uint32_t at = s_binoff[d] + my_cnt[d] + (key[s] >> 16);
            if (PASS == 1) {
                reinterpret_cast<uint2 *>(s_stage)[at] = make_uint2(val[s], pix[s]);
            } else {
                s_stage[at] = val[s];
                s_sbin[at] = static_cast<unsigned short>(d);
            }
        }
    }
    __syncthreads();
    const int n_tile = s_ntile;                                                          // kept events of this tile
    for (int i = threadIdx.x; i < n_tile; i += kTileThreads) {
        if (PASS == 1) {
            const uint2 q = reinterpret_cast<const uint2 *>(s_stage)[i];
            const uint32_t d = q.y & dmask;
            p.pairs[s_base[d] + i] = (static_cast<uint64_t>(q.y) << 32) | q.x;
        } else {
            p.csr_ev[s_base[s_sbin[i]] + i] = s_stage[i];
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
            lrank[j] = atomicAdd(&s_cls[size_class(v[j])], 1);
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


}  // namespace

cudaError_t ingest_configure()
{
    // sized for the largest digit (2048 bins)
    cudaError_t e = cudaFuncSetAttribute(k_part<1>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                         static_cast<int>(PartSmem<1>::bytes(2048)));
    if (e != cudaSuccess) return e;
    return cudaFuncSetAttribute(k_part<2>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                static_cast<int>(PartSmem<2>::bytes(2048)));
}

int ingest_tile_events() { return kTile; }
int ingest_chunk_tiles() { return kChunkTiles; }

int launch_ingest(const IngestParams &p, cudaStream_t st)
{
    const int n_tiles = (p.np + kScanTile - 1) / kScanTile;
    const int ev_tiles = static_cast<int>((p.n + kTile - 1) / kTile);
    const int bins1 = 1 << p.bits1, bins2 = 1 << p.bits2;
    const size_t part1_smem = PartSmem<1>::bytes(bins1), part2_smem = PartSmem<2>::bytes(bins2);
    int launches = 0;
    k_init<<<(p.np + 255) / 256, 256, 0, st>>>(p); ++launches;
    if (ev_tiles > 0) {
        k_dhist<1><<<ev_tiles, kTileThreads, bins1 * 4, st>>>(p); ++launches;
        k_binscan<1><<<(bins1 + 31) / 32, 1024, 0, st>>>(p); ++launches;
        k_part<1><<<ev_tiles, kTileThreads, part1_smem, st>>>(p); ++launches;
        k_dhist<2><<<ev_tiles, kTileThreads, (1 + kLoSpan) * bins2 * 4, st>>>(p); ++launches;
        k_binscan<2><<<(bins2 + 31) / 32, 1024, 0, st>>>(p); ++launches;
        k_part<2><<<ev_tiles, kTileThreads, part2_smem, st>>>(p); ++launches;
    }
    k_scan_reduce<<<n_tiles, 1024, 0, st>>>(p); ++launches;
    k_scan_tiles<<<1, 1024, 0, st>>>(p, n_tiles); ++launches;
    k_scan_apply<<<n_tiles, 1024, 0, st>>>(p); ++launches;
    return launches;
}

}  // namespace ddhf
