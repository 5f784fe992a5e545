// ccl.cu -- a8: 8-connected component labelling of the detection mask, bounding boxes and
// the A_min filter ("We apply 8-connected component labeling to the boolean mask ... extract
// their bounding boxes.  Small boxes below the area threshold A_min are removed", PAPER.md
// L164).  Readings: R17 (area = bounding-box area), R18 (label = minimum linear pixel index of
// the component, boxes in ascending label order).
//
// Union-find with atomicMin so that the root of every tree is the smallest linear index of its
// component, which makes labels and box order deterministic.  The mask is at most a few MB and
// normally sparse, so the stage is bound by launch latency, not by bandwidth: four kernels.
//
//   parent[] arrives filled with INT_MAX (k_init of the ingest stage): "no parent yet".  A node
//   is a root while parent[x] >= x, and links only ever go to smaller indices.
//   k_ccl_merge     every mask pixel resets its box record and unites with the start of its
//                   horizontal run and with its N (else NW, NE) neighbours
//   k_ccl_label     parent[i] = root (labels; -1 off the mask); box record of the root updated
//   k_ccl_boxes     per tile of 4096 pixels: roots, roots whose box passes A_min, and their ordered compaction
//                   into boxes[] (ascending label) with a chained count over the tiles
//   k_box_merge_pairs   (optional) eq. 12: boxes with close centres merged into the final detections
#include "ddhf_internal.cuh"

namespace ddhf {

namespace {

constexpr int kTile = 4096;      // 1024 threads x 4

__device__ __forceinline__ int uf_find(int *parent, int x)
{
    // find with path halving; parent[] only ever decreases, so concurrent halving is safe
    int p = *reinterpret_cast<volatile int *>(parent + x);
    while (p < x) {
        const int gp = *reinterpret_cast<volatile int *>(parent + p);
        if (gp < p) atomicMin(parent + x, gp);
        x = p;
        p = gp;
    }
    return x;
}

__device__ __forceinline__ void uf_union(int *parent, int a, int b)
{
    while (true) {
        a = uf_find(parent, a);
        b = uf_find(parent, b);
        if (a == b) return;
        if (a < b) { const int t = a; a = b; b = t; }     // link the larger root under the smaller
        const int old = atomicMin(parent + a, b);
        if (old >= a) return;                             // a was still a root
        a = old;                                          // somebody linked a first: unite that with b
    }
}

__global__ void k_ccl_merge(CclParams p)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    const int lane = threadIdx.x & 31;
    const bool m = (i < p.np) && p.mask[i];
    // horizontal runs inside the warp's 32-pixel span (cut at row starts): every pixel of a run
    // unites directly with the run's first pixel, which keeps the trees flat
    const unsigned bits = __ballot_sync(0xffffffffu, m);
    const unsigned rs = __ballot_sync(0xffffffffu, i < p.np && (i % p.width) == 0);
    if (!m) return;
    const unsigned starts = bits & (~(bits << 1) | rs | 1u);
    const unsigned upto = starts & (0xffffffffu >> (31 - lane));
    const int run0 = i - (lane - (31 - __clz(upto)));
    int *c = p.rec + 5 * static_cast<size_t>(i);
    c[0] = 0x7fffffff; c[1] = 0x7fffffff; c[2] = -1; c[3] = -1; c[4] = 0;
    const int x = i % p.width, y = i / p.width;
    if (run0 != i) uf_union(p.parent, i, run0);
    else if (x > 0 && p.mask[i - 1]) uf_union(p.parent, i, i - 1);                   // W across a span boundary
    if (y > 0) {
        const int up = i - p.width;
        if (p.mask[up]) {
            uf_union(p.parent, i, up);                    // N (NW and NE are in N's run)
        } else {
            if (x > 0 && p.mask[up - 1]) uf_union(p.parent, i, up - 1);             // NW
            if (x + 1 < p.width && p.mask[up + 1]) uf_union(p.parent, i, up + 1);   // NE
        }
    }
}

__global__ void k_ccl_label(CclParams p)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    const int lane = threadIdx.x & 31;
    const bool m = (i < p.np) && p.mask[i];
    if (i < p.np && !m) p.parent[i] = -1;
    const unsigned act = __ballot_sync(0xffffffffu, m);
    if (!m) return;
    const int r = uf_find(p.parent, i);
    p.parent[i] = r;
    const int x = i % p.width, y = i / p.width;
    // the pixels of the warp that share a root update its record once (a dense mask is a few large
    // components: one atomic per pixel and field on the same five words serialises the whole kernel)
    const unsigned peers = __match_any_sync(act, r);
    const int x0 = __reduce_min_sync(peers, x), y0 = __reduce_min_sync(peers, y);
    const int x1 = __reduce_max_sync(peers, x), y1 = __reduce_max_sync(peers, y);
    if (lane == __ffs(peers) - 1) {
        int *c = p.rec + 5 * static_cast<size_t>(r);
        atomicMin(c + 0, x0);
        atomicMin(c + 1, y0);
        atomicMax(c + 2, x1);
        atomicMax(c + 3, y1);
        atomicAdd(c + 4, __popc(peers));
    }
}

// 0: not a root, 1: root, 3: root whose bounding box passes A_min
__device__ __forceinline__ int root_flags(const CclParams &p, int i)
{
    if (i >= p.np || !p.mask[i] || p.parent[i] != i) return 0;
    const int *c = p.rec + 5 * static_cast<size_t>(i);
    const long long area = static_cast<long long>(c[2] - c[0] + 1) * (c[3] - c[1] + 1);
    return area >= p.a_min ? 3 : 1;
}

__device__ __forceinline__ int block_sum(int a, int *s)
{
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    a = __reduce_add_sync(0xffffffffu, a);
    if (lane == 0) s[wid] = a;
    __syncthreads();
    int t = 0;
    if (wid == 0) {
        t = s[lane];
        t = __reduce_add_sync(0xffffffffu, t);
        if (lane == 0) s[32] = t;
    }
    __syncthreads();
    t = s[32];
    __syncthreads();
    return t;
}

// ---- k_ccl_boxes: count the roots of every tile and emit the passing ones in order, one pass -----------------
// Tiles take tickets (so that a tile only ever waits for tiles that are already running), publish their number
// of passing roots (tile_state[t] = count << 1 | 1; zeroed by the ingest stage) and add up the published counts of
// the tiles before them: an ordered compaction without a second kernel.
__global__ void __launch_bounds__(1024) k_ccl_boxes(CclParams p, int n_tiles)
{
    __shared__ int s[33];
    __shared__ int s_scan[33];
    __shared__ int s_tile;
    if (threadIdx.x == 0) s_tile = atomicAdd(p.tile_state + 1024, 1);
    __syncthreads();
    const int tile = s_tile;
    const int base = tile * kTile + threadIdx.x * 4;
    int f[4], roots = 0, a = 0;
#pragma unroll
    for (int j = 0; j < 4; ++j) {
        const int fl = root_flags(p, base + j);
        roots += fl & 1;
        f[j] = fl >> 1;
        a += f[j];
    }
    const int tr = block_sum(roots, s);
    const int tp = block_sum(a, s);
    if (threadIdx.x == 0) {
        atomicExch(p.tile_state + tile, (tp << 1) | 1);
        if (tr) atomicAdd(&p.counters[DDHF_CNT_N_COMPONENTS], tr);
    }
    // boxes in the tiles before this one (n_tiles <= 1024: one predecessor per thread)
    int before = 0;
    if (static_cast<int>(threadIdx.x) < tile) {
        int v;
        do { v = *reinterpret_cast<volatile int *>(p.tile_state + threadIdx.x); } while ((v & 1) == 0);
        before = v >> 1;
    }
    before = block_sum(before, s);
    if (tile == n_tiles - 1 && threadIdx.x == 0) {
        const int total = before + tp;
        p.counters[DDHF_CNT_N_BOXES_TOTAL] = total;
        p.counters[DDHF_CNT_N_BOXES] = min(total, p.max_boxes);
        if (total > p.max_boxes) atomicOr(&p.counters[DDHF_CNT_OVERFLOW], 2);
    }
    if (tp == 0) return;
    // exclusive scan over the block
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    int inc = a;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const int t = __shfl_up_sync(0xffffffffu, inc, o);
        if (lane >= o) inc += t;
    }
    if (lane == 31) s_scan[wid] = inc;
    __syncthreads();
    if (wid == 0) {
        const int w = s_scan[lane];
        int x = w;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const int t = __shfl_up_sync(0xffffffffu, x, o);
            if (lane >= o) x += t;
        }
        s_scan[lane] = x - w;
    }
    __syncthreads();
    int pos = before + inc - a + s_scan[wid];
#pragma unroll
    for (int j = 0; j < 4; ++j) {
        if (!f[j]) continue;
        if (pos < p.max_boxes) {
            const int i = base + j;
            const int *c = p.rec + 5 * static_cast<size_t>(i);
            ddhf_box b;
            b.x0 = c[0]; b.y0 = c[1]; b.x1 = c[2]; b.y1 = c[3]; b.n_pix = c[4];
            b.label = i;
            p.boxes[pos] = b;
            if (p.merge_parent) p.merge_parent[pos] = pos;       // every box starts as its own detection (eq. 12 merge)
        }
        ++pos;
    }
}

// ---- a9: box merge, eq. 12 ---------------------------------------------------
// "two boxes ... are merged if dist(c1, c2) < alpha max(w1, h1, w2, h2)".  Readings R27-R29: box
// centres, the rule evaluated on the boxes that entered the step, merging transitive.  Every pair is
// tested in double precision with the same expression as the oracle; the pair matrix is cut into
// 64 x 64 tiles spread over the grid (4096 boxes = 8.4 M pairs: one CTA needed 52 ms), pairs that pass
// are united in a union-find over box indices in the workspace (root = smallest index = smallest label,
// since boxes[] is ascending by label), and one CTA emits the roots in order.
constexpr int kMergeThreads = 256;
constexpr int kMergeTile = 64;

constexpr int kMergeSmall = 128;      // up to this many boxes one CTA does the whole step in shared memory

__device__ __forceinline__ int mg_find(volatile int *par, int x)
{
    int p = par[x];
    while (p != x) { x = p; p = par[x]; }
    return x;
}

// The usual case, a handful of boxes: all pairs, union-find, records and ordered emit by one CTA in
// shared memory (a few microseconds; the general path below costs three times that in global atomics).
__device__ __forceinline__ void merge_small(const CclParams &p, int n)
{
    __shared__ int s_par[kMergeSmall], s_rec[kMergeSmall][5];
    for (int i = threadIdx.x; i < n; i += kMergeThreads) {
        s_par[i] = i;
        s_rec[i][0] = 0x7fffffff; s_rec[i][1] = 0x7fffffff; s_rec[i][2] = -1; s_rec[i][3] = -1; s_rec[i][4] = 0;
    }
    __syncthreads();
    const double alpha = static_cast<double>(p.merge_alpha);
    for (int q = threadIdx.x; q < n * n; q += kMergeThreads) {
        const int i = q / n, j = q % n;
        if (i >= j) continue;
        const ddhf_box a = p.boxes[i], b = p.boxes[j];
        const double dx = 0.5 * (a.x0 + a.x1) - 0.5 * (b.x0 + b.x1), dy = 0.5 * (a.y0 + a.y1) - 0.5 * (b.y0 + b.y1);
        const double dist = sqrt(dx * dx + dy * dy);
        const double m = static_cast<double>(max(max(a.x1 - a.x0 + 1, a.y1 - a.y0 + 1), max(b.x1 - b.x0 + 1, b.y1 - b.y0 + 1)));
        if (dist < alpha * m) {
            int x = i, y = j;
            while (true) {                               // unite: larger root under the smaller
                x = mg_find(s_par, x);
                y = mg_find(s_par, y);
                if (x == y) break;
                if (x < y) { const int t = x; x = y; y = t; }
                const int old = atomicMin(&s_par[x], y);
                if (old == x) break;
                x = old;
            }
        }
    }
    __syncthreads();
    for (int i = threadIdx.x; i < n; i += kMergeThreads) {
        const int r = mg_find(s_par, i);
        const ddhf_box b = p.boxes[i];
        atomicMin(&s_rec[r][0], b.x0);
        atomicMin(&s_rec[r][1], b.y0);
        atomicMax(&s_rec[r][2], b.x1);
        atomicMax(&s_rec[r][3], b.y1);
        atomicAdd(&s_rec[r][4], b.n_pix);
    }
    __syncthreads();
    if (threadIdx.x == 0) {                              // roots in ascending index = ascending label
        int k = 0;
        for (int i = 0; i < n; ++i) {
            if (s_par[i] != i) continue;
            ddhf_box b;
            b.x0 = s_rec[i][0]; b.y0 = s_rec[i][1]; b.x1 = s_rec[i][2]; b.y1 = s_rec[i][3]; b.n_pix = s_rec[i][4];
            b.label = p.boxes[i].label;
            p.merged[k++] = b;
        }
        p.counters[DDHF_CNT_N_MERGED] = k;
    }
}

__global__ void __launch_bounds__(kMergeThreads) k_box_merge_pairs(CclParams p)
{
    __shared__ double s_cx[2][kMergeTile], s_cy[2][kMergeTile], s_m[2][kMergeTile];
    const int n = min(p.counters[DDHF_CNT_N_BOXES], p.max_boxes);
    if (n <= kMergeSmall) {
        if (blockIdx.x == 0) merge_small(p, n);
        return;
    }
    const int nt = (n + kMergeTile - 1) / kMergeTile;
    const int n_tiles = nt * (nt + 1) / 2;
    const double alpha = static_cast<double>(p.merge_alpha);
    for (int tile = blockIdx.x; tile < n_tiles; tile += gridDim.x) {
        // tile (ti, tj), ti <= tj, from the linear index tile = tj (tj + 1) / 2 + ti
        int tj = static_cast<int>((sqrt(8.0 * tile + 1.0) - 1.0) * 0.5);
        while (tj * (tj + 1) / 2 > tile) --tj;
        while ((tj + 1) * (tj + 2) / 2 <= tile) ++tj;
        const int ti = tile - tj * (tj + 1) / 2;
        __syncthreads();
        if (threadIdx.x < 2 * kMergeTile) {
            const int side = threadIdx.x / kMergeTile, k = threadIdx.x % kMergeTile;
            const int idx = (side ? tj : ti) * kMergeTile + k;
            if (idx < n) {
                const ddhf_box b = p.boxes[idx];
                s_cx[side][k] = 0.5 * (b.x0 + b.x1);
                s_cy[side][k] = 0.5 * (b.y0 + b.y1);
                s_m[side][k] = static_cast<double>(max(b.x1 - b.x0 + 1, b.y1 - b.y0 + 1));
            }
        }
        __syncthreads();
        for (int q = threadIdx.x; q < kMergeTile * kMergeTile; q += kMergeThreads) {
            const int a = q / kMergeTile, b = q % kMergeTile;
            const int i = ti * kMergeTile + a, j = tj * kMergeTile + b;
            if (i >= j || j >= n) continue;
            const double dx = s_cx[0][a] - s_cx[1][b], dy = s_cy[0][a] - s_cy[1][b];
            const double dist = sqrt(dx * dx + dy * dy);
            const double m = s_m[0][a] > s_m[1][b] ? s_m[0][a] : s_m[1][b];
            if (dist < alpha * m && uf_find(p.merge_parent, i) != uf_find(p.merge_parent, j))
                uf_union(p.merge_parent, i, j);
        }
    }
    // the last CTA to finish emits the roots in ascending index (= ascending label) with the union of
    // their members' boxes
    __shared__ int s_w[33];
    __shared__ bool s_last;
    __threadfence();
    __syncthreads();
    if (threadIdx.x == 0) s_last = (atomicAdd(p.merge_sync, 1) == static_cast<int>(gridDim.x) - 1);
    __syncthreads();
    if (!s_last) return;
    __threadfence();
    constexpr int NT = kMergeThreads;
    int *rec = p.merge_rec;
    for (int i = threadIdx.x; i < n; i += NT) {
        int *c = rec + 5 * i;
        c[0] = 0x7fffffff; c[1] = 0x7fffffff; c[2] = -1; c[3] = -1; c[4] = 0;
    }
    __syncthreads();
    for (int i = threadIdx.x; i < n; i += NT) {
        const int r = uf_find(p.merge_parent, i);
        const ddhf_box b = p.boxes[i];
        int *c = rec + 5 * r;
        atomicMin(c + 0, b.x0);
        atomicMin(c + 1, b.y0);
        atomicMax(c + 2, b.x1);
        atomicMax(c + 3, b.y1);
        atomicAdd(c + 4, b.n_pix);
    }
    __syncthreads();
    // ordered emit: thread t owns a contiguous range of box indices; exclusive scan of the root counts
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    const int per = (n + NT - 1) / NT;
    const int beg = min(threadIdx.x * per, n), end = min(beg + per, n);
    int cnt = 0;
    for (int i = beg; i < end; ++i) cnt += (__ldcg(p.merge_parent + i) >= i);
    int inc = cnt;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const int v = __shfl_up_sync(0xffffffffu, inc, o);
        if (lane >= o) inc += v;
    }
    if (lane == 31) s_w[wid] = inc;
    __syncthreads();
    if (wid == 0) {
        const int w = (lane < NT / 32) ? s_w[lane] : 0;
        int x = w;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const int v = __shfl_up_sync(0xffffffffu, x, o);
            if (lane >= o) x += v;
        }
        s_w[lane] = x - w;
        if (lane == 31) s_w[32] = x;
    }
    __syncthreads();
    int k = inc - cnt + s_w[wid];
    for (int i = beg; i < end; ++i) {
        if (__ldcg(p.merge_parent + i) < i) continue;
        const int *c = rec + 5 * i;
        ddhf_box b;
        b.x0 = c[0]; b.y0 = c[1]; b.x1 = c[2]; b.y1 = c[3]; b.n_pix = c[4];
        b.label = p.boxes[i].label;
        p.merged[k++] = b;
    }
    if (threadIdx.x == 0) p.counters[DDHF_CNT_N_MERGED] = s_w[32];
}

}  // namespace


int launch_ccl(const CclParams &p, cudaStream_t st)
{
    const int g256 = (p.np + 255) / 256;
    const int n_tiles = (p.np + kTile - 1) / kTile;
    int launches = 0;
    k_ccl_merge<<<g256, 256, 0, st>>>(p); ++launches;
    k_ccl_label<<<g256, 256, 0, st>>>(p); ++launches;
    k_ccl_boxes<<<n_tiles, 1024, 0, st>>>(p, n_tiles); ++launches;
    if (p.merged != nullptr) {
        const int nt = (p.max_boxes + kMergeTile - 1) / kMergeTile;
        const int pair_tiles = nt * (nt + 1) / 2;
        k_box_merge_pairs<<<pair_tiles < 296 ? pair_tiles : 296, kMergeThreads, 0, st>>>(p); ++launches;
    }
    return launches;
}

}  // namespace ddhf
