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
//   k_ccl_count     per tile of 4096 pixels: roots, and roots whose box passes A_min
//   k_ccl_emit      ordered compaction of the passing roots into boxes[] (ascending label)
//   k_box_merge     (optional) eq. 12: boxes with close centres merged into the final detections
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
    if (i >= p.np) return;
    if (!p.mask[i]) { p.parent[i] = -1; return; }
    const int r = uf_find(p.parent, i);
    p.parent[i] = r;
    const int x = i % p.width, y = i / p.width;
    int *c = p.rec + 5 * static_cast<size_t>(r);
    atomicMin(c + 0, x);
    atomicMin(c + 1, y);
    atomicMax(c + 2, x);
    atomicMax(c + 3, y);
    atomicAdd(c + 4, 1);
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

__global__ void __launch_bounds__(1024) k_ccl_count(CclParams p)
{
    __shared__ int s[33];
    const int base = blockIdx.x * kTile + threadIdx.x * 4;
    int roots = 0, pass = 0;
#pragma unroll
    for (int j = 0; j < 4; ++j) {
        const int f = root_flags(p, base + j);
        roots += f & 1;
        pass += f >> 1;
    }
    const int tr = block_sum(roots, s);
    const int tp = block_sum(pass, s);
    if (threadIdx.x == 0) {
        p.tile_sum[blockIdx.x] = tp;
        if (tr) atomicAdd(&p.counters[DDHF_CNT_N_COMPONENTS], tr);
    }
}

__global__ void __launch_bounds__(1024) k_ccl_emit(CclParams p, int n_tiles)
{
    __shared__ int s[33];
    __shared__ int s_scan[33];
    // boxes before this tile, and (block 0) the total
    int before = 0, total = 0;
    for (int t = threadIdx.x; t < n_tiles; t += 1024) {
        const int v = p.tile_sum[t];
        total += v;
        if (t < static_cast<int>(blockIdx.x)) before += v;
    }
    before = block_sum(before, s);
    if (blockIdx.x == 0) {
        total = block_sum(total, s);
        if (threadIdx.x == 0) {
            p.counters[DDHF_CNT_N_BOXES_TOTAL] = total;
            p.counters[DDHF_CNT_N_BOXES] = min(total, p.max_boxes);
            if (total > p.max_boxes) atomicOr(&p.counters[DDHF_CNT_OVERFLOW], 2);
        }
    }
    if (p.tile_sum[blockIdx.x] == 0) return;
    const int base = blockIdx.x * kTile + threadIdx.x * 4;
    int f[4], a = 0;
#pragma unroll
    for (int j = 0; j < 4; ++j) { f[j] = root_flags(p, base + j) >> 1; a += f[j]; }
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
        }
        ++pos;
    }
}

// ---- a9: box merge, eq. 12 ---------------------------------------------------
// "two boxes ... are merged if dist(c1, c2) < alpha max(w1, h1, w2, h2)".  Readings R27-R29: box
// centres, the rule evaluated on the boxes that entered the step, merging transitive.  A handful of
// boxes: one CTA, union-find over box indices in shared memory (root = smallest index = smallest
// label, since boxes[] is ascending by label), all pairs tested in double precision with the same
// expression as the oracle.
constexpr int kMergeThreads = 256;

__device__ __forceinline__ int mg_find(volatile int *par, int x)
{
    int p = par[x];
    while (p != x) { x = p; p = par[x]; }
    return x;
}

__global__ void __launch_bounds__(kMergeThreads) k_box_merge(CclParams p)
{
    extern __shared__ int s_par[];                       // [n] parents, then [n][5] merged records
    __shared__ int s_out;
    const int n = min(p.counters[DDHF_CNT_N_BOXES], p.max_boxes);
    int *s_rec = s_par + n;
    for (int i = threadIdx.x; i < n; i += kMergeThreads) s_par[i] = i;
    if (threadIdx.x == 0) s_out = 0;
    __syncthreads();
    const double alpha = static_cast<double>(p.merge_alpha);
    const long long n_pairs = static_cast<long long>(n) * (n - 1) / 2;
    for (long long q = threadIdx.x; q < n_pairs; q += kMergeThreads) {
        // pair (i, j), i < j, from the linear index q = j (j - 1) / 2 + i
        int j = static_cast<int>((1.0 + sqrt(1.0 + 8.0 * static_cast<double>(q))) * 0.5);
        while (static_cast<long long>(j) * (j - 1) / 2 > q) --j;
        while (static_cast<long long>(j + 1) * j / 2 <= q) ++j;
        const int i = static_cast<int>(q - static_cast<long long>(j) * (j - 1) / 2);
        const ddhf_box a = p.boxes[i], b = p.boxes[j];
        const double cxa = 0.5 * (a.x0 + a.x1), cya = 0.5 * (a.y0 + a.y1);
        const double cxb = 0.5 * (b.x0 + b.x1), cyb = 0.5 * (b.y0 + b.y1);
        const double dist = sqrt((cxa - cxb) * (cxa - cxb) + (cya - cyb) * (cya - cyb));
        double m = a.x1 - a.x0 + 1;
        if (a.y1 - a.y0 + 1 > m) m = a.y1 - a.y0 + 1;
        if (b.x1 - b.x0 + 1 > m) m = b.x1 - b.x0 + 1;
        if (b.y1 - b.y0 + 1 > m) m = b.y1 - b.y0 + 1;
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
        int *c = s_rec + 5 * i;
        c[0] = 0x7fffffff; c[1] = 0x7fffffff; c[2] = -1; c[3] = -1; c[4] = 0;
    }
    __syncthreads();
    for (int i = threadIdx.x; i < n; i += kMergeThreads) {
        const int r = mg_find(s_par, i);
        const ddhf_box b = p.boxes[i];
        int *c = s_rec + 5 * r;
        atomicMin(c + 0, b.x0);
        atomicMin(c + 1, b.y0);
        atomicMax(c + 2, b.x1);
        atomicMax(c + 3, b.y1);
        atomicAdd(c + 4, b.n_pix);
    }
    __syncthreads();
    // ordered emit: roots in ascending index (= ascending label); one thread walks them (n is small)
    if (threadIdx.x == 0) {
        int k = 0;
        for (int i = 0; i < n; ++i) {
            if (s_par[i] != i) continue;
            const int *c = s_rec + 5 * i;
            ddhf_box b;
            b.x0 = c[0]; b.y0 = c[1]; b.x1 = c[2]; b.y1 = c[3]; b.n_pix = c[4];
            b.label = p.boxes[i].label;
            p.merged[k++] = b;
        }
        p.counters[DDHF_CNT_N_MERGED] = k;
    }
}

}  // namespace

cudaError_t ccl_configure(int max_boxes)
{
    return cudaFuncSetAttribute(k_box_merge, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                static_cast<int>(static_cast<size_t>(max_boxes) * 6 * sizeof(int)));
}

int launch_ccl(const CclParams &p, cudaStream_t st)
{
    const int g256 = (p.np + 255) / 256;
    const int n_tiles = (p.np + kTile - 1) / kTile;
    int launches = 0;
    k_ccl_merge<<<g256, 256, 0, st>>>(p); ++launches;
    k_ccl_label<<<g256, 256, 0, st>>>(p); ++launches;
    k_ccl_count<<<n_tiles, 1024, 0, st>>>(p); ++launches;
    k_ccl_emit<<<n_tiles, 1024, 0, st>>>(p, n_tiles); ++launches;
    if (p.merged != nullptr) {
        k_box_merge<<<1, kMergeThreads, static_cast<size_t>(p.max_boxes) * 6 * sizeof(int), st>>>(p); ++launches;
    }
    return launches;
}

}  // namespace ddhf
