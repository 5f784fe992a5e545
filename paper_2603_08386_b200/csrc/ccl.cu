// ccl.cu -- a8: 8-connected component labelling of the detection mask, bounding boxes and
// the A_min filter ("We apply 8-connected component labeling to the boolean mask ... extract
// their bounding boxes.  Small boxes below the area threshold A_min are removed", PAPER.md
// L164).  Readings: R17 (area = bounding-box area), R18 (label = minimum linear pixel index of
// the component, boxes in ascending label order).
//
// Union-find with atomicMin so that the root of every tree is the smallest linear index of its
// component, which makes labels and box order deterministic.  The mask is at most 0.9 MB, so
// the stage is bound by launch latency, not by bandwidth: few, small kernels.
#include "ddhf_internal.cuh"

namespace ddhf {

namespace {

constexpr int kTile = 4096;      // 1024 threads x 4

__device__ __forceinline__ int uf_find(int *parent, int x)
{
    // find with path halving; parent[] only ever decreases, so concurrent halving is safe
    int p = *reinterpret_cast<volatile int *>(parent + x);
    while (p != x) {
        const int gp = *reinterpret_cast<volatile int *>(parent + p);
        if (gp != p) atomicMin(parent + x, gp);
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
        if (old == a) return;
        a = old;
    }
}

// Every mask pixel starts as a child of the first pixel of its horizontal run inside the
// warp's 32-pixel span (runs are cut at row starts), so the union-find trees start flat.
__global__ void k_ccl_init(CclParams p)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    const int lane = threadIdx.x & 31;
    const bool m = (i < p.np) && p.mask[i];
    const unsigned bits = __ballot_sync(0xffffffffu, m);
    const unsigned rs = __ballot_sync(0xffffffffu, (i % p.width) == 0);
    const unsigned starts = bits & (~(bits << 1) | rs | 1u);
    const unsigned upto = starts & (0xffffffffu >> (31 - lane));
    if (i < p.np) p.parent[i] = m ? i - (lane - (31 - __clz(upto))) : -1;
}

__global__ void k_ccl_merge(CclParams p)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= p.np || !p.mask[i]) return;
    const int x = i % p.width, y = i / p.width;
    // W: only where a run was cut at a span boundary
    if (x > 0 && p.mask[i - 1] && (threadIdx.x & 31) == 0) uf_union(p.parent, i, i - 1);
    if (y > 0) {
        const int up = i - p.width;
        if (p.mask[up]) {
            uf_union(p.parent, i, up);                    // N (NW and NE are then in N's run)
        } else {
            if (x > 0 && p.mask[up - 1]) uf_union(p.parent, i, up - 1);             // NW
            if (x + 1 < p.width && p.mask[up + 1]) uf_union(p.parent, i, up + 1);   // NE
        }
    }
}

__global__ void k_ccl_compress(CclParams p)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= p.np || !p.mask[i]) return;
    p.parent[i] = uf_find(p.parent, i);
}

// ---- ordered compaction (reduce / scan tiles / apply) over a flag per element -------------
__device__ __forceinline__ int block_scan1(int &a, int *s)
{
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    int ia = a;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const int t = __shfl_up_sync(0xffffffffu, ia, o);
        if (lane >= o) ia += t;
    }
    if (lane == 31) s[wid] = ia;
    __syncthreads();
    if (wid == 0) {
        const int w = s[lane];
        int x = w;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const int t = __shfl_up_sync(0xffffffffu, x, o);
            if (lane >= o) x += t;
        }
        s[lane] = x - w;
        if (lane == 31) s[32] = x;
    }
    __syncthreads();
    a = ia - a + s[wid];
    const int tot = s[32];
    __syncthreads();
    return tot;
}

// mode 0: flag = pixel is a root (parent[i] == i), n = np
// mode 1: flag = component passes A_min, n = number of components (device counter)
template <int MODE>
__device__ __forceinline__ int flag_of(const CclParams &p, int i, int n)
{
    if (i >= n) return 0;
    if (MODE == 0) return p.parent[i] == i;
    const int *c = p.comp + 5 * i;
    const long long area = static_cast<long long>(c[2] - c[0] + 1) * (c[3] - c[1] + 1);
    return area >= p.a_min;
}

template <int MODE>
__global__ void __launch_bounds__(1024) k_flag_reduce(CclParams p)
{
    __shared__ int s[33];
    const int n = MODE == 0 ? p.np : min(p.counters[DDHF_CNT_N_COMPONENTS], p.comp_cap);
    const int base = blockIdx.x * kTile + threadIdx.x * 4;
    if (blockIdx.x * kTile >= n) { if (threadIdx.x == 0) p.tile_sum[blockIdx.x] = 0; return; }
    int a = 0;
#pragma unroll
    for (int j = 0; j < 4; ++j) a += flag_of<MODE>(p, base + j, n);
    const int tot = block_scan1(a, s);
    if (threadIdx.x == 0) p.tile_sum[blockIdx.x] = tot;
}

template <int MODE>
__global__ void __launch_bounds__(1024) k_flag_tiles(CclParams p, int n_tiles)
{
    __shared__ int s[33];
    int a = threadIdx.x < n_tiles ? p.tile_sum[threadIdx.x] : 0;
    const int tot = block_scan1(a, s);
    if (threadIdx.x < n_tiles) p.tile_off[threadIdx.x] = a;
    if (threadIdx.x == 0) {
        if (MODE == 0) {
            p.counters[DDHF_CNT_N_COMPONENTS] = tot;
        } else {
            p.counters[DDHF_CNT_N_BOXES_TOTAL] = tot;
            p.counters[DDHF_CNT_N_BOXES] = min(tot, p.max_boxes);
            if (tot > p.max_boxes) atomicOr(&p.counters[DDHF_CNT_OVERFLOW], 2);
        }
    }
}

template <int MODE>
__global__ void __launch_bounds__(1024) k_flag_apply(CclParams p)
{
    __shared__ int s[33];
    const int n = MODE == 0 ? p.np : min(p.counters[DDHF_CNT_N_COMPONENTS], p.comp_cap);
    if (blockIdx.x * kTile >= n) return;
    const int base = blockIdx.x * kTile + threadIdx.x * 4;
    int f[4], a = 0;
#pragma unroll
    for (int j = 0; j < 4; ++j) { f[j] = flag_of<MODE>(p, base + j, n); a += f[j]; }
    block_scan1(a, s);
    int pos = p.tile_off[blockIdx.x] + a;
#pragma unroll
    for (int j = 0; j < 4; ++j) {
        if (!f[j]) continue;
        const int i = base + j;
        if (MODE == 0) {
            p.slot[i] = pos;
            if (pos < p.comp_cap) {
                p.comp_label[pos] = i;
                int *c = p.comp + 5 * pos;
                c[0] = 0x7fffffff; c[1] = 0x7fffffff; c[2] = -1; c[3] = -1; c[4] = 0;
            }
        } else if (pos < p.max_boxes) {
            const int *c = p.comp + 5 * i;
            ddhf_box b;
            b.x0 = c[0]; b.y0 = c[1]; b.x1 = c[2]; b.y1 = c[3]; b.n_pix = c[4];
            b.label = p.comp_label[i];
            p.boxes[pos] = b;
        }
        ++pos;
    }
}

__global__ void k_box_accum(CclParams p)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= p.np || !p.mask[i]) return;
    const int s = p.slot[p.parent[i]];
    if (s >= p.comp_cap) return;
    const int x = i % p.width, y = i / p.width;
    int *c = p.comp + 5 * s;
    atomicMin(c + 0, x);
    atomicMin(c + 1, y);
    atomicMax(c + 2, x);
    atomicMax(c + 3, y);
    atomicAdd(c + 4, 1);
}

}  // namespace

int launch_ccl(const CclParams &p, cudaStream_t st)
{
    const int g256 = (p.np + 255) / 256;
    const int n_tiles = (p.np + kTile - 1) / kTile;
    const int c_tiles = (p.comp_cap + kTile - 1) / kTile;
    int launches = 0;
    k_ccl_init<<<g256, 256, 0, st>>>(p); ++launches;
    k_ccl_merge<<<g256, 256, 0, st>>>(p); ++launches;
    k_ccl_compress<<<g256, 256, 0, st>>>(p); ++launches;
    k_flag_reduce<0><<<n_tiles, 1024, 0, st>>>(p); ++launches;
    k_flag_tiles<0><<<1, 1024, 0, st>>>(p, n_tiles); ++launches;
    k_flag_apply<0><<<n_tiles, 1024, 0, st>>>(p); ++launches;
    k_box_accum<<<g256, 256, 0, st>>>(p); ++launches;
    k_flag_reduce<1><<<c_tiles, 1024, 0, st>>>(p); ++launches;
    k_flag_tiles<1><<<1, 1024, 0, st>>>(p, c_tiles); ++launches;
    k_flag_apply<1><<<c_tiles, 1024, 0, st>>>(p); ++launches;
    return launches;
}

}  // namespace ddhf
