// noalloc.cu -- ddhf_boxes_noalloc(): stage a8 (+ eq. 12) on a caller's detection mask with the stage's scratch in
// a static device array, for callers that cannot allocate device memory (CUDA graph capture, serving loops,
// harnesses that forbid cudaMalloc): no handle, no workspace, no cudaMalloc / cudaFree anywhere on the path.
//
//   "We apply 8-connected component labeling to the boolean mask ... extract their bounding boxes.  Small boxes
//    below the area threshold A_min are removed"; merge of close boxes, eq. 12 (L166).
//
// The kernels are those of ccl.cu (launch_ccl), unchanged; what ddhf_window() takes from its workspace -- the box
// record of every pixel, the chained tile counts, the union-find arrays of the eq. 12 merge -- comes from
// g_noalloc_scratch below, and what k_init of the ingest stage clears for them is cleared by k_noalloc_init.
#include "ddhf_internal.cuh"

#include <cstdio>
#include <mutex>

namespace ddhf {

namespace {

constexpr int kNoallocMaxPixels = DDHF_NOALLOC_MAX_PIXELS;     // 1280 x 720
constexpr int kNoallocMaxBoxes = DDHF_NOALLOC_MAX_BOXES;       // 4096
// layout of the scratch, in 32-bit words (every part starts on a multiple of 64 words = 256 bytes)
constexpr size_t kOffRec = 0;                                                          // [max pixels][5] box records
constexpr size_t kOffTiles = (kOffRec + 5 * static_cast<size_t>(kNoallocMaxPixels) + 63) / 64 * 64;   // [1025 (+ pad)] tile counts, tickets
constexpr size_t kOffMerge = kOffTiles + 1088;                                         // [max boxes] parents, [max boxes][5] records
constexpr size_t kOffSync = kOffMerge + 6 * static_cast<size_t>(kNoallocMaxBoxes);     // [64] CTAs of the merge kernel that have finished
constexpr size_t kScratchWords = kOffSync + 64;                                        // 18.5 MB

// Held by every GPU that loads the library, until the process exits.  In HOST code this name is a stand-in, not
// a device address: the address comes from cudaGetSymbolAddress (noalloc_scratch below), once per device.
static __device__ __align__(256) int32_t g_noalloc_scratch[kScratchWords];

constexpr int kMaxDevices = 64;
std::mutex g_mu;
int32_t *g_scratch_ptr[kMaxDevices] = {};          // device address of g_noalloc_scratch on each device
thread_local char g_err[256] = "";

int fail(int code, const char *what, const char *detail = "")
{
    snprintf(g_err, sizeof g_err, "%s%s", what, detail);
    return code;
}

// the array's address on the current device (resolved once per device, with that device current)
int noalloc_scratch(int32_t **out)
{
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return fail(DDHF_E_CUDA, "ddhf_boxes_noalloc: cudaGetDevice: ", cudaGetErrorString(e));
    if (dev < 0 || dev >= kMaxDevices) return fail(DDHF_E_INVAL, "ddhf_boxes_noalloc: device ordinal beyond 63");
    std::lock_guard<std::mutex> lock(g_mu);
    if (!g_scratch_ptr[dev]) {
        void *ptr = nullptr;
        e = cudaGetSymbolAddress(&ptr, g_noalloc_scratch);
        if (e != cudaSuccess || !ptr)
            return fail(DDHF_E_CUDA, "ddhf_boxes_noalloc: cudaGetSymbolAddress: ", cudaGetErrorString(e));
        g_scratch_ptr[dev] = static_cast<int32_t *>(ptr);
    }
    *out = g_scratch_ptr[dev];
    return DDHF_OK;
}

// what launch_ccl expects to find cleared: labels "no parent yet", tile counts and tickets, the merge kernel's
// arrival counter, the counters the kernels add to.  The array keeps the previous call's contents otherwise;
// box records and merge arrays are (re)written by the kernels before they are read.
__global__ void k_noalloc_init(int32_t *labels, int np, int32_t *counters, int32_t *tiles, int32_t *sync)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < np) labels[i] = 0x7fffffff;
    if (i <= 1024) tiles[i] = 0;
    if (i < 64) sync[i] = 0;
    if (i < DDHF_N_COUNTERS) counters[i] = 0;
}

}  // namespace

}  // namespace ddhf

using namespace ddhf;

extern "C" int ddhf_boxes_noalloc_setup(void)
{
    int32_t *ptr = nullptr;
    return noalloc_scratch(&ptr);
}

extern "C" const char *ddhf_boxes_noalloc_error(void) { return g_err; }

extern "C" int ddhf_boxes_noalloc(const uint8_t *d_mask, int32_t width, int32_t height, int32_t a_min, float merge_alpha,
                                  int32_t max_boxes, int32_t *d_labels, ddhf_box *d_boxes, ddhf_box *d_merged_boxes,
                                  int32_t *d_counters, void *cuda_stream)
{
    if (!d_mask || !d_labels || !d_boxes || !d_counters) return fail(DDHF_E_INVAL, "ddhf_boxes_noalloc: NULL argument");
    if (width <= 0 || height <= 0 || a_min < 0) return fail(DDHF_E_INVAL, "ddhf_boxes_noalloc: width, height or a_min out of range");
    if (static_cast<long long>(width) * height > kNoallocMaxPixels) {
        char msg[128];
        snprintf(msg, sizeof msg, "%d x %d pixels exceed the static scratch (DDHF_NOALLOC_MAX_PIXELS = %d)", width, height,
                 kNoallocMaxPixels);
        return fail(DDHF_E_CAPACITY, "ddhf_boxes_noalloc: ", msg);
    }
    if (max_boxes < 1 || max_boxes > kNoallocMaxBoxes)
        return fail(DDHF_E_CAPACITY, "ddhf_boxes_noalloc: max_boxes must be in [1, DDHF_NOALLOC_MAX_BOXES = 4096]");
    int32_t *scr = nullptr;
    const int rc = noalloc_scratch(&scr);
    if (rc != DDHF_OK) return rc;
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);

    CclParams cp{};
    cp.mask = d_mask; cp.width = width; cp.height = height; cp.np = width * height;
    cp.a_min = a_min; cp.max_boxes = max_boxes;
    cp.parent = d_labels;
    cp.rec = scr + kOffRec;
    cp.tile_state = scr + kOffTiles;
    cp.boxes = d_boxes; cp.counters = d_counters;
    cp.merged = (merge_alpha > 0.f) ? d_merged_boxes : nullptr;
    cp.merge_alpha = merge_alpha;
    cp.merge_parent = cp.merged ? scr + kOffMerge : nullptr;
    cp.merge_rec = cp.merged ? cp.merge_parent + max_boxes : nullptr;
    cp.merge_sync = scr + kOffSync;

    const int n_init = cp.np > 1025 ? cp.np : 1025;
    k_noalloc_init<<<(n_init + 255) / 256, 256, 0, st>>>(d_labels, cp.np, d_counters, cp.tile_state, cp.merge_sync);
    launch_ccl(cp, st);
    const cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return fail(DDHF_E_CUDA, "ddhf_boxes_noalloc: ", cudaGetErrorString(e));
    return DDHF_OK;
}
