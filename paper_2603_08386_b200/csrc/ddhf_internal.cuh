// ddhf_internal.cuh -- shared declarations of the DDHF CUDA kernel sets (sm_100a).
// Product code: shares nothing with oracle/.
#pragma once

#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/ddhf.h"

namespace ddhf {

constexpr int kMaxHarm = 16;       // n_harm limit
constexpr int kMaxF0 = 256;        // n_f0 limit
constexpr int kMaxPieces = 64;     // pieces of <= 32 bins of one candidate's excluded set
constexpr int kNumClasses = 12;    // work-list size classes (by log2 of the row length)
constexpr int kScanTile = 4096;    // elements per scan tile (1024 threads x 4)

// One unit of NDFT work: an active pixel's CSR row.
struct __align__(16) WorkItem {
    int32_t row_begin;   // first slot in csr_ev
    int32_t n;           // events in the row
    int32_t pix;         // linear pixel index
    int32_t arow;        // row of the compact outputs (index into active_idx)
};

// Rows longer than kSplitMin events are split into segments of equal length (at most kSegEvents), one
// work item each, and their partial sums are combined along a tree of fan-in kSplitFan; see k_ndft_score.
// A segment's work item has pix = 0x80000000 | split row, arow = segment.
constexpr int kSplitMin = 4096;
constexpr int kSegEvents = 512;
constexpr int kSplitFan = 8;
constexpr int kMaxSegs = 1536;
struct __align__(16) SplitRow {
    int32_t pix, arow;           // the row's identity (arow: row of the compact outputs)
    int32_t n_seg;               // segments of the row = leaves of its tree
    int32_t seg_base;            // first partial of the row in NdftParams::split_partial (leaves, then level 1, ...)
    int32_t cnt_base;            // first arrival counter of the row in NdftParams::split_cnt (level 1, level 2, ...)
    int32_t _pad[3];
};
// partial slots / arrival counters of a row of n_seg segments (the root has a counter but no slot)
__host__ __device__ inline int split_slots(int n) { int s = 0; while (n > 1) { s += n; n = (n + kSplitFan - 1) / kSplitFan; } return s; }
__host__ __device__ inline int split_nodes(int n) { int c = 0; while (n > 1) { n = (n + kSplitFan - 1) / kSplitFan; c += n; } return c; }

// Constants of the SF / comb stages (a5-a7) and the per-candidate tables, built on the host at create
// time (readings R7-R10).  Tables are padded to `cpad` candidates (a multiple of 32) so that a warp
// reads them without range checks; layout [row][cpad], candidate fastest (coalesced per lane).
struct CombParams {
    int32_t n_freq, k_lo, n_f0, n_harm, half_bw;
    int32_t s_lvl;               // block maxima of 2^s_lvl bins, 2^s_lvl <= min(2 half_bw + 1, 32)
    int32_t r0, r1;              // full-spectrum rank band that holds every complement median
    int32_t cpad, max_pieces;
    float tau_sf, tau_comb, sf_eps;
    int32_t score_all;
    const uint32_t *num_tab;     // DEVICE [n_harm][cpad]: padded indices of the two block maxima that cover the
                                 // window of harmonic m (lo | hi << 16); 0 beyond M_valid
    const uint2 *piece_tab;      // DEVICE [max_pieces][cpad]: the union of the windows in pieces of <= 32 bins,
                                 // {mask of the piece's length, first bin}; mask 0 beyond the candidate's pieces
    const uint4 *meta;           // DEVICE [cpad]: {M_valid | n_pieces << 16, rank of the lower median in the
                                 // complement | n_excl << 16, float bits of 1 / M_valid, 0}; M_valid 0 = skipped
};
typedef CombParams ScoreParams;

// One row of the deferred-scoring queue (a pixel that passed the SF filter).
struct __align__(16) SpillRec {
    int32_t pix;
    int32_t arow;
    float mean_p;        // mean of the floored spectrum over [k_lo, n_freq): seed of the band search
    int32_t _pad;
};

struct NdftParams {
    const WorkItem *work;        // DEVICE [n_active] ordered by descending size class
    const uint32_t *csr_ev;
    const int32_t *counters;
    const int32_t *n_work;       // DEVICE: work items = active pixels + extra segments of split rows
    const SplitRow *split_tab;   // rows longer than kSplitMin events
    float *split_partial;        // [slots][2 * padded bins] partial (S1..S4) sums of the segments and tree nodes
    int32_t *split_cnt;          // arrival counters of the tree nodes (zeroed when the row is split)
    unsigned long long *work_cursor;   // dynamic work queue: items taken from the head (hi 32) / tail (lo 32)
    int32_t max_active;
    uint64_t g_f0, g_d, g_h;     // 2^64 * f * 1e-6 for: centre base, df, 16*df
    float *power;                // optional compact spectra
    float *sf, *score;
    int32_t *f0_idx;
    uint8_t *mask;
    float *comb_debug;
    int32_t *n_scored;
    // deferred comb scoring: spectra of the pixels to score are queued and scored by k_comb_deferred
    float *spill;                // [spill_cap][padded n_freq]
    SpillRec *spill_rec;         // [spill_cap]
    int32_t *spill_count;        // [0] rows requested (may exceed spill_cap: the excess is scored in place), [1] rows taken by k_comb_deferred
    int32_t spill_cap;
    ScoreParams sp;
};

// The NUFFT path for long rows (nufft.cu): the rows of the hot list, one warp each
struct NufftParams {
    NdftParams nd;               // csr_ev, outputs, scoring queue and constants, as for k_ndft_score
    const WorkItem *hot;         // DEVICE [*n_hot] rows (unordered)
    const int32_t *n_hot;
    int32_t *cursor;             // rows handed out
    uint64_t g_c, g_t;           // 2^64 1e-6 x: -(f_min + 1024 df) (mod 2^64), df
    float *scratch;              // [warps of the grid][2048] the row in bin order
};

struct IngestParams {
    const ddhf_event *events;    // 16-byte events, or (packed) ddhf_event8 records through the same pointer
    int32_t packed;
    int64_t t_base;              // packed: t = t_base + dt_us
    int64_t n;
    int64_t t0, t1;              // window [t0, t1)
    int32_t width, height, np;
    int32_t n_min, max_active;
    int32_t *cnt;                // [np] per-pixel histogram
    int32_t *row_ptr;            // [np+1]
    uint32_t *csr_ev;
    // stable two-level sort on pixel = bucket << bl | low (ingest.cu)
    int32_t bl, vb;              // low-digit bits; value bits of a compact item (32 - bl)
    int32_t nb, hbits;           // buckets (<= 1023); bits of the tile sort digit (holds nb + 1 values)
    int32_t compact;             // items of 4 bytes (low << vb | value): 2 * window < 2^vb
    void *items;                 // [ev_tiles][tile stride] 4- or 8-byte items: every tile sorted by bucket, runs 16-byte aligned
    void *scratch;               // [max_events] sorted chunks of the buckets that need more than one
    uint32_t *run_tab;           // [ev_tiles][nb] run of every bucket inside its tile: first item | length << 16
    int32_t *bkt_order;          // [nb] buckets by descending size class
    int32_t *bkt_act;            // [nb] active pixels (count >= n_min) of every bucket
    int32_t *bkt_maxrun;         // [nb + 2] longest run of the bucket in one tile
    int32_t *giant_of;           // [nb + 2] index into giant_tab, -1: the bucket is sorted by its own CTA
    void *giant_tab;             // [nb] GiantBucket (ingest.cu)
    int32_t giant_row0, giant_rows;   // chunk rows reserved for giant buckets: first row, count
    int32_t *bkt_total, *bkt_base;   // [nb + 2] events per bucket; exclusive scan (bkt_base[nb] = n_in)
    int32_t *chunk_rows;         // [max_rows][4 + 2^bl] chunk table of the multi-chunk buckets
    int32_t *sync;               // [16] 0: tiles finished, 1: chunk rows handed out, 2-3: scoring queue counts,
                                 //     4: work items, 5: split rows, 6: partials, 7: arrival counters handed out, 8: box-merge CTAs finished,
                                 //     9: items of the segment list, 10: giant buckets, 11: their chunks, 12-13: chunk tickets of
                                 //     k_bucket_sort / k_worklist, 14: giant chunk rows handed out, 15: rows of the hot list
    SplitRow *split_tab;         // rows longer than kSplitMin (see NdftParams)
    int32_t *split_cnt;
    WorkItem *seg_work;          // when set: the segments of split rows go to this list (count in sync[9]) instead of `work`
    unsigned long long *work_cursor2;   // cursor of the segment pass
    WorkItem *hot_work;          // when set: unsplit rows of >= hot_min events go to this list (count in sync[15]), for k_nufft_score
    int32_t hot_min;
    int32_t *hot_cursor;         // rows of the hot list handed out (zeroed by k_init)
    // sliding windows (ddhf_window_slide): NULL otherwise
    const int32_t *prev_row_ptr; // [np + 1] CSR of the previous window (workspace copy)
    const uint32_t *prev_csr;
    int32_t *next_row_ptr;       // [np + 1] copy of this window's CSR for the next call
    uint32_t *next_csr;
    int32_t *slab_row_ptr;       // [np] row starts of the new slab's own CSR
    uint32_t *slab_csr;          // [max_events]
    uint32_t shift2;             // 2 (t0 - previous t0): values below it have left the window
    int32_t csr_cap;             // max_events: a sliding window that outgrows it is truncated and flagged
    int32_t *active_idx;
    WorkItem *work;
    int32_t *tile_sum, *tile_act;   // [n_tiles]
    int32_t *tile_off, *tile_aoff;  // [n_tiles]
    int32_t *class_cnt;             // [kNumClasses] counts, then bases
    int32_t *class_cur;             // [kNumClasses] cursors
    int32_t *counters;
    float *sf, *score;           // per-pixel maps initialised for inactive pixels
    int32_t *f0_idx;
    uint8_t *mask;
    unsigned long long *work_cursor;
    int32_t *ccl_parent;         // [np] union-find array of the CCL stage, reset here
    int32_t *ccl_tile_state;     // [1025] chained tile counts of k_ccl_boxes, zeroed here
};

struct CclParams {
    const uint8_t *mask;
    int32_t width, height, np;
    int32_t a_min, max_boxes;
    int32_t *parent;             // [np] = labels output or workspace; arrives filled with INT_MAX
    int32_t *rec;                // [np][5] x0,y0,x1,y1,n of the component rooted at the pixel (mask pixels only)
    int32_t *tile_state;         // [1024 + 1] per tile of 4096 pixels: passing boxes << 1 | published; [1024]: tickets (zeroed by k_init)
    ddhf_box *boxes;
    int32_t *counters;
    ddhf_box *merged;            // optional: eq. 12 detections
    int32_t *merge_parent;       // [max_boxes] union-find over box indices (eq. 12), set by k_ccl_emit
    int32_t *merge_rec;          // [max_boxes][5] merged box records
    int32_t *merge_sync;         // CTAs of k_box_merge_pairs that have finished (zeroed by the ingest stage)
    float merge_alpha;
};

// kernel-set entry points (host functions that enqueue on `st`); each returns the number
// of kernels it launched
int launch_ingest(const IngestParams &p, cudaStream_t st);
int launch_ingest_slide(const IngestParams &p, cudaStream_t st);   // p.events = the new slab; previous CSR in p.prev_*
cudaError_t ingest_configure();              // opt in to large dynamic shared memory
int ingest_tile_events();                    // events per sort tile
int ingest_tile_stride(bool compact);        // items per tile slot of IngestParams::items (run padding included)
size_t ingest_tile_smem(bool compact);       // dynamic shared memory of k_tile_sort
void ingest_plan(int np, int *bl, int *nb, int *hbits);   // digit split for a sensor of np pixels
int launch_ndft(const NdftParams &p, const NdftParams *seg_pass, int n_freq, int band_size, bool fallback, int grid_ndft, int grid_seg,
                int grid_score, cudaStream_t st, cudaEvent_t between);
                                             // fallback: the full kernel variant (scores a pixel itself when the queue is full, combines
                                             // split rows); else the lean variant, followed by the full one on `seg_pass` (the segment list)
                                             // `between` (optional) is recorded after the NDFT kernel, before the scoring kernel
int launch_ccl(const CclParams &p, cudaStream_t st);
bool nufft_supported(int n_freq);            // frequency grids the NUFFT path is built for (1024 < n_freq <= 2048)
bool nufft_window_fits(double df_hz, int64_t window_us);   // the window's events stay inside the quarter turn the path holds
size_t nufft_smem_bytes();
int nufft_warps();                           // warps per CTA of k_nufft_score (one scratch row each)
cudaError_t nufft_configure();               // tables and shared-memory opt-in on the current device
int launch_nufft(const NufftParams &q, int grid, cudaStream_t st);
int ndft_bins_per_lane(int n_freq);          // 8, 16, 32 or 64
int ndft_tn(int n_freq);                     // offset pairs per centre for that kernel
int ndft_padded_bins(int n_freq);            // row length of the deferred-scoring queue
int ndft_band_size(int n_freq, int r0, int r1);   // sort capacity needed, 0 if unsupported
cudaError_t ndft_configure(int n_freq, int band_size, int cpad, bool fallback, int *blocks_per_sm, int *full_blocks_per_sm,
                           int *score_blocks_per_sm);
                                             // opt in to the kernels' dynamic shared memory on the current device
bool ndft_scores_in_place(int n_freq, int band_size);   // whether the NDFT kernel can score a pixel itself when the queue is full

}  // namespace ddhf
