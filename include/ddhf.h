/*
 * ddhf.h -- C ABI of the DDHF hot path for NVIDIA B200 (sm_100a).
 *
 * DDHF = "Drone Detection via Harmonic Fingerprinting", arXiv 2603.08386.  Citations
 * below are PAPER.md line numbers ("L93") with the equation or section they fall in;
 * "R<n>" is reading n of DESIGN.md section 3, taken where the paper is silent.
 *
 * One call, ddhf_window(), runs the whole per-window path of the paper's section 3.5 on
 * one GPU, entirely in hand-written CUDA kernels (there is no CPU fallback):
 *
 *   a0-a3  ingest: keep events inside [t0, t0+window) and the sensor, bucket them per
 *          pixel into CSR form, stable in input order            ("sorted by pixel index", L137)
 *   a4     per active pixel (>= n_min events, L137) the Non-uniform DFT power spectrum
 *          P_j = | sum_k w_k exp(-2 pi i f_j t_k) |^2,  w_k = +-1  (eq. 6)
 *   a5     spectral flatness SF = geometric / arithmetic mean of P (eq. 7)
 *   a6     median-normalised harmonic comb SNR_M over the f0 candidates, its maximum and
 *          argmax                                                 (eq. 8-11)
 *   a7     mask = active and SF <= tau_sf and max SNR_M >= tau_comb      (L107, L131, L139)
 *   a8     8-connected components of the mask, bounding boxes, A_min filter      (L164)
 *   a9     boxes whose centres are closer than alpha x their largest side are merged
 *          into the final detections                                  (eq. 12)
 *
 * Conventions
 *   - Every function returns 0 (DDHF_OK) or a negative DDHF_E_* code; nothing throws
 *     across the ABI.  ddhf_last_error() gives the text for the last failure on a handle.
 *   - Pointers are marked DEVICE or HOST.  The caller owns every buffer (events,
 *     workspace, outputs); the handle owns only small constant tables, per-stage CUDA
 *     events and, for ddhf_window_host(), its own staging buffers.
 *   - ddhf_window() only enqueues work on the given CUDA stream and never synchronises;
 *     outputs are valid once the stream has been synchronised by the caller.
 *   - Data-dependent conditions cannot be returned synchronously; they are counted on
 *     the device in ddhf_outputs.counters.
 */
#ifndef DDHF_H
#define DDHF_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define DDHF_OK            0
#define DDHF_E_INVAL      (-1)   /* bad argument or unsupported configuration            */
#define DDHF_E_CAPACITY   (-2)   /* n > max_events                                       */
#define DDHF_E_CUDA       (-3)   /* a CUDA runtime call failed (text in ddhf_last_error) */
#define DDHF_E_NOMEM      (-4)

/* ddhf_config.flags */
#define DDHF_FLAG_SCORE_ALL   1u  /* comb score on every active pixel (R14); default is the
                                     paper's order: only where SF <= tau_sf (L139)        */
#define DDHF_FLAG_TIMING      2u  /* record per-stage CUDA events (ddhf_stage_ms)          */
#define DDHF_FLAG_NUFFT       4u  /* spectra of long rows by a type-1 non-uniform FFT (footnote 1:
                                     "NUFFTs [22] offer asymptotic acceleration for large sample counts") instead
                                     of the direct sum of eq. 6.  Rows of at least (flags >> 16) events take it
                                     (0: DDHF_NUFFT_MIN_DEFAULT); longer than 4096 events they are split and
                                     summed directly as always.  Approximate: spreading on a 2x oversampled
                                     grid with an 8-cell kernel, aliasing error <= 1e-6 of sum |w| in amplitude,
                                     i.e. far inside the 1e-3-of-peak power tolerance of the direct path; the
                                     cost of such a row does not depend on its length.  Honoured only where it
                                     applies: 1024 < n_freq <= 2048, one queue row per pixel (max_scored = 0
                                     default), and windows with df_hz * window <= 0.24 (events within a quarter
                                     turn of the finest grid phase); otherwise the call runs the direct path. */
#define DDHF_NUFFT_MIN_DEFAULT 64

/* indices into ddhf_outputs.counters (int32[DDHF_N_COUNTERS]) */
#define DDHF_CNT_N_IN          0  /* events kept (inside window and sensor)                */
#define DDHF_CNT_N_DROPPED     1  /* events outside [t0, t0+window) or the sensor (R19)    */
#define DDHF_CNT_N_ACTIVE      2  /* pixels with >= n_min events (before truncation)       */
#define DDHF_CNT_N_BOXES       3  /* boxes written (<= max_boxes)                          */
#define DDHF_CNT_N_BOXES_TOTAL 4  /* components that passed A_min                          */
#define DDHF_CNT_OVERFLOW      5  /* bit 0: n_active > max_active, bit 1: boxes > max_boxes,
                                     bit 2: sliding window > max_events                   */
#define DDHF_CNT_N_SCORED      6  /* active pixels on which the comb score was evaluated   */
#define DDHF_CNT_N_COMPONENTS  7  /* connected components before the A_min filter          */
#define DDHF_CNT_N_MERGED      8  /* detections written to merged_boxes (eq. 12)           */
#define DDHF_CNT_N_GIANT       9  /* buckets of the ingest sort that were cut into chunks for
                                     several CTAs (> 65536 events in 2^bL pixels)          */
#define DDHF_N_COUNTERS        16 /* 10..15 reserved, written as 0                         */

/* Event tuple (x, y, p, t) of a temporal-contrast sensor (L55).  16 bytes. */
typedef struct {
    uint16_t x, y;       /* pixel coordinates                                             */
    int16_t  p;          /* polarity: > 0 is mapped to w = +1, anything else to -1 (L139)  */
    uint16_t _pad;
    int64_t  t_us;       /* timestamp in microseconds                                      */
} ddhf_event;

/* The same tuple in 8 bytes, for streams that cross PCIe every window: coordinates as above, the polarity in
 * bit 15 of y_p (1: w = +1, 0: w = -1; sensors are < 32768 rows), the timestamp as an offset in microseconds
 * from a base time that is passed with the call (71 minutes of range).  No information is lost: t = t_base_us
 * + dt_us, and every result is bit-identical to the 16-byte form (the CSR value is (t - t0) << 1 | polarity). */
typedef struct {
    uint16_t x;
    uint16_t y_p;        /* y | (p > 0) << 15                                              */
    uint32_t dt_us;      /* t_us - t_base_us                                               */
} ddhf_event8;

/* Bounding box of one connected component, inclusive corners. */
typedef struct {
    int32_t x0, y0, x1, y1;
    int32_t n_pix;       /* pixels in the component                                        */
    int32_t label;       /* minimum linear pixel index (y*width + x) of the component (R18) */
} ddhf_box;

typedef struct {
    int32_t width, height;          /* sensor W x H; pixel index = y*width + x            */
    double  f_min_hz, df_hz;        /* frequency grid f_j = f_min + j*df, j < n_freq (R3);
                                       the paper's integer modes are f_min = 0, df = 1/window */
    int32_t n_freq;                 /* 8 <= n_freq <= 2048                                */
    double  f0_min_hz, f0_step_hz;  /* fundamental candidates f0_c = f0_min + c*step (R12) */
    int32_t n_f0;                   /* 1 <= n_f0 <= 256                                   */
    int32_t n_harm;                 /* M of eq. 8, Table 2; <= 16                    */
    int32_t half_bw_bins;           /* d_k of eq. 8 in bins, Table 2                 */
    int32_t h_min;                  /* min matched harmonics, L115 / Table 2         */
    int32_t n_min;                  /* min events per active pixel, L137 / Table 2   */
    int32_t a_min;                  /* min bounding-box area in px, L164 / Table 2   */
    float   merge_alpha;            /* alpha of eq. 12 (L166, Table 2: 19.05); <= 0
                                       leaves merged_boxes untouched                       */
    float   tau_sf, tau_comb;       /* thresholds, L107 / L131                            */
    float   sf_eps;                 /* floor under log P and under the median (R6, R11)   */
    int32_t k_lo;                   /* first bin used by SF and the comb (R6)             */
    int64_t max_events;             /* capacity: events per window                        */
    int32_t max_active;             /* capacity: rows of the compact power output         */
    int32_t max_boxes;              /* capacity: boxes                                    */
    int32_t max_scored;             /* capacity (rows of n_freq floats) of the deferred comb-
                                       scoring queue in the workspace; 0 = one row per pixel
                                       if that is below 1/16 of the device memory (the NDFT
                                       kernel then runs its lean variant), else min(NP, 32768).
                                       Pixels beyond it are scored in place: same results   */
    uint32_t flags;                 /* DDHF_FLAG_*                                        */
} ddhf_config;

/* Outputs of one window.  All DEVICE pointers, allocated by the caller, sizes fixed by the
 * config (NP = width*height).  Pointers marked optional may be NULL. */
typedef struct {
    int32_t  *row_ptr;     /* [NP+1]  CSR row starts; row p holds pixel p's events          */
    uint32_t *csr_ev;      /* [max_events]  (t - t0) << 1 | (p > 0), input order per row    */
    int32_t  *active_idx;  /* [max_active]  ascending pixel indices with >= n_min events    */
    float    *power;       /* optional [max_active * n_freq]  row r <-> active_idx[r]       */
    float    *sf;          /* [NP]  spectral flatness, NaN where the pixel is not active    */
    float    *score;       /* [NP]  max_c SNR_M, 0 where not evaluated                      */
    int32_t  *f0_idx;      /* [NP]  argmax candidate (first maximum), -1 where none         */
    uint8_t  *mask;        /* [NP]  detection mask                                          */
    int32_t  *labels;      /* optional [NP]  component label (min linear index), -1 off-mask */
    ddhf_box *boxes;       /* [max_boxes]  boxes that passed A_min, ascending label         */
    int32_t  *counters;    /* [DDHF_N_COUNTERS]                                             */
    ddhf_box *merged_boxes;/* optional [max_boxes]  final detections: boxes merged by eq. 12 (L166;
                              R27-R29: box centres, transitive, evaluated on the boxes that passed
                              A_min and fit in boxes[]), ascending label                        */
    float    *comb_debug;  /* optional [max_active * n_f0 * 3]  per candidate (SNR_M, N, median)
                              of eq. 10 / 8 / 9 for rows whose comb was evaluated; tests only */
} ddhf_outputs;

/* Same, HOST pointers, for ddhf_window_host(); any pointer may be NULL (not copied back). */
typedef struct {
    int32_t  *row_ptr;
    uint32_t *csr_ev;
    int32_t  *active_idx;
    float    *power;
    float    *sf;
    float    *score;
    int32_t  *f0_idx;
    uint8_t  *mask;
    int32_t  *labels;
    ddhf_box *boxes;
    int32_t  *counters;
    ddhf_box *merged_boxes;
} ddhf_host_outputs;

typedef struct ddhf_handle ddhf_handle;

/* Validate the configuration, build the constant tables (harmonic windows of every
 * candidate per R7-R9, fixed-point frequency constants) and upload them to the current
 * CUDA device.  *out is set to NULL on failure.  HOST pointers. */
int ddhf_create(const ddhf_config *cfg, ddhf_handle **out);

/* Bytes of DEVICE scratch ddhf_window() needs (a function of the config only). */
size_t ddhf_workspace_bytes(const ddhf_handle *h);

/* Run a0-a8 on one window.  d_events: DEVICE, n records, any order (CSR rows keep input
 * order, R20); t0_us / window_us define the half-open window [t0, t0+window) (R19),
 * 0 < window_us < 2^31.  d_workspace: DEVICE, >= ddhf_workspace_bytes(), 256-byte aligned,
 * contents irrelevant on entry.  out: HOST struct of DEVICE pointers.  cuda_stream: a
 * cudaStream_t (NULL = default stream).  Asynchronous.  Errors: DDHF_E_INVAL (NULL
 * pointers, window out of range), DDHF_E_CAPACITY (n > max_events), DDHF_E_CUDA. */
int ddhf_window(ddhf_handle *h, const ddhf_event *d_events, int64_t n, int64_t t0_us,
                int64_t window_us, void *d_workspace, const ddhf_outputs *out,
                void *cuda_stream);

/* ddhf_window() on 8-byte events (ddhf_event8, DEVICE): t = t_base_us + dt_us.  Same outputs, bit for bit. */
int ddhf_window_packed(ddhf_handle *h, const ddhf_event8 *d_events, int64_t n, int64_t t_base_us, int64_t t0_us,
                       int64_t window_us, void *d_workspace, const ddhf_outputs *out, void *cuda_stream);

/* Sliding windows ("Events are streamed in temporal windows"): advance the
 * window kept in the workspace to [t0, t0+window).  d_new_events: DEVICE, the n_new events that follow,
 * in the stream, the events handed over by the previous call.  The row of a pixel becomes the previous
 * row's events that are still inside the window (re-based to the new t0) followed by its new events: the
 * input order of the window's slice of the stream, so row_ptr / csr_ev are bit-identical to ddhf_window()
 * on that slice (R20), and so is everything downstream; only the new slab is sorted.  The first call (and
 * any call with another workspace, another window length, or t0 moved backwards or by a whole window or
 * more) starts a sequence: its events are the whole first window.  counters[n_dropped] counts the new
 * events outside the window or the sensor.  If the window outgrows max_events it is truncated and bit 2 of
 * counters[overflow] is set.  The workspace must not be used by other calls in between (ddhf_window()
 * on the same workspace keeps the state intact; ddhf_slide_reset() forgets it).  Otherwise as ddhf_window(). */
int ddhf_window_slide(ddhf_handle *h, const ddhf_event *d_new_events, int64_t n_new, int64_t t0_us,
                      int64_t window_us, void *d_workspace, const ddhf_outputs *out,
                      void *cuda_stream);
int ddhf_slide_reset(ddhf_handle *h);

/* End-to-end variant: h_events is HOST memory (pinned for full PCIe speed).  Copies the
 * events to the device, runs ddhf_window() on buffers owned by the handle (allocated on
 * first use), copies every non-NULL output back and synchronises the stream. */
int ddhf_window_host(ddhf_handle *h, const ddhf_event *h_events, int64_t n, int64_t t0_us,
                     int64_t window_us, const ddhf_host_outputs *out, void *cuda_stream);

/* Pipelined end-to-end variant (two windows in flight): ddhf_host_submit() enqueues the
 * host->device copy of the events on an internal copy stream, the window on `cuda_stream`
 * (after the copy) and the device->host copies of the requested outputs, and returns without
 * waiting, so that the copy of window i+1 overlaps the kernels of window i (SURVEY 8(f)-3:
 * double-buffered H2D).  ddhf_host_wait() blocks until the OLDEST submitted window is complete;
 * its outputs are then valid.  h_events and every buffer named in `out` are HOST memory (pinned,
 * or the copies are not asynchronous) and must stay valid and untouched until that wait returns.
 * Only the fixed-size outputs are supported here: row_ptr, sf, score, f0_idx, mask, labels, boxes
 * (all max_boxes records are copied) and counters; csr_ev, active_idx and power must be NULL.
 * Errors: DDHF_E_INVAL (NULL arguments, unsupported output requested, more than two windows in
 * flight on submit, none in flight on wait), DDHF_E_CAPACITY, DDHF_E_CUDA. */
int ddhf_host_submit(ddhf_handle *h, const ddhf_event *h_events, int64_t n, int64_t t0_us,
                     int64_t window_us, const ddhf_host_outputs *out, void *cuda_stream);
int ddhf_host_wait(ddhf_handle *h);
/* ddhf_host_submit() on 8-byte events (HOST, pinned): half the bytes over PCIe per window. */
int ddhf_host_submit_packed(ddhf_handle *h, const ddhf_event8 *h_events, int64_t n, int64_t t_base_us, int64_t t0_us,
                            int64_t window_us, const ddhf_host_outputs *out, void *cuda_stream);

/* With DDHF_FLAG_TIMING: waits for the last ddhf_window() on this handle and returns the
 * device time of its stages in ms: [0] ingest a0-a3, [1] the NDFT kernel (a4, a5 and the
 * queueing of the spectra to score), [2] deferred comb scoring a6-a7, [3] CCL + boxes a8,
 * [4] total.  ms: HOST float[5]. */
int ddhf_stage_ms(ddhf_handle *h, float *ms);

/* Number of kernels ddhf_window() launches per call (constant for a handle). */
int ddhf_launches_per_window(const ddhf_handle *h);

/* FP32 FMA throughput probe: runs register-resident FMA chains on every SM for at least
 * `ms_target` milliseconds each and reports the achieved TFLOP/s (2 flop per FMA) -- the
 * measured ceiling the NDFT roofline is quoted against.  tflops_out: HOST float[2],
 * [0] scalar FFMA, [1] packed FFMA2 (fma.rn.f32x2).  Synchronous. */
int ddhf_fma_peak_probe(float ms_target, float *tflops_out, void *cuda_stream);

int ddhf_destroy(ddhf_handle *h);

/* ---- Entry point that allocates nothing ---------------------------------------------------------------------
 * Stage a8 on a caller's mask: 8-connected component labelling, bounding boxes, the A_min filter
 * and, if merge_alpha > 0, the final detections of eq. 12 (L166) -- the same kernels ddhf_window() runs after the
 * comb stage, results bit-identical.  For callers that cannot allocate device memory (CUDA graph capture, serving
 * loops, harnesses that forbid cudaMalloc): no handle, no workspace; the stage's scratch is a static device array
 * inside the library (18.5 MB, held by every GPU that loads the library until the process exits), sized for
 *     width * height <= DDHF_NOALLOC_MAX_PIXELS (1280 x 720)   and   max_boxes <= DDHF_NOALLOC_MAX_BOXES;
 * anything larger is refused with DDHF_E_CAPACITY.  No cudaMalloc, cudaFree or allocating library call is made,
 * here or in ddhf_boxes_noalloc_setup().
 *   d_mask           DEVICE [width*height] bytes, nonzero = detection (input, not modified)
 *   d_labels         DEVICE [width*height] out: component label (min linear index), -1 off the mask
 *   d_boxes          DEVICE [max_boxes] out: boxes that passed a_min, ascending label
 *   d_merged_boxes   DEVICE [max_boxes] out: eq. 12 detections; may be NULL (or merge_alpha <= 0): not written
 *   d_counters       DEVICE int32[DDHF_N_COUNTERS] out: N_COMPONENTS, N_BOXES, N_BOXES_TOTAL, N_MERGED and
 *                    OVERFLOW bit 1 as for ddhf_window(); the other entries are written as 0
 * Only enqueues on `cuda_stream` (five kernels), never synchronises.  Every call on a device shares the one
 * array: calls that overlap on the GPU (different streams without an ordering between them, or two processes'
 * worth of threads on one device) race -- order them.  The array keeps the previous call's contents; what must
 * start cleared is cleared by the call itself.  ddhf_boxes_noalloc_setup() resolves the array's device address
 * for the CURRENT device (cudaGetSymbolAddress; once per device, idempotent, thread-safe); the entry point does
 * it on first use, so call setup beforehand where that must not happen at call time (before a stream capture).
 * Errors: DDHF_E_INVAL / DDHF_E_CAPACITY / DDHF_E_CUDA, text from ddhf_boxes_noalloc_error() (per thread). */
#define DDHF_NOALLOC_MAX_PIXELS 921600
#define DDHF_NOALLOC_MAX_BOXES  4096
int ddhf_boxes_noalloc_setup(void);
int ddhf_boxes_noalloc(const uint8_t *d_mask, int32_t width, int32_t height, int32_t a_min, float merge_alpha,
                       int32_t max_boxes, int32_t *d_labels, ddhf_box *d_boxes, ddhf_box *d_merged_boxes,
                       int32_t *d_counters, void *cuda_stream);
const char *ddhf_boxes_noalloc_error(void);

/* Text of the last error on this handle (or of the last failed ddhf_create if h is NULL). */
const char *ddhf_last_error(const ddhf_handle *h);

const char *ddhf_version(void);

#ifdef __cplusplus
}
#endif
#endif /* DDHF_H */
