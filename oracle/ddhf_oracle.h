/*
 * ddhf_oracle.h -- float64 CPU ORACLE for the DDHF hot path (arXiv 2603.08386).
 *
 * TEST INFRASTRUCTURE ONLY.  Only tests/, __graft_entry__.smoke() and bench.py's
 * cpu_baseline / --impl reference legs may build, link, import or call anything under
 * oracle/.  The product (paper_2603_08386_b200/, include/ddhf.h) never does, and the
 * oracle shares no source, header, table generator or helper with it.
 *
 * Every function is the plain definition from the paper, written out as direct loops in
 * double precision: one cos/sin per (bin, event) term, no recurrences, no FFT, no
 * blocking or reordering.  Citations are PAPER.md line numbers ("L93") plus the equation
 * or section; "R<n>" is reading n of DESIGN.md section 3 (taken where the paper is
 * silent or ambiguous).
 *
 * Parity pins (tests/test_oracle_*.py, none of which re-type these formulas):
 *   ndft_power      FFT on uniform samples, FFT of a sparse integer-timestamp sequence,
 *                   Parseval, single event = flat w^2, closed form of a periodic ON/OFF
 *                   train 4 N^2 sin^2(pi m tau) (tests/golden/periodic_train.txt), shift /
 *                   polarity-flip invariance, P_0 = (sum w)^2
 *   spectral_flatness  flat -> 1, one spike on a flat floor (closed form), scale invariance
 *   comb_score      hand-built spectra with known N, median and SNR; window-edge,
 *                   M_valid-prefix, h_min, overlapping-window and even-count cases
 *   bucket          numpy stable argsort / bincount / cumsum
 *   ccl_boxes       scipy.ndimage.label with the 3x3 structure + find_objects
 *   merge_boxes     hand-placed boxes (far / near / chain), scipy.sparse.csgraph.connected_components
 *                   on an adjacency built independently in numpy
 * No function here is "parity unpinned".
 */
#ifndef DDHF_ORACLE_H
#define DDHF_ORACLE_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

/* Event tuple (x, y, p, t).  Same 16-byte memory layout as the numpy
 * dtype in workloads.py (declared independently here). */
typedef struct {
    uint16_t x, y;
    int16_t p;          /* polarity; > 0 means +1, anything else -1 (L139, R21) */
    uint16_t pad;
    int64_t t_us;
} orc_event;

typedef struct {
    int32_t x0, y0, x1, y1;   /* inclusive corners */
    int32_t n_pix;
    int32_t label;            /* minimum linear pixel index of the component (R18) */
} orc_box;

typedef struct {
    int32_t width, height;
    double f_min_hz, df_hz;       /* uniform grid f_j = f_min + j df            (R3, R4) */
    int32_t n_freq;
    double f0_min_hz, f0_step_hz; /* candidates f0_c = f0_min + c step          (R12)    */
    int32_t n_f0;
    int32_t n_harm;               /* M of eq. 8 (Table 2)                          */
    int32_t half_bw_bins;         /* d_k of eq. 8 (Table 2)                         */
    int32_t h_min;                /* min matched harmonics (L115, Table 2)          */
    int32_t n_min;                /* min events per pixel (L137, Table 2)           */
    int32_t a_min;                /* min box area in px (L164, Table 2)             */
    double tau_sf, tau_comb;      /* L107, L131                                          */
    double sf_eps;                /* floor under log / division (R6, R11)                */
    int32_t k_lo;                 /* first bin used by SF and the comb (R6)              */
    int32_t score_all;            /* 1: comb score on every active pixel (R14);
                                     0: only where SF <= tau_sf (paper order, L139)      */
} orc_config;

/* a0-a3: filter to window/sensor, stable counting sort by pixel = y*W + x  (L137, R19, R20).
 * row_ptr[NP+1], csr_ev[n] (only the first row_ptr[NP] entries are written),
 * csr value = (t - t0) << 1 | (p > 0).  Returns the number of dropped events. */
int64_t orc_bucket(const orc_event *ev, int64_t n, int32_t width, int32_t height,
                   int64_t t0_us, int64_t window_us, int32_t *row_ptr, uint32_t *csr_ev);

/* a4: eq. 6 (L93) on a Hz grid: P_j = | sum_k w_k exp(-2 pi i f_j t_k 1e-6) |^2  (R1-R3). */
void orc_ndft_power(const int64_t *t_us, const double *w, int64_t n,
                    double f_min_hz, double df_hz, int32_t n_freq, double *power);

/* a5: eq. 7 (L104) over bins [k_lo, n_freq) with floor eps (R6). */
double orc_spectral_flatness(const double *power, int32_t n_freq, int32_t k_lo, double eps);

/* a6: eq. 8-11 (L113-131).  snr_out (optional, n_f0 doubles) receives SNR_M per candidate
 * (0 where skipped).  Returns max SNR (0 if no candidate is valid); *f0_idx = first argmax
 * or -1. */
double orc_comb_score(const double *power, const orc_config *cfg, int32_t *f0_idx,
                      double *snr_out, double *num_out, double *med_out);

/* a8: 8-connected components, label = min linear index; boxes sorted by label, kept if
 * bounding-box area >= a_min (L164, R17, R18).  labels[NP] (-1 off-mask).  Returns the
 * number of boxes written (at most max_boxes; *n_total = number that passed the filter). */
int32_t orc_ccl_boxes(const uint8_t *mask, int32_t width, int32_t height, int32_t a_min,
                      int32_t *labels, orc_box *boxes, int32_t max_boxes, int32_t *n_total);

/* Box merge, eq. 12 (L166): two boxes are merged if dist(c1, c2) < alpha max(w1, h1, w2, h2).
 * Readings R27-R29: c = centre of the bounding box, w = x1 - x0 + 1, h = y1 - y0 + 1; the rule is
 * evaluated on the boxes that enter the step and merging is transitive (connected components
 * of the "close" relation); a merged box is the bounding box of its members, n_pix their sum,
 * label their smallest label; output ascending by label.  out has room for n boxes.  Returns
 * the number of merged boxes. */
int32_t orc_merge_boxes(const orc_box *boxes, int32_t n, double alpha, orc_box *out);

/* Whole window: a0-a8.  All output pointers are host memory owned by the caller; power
 * (n_active x n_freq doubles, row r <-> active_idx[r]) and labels may be NULL.
 * counters[5] = { n_in (kept events), n_dropped, n_active, n_boxes written, n_boxes passing
 * A_min }.  OpenMP over pixels. */
int orc_window(const orc_config *cfg, const orc_event *ev, int64_t n, int64_t t0_us,
               int64_t window_us, int32_t *row_ptr, uint32_t *csr_ev, int32_t *active_idx,
               double *power, int64_t power_rows_cap, double *sf, double *score,
               int32_t *f0_idx, uint8_t *mask, int32_t *labels, orc_box *boxes,
               int32_t max_boxes, int64_t *counters);

int orc_num_threads(void);

#ifdef __cplusplus
}
#endif
#endif
