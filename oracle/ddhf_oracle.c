/*
 * ddhf_oracle.c -- float64 CPU ORACLE for the DDHF hot path (arXiv 2603.08386).
 * TEST INFRASTRUCTURE ONLY -- see ddhf_oracle.h for who may use it, the citations
 * convention and the list of pins.  Plain C, direct loops, double precision.
 */
#include "ddhf_oracle.h"

#include <math.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define ORC_PI 3.14159265358979323846264338327950288

int orc_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/* ---------------------------------------------------------------------------------- */
/* a0-a3  "sorted by pixel index" (L137).  Events outside [t0, t0+window) or outside   */
/* the sensor are dropped (R19); order inside a pixel is input order (R20).            */
/* ---------------------------------------------------------------------------------- */
int64_t orc_bucket(const orc_event *ev, int64_t n, int32_t width, int32_t height,
                   int64_t t0_us, int64_t window_us, int32_t *row_ptr, uint32_t *csr_ev)
{
    const int64_t np = (int64_t)width * height;
    int64_t dropped = 0;
    for (int64_t i = 0; i <= np; ++i) row_ptr[i] = 0;
    /* count */
    for (int64_t i = 0; i < n; ++i) {
        const orc_event *e = &ev[i];
        if (e->t_us < t0_us || e->t_us >= t0_us + window_us || e->x >= width || e->y >= height) {
            ++dropped;
            continue;
        }
        row_ptr[(int64_t)e->y * width + e->x + 1] += 1;
    }
    /* exclusive scan */
    for (int64_t i = 0; i < np; ++i) row_ptr[i + 1] += row_ptr[i];
    /* stable placement */
    int32_t *cursor = (int32_t *)malloc(sizeof(int32_t) * (size_t)(np > 0 ? np : 1));
    for (int64_t i = 0; i < np; ++i) cursor[i] = row_ptr[i];
    for (int64_t i = 0; i < n; ++i) {
        const orc_event *e = &ev[i];
        if (e->t_us < t0_us || e->t_us >= t0_us + window_us || e->x >= width || e->y >= height)
            continue;
        const int64_t pix = (int64_t)e->y * width + e->x;
        const uint32_t t_rel = (uint32_t)(e->t_us - t0_us);
        csr_ev[cursor[pix]++] = (t_rel << 1) | (e->p > 0 ? 1u : 0u);
    }
    free(cursor);
    return dropped;
}

/* ---------------------------------------------------------------------------------- */
/* a4  eq. 6 (L93):  F = sum_j p_j exp(i k t_j),  P = |F|^2 (L96).                     */
/* Hz grid and minus sign: R1-R3 (P is the same for either sign since p is real).      */
/* ---------------------------------------------------------------------------------- */
void orc_ndft_power(const int64_t *t_us, const double *w, int64_t n,
                    double f_min_hz, double df_hz, int32_t n_freq, double *power)
{
    for (int32_t j = 0; j < n_freq; ++j) {
        const double f = f_min_hz + (double)j * df_hz;
        double re = 0.0, im = 0.0;
        for (int64_t k = 0; k < n; ++k) {
            const double ang = -2.0 * ORC_PI * f * ((double)t_us[k] * 1e-6);
            re += w[k] * cos(ang);
            im += w[k] * sin(ang);
        }
        power[j] = re * re + im * im;
    }
}

/* ---------------------------------------------------------------------------------- */
/* a5  eq. 7 (L104): SF = exp(mean log P) / mean P over bins [k_lo, n_freq), P floored  */
/* at eps (R6).                                                                        */
/* ---------------------------------------------------------------------------------- */
double orc_spectral_flatness(const double *power, int32_t n_freq, int32_t k_lo, double eps)
{
    const int32_t nb = n_freq - k_lo;
    if (nb <= 0) return NAN;
    double slog = 0.0, ssum = 0.0;
    for (int32_t k = k_lo; k < n_freq; ++k) {
        const double p = power[k] > eps ? power[k] : eps;
        slog += log(p);
        ssum += p;
    }
    return exp(slog / nb) / (ssum / nb);
}

/* ---------------------------------------------------------------------------------- */
/* a6  eq. 8-11 (L113-131).                                                            */
/* ---------------------------------------------------------------------------------- */
static int cmp_double(const void *a, const void *b)
{
    const double x = *(const double *)a, y = *(const double *)b;
    return (x > y) - (x < y);
}

double orc_comb_score(const double *power, const orc_config *cfg, int32_t *f0_idx,
                      double *snr_out, double *num_out, double *med_out)
{
    const int32_t nf = cfg->n_freq, d = cfg->half_bw_bins, klo = cfg->k_lo;
    unsigned char *excl = (unsigned char *)malloc((size_t)(nf > 0 ? nf : 1));
    double *comp = (double *)malloc(sizeof(double) * (size_t)(nf > 0 ? nf : 1));
    double best = 0.0;
    int32_t best_c = -1;

    for (int32_t c = 0; c < cfg->n_f0; ++c) {
        const double f0 = cfg->f0_min_hz + (double)c * cfg->f0_step_hz;   /* candidate omega (R12) */
        if (snr_out) snr_out[c] = 0.0;
        if (num_out) num_out[c] = 0.0;
        if (med_out) med_out[c] = 0.0;

        /* M_valid(omega): leading harmonics whose window lies in-band (L115, R7, R8) */
        int32_t m_valid = 0;
        for (int32_t m = 1; m <= cfg->n_harm; ++m) {
            const int64_t km = (int64_t)floor(((double)m * f0 - cfg->f_min_hz) / cfg->df_hz + 0.5);
            if (km - d < klo || km + d > nf - 1) break;
            m_valid = m;
        }
        if (m_valid < cfg->h_min || m_valid < 1) continue;                 /* L115 */

        /* eq. 8: N = mean over valid harmonics of the max in |k - m omega| <= d_k;
         * eq. 9: H = union of the windows (R9) */
        memset(excl, 0, (size_t)nf);
        double num = 0.0;
        for (int32_t m = 1; m <= m_valid; ++m) {
            const int64_t km = (int64_t)floor(((double)m * f0 - cfg->f_min_hz) / cfg->df_hz + 0.5);
            double mx = power[km - d];
            for (int64_t k = km - d; k <= km + d; ++k) {
                if (power[k] > mx) mx = power[k];
                excl[k] = 1;
            }
            num += mx;
        }
        num /= (double)m_valid;

        /* median of the complement over [k_lo, n_freq): lower median (L124, R10) */
        int32_t nc = 0;
        for (int32_t k = klo; k < nf; ++k)
            if (!excl[k]) comp[nc++] = power[k];
        if (nc == 0) continue;
        qsort(comp, (size_t)nc, sizeof(double), cmp_double);
        const double med = comp[(nc - 1) / 2];

        /* eq. 10, with the floor of R11 */
        const double snr = num / (med > cfg->sf_eps ? med : cfg->sf_eps);
        if (snr_out) snr_out[c] = snr;
        if (num_out) num_out[c] = num;
        if (med_out) med_out[c] = med;
        if (best_c < 0 || snr > best) {        /* eq. 11: max over omega; first max wins (R16) */
            best = snr;
            best_c = c;
        }
    }
    free(excl);
    free(comp);
    *f0_idx = best_c;
    return best_c < 0 ? 0.0 : best;
}

/* ---------------------------------------------------------------------------------- */
/* a8  8-connected component labelling + bounding boxes + A_min filter (L164).          */
/* Raster scan; the first pixel of a component met in raster order is its minimum       */
/* linear index, which is the label (R18); boxes therefore come out sorted by label.    */
/* ---------------------------------------------------------------------------------- */
int32_t orc_ccl_boxes(const uint8_t *mask, int32_t width, int32_t height, int32_t a_min,
                      int32_t *labels, orc_box *boxes, int32_t max_boxes, int32_t *n_total)
{
    const int64_t np = (int64_t)width * height;
    int32_t *lab = labels ? labels : (int32_t *)malloc(sizeof(int32_t) * (size_t)(np > 0 ? np : 1));
    int32_t *stack = (int32_t *)malloc(sizeof(int32_t) * (size_t)(np > 0 ? np : 1));
    for (int64_t i = 0; i < np; ++i) lab[i] = -1;
    int32_t n_out = 0, n_pass = 0;
    for (int64_t s = 0; s < np; ++s) {
        if (!mask[s] || lab[s] >= 0) continue;
        orc_box b;
        b.x0 = b.x1 = (int32_t)(s % width);
        b.y0 = b.y1 = (int32_t)(s / width);
        b.n_pix = 0;
        b.label = (int32_t)s;
        int64_t top = 0;
        stack[top++] = (int32_t)s;
        lab[s] = (int32_t)s;
        while (top > 0) {
            const int32_t q = stack[--top];
            const int32_t qx = q % width, qy = q / width;
            b.n_pix += 1;
            if (qx < b.x0) b.x0 = qx;
            if (qx > b.x1) b.x1 = qx;
            if (qy < b.y0) b.y0 = qy;
            if (qy > b.y1) b.y1 = qy;
            for (int32_t dy = -1; dy <= 1; ++dy)
                for (int32_t dx = -1; dx <= 1; ++dx) {
                    if (!dx && !dy) continue;
                    const int32_t nx = qx + dx, ny = qy + dy;
                    if (nx < 0 || ny < 0 || nx >= width || ny >= height) continue;
                    const int64_t r = (int64_t)ny * width + nx;
                    if (mask[r] && lab[r] < 0) {
                        lab[r] = (int32_t)s;
                        stack[top++] = (int32_t)r;
                    }
                }
        }
        const int64_t area = (int64_t)(b.x1 - b.x0 + 1) * (b.y1 - b.y0 + 1);   /* R17 */
        if (area >= a_min) {
            if (n_out < max_boxes) boxes[n_out++] = b;
            ++n_pass;
        }
    }
    free(stack);
    if (!labels) free(lab);
    if (n_total) *n_total = n_pass;
    return n_out;
}

/* ---------------------------------------------------------------------------------- */
/* Box merge, eq. 12 (L166-176): merged if dist(c1, c2) < alpha * max(w1, h1, w2, h2).   */
/* Transitive closure by repeated relabelling (plain and slow), R27-R29.                 */
/* ---------------------------------------------------------------------------------- */
int32_t orc_merge_boxes(const orc_box *boxes, int32_t n, double alpha, orc_box *out)
{
    if (n <= 0) return 0;
    int32_t *grp = (int32_t *)malloc(sizeof(int32_t) * (size_t)n);
    for (int32_t i = 0; i < n; ++i) grp[i] = i;
    int changed = 1;
    while (changed) {                                   /* propagate the smallest index */
        changed = 0;
        for (int32_t i = 0; i < n; ++i)
            for (int32_t j = 0; j < n; ++j) {
                if (i == j || grp[i] == grp[j]) continue;
                const double cxi = 0.5 * (boxes[i].x0 + boxes[i].x1), cyi = 0.5 * (boxes[i].y0 + boxes[i].y1);
                const double cxj = 0.5 * (boxes[j].x0 + boxes[j].x1), cyj = 0.5 * (boxes[j].y0 + boxes[j].y1);
                const double dist = sqrt((cxi - cxj) * (cxi - cxj) + (cyi - cyj) * (cyi - cyj));
                double m = boxes[i].x1 - boxes[i].x0 + 1;
                if (boxes[i].y1 - boxes[i].y0 + 1 > m) m = boxes[i].y1 - boxes[i].y0 + 1;
                if (boxes[j].x1 - boxes[j].x0 + 1 > m) m = boxes[j].x1 - boxes[j].x0 + 1;
                if (boxes[j].y1 - boxes[j].y0 + 1 > m) m = boxes[j].y1 - boxes[j].y0 + 1;
                if (dist < alpha * m) {                 /* eq. 12 */
                    const int32_t g = grp[i] < grp[j] ? grp[i] : grp[j];
                    grp[i] = g;
                    grp[j] = g;
                    changed = 1;
                }
            }
    }
    int32_t n_out = 0;
    for (int32_t g = 0; g < n; ++g) {                   /* groups in ascending smallest member */
        int first = 1;
        orc_box b = boxes[g];
        for (int32_t i = 0; i < n; ++i) {
            if (grp[i] != g) continue;
            if (first) { b = boxes[i]; first = 0; continue; }
            if (boxes[i].x0 < b.x0) b.x0 = boxes[i].x0;
            if (boxes[i].y0 < b.y0) b.y0 = boxes[i].y0;
            if (boxes[i].x1 > b.x1) b.x1 = boxes[i].x1;
            if (boxes[i].y1 > b.y1) b.y1 = boxes[i].y1;
            b.n_pix += boxes[i].n_pix;
            if (boxes[i].label < b.label) b.label = boxes[i].label;
        }
        if (!first) out[n_out++] = b;
    }
    free(grp);
    return n_out;
}

/* ---------------------------------------------------------------------------------- */
/* Whole window, L137-139 + L164: bucket -> per active pixel NDFT power -> SF -> comb   */
/* -> mask -> CCL/boxes.                                                               */
/* ---------------------------------------------------------------------------------- */
int orc_window(const orc_config *cfg, const orc_event *ev, int64_t n, int64_t t0_us,
               int64_t window_us, int32_t *row_ptr, uint32_t *csr_ev, int32_t *active_idx,
               double *power, int64_t power_rows_cap, double *sf, double *score,
               int32_t *f0_idx, uint8_t *mask, int32_t *labels, orc_box *boxes,
               int32_t max_boxes, int64_t *counters)
{
    const int64_t np = (int64_t)cfg->width * cfg->height;
    const int32_t nf = cfg->n_freq;

    const int64_t dropped = orc_bucket(ev, n, cfg->width, cfg->height, t0_us, window_us,
                                       row_ptr, csr_ev);
    /* active pixels: at least n_min events (L137, R15), ascending pixel index */
    int64_t n_active = 0;
    for (int64_t p = 0; p < np; ++p) {
        sf[p] = NAN;
        score[p] = 0.0;
        f0_idx[p] = -1;
        mask[p] = 0;
        if (row_ptr[p + 1] - row_ptr[p] >= cfg->n_min && row_ptr[p + 1] - row_ptr[p] >= 1)
            active_idx[n_active++] = (int32_t)p;
    }

#pragma omp parallel
    {
        double *pw = (double *)malloc(sizeof(double) * (size_t)nf);
        int64_t cap = 64;
        int64_t *tt = (int64_t *)malloc(sizeof(int64_t) * (size_t)cap);
        double *ww = (double *)malloc(sizeof(double) * (size_t)cap);
#pragma omp for schedule(dynamic, 16)
        for (int64_t r = 0; r < n_active; ++r) {
            const int64_t p = active_idx[r];
            const int64_t beg = row_ptr[p], cnt = row_ptr[p + 1] - row_ptr[p];
            if (cnt > cap) {
                cap = cnt * 2;
                tt = (int64_t *)realloc(tt, sizeof(int64_t) * (size_t)cap);
                ww = (double *)realloc(ww, sizeof(double) * (size_t)cap);
            }
            for (int64_t k = 0; k < cnt; ++k) {
                tt[k] = (int64_t)(csr_ev[beg + k] >> 1);             /* t - t0 (R2)       */
                ww[k] = (csr_ev[beg + k] & 1u) ? 1.0 : -1.0;         /* polarity -> +-1 (L139) */
            }
            double *dst = (power && r < power_rows_cap) ? power + r * (int64_t)nf : pw;
            orc_ndft_power(tt, ww, cnt, cfg->f_min_hz, cfg->df_hz, nf, dst);
            const double s = orc_spectral_flatness(dst, nf, cfg->k_lo, cfg->sf_eps);
            sf[p] = s;
            const int sf_ok = (s <= cfg->tau_sf);                    /* discard if SF > tau_sf (L107) */
            if (cfg->score_all || sf_ok) {
                int32_t fi;
                score[p] = orc_comb_score(dst, cfg, &fi, NULL, NULL, NULL);
                f0_idx[p] = fi;
            }
            mask[p] = (uint8_t)(sf_ok && f0_idx[p] >= 0 && score[p] >= cfg->tau_comb);   /* eq. 11 */
        }
        free(pw);
        free(tt);
        free(ww);
    }

    int32_t n_total = 0;
    const int32_t nb = orc_ccl_boxes(mask, cfg->width, cfg->height, cfg->a_min, labels, boxes,
                                     max_boxes, &n_total);
    counters[0] = n - dropped;
    counters[1] = dropped;
    counters[2] = n_active;
    counters[3] = nb;
    counters[4] = n_total;
    return 0;
}
