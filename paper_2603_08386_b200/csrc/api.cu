// api.cu -- the C ABI of include/ddhf.h: handle, constant tables, workspace layout, the
// per-window launch sequence and the host-buffer (end-to-end) variant.
#include <algorithm>
#include <math.h>
#include <stdio.h>
#include <string.h>

#include <string>
#include <vector>

#include "ddhf_internal.cuh"

namespace ddhf {
int fma_probe(float ms_target, float *tflops, cudaStream_t st);
}

using namespace ddhf;

struct ddhf_handle {
    ddhf_config cfg;
    int np = 0;
    int sm_count = 0;
    int n_tiles = 0;
    int launches = 0;
    int bl = 5, nb = 1, hbits = 1;          // ingest digit split (ingest_plan)
    int giant_row0 = 0, giant_rows = 0;     // chunk rows reserved for giant buckets
    int spill_cap = 0;
    bool fallback = true;                  // the NDFT kernel variant with in-place scoring (queue smaller than the sensor)
    ScoreParams sp{};
    uint64_t g_f0 = 0, g_d = 0, g_h = 0;
    bool nufft = false;                     // DDHF_FLAG_NUFFT and the grid / queue allow it
    int nufft_min = 0;                      // rows of at least that many events take the NUFFT path
    uint64_t g_nc = 0, g_nt = 0;            // its frequency constants (nufft.cu)
    size_t off_hot = 0, off_nuscr = 0;
    unsigned char *d_tables = nullptr;      // comb tables (num_tab | piece_tab | meta)
    int band_size = 0;
    int ndft_blocks_per_sm = 1, full_blocks_per_sm = 1, score_blocks_per_sm = 1;
    // workspace offsets (bytes)
    size_t off_cnt = 0, off_items = 0, off_scratch = 0, off_work = 0, off_tiles = 0, off_class = 0, off_cursor = 0, off_runs = 0, off_bkt = 0, off_rows = 0, off_spill = 0, off_spillrec = 0,
           off_parent = 0, off_rec = 0, off_ctiles = 0, off_merge = 0, off_giant = 0, off_slide = 0, off_segwork = 0, off_split = 0, off_splitcnt = 0, off_partial = 0, ws_bytes = 0;
    cudaEvent_t ev[5] = {nullptr, nullptr, nullptr, nullptr, nullptr};
    bool timed_once = false;
    // buffers of the host-buffer variant
    ddhf_event *hb_events = nullptr;
    void *hb_ws = nullptr;
    ddhf_outputs hb_out{};
    bool hb_ready = false;
    // double-buffered pipeline of ddhf_host_submit / ddhf_host_wait
    struct PipeSlot {
        ddhf_event *events = nullptr;
        void *ws = nullptr;
        ddhf_outputs out{};
        cudaEvent_t copied = nullptr, kernels = nullptr, done = nullptr;
    } pipe[2];
    cudaStream_t copy_stream = nullptr, d2h_stream = nullptr;   // H2D of the next window / D2H of the finished one, both beside the kernels
    bool pipe_ready = false;
    long long pipe_head = 0, pipe_tail = 0;      // windows submitted / waited for
    // sliding-window state (ddhf_window_slide): the previous window's CSR lives in the workspace
    bool slide_valid = false;
    int64_t slide_t0 = 0, slide_window = 0;
    void *slide_ws = nullptr;
    int slide_parity = 0;
    std::string err;
};

static std::string g_create_err;

static int fail(ddhf_handle *h, int code, const std::string &msg)
{
    if (h) h->err = msg; else g_create_err = msg;
    return code;
}

static size_t align_up(size_t x, size_t a = 256) { return (x + a - 1) / a * a; }

static uint64_t freq_const(double f_hz)
{
    // round(2^64 * f * 1e-6) mod 2^64: phase in turns of f at integer microsecond t is hi32(G * t).
    // Only the fractional part of f * 1e-6 (cycles per microsecond) matters; it is scaled in two
    // 32-bit halves so that no signed 64-bit conversion can overflow, whatever f is.
    long double x = static_cast<long double>(f_hz) / 1.0e6L;
    x -= floorl(x);
    const long double hi = floorl(ldexpl(x, 32));
    const long double lo = roundl(ldexpl(ldexpl(x, 32) - hi, 32));
    return (static_cast<uint64_t>(hi) << 32) + static_cast<uint64_t>(lo);     // lo == 2^32 carries into hi
}

extern "C" const char *ddhf_version(void) { return "ddhf-b200 0.1 (sm_100a)"; }

extern "C" const char *ddhf_last_error(const ddhf_handle *h)
{
    return h ? h->err.c_str() : g_create_err.c_str();
}

extern "C" int ddhf_create(const ddhf_config *cfg, ddhf_handle **out)
{
    if (out) *out = nullptr;
    if (!cfg || !out) return fail(nullptr, DDHF_E_INVAL, "ddhf_create: NULL argument");
    const ddhf_config &c = *cfg;
    const long long np = static_cast<long long>(c.width) * c.height;
    if (c.width < 1 || c.height < 1 || c.width > 65535 || c.height > 65535 || np > (4ll << 20))
        return fail(nullptr, DDHF_E_INVAL, "ddhf_create: sensor size out of range (<= 4 Mi pixels)");
    if (c.n_freq < 8 || c.n_freq > 2048)
        return fail(nullptr, DDHF_E_INVAL, "ddhf_create: n_freq must be in [8, 2048]");
    if (!(c.df_hz > 0) || !(c.f_min_hz >= 0) || c.f_min_hz + (c.n_freq + 64) * c.df_hz >= 4.0e5)
        return fail(nullptr, DDHF_E_INVAL, "ddhf_create: frequency grid out of range (0 <= f < 400 kHz)");
    if (c.n_f0 < 1 || c.n_f0 > kMaxF0 || c.n_harm < 1 || c.n_harm > kMaxHarm || c.half_bw_bins < 0 ||
        c.h_min < 1 || !(c.f0_step_hz >= 0) || !(c.f0_min_hz > 0))
        return fail(nullptr, DDHF_E_INVAL, "ddhf_create: comb parameters out of range");
    if (c.k_lo < 0 || c.k_lo >= c.n_freq || !(c.sf_eps > 0))
        return fail(nullptr, DDHF_E_INVAL, "ddhf_create: k_lo / sf_eps out of range");
    if (c.max_events < 1 || c.max_events >= (1ll << 31) || c.max_active < 1 || c.max_boxes < 1)
        return fail(nullptr, DDHF_E_INVAL, "ddhf_create: capacities out of range");

    ddhf_handle *h = new (std::nothrow) ddhf_handle();
    if (!h) return fail(nullptr, DDHF_E_NOMEM, "ddhf_create: out of host memory");
    h->cfg = c;
    h->np = static_cast<int>(np);
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess ||
        cudaDeviceGetAttribute(&h->sm_count, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) {
        delete h;
        return fail(nullptr, DDHF_E_CUDA, "ddhf_create: no CUDA device");
    }

    // ---- comb tables (R7-R10): harmonic centres, validity prefix, union of the windows, median rank ------
    const int nb = c.n_freq - c.k_lo, d = c.half_bw_bins;
    const int nbl = ndft_bins_per_lane(c.n_freq);
    const int cpad = (c.n_f0 + 31) / 32 * 32;
    const int wlen = 2 * d + 1;
    int s_lvl = 0;
    while (s_lvl < 5 && (2 << s_lvl) <= wlen) ++s_lvl;               // 2^s_lvl <= min(wlen, 32)
    const int blk = 1 << s_lvl;
    if (wlen > 2 * blk) {
        delete h;
        return fail(nullptr, DDHF_E_INVAL, "ddhf_create: half_bw_bins must be <= 31 (harmonic window <= 63 bins)");
    }
    auto padk = [nbl](long long k) { return static_cast<uint32_t>(k + k / nbl); };
    struct Cand { int mv = 0, rank = 0, n_excl = 0; std::vector<int> kc; std::vector<std::pair<int, int>> pieces; };
    std::vector<Cand> cand(c.n_f0);
    int r0 = 1 << 30, r1 = -1, max_pieces = 1;
    for (int ci = 0; ci < c.n_f0; ++ci) {
        Cand &t = cand[ci];
        const double f0 = c.f0_min_hz + ci * c.f0_step_hz;
        for (int m = 1; m <= c.n_harm; ++m) {
            const long long km = static_cast<long long>(floor((m * f0 - c.f_min_hz) / c.df_hz + 0.5));
            if (km - d < c.k_lo || km + d > c.n_freq - 1) break;
            t.kc.push_back(static_cast<int>(km));
        }
        int mv = static_cast<int>(t.kc.size());
        if (mv < c.h_min) continue;
        // union of the windows as disjoint intervals (centres rise with m), cut into pieces of <= 32 bins
        std::vector<std::pair<int, int>> iv;
        int n_excl = 0;
        for (int m = 0; m < mv; ++m) {
            const int lo = t.kc[m] - d, hi = t.kc[m] + d;
            if (!iv.empty() && lo <= iv.back().second) {
                if (hi > iv.back().second) { n_excl += hi - iv.back().second; iv.back().second = hi; }
            } else {
                iv.emplace_back(lo, hi);
                n_excl += hi - lo + 1;
            }
        }
        const int n_comp = nb - n_excl;
        if (n_comp <= 0) continue;
        for (const auto &q : iv)
            for (int s = q.first; s <= q.second; s += 32)
                t.pieces.emplace_back(s, std::min(32, q.second - s + 1));
        t.mv = mv;
        t.n_excl = n_excl;
        t.rank = (n_comp - 1) / 2;
        r0 = std::min(r0, t.rank);
        r1 = std::max(r1, t.rank + n_excl);
        max_pieces = std::max(max_pieces, static_cast<int>(t.pieces.size()));
    }
    if (r1 < 0) { r0 = 0; r1 = 0; }
    const int band_size = ndft_band_size(c.n_freq, r0, r1);
    if (band_size == 0 || max_pieces > kMaxPieces) {
        delete h;
        return fail(nullptr, DDHF_E_INVAL,
                    "ddhf_create: harmonic windows exclude too many bins for the band sorter "
                    "(the union of a candidate's windows must stay below about 900 of 2048 bins; "
                    "n_harm * (2 half_bw_bins + 1) too large for n_freq)");
    }
    {
        // one device buffer: num_tab [n_harm][cpad] u32 | piece_tab [max_pieces][cpad] uint2 | meta [cpad] uint4
        // rows padded to a multiple of 8 (the kernel reads the tables 8 rows at a time, unconditionally)
        const size_t n_num = static_cast<size_t>((c.n_harm + 7) / 8 * 8) * cpad, n_pc = static_cast<size_t>((max_pieces + 7) / 8 * 8) * cpad;
        const size_t off_pc = align_up(n_num * sizeof(uint32_t), 16), off_meta = align_up(off_pc + n_pc * sizeof(uint2), 16);
        const size_t bytes = off_meta + static_cast<size_t>(cpad) * sizeof(uint4);
        std::vector<unsigned char> host(bytes, 0);
        uint32_t *num_tab = reinterpret_cast<uint32_t *>(host.data());
        uint2 *piece_tab = reinterpret_cast<uint2 *>(host.data() + off_pc);
        uint4 *meta = reinterpret_cast<uint4 *>(host.data() + off_meta);
        for (int ci = 0; ci < c.n_f0; ++ci) {
            const Cand &t = cand[ci];
            if (t.mv == 0) continue;
            for (int m = 0; m < t.mv; ++m)
                num_tab[static_cast<size_t>(m) * cpad + ci] = padk(t.kc[m] - d) | (padk(t.kc[m] + d - blk + 1) << 16);
            for (size_t q = 0; q < t.pieces.size(); ++q) {
                const int len = t.pieces[q].second;
                piece_tab[q * cpad + ci] = make_uint2(len >= 32 ? 0xffffffffu : ((1u << len) - 1u),
                                                      static_cast<uint32_t>(t.pieces[q].first));
            }
            const float inv_mv = 1.0f / static_cast<float>(t.mv);
            uint32_t inv_bits;
            memcpy(&inv_bits, &inv_mv, 4);
            meta[ci] = make_uint4(static_cast<uint32_t>(t.mv) | (static_cast<uint32_t>(t.pieces.size()) << 16),
                                  static_cast<uint32_t>(t.rank) | (static_cast<uint32_t>(t.n_excl) << 16), inv_bits, 0u);
        }
        if (cudaMalloc(&h->d_tables, bytes) != cudaSuccess ||
            cudaMemcpy(h->d_tables, host.data(), bytes, cudaMemcpyHostToDevice) != cudaSuccess) {
            const std::string msg = std::string("ddhf_create: ") + cudaGetErrorString(cudaGetLastError());
            if (h->d_tables) cudaFree(h->d_tables);
            delete h;
            return fail(nullptr, DDHF_E_CUDA, msg);
        }
        h->sp.num_tab = reinterpret_cast<const uint32_t *>(h->d_tables);
        h->sp.piece_tab = reinterpret_cast<const uint2 *>(h->d_tables + off_pc);
        h->sp.meta = reinterpret_cast<const uint4 *>(h->d_tables + off_meta);
    }
    h->band_size = band_size;
    {
        // deferred-scoring queue: one row (the padded spectrum) per pixel to score.  Default: a row for every
        // pixel when that stays below 1/16 of the device's memory (1280x720 at 2048 bins: 7.5 GB of the
        // workspace on a 180 GB part) -- the NDFT kernel then never scores in place and runs its lean variant;
        // else 32 Ki rows with the in-place fallback.  max_scored > 0 sets the row count explicitly.
        const size_t row_bytes = sizeof(float) * static_cast<size_t>(ndft_padded_bins(c.n_freq));
        size_t mem_free = 0, mem_total = 0;
        cudaMemGetInfo(&mem_free, &mem_total);
        h->spill_cap = (row_bytes * static_cast<size_t>(h->np) <= mem_total / 16) ? h->np : (h->np < 32768 ? h->np : 32768);
        if (c.max_scored > 0) h->spill_cap = c.max_scored < h->np ? c.max_scored : h->np;
        if (!ndft_scores_in_place(c.n_freq, band_size)) h->spill_cap = h->np;      // every pixel must fit in the queue
        h->fallback = h->spill_cap < h->np;
    }
    if (ingest_configure() != cudaSuccess ||
        ndft_configure(c.n_freq, band_size, cpad, h->fallback, &h->ndft_blocks_per_sm, &h->full_blocks_per_sm,
                       &h->score_blocks_per_sm) != cudaSuccess) {
        const std::string msg = std::string("ddhf_create: ") + cudaGetErrorString(cudaGetLastError());
        cudaFree(h->d_tables);
        delete h;
        return fail(nullptr, DDHF_E_CUDA, msg);
    }
    h->sp.n_freq = c.n_freq; h->sp.k_lo = c.k_lo; h->sp.n_f0 = c.n_f0; h->sp.n_harm = c.n_harm; h->sp.half_bw = d;
    h->sp.s_lvl = s_lvl; h->sp.r0 = r0; h->sp.r1 = r1; h->sp.cpad = cpad; h->sp.max_pieces = max_pieces;
    h->sp.tau_sf = c.tau_sf; h->sp.tau_comb = c.tau_comb; h->sp.sf_eps = c.sf_eps;
    h->sp.score_all = (c.flags & DDHF_FLAG_SCORE_ALL) ? 1 : 0;

    // ---- fixed-point frequency constants of the factorised NDFT ------------------------------
    const int tn = ndft_tn(c.n_freq);
    // negated (mod 2^64): the kernel evaluates (sin, cos) of -2 pi f t directly
    h->g_h = 0ull - freq_const(16.0 * c.df_hz);
    h->g_d = 0ull - freq_const(c.df_hz);
    h->g_f0 = 0ull - freq_const(c.f_min_hz + (32.0 * tn - 16.0) * c.df_hz);
    // NUFFT path for long rows: needs the 4096-cell grid and a queue row per pixel (it never scores in place)
    if ((c.flags & DDHF_FLAG_NUFFT) && nufft_supported(c.n_freq) && !h->fallback) {
        if (nufft_configure() != cudaSuccess) {
            const std::string msg = std::string("ddhf_create: ") + cudaGetErrorString(cudaGetLastError());
            cudaFree(h->d_tables);
            delete h;
            return fail(nullptr, DDHF_E_CUDA, msg);
        }
        h->nufft = true;
        h->nufft_min = static_cast<int>(c.flags >> 16) ? static_cast<int>(c.flags >> 16) : DDHF_NUFFT_MIN_DEFAULT;
        h->g_nc = 0ull - freq_const(c.f_min_hz + 1024.0 * c.df_hz);
        h->g_nt = freq_const(c.df_hz);
    }

    // ---- workspace layout -----------------------------------------------------------------------
    h->n_tiles = (h->np + kScanTile - 1) / kScanTile;
    size_t o = 0;
    h->off_cnt = o;        o = align_up(o + sizeof(int32_t) * h->np);
    {
        // tile slots of the bucket-sorted items: 4-byte items in slots of ingest_tile_stride(true), 8-byte in (false)
        const size_t ev_tiles = (static_cast<size_t>(c.max_events) + ingest_tile_events() - 1) / ingest_tile_events();
        const size_t a = 4u * ingest_tile_stride(true), b = 8u * ingest_tile_stride(false);
        h->off_items = o;  o = align_up(o + ev_tiles * (a > b ? a : b));
    }
    h->off_scratch = o;    o = align_up(o + sizeof(uint64_t) * static_cast<size_t>(c.max_events));
    // work list: one item per active pixel, one more per extra segment of a split row (rows > kSplitMin
    // events in segments of <= kSegEvents); partial sums and arrival counters of the segment trees
    const size_t max_segs = static_cast<size_t>(c.max_events) / kSegEvents + static_cast<size_t>(c.max_events) / kSplitMin + 2;
    const size_t max_rows = static_cast<size_t>(c.max_events) / kSplitMin + 1;          // rows that can be split
    const size_t max_slots = max_segs * kSplitFan / (kSplitFan - 1) + 4 * max_rows + 64;   // leaves + inner nodes, rounding per level
    h->off_work = o;       o = align_up(o + sizeof(WorkItem) * (static_cast<size_t>(h->np) + max_segs));
    h->off_segwork = o;    o = align_up(o + sizeof(WorkItem) * max_segs);            // segment list of the lean NDFT variant
    h->off_split = o;      o = align_up(o + sizeof(SplitRow) * max_rows);
    h->off_splitcnt = o;   o = align_up(o + sizeof(int32_t) * (max_segs + 4 * max_rows + 64));
    h->off_partial = o;    o = align_up(o + sizeof(float) * max_slots * 2 * ndft_padded_bins(c.n_freq));
    h->off_tiles = o;      o = align_up(o + sizeof(int32_t) * 4 * 1024);
    h->off_class = o;      o = align_up(o + sizeof(int32_t) * 2 * kNumClasses);
    h->off_cursor = o;     o = align_up(o + 256);
    {
        // stable two-level sort on the pixel index (ingest.cu): run table of the tiles, bucket totals and
        // bases, chunk table of the buckets that need more than one chunk (at most 2 n / capacity + nb rows)
        ingest_plan(h->np, &h->bl, &h->nb, &h->hbits);
        const size_t ev_tiles = (static_cast<size_t>(c.max_events) + ingest_tile_events() - 1) / ingest_tile_events();
        h->off_runs = o;    o = align_up(o + sizeof(uint32_t) * ev_tiles * static_cast<size_t>(h->nb));
        h->off_bkt = o;     o = align_up(o + sizeof(int32_t) * 6 * (static_cast<size_t>(h->nb) + 2));
        h->off_giant = o;   o = align_up(o + 32 * (static_cast<size_t>(h->nb) + 2));
        // chunk rows: header + counts + bases per pixel of a bucket; the one-CTA path needs at most 2 n / capacity + nb
        // rows, the giant buckets get 4 rows per tile more (a bucket that finds no room there stays on the one-CTA path)
        h->giant_row0 = static_cast<int>(2 * ev_tiles + h->nb + 2);
        h->giant_rows = static_cast<int>(4 * ev_tiles + 64);
        h->off_rows = o;    o = align_up(o + sizeof(int32_t) * (static_cast<size_t>(h->giant_row0) + h->giant_rows) * (4 + (static_cast<size_t>(2) << h->bl)));
    }
    // deferred-scoring queue (row count decided above)
    h->off_spill = o;      o = align_up(o + sizeof(float) * static_cast<size_t>(h->spill_cap) * ndft_padded_bins(c.n_freq));
    h->off_spillrec = o;   o = align_up(o + sizeof(SpillRec) * static_cast<size_t>(h->spill_cap));
    h->off_parent = o;     o = align_up(o + sizeof(int32_t) * h->np);
    h->off_rec = o;        o = align_up(o + sizeof(int32_t) * 5 * static_cast<size_t>(h->np));
    h->off_ctiles = o;     o = align_up(o + sizeof(int32_t) * 1032);
    // sliding windows: two copies of (row_ptr, csr_ev) used alternately, the new slab's own CSR
    h->off_slide = o;      o = align_up(o + 2 * (sizeof(int32_t) * (static_cast<size_t>(h->np) + 2) + sizeof(uint32_t) * static_cast<size_t>(c.max_events))
                                         + sizeof(int32_t) * static_cast<size_t>(h->np) + sizeof(uint32_t) * static_cast<size_t>(c.max_events) + 1024);
    h->off_merge = o;      o = align_up(o + sizeof(int32_t) * 6 * static_cast<size_t>(c.max_boxes));
    if (h->nufft) {
        h->off_hot = o;    o = align_up(o + sizeof(WorkItem) * static_cast<size_t>(h->np));
        h->off_nuscr = o;  o = align_up(o + sizeof(float) * 2048 * static_cast<size_t>(h->sm_count) * nufft_warps());
    }
    h->ws_bytes = o;

    if (c.flags & DDHF_FLAG_TIMING)
        for (int i = 0; i < 5; ++i) cudaEventCreate(&h->ev[i]);
    *out = h;
    return DDHF_OK;
}

extern "C" size_t ddhf_workspace_bytes(const ddhf_handle *h) { return h ? h->ws_bytes : 0; }

extern "C" int ddhf_launches_per_window(const ddhf_handle *h) { return h ? h->launches : 0; }

// mode 0: one window from scratch; 1: first window of a sliding sequence (from scratch, CSR saved in the
// workspace); 2: slide (d_events = the new slab, shift = t0 - previous t0)
static int run_window(ddhf_handle *h, const ddhf_event *d_events, int64_t n, int64_t t0_us,
                      int64_t window_us, void *d_workspace, const ddhf_outputs *out,
                      void *cuda_stream, int mode, int64_t shift_us, bool packed = false, int64_t t_base_us = 0)
{
    if (!h) return DDHF_E_INVAL;
    if (!out || !d_workspace || (n > 0 && !d_events))
        return fail(h, DDHF_E_INVAL, "ddhf_window: NULL argument");
    if (!out->row_ptr || !out->csr_ev || !out->active_idx || !out->sf || !out->score || !out->f0_idx ||
        !out->mask || !out->boxes || !out->counters)
        return fail(h, DDHF_E_INVAL, "ddhf_window: a required output pointer is NULL");
    if (n < 0 || window_us <= 0 || window_us >= (1ll << 31))
        return fail(h, DDHF_E_INVAL, "ddhf_window: n or window_us out of range");
    if (n > h->cfg.max_events) return fail(h, DDHF_E_CAPACITY, "ddhf_window: n > max_events");
    if (packed && h->cfg.height > 32768)
        return fail(h, DDHF_E_INVAL, "ddhf_window_packed: 8-byte events hold y < 32768");
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    char *ws = static_cast<char *>(d_workspace);
    const ddhf_config &c = h->cfg;
    const bool timing = (c.flags & DDHF_FLAG_TIMING) != 0;

    int32_t *cp_parent = out->labels ? out->labels : reinterpret_cast<int32_t *>(ws + h->off_parent);
    IngestParams ip{};
    ip.events = d_events; ip.n = n; ip.t0 = t0_us; ip.t1 = t0_us + window_us;
    ip.packed = packed ? 1 : 0; ip.t_base = t_base_us;
    ip.width = c.width; ip.height = c.height; ip.np = h->np;
    ip.n_min = c.n_min; ip.max_active = c.max_active;
    ip.cnt = reinterpret_cast<int32_t *>(ws + h->off_cnt);
    ip.row_ptr = out->row_ptr; ip.csr_ev = out->csr_ev;
    ip.items = ws + h->off_items; ip.scratch = ws + h->off_scratch;
    ip.active_idx = out->active_idx;
    ip.work = reinterpret_cast<WorkItem *>(ws + h->off_work);
    int32_t *tiles = reinterpret_cast<int32_t *>(ws + h->off_tiles);
    ip.tile_sum = tiles; ip.tile_act = tiles + 1024; ip.tile_off = tiles + 2048; ip.tile_aoff = tiles + 3072;
    ip.class_cnt = reinterpret_cast<int32_t *>(ws + h->off_class);
    ip.class_cur = ip.class_cnt + kNumClasses;
    ip.counters = out->counters;
    ip.sf = out->sf; ip.score = out->score; ip.f0_idx = out->f0_idx; ip.mask = out->mask;
    ip.work_cursor = reinterpret_cast<unsigned long long *>(ws + h->off_cursor);
    ip.bl = h->bl; ip.vb = 32 - h->bl; ip.nb = h->nb; ip.hbits = h->hbits;
    ip.compact = (2 * window_us <= (1ll << ip.vb)) ? 1 : 0;               // value = (t - t0) << 1 | polarity
    ip.run_tab = reinterpret_cast<uint32_t *>(ws + h->off_runs);
    ip.bkt_total = reinterpret_cast<int32_t *>(ws + h->off_bkt);
    ip.bkt_base = ip.bkt_total + h->nb + 2;
    ip.bkt_order = ip.bkt_base + h->nb + 2;
    ip.bkt_act = ip.bkt_order + h->nb + 2;
    ip.bkt_maxrun = ip.bkt_act + h->nb + 2;
    ip.giant_of = ip.bkt_maxrun + h->nb + 2;
    ip.giant_tab = ws + h->off_giant;
    ip.giant_row0 = h->giant_row0; ip.giant_rows = h->giant_rows;
    ip.chunk_rows = reinterpret_cast<int32_t *>(ws + h->off_rows);
    ip.sync = reinterpret_cast<int32_t *>(ws + h->off_cursor + 16);       // [16]; the scoring queue counts are sync[2..3]

    if (mode != 0) {
        // state buffers: {row_ptr [np + 2], csr [max_events]} x 2, then the slab's {row starts [np], csr [max_events]}
        const size_t rp_bytes = sizeof(int32_t) * (static_cast<size_t>(h->np) + 2), cs_bytes = sizeof(uint32_t) * static_cast<size_t>(c.max_events);
        char *s0 = ws + h->off_slide, *s1 = s0 + rp_bytes + cs_bytes, *s2 = s1 + rp_bytes + cs_bytes;
        char *prev = h->slide_parity ? s1 : s0, *next = h->slide_parity ? s0 : s1;
        ip.next_row_ptr = reinterpret_cast<int32_t *>(next);
        ip.next_csr = reinterpret_cast<uint32_t *>(next + rp_bytes);
        if (mode == 2) {
            ip.prev_row_ptr = reinterpret_cast<const int32_t *>(prev);
            ip.prev_csr = reinterpret_cast<const uint32_t *>(prev + rp_bytes);
            ip.slab_row_ptr = reinterpret_cast<int32_t *>(s2);
            ip.slab_csr = reinterpret_cast<uint32_t *>(s2 + sizeof(int32_t) * static_cast<size_t>(h->np));
            ip.shift2 = static_cast<uint32_t>(2 * shift_us);
        }
        ip.csr_cap = static_cast<int32_t>(c.max_events);
    }
    ip.split_tab = reinterpret_cast<SplitRow *>(ws + h->off_split);
    if (!h->fallback && ndft_bins_per_lane(c.n_freq) == 64) {      // lean 2048-bin kernel: segments in a second pass
        ip.seg_work = reinterpret_cast<WorkItem *>(ws + h->off_segwork);
        ip.work_cursor2 = reinterpret_cast<unsigned long long *>(ws + h->off_cursor + 96);
    }
    ip.split_cnt = reinterpret_cast<int32_t *>(ws + h->off_splitcnt);
    ip.ccl_parent = cp_parent;
    const bool use_nufft = h->nufft && nufft_window_fits(c.df_hz, window_us);
    if (use_nufft) {
        ip.hot_work = reinterpret_cast<WorkItem *>(ws + h->off_hot);
        ip.hot_min = h->nufft_min;
        ip.hot_cursor = reinterpret_cast<int32_t *>(ws + h->off_cursor + 104);
    }

    NdftParams np{};
    np.work = ip.work; np.csr_ev = out->csr_ev; np.counters = out->counters;
    np.work_cursor = ip.work_cursor; np.max_active = c.max_active;
    np.n_work = ip.sync + 4; np.split_tab = ip.split_tab; np.split_cnt = ip.split_cnt;
    np.split_partial = reinterpret_cast<float *>(ws + h->off_partial);
    np.g_f0 = h->g_f0; np.g_d = h->g_d; np.g_h = h->g_h;
    np.power = out->power; np.sf = out->sf; np.score = out->score; np.f0_idx = out->f0_idx;
    np.mask = out->mask; np.comb_debug = out->comb_debug;
    np.n_scored = out->counters + DDHF_CNT_N_SCORED;
    np.spill = reinterpret_cast<float *>(ws + h->off_spill);
    np.spill_rec = reinterpret_cast<SpillRec *>(ws + h->off_spillrec);
    np.spill_count = reinterpret_cast<int32_t *>(ws + h->off_cursor + 24);
    np.spill_cap = h->spill_cap;
    np.sp = h->sp;

    CclParams cp{};
    cp.mask = out->mask; cp.width = c.width; cp.height = c.height; cp.np = h->np;
    cp.a_min = c.a_min; cp.max_boxes = c.max_boxes;
    cp.parent = cp_parent;
    cp.rec = reinterpret_cast<int32_t *>(ws + h->off_rec);
    cp.tile_state = reinterpret_cast<int32_t *>(ws + h->off_ctiles);
    ip.ccl_tile_state = cp.tile_state;
    cp.boxes = out->boxes; cp.counters = out->counters;
    cp.merged = (c.merge_alpha > 0.f) ? out->merged_boxes : nullptr;
    cp.merge_alpha = c.merge_alpha;
    cp.merge_parent = cp.merged ? reinterpret_cast<int32_t *>(ws + h->off_merge) : nullptr;
    cp.merge_rec = cp.merge_parent ? cp.merge_parent + c.max_boxes : nullptr;
    cp.merge_sync = ip.sync + 8;

    int launches = 0;
    if (timing) cudaEventRecord(h->ev[0], st);
    launches += (mode == 2) ? launch_ingest_slide(ip, st) : launch_ingest(ip, st);
    if (timing) cudaEventRecord(h->ev[1], st);
    if (use_nufft) {
        NufftParams nq{};
        nq.nd = np; nq.hot = ip.hot_work; nq.n_hot = ip.sync + 15; nq.cursor = ip.hot_cursor;
        nq.g_c = h->g_nc; nq.g_t = h->g_nt;
        nq.scratch = reinterpret_cast<float *>(ws + h->off_nuscr);
        launches += launch_nufft(nq, h->sm_count, st);
    }
    NdftParams seg = np;                                   // the segment pass of the lean variant
    seg.work = ip.seg_work; seg.n_work = ip.sync + 9; seg.work_cursor = ip.work_cursor2;
    launches += launch_ndft(np, ip.seg_work ? &seg : nullptr, c.n_freq, h->band_size, h->fallback,
                            h->sm_count * h->ndft_blocks_per_sm, h->sm_count * h->full_blocks_per_sm,
                            h->sm_count * h->score_blocks_per_sm, st, timing ? h->ev[2] : nullptr);
    if (timing) cudaEventRecord(h->ev[3], st);
    launches += launch_ccl(cp, st);
    if (timing) { cudaEventRecord(h->ev[4], st); h->timed_once = true; }
    h->launches = launches;
    const cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return fail(h, DDHF_E_CUDA, std::string("ddhf_window: ") + cudaGetErrorString(e));
    return DDHF_OK;
}

extern "C" int ddhf_window(ddhf_handle *h, const ddhf_event *d_events, int64_t n, int64_t t0_us,
                           int64_t window_us, void *d_workspace, const ddhf_outputs *out,
                           void *cuda_stream)
{
    return run_window(h, d_events, n, t0_us, window_us, d_workspace, out, cuda_stream, 0, 0);
}

extern "C" int ddhf_window_packed(ddhf_handle *h, const ddhf_event8 *d_events, int64_t n, int64_t t_base_us, int64_t t0_us,
                                  int64_t window_us, void *d_workspace, const ddhf_outputs *out, void *cuda_stream)
{
    return run_window(h, reinterpret_cast<const ddhf_event *>(d_events), n, t0_us, window_us, d_workspace, out, cuda_stream,
                      0, 0, true, t_base_us);
}

extern "C" int ddhf_window_slide(ddhf_handle *h, const ddhf_event *d_new_events, int64_t n_new, int64_t t0_us,
                                 int64_t window_us, void *d_workspace, const ddhf_outputs *out,
                                 void *cuda_stream)
{
    if (!h) return DDHF_E_INVAL;
    // a continuation needs the state of the previous call: same workspace, same window length, t0 not
    // moved backwards and by less than a window; anything else starts a new sequence from scratch
    const bool cont = h->slide_valid && h->slide_ws == d_workspace && h->slide_window == window_us &&
                      t0_us >= h->slide_t0 && t0_us - h->slide_t0 < window_us;
    const int rc = run_window(h, d_new_events, n_new, t0_us, window_us, d_workspace, out, cuda_stream,
                              cont ? 2 : 1, cont ? t0_us - h->slide_t0 : 0);
    if (rc != DDHF_OK) { h->slide_valid = false; return rc; }
    h->slide_valid = true;
    h->slide_t0 = t0_us;
    h->slide_window = window_us;
    h->slide_ws = d_workspace;
    h->slide_parity ^= 1;
    return DDHF_OK;
}

extern "C" int ddhf_slide_reset(ddhf_handle *h)
{
    if (!h) return DDHF_E_INVAL;
    h->slide_valid = false;
    return DDHF_OK;
}

extern "C" int ddhf_stage_ms(ddhf_handle *h, float *ms)
{
    if (!h || !ms) return DDHF_E_INVAL;
    if (!(h->cfg.flags & DDHF_FLAG_TIMING) || !h->timed_once)
        return fail(h, DDHF_E_INVAL, "ddhf_stage_ms: handle was not created with DDHF_FLAG_TIMING or no window ran");
    if (cudaEventSynchronize(h->ev[4]) != cudaSuccess)
        return fail(h, DDHF_E_CUDA, std::string("ddhf_stage_ms: ") + cudaGetErrorString(cudaGetLastError()));
    for (int i = 0; i < 4; ++i) cudaEventElapsedTime(&ms[i], h->ev[i], h->ev[i + 1]);
    cudaEventElapsedTime(&ms[4], h->ev[0], h->ev[4]);
    return DDHF_OK;
}

// ---- device buffers owned by the handle for the host-buffer entry points -----------------------
// One set for ddhf_window_host(), two for the pipeline of ddhf_host_submit().  A set is either
// complete or absent: a failed allocation frees what was allocated before it.
static void free_set(ddhf_event *&events, void *&ws, ddhf_outputs &o)
{
    void *bufs[] = {events, ws, o.row_ptr, o.csr_ev, o.active_idx, o.power, o.sf, o.score, o.f0_idx, o.mask,
                    o.labels, o.boxes, o.counters, o.merged_boxes};
    for (void *b : bufs) if (b) cudaFree(b);
    events = nullptr;
    ws = nullptr;
    o = ddhf_outputs{};
}

static cudaError_t alloc_set(const ddhf_handle *h, ddhf_event *&events, void *&ws, ddhf_outputs &o)
{
    const ddhf_config &c = h->cfg;
    const size_t np = h->np;
    o = ddhf_outputs{};
    events = nullptr;
    ws = nullptr;
    cudaError_t e = cudaSuccess;
    auto get = [&e](auto &ptr, size_t bytes) {
        if (e == cudaSuccess) e = cudaMalloc(reinterpret_cast<void **>(&ptr), bytes ? bytes : 1);
    };
    get(events, sizeof(ddhf_event) * static_cast<size_t>(c.max_events));
    get(ws, h->ws_bytes);
    get(o.row_ptr, sizeof(int32_t) * (np + 1));
    get(o.csr_ev, sizeof(uint32_t) * static_cast<size_t>(c.max_events));
    get(o.active_idx, sizeof(int32_t) * static_cast<size_t>(c.max_active));
    get(o.sf, sizeof(float) * np);
    get(o.score, sizeof(float) * np);
    get(o.f0_idx, sizeof(int32_t) * np);
    get(o.mask, np);
    get(o.labels, sizeof(int32_t) * np);
    get(o.boxes, sizeof(ddhf_box) * static_cast<size_t>(c.max_boxes));
    get(o.merged_boxes, sizeof(ddhf_box) * static_cast<size_t>(c.max_boxes));
    get(o.counters, sizeof(int32_t) * DDHF_N_COUNTERS);
    if (e != cudaSuccess) free_set(events, ws, o);
    return e;
}

static int check_host_args(ddhf_handle *h, const char *who, const ddhf_event *h_events, int64_t n,
                           int64_t window_us, const ddhf_host_outputs *out)
{
    if (!out || (n > 0 && !h_events)) return fail(h, DDHF_E_INVAL, std::string(who) + ": NULL argument");
    if (n < 0 || window_us <= 0 || window_us >= (1ll << 31))
        return fail(h, DDHF_E_INVAL, std::string(who) + ": n or window_us out of range");
    if (n > h->cfg.max_events) return fail(h, DDHF_E_CAPACITY, std::string(who) + ": n > max_events");
    return DDHF_OK;
}

#define HB_CHECK(call)                                                                         \
    do {                                                                                       \
        const cudaError_t e_ = (call);                                                         \
        if (e_ != cudaSuccess)                                                                 \
            return fail(h, DDHF_E_CUDA, std::string("ddhf_window_host: ") + cudaGetErrorString(e_)); \
    } while (0)

extern "C" int ddhf_window_host(ddhf_handle *h, const ddhf_event *h_events, int64_t n, int64_t t0_us,
                                int64_t window_us, const ddhf_host_outputs *out, void *cuda_stream)
{
    if (!h) return DDHF_E_INVAL;
    const int arg_rc = check_host_args(h, "ddhf_window_host", h_events, n, window_us, out);     // before any copy
    if (arg_rc != DDHF_OK) return arg_rc;
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    const ddhf_config &c = h->cfg;
    const size_t np = h->np;
    if (!h->hb_ready) {
        HB_CHECK(alloc_set(h, h->hb_events, h->hb_ws, h->hb_out));
        h->hb_ready = true;
    }
    if (out->power && !h->hb_out.power)
        HB_CHECK(cudaMalloc(&h->hb_out.power, sizeof(float) * static_cast<size_t>(c.max_active) * c.n_freq));
    ddhf_outputs dev = h->hb_out;
    if (!out->power) dev.power = nullptr;

    if (n > 0) HB_CHECK(cudaMemcpyAsync(h->hb_events, h_events, sizeof(ddhf_event) * static_cast<size_t>(n),
                                        cudaMemcpyHostToDevice, st));
    const int rc = ddhf_window(h, h->hb_events, n, t0_us, window_us, h->hb_ws, &dev, st);
    if (rc != DDHF_OK) { cudaStreamSynchronize(st); return rc; }

    int32_t cnt[DDHF_N_COUNTERS];
    HB_CHECK(cudaMemcpyAsync(cnt, dev.counters, sizeof(cnt), cudaMemcpyDeviceToHost, st));
    if (out->mask) HB_CHECK(cudaMemcpyAsync(out->mask, dev.mask, np, cudaMemcpyDeviceToHost, st));
    if (out->sf) HB_CHECK(cudaMemcpyAsync(out->sf, dev.sf, sizeof(float) * np, cudaMemcpyDeviceToHost, st));
    if (out->score) HB_CHECK(cudaMemcpyAsync(out->score, dev.score, sizeof(float) * np, cudaMemcpyDeviceToHost, st));
    if (out->f0_idx) HB_CHECK(cudaMemcpyAsync(out->f0_idx, dev.f0_idx, sizeof(int32_t) * np, cudaMemcpyDeviceToHost, st));
    if (out->labels) HB_CHECK(cudaMemcpyAsync(out->labels, dev.labels, sizeof(int32_t) * np, cudaMemcpyDeviceToHost, st));
    if (out->row_ptr) HB_CHECK(cudaMemcpyAsync(out->row_ptr, dev.row_ptr, sizeof(int32_t) * (np + 1), cudaMemcpyDeviceToHost, st));
    HB_CHECK(cudaStreamSynchronize(st));
    const size_t n_in = static_cast<size_t>(cnt[DDHF_CNT_N_IN]);
    const size_t n_act = static_cast<size_t>(cnt[DDHF_CNT_N_ACTIVE] < c.max_active ? cnt[DDHF_CNT_N_ACTIVE] : c.max_active);
    const size_t n_box = static_cast<size_t>(cnt[DDHF_CNT_N_BOXES]);
    if (out->counters) memcpy(out->counters, cnt, sizeof(cnt));
    if (out->csr_ev && n_in) HB_CHECK(cudaMemcpyAsync(out->csr_ev, dev.csr_ev, sizeof(uint32_t) * n_in, cudaMemcpyDeviceToHost, st));
    if (out->active_idx && n_act) HB_CHECK(cudaMemcpyAsync(out->active_idx, dev.active_idx, sizeof(int32_t) * n_act, cudaMemcpyDeviceToHost, st));
    if (out->power && n_act) HB_CHECK(cudaMemcpyAsync(out->power, dev.power, sizeof(float) * n_act * c.n_freq, cudaMemcpyDeviceToHost, st));
    if (out->boxes && n_box) HB_CHECK(cudaMemcpyAsync(out->boxes, dev.boxes, sizeof(ddhf_box) * n_box, cudaMemcpyDeviceToHost, st));
    const size_t n_mrg = static_cast<size_t>(cnt[DDHF_CNT_N_MERGED]);
    if (out->merged_boxes && n_mrg) HB_CHECK(cudaMemcpyAsync(out->merged_boxes, dev.merged_boxes, sizeof(ddhf_box) * n_mrg, cudaMemcpyDeviceToHost, st));
    HB_CHECK(cudaStreamSynchronize(st));
    return DDHF_OK;
}

static int host_submit(ddhf_handle *h, const void *h_events, int64_t n, int64_t t0_us, int64_t window_us,
                       const ddhf_host_outputs *out, void *cuda_stream, bool packed, int64_t t_base_us)
{
    if (!h) return DDHF_E_INVAL;
    const int arg_rc = check_host_args(h, "ddhf_host_submit", static_cast<const ddhf_event *>(h_events), n, window_us, out);
    if (arg_rc != DDHF_OK) return arg_rc;
    if (out->csr_ev || out->active_idx || out->power)
        return fail(h, DDHF_E_INVAL, "ddhf_host_submit: csr_ev, active_idx and power are not available in the pipelined call");
    if (h->pipe_head - h->pipe_tail >= 2)
        return fail(h, DDHF_E_INVAL, "ddhf_host_submit: two windows already in flight, call ddhf_host_wait");
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    const ddhf_config &c = h->cfg;
    const size_t np = h->np;
    auto cuda_fail = [h](cudaError_t e) {
        return fail(h, DDHF_E_CUDA, std::string("ddhf_host_submit: ") + cudaGetErrorString(e));
    };
    if (!h->pipe_ready) {
        // all or nothing: a failure part-way leaves no buffer behind, so the next call starts clean
        cudaError_t e = cudaSuccess;
        if (!h->copy_stream) e = cudaStreamCreateWithFlags(&h->copy_stream, cudaStreamNonBlocking);
        if (e == cudaSuccess && !h->d2h_stream) e = cudaStreamCreateWithFlags(&h->d2h_stream, cudaStreamNonBlocking);
        for (auto &s : h->pipe) {
            if (e == cudaSuccess) e = alloc_set(h, s.events, s.ws, s.out);
            if (e == cudaSuccess && !s.copied) e = cudaEventCreateWithFlags(&s.copied, cudaEventDisableTiming);
            if (e == cudaSuccess && !s.kernels) e = cudaEventCreateWithFlags(&s.kernels, cudaEventDisableTiming);
            if (e == cudaSuccess && !s.done) e = cudaEventCreateWithFlags(&s.done, cudaEventDisableTiming);
        }
        if (e != cudaSuccess) {
            for (auto &s : h->pipe) free_set(s.events, s.ws, s.out);
            return cuda_fail(e);
        }
        h->pipe_ready = true;
    }
    ddhf_handle::PipeSlot &s = h->pipe[h->pipe_head & 1];
    // the slot's previous window (two submits ago) has been waited for, so its buffers are free
    cudaError_t e = cudaSuccess;
    if (n > 0) e = cudaMemcpyAsync(s.events, h_events, (packed ? sizeof(ddhf_event8) : sizeof(ddhf_event)) * static_cast<size_t>(n),
                                   cudaMemcpyHostToDevice, h->copy_stream);
    if (e == cudaSuccess) e = cudaEventRecord(s.copied, h->copy_stream);
    if (e == cudaSuccess) e = cudaStreamWaitEvent(st, s.copied, 0);
    if (e != cudaSuccess) {
        cudaStreamSynchronize(h->copy_stream);            // nothing was enqueued on `st`: the slot stays free
        return cuda_fail(e);
    }
    const int rc = run_window(h, s.events, n, t0_us, window_us, s.ws, &s.out, st, 0, 0, packed, t_base_us);
    const ddhf_outputs &d = s.out;
    // the results leave on a stream of their own, so that the next window's kernels start at once
    auto d2h = [&](void *dst, const void *src, size_t bytes) {
        if (e == cudaSuccess && dst) e = cudaMemcpyAsync(dst, src, bytes, cudaMemcpyDeviceToHost, h->d2h_stream);
    };
    if (rc == DDHF_OK) {
        e = cudaEventRecord(s.kernels, st);
        if (e == cudaSuccess) e = cudaStreamWaitEvent(h->d2h_stream, s.kernels, 0);
        d2h(out->counters, d.counters, sizeof(int32_t) * DDHF_N_COUNTERS);
        d2h(out->mask, d.mask, np);
        d2h(out->boxes, d.boxes, sizeof(ddhf_box) * static_cast<size_t>(c.max_boxes));
        d2h(out->merged_boxes, d.merged_boxes, sizeof(ddhf_box) * static_cast<size_t>(c.max_boxes));
        d2h(out->sf, d.sf, sizeof(float) * np);
        d2h(out->score, d.score, sizeof(float) * np);
        d2h(out->f0_idx, d.f0_idx, sizeof(int32_t) * np);
        d2h(out->labels, d.labels, sizeof(int32_t) * np);
        d2h(out->row_ptr, d.row_ptr, sizeof(int32_t) * (np + 1));
    }
    if (rc != DDHF_OK || e != cudaSuccess) {
        // kernels or copies of this window may already be queued on the slot's buffers: drain them so
        // that the slot can be reused by the next submit, and report the failure (nothing is in flight)
        cudaStreamSynchronize(st);
        cudaStreamSynchronize(h->d2h_stream);
        return rc != DDHF_OK ? rc : cuda_fail(e);
    }
    if ((e = cudaEventRecord(s.done, h->d2h_stream)) != cudaSuccess) {
        cudaStreamSynchronize(st);
        cudaStreamSynchronize(h->d2h_stream);
        return cuda_fail(e);
    }
    ++h->pipe_head;
    return DDHF_OK;
}

extern "C" int ddhf_host_submit(ddhf_handle *h, const ddhf_event *h_events, int64_t n, int64_t t0_us,
                                int64_t window_us, const ddhf_host_outputs *out, void *cuda_stream)
{
    return host_submit(h, h_events, n, t0_us, window_us, out, cuda_stream, false, 0);
}

extern "C" int ddhf_host_submit_packed(ddhf_handle *h, const ddhf_event8 *h_events, int64_t n, int64_t t_base_us, int64_t t0_us,
                                       int64_t window_us, const ddhf_host_outputs *out, void *cuda_stream)
{
    return host_submit(h, h_events, n, t0_us, window_us, out, cuda_stream, true, t_base_us);
}

extern "C" int ddhf_host_wait(ddhf_handle *h)
{
    if (!h) return DDHF_E_INVAL;
    if (h->pipe_head == h->pipe_tail) return fail(h, DDHF_E_INVAL, "ddhf_host_wait: no window in flight");
    ddhf_handle::PipeSlot &s = h->pipe[h->pipe_tail & 1];
    const cudaError_t e = cudaEventSynchronize(s.done);
    ++h->pipe_tail;
    if (e != cudaSuccess) return fail(h, DDHF_E_CUDA, std::string("ddhf_host_wait: ") + cudaGetErrorString(e));
    return DDHF_OK;
}

extern "C" int ddhf_fma_peak_probe(float ms_target, float *tflops_out, void *cuda_stream)
{
    if (!tflops_out) return DDHF_E_INVAL;
    return fma_probe(ms_target, tflops_out, static_cast<cudaStream_t>(cuda_stream));
}

extern "C" int ddhf_destroy(ddhf_handle *h)
{
    if (!h) return DDHF_OK;
    if (h->d_tables) cudaFree(h->d_tables);
    for (int i = 0; i < 5; ++i) if (h->ev[i]) cudaEventDestroy(h->ev[i]);
    free_set(h->hb_events, h->hb_ws, h->hb_out);
    for (auto &s : h->pipe) {
        free_set(s.events, s.ws, s.out);
        if (s.copied) cudaEventDestroy(s.copied);
        if (s.kernels) cudaEventDestroy(s.kernels);
        if (s.done) cudaEventDestroy(s.done);
    }
    if (h->copy_stream) cudaStreamDestroy(h->copy_stream);
    if (h->d2h_stream) cudaStreamDestroy(h->d2h_stream);
    delete h;
    return DDHF_OK;
}
