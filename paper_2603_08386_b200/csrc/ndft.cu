// ndft.cu -- a4-a7: per-pixel NDFT power spectrum and spectral flatness (k_ndft_score) and the
// harmonic-comb score of the pixels that pass the SF filter (k_comb_deferred).
//
//   a4  X_j = sum_k w_k exp(-2 pi i f_j t_k),  P_j = |X_j|^2          (eq. 6)
//   a5  SF = geometric mean / arithmetic mean of P                  (eq. 7)
//   a6  SNR_M(w) = N(w) / median(P outside the harmonic windows)    (eq. 8-10)
//   a7  mask = SF <= tau_sf and max_w SNR_M >= tau_comb              (L107, eq. 11)
//
// Design (B200, plain FP32 pipes -- the per-pixel Vandermonde has no operand shared between
// pixels, so this is ALU work, not a tensor-core contraction):
//
// * One warp owns one pixel at a time and all of its bins; lane l holds the bins
//   j = l + 32 i, i < NBL.  Warps pull pixels from a device-side queue ordered by
//   descending row length, so the heavy tail (config 4) is spread over the grid.
// * The direct sum is factorised exactly, not approximated: with the bins of a lane split
//   into TM groups of 2 TN bins around a centre frequency, f_j = f_c +- (m + 1/2) 32 df and
//       w e^{-i th_c} e^{-+i ph_m}
//   needs only the four real products a_r b_r, a_r b_i, a_i b_r, a_i b_i of the centre
//   phasor a (per lane, per event) and the offset phasor b (shared by all lanes, per event,
//   read as a shared-memory broadcast).  Accumulating those four products costs 4 FMA for 2
//   bins = 2 FMA per (pixel, bin, event) term, issued as packed FFMA2 (fma.rn.f32x2).  There
//   is no recurrence along frequency or time, hence no drift to resync.
// * Phases are exact 32-bit fixed point "turns": hi32(G * t) with G = 2^64 f 1e-6, so a
//   5 kHz x 0.1 s = 500-cycle phase keeps 2^-32 turn resolution before it reaches the SFU.
// * Power and spectral flatness are the kernel's epilogue, straight from the accumulators; the
//   optional compact spectrum output is a streaming store.  A pixel that needs the comb score
//   queues its spectrum (8 KB) for k_comb_deferred, which runs the latency-bound scoring code at
//   an occupancy this 168-register kernel cannot offer; when the queue is full the same
//   comb_score() runs in place, so the result does not depend on the path.
// * The complement median of every candidate is an order statistic of the full spectrum
//   in a narrow rank band [r0, r1] known at create time.  The band is isolated by a few
//   counting passes over the spectrum, sorted once per pixel in registers (bitonic), and each
//   candidate then only corrects the rank for its own excluded bins (prefix counts from warp
//   ballots + a bitmask of excluded in-band positions).  Window maxima of eq. 8 come from a
//   table of forward block maxima built by warp shuffles.
#include "comb.cuh"

namespace ddhf {

namespace {

#ifndef DDHF_NDFT_WARPS
#define DDHF_NDFT_WARPS 12         // warps per CTA: 12 x 32 threads x 168 registers fill the 64 K register file
#endif
#ifndef DDHF_NDFT_HEAD_WARPS
#define DDHF_NDFT_HEAD_WARPS 2     // of every 3 warps, how many start from the long-row end of the work list
#endif
#ifndef DDHF_PU
#define DDHF_PU 4                 // table passes issued together
#endif
#ifndef DDHF_NDFT_BLOCKS
#define DDHF_NDFT_BLOCKS 1         // CTAs per SM
#endif
constexpr int kWarps = DDHF_NDFT_WARPS;
#ifndef DDHF_NDFT_WARPS_SMALL
#define DDHF_NDFT_WARPS_SMALL 16   // kernels of <= 32 bins per lane need <= 128 registers: four warps per sub-partition
#endif
// warps per CTA of the kernel with NBL bins per lane
__host__ __device__ constexpr int warps_of(int nbl) { return nbl >= 64 ? kWarps : DDHF_NDFT_WARPS_SMALL; }
constexpr int kEC = 32;            // events per table chunk
constexpr unsigned kFull = 0xffffffffu;

// Per-warp shared memory of k_ndft_score: the phasor table / phase words of the event loop and the
// staged CSR events; the scoring scratch of comb.cuh (in-place scoring, only when the deferred queue is
// full) aliases the table.  INPLACE = false (lean variant, or band sorter of 1024 values): the queue holds every pixel,
// and the small layout leaves the L1 cache to the kernel's spills and global loads.
template <int TM, int TN, int BS, bool FB>
struct Layout {
    static constexpr int NBL = TM * 2 * TN;                 // bins per lane
    static constexpr int NB = NBL * 32;                     // padded spectrum length
    static constexpr bool INPLACE = FB && BS <= 512;
    static constexpr int TAB_WORDS = kEC * TN * 2 + kEC * 4;
    static constexpr int EV_WORDS = 2 * kEC;                // staged CSR events, double buffered
    __host__ __device__ static constexpr int scratch_words(int cpad)
    {
        return INPLACE && CombSmem<NBL, BS>::words(cpad) > TAB_WORDS ? CombSmem<NBL, BS>::words(cpad) : TAB_WORDS;
    }
    __host__ __device__ static constexpr int warp_words(int cpad) { return ((scratch_words(cpad) + EV_WORDS + 3) / 4) * 4; }
    static size_t smem_bytes(int cpad) { return static_cast<size_t>(warp_words(cpad)) * 4 * warps_of(NBL); }
};

__device__ __forceinline__ uint32_t phase_u32(uint64_t g, uint32_t t)
{
    // hi 32 bits of (g * t mod 2^64): the phase f*t in turns, 2^-32 resolution
    return static_cast<uint32_t>(g >> 32) * t + __umulhi(static_cast<uint32_t>(g), t);
}

// (sin, cos) of 2 pi (turns - 1/2), turns = ph / 2^32.  The half-turn offset only flips the
// sign of both components; every phasor of the kernel carries it, and centre x offset
// phasors are always multiplied, so it cancels.  Argument of the SFU is in [-pi, pi).
__device__ __forceinline__ void sincos_u32(uint32_t ph, float &s, float &c)
{
    // 1 + turns in [1, 2) from the top 23 phase bits; 2 pi (that - 3/2) in one FMA
    const float r = fmaf(__uint_as_float((ph >> 9) | 0x3f800000u), 6.283185307179586f, -9.42477796076938f);
    s = __sinf(r);
    c = __cosf(r);
}

// The work list is ordered by descending row length.  Warps take items from both ends: "head"
// warps the long rows (FMA-pipe bound), "tail" warps the short ones (dominated by the
// per-pixel epilogue, latency bound), so that every SM sub-partition always holds a mix of
// the two and neither the FMA pipe nor the issue slots sit idle for a whole phase of the
// kernel.  One 64-bit counter holds both cursors; an item is valid while head + tail < n.
// Tail warps claim kTailBatch items per atomic (short rows cost about a thousand cycles each, so a
// global atomic per pixel is a visible stall); item i of a claim made at (h, t) is valid while
// h + t + i < n.  Returns the first index of the claim and its valid count.
#ifndef DDHF_TAIL_BATCH
#define DDHF_TAIL_BATCH 4
#endif
constexpr int kTailBatch = DDHF_TAIL_BATCH;
constexpr unsigned kTailBatchMinLeft = 65536u;      // items left below which tail warps stop batching

__device__ __forceinline__ int fetch_items(unsigned long long *cursor, bool head, int n_items, int &cnt, unsigned &seen_used)
{
    // near the end of the list (or in a short list, where the tail holds long rows or segments of a split
    // row) tail warps claim one item at a time, so that no warp sits on a batch of expensive items while
    // others idle.  `seen_used` = items handed out as of this warp's previous claim: a hint, the atomic decides.
    const unsigned n = static_cast<unsigned>(n_items);
    const bool batch = !head && seen_used + kTailBatchMinLeft < n;
    const unsigned b = batch ? static_cast<unsigned>(kTailBatch) : 1u;
    const unsigned long long old = atomicAdd(cursor, head ? (1ull << 32) : static_cast<unsigned long long>(b));
    const unsigned h = static_cast<unsigned>(old >> 32), t = static_cast<unsigned>(old);
    const unsigned used = h + t;
    seen_used = used;
    cnt = (used >= n) ? 0 : static_cast<int>(min(b, n - used));
    return head ? static_cast<int>(h) : n_items - 1 - static_cast<int>(t);
}

__device__ __forceinline__ void stage_event(uint32_t *dst_smem, const uint32_t *src)
{
    const unsigned d = static_cast<unsigned>(__cvta_generic_to_shared(dst_smem));
    asm volatile("cp.async.ca.shared.global [%0], [%1], 4;" ::"r"(d), "l"(src) : "memory");
}

__device__ __forceinline__ void stage_wait()
{
    asm volatile("cp.async.wait_all;" ::: "memory");
}

__device__ __forceinline__ WorkItem make_item()
{
    WorkItem w;
    w.row_begin = 0; w.n = 0; w.pix = 0; w.arow = 0;
    return w;
}

// ----------------------------------------------------------------------------------------
// The fused kernel.
// ----------------------------------------------------------------------------------------
// FULL: n_freq fills the padded grid (n_freq == 32 NBL) and k_lo <= 32, so no per-bin range checks
// FB: carries the in-place scoring fallback for a full queue (launched only when the queue is smaller than
// the sensor: the fallback's code costs the lean kernel 1.7 % of its time just by being there)
template <int TM, int TN, int BS, bool FULL, bool FB>
#ifdef DDHF_NDFT_MAXNREG
__global__ void __maxnreg__(DDHF_NDFT_MAXNREG) k_ndft_score(NdftParams p)
#else
__global__ void __launch_bounds__(warps_of(TM * 2 * TN) * 32, DDHF_NDFT_BLOCKS) k_ndft_score(NdftParams p)
#endif
{
    using L = Layout<TM, TN, BS, FB>;
    constexpr int NBL = L::NBL;
    extern __shared__ __align__(16) uint32_t smem_raw[];
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    const int cpad = p.sp.cpad;
    uint32_t *scr = smem_raw + wid * L::warp_words(cpad);
    float2 *btab = reinterpret_cast<float2 *>(scr);                 // [kEC][TN]
    uint4 *phs = reinterpret_cast<uint4 *>(scr + kEC * TN * 2);     // [kEC]

    const int n_items = *p.n_work;                     // active pixels + the extra segments of split rows
    const ScoreParams &sp = p.sp;
    constexpr int EPP = 32 / TN;       // events per table pass
    constexpr bool full_grid = FULL;
    const bool store_power = p.power != nullptr;

    // dynamic work queue with one item of look-ahead: the next work item is loaded while the
    // current pixel is being processed, and its first events are staged in shared memory by
    // cp.async (no register holds data in flight, so nothing waits on a spill)
    uint32_t *ev_s = scr + L::scratch_words(cpad);                  // [2][kEC]
    int evb = 0;                                                    // staging buffer in use
    const bool head = (wid % 3) < DDHF_NDFT_HEAD_WARPS;
    int claim_left = 0;                                             // items of the current claim not yet started
    int idx = 0;
    unsigned seen_used = 0u;
    if (lane == 0) idx = fetch_items(p.work_cursor, head, n_items, claim_left, seen_used);
    idx = __shfl_sync(kFull, idx, 0);
    claim_left = __shfl_sync(kFull, claim_left, 0);
    if (claim_left == 0) idx = n_items;
    --claim_left;
    WorkItem it_next = make_item();
    if (idx < n_items) {
        it_next = p.work[idx];
        if (lane < it_next.n) stage_event(ev_s + lane, p.csr_ev + it_next.row_begin + lane);
    }

    while (idx < n_items) {
        const WorkItem it = it_next;
        // next item: the following one of the claim (tail warps walk down the list), or a new claim
        // (claimed before the row is processed, except by the segments of a split row: a warp that starts a
        // segment must not sit on a second one that an idle warp could take)
        int next_idx = idx - 1, next_cnt = claim_left;
        const bool claim_early = it.pix >= 0;
        if (claim_left <= 0 && claim_early && lane == 0) next_idx = fetch_items(p.work_cursor, head, n_items, next_cnt, seen_used);

        float2 acc1[TM][TN], acc2[TM][TN];     // (S1, S4) and (S3, S2)
#pragma unroll
        for (int g = 0; g < TM; ++g)
#pragma unroll
            for (int m = 0; m < TN; ++m) {
                acc1[g][m] = make_float2(0.f, 0.f);
                acc2[g][m] = make_float2(0.f, 0.f);
            }

        // an active pixel has at least one event: do-while, so the accumulators are set up once
        int base = 0;
        do {
            const int nc = min(kEC, it.n - base);
            // ---- per-event phase words and the offset-phasor table of this chunk ----------
            stage_wait();
            const uint32_t v = ev_s[evb * kEC + lane];
            evb ^= 1;
            if (base + kEC + lane < it.n)                         // stage the next chunk
                stage_event(ev_s + evb * kEC + lane, p.csr_ev + it.row_begin + base + kEC + lane);
            if (lane < nc) {
                const uint32_t t = v >> 1;
                // .w: sign mask of the weight, w = +1 if bit 0 of the CSR value else -1
                phs[lane] = make_uint4(phase_u32(p.g_f0, t), phase_u32(p.g_d, t), phase_u32(p.g_h, t),
                                       (v & 1u) ? 0u : 0x80000000u);
            }
            __syncwarp();
            const int n_pass = (nc + EPP - 1) / EPP;
            // PU passes at a time: their phase -> SFU -> store chains are independent
            constexpr int PU = (kEC / EPP) < DDHF_PU ? (kEC / EPP) : DDHF_PU;
            {
                const int e_l = lane / TN, m_l = lane % TN;
                const uint32_t mult = static_cast<uint32_t>(2 * m_l + 1);
#pragma unroll 1
                for (int ps0 = 0; ps0 < n_pass; ps0 += PU) {
#pragma unroll
                    for (int u = 0; u < PU; ++u) {
                        const int e = (ps0 + u) * EPP + e_l;
                        if (e < kEC) {
                            const uint2 hw = *reinterpret_cast<const uint2 *>(&phs[e].z);
                            float sn, cs;
                            sincos_u32(hw.x * mult, sn, cs);
                            // b = w e^{-i phi} up to the common sign of every phasor of the kernel
                            btab[e * TN + m_l] = make_float2(__uint_as_float(__float_as_uint(cs) ^ hw.y),
                                                             __uint_as_float(__float_as_uint(sn) ^ hw.y));
                        }
                    }
                }
            }
            __syncwarp();
            // ---- accumulate: 4 real products per (centre, offset pair, event) --------------
            // software pipelined by hand, two events per trip: the centre phasors of the next
            // event (shared-memory read, integer phase, two SFU ops per centre) are produced under
            // the FFMA2 block of the current one, in alternating register sets (no copies)
            static_assert(TM <= 2, "centre stride is applied as one shift");
            constexpr int kLog4TN = (TN == 16) ? 6 : (TN == 8) ? 5 : (TN == 4) ? 4 : 3;
            float a0r[TM], a0i[TM], a1r[TM], a1i[TM];
            const uint32_t lane_u = static_cast<uint32_t>(lane);
#define DDHF_CENTRES(AR, AI, K)                                                                  \
            {                                                                                    \
                const uint4 ph = phs[K];                                                         \
                const uint32_t pc0 = ph.x + lane_u * ph.y;                                       \
                _Pragma("unroll") for (int g = 0; g < TM; ++g)                                   \
                    sincos_u32(pc0 + (g ? (ph.z << kLog4TN) : 0u), AI[g], AR[g]);               \
            }
#define DDHF_FMA_BLOCK(AR, AI, K)                                                                \
            {                                                                                    \
                const float4 *brow = reinterpret_cast<const float4 *>(btab + (K) * TN);          \
                _Pragma("unroll") for (int m2 = 0; m2 < TN / 2; ++m2) {                          \
                    const float4 bb = brow[m2];                                                  \
                    const float2 b0 = make_float2(bb.x, bb.y), b1 = make_float2(bb.z, bb.w);     \
                    _Pragma("unroll") for (int g = 0; g < TM; ++g) {                             \
                        const float2 arr = make_float2(AR[g], AR[g]), aii = make_float2(AI[g], AI[g]); \
                        acc1[g][2 * m2] = __ffma2_rn(arr, b0, acc1[g][2 * m2]);                  \
                        acc2[g][2 * m2] = __ffma2_rn(aii, b0, acc2[g][2 * m2]);                  \
                        acc1[g][2 * m2 + 1] = __ffma2_rn(arr, b1, acc1[g][2 * m2 + 1]);          \
                        acc2[g][2 * m2 + 1] = __ffma2_rn(aii, b1, acc2[g][2 * m2 + 1]);          \
                    }                                                                            \
                }                                                                                \
            }
            const int nce = nc;
            DDHF_CENTRES(a0r, a0i, 0)
            int k = 0;
#pragma unroll 1
            for (; k + 1 < nce; k += 2) {
                DDHF_CENTRES(a1r, a1i, k + 1)
                DDHF_FMA_BLOCK(a0r, a0i, k)
                DDHF_CENTRES(a0r, a0i, min(k + 2, nce - 1))
                DDHF_FMA_BLOCK(a1r, a1i, k + 1)
            }
            if (k < nce) DDHF_FMA_BLOCK(a0r, a0i, k)
#undef DDHF_CENTRES
#undef DDHF_FMA_BLOCK
            __syncwarp();
            base += kEC;
        } while (base < it.n);

        // the next pixel's work item and first events are fetched under the epilogue
        if (claim_left <= 0) {
            if (!claim_early && lane == 0) next_idx = fetch_items(p.work_cursor, head, n_items, next_cnt, seen_used);
            idx = __shfl_sync(kFull, next_idx, 0);
            claim_left = __shfl_sync(kFull, next_cnt, 0);
            if (claim_left == 0) idx = n_items;
        } else {
            idx = next_idx;
        }
        --claim_left;
        if (idx < n_items) it_next = p.work[idx];

        // ---- split rows: a row longer than kSplitMin events is accumulated by several warps, one segment
        // of <= kSegEvents events each (S1..S4 are linear in the events).  The partial sums are combined
        // along a fixed tree of fan-in kSplitFan: the warp that arrives last at a node adds the node's
        // children in index order, whoever that warp is, so the result does not depend on the schedule;
        // the warp that completes the root runs the row's epilogue.
        int out_pix = it.pix, out_arow = it.arow;
        if ((FB || NBL < 64) && it.pix < 0) {     // (the 168-register 2048-bin lean kernel leaves segments to a second pass)
            const SplitRow *sr = p.split_tab + (it.pix & 0x7fffffff);
            constexpr int PW = 2 * NBL * 32;                       // floats per partial
            int n_l = sr->n_seg, idx_l = it.arow;                  // nodes of the current level, this warp's node
            int slot0 = sr->seg_base, cnt0 = sr->cnt_base;         // first partial / first counter of the level
            bool last = true;
            while (n_l > 1) {
                float *mine = p.split_partial + static_cast<size_t>(slot0 + idx_l) * PW + lane;
#pragma unroll
                for (int g = 0; g < TM; ++g)
#pragma unroll
                    for (int m = 0; m < TN; ++m) {
                        const int k = (g * TN + m) * 4;
                        __stcg(mine + (k + 0) * 32, acc1[g][m].x);
                        __stcg(mine + (k + 1) * 32, acc1[g][m].y);
                        __stcg(mine + (k + 2) * 32, acc2[g][m].x);
                        __stcg(mine + (k + 3) * 32, acc2[g][m].y);
                    }
                __threadfence();
                __syncwarp();
                const int parent = idx_l / kSplitFan;
                const int c_beg = parent * kSplitFan, c_end = min(n_l, c_beg + kSplitFan);
                int done = 0;
                if (lane == 0) done = atomicAdd(p.split_cnt + cnt0 + parent, 1);
                done = __shfl_sync(kFull, done, 0);
                if (done != c_end - c_beg - 1) { last = false; break; }
                __threadfence();
#pragma unroll
                for (int g = 0; g < TM; ++g)
#pragma unroll
                    for (int m = 0; m < TN; ++m) {
                        acc1[g][m] = make_float2(0.f, 0.f);
                        acc2[g][m] = make_float2(0.f, 0.f);
                    }
#pragma unroll 1
                for (int c = c_beg; c < c_end; ++c) {
                    const float *ps = p.split_partial + static_cast<size_t>(slot0 + c) * PW + lane;
#pragma unroll
                    for (int g = 0; g < TM; ++g)
#pragma unroll
                        for (int m = 0; m < TN; ++m) {
                            const int k = (g * TN + m) * 4;
                            acc1[g][m].x += __ldcg(ps + (k + 0) * 32);
                            acc1[g][m].y += __ldcg(ps + (k + 1) * 32);
                            acc2[g][m].x += __ldcg(ps + (k + 2) * 32);
                            acc2[g][m].y += __ldcg(ps + (k + 3) * 32);
                        }
                }
                slot0 += n_l;
                n_l = (n_l + kSplitFan - 1) / kSplitFan;
                cnt0 += n_l;
                idx_l = parent;
            }
            if (!last) {
                // another warp finishes the row: no epilogue; the next pixel's first events are staged here
                if (idx < n_items && lane < it_next.n)
                    stage_event(ev_s + evb * kEC + lane, p.csr_ev + it_next.row_begin + lane);
                __syncwarp();
                continue;
            }
            out_pix = sr->pix;
            out_arow = sr->arow;
        }

        // ---- epilogue: powers, optional spectrum store, spectral flatness -------------------
        float preg[NBL];
#pragma unroll
        for (int g = 0; g < TM; ++g)
#pragma unroll
            for (int m = 0; m < TN; ++m) {
                const float s1 = acc1[g][m].x, s4 = acc1[g][m].y, s3 = acc2[g][m].x, s2 = acc2[g][m].y;
                const float rp = s1 - s2, ip = s4 + s3;       // bin centre + (m + 1/2) 32 df
                const float rm = s1 + s2, im = s3 - s4;       // bin centre - (m + 1/2) 32 df
                preg[g * 2 * TN + TN + m] = rp * rp + ip * ip;
                preg[g * 2 * TN + TN - 1 - m] = rm * rm + im * im;
            }
        const bool has_row = out_arow < p.max_active;
        if (store_power && has_row) {
            float *dst = p.power + static_cast<size_t>(out_arow) * sp.n_freq + lane;
#pragma unroll
            for (int i = 0; i < NBL; ++i)
                if (full_grid || i * 32 + lane < sp.n_freq) __stcs(dst + i * 32, preg[i]);
        }
        float slog = 0.f, ssum = 0.f;
        if (full_grid) {
            // every bin is in range; only the first k_lo bins (register 0) are left out.  Bins are
            // taken in pairs, log2(a b) = log2 a + log2 b (one SFU op per two bins; a b stays a
            // normal number: sf_eps^2 >= 1e-36 is checked, P <= n^2 < 2^62), four partial sums
            const bool in0 = lane >= sp.k_lo;
            float sl[4] = {0.f, 0.f, 0.f, 0.f}, ss[4] = {0.f, 0.f, 0.f, 0.f};
            if (sp.sf_eps >= 1e-18f) {
#pragma unroll
                for (int i = 0; i < NBL; i += 2) {
                    float a = fmaxf(preg[i], sp.sf_eps);
                    const float b = fmaxf(preg[i + 1], sp.sf_eps);
                    float sa = a;
                    if (i == 0) { sa = in0 ? a : 0.f; a = in0 ? a : 1.f; }
                    sl[(i >> 1) & 3] += __log2f(a * b);
                    ss[(i >> 1) & 3] += sa + b;
                }
            } else {
#pragma unroll
                for (int i = 0; i < NBL; ++i) {
                    const float pt = fmaxf(preg[i], sp.sf_eps);
                    const bool in = (i > 0) || in0;
                    sl[i & 3] += in ? __log2f(pt) : 0.f;
                    ss[i & 3] += in ? pt : 0.f;
                }
            }
            slog = (sl[0] + sl[1]) + (sl[2] + sl[3]);
            ssum = (ss[0] + ss[1]) + (ss[2] + ss[3]);
        } else {
#pragma unroll
            for (int i = 0; i < NBL; ++i) {
                const int j = i * 32 + lane;
                if (j >= sp.k_lo && j < sp.n_freq) {
                    const float pt = fmaxf(preg[i], sp.sf_eps);
                    slog += __log2f(pt);
                    ssum += pt;
                }
            }
        }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            slog += __shfl_xor_sync(kFull, slog, o);
            ssum += __shfl_xor_sync(kFull, ssum, o);
        }
        if (idx < n_items && lane < it_next.n)
            stage_event(ev_s + evb * kEC + lane, p.csr_ev + it_next.row_begin + lane);
        const float inv_nb = 1.f / static_cast<float>(sp.n_freq - sp.k_lo);
        const float mean_p = ssum * inv_nb;
        const float sfv = exp2f(slog * inv_nb) / mean_p;         // eq. 7
        const bool sf_ok = sfv <= sp.tau_sf;                     // discard if SF > tau_sf (L107)

        float score = 0.f;
        int f0 = -1;
        bool deferred = false;
        if (sp.score_all || sf_ok) {
            // queue the spectrum for k_comb_deferred; if the queue is full, score it here
            int slot = 0;
            if (lane == 0) slot = atomicAdd(p.spill_count, 1);
            slot = __shfl_sync(kFull, slot, 0);
            if (slot < p.spill_cap) {
                deferred = true;
                float *dst = p.spill + static_cast<size_t>(slot) * L::NB + lane;
#pragma unroll
                for (int i = 0; i < NBL; ++i) dst[i * 32] = preg[i];
                if (lane == 0) {
                    SpillRec r;
                    r.pix = out_pix; r.arow = has_row ? out_arow : -1; r.mean_p = mean_p; r._pad = 0;
                    p.spill_rec[slot] = r;
                }
            } else if (L::INPLACE) {
                // the queue is full: score here.  comb_score() wants the lane's bins contiguous
                // (NBL lane + i); they are strided (32 i + lane) in the accumulators: transpose through
                // the scratch (bin k at k + k / NBL, conflict-free both ways)
                float *T = reinterpret_cast<float *>(scr);
                __syncwarp();
#pragma unroll
                for (int i = 0; i < NBL; ++i) {
                    const int k = i * 32 + lane;
                    T[k + k / NBL] = preg[i];
                }
                __syncwarp();
                float *dbg = (p.comb_debug != nullptr && has_row)
                                 ? p.comb_debug + static_cast<size_t>(out_arow) * sp.n_f0 * 3 : nullptr;
                const float2 r = comb_score_from_smem<NBL, L::INPLACE ? BS : 256>(scr, sp, mean_p, lane, dbg);
                score = r.x;
                f0 = __float_as_int(r.y);
                if (lane == 0) atomicAdd(p.n_scored, 1);
            }
        }
        if (lane == 0) {
            p.sf[out_pix] = sfv;
            if (!deferred) {
                p.score[out_pix] = score;
                p.f0_idx[out_pix] = f0;
                p.mask[out_pix] = (sf_ok && f0 >= 0 && score >= sp.tau_comb) ? 1 : 0;   // eq. 11
            }
        }
        __syncwarp();
    }
}


// ----------------------------------------------------------------------------------------
// Deferred comb scoring: one warp per queued pixel, at an occupancy the 168-register NDFT
// kernel cannot offer (the code is latency-bound: dependent shared-memory and shuffle chains).
// Same comb_score() as the in-place path, on the same float spectrum, so results are identical
// whichever path scores a pixel.
// ----------------------------------------------------------------------------------------
constexpr int kScoreWarps = 4;

template <int NBL, int BS>
__global__ void __launch_bounds__(kScoreWarps * 32, 4) k_comb_deferred(NdftParams p)
{
    using S = CombSmem<NBL, BS>;
    constexpr int NB = NBL * 32;
    extern __shared__ __align__(16) uint32_t smem_raw[];
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    const ScoreParams &sp = p.sp;
    uint32_t *scr = smem_raw + wid * S::words(sp.cpad);
    const int n_rows = min(*p.spill_count, p.spill_cap);
    // rows are handed out one at a time (their cost varies with the band search): spill_count[1]
    // is the consumer cursor, zeroed with the producer count by the ingest stage
    while (true) {
        int row = 0;
        if (lane == 0) row = atomicAdd(p.spill_count + 1, 1);
        row = __shfl_sync(kFull, row, 0);
        if (row >= n_rows) break;
        const SpillRec r = p.spill_rec[row];
        // the lane's NBL consecutive bins: NBL / 4 128-bit loads (the row is read exactly once)
        const float4 *src = reinterpret_cast<const float4 *>(p.spill + static_cast<size_t>(row) * NB + NBL * lane);
        float preg[NBL];
#pragma unroll
        for (int i = 0; i < NBL / 4; ++i) {
            const float4 v = __ldcs(src + i);
            preg[4 * i] = v.x; preg[4 * i + 1] = v.y; preg[4 * i + 2] = v.z; preg[4 * i + 3] = v.w;
        }
        float score;
        int f0;
        float *dbg = (p.comb_debug != nullptr && r.arow >= 0)
                         ? p.comb_debug + static_cast<size_t>(r.arow) * sp.n_f0 * 3 : nullptr;
        comb_score<NBL, BS>(preg, scr, sp, r.mean_p, lane, score, f0, dbg);
        if (lane == 0) {
            // the pixel is in the queue because SF <= tau_sf or score_all; the mask needs both
            const bool sf_ok = p.sf[r.pix] <= sp.tau_sf;
            p.score[r.pix] = score;
            p.f0_idx[r.pix] = f0;
            p.mask[r.pix] = (sf_ok && f0 >= 0 && score >= sp.tau_comb) ? 1 : 0;       // eq. 11
        }
        __syncwarp();
    }
    if (blockIdx.x == 0 && threadIdx.x == 0) atomicAdd(p.n_scored, n_rows);
}

template <int TM, int TN, int BS, bool FULL, bool FB>
int launch_one(const NdftParams &p, const NdftParams *seg_pass, int grid_ndft, int grid_seg, int grid_score, cudaStream_t st,
               cudaEvent_t between)
{
    using L = Layout<TM, TN, BS, FB>;
    const size_t score_smem = static_cast<size_t>(CombSmem<L::NBL, BS>::words(p.sp.cpad)) * 4 * kScoreWarps;
    int launches = 2;
    k_ndft_score<TM, TN, BS, FULL, FB><<<grid_ndft, warps_of(L::NBL) * 32, L::smem_bytes(p.sp.cpad), st>>>(p);
    if (!FB && L::NBL == 64 && seg_pass) {
        // the lean variant's work list holds whole rows only; the segments of split rows go through the
        // full variant (it leaves at once when there are none)
        using LF = Layout<TM, TN, BS, true>;
        k_ndft_score<TM, TN, BS, FULL, true><<<grid_seg, warps_of(L::NBL) * 32, LF::smem_bytes(p.sp.cpad), st>>>(*seg_pass);
        ++launches;
    }
    if (between) cudaEventRecord(between, st);
    k_comb_deferred<L::NBL, BS><<<grid_score, kScoreWarps * 32, score_smem, st>>>(p);
    return launches;
}

template <int TM, int TN, int BS, bool FULL, bool FB>
cudaError_t configure_one(int cpad, int *blocks_per_sm, int *score_blocks_per_sm)
{
    using L = Layout<TM, TN, BS, FB>;
    const size_t smem = L::smem_bytes(cpad);
    const size_t score_smem = static_cast<size_t>(CombSmem<L::NBL, BS>::words(cpad)) * 4 * kScoreWarps;
    cudaError_t e = cudaFuncSetAttribute(k_ndft_score<TM, TN, BS, FULL, FB>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                         static_cast<int>(smem));
    if (e != cudaSuccess) return e;
    e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(blocks_per_sm, k_ndft_score<TM, TN, BS, FULL, FB>, warps_of(L::NBL) * 32, smem);
    if (e != cudaSuccess) return e;
    if (*blocks_per_sm < 1) return cudaErrorLaunchOutOfResources;
    e = cudaFuncSetAttribute(k_comb_deferred<L::NBL, BS>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                             static_cast<int>(score_smem));
    if (e != cudaSuccess) return e;
    e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(score_blocks_per_sm, k_comb_deferred<L::NBL, BS>,
                                                      kScoreWarps * 32, score_smem);
    if (e != cudaSuccess) return e;
    if (*score_blocks_per_sm < 1) return cudaErrorLaunchOutOfResources;
    return cudaSuccess;
}

}  // namespace

int ndft_bins_per_lane(int n_freq)
{
    if (n_freq <= 256) return 8;
    if (n_freq <= 512) return 16;
    if (n_freq <= 1024) return 32;
    return 64;
}

int ndft_padded_bins(int n_freq) { return ndft_bins_per_lane(n_freq) * 32; }

int ndft_tn(int n_freq)
{
    const int nbl = ndft_bins_per_lane(n_freq);
    return nbl == 64 ? 16 : nbl == 32 ? 8 : nbl / 2;      // 32 bins per lane: two centres x 8 offset pairs
}

int ndft_band_size(int n_freq, int r0, int r1)
{
    // sort capacity: the rank band [r0, r1] plus room for the band-limit search to land in (16 ranks on
    // either side at least); a spectrum that fits the smallest sorter is sorted whole
    const int need = r1 - r0 + 1;
    const int nb = ndft_bins_per_lane(n_freq) * 32;
    if (nb <= 256 || need + 32 <= 256) return (need <= 256) ? 256 : 0;
    if (nb <= 512 || need + 64 <= 512) return (need <= 512) ? 512 : 0;
    if (nb <= 1024 || need + 128 <= 1024) return (need <= 1024) ? 1024 : 0;
    return 0;
}

bool ndft_scores_in_place(int n_freq, int band_size) { (void)n_freq; return band_size <= 512; }

namespace {

// one dispatch for configure and launch: f.template operator()<TM, TN, BS>()
template <typename F>
auto dispatch(int n_freq, int bs, F &&f)
{
    const int nbl = ndft_bins_per_lane(n_freq);
    if (nbl == 8) return f.template operator()<1, 4, 256>();
    if (nbl == 16) return bs == 256 ? f.template operator()<1, 8, 256>() : f.template operator()<1, 8, 512>();
    if (nbl == 32) return bs == 256 ? f.template operator()<2, 8, 256>()
                        : bs == 512 ? f.template operator()<2, 8, 512>() : f.template operator()<2, 8, 1024>();
    return bs == 256 ? f.template operator()<2, 16, 256>()
         : bs == 512 ? f.template operator()<2, 16, 512>() : f.template operator()<2, 16, 1024>();
}

struct ConfigureFn {
    int cpad; bool fb; int *b1, *bf, *b2;
    template <int TM, int TN, int BS> cudaError_t operator()() const
    {
        int x, y;
        // the full variant is always needed (as the main kernel, or for the segment pass)
        cudaError_t e = configure_one<TM, TN, BS, true, true>(cpad, bf, b2);
        if (e != cudaSuccess) return e;
        e = configure_one<TM, TN, BS, false, true>(cpad, &x, &y);
        if (e != cudaSuccess) return e;
        *bf = x < *bf ? x : *bf; *b2 = y < *b2 ? y : *b2;
        *b1 = *bf;
        if (!fb) {
            e = configure_one<TM, TN, BS, true, false>(cpad, b1, &y);
            if (e != cudaSuccess) return e;
            e = configure_one<TM, TN, BS, false, false>(cpad, &x, &y);
            if (e == cudaSuccess) *b1 = x < *b1 ? x : *b1;
        }
        return e;
    }
};

struct LaunchFn {
    const NdftParams &p; const NdftParams *seg; bool full, fb; int g1, gs, g2; cudaStream_t st; cudaEvent_t between;
    template <int TM, int TN, int BS> int operator()() const
    {
        if (fb)
            return full ? launch_one<TM, TN, BS, true, true>(p, seg, g1, gs, g2, st, between)
                        : launch_one<TM, TN, BS, false, true>(p, seg, g1, gs, g2, st, between);
        return full ? launch_one<TM, TN, BS, true, false>(p, seg, g1, gs, g2, st, between)
                    : launch_one<TM, TN, BS, false, false>(p, seg, g1, gs, g2, st, between);
    }
};

}  // namespace

cudaError_t ndft_configure(int n_freq, int band_size, int cpad, bool fallback, int *blocks_per_sm, int *full_blocks_per_sm,
                           int *score_blocks_per_sm)
{
    return dispatch(n_freq, band_size, ConfigureFn{cpad, fallback, blocks_per_sm, full_blocks_per_sm, score_blocks_per_sm});
}

int launch_ndft(const NdftParams &p, const NdftParams *seg_pass, int n_freq, int band_size, bool fallback, int grid_ndft, int grid_seg,
                int grid_score, cudaStream_t st, cudaEvent_t between)
{
    const bool full = (n_freq == ndft_bins_per_lane(n_freq) * 32) && (p.sp.k_lo <= 32);
    return dispatch(n_freq, band_size, LaunchFn{p, seg_pass, full, fallback, grid_ndft, grid_seg, grid_score, st, between});
}

}  // namespace ddhf
