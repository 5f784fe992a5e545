// comb.cuh -- a6: median-normalised harmonic comb score of one pixel, one warp per pixel.
//
//   N(w)     = mean over the valid harmonics m of  max_{|k - k_m| <= d} P_k         (eq. 8)
//   H(w)     = union of the harmonic windows, median taken over its complement       (eq. 9)
//   SNR_M(w) = N(w) / median                                                          (eq. 10)
//   score    = max_w SNR_M(w), f0 = first argmax                                      (eq. 11)
//
// Readings R7-R11, R16 of DESIGN.md (window centres, validity prefix, union, lower median, floor).
//
// Design (what the 11.7 k warp instructions per pixel of the first version became):
//
// * The lane owns NBL CONSECUTIVE bins (lane l: bins NBL l .. NBL l + NBL - 1) in registers.  Every
//   stage that walks the whole spectrum (rank counting, classification, block maxima) is then plain
//   register arithmetic with a warp scan at the end, instead of one ballot per 32 bins.
// * Every candidate's complement median is an order statistic of the full spectrum inside the rank
//   band [r0, r1] fixed at create time (a candidate removes <= n_excl bins).  The band is bracketed
//   by counting passes over the registers (two pivots per pass; first pivots from the exponential
//   model of a noise spectrum, then a secant through the two measured ranks, bisection of the key
//   interval every third pass so the search always ends; a collapsed bracket = heavy ties, split by
//   bin order), compacted in bin order and sorted once (bitonic, in registers).
// * Window maxima: forward block maxima M[k] = max P[k .. k + 2^s - 1] by s doubling steps in
//   registers (one FMNMX per bin and step), two table lookups per harmonic.
// * Per candidate (one per lane): the excluded bins below / inside the band are counted by popcounts
//   of <= 32-bin pieces of the two classification bitmaps (tables built at create time).  That
//   gives the candidate's median up to the excluded bins that fall inside the band: an interval
//   [s[j], s[j + n_in]] of the sorted band, hence an interval for SNR_M.  Only candidates whose upper
//   bound reaches the best lower bound are evaluated exactly (usually a handful): their in-band
//   excluded values are gathered and the rank equation a = j + #{v <= s[a]} is iterated to its
//   least fixed point, which is the lower median of the complement as a multiset.  Pruned candidates
//   are strictly below the maximum, so score and argmax are the same as evaluating all of them.
#pragma once

#include "ddhf_internal.cuh"

namespace ddhf {
namespace {

constexpr unsigned kFullWarp = 0xffffffffu;
constexpr uint32_t kInfKey = 0x7f800000u;      // +inf: above every spectrum value; marks bins outside [k_lo, n_freq)
constexpr int kCoopMax = 6;                    // contenders up to which the warp evaluates them one at a time
constexpr int kVCap = 32;                      // in-band excluded values gathered per candidate (more: slow walk)

template <int N> struct Log2 { static constexpr int v = 1 + Log2<N / 2>::v; };
template <> struct Log2<1> { static constexpr int v = 0; };

// Per-warp shared-memory layout of the scoring scratch, in 32-bit words.
template <int NBL, int BS>
struct CombSmem {
    static constexpr int NB = NBL * 32;
    static constexpr int NW = NBL;                          // 32-bit words of a per-bin bitmap
    static constexpr int E = BS / 32;                       // sorted values per lane
    static constexpr int M_WORDS = NB + 32;                 // block maxima, bin k at k + k / NBL
    static constexpr int BAL_WORDS = 4 * NW;                // uint4 {below[w], below[w+1], inband[w], inband[w+1]}
    static constexpr int INBC_WORDS = NW;                   // in-band bins before word w
    static constexpr int BAND_WORDS = BS;                   // band values in bin order
    static constexpr int SORT_WORDS = BS + 32;              // band values ascending, index a at a + a / E
    static constexpr int VLIST_WORDS = kVCap * 32;          // [kVCap][lane]; aliases the block maxima (dead by then)
    static_assert(VLIST_WORDS <= M_WORDS || NBL < 32, "gather list must fit in the block-maxima region");
    static constexpr int M_REGION = M_WORDS > VLIST_WORDS ? M_WORDS : VLIST_WORDS;
    static constexpr int FIXED_WORDS = M_REGION + BAL_WORDS + INBC_WORDS + BAND_WORDS + SORT_WORDS;
    // + per candidate: (N, j | n_in << 16) and a contender list, sized at run time (cpad)
    __host__ __device__ static constexpr int words(int cpad) { return ((FIXED_WORDS + 3 * cpad + 3) / 4) * 4; }
};

// Compare-exchange steps j = J, J/2, .., 1 on the lane's E registers; asc: this lane sorts ascending.
template <int E, int J>
__device__ __forceinline__ void bitonic_reg_steps(float (&x)[E], bool asc)
{
#pragma unroll
    for (int j = J; j > 0; j >>= 1) {
#pragma unroll
        for (int r = 0; r < E; ++r) {
            if ((r & j) == 0) {
                const float a = x[r], b = x[r | j];
                x[r] = asc ? fminf(a, b) : fmaxf(a, b);
                x[r | j] = asc ? fmaxf(a, b) : fminf(a, b);
            }
        }
    }
}

// Bitonic sort of 32 E values, element (lane, r) <-> position lane E + r.  The merges that cross lanes
// are rolled loops (the code of a fully unrolled network does not fit the instruction cache next to the
// rest of the scoring code); their register steps are the same code for every merge size.
template <int E>
__device__ __forceinline__ void bitonic_sort_regs(float (&x)[E], int lane)
{
    // merge sizes 2 .. E: inside the registers, direction from the register index (and the lane for k = E)
#pragma unroll
    for (int k = 2; k <= E; k <<= 1) {
#pragma unroll
        for (int j = k >> 1; j > 0; j >>= 1) {
#pragma unroll
            for (int r = 0; r < E; ++r) {
                if ((r & j) == 0) {
                    const bool asc = (k < E) ? ((r & k) == 0) : ((lane & 1) == 0);
                    const float a = x[r], b = x[r | j];
                    x[r] = asc ? fminf(a, b) : fmaxf(a, b);
                    x[r | j] = asc ? fmaxf(a, b) : fminf(a, b);
                }
            }
        }
    }
    // merge sizes 2 E .. 32 E: kl = lanes per merged run
#pragma unroll 1
    for (int kl = 2; kl <= 32; kl <<= 1) {
        const bool asc = (kl == 32) ? true : ((lane & kl) == 0);
#pragma unroll 1
        for (int lm = kl >> 1; lm > 0; lm >>= 1) {
            const bool take_min = ((lane & lm) == 0) == asc;
#pragma unroll
            for (int r = 0; r < E; ++r) {
                const float o = __shfl_xor_sync(kFullWarp, x[r], lm);
                x[r] = take_min ? fminf(x[r], o) : fmaxf(x[r], o);
            }
        }
        bitonic_reg_steps<E, E / 2>(x, asc);
    }
}

__device__ __forceinline__ int warp_excl_scan(int v, int lane, int &total)
{
    int inc = v;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const int t = __shfl_up_sync(kFullWarp, inc, o);
        if (lane >= o) inc += t;
    }
    total = __shfl_sync(kFullWarp, inc, 31);
    return inc - v;
}

// One side of the band-limit search: the wanted key has  lo_ok <= #{key < it} <= hi_ok.
struct BandSide {
    uint32_t a, b;       // bracket: #{key < a} < lo_ok (too low), #{key < b} > hi_ok (too high)
    int ca, cb;
    uint32_t key;        // result
    int cnt, ties;       // #{key < result}; tied bins (== result) that are taken as well, in bin order
    bool done;
};

__device__ __forceinline__ void band_side_update(BandSide &s, uint32_t p, int c, int lo_ok, int hi_ok)
{
    if (s.done) return;
    if (c < lo_ok) {
        if (p > s.a) { s.a = p; s.ca = c; }
    } else if (c > hi_ok) {
        if (p < s.b) { s.b = p; s.cb = c; }
    } else {
        s.done = true; s.key = p; s.cnt = c; s.ties = 0;
    }
}

// Next trial key of one side.  (x1, c1), (x2, c2): two measured (value, rank) points (the two pivots of the
// last pass if they differ, else the bracket ends); `bisect`: plain bisection of the key interval.
__device__ __forceinline__ uint32_t band_next_pivot(const BandSide &s, float target, uint32_t p1, int c1,
                                                    uint32_t p2, int c2, bool bisect)
{
    uint32_t p = s.a + ((s.b - s.a) >> 1);
    if (!bisect) {
        if (p1 == p2) { p1 = s.a; c1 = s.ca; p2 = s.b; c2 = s.cb; }
        if (p2 < kInfKey && p1 < kInfKey && p1 != p2 && c1 != c2) {
            const float v1 = __uint_as_float(p1), v2 = __uint_as_float(p2);
            const float f1 = static_cast<float>(c1), f2 = static_cast<float>(c2);
            const bool use2 = fabsf(f2 - target) < fabsf(f1 - target);
            const float v = (use2 ? v2 : v1) + (target - (use2 ? f2 : f1)) * (v2 - v1) / (f2 - f1);
            if (v > 0.f && v < 3.0e38f) p = __float_as_uint(v);
        }
    }
    return min(max(p, s.a + 1u), s.b - 1u);
}

// ---------------------------------------------------------------------------------------------------
// p[i]: power of bin NBL * lane + i (destroyed).  sm: CombSmem<NBL, BS>::words(cp.cpad) words of this
// warp's shared memory.  Returns (score, f0 index) on every lane.
// ---------------------------------------------------------------------------------------------------
template <int NBL, int BS>
__device__ __forceinline__ void comb_score(float (&p)[NBL], uint32_t *sm, const CombParams &cp, float mean_p,
                                           int lane, float &score_out, int &f0_out, float *dbg)
{
    using S = CombSmem<NBL, BS>;
    constexpr int NB = S::NB;
    constexpr int E = S::E;
    constexpr int LOG_E = Log2<E>::v;
    constexpr int WL = (NBL >= 32) ? NBL / 32 : 1;          // bitmap words (or the part of one) per lane
    float *Ms = reinterpret_cast<float *>(sm);
    uint4 *bal = reinterpret_cast<uint4 *>(sm + S::M_REGION);
    uint32_t *inbc = sm + S::M_REGION + S::BAL_WORDS;
    float *bandv = reinterpret_cast<float *>(inbc + S::INBC_WORDS);
    float *sortv = bandv + S::BAND_WORDS;
    float *vlist = Ms;                                                      // after the numerators are done
    uint2 *cand_s = reinterpret_cast<uint2 *>(sortv + S::SORT_WORDS);       // 8-byte aligned: FIXED_WORDS is even
    unsigned short *clist = reinterpret_cast<unsigned short *>(cand_s + cp.cpad);

    const int nb = cp.n_freq - cp.k_lo;
    const int r0 = cp.r0, r1 = cp.r1;

    // ---- 0: bins outside [k_lo, n_freq) never take part: +inf sorts above everything ---------------
    if (cp.k_lo <= 4 && cp.n_freq == NB) {
        if (lane == 0) {
#pragma unroll
            for (int i = 0; i < 4; ++i)
                if (i < cp.k_lo) p[i] = __uint_as_float(kInfKey);
        }
    } else {
#pragma unroll
        for (int i = 0; i < NBL; ++i) {
            const int j = NBL * lane + i;
            if (j < cp.k_lo || j >= cp.n_freq) p[i] = __uint_as_float(kInfKey);
        }
    }

    // ---- A: band limits by counting passes over the registers ----------------------------------------
    BandSide L, U;
    L.a = 0u; L.ca = 0; L.b = kInfKey; L.cb = nb; L.key = 0u; L.cnt = 0; L.ties = 0; L.done = true;
    U = L; U.key = kInfKey; U.cnt = nb;
    if (nb > BS) {
        const int slack = (BS - (r1 - r0 + 1)) >> 1;
        const int L0 = r0 - slack, L1 = r0, U0 = r1 + 1, U1 = r1 + 1 + slack;
        L.done = (L0 <= 0);                     // key 0 (nothing below) already fits
        U.done = (nb <= U1);                    // +inf (everything below) already fits
        const float nbf = static_cast<float>(nb);
        const float tgL = r0 - 0.5f * slack, tgU = r1 + 1 + 0.5f * slack;
        // first pivots: quantiles of an exponential spectrum with the measured mean
        uint32_t pvL = __float_as_uint(-mean_p * __logf(fmaxf(1.f - tgL / nbf, 1e-3f)));
        uint32_t pvU = __float_as_uint(-mean_p * __logf(fmaxf(1.f - tgU / nbf, 1e-3f)));
        pvL = min(max(pvL, 1u), kInfKey - 1u);
        pvU = min(max(pvU, pvL + 1u), kInfKey - 1u);
#pragma unroll 1
        for (int it = 0; !(L.done && U.done); ++it) {
            if (L.done) pvL = pvU;
            if (U.done) pvU = pvL;
            uint32_t gl = 0, gu = 0;
#pragma unroll
            for (int i = 0; i < NBL; ++i) {
                // count += (key >= pivot): sub.cc leaves CF = 1 when there is no borrow (checked on sm_100a),
                // addc adds it: 2 instructions per comparison
                uint32_t t;
                asm("{sub.cc.u32 %1, %2, %3;\n\taddc.u32 %0, %0, 0;}" : "+r"(gl), "=r"(t) : "r"(__float_as_uint(p[i])), "r"(pvL));
                asm("{sub.cc.u32 %1, %2, %3;\n\taddc.u32 %0, %0, 0;}" : "+r"(gu), "=r"(t) : "r"(__float_as_uint(p[i])), "r"(pvU));
            }
            const uint32_t cl = NBL - gl, cu = NBL - gu;          // bins outside [k_lo, n_freq) are +inf: never below
            const int cl_w = static_cast<int>(__reduce_add_sync(kFullWarp, cl));
            const int cu_w = static_cast<int>(__reduce_add_sync(kFullWarp, cu));
            band_side_update(L, pvL, cl_w, L0, L1);
            band_side_update(L, pvU, cu_w, L0, L1);
            band_side_update(U, pvL, cl_w, U0, U1);
            band_side_update(U, pvU, cu_w, U0, U1);
            // a bracket of two adjacent keys: the lower one is tied across the whole accepted range;
            // take exactly as many of the tied bins (in bin order) as the wanted rank asks for
            if (!L.done && L.b - L.a <= 1u) { L.done = true; L.key = L.a; L.cnt = L.ca; L.ties = r0 - L.ca; }
            if (!U.done && U.b - U.a <= 1u) { U.done = true; U.key = U.a; U.cnt = U.ca; U.ties = (r1 + 1) - U.ca; }
            const bool bisect = (it % 3) == 2;
            const uint32_t nL = L.done ? 0u : band_next_pivot(L, tgL, pvL, cl_w, pvU, cu_w, bisect);
            const uint32_t nU = U.done ? 0u : band_next_pivot(U, tgU, pvL, cl_w, pvU, cu_w, bisect);
            pvL = nL; pvU = nU;
        }
    }
    const uint32_t Lkey = L.key, Ukey = U.key;
    const int cnt_below = L.cnt + L.ties;                 // bins whose rank is below the band
    const int nband = min((U.cnt + U.ties) - cnt_below, BS);

    // a copy of the lane's bins in shared memory (the block maxima overwrite it later): registers cannot be
    // indexed by a run-time position, the rolled loops below (ties, compaction) read the copy
    float *mine = Ms + lane * (NBL + 1);
#pragma unroll
    for (int i = 0; i < NBL; ++i) mine[i] = p[i];
    __syncwarp();

    // ---- B: classification bitmaps (below the band / inside it), bit b of the lane's word <-> bin ----
    constexpr int CNT = (NBL >= 32) ? 32 : NBL;             // bins per bitmap word of the lane
    uint32_t mb[WL], mi[WL];
    if ((L.ties | U.ties) == 0) {
#pragma unroll
        for (int w = 0; w < WL; ++w) {
            uint32_t below = 0u, lt_u = 0u;
#pragma unroll
            for (int b = CNT - 1; b >= 0; --b) {
                const uint32_t key = __float_as_uint(p[w * 32 + b]);
                // keys and limits are < 2^31: the sign bit of the difference is (key < limit)
                below = __funnelshift_l(key - Lkey, below, 1);
                lt_u = __funnelshift_l(key - Ukey, lt_u, 1);
            }
            mb[w] = below;
            mi[w] = lt_u & ~below;
        }
    } else {
        // heavy ties at a band limit (rare): the bins equal to the limit are taken in bin order
        int eqL = 0, eqU = 0;
#pragma unroll 1
        for (int i = 0; i < NBL; ++i) {
            const uint32_t key = __float_as_uint(mine[i]);
            eqL += (key == Lkey) ? 1 : 0;
            eqU += (key == Ukey) ? 1 : 0;
        }
        int tot;
        int runL = warp_excl_scan(eqL, lane, tot);
        int runU = warp_excl_scan(eqU, lane, tot);
#pragma unroll
        for (int w = 0; w < WL; ++w) {
            uint32_t below = 0u, inb = 0u;
#pragma unroll 1
            for (int b = 0; b < CNT; ++b) {
                const uint32_t key = __float_as_uint(mine[w * 32 + b]);
                bool bl = key < Lkey, le = key < Ukey;
                if (key == Lkey) { bl = bl || (runL < L.ties); ++runL; }
                if (key == Ukey) { le = le || (runU < U.ties); ++runU; }
                below |= (bl ? 1u : 0u) << b;
                inb |= ((le && !bl) ? 1u : 0u) << b;
            }
            mb[w] = below;
            mi[w] = inb;
        }
    }

    // ---- C: in-band values compacted in bin order; bitmaps and prefix counts to shared memory ----------
    {
        int n_in = 0;
#pragma unroll
        for (int w = 0; w < WL; ++w) n_in += __popc(mi[w]);
        int total;
        const int ex = warp_excl_scan(n_in, lane, total);
        // the in-band bins are few (a dozen per lane): walk the set bits
        int pos = ex;
#pragma unroll
        for (int w = 0; w < WL; ++w) {
            uint32_t m = mi[w];
            while (m) {
                const int b = __ffs(m) - 1;
                m &= m - 1u;
                if (pos < BS) bandv[pos] = mine[w * 32 + b];
                ++pos;
            }
        }
        __syncwarp();
        if constexpr (NBL >= 32) {
            const uint32_t nb_b = __shfl_down_sync(kFullWarp, mb[0], 1), nb_i = __shfl_down_sync(kFullWarp, mi[0], 1);
            const uint32_t xb = (lane == 31) ? 0u : nb_b, xi = (lane == 31) ? 0u : nb_i;
            if (WL == 2) {
                bal[2 * lane] = make_uint4(mb[0], mb[WL - 1], mi[0], mi[WL - 1]);
                bal[2 * lane + 1] = make_uint4(mb[WL - 1], xb, mi[WL - 1], xi);
                inbc[2 * lane] = ex;
                inbc[2 * lane + 1] = ex + __popc(mi[0]);
            } else {
                bal[lane] = make_uint4(mb[0], xb, mi[0], xi);
                inbc[lane] = ex;
            }
        } else {
            // several lanes share one bitmap word
            constexpr int LPW = 32 / NBL;
            uint32_t fb = mb[0] << (NBL * (lane % LPW)), fi = mi[0] << (NBL * (lane % LPW));
#pragma unroll
            for (int o = 1; o < LPW; o <<= 1) {
                fb |= __shfl_xor_sync(kFullWarp, fb, o);
                fi |= __shfl_xor_sync(kFullWarp, fi, o);
            }
            const uint32_t nb_b = __shfl_down_sync(kFullWarp, fb, LPW), nb_i = __shfl_down_sync(kFullWarp, fi, LPW);
            const bool last = lane + LPW >= 32;
            if ((lane % LPW) == 0) {
                bal[lane / LPW] = make_uint4(fb, last ? 0u : nb_b, fi, last ? 0u : nb_i);
                inbc[lane / LPW] = ex;
            }
        }
    }

    // ---- W: forward block maxima M[k] = max P[k .. k + 2^s - 1] in registers (destroys p) --------------
#pragma unroll
    for (int t = 0; t < 5; ++t) {
        if (t < cp.s_lvl) {
            // values of the following lanes that this step needs, fetched before anything is updated
            float nbv[(1 << 4) < NBL ? (1 << 4) : NBL];
            const int sh = 1 << t;
            constexpr int MAXN = (1 << 4) < NBL ? (1 << 4) : NBL;
#pragma unroll
            for (int r = 0; r < MAXN; ++r) {
                // register r is needed from lane + (sh_c + i) / NBL for the i with (i + sh_c) % NBL == r
                if (r < sh || sh >= NBL) {
                    const int i = ((r - sh) % NBL + NBL) % NBL;
                    const int lo = (i + sh) / NBL;
                    nbv[r] = __shfl_down_sync(kFullWarp, p[r], lo > 0 ? lo : 1);
                }
            }
#pragma unroll
            for (int i = 0; i < NBL; ++i) {
                const int src = i + sh;
                if (src < NBL) p[i] = fmaxf(p[i], p[src]);        // p[src] not yet updated (ascending i)
                else p[i] = fmaxf(p[i], nbv[src % NBL]);
            }
        }
    }
    __syncwarp();
#pragma unroll
    for (int i = 0; i < NBL; ++i) mine[i] = p[i];
    __syncwarp();

    // ---- D: sort the band (ascending) in registers ---------------------------------------------------------
    {
        float x[E];
#pragma unroll
        for (int r = 0; r < E; ++r) {
            const int idx = r * 32 + lane;
            x[r] = (idx < nband) ? bandv[idx] : __uint_as_float(kInfKey);
        }
        bitonic_sort_regs<E>(x, lane);
#pragma unroll
        for (int r = 0; r < E; ++r) sortv[lane * (E + 1) + r] = x[r];
    }
    __syncwarp();
    auto sorted_at = [&](int a) { return sortv[a + (a >> LOG_E)]; };
    const int last = max(nband - 1, 0);
    const int cpad = cp.cpad;

    // ---- F1: every candidate: numerator, excluded bins below / inside the band, SNR interval -------------
    float lb_max = 0.f;
#pragma unroll 1
    for (int c0 = 0; c0 < cp.n_f0; c0 += 32) {
        const int c = c0 + lane;
        const uint4 meta = cp.meta[c];
        const int mv = static_cast<int>(meta.x & 0xffffu);
        // table entries first (independent loads in flight), then the shared-memory lookups
        float num = 0.f;
#pragma unroll 1
        const uint32_t *nt = cp.num_tab + c;                  // rows padded to a multiple of 8 (zero entries)
        for (int m0 = 0; m0 < cp.n_harm; m0 += 8, nt += 8 * cpad) {
            uint32_t e[8];
#pragma unroll
            for (int u = 0; u < 8; ++u) e[u] = nt[u * cpad];
            float w[8];
#pragma unroll
            for (int u = 0; u < 8; ++u) w[u] = fmaxf(Ms[e[u] & 0xffffu], Ms[e[u] >> 16]);
#pragma unroll
            for (int u = 0; u < 8; ++u) num += (m0 + u < mv) ? w[u] : 0.f;
        }
        num *= __uint_as_float(meta.z);                       // 1 / M_valid
        int e_low = 0, n_in = 0;
#pragma unroll 1
        const uint2 *pt = cp.piece_tab + c;                   // rows padded to a multiple of 8 (mask 0)
        for (int q0 = 0; q0 < cp.max_pieces; q0 += 8, pt += 8 * cpad) {
            uint2 pc[8];                                      // {mask of the piece's length, first bin}
#pragma unroll
            for (int u = 0; u < 8; ++u) pc[u] = pt[u * cpad];
            uint4 a[8];
#pragma unroll
            for (int u = 0; u < 8; ++u) a[u] = bal[pc[u].y >> 5];
#pragma unroll
            for (int u = 0; u < 8; ++u) {
                e_low += __popc(__funnelshift_r(a[u].x, a[u].y, pc[u].y) & pc[u].x);
                n_in += __popc(__funnelshift_r(a[u].z, a[u].w, pc[u].y) & pc[u].x);
            }
        }
        int j = static_cast<int>(meta.y & 0xffffu) - (cnt_below - e_low);   // rank in the band if nothing of it were excluded
        j = min(max(j, 0), last);
        const float s_hi = sorted_at(min(j + n_in, last));
        if (mv > 0) lb_max = fmaxf(lb_max, __fdividef(num, fmaxf(s_hi, cp.sf_eps)));
        cand_s[c] = make_uint2(__float_as_uint(num), static_cast<uint32_t>(j) | (static_cast<uint32_t>(n_in) << 16));
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) lb_max = fmaxf(lb_max, __shfl_xor_sync(kFullWarp, lb_max, o));
    __syncwarp();

    // ---- F2: contenders: upper bound of SNR_M reaches the best lower bound (all of them when debugging) ----
    int n_cont = 0;
    {
        const float thr = lb_max * (1.f - 8e-6f);
#pragma unroll 1
        for (int c0 = 0; c0 < cp.n_f0; c0 += 32) {
            const int c = c0 + lane;
            const uint4 meta = cp.meta[c];
            const uint2 cs = cand_s[c];
            const float ub = __fdividef(__uint_as_float(cs.x), fmaxf(sorted_at(cs.y & 0xffffu), cp.sf_eps));
            const bool cont = (meta.x & 0xffffu) != 0u && (dbg != nullptr || ub * (1.f + 8e-6f) >= thr);
            const uint32_t bm = __ballot_sync(kFullWarp, cont);
            if (cont) clist[n_cont + __popc(bm & ((1u << lane) - 1u))] = static_cast<unsigned short>(c);
            n_cont += __popc(bm);
        }
    }
    __syncwarp();

    // ---- F3: exact complement median of the contenders -----------------------------------------------------
    float best = 0.f;
    int best_c = 0x7fffffff;
    if (n_cont <= kCoopMax && dbg == nullptr) {
        // a few contenders (the usual case): the whole warp works on one at a time, one piece per lane
        float *glist = vlist;                                  // the candidate's in-band excluded values, <= BS
#pragma unroll 1
        for (int ci = 0; ci < n_cont; ++ci) {
            const int c = clist[ci];
            const uint2 cs = cand_s[c];
            const float num = __uint_as_float(cs.x);
            const int j = static_cast<int>(cs.y & 0xffffu), n_in = static_cast<int>(cs.y >> 16);
            int a = j;
            if (n_in > 0) {
                const int np = static_cast<int>(cp.meta[c].x >> 16);
                int base = 0;
#pragma unroll 1
                for (int q0 = 0; q0 < np; q0 += 32) {
                    const int q = q0 + lane;
                    const uint2 pc = (q < np) ? cp.piece_tab[q * cpad + c] : make_uint2(0u, 0u);
                    const uint4 aa = bal[pc.y >> 5];
                    uint32_t inb = __funnelshift_r(aa.z, aa.w, pc.y) & pc.x;
                    int ib = inbc[pc.y >> 5] + __popc(aa.z & ((1u << (pc.y & 31u)) - 1u));
                    int tot;
                    int pos = base + warp_excl_scan(__popc(inb), lane, tot);
                    while (inb) {
                        inb &= inb - 1u;
                        glist[min(pos, BS - 1)] = bandv[min(ib, BS - 1)];
                        ++pos; ++ib;
                    }
                    base += tot;
                }
                __syncwarp();
                const int n = min(base, BS);
                // least fixed point of a = j + #{excluded in-band values <= s[a]}, from a = j
                while (true) {
                    const float x = sorted_at(min(a, last));
                    int cnt = 0;
                    for (int t0 = 0; t0 < n; t0 += 32) {
                        const float v = (t0 + lane < n) ? glist[t0 + lane] : __uint_as_float(kInfKey);
                        cnt += __popc(__ballot_sync(kFullWarp, v <= x));
                    }
                    if (j + cnt == a) break;
                    a = j + cnt;
                }
                __syncwarp();
            }
            const float med = sorted_at(min(a, last));
            const float snr = num / fmaxf(med, cp.sf_eps);
            if (best_c == 0x7fffffff || snr > best || (snr == best && c < best_c)) { best = snr; best_c = c; }
        }
    } else
#pragma unroll 1
    for (int b0 = 0; b0 < n_cont; b0 += 32) {
        const bool act = b0 + lane < n_cont;
        const int c = act ? clist[b0 + lane] : 0;
        const uint2 cs = cand_s[c];
        const float num = __uint_as_float(cs.x);
        const int j = static_cast<int>(cs.y & 0xffffu);
        const int n_in = act ? static_cast<int>(cs.y >> 16) : 0;
        const int np = act ? static_cast<int>(cp.meta[c].x >> 16) : 0;
        // gather the candidate's excluded values that lie inside the band
        int n = 0;
        if (__any_sync(kFullWarp, n_in > 0)) {
#pragma unroll 1
            for (int q0 = 0; q0 < cp.max_pieces; q0 += 4) {
                uint2 pc[4];
#pragma unroll
                for (int u = 0; u < 4; ++u)
                    pc[u] = (q0 + u < np && n_in > 0) ? cp.piece_tab[(q0 + u) * cpad + c] : make_uint2(0u, 0u);
                uint4 aa[4];
                int ib0[4];
#pragma unroll
                for (int u = 0; u < 4; ++u) { aa[u] = bal[pc[u].y >> 5]; ib0[u] = inbc[pc[u].y >> 5]; }
#pragma unroll
                for (int u = 0; u < 4; ++u) {
                    uint32_t inb = __funnelshift_r(aa[u].z, aa[u].w, pc[u].y) & pc[u].x;
                    int ib = ib0[u] + __popc(aa[u].z & ((1u << (pc[u].y & 31u)) - 1u));     // in-band bins before the piece
                    while (inb) {
                        inb &= inb - 1u;
                        if (n < kVCap) vlist[n * 32 + lane] = bandv[min(ib, BS - 1)];
                        ++n; ++ib;
                    }
                }
            }
        }
        // least fixed point of a = j + #{excluded in-band values <= s[a]}, from a = j
        int a = j;
        if (n > kVCap) {
            // more excluded values inside the band than the list holds: count by walking the pieces
            while (true) {
                const float x = sorted_at(min(a, last));
                int cnt = 0;
                for (int q = 0; q < np; ++q) {
                    const uint2 pc = cp.piece_tab[q * cpad + c];
                    const uint4 aa = bal[pc.y >> 5];
                    uint32_t inb = __funnelshift_r(aa.z, aa.w, pc.y) & pc.x;
                    int ib = inbc[pc.y >> 5] + __popc(aa.z & ((1u << (pc.y & 31u)) - 1u));
                    while (inb) {
                        inb &= inb - 1u;
                        cnt += (bandv[min(ib, BS - 1)] <= x) ? 1 : 0;
                        ++ib;
                    }
                }
                if (j + cnt == a) break;
                a = j + cnt;
            }
            n = 0;
        }
        __syncwarp();
        if (__any_sync(kFullWarp, n > 0)) {
            float v[kVCap];                                   // the lane's list, +inf beyond its end
#pragma unroll
            for (int t = 0; t < kVCap; ++t) v[t] = (t < n) ? vlist[t * 32 + lane] : __uint_as_float(kInfKey);
            bool moving = n > 0;
            while (__any_sync(kFullWarp, moving)) {
                const float x = sorted_at(min(a, last));
                int cnt = 0;
#pragma unroll
                for (int t = 0; t < kVCap; ++t) cnt += (v[t] <= x) ? 1 : 0;
                moving = moving && (j + cnt != a);
                if (moving) a = j + cnt;
            }
        }
        const float med = sorted_at(min(a, last));
        const float snr = num / fmaxf(med, cp.sf_eps);
        if (act) {
            if (dbg != nullptr) {
                dbg[c * 3 + 0] = snr;
                dbg[c * 3 + 1] = num;
                dbg[c * 3 + 2] = med;
            }
            if (best_c == 0x7fffffff || snr > best || (snr == best && c < best_c)) { best = snr; best_c = c; }
        }
        __syncwarp();
    }
    // eq. 11: max over candidates, first maximum wins
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        const float ob = __shfl_xor_sync(kFullWarp, best, o);
        const int oc = __shfl_xor_sync(kFullWarp, best_c, o);
        const bool take = (oc != 0x7fffffff) && (best_c == 0x7fffffff || ob > best || (ob == best && oc < best_c));
        if (take) { best = ob; best_c = oc; }
    }
    score_out = (best_c == 0x7fffffff) ? 0.f : best;
    f0_out = (best_c == 0x7fffffff) ? -1 : best_c;
}

// The same, out of line, for a caller that cannot afford the registers (the NDFT kernel scores a pixel
// itself only when the deferred queue is full).  The spectrum arrives in the block-maxima region of `sm`
// (bin k at k + k / NBL), which comb_score() overwrites only after it has consumed the registers.
template <int NBL, int BS>
__device__ __noinline__ float2 comb_score_from_smem(uint32_t *sm, const CombParams &cp, float mean_p, int lane, float *dbg)
{
    float p[NBL];
    const float *T = reinterpret_cast<const float *>(sm);
#pragma unroll
    for (int i = 0; i < NBL; ++i) p[i] = T[lane * (NBL + 1) + i];
    __syncwarp();
    float score;
    int f0;
    comb_score<NBL, BS>(p, sm, cp, mean_p, lane, score, f0, dbg);
    return make_float2(score, __int_as_float(f0));
}

}  // namespace
}  // namespace ddhf
