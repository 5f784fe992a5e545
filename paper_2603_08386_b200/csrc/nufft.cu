// nufft.cu -- SURVEY 8(f)-4: the power spectrum of a long row by a type-1 non-uniform FFT instead of the
// direct sum (footnote 1 of section 3.3: "NUFFTs [22] offer asymptotic acceleration for large
// sample counts").  Optional (DDHF_FLAG_NUFFT), approximate (the error bound is part of the interface: see
// include/ddhf.h), and reported apart from the "terms" metric: a row that takes this path costs the same
// whatever its length, so a rate in (pixel x bin x event) terms means nothing for it.
//
//   X_k = sum_j w_j e^{-2 pi i (f_min + k df) t_j},  k < 2048        (eq. 6)
//       = sum_j c_j e^{-2 pi i k' th_j},   k' = k - 1024,  th_j = df t_j,  c_j = w_j e^{-2 pi i (f_min + 1024 df) t_j}
//
// 1. Spreading: every event adds c_j phi((n' - N th_j) / 4) to the 8 cells n' nearest to N th_j of a uniform
//    grid of N = 4096 cells per turn (upsampling 2 for modes |k'| <= 1024), phi(z) = exp(beta (sqrt(1 - z^2) - 1)),
//    beta = 2.3 x 8: the "exponential of semicircle" kernel.  The events of a window cover df x window < 1/4 of
//    a turn on every grid of BASELINE.json (the frequency grid is finer than 1 / window), so only the first
//    1024 cells are ever touched; they live in the warp's shared memory.  Windows for which that does not
//    hold take the direct path.
// 2. FFT: Y_q = sum_{n < 1024} x_n e^{-2 pi i n q / 4096} for the 2048 wanted q = k' mod 4096, as four
//    1024-point FFTs (q = 4 m + r: the input times e^{-2 pi i n r / 4096}), each one 32 x 32: lane n1 transforms
//    x[n1 + 32 n2] over n2 in registers, twiddles, the warp transposes through shared memory, lane m2
//    transforms over n1.  Of the 32 outputs per lane 16 are wanted; the rest is dead code.
// 3. Deconvolution and power: P_k = |Y_q|^2 / psi^(k')^2, psi^ the Fourier transform of the kernel
//    (host, double precision, at create time).  A shift of the grid origin only turns the phase of Y.
// The row then goes through the same epilogue as in k_ndft_score (spectral flatness, scoring queue).
#include "ddhf_internal.cuh"

#include <cmath>
#include <vector>

namespace ddhf {

namespace {

constexpr int kTaps = 8;                   // spreading width in cells
constexpr int kFine = 4096;                // cells per turn
constexpr int kCells = 1024;               // cells a window may touch (a quarter turn)
constexpr int kNuWarps = 12;               // warps per CTA: 16.25 KB of shared memory each
constexpr int kTPitch = 33;                // row pitch of the transpose buffer in float2
constexpr int kWarpF2 = kCells + 32 * kTPitch;   // float2 per warp: grid + transpose buffer
constexpr unsigned kFull = 0xffffffffu;
constexpr double kPi = 3.14159265358979323846;
constexpr double kBeta = 2.30 * kTaps;

__constant__ float2 c_w128[4][32];         // e^{-2 pi i n2 r / 128}
__device__ float2 g_tw[4 * 32 * 32];       // [r][m2][n1] e^{-2 pi i n1 (4 m2 + r) / 4096}
__device__ float g_deconv[4 * 16 * 32];    // [r][jj][lane] 1 / psi^(k - 1024)^2 of bin k = 128 jj + 4 lane + r

__device__ __forceinline__ uint32_t phase_u32(uint64_t g, uint32_t t)
{
    // hi 32 bits of (g * t mod 2^64): f t in turns, 2^-32 resolution
    return static_cast<uint32_t>(g >> 32) * t + __umulhi(static_cast<uint32_t>(g), t);
}

// -(sin, cos) of 2 pi ph / 2^32 (the common sign does not reach the power)
__device__ __forceinline__ void sincos_u32(uint32_t ph, float &s, float &c)
{
    const float r = fmaf(__uint_as_float((ph >> 9) | 0x3f800000u), 6.283185307179586f, -9.42477796076938f);
    s = __sinf(r);
    c = __cosf(r);
}

// ---- 32-point FFT in registers: radix-2 decimation in frequency, twiddles are immediates, the result is in
// bit-reversed order (a compile-time renaming) ----------------------------------------------------------------
__host__ __device__ constexpr double cx_cos(double x)
{
    double x2 = x * x, term = 1.0, sum = 1.0;
    for (int i = 1; i <= 16; ++i) { term *= -x2 / ((2 * i - 1) * (2 * i)); sum += term; }
    return sum;
}
__host__ __device__ constexpr double cx_sin(double x)
{
    double x2 = x * x, term = x, sum = x;
    for (int i = 1; i <= 16; ++i) { term *= -x2 / ((2 * i) * (2 * i + 1)); sum += term; }
    return sum;
}
__host__ __device__ constexpr int brev5(int m) { return ((m & 1) << 4) | ((m & 2) << 2) | (m & 4) | ((m & 8) >> 2) | ((m & 16) >> 4); }

template <int S, int I>
__device__ __forceinline__ void bfly(float2 (&v)[32])
{
    constexpr int LEN = 32 >> S, HALF = LEN / 2;
    constexpr int J = I % HALF, LO = (I / HALF) * LEN + J, HI = LO + HALF;
    constexpr int K = J * (32 / LEN);                       // twiddle e^{-2 pi i K / 32}
    const float2 a = v[LO], b = v[HI];
    v[LO] = make_float2(a.x + b.x, a.y + b.y);
    const float dx = a.x - b.x, dy = a.y - b.y;
    if constexpr (K == 0) {
        v[HI] = make_float2(dx, dy);
    } else if constexpr (K == 8) {
        v[HI] = make_float2(dy, -dx);                       // times -i
    } else {
        constexpr float c = static_cast<float>(cx_cos(2.0 * kPi * K / 32.0));
        constexpr float s = static_cast<float>(cx_sin(2.0 * kPi * K / 32.0));
        v[HI] = make_float2(fmaf(dy, s, dx * c), fmaf(-dx, s, dy * c));     // (dx + i dy)(c - i s)
    }
}

template <int T>
__device__ __forceinline__ void fft32_from(float2 (&v)[32])
{
    if constexpr (T < 80) {
        bfly<T / 16, T % 16>(v);
        fft32_from<T + 1>(v);
    }
}

// v[brev5(m)] = sum_n v[n] e^{-2 pi i n m / 32}
__device__ __forceinline__ void fft32(float2 (&v)[32]) { fft32_from<0>(v); }

}  // namespace

namespace {

// ---- k_nufft_score: one warp per row of the hot list --------------------------------------------------------
__global__ void __launch_bounds__(kNuWarps * 32, 1) k_nufft_score(NufftParams q)
{
    extern __shared__ __align__(16) uint32_t smem_raw[];
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    float2 *grid = reinterpret_cast<float2 *>(smem_raw) + wid * kWarpF2;    // [kCells]
    float2 *tbuf = grid + kCells;                                           // [32][kTPitch]
    const NdftParams &p = q.nd;
    const ScoreParams &sp = p.sp;
    // the row's spectrum in bin order; every lane reads back only what it wrote itself (bins 128 jj + 4 lane + r)
    float *prow = q.scratch + static_cast<size_t>(blockIdx.x * kNuWarps + wid) * 2048;
    const int n_hot = *q.n_hot;
    const int tap = lane & 7, grp = lane >> 3;
    const float tap_off = static_cast<float>(tap - 3);
    const bool pair_logs = sp.sf_eps >= 1e-18f;        // log2(a b) of two floored powers stays a normal number

    while (true) {
        int idx = 0;
        if (lane == 0) idx = atomicAdd(q.cursor, 1);
        idx = __shfl_sync(kFull, idx, 0);
        if (idx >= n_hot) break;
        const WorkItem it = q.hot[idx];

        // ---- 1. spreading ---------------------------------------------------------------------------------
        {
            float4 *g4 = reinterpret_cast<float4 *>(grid);
#pragma unroll
            for (int i = 0; i < kCells / 64; ++i) g4[i * 32 + lane] = make_float4(0.f, 0.f, 0.f, 0.f);
        }
        __syncwarp();
        uint32_t v_next = (lane < it.n) ? __ldg(p.csr_ev + it.row_begin + lane) : 0u;
#pragma unroll 1
        for (int base = 0; base < it.n; base += 32) {
            const uint32_t v = v_next;
            if (base + 32 + lane < it.n) v_next = __ldg(p.csr_ev + it.row_begin + base + 32 + lane);
            const uint32_t t = v >> 1;
            float sn, cs;
            sincos_u32(phase_u32(q.g_c, t), sn, cs);
            const uint32_t sgn = (v & 1u) ? 0u : 0x80000000u;             // w = +1 if bit 0 else -1
            cs = __uint_as_float(__float_as_uint(cs) ^ sgn);
            sn = __uint_as_float(__float_as_uint(sn) ^ sgn);
            const uint32_t pt = phase_u32(q.g_t, t);                      // th in turns; N th = top 12 bits . rest
            const int n0 = static_cast<int>(pt >> 20);
            const float fr = static_cast<float>(pt << 12) * 2.3283064365386963e-10f;
            const int nc = min(32, it.n - base);
#pragma unroll 1
            for (int e0 = 0; e0 < nc; e0 += 4) {
                // four events at a time, one tap per lane
                const int e = e0 + grp;
                const float cr = __shfl_sync(kFull, cs, e), ci = __shfl_sync(kFull, sn, e);
                const int nn = __shfl_sync(kFull, n0, e);
                const float f = __shfl_sync(kFull, fr, e);
                const bool valid = e < nc;
                const float d = tap_off - f;                              // cell - N th in (-4, 4]
                const float s = sqrtf(fmaxf(fmaf(d * 0.0625f, -d, 1.f), 0.f));
                const float phi = exp2f(static_cast<float>(kBeta * 1.4426950408889634) * (s - 1.f));
                float2 *cell = grid + nn + tap;
                // the windows of the four events may overlap: one event at a time adds to the grid
#pragma unroll
                for (int g = 0; g < 4; ++g) {
                    if (grp == g && valid) {
                        float2 c = *cell;
                        c.x = fmaf(cr, phi, c.x);
                        c.y = fmaf(ci, phi, c.y);
                        *cell = c;
                    }
                    __syncwarp();
                }
            }
        }
        __syncwarp();

        // ---- 2. + 3. four 1024-point FFTs, deconvolution, power, sums of the spectral flatness -------------
        float slog = 0.f, ssum = 0.f;
#pragma unroll 1
        for (int r = 0; r < 4; ++r) {
            float2 v[32];
            if (r == 0) {
#pragma unroll
                for (int n2 = 0; n2 < 32; ++n2) v[n2] = grid[lane + 32 * n2];
            } else {
#pragma unroll
                for (int n2 = 0; n2 < 32; ++n2) {
                    const float2 x = grid[lane + 32 * n2], w = c_w128[r][n2];
                    v[n2] = make_float2(fmaf(-x.y, w.y, x.x * w.x), fmaf(x.y, w.x, x.x * w.y));
                }
            }
            fft32(v);                                                    // over n2: v[brev5(m2)]
            const float2 *tw = g_tw + r * 1024 + lane;
#pragma unroll
            for (int m2 = 0; m2 < 32; ++m2) {
                const float2 x = v[brev5(m2)], w = __ldg(tw + m2 * 32);
                tbuf[m2 * kTPitch + lane] = make_float2(fmaf(-x.y, w.y, x.x * w.x), fmaf(x.y, w.x, x.x * w.y));
            }
            __syncwarp();
#pragma unroll
            for (int n1 = 0; n1 < 32; ++n1) v[n1] = tbuf[lane * kTPitch + n1];
            __syncwarp();
            fft32(v);                                                    // over n1: v[brev5(m1)]
            const float *dc = g_deconv + r * 512 + lane;
            const int k0 = 4 * lane + r;
#pragma unroll
            for (int jj = 0; jj < 16; jj += 2) {
                float pw[2], fl[2];
                bool in[2];
#pragma unroll
                for (int u = 0; u < 2; ++u) {
                    const int j = jj + u, m1 = (j < 8) ? j + 24 : j - 8;   // k' = k - 1024 < 0 first
                    const float2 y = v[brev5(m1)];
                    const int k = 128 * j + k0;
                    pw[u] = (y.x * y.x + y.y * y.y) * __ldg(dc + j * 32);
                    prow[k] = pw[u];
                    in[u] = k >= sp.k_lo && k < sp.n_freq;
                    fl[u] = fmaxf(pw[u], sp.sf_eps);
                }
                if (pair_logs) {
                    slog += __log2f((in[0] ? fl[0] : 1.f) * (in[1] ? fl[1] : 1.f));
                } else {
                    slog += (in[0] ? __log2f(fl[0]) : 0.f) + (in[1] ? __log2f(fl[1]) : 0.f);
                }
                ssum += (in[0] ? fl[0] : 0.f) + (in[1] ? fl[1] : 0.f);
            }
        }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            slog += __shfl_xor_sync(kFull, slog, o);
            ssum += __shfl_xor_sync(kFull, ssum, o);
        }

        // ---- epilogue: as in k_ndft_score ---------------------------------------------------------------
        const float inv_nb = 1.f / static_cast<float>(sp.n_freq - sp.k_lo);
        const float mean_p = ssum * inv_nb;
        const float sfv = exp2f(slog * inv_nb) / mean_p;         // eq. 7
        const bool sf_ok = sfv <= sp.tau_sf;                     // discard if SF > tau_sf (L107)
        const bool has_row = it.arow < p.max_active;
        if (p.power != nullptr && has_row) {
            __syncwarp();                                        // the row was written by all lanes
            float *dst = p.power + static_cast<size_t>(it.arow) * sp.n_freq;
#pragma unroll 4
            for (int k = lane; k < sp.n_freq; k += 32) __stcs(dst + k, prow[k]);
        }
        bool deferred = false;
        if (sp.score_all || sf_ok) {
            int slot = 0;
            if (lane == 0) slot = atomicAdd(p.spill_count, 1);
            slot = __shfl_sync(kFull, slot, 0);
            if (slot < p.spill_cap) {        // always: this path runs only when the queue holds a row per pixel
                deferred = true;
                float4 *dst = reinterpret_cast<float4 *>(p.spill + static_cast<size_t>(slot) * 2048);
                const float4 *src = reinterpret_cast<const float4 *>(prow);
#pragma unroll
                for (int i = 0; i < 16; ++i) dst[i * 32 + lane] = src[i * 32 + lane];
                if (lane == 0) {
                    SpillRec rec;
                    rec.pix = it.pix; rec.arow = has_row ? it.arow : -1; rec.mean_p = mean_p; rec._pad = 0;
                    p.spill_rec[slot] = rec;
                }
            }
        }
        if (lane == 0) {
            p.sf[it.pix] = sfv;
            if (!deferred) {
                p.score[it.pix] = 0.f;
                p.f0_idx[it.pix] = -1;
                p.mask[it.pix] = 0;
            }
        }
        __syncwarp();
    }
}

}  // namespace

// ---- host side ------------------------------------------------------------------------------------------------
bool nufft_supported(int n_freq) { return ndft_bins_per_lane(n_freq) == 64; }     // the 4096-cell grid: 1024 < n_freq <= 2048

bool nufft_window_fits(double df_hz, int64_t window_us)
{
    // cells touched: [0, N df window] widened by the taps; one cell of margin for the rounding of the phase
    const double span = df_hz * static_cast<double>(window_us) * 1e-6 * kFine;
    return df_hz > 0.0 && span + kTaps + 1 <= kCells;
}

size_t nufft_smem_bytes() { return sizeof(float2) * kWarpF2 * kNuWarps; }
int nufft_warps() { return kNuWarps; }

cudaError_t nufft_configure()
{
    // the tables depend on nothing but the kernel's own constants: (re)written at every create
    std::vector<float2> w128(4 * 32), tw(4 * 32 * 32);
    for (int r = 0; r < 4; ++r)
        for (int n2 = 0; n2 < 32; ++n2) {
            const double a = -2.0 * kPi * (n2 * r) / 128.0;
            w128[r * 32 + n2] = make_float2(static_cast<float>(cos(a)), static_cast<float>(sin(a)));
        }
    for (int r = 0; r < 4; ++r)
        for (int m2 = 0; m2 < 32; ++m2)
            for (int n1 = 0; n1 < 32; ++n1) {
                const double a = -2.0 * kPi * (n1 * (4 * m2 + r)) / static_cast<double>(kFine);
                tw[(r * 32 + m2) * 32 + n1] = make_float2(static_cast<float>(cos(a)), static_cast<float>(sin(a)));
            }
    // psi^(k') = integral over d in [-4, 4] of phi(d / 4) cos(2 pi k' d / N): Simpson, 8192 intervals
    std::vector<float> dec(4 * 16 * 32);
    const int n_int = 8192;
    const double hw = kTaps / 2.0, hstep = 2.0 * hw / n_int;
    std::vector<double> ph(n_int + 1);
    for (int i = 0; i <= n_int; ++i) {
        const double z = (-hw + i * hstep) / hw, u = 1.0 - z * z;
        ph[i] = exp(kBeta * (sqrt(u > 0.0 ? u : 0.0) - 1.0));
    }
    for (int k = 0; k < 2048; ++k) {
        const double om = 2.0 * kPi * (k - 1024) / static_cast<double>(kFine);
        double acc = 0.0;
        for (int i = 0; i <= n_int; ++i) {
            const double wgt = (i == 0 || i == n_int) ? 1.0 : (i & 1) ? 4.0 : 2.0;
            acc += wgt * ph[i] * cos(om * (-hw + i * hstep));
        }
        const double psi = acc * hstep / 3.0;
        const int jj = k >> 7, lane = (k & 127) >> 2, r = k & 3;
        dec[(r * 16 + jj) * 32 + lane] = static_cast<float>(1.0 / (psi * psi));
    }
    cudaError_t e = cudaMemcpyToSymbol(c_w128, w128.data(), sizeof(float2) * w128.size());
    if (e != cudaSuccess) return e;
    e = cudaMemcpyToSymbol(g_tw, tw.data(), sizeof(float2) * tw.size());
    if (e != cudaSuccess) return e;
    e = cudaMemcpyToSymbol(g_deconv, dec.data(), sizeof(float) * dec.size());
    if (e != cudaSuccess) return e;
    return cudaFuncSetAttribute(k_nufft_score, cudaFuncAttributeMaxDynamicSharedMemorySize, static_cast<int>(nufft_smem_bytes()));
}

int launch_nufft(const NufftParams &q, int grid, cudaStream_t st)
{
    k_nufft_score<<<grid, kNuWarps * 32, nufft_smem_bytes(), st>>>(q);
    return 1;
}

}  // namespace ddhf
