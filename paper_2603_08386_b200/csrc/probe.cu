// probe.cu -- FP32 FMA throughput probe: the measured ceiling the NDFT roofline is quoted
// against ("an FMA microbenchmark measured in the same run").
// Register-resident chains, no memory traffic: scalar FFMA and packed FFMA2 (fma.rn.f32x2).
#include "ddhf_internal.cuh"

namespace ddhf {

namespace {

constexpr int kChains = 16;
constexpr int kInner = 64;

__global__ void __launch_bounds__(256) k_fma_scalar(float *out, int iters, float a, float b)
{
    float x[kChains];
#pragma unroll
    for (int i = 0; i < kChains; ++i) x[i] = threadIdx.x * 1e-3f + i;
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int r = 0; r < kInner; ++r)
#pragma unroll
            for (int i = 0; i < kChains; ++i) x[i] = fmaf(x[i], a, b);
    }
    float s = 0.f;
#pragma unroll
    for (int i = 0; i < kChains; ++i) s += x[i];
    if (s == 123.456f) out[0] = s;
}

__global__ void __launch_bounds__(256) k_fma_packed(float *out, int iters, float a, float b)
{
    float2 x[kChains];
    const float2 aa = make_float2(a, a * 0.999f), bb = make_float2(b, b * 1.001f);
#pragma unroll
    for (int i = 0; i < kChains; ++i) x[i] = make_float2(threadIdx.x * 1e-3f + i, i * 0.5f);
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int r = 0; r < kInner; ++r)
#pragma unroll
            for (int i = 0; i < kChains; ++i) x[i] = __ffma2_rn(x[i], aa, bb);
    }
    float s = 0.f;
#pragma unroll
    for (int i = 0; i < kChains; ++i) s += x[i].x + x[i].y;
    if (s == 123.456f) out[0] = s;
}

}  // namespace

int fma_probe(float ms_target, float *tflops, cudaStream_t st)
{
    int dev = 0, sms = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return DDHF_E_CUDA;
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    float *d_out = nullptr;
    if (cudaMalloc(&d_out, 16) != cudaSuccess) return DDHF_E_CUDA;
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0);
    cudaEventCreate(&e1);
    const int blocks = sms * 8, threads = 256;
    for (int variant = 0; variant < 2; ++variant) {
        int iters = 64;
        float ms = 0.f;
        for (int attempt = 0; attempt < 12; ++attempt) {
            cudaEventRecord(e0, st);
            if (variant == 0) k_fma_scalar<<<blocks, threads, 0, st>>>(d_out, iters, 0.9999f, 1e-4f);
            else k_fma_packed<<<blocks, threads, 0, st>>>(d_out, iters, 0.9999f, 1e-4f);
            cudaEventRecord(e1, st);
            if (cudaEventSynchronize(e1) != cudaSuccess) { cudaFree(d_out); return DDHF_E_CUDA; }
            cudaEventElapsedTime(&ms, e0, e1);
            if (ms >= ms_target) break;
            iters *= 2;
        }
        const double fma = static_cast<double>(blocks) * threads * iters * kInner * kChains * (variant ? 2.0 : 1.0);
        tflops[variant] = static_cast<float>(2.0 * fma / (ms * 1e-3) / 1e12);
    }
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    cudaFree(d_out);
    return cudaGetLastError() == cudaSuccess ? DDHF_OK : DDHF_E_CUDA;
}

}  // namespace ddhf
