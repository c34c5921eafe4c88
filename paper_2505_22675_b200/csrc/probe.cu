// probe.cu -- bathy_probe_fp32: an FMA-chain microbenchmark that MEASURES the FP32 ALU peak the kriging
// roofline is reported against ("the builder measures an FMA-chain microbenchmark and
// records actual clocks").  No method arithmetic; bench.py times it with CUDA events.
#include "common.cuh"

namespace bathy {
namespace {

constexpr int kProbeThreads = 512;
constexpr int kChains = 16;          // independent accumulators per thread: hides the FMA latency at any occupancy

template <int PACKED>
__global__ void __launch_bounds__(kProbeThreads)
fp32_probe_kernel(long long iters, float seed, float* __restrict__ sink)
{
    const float a = 1.0f + seed * 1e-7f, b = seed * 1e-9f + (float)threadIdx.x * 1e-12f;
    if (PACKED) {
        u64 acc[kChains / 2];
#pragma unroll
        for (int c = 0; c < kChains / 2; ++c) acc[c] = pack2((float)c, (float)c + 0.5f);
        const u64 a2 = pack2(a, a), b2 = pack2(b, b);
        for (long long i = 0; i < iters; ++i) {
#pragma unroll
            for (int c = 0; c < kChains / 2; ++c) acc[c] = ffma2(acc[c], a2, b2);
        }
        float s = 0.0f;
#pragma unroll
        for (int c = 0; c < kChains / 2; ++c) s += lo_of(acc[c]) + hi_of(acc[c]);
        if (s == 12345.678f) sink[0] = s;                  // never true: keeps the chains alive
    } else {
        float acc[kChains];
#pragma unroll
        for (int c = 0; c < kChains; ++c) acc[c] = (float)c;
        for (long long i = 0; i < iters; ++i) {
#pragma unroll
            for (int c = 0; c < kChains; ++c) acc[c] = fmaf(acc[c], a, b);
        }
        float s = 0.0f;
#pragma unroll
        for (int c = 0; c < kChains; ++c) s += acc[c];
        if (s == 12345.678f) sink[0] = s;
    }
}

}  // namespace
}  // namespace bathy

using namespace bathy;

extern "C" BATHY_API int bathy_probe_fp32(int32_t packed, int64_t iters, int32_t ctas_per_sm, float* d_sink,
                                          double* flop_out, void* cuda_stream)
{
    if (!d_sink || !flop_out) return BATHY_ERR_NULL;
    if (iters < 1 || ctas_per_sm < 1 || ctas_per_sm > 4) return BATHY_ERR_SIZE;
    int dev = 0, sms = kSMs;
    BATHY_CUDA_TRY(cudaGetDevice(&dev));
    BATHY_CUDA_TRY(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
    const int grid = sms * ctas_per_sm;
    cudaStream_t s = static_cast<cudaStream_t>(cuda_stream);
    if (packed) fp32_probe_kernel<1><<<grid, kProbeThreads, 0, s>>>((long long)iters, 1.0f, d_sink);
    else        fp32_probe_kernel<0><<<grid, kProbeThreads, 0, s>>>((long long)iters, 1.0f, d_sink);
    count_launch();
    // every thread retires kChains FMAs (2 flop each) per iteration, in either variant
    *flop_out = 2.0 * (double)kChains * (double)iters * (double)kProbeThreads * (double)grid;
    return launch_status();
}
