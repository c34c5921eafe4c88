// tma_probe.cu -- bathy_probe_tma: a minimal cp.async.bulk.tensor.2d (TMA) tile load, kept as the committed
// reproduction for DESIGN.md's question "do TMA tensor loads work on this pool's B200s?" (round-1 claimed a trap).
// The load follows every rule of the PTX ISA for a tiled 2-D map: inner box bytes a multiple of 16, global row
// pitch a multiple of 16 bytes, 128-byte aligned shared-memory destination, tensor map passed as a
// __grid_constant__ kernel parameter, mbarrier expect_tx equal to the full box bytes.  Measured on the pool's B200s
// (profiles/r2_tma_probe.md): the load works when the box's first column x0 is a multiple of 4 floats (16 bytes) and
// raises an illegal-instruction exception otherwise -- the trap round 1 ran into with windows starting at 64 t - 11.
// No method arithmetic.
#include "common.cuh"
#include <cuda.h>

namespace bathy {
namespace {

constexpr int kBoxW = 88, kBoxH = 54;            // 88 floats = 352 bytes (a multiple of 16): the spline window, padded

__global__ void __launch_bounds__(128)
tma_probe_kernel(const __grid_constant__ CUtensorMap map, int x0, int y0, float* __restrict__ out)
{
    __shared__ __align__(128) float tile[kBoxH * kBoxW];
    __shared__ __align__(8) unsigned long long bar;
    const unsigned bar_a = (unsigned)__cvta_generic_to_shared(&bar);
    const unsigned dst_a = (unsigned)__cvta_generic_to_shared(tile);
    if (threadIdx.x == 0) {
        asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" :: "r"(bar_a) : "memory");
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" :: "r"(bar_a), "r"((unsigned)(kBoxH * kBoxW * sizeof(float))) : "memory");
        asm volatile("cp.async.bulk.tensor.2d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3}], [%4];"
                     :: "r"(dst_a), "l"(&map), "r"(x0), "r"(y0), "r"(bar_a) : "memory");
    }
    unsigned done = 0;
    for (int it = 0; it < (1 << 22) && !done; ++it) {      // bounded: a load that never completes must not hang the GPU
        asm volatile("{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], 0;\n\tselp.u32 %0, 1, 0, p;\n\t}"
                     : "=r"(done) : "r"(bar_a) : "memory");
    }
    for (int i = threadIdx.x; i < kBoxH * kBoxW; i += blockDim.x) out[i] = done ? tile[i] : -12345.0f;
}

typedef CUresult (*encode_fn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                              const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                              CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

}  // namespace
}  // namespace bathy

using namespace bathy;

// d_in: [ny][nx] fp32 with nx a multiple of 4; d_out: [54 * 88] fp32.  Loads the box whose first element is
// (x0, y0); elements outside the tensor arrive as zeros.  Returns BATHY_ERR_CUDA if the tensor map cannot be encoded.
extern "C" BATHY_API int bathy_probe_tma(const float* d_in, int32_t nx, int32_t ny, int32_t x0, int32_t y0, float* d_out,
                                         void* cuda_stream)
{
    if (!d_in || !d_out) return BATHY_ERR_NULL;
    if (nx < 4 || ny < 1 || (nx & 3) || (x0 & 3) || (reinterpret_cast<uintptr_t>(d_in) & 15)) return BATHY_ERR_GEOMETRY;
    void* fn = nullptr;
    cudaDriverEntryPointQueryResult qres;
    BATHY_CUDA_TRY(cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qres));
    if (!fn || qres != cudaDriverEntryPointSuccess) return BATHY_ERR_CUDA;
    CUtensorMap map;
    const cuuint64_t dims[2] = {(cuuint64_t)nx, (cuuint64_t)ny};
    const cuuint64_t strides[1] = {(cuuint64_t)nx * sizeof(float)};
    const cuuint32_t box[2] = {kBoxW, kBoxH};
    const cuuint32_t estr[2] = {1, 1};
    const CUresult r = reinterpret_cast<encode_fn>(fn)(&map, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 2, const_cast<float*>(d_in), dims, strides,
                                                       box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE,
                                                       CU_TENSOR_MAP_L2_PROMOTION_NONE, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) return BATHY_ERR_CUDA;
    tma_probe_kernel<<<1, 128, 0, static_cast<cudaStream_t>(cuda_stream)>>>(map, x0, y0, d_out);
    count_launch();
    return launch_status();
}
