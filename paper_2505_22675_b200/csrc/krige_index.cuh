// krige_index.cuh -- the library-owned sounding index.
#pragma once
#include "common.cuh"

struct krige_index {
    uint32_t magic;             // kIndexMagic while alive
    int64_t  n;                 // soundings
    float    xmin, ymin;        // lower corner of the bounding box
    float    cell, inv_cell;    // cell edge and its fp32 reciprocal
    int32_t  ncx, ncy;          // cell grid
    float    step_hint;         // mean spacing sqrt(area / n), seeds the first search radius
    float4*  d_pts;             // [n] cell-sorted (x, y, z, original index as int bits)
    int32_t* d_cell_start;      // [ncx*ncy + 1] exclusive prefix of the per-cell counts
};

namespace bathy {
constexpr uint32_t kIndexMagic = 0x4b524947u;   // "KRIG"

// The cell of a coordinate, as the index build computes it (fp32, truncation, clamped).
__device__ __forceinline__ int cell_of(float v, float vmin, float inv_cell, int nc)
{
    int c = (int)((v - vmin) * inv_cell);
    return min(max(c, 0), nc - 1);
}
}  // namespace bathy
