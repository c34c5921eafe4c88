// krige_index.cuh -- the library-owned sounding index.
//
// Everything a kernel needs to know about the cell grid lives in a DEVICE header that the build
// kernels write and krige_predict reads, so that building (or appending to) an index never has to
// bring the bounding box back to the host: every call only enqueues work.
#pragma once
#include "common.cuh"

namespace bathy {

struct IndexHeader {
    float   xmin, ymin;         // lower corner of the cell grid
    float   cell, inv_cell;     // cell edge and its fp32 reciprocal
    int32_t ncx, ncy;           // cell grid
    float   step_hint;          // mean spacing sqrt(area / n), seeds the first search radius
    int32_t status;             // BATHY_OK, or BATHY_ERR_GEOMETRY once a non-finite coordinate was seen
    int32_t n;                  // soundings in the index
    float   bb[4];              // xmin, xmax, ymin, ymax of all soundings so far
    float   changed[4];         // xmin, xmax, ymin, ymax of the soundings of the last append
    int32_t pad[3];
};

}  // namespace bathy

struct krige_index {
    uint32_t magic;             // kIndexMagic while alive
    int64_t  n;                 // soundings (host count: the sum of what was appended)
    int64_t  capacity;          // soundings the point buffers hold
    int64_t  cells_cap;         // cells the cell arrays hold
    int      device;            // CUDA device the memory lives on
    bathy::IndexHeader* d_hdr;  // device header (what the kernels read)
    cudaStream_t stream;        // stream of the last build / append (krige_free_index waits on it)
    int      used_elsewhere;    // set once work that reads the index was issued on any other stream: krige_free_index
                                // then waits for the whole device (written with __atomic_store_n: predicts may run concurrently)
    float4*  d_pts;             // [capacity] cell-sorted (x, y, z, original index as int bits)
    float4*  d_pts_alt;         // [capacity] second buffer of an appendable index (ping-pong), else NULL
    int32_t* d_cell_start;      // [cells_cap + 1] exclusive prefix of the per-cell counts
    int32_t* d_cell_start_alt;  // [cells_cap + 1] second buffer of an appendable index, else NULL
};

namespace bathy {
constexpr uint32_t kIndexMagic = 0x4b524947u;   // "KRIG"

// An index belongs to the device it was built on: with another device current, its pointers are foreign and a
// launch would fault with a sticky context error instead of a status code.
inline bool index_on_current_device(const krige_index* idx)
{
    int dev = -1;
    return cudaGetDevice(&dev) == cudaSuccess && dev == idx->device;
}

// The cell of a coordinate, as the index build computes it (fp32, truncation, clamped).
__device__ __forceinline__ int cell_of(float v, float vmin, float inv_cell, int nc)
{
    int c = (int)((v - vmin) * inv_cell);
    return min(max(c, 0), nc - 1);
}
}  // namespace bathy
