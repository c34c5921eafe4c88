// krige_index.cu -- krige_build_index: bounding box -> cell id per sounding
// -> histogram -> exclusive scan -> scatter of (x, y, z, original index), counting sort by cell.
// Replaces the paper's per-thread "nearest n valid candidate neighbors" window scan
// for scattered soundings.  One-off per survey; HBM/atomic bound.
#include "krige_index.cuh"
#include <new>

namespace bathy {

namespace {

constexpr int kThreads = 256;

// ---- bounding box: per-block partials, then one block folds them (no float atomics: deterministic)
__global__ void __launch_bounds__(kThreads)
bbox_partial_kernel(const float* __restrict__ x, const float* __restrict__ y, int64_t n, float4* __restrict__ partial)
{
    float xmin = INFINITY, xmax = -INFINITY, ymin = INFINITY, ymax = -INFINITY;
    bool bad = false;
    for (int64_t i = (int64_t)blockIdx.x * kThreads + threadIdx.x; i < n; i += (int64_t)gridDim.x * kThreads) {
        const float a = x[i], b = y[i];
        bad |= !(isfinite(a) && isfinite(b));
        xmin = fminf(xmin, a); xmax = fmaxf(xmax, a);
        ymin = fminf(ymin, b); ymax = fmaxf(ymax, b);
    }
    if (bad) xmin = NAN;                                   // poison: reported as a geometry error
    __shared__ float4 s[kThreads / 32];
    for (int o = 16; o > 0; o >>= 1) {
        const float oxmin = __shfl_xor_sync(0xffffffffu, xmin, o);
        xmin = (isnan(xmin) || isnan(oxmin)) ? NAN : fminf(xmin, oxmin);
        xmax = fmaxf(xmax, __shfl_xor_sync(0xffffffffu, xmax, o));
        ymin = fminf(ymin, __shfl_xor_sync(0xffffffffu, ymin, o));
        ymax = fmaxf(ymax, __shfl_xor_sync(0xffffffffu, ymax, o));
    }
    if ((threadIdx.x & 31) == 0) s[threadIdx.x >> 5] = make_float4(xmin, xmax, ymin, ymax);
    __syncthreads();
    if (threadIdx.x == 0) {
        float4 r = s[0];
        for (int w = 1; w < kThreads / 32; ++w) {
            r.x = (isnan(r.x) || isnan(s[w].x)) ? NAN : fminf(r.x, s[w].x);
            r.y = fmaxf(r.y, s[w].y); r.z = fminf(r.z, s[w].z); r.w = fmaxf(r.w, s[w].w);
        }
        partial[blockIdx.x] = r;
    }
}

__global__ void bbox_final_kernel(const float4* __restrict__ partial, int nb, float4* __restrict__ out)
{
    // one warp: lanes stride over the partials, then a shuffle tree (min/max are order independent:
    // deterministic)
    float xmin = INFINITY, xmax = -INFINITY, ymin = INFINITY, ymax = -INFINITY;
    bool bad = false;
    for (int b = threadIdx.x; b < nb; b += 32) {
        const float4 p = partial[b];
        bad |= isnan(p.x);
        xmin = fminf(xmin, p.x); xmax = fmaxf(xmax, p.y); ymin = fminf(ymin, p.z); ymax = fmaxf(ymax, p.w);
    }
    for (int o = 16; o > 0; o >>= 1) {
        xmin = fminf(xmin, __shfl_xor_sync(0xffffffffu, xmin, o));
        xmax = fmaxf(xmax, __shfl_xor_sync(0xffffffffu, xmax, o));
        ymin = fminf(ymin, __shfl_xor_sync(0xffffffffu, ymin, o));
        ymax = fmaxf(ymax, __shfl_xor_sync(0xffffffffu, ymax, o));
    }
    bad = __any_sync(0xffffffffu, bad);
    if (threadIdx.x == 0) *out = make_float4(bad ? NAN : xmin, xmax, ymin, ymax);
}

// ---- histogram of soundings per cell
__global__ void __launch_bounds__(kThreads)
cell_count_kernel(const float* __restrict__ x, const float* __restrict__ y, int64_t n,
                  float xmin, float ymin, float inv_cell, int ncx, int ncy, int32_t* __restrict__ count)
{
    for (int64_t i = (int64_t)blockIdx.x * kThreads + threadIdx.x; i < n; i += (int64_t)gridDim.x * kThreads) {
        const int c = cell_of(y[i], ymin, inv_cell, ncy) * ncx + cell_of(x[i], xmin, inv_cell, ncx);
        atomicAdd(count + c, 1);
    }
}

// ---- exclusive scan of int32 counts: per-block scan + block sums, scan of sums, add back
constexpr int kScanItems = 8;
constexpr int kScanBlock = kThreads * kScanItems;

__global__ void __launch_bounds__(kThreads)
scan_block_kernel(const int32_t* __restrict__ in, int32_t* __restrict__ out, int64_t n, int32_t* __restrict__ sums)
{
    __shared__ int32_t s_warp[kThreads / 32];
    const int64_t base = (int64_t)blockIdx.x * kScanBlock + (int64_t)threadIdx.x * kScanItems;
    int32_t v[kScanItems];
    int32_t tsum = 0;
#pragma unroll
    for (int e = 0; e < kScanItems; ++e) {
        v[e] = (base + e < n) ? in[base + e] : 0;
        tsum += v[e];
    }
    int32_t inc = tsum;                                    // inclusive scan of thread sums in the warp
    for (int o = 1; o < 32; o <<= 1) {
        const int32_t up = __shfl_up_sync(0xffffffffu, inc, o);
        if ((threadIdx.x & 31) >= o) inc += up;
    }
    if ((threadIdx.x & 31) == 31) s_warp[threadIdx.x >> 5] = inc;
    __syncthreads();
    int32_t woff = 0;
    for (int w = 0; w < (int)(threadIdx.x >> 5); ++w) woff += s_warp[w];
    int32_t run = woff + inc - tsum;
#pragma unroll
    for (int e = 0; e < kScanItems; ++e) {
        if (base + e < n) out[base + e] = run;
        run += v[e];
    }
    if (threadIdx.x == kThreads - 1) sums[blockIdx.x] = run;
}

__global__ void __launch_bounds__(kThreads)
scan_sums_kernel(int32_t* __restrict__ sums, int nb)
{
    // one block: serial over chunks of kThreads, warp-scan inside
    __shared__ int32_t s_warp[kThreads / 32];
    __shared__ int32_t s_carry;
    if (threadIdx.x == 0) s_carry = 0;
    __syncthreads();
    for (int base = 0; base < nb; base += kThreads) {
        const int i = base + threadIdx.x;
        const int32_t v = (i < nb) ? sums[i] : 0;
        int32_t inc = v;
        for (int o = 1; o < 32; o <<= 1) {
            const int32_t up = __shfl_up_sync(0xffffffffu, inc, o);
            if ((threadIdx.x & 31) >= o) inc += up;
        }
        if ((threadIdx.x & 31) == 31) s_warp[threadIdx.x >> 5] = inc;
        __syncthreads();
        int32_t woff = s_carry;
        for (int w = 0; w < (int)(threadIdx.x >> 5); ++w) woff += s_warp[w];
        if (i < nb) sums[i] = woff + inc - v;
        __syncthreads();
        if (threadIdx.x == kThreads - 1) s_carry = woff + inc;
        __syncthreads();
    }
}

__global__ void __launch_bounds__(kThreads)
scan_add_kernel(int32_t* __restrict__ out, int64_t n, const int32_t* __restrict__ sums, int32_t total)
{
    const int64_t base = (int64_t)blockIdx.x * kScanBlock;
    const int32_t off = sums[blockIdx.x];
    for (int e = threadIdx.x; e < kScanBlock; e += kThreads)
        if (base + e < n) out[base + e] += off;
    if (blockIdx.x == 0 && threadIdx.x == 0) out[n] = total;
}

// ---- scatter by cell (atomic cursor), then order every cell by original index so that the
//      index -- and with it every later result -- does not depend on atomic arrival order
__global__ void __launch_bounds__(kThreads)
scatter_kernel(const float* __restrict__ x, const float* __restrict__ y, const float* __restrict__ z, int64_t n,
               float xmin, float ymin, float inv_cell, int ncx, int ncy,
               int32_t* __restrict__ cursor, float4* __restrict__ tmp)
{
    for (int64_t i = (int64_t)blockIdx.x * kThreads + threadIdx.x; i < n; i += (int64_t)gridDim.x * kThreads) {
        const float a = x[i], b = y[i];
        const int c = cell_of(b, ymin, inv_cell, ncy) * ncx + cell_of(a, xmin, inv_cell, ncx);
        const int32_t p = atomicAdd(cursor + c, 1);
        tmp[p] = make_float4(a, b, z[i], __int_as_float((int32_t)i));
    }
}

__global__ void __launch_bounds__(kThreads)
order_cells_kernel(const float4* __restrict__ tmp, int64_t n, float xmin, float ymin, float inv_cell,
                   int ncx, int ncy, const int32_t* __restrict__ cell_start, float4* __restrict__ pts)
{
    for (int64_t p = (int64_t)blockIdx.x * kThreads + threadIdx.x; p < n; p += (int64_t)gridDim.x * kThreads) {
        const float4 me = tmp[p];
        const int c = cell_of(me.y, ymin, inv_cell, ncy) * ncx + cell_of(me.x, xmin, inv_cell, ncx);
        const int32_t s = cell_start[c], e = cell_start[c + 1];
        const int32_t my = __float_as_int(me.w);
        int32_t rank = 0;
        for (int32_t q = s; q < e; ++q) rank += (__float_as_int(tmp[q].w) < my);
        pts[s + rank] = me;
    }
}

inline int grid_for(int64_t n)
{
    int64_t b = (n + kThreads - 1) / kThreads;
    const int64_t cap = (int64_t)kSMs * 8;
    return (int)(b < cap ? (b < 1 ? 1 : b) : cap);
}

}  // namespace


// The default memory pool gives freed blocks back to the driver at every synchronisation unless its
// release threshold is raised; with it raised, cudaMallocAsync of the index and its scratch is a
// pointer bump after the first call.  Once per device.
static void pool_keep_warm()
{
    static bool done[64] = {};
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= 64 || done[dev]) return;
    cudaMemPool_t pool;
    if (cudaDeviceGetDefaultMemPool(&pool, dev) == cudaSuccess) {
        unsigned long long keep = 1ull << 31;              // hold up to 2 GiB of freed blocks
        cudaMemPoolSetAttribute(pool, cudaMemPoolAttrReleaseThreshold, &keep);
    }
    done[dev] = true;
}

int build_index(const float* d_x, const float* d_y, const float* d_z, int64_t n, float cell_size,
                cudaStream_t stream, krige_index** out_index)
{
    *out_index = nullptr;
    // 1. bounding box
    pool_keep_warm();
    const int nb = grid_for(n);
    float4* d_partial = nullptr;
    BATHY_CUDA_TRY(cudaMallocAsync(&d_partial, sizeof(float4) * (size_t)(nb + 1), stream));
    bbox_partial_kernel<<<nb, kThreads, 0, stream>>>(d_x, d_y, n, d_partial);
    bbox_final_kernel<<<1, 32, 0, stream>>>(d_partial, nb, d_partial + nb);
    count_launch(2);
    float4 bb;
    BATHY_CUDA_TRY(cudaMemcpyAsync(&bb, d_partial + nb, sizeof(float4), cudaMemcpyDeviceToHost, stream));
    BATHY_CUDA_TRY(cudaStreamSynchronize(stream));
    BATHY_CUDA_TRY(cudaFreeAsync(d_partial, stream));
    if (!(isfinite(bb.x) && isfinite(bb.y) && isfinite(bb.z) && isfinite(bb.w))) return BATHY_ERR_GEOMETRY;

    // 2. cell grid
    const double w = (double)bb.y - (double)bb.x, h = (double)bb.w - (double)bb.z;
    double cell = cell_size;
    if (!(cell > 0.0)) {
        const double area = w * h;
        if (area > 0.0) cell = sqrt(8.0 * area / (double)n);           // about 8 soundings per cell
        else if (w > 0.0 || h > 0.0) cell = 8.0 * (w > h ? w : h) / (double)n;
        else cell = 1.0;
        if (!(cell > 0.0) || !isfinite(cell)) cell = 1.0;
    }
    int ncx = 1, ncy = 1;
    float cellf = 0.0f, inv = 0.0f;
    for (int it = 0; it < 64; ++it) {
        cellf = (float)cell;
        if (!(cellf > 0.0f) || !isfinite(cellf)) return BATHY_ERR_GEOMETRY;
        inv = 1.0f / cellf;
        const double fx = (double)((bb.y - bb.x) * inv), fy = (double)((bb.w - bb.z) * inv);   // as cell_of computes it
        if (fx < 32768.0 && fy < 32768.0 && (floor(fx) + 1.0) * (floor(fy) + 1.0) <= (double)(1 << 26)) {
            ncx = (int)fx + 1;
            ncy = (int)fy + 1;
            break;
        }
        cell *= 2.0;
        if (it == 63) return BATHY_ERR_SIZE;
    }
    const int64_t ncells = (int64_t)ncx * ncy;

    // 3. allocate the index
    krige_index* idx = new (std::nothrow) krige_index();
    if (!idx) return BATHY_ERR_CUDA;
    idx->magic = 0;
    idx->n = n;
    idx->xmin = bb.x; idx->ymin = bb.z;
    idx->cell = cellf; idx->inv_cell = inv;
    idx->ncx = ncx; idx->ncy = ncy;
    {
        const double area = (w > 0 ? w : cell) * (h > 0 ? h : cell);
        idx->step_hint = (float)sqrt(area / (double)n);
    }
    idx->d_pts = nullptr; idx->d_cell_start = nullptr;
    float4* d_tmp = nullptr;
    int32_t* d_cursor = nullptr;
    int32_t* d_sums = nullptr;
    const int nsb = (int)((ncells + kScanBlock - 1) / kScanBlock);
    // stream-ordered allocations from the device's default pool (kept warm, see pool_keep_warm):
    // a synchronous cudaMalloc costs more than all the kernels of the build together
    cudaError_t e = cudaMallocAsync(&idx->d_pts, sizeof(float4) * (size_t)n, stream);
    if (e == cudaSuccess) e = cudaMallocAsync(&idx->d_cell_start, sizeof(int32_t) * (size_t)(ncells + 1), stream);
    if (e == cudaSuccess) e = cudaMallocAsync(&d_tmp, sizeof(float4) * (size_t)n, stream);
    if (e == cudaSuccess) e = cudaMallocAsync(&d_cursor, sizeof(int32_t) * (size_t)(ncells + 1), stream);
    if (e == cudaSuccess) e = cudaMallocAsync(&d_sums, sizeof(int32_t) * (size_t)(nsb + 1), stream);
    if (e == cudaSuccess) e = cudaMemsetAsync(d_cursor, 0, sizeof(int32_t) * (size_t)(ncells + 1), stream);
    if (e != cudaSuccess) {
        cudaGetLastError();
        if (d_tmp) cudaFreeAsync(d_tmp, stream);
        if (d_cursor) cudaFreeAsync(d_cursor, stream);
        if (d_sums) cudaFreeAsync(d_sums, stream);
        if (idx->d_pts) cudaFreeAsync(idx->d_pts, stream);
        if (idx->d_cell_start) cudaFreeAsync(idx->d_cell_start, stream);
        delete idx;
        return BATHY_ERR_CUDA;
    }

    // 4. histogram -> exclusive scan -> scatter -> order cells
    const int g = grid_for(n);
    cell_count_kernel<<<g, kThreads, 0, stream>>>(d_x, d_y, n, idx->xmin, idx->ymin, inv, ncx, ncy, d_cursor);
    scan_block_kernel<<<nsb, kThreads, 0, stream>>>(d_cursor, idx->d_cell_start, ncells, d_sums);
    scan_sums_kernel<<<1, kThreads, 0, stream>>>(d_sums, nsb);
    scan_add_kernel<<<nsb, kThreads, 0, stream>>>(idx->d_cell_start, ncells, d_sums, (int32_t)n);
    cudaMemcpyAsync(d_cursor, idx->d_cell_start, sizeof(int32_t) * (size_t)ncells, cudaMemcpyDeviceToDevice, stream);
    scatter_kernel<<<g, kThreads, 0, stream>>>(d_x, d_y, d_z, n, idx->xmin, idx->ymin, inv, ncx, ncy, d_cursor, d_tmp);
    order_cells_kernel<<<g, kThreads, 0, stream>>>(d_tmp, n, idx->xmin, idx->ymin, inv, ncx, ncy, idx->d_cell_start, idx->d_pts);
    count_launch(6);
    const int st = launch_status();
    cudaFreeAsync(d_tmp, stream);
    cudaFreeAsync(d_cursor, stream);
    cudaFreeAsync(d_sums, stream);
    if (st != BATHY_OK) {
        if (idx->d_pts) cudaFreeAsync(idx->d_pts, stream);
        if (idx->d_cell_start) cudaFreeAsync(idx->d_cell_start, stream);
        delete idx;
        return st;
    }
    idx->magic = kIndexMagic;
    *out_index = idx;
    return BATHY_OK;
}

void free_index(krige_index* idx)
{
    if (!idx || idx->magic != kIndexMagic) return;
    cudaDeviceSynchronize();
    idx->magic = 0;
    cudaFreeAsync(idx->d_pts, 0);                          // (the device is idle: synchronised above)
    cudaFreeAsync(idx->d_cell_start, 0);
    delete idx;
}

// Stream-ordered release: the memory goes back to the pool when `stream` reaches this point; no host
// synchronisation.
void free_index_async(krige_index* idx, cudaStream_t stream)
{
    if (!idx || idx->magic != kIndexMagic) return;
    idx->magic = 0;
    cudaFreeAsync(idx->d_pts, stream);
    cudaFreeAsync(idx->d_cell_start, stream);
    delete idx;
}

}  // namespace bathy
