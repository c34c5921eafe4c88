// krige_index.cu -- krige_build_index / krige_index_create / krige_index_append (SURVEY.md 8(a) row K1,
// 8(f) NEXT-3): bounding box -> cell grid (sized ON THE DEVICE) -> cell id per sounding -> histogram ->
// exclusive scan -> scatter of (x, y, z, original index), counting sort by cell, stable in the original
// index.  Replaces the paper's per-thread "nearest n valid candidate neighbors" window scan
// for scattered soundings.  HBM/atomic bound.  Every call only ENQUEUES work: the cell
// grid lives in a device header (krige_index.cuh), nothing comes back to the host inside a call.
// An append merges a new batch of soundings into the sorted arrays (old soundings shift right by the
// number of new ones in the cells before theirs, the new ones follow the old ones of their cell in
// original-index order), so that create + append(A) + append(B) is bit-identical to create + append(A|B).
#include "krige_index.cuh"
#include <atomic>
#include <new>
#include <string.h>

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


// ---- cell grid from the bounding box, on the device (one thread).  mode 0: the grid covers the
//      bounding box `bb` of the soundings (krige_build_index); mode 1: the grid covers the caller's
//      extent `ext` (krige_index_create) and bb only seeds the running bounding box.
__global__ void size_grid_kernel(const float4* __restrict__ bb_in, float4 ext, int mode, long long n, float cell_size,
                                 long long cells_cap, IndexHeader* __restrict__ hdr)
{
    if (threadIdx.x != 0 || blockIdx.x != 0) return;
    IndexHeader h;
    const float4 bb = mode == 0 ? *bb_in : ext;            // xmin, xmax, ymin, ymax
    h.status = BATHY_OK;
    if (!(isfinite(bb.x) && isfinite(bb.y) && isfinite(bb.z) && isfinite(bb.w))) h.status = BATHY_ERR_GEOMETRY;
    const double w = (double)bb.y - (double)bb.x, hh = (double)bb.w - (double)bb.z;
    const double nn = (double)(n > 0 ? n : 1);
    double cell = cell_size;
    if (!(cell > 0.0)) {
        const double area = w * hh;
        if (area > 0.0) cell = sqrt(8.0 * area / nn);                  // about 8 soundings per cell
        else if (w > 0.0 || hh > 0.0) cell = 8.0 * (w > hh ? w : hh) / nn;
        else cell = 1.0;
        if (!(cell > 0.0) || !isfinite(cell)) cell = 1.0;
    }
    int ncx = 1, ncy = 1;
    float cellf = 1.0f, inv = 1.0f;
    for (int it = 0; it < 200; ++it) {
        cellf = (float)cell;
        if (!(cellf > 0.0f) || !isfinite(cellf)) { h.status = BATHY_ERR_GEOMETRY; cellf = 1.0f; inv = 1.0f; ncx = ncy = 1; break; }
        inv = 1.0f / cellf;
        const double fx = (double)((bb.y - bb.x) * inv), fy = (double)((bb.w - bb.z) * inv);   // as cell_of computes it
        if (fx < 32768.0 && fy < 32768.0 && (floor(fx) + 1.0) * (floor(fy) + 1.0) <= (double)cells_cap) {
            ncx = (int)fx + 1;
            ncy = (int)fy + 1;
            break;
        }
        cell *= 2.0;
        if (it == 199) { h.status = BATHY_ERR_GEOMETRY; ncx = ncy = 1; }
    }
    if (h.status != BATHY_OK) { ncx = ncy = 1; }
    h.xmin = (h.status == BATHY_OK) ? bb.x : 0.0f; h.ymin = (h.status == BATHY_OK) ? bb.z : 0.0f;
    h.cell = cellf; h.inv_cell = inv; h.ncx = ncx; h.ncy = ncy;
    const double area = (w > 0 ? w : cell) * (hh > 0 ? hh : cell);
    h.step_hint = (float)sqrt(area / nn);
    h.n = 0;
    h.bb[0] = INFINITY; h.bb[1] = -INFINITY; h.bb[2] = INFINITY; h.bb[3] = -INFINITY;
    h.changed[0] = INFINITY; h.changed[1] = -INFINITY; h.changed[2] = INFINITY; h.changed[3] = -INFINITY;
    h.pad[0] = h.pad[1] = h.pad[2] = 0;
    *hdr = h;
}

// ---- after an append: count, running bounding box, bounding box of the batch, poisoned input
__global__ void header_update_kernel(IndexHeader* __restrict__ hdr, const float4* __restrict__ bb_new, int n_new,
                                     float* __restrict__ changed_out)
{
    if (threadIdx.x != 0 || blockIdx.x != 0) return;
    const float4 b = *bb_new;
    if (!(isfinite(b.x) && isfinite(b.y) && isfinite(b.z) && isfinite(b.w))) hdr->status = BATHY_ERR_GEOMETRY;
    hdr->n += n_new;
    hdr->bb[0] = fminf(hdr->bb[0], b.x); hdr->bb[1] = fmaxf(hdr->bb[1], b.y);
    hdr->bb[2] = fminf(hdr->bb[2], b.z); hdr->bb[3] = fmaxf(hdr->bb[3], b.w);
    hdr->changed[0] = b.x; hdr->changed[1] = b.y; hdr->changed[2] = b.z; hdr->changed[3] = b.w;
    if (changed_out) { changed_out[0] = b.x; changed_out[1] = b.y; changed_out[2] = b.z; changed_out[3] = b.w; }
    // mean spacing over the area the soundings cover so far (seeds the first search radius)
    const double w = (double)hdr->bb[1] - (double)hdr->bb[0], h = (double)hdr->bb[3] - (double)hdr->bb[2];
    const double c = hdr->cell;
    if (hdr->n > 0 && isfinite(w) && isfinite(h)) hdr->step_hint = (float)sqrt((w > 0 ? w : c) * (h > 0 ? h : c) / (double)hdr->n);
}

// ---- The cell arrays are allocated for the host-known capacity `cap` (+ 1), but the grid the device sized may be
//      far smaller (a caller's cell size asks for up to 4 cells per sounding of CAPACITY).  Only entries
//      [0, ncx*ncy] are ever read -- by the kernels below and by krige_predict -- so the per-append sweeps (zeroing,
//      scan, add-back) stop there: an append costs O(batch + cells in use + soundings held), not O(capacity).
__device__ __forceinline__ int64_t cells_in_use(const IndexHeader* __restrict__ hdr, int64_t cap)
{
    const int64_t m = (int64_t)hdr->ncx * hdr->ncy + 1;      // entry ncx*ncy holds the total
    return m < cap ? m : cap;
}

__global__ void __launch_bounds__(kThreads)
zero_counts_kernel(int32_t* __restrict__ count, int64_t cap, const IndexHeader* __restrict__ hdr)
{
    const int64_t n = cells_in_use(hdr, cap);
    for (int64_t i = (int64_t)blockIdx.x * kThreads + threadIdx.x; i < n; i += (int64_t)gridDim.x * kThreads) count[i] = 0;
}

// ---- histogram of the new soundings per cell
__global__ void __launch_bounds__(kThreads)
cell_count_kernel(const float* __restrict__ x, const float* __restrict__ y, int64_t n,
                  const IndexHeader* __restrict__ hdr, int32_t* __restrict__ count)
{
    const float xmin = hdr->xmin, ymin = hdr->ymin, inv_cell = hdr->inv_cell;
    const int ncx = hdr->ncx, ncy = hdr->ncy;
    for (int64_t i = (int64_t)blockIdx.x * kThreads + threadIdx.x; i < n; i += (int64_t)gridDim.x * kThreads) {
        const int c = cell_of(y[i], ymin, inv_cell, ncy) * ncx + cell_of(x[i], xmin, inv_cell, ncx);
        atomicAdd(count + c, 1);
    }
}

// ---- exclusive scan of int32 counts: per-block scan + block sums, scan of sums, add back
constexpr int kScanItems = 8;
constexpr int kScanBlock = kThreads * kScanItems;

__global__ void __launch_bounds__(kThreads)
scan_block_kernel(const int32_t* __restrict__ in, int32_t* __restrict__ out, int64_t cap, const IndexHeader* __restrict__ hdr,
                  int32_t* __restrict__ sums)
{
    __shared__ int32_t s_warp[kThreads / 32];
    const int64_t n = cells_in_use(hdr, cap);
    if ((int64_t)blockIdx.x * kScanBlock >= n) {             // beyond the grid in use: nothing to scan, a zero block sum
        if (threadIdx.x == 0) sums[blockIdx.x] = 0;
        return;
    }
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

// prefix[c] += block offset (the exclusive prefix of the NEW soundings per cell, prefix[cap] = total),
// cursor[c] = prefix[c] (where the scatter puts the next sounding of cell c; overwrites the counts), and
// start_new[c] = start_old[c] + prefix[c] (start_old == NULL: an empty index)
__global__ void __launch_bounds__(kThreads)
scan_add_kernel(int32_t* __restrict__ prefix, int64_t cap, const IndexHeader* __restrict__ hdr, const int32_t* __restrict__ sums,
                int32_t total, const int32_t* __restrict__ start_old, int32_t* __restrict__ start_new, int32_t* __restrict__ cursor)
{
    const int64_t n = cells_in_use(hdr, cap);
    const int64_t base = (int64_t)blockIdx.x * kScanBlock;
    if (blockIdx.x == 0 && threadIdx.x == 0) {
        prefix[cap] = total;
        start_new[cap] = total + (start_old ? start_old[cap] : 0);
    }
    if (base >= n) return;
    const int32_t off = sums[blockIdx.x];
    for (int e = threadIdx.x; e < kScanBlock; e += kThreads)
        if (base + e < n) {
            const int32_t v = prefix[base + e] + off;
            prefix[base + e] = v;
            cursor[base + e] = v;
            start_new[base + e] = v + (start_old ? start_old[base + e] : 0);
        }
}

// ---- the soundings already in the index move right by the number of new soundings in the cells before theirs
__global__ void __launch_bounds__(kThreads)
shift_old_kernel(const float4* __restrict__ src, int64_t n_old, const IndexHeader* __restrict__ hdr,
                 const int32_t* __restrict__ prefix, float4* __restrict__ dst)
{
    const float xmin = hdr->xmin, ymin = hdr->ymin, inv_cell = hdr->inv_cell;
    const int ncx = hdr->ncx, ncy = hdr->ncy;
    for (int64_t p = (int64_t)blockIdx.x * kThreads + threadIdx.x; p < n_old; p += (int64_t)gridDim.x * kThreads) {
        const float4 me = src[p];
        const int c = cell_of(me.y, ymin, inv_cell, ncy) * ncx + cell_of(me.x, xmin, inv_cell, ncx);
        dst[p + prefix[c]] = me;
    }
}

// ---- the new soundings: scatter by cell into a scratch array (atomic cursor), then place every one behind
//      the old soundings of its cell, ordered by original index, so that the index -- and with it every
//      later result -- does not depend on atomic arrival order
__global__ void __launch_bounds__(kThreads)
scatter_kernel(const float* __restrict__ x, const float* __restrict__ y, const float* __restrict__ z, int64_t n,
               int32_t first_index, const IndexHeader* __restrict__ hdr, int32_t* __restrict__ cursor, float4* __restrict__ tmp)
{
    const float xmin = hdr->xmin, ymin = hdr->ymin, inv_cell = hdr->inv_cell;
    const int ncx = hdr->ncx, ncy = hdr->ncy;
    for (int64_t i = (int64_t)blockIdx.x * kThreads + threadIdx.x; i < n; i += (int64_t)gridDim.x * kThreads) {
        const float a = x[i], b = y[i];
        const int c = cell_of(b, ymin, inv_cell, ncy) * ncx + cell_of(a, xmin, inv_cell, ncx);
        const int32_t p = atomicAdd(cursor + c, 1);
        tmp[p] = make_float4(a, b, z[i], __int_as_float(first_index + (int32_t)i));
    }
}

__global__ void __launch_bounds__(kThreads)
order_cells_kernel(const float4* __restrict__ tmp, int64_t n, const IndexHeader* __restrict__ hdr,
                   const int32_t* __restrict__ prefix, const int32_t* __restrict__ start_new, float4* __restrict__ pts)
{
    const float xmin = hdr->xmin, ymin = hdr->ymin, inv_cell = hdr->inv_cell;
    const int ncx = hdr->ncx, ncy = hdr->ncy;
    for (int64_t p = (int64_t)blockIdx.x * kThreads + threadIdx.x; p < n; p += (int64_t)gridDim.x * kThreads) {
        const float4 me = tmp[p];
        const int c = cell_of(me.y, ymin, inv_cell, ncy) * ncx + cell_of(me.x, xmin, inv_cell, ncx);
        const int32_t s = prefix[c], e = prefix[c + 1];
        const int32_t my = __float_as_int(me.w);
        int32_t rank = 0;
        for (int32_t q = s; q < e; ++q) rank += (__float_as_int(tmp[q].w) < my);
        // the cell's new segment ends where the next cell starts: old soundings first, then the new ones
        pts[start_new[c + 1] - (e - s) + rank] = me;
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
// pointer bump after the first call.  Once per device (bathy.h documents the side effect).
void pool_keep_warm()
{
    static std::atomic<uint64_t> done{0};
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= 64) return;
    if (done.load(std::memory_order_acquire) & (1ull << dev)) return;
    cudaMemPool_t pool;
    if (cudaDeviceGetDefaultMemPool(&pool, dev) == cudaSuccess) {
        unsigned long long keep = 1ull << 31;              // hold up to 2 GiB of freed blocks
        cudaMemPoolSetAttribute(pool, cudaMemPoolAttrReleaseThreshold, &keep);
    }
    done.fetch_or(1ull << dev, std::memory_order_release);
}

namespace {

// stream-ordered scratch that is released on every path out of a function
struct Scratch {
    cudaStream_t s;
    void* p[8];
    int n = 0;
    explicit Scratch(cudaStream_t st) : s(st) {}
    template <class T> bool get(T** out, size_t count)
    {
        void* q = nullptr;
        if (n >= 8 || cudaMallocAsync(&q, sizeof(T) * (count ? count : 1), s) != cudaSuccess) { cudaGetLastError(); return false; }
        p[n++] = q;
        *out = static_cast<T*>(q);
        return true;
    }
    ~Scratch() { for (int i = 0; i < n; ++i) cudaFreeAsync(p[i], s); }
};

void release_index_memory(krige_index* idx, cudaStream_t stream)
{
    if (idx->d_pts) cudaFreeAsync(idx->d_pts, stream);
    if (idx->d_pts_alt) cudaFreeAsync(idx->d_pts_alt, stream);
    if (idx->d_cell_start) cudaFreeAsync(idx->d_cell_start, stream);
    if (idx->d_cell_start_alt) cudaFreeAsync(idx->d_cell_start_alt, stream);
    if (idx->d_hdr) cudaFreeAsync(idx->d_hdr, stream);
    idx->magic = 0;
    delete idx;
}

// Allocates an index with room for `capacity` soundings and `cells_cap` cells (appendable: with the
// second set of buffers an append writes into).
int alloc_index(int64_t capacity, int64_t cells_cap, bool appendable, cudaStream_t stream, krige_index** out)
{
    pool_keep_warm();
    krige_index* idx = new (std::nothrow) krige_index();
    if (!idx) return BATHY_ERR_CUDA;
    memset(idx, 0, sizeof(*idx));
    idx->capacity = capacity; idx->cells_cap = cells_cap; idx->stream = stream;
    cudaGetDevice(&idx->device);
    cudaError_t e = cudaMallocAsync(&idx->d_pts, sizeof(float4) * (size_t)capacity, stream);
    if (e == cudaSuccess) e = cudaMallocAsync(&idx->d_cell_start, sizeof(int32_t) * (size_t)(cells_cap + 1), stream);
    if (e == cudaSuccess && appendable) e = cudaMallocAsync(&idx->d_pts_alt, sizeof(float4) * (size_t)capacity, stream);
    if (e == cudaSuccess && appendable) e = cudaMallocAsync(&idx->d_cell_start_alt, sizeof(int32_t) * (size_t)(cells_cap + 1), stream);
    if (e == cudaSuccess) e = cudaMallocAsync(&idx->d_hdr, sizeof(IndexHeader), stream);
    if (e == cudaSuccess) e = cudaMemsetAsync(idx->d_cell_start, 0, sizeof(int32_t) * (size_t)(cells_cap + 1), stream);
    if (e != cudaSuccess) {
        cudaGetLastError();
        release_index_memory(idx, stream);
        return BATHY_ERR_CUDA;
    }
    *out = idx;
    return BATHY_OK;
}

// Merges n_new soundings into the index (whose device header is already sized).  size_first: the cell
// grid is sized from the batch's own bounding box first (krige_build_index).
int merge_soundings(krige_index* idx, const float* d_x, const float* d_y, const float* d_z, int64_t n_new,
                    bool size_first, float cell_size, float* d_changed, cudaStream_t stream)
{
    const int64_t n_old = idx->n, cells = idx->cells_cap;
    const bool pingpong = idx->d_pts_alt != nullptr;
    const int nb = grid_for(n_new);
    const int nsb = (int)((cells + kScanBlock - 1) / kScanBlock);
    Scratch sc(stream);
    float4* d_bb = nullptr; float4* d_tmp = nullptr;
    int32_t *d_count = nullptr, *d_prefix = nullptr, *d_sums = nullptr;
    if (!sc.get(&d_bb, (size_t)nb + 1) || !sc.get(&d_tmp, (size_t)n_new) || !sc.get(&d_count, (size_t)cells + 1) ||
        !sc.get(&d_prefix, (size_t)cells + 1) || !sc.get(&d_sums, (size_t)nsb + 1))
        return BATHY_ERR_CUDA;
    float4* pts_dst = pingpong ? idx->d_pts_alt : idx->d_pts;
    int32_t* start_dst = pingpong ? idx->d_cell_start_alt : idx->d_cell_start;
    const int32_t* start_old = pingpong ? idx->d_cell_start : nullptr;   // (a one-shot build starts from an empty index)

    bbox_partial_kernel<<<nb, kThreads, 0, stream>>>(d_x, d_y, n_new, d_bb);
    bbox_final_kernel<<<1, 32, 0, stream>>>(d_bb, nb, d_bb + nb);
    if (size_first)
        size_grid_kernel<<<1, 32, 0, stream>>>(d_bb + nb, make_float4(0, 0, 0, 0), 0, (long long)n_new, cell_size, (long long)cells, idx->d_hdr);
    zero_counts_kernel<<<grid_for(cells + 1), kThreads, 0, stream>>>(d_count, cells + 1, idx->d_hdr);
    cell_count_kernel<<<nb, kThreads, 0, stream>>>(d_x, d_y, n_new, idx->d_hdr, d_count);
    scan_block_kernel<<<nsb, kThreads, 0, stream>>>(d_count, d_prefix, cells, idx->d_hdr, d_sums);
    scan_sums_kernel<<<1, kThreads, 0, stream>>>(d_sums, nsb);
    scan_add_kernel<<<nsb, kThreads, 0, stream>>>(d_prefix, cells, idx->d_hdr, d_sums, (int32_t)n_new, start_old, start_dst, d_count);
    int launches = 10 + (size_first ? 1 : 0);   // bbox x2, zero, count, scan x3, scatter, order, header update
    if (n_old > 0) {
        shift_old_kernel<<<grid_for(n_old), kThreads, 0, stream>>>(idx->d_pts, n_old, idx->d_hdr, d_prefix, pts_dst);
        ++launches;
    }
    scatter_kernel<<<nb, kThreads, 0, stream>>>(d_x, d_y, d_z, n_new, (int32_t)n_old, idx->d_hdr, d_count, d_tmp);
    order_cells_kernel<<<nb, kThreads, 0, stream>>>(d_tmp, n_new, idx->d_hdr, d_prefix, start_dst, pts_dst);
    header_update_kernel<<<1, 32, 0, stream>>>(idx->d_hdr, d_bb + nb, (int)n_new, d_changed);
    count_launch(launches);
    const int st = launch_status();
    if (st != BATHY_OK) return st;
    if (pingpong) {
        float4* t = idx->d_pts; idx->d_pts = idx->d_pts_alt; idx->d_pts_alt = t;
        int32_t* u = idx->d_cell_start; idx->d_cell_start = idx->d_cell_start_alt; idx->d_cell_start_alt = u;
    }
    idx->n = n_old + n_new;
    if (stream != idx->stream) __atomic_store_n(&idx->used_elsewhere, 1, __ATOMIC_RELEASE);   // earlier work stays on the old stream
    idx->stream = stream;
    return BATHY_OK;
}

}  // namespace

// krige_build_index: one-shot index over the bounding box of the soundings; the cell grid is sized on the
// device (about 8 soundings per cell, or the caller's cell size, enlarged until the grid fits the
// host-known cell capacity).  Enqueue only.
int build_index(const float* d_x, const float* d_y, const float* d_z, int64_t n, float cell_size,
                cudaStream_t stream, krige_index** out_index)
{
    *out_index = nullptr;
    // automatic: n/8 cells plus the perimeter terms; a caller's cell size may ask for up to 4 cells per sounding
    int64_t cells_cap = (cell_size > 0.0f) ? 4 * n + 4096 : n / 4 + 4096;
    if (cells_cap > (int64_t)1 << 26) cells_cap = (int64_t)1 << 26;
    krige_index* idx = nullptr;
    int rc = alloc_index(n, cells_cap, false, stream, &idx);
    if (rc) return rc;
    rc = merge_soundings(idx, d_x, d_y, d_z, n, true, cell_size, nullptr, stream);
    if (rc) { release_index_memory(idx, stream); return rc; }
    idx->magic = kIndexMagic;
    *out_index = idx;
    return BATHY_OK;
}

// krige_index_create: an empty, appendable index over the caller's extent (the planned survey area).
int create_index(float xmin, float xmax, float ymin, float ymax, float cell_size, int64_t capacity,
                 cudaStream_t stream, krige_index** out_index)
{
    *out_index = nullptr;
    int64_t cells_cap = (cell_size > 0.0f) ? 4 * capacity + 4096 : capacity / 4 + 4096;
    if (cells_cap > (int64_t)1 << 26) cells_cap = (int64_t)1 << 26;
    krige_index* idx = nullptr;
    int rc = alloc_index(capacity, cells_cap, true, stream, &idx);
    if (rc) return rc;
    cudaError_t e = cudaMemsetAsync(idx->d_cell_start_alt, 0, sizeof(int32_t) * (size_t)(cells_cap + 1), stream);
    size_grid_kernel<<<1, 32, 0, stream>>>(nullptr, make_float4(xmin, xmax, ymin, ymax), 1, (long long)capacity, cell_size,
                                           (long long)cells_cap, idx->d_hdr);
    count_launch();
    if (e != cudaSuccess || launch_status() != BATHY_OK) { cudaGetLastError(); release_index_memory(idx, stream); return BATHY_ERR_CUDA; }
    idx->magic = kIndexMagic;
    *out_index = idx;
    return BATHY_OK;
}

int append_index(krige_index* idx, const float* d_x, const float* d_y, const float* d_z, int64_t n,
                 float* d_changed, cudaStream_t stream)
{
    if (!idx->d_pts_alt) return BATHY_ERR_INDEX;           // built by krige_build_index: not appendable
    if (!index_on_current_device(idx)) return BATHY_ERR_INDEX;
    if (idx->n + n > idx->capacity) return BATHY_ERR_SIZE;
    return merge_soundings(idx, d_x, d_y, d_z, n, false, 0.0f, d_changed, stream);
}

// Host copy of the header: waits for the stream of the last build / append (the only index call that
// synchronises the host, besides krige_free_index).
int index_header(const krige_index* idx, IndexHeader* out)
{
    if (!index_on_current_device(idx)) return BATHY_ERR_INDEX;
    if (cudaMemcpyAsync(out, idx->d_hdr, sizeof(IndexHeader), cudaMemcpyDeviceToHost, idx->stream) != cudaSuccess ||
        cudaStreamSynchronize(idx->stream) != cudaSuccess) { cudaGetLastError(); return BATHY_ERR_CUDA; }
    return BATHY_OK;
}

void free_index(krige_index* idx)
{
    if (!idx || idx->magic != kIndexMagic) return;
    int cur = 0;
    cudaGetDevice(&cur);
    if (cur != idx->device) cudaSetDevice(idx->device);
    // Every kernel that reads the index must have finished before its memory returns to the pool.  When all of them
    // were issued on the stream of the last build / append, waiting for that stream is enough; once a krige_predict
    // (or an earlier append) went to another stream, only the device-wide wait is safe.
    if (__atomic_load_n(&idx->used_elsewhere, __ATOMIC_ACQUIRE)) cudaDeviceSynchronize();
    else cudaStreamSynchronize(idx->stream);
    cudaGetLastError();
    release_index_memory(idx, idx->stream);
    if (cur != idx->device) cudaSetDevice(cur);
}

// Stream-ordered release: the memory goes back to the pool when `stream` reaches this point; no host
// synchronisation.
void free_index_async(krige_index* idx, cudaStream_t stream)
{
    if (!idx || idx->magic != kIndexMagic) return;
    release_index_memory(idx, stream);
}

}  // namespace bathy
