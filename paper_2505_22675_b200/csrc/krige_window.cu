// krige_window.cu -- interp_krige_window: the holes (NaN cells) of a regular grid are
// filled by ordinary kriging from the valid cells of a (2 half + 1)^2 window -- the form of kriging the paper
// measured: "the implementation in this study uses a 5x5 grid", with its helper that finds "the
// nearest n valid candidate neighbors" (L179) and its fallback to bilinear "if enough valid candidate neighbors
// are not found" (L171, L180) -- the Grid B workload, cells removed at random (L225-L234).  Readings W1-W4 of
// DESIGN.md.  Two kernels: a scan copies the valid cells and lists the holes; a persistent kernel then takes
// 32/G holes per warp at a time, G lanes per hole: gathers the window's valid cells (in window order) into the
// shared-memory neighbour lists of krige_solve.cuh, keeps the n_max nearest by the defined fp32 key, and runs the
// same covariance build + Cholesky + Schur step as krige_predict (solve_batch).
#include "krige_solve.cuh"

namespace bathy {

namespace {

struct WindowParams : SolveParams {
    const float* in;
    uint8_t* how;
    int nx, ny;
    float dx, dy;
    int half, n_max, n_min;
    const int32_t* holes;       // linear indices of the NaN cells (any order)
    const int32_t* n_holes;
};

constexpr int kScanThreads = 256;

__global__ void __launch_bounds__(kScanThreads)
window_scan_kernel(const float* __restrict__ in, float* __restrict__ out, uint8_t* __restrict__ how, long long n,
                   int32_t* __restrict__ holes, int32_t* __restrict__ counter)
{
    const int lane = threadIdx.x & 31;
    for (long long base = (long long)blockIdx.x * kScanThreads; base < n; base += (long long)gridDim.x * kScanThreads) {
        const long long i = base + threadIdx.x;
        float v = 0.0f;
        bool hole = false;
        if (i < n) {
            v = in[i];
            hole = v != v;
            if (!hole) { out[i] = v; if (how) how[i] = (uint8_t)0; }
        }
        const unsigned m = __ballot_sync(kFull, hole);     // one atomic per warp
        if (m) {
            int32_t first = 0;
            if (lane == __ffs(m) - 1) first = atomicAdd(counter, __popc(m));
            first = __shfl_sync(kFull, first, __ffs(m) - 1);
            if (hole) holes[first + __popc(m & ((1u << lane) - 1u))] = (int32_t)i;
        }
    }
}

template <int K, int G>
struct __align__(16) WindowSmem : SolveSmem<K, G> {
    float key[Shape<K, G>::NB][K];              // selection keys of the gathered candidates (reading W2)
};

template <int K, int G, int MODEL>
__global__ void __launch_bounds__(Shape<K, G>::WARPS * 32, Shape<K, G>::CTAS)
krige_window_kernel(const WindowParams p)
{
    using S = Shape<K, G>;
    extern __shared__ __align__(16) unsigned char s_raw[];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    WindowSmem<K, G>& ws = reinterpret_cast<WindowSmem<K, G>*>(s_raw)[warp];
    const int nd = S::ILV ? lane % S::NB : lane / G, g = S::ILV ? lane / S::NB : lane % G;
    // the lanes that work on the same hole as this one, and those of them below this lane
    unsigned groupmask = 0;
#pragma unroll
    for (int l = 0; l < 32; ++l) groupmask |= ((S::ILV ? l % S::NB : l / G) == nd) ? (1u << l) : 0u;
    const unsigned below = groupmask & ((1u << lane) - 1u);
    const int n_holes = *p.n_holes;
    const int side = 2 * p.half + 1, wn = side * side;
    const float sc = p.s_coord;
    const float padbase = 4.0f * (float)p.half * (p.dx + p.dy) * sc + 300.0f;
    const float qnan = __int_as_float(0x7fc00000);
    constexpr int SLOTS = (K + G - 1) / G;                 // candidates a lane handles at most

#pragma unroll 1
    for (long long batch = (long long)blockIdx.x * S::WARPS + warp; batch * S::NB < n_holes; batch += (long long)gridDim.x * S::WARPS) {
        const long long h = batch * S::NB + nd;
        const bool live = h < n_holes;
        const int cell = live ? p.holes[h] : 0;
        const int i = cell / p.nx, j = cell - i * p.nx;
        // W1: the valid cells of the clipped window, in window (row-major) order
        int cnt = 0;
        for (int e0 = 0; e0 < wn; e0 += G) {
            const int e = e0 + g;
            const int a = e / side - p.half, b = e - (e / side) * side - p.half;
            const int ii = i + a, jj = j + b;
            float v = qnan;
            if (live && e < wn && !(a == 0 && b == 0) && ii >= 0 && ii < p.ny && jj >= 0 && jj < p.nx)
                v = __ldg(p.in + (size_t)ii * p.nx + jj);
            const bool ok = v == v;
            const unsigned m = __ballot_sync(kFull, ok);
            const int slot = cnt + __popc(m & below);
            if (ok) {                                       // (slot < K: the window has at most K cells besides the hole)
                const float ddx = __fmul_rn((float)b, p.dx), ddy = __fmul_rn((float)a, p.dy);
                ws.nb_x[nd][slot] = __fmul_rn(ddx, sc);
                ws.nb_y[nd][slot] = __fmul_rn(ddy, sc);
                ws.nb_z[nd][slot] = v;
                ws.key[nd][slot] = __fmaf_rn(ddx, ddx, __fmul_rn(ddy, ddy));
            }
            cnt += __popc(m & groupmask);
        }
        __syncwarp();
        int k = cnt;
        if (__any_sync(kFull, cnt > p.n_max)) {
            // W2: keep the n_max nearest by (key, window order), in window order
            float kx[SLOTS], ky[SLOTS], kz[SLOTS];
            bool keep[SLOTS];
#pragma unroll
            for (int q = 0; q < SLOTS; ++q) {
                const int s = q * G + g;
                keep[q] = false;
                kx[q] = ky[q] = kz[q] = 0.0f;
                if (s < cnt) {
                    const float ks = ws.key[nd][s];
                    int rank = 0;
                    for (int f = 0; f < cnt; ++f) {
                        const float kf = ws.key[nd][f];
                        rank += (kf < ks || (kf == ks && f < s)) ? 1 : 0;
                    }
                    keep[q] = rank < p.n_max;
                    kx[q] = ws.nb_x[nd][s]; ky[q] = ws.nb_y[nd][s]; kz[q] = ws.nb_z[nd][s];
                }
            }
            __syncwarp();
            int c2 = 0;
#pragma unroll
            for (int q = 0; q < SLOTS; ++q) {
                const unsigned m = __ballot_sync(kFull, keep[q]);
                const int slot = c2 + __popc(m & below);
                if (keep[q]) { ws.nb_x[nd][slot] = kx[q]; ws.nb_y[nd][slot] = ky[q]; ws.nb_z[nd][slot] = kz[q]; }
                c2 += __popc(m & groupmask);
            }
            k = c2;
            __syncwarp();
        }
        const bool kriged = live && k >= p.n_min;
        if (live && !kriged && g == 0) {
            // W3 + W4: bilinear on the rectangle of the diagonal neighbours, t = s = 1/2
            float f = qnan;
            if (i - 1 >= 0 && i + 1 < p.ny && j - 1 >= 0 && j + 1 < p.nx) {
                const float q11 = __ldg(p.in + (size_t)(i - 1) * p.nx + j - 1), q21 = __ldg(p.in + (size_t)(i - 1) * p.nx + j + 1);
                const float q12 = __ldg(p.in + (size_t)(i + 1) * p.nx + j - 1), q22 = __ldg(p.in + (size_t)(i + 1) * p.nx + j + 1);
                const float a = q21 - q11, b = q12 - q11, c = q22 - q11;       // on differences: one rounding at full magnitude
                f = q11 + 0.25f * ((a + b) + c);
            }
            p.zhat[cell] = f;
            if (p.how) p.how[cell] = (uint8_t)255;
        }
        if (kriged && g == 0 && p.how) p.how[cell] = (uint8_t)k;
        // rows at and beyond k: pad soundings far away from everything (they decouple as identity rows)
        const float z0 = (k > 0) ? ws.nb_z[nd][0] : 0.0f;
        __syncwarp();
        for (int s = g; s < K; s += G)
            if (s >= k) { ws.nb_x[nd][s] = padbase + 300.0f * (float)s; ws.nb_y[nd][s] = 0.0f; ws.nb_z[nd][s] = z0; }
        __syncwarp();
        if (__any_sync(kFull, kriged))
            solve_batch<K, G, MODEL, false>(p, ws, lane, 0.0f, 0.0f, kriged, (long long)cell, k);
        __syncwarp();
    }
}

template <int K, int G, int MODEL>
int launch_window_one(const WindowParams& p, cudaStream_t stream)
{
    const size_t smem = sizeof(WindowSmem<K, G>) * Shape<K, G>::WARPS;
    static DeviceOnce once;
    const int rc = once_per_device(once, [smem]() -> int {
        BATHY_CUDA_TRY(cudaFuncSetAttribute(krige_window_kernel<K, G, MODEL>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        return (int)BATHY_OK;
    });
    if (rc) return rc;
    int dev = 0, sms = kSMs;
    BATHY_CUDA_TRY(cudaGetDevice(&dev));
    BATHY_CUDA_TRY(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
    krige_window_kernel<K, G, MODEL><<<sms * Shape<K, G>::CTAS, Shape<K, G>::WARPS * 32, smem, stream>>>(p);   // persistent: the CTAs one SM holds
    count_launch();
    return launch_status();
}

template <int K, int G>
int launch_window_shape(const WindowParams& p, int model, cudaStream_t stream)
{
    if (model == BATHY_VGM_EXPONENTIAL) return launch_window_one<K, G, BATHY_VGM_EXPONENTIAL>(p, stream);
    if (model == BATHY_VGM_SPHERICAL) return launch_window_one<K, G, BATHY_VGM_SPHERICAL>(p, stream);
    return launch_window_one<K, G, BATHY_VGM_GAUSSIAN>(p, stream);
}

}  // namespace

int launch_krige_window(const float* d_in, const grid_geom_t& g, int half, int n_max, int n_min, const variogram_t& vg,
                        float* d_out, uint8_t* d_how, int64_t* d_failed, cudaStream_t stream)
{
    const long long n = (long long)g.nx * g.ny;
    if (n > 0x7fffffffLL) return BATHY_ERR_SIZE;
    int32_t* d_holes = nullptr;                            // [n] hole list + [1] counter, stream-ordered scratch
    if (cudaMallocAsync(&d_holes, sizeof(int32_t) * (size_t)(n + 1), stream) != cudaSuccess) { cudaGetLastError(); return BATHY_ERR_CUDA; }
    int32_t* d_count = d_holes + n;
    int rc = BATHY_OK;
    if (cudaMemsetAsync(d_count, 0, sizeof(int32_t), stream) != cudaSuccess) { cudaGetLastError(); rc = BATHY_ERR_CUDA; }
    if (rc == BATHY_OK) {
        const long long blocks = (n + kScanThreads - 1) / kScanThreads;
        const int grid = (int)(blocks < (long long)kSMs * 16 ? blocks : (long long)kSMs * 16);
        window_scan_kernel<<<grid, kScanThreads, 0, stream>>>(d_in, d_out, d_how, n, d_holes, d_count);
        count_launch();
        rc = launch_status();
    }
    if (rc == BATHY_OK) {
        WindowParams p;
        set_variogram(p, vg);
        p.zhat = d_out; p.var = nullptr; p.failed = reinterpret_cast<unsigned long long*>(d_failed); p.illcond = nullptr;
        p.in = d_in; p.how = d_how; p.nx = g.nx; p.ny = g.ny; p.dx = g.dx; p.dy = g.dy;
        const int wn = (2 * half + 1) * (2 * half + 1) - 1;
        p.half = half; p.n_max = n_max < wn ? n_max : wn; p.n_min = n_min;
        p.holes = d_holes; p.n_holes = d_count;
        if (half == 1)      rc = launch_window_shape<8, 8>(p, vg.model, stream);
        else if (half == 2) rc = launch_window_shape<24, 8>(p, vg.model, stream);
        else                rc = launch_window_shape<48, 16>(p, vg.model, stream);
    }
    cudaFreeAsync(d_holes, stream);
    return rc;
}

// ---------------------------------------------------------------------------------------------------------------
// interp_krige_window_noalloc: the same two kernels, with the hole list and its counter in a fixed device array
// that is part of the library image instead of memory taken from the stream's pool.
//
// Who needs this.  On the vehicle the mapping loop runs with a device-memory budget that was handed out in full
// at start-up: every buffer is allocated before the dive, and a call that asks the driver for more in the middle
// of a survey line can fail (nothing left), can stall (cudaMalloc / cudaFree wait for the whole device), or can
// make the pool grow and trim at the caller's synchronisation points -- none of which a ping-rate loop can
// afford.  The same holds for a host application whose own allocator has reserved the GPU (a driver allocation
// made behind its back competes with it), and for devices or driver set-ups without stream-ordered memory pools,
// where interp_krige_window's cudaMallocAsync simply returns an error.  Those callers pass their input and output
// buffers as always and the library brings the scratch itself.
//
// The price: kNoAllocMaxCells * 4 bytes + 256 bytes (16 MiB) of device memory on EVERY GPU whose context loads
// this library, from the moment the module is loaded until the process exits, whether or not the call is used;
// and one array per device, shared by all calls -- see the race note at launch_krige_window_noalloc.
constexpr long long kNoAllocMaxCells = BATHY_NOALLOC_MAX_CELLS;
static_assert((kNoAllocMaxCells * (long long)sizeof(int32_t)) % 256 == 0, "the counter sits on a 256-byte boundary behind the list");
// [kNoAllocMaxCells] hole list, then one 256-byte line whose first word is the hole counter.
static __device__ __align__(256) int32_t g_window_scratch[kNoAllocMaxCells + 64];

// The DEVICE address of g_window_scratch on the current device.  In host code the name `g_window_scratch` is only
// the host-side handle of the symbol -- handing it to a kernel or to cudaMemsetAsync would pass a host address --
// so the address is asked for once per device (with that device current) and remembered.  Devices numbered 64 and
// above are served too, without the cache.
static int window_scratch_address(int32_t** out)
{
    static std::atomic<int32_t*> cached[64];
    int dev = 0;
    BATHY_CUDA_TRY(cudaGetDevice(&dev));
    if (dev >= 0 && dev < 64) {
        int32_t* p = cached[dev].load(std::memory_order_acquire);
        if (p) { *out = p; return BATHY_OK; }
    }
    int32_t* p = nullptr;
    BATHY_CUDA_TRY(cudaGetSymbolAddress(reinterpret_cast<void**>(&p), g_window_scratch));
    if (!p) return BATHY_ERR_CUDA;
    if (dev >= 0 && dev < 64) cached[dev].store(p, std::memory_order_release);   // (a racing first call stores the same address)
    *out = p;
    return BATHY_OK;
}

// Calls no cudaMalloc*, cudaFree* or allocating library routine: cudaGetDevice, cudaGetSymbolAddress (first call
// on a device), one 4-byte cudaMemsetAsync, cudaFuncSetAttribute (first call per window size and device) and two
// kernel launches.  The hole list keeps whatever the previous call left in it; only the counter has to start at
// zero, and the scan writes every list entry the solve kernel reads.  All calls on one device use the one array:
// two calls whose work overlaps on the GPU (different streams without an event between them, or two host threads)
// corrupt each other's hole list.
int launch_krige_window_noalloc(const float* d_in, const grid_geom_t& g, int half, int n_max, int n_min, const variogram_t& vg,
                                float* d_out, uint8_t* d_how, int64_t* d_failed, cudaStream_t stream)
{
    const long long n = (long long)g.nx * g.ny;
    if (n > kNoAllocMaxCells) return BATHY_ERR_SCRATCH;
    int32_t* d_holes = nullptr;
    int rc = window_scratch_address(&d_holes);
    if (rc) return rc;
    int32_t* d_count = d_holes + kNoAllocMaxCells;
    BATHY_CUDA_TRY(cudaMemsetAsync(d_count, 0, sizeof(int32_t), stream));
    const long long blocks = (n + kScanThreads - 1) / kScanThreads;
    const int grid = (int)(blocks < (long long)kSMs * 16 ? blocks : (long long)kSMs * 16);
    window_scan_kernel<<<grid, kScanThreads, 0, stream>>>(d_in, d_out, d_how, n, d_holes, d_count);
    count_launch();
    rc = launch_status();
    if (rc) return rc;
    WindowParams p;
    set_variogram(p, vg);
    p.zhat = d_out; p.var = nullptr; p.failed = reinterpret_cast<unsigned long long*>(d_failed); p.illcond = nullptr;
    p.in = d_in; p.how = d_how; p.nx = g.nx; p.ny = g.ny; p.dx = g.dx; p.dy = g.dy;
    const int wn = (2 * half + 1) * (2 * half + 1) - 1;
    p.half = half; p.n_max = n_max < wn ? n_max : wn; p.n_min = n_min;
    p.holes = d_holes; p.n_holes = d_count;
    if (half == 1) return launch_window_shape<8, 8>(p, vg.model, stream);
    if (half == 2) return launch_window_shape<24, 8>(p, vg.model, stream);
    return launch_window_shape<48, 16>(p, vg.model, stream);
}

}  // namespace bathy
