// api.cu -- the extern "C" boundary of libbathy.so (include/bathy.h): argument checks, host-buffer
// forms, error strings.  Every step of the path runs in the kernels of the other .cu files.
#include "krige_index.cuh"
#include <atomic>

namespace bathy {

int launch_bilinear(const float*, const grid_geom_t&, float*, const grid_geom_t&, cudaStream_t);
int launch_catmull_rom(const float*, const grid_geom_t&, float*, const grid_geom_t&, cudaStream_t);
size_t spline_workspace_bytes(const grid_geom_t&, const grid_geom_t&);
int launch_spline(const float*, const grid_geom_t&, float*, const grid_geom_t&, void*, cudaStream_t, int path);
int build_index(const float*, const float*, const float*, int64_t, float, cudaStream_t, krige_index**);
int create_index(float, float, float, float, float, int64_t, cudaStream_t, krige_index**);
int append_index(krige_index*, const float*, const float*, const float*, int64_t, float*, cudaStream_t);
int index_header(const krige_index*, IndexHeader*);
void free_index(krige_index*);
void free_index_async(krige_index*, cudaStream_t);
int launch_predict(const krige_index*, const grid_geom_t&, const variogram_t&, int, float*, float*, int32_t*, int64_t*,
                   int64_t*, cudaStream_t, const krige_aniso_t* aniso_or_null);

int launch_krige_window(const float*, const grid_geom_t&, int, int, int, const variogram_t&, float*, uint8_t*, int64_t*,
                        cudaStream_t);
int launch_krige_window_noalloc(const float*, const grid_geom_t&, int, int, int, const variogram_t&, float*, uint8_t*, int64_t*,
                                cudaStream_t);

void pool_keep_warm();           // krige_index.cu: raises the release threshold of the device's default memory pool, once per device

extern std::atomic<bool> g_bilinear_tma;
static std::atomic<int64_t> g_launches{0};
static std::atomic<int> g_spline_path{0};
void count_launch(int n) { g_launches.fetch_add(n, std::memory_order_relaxed); }

static int check_variogram(const variogram_t& v)
{
    if (v.model != BATHY_VGM_EXPONENTIAL && v.model != BATHY_VGM_SPHERICAL && v.model != BATHY_VGM_GAUSSIAN) return BATHY_ERR_VARIOGRAM;
    if (!isfinite(v.range) || !isfinite(v.sill) || !isfinite(v.nugget)) return BATHY_ERR_VARIOGRAM;
    if (!(v.range > 0.0f) || !(v.sill > 0.0f) || v.nugget < 0.0f || v.nugget > v.sill) return BATHY_ERR_VARIOGRAM;
    return BATHY_OK;
}

// RAII device scratch for the host-buffer forms
struct DevBuf {
    void* p = nullptr;
    cudaStream_t s;
    explicit DevBuf(cudaStream_t st) : s(st) { pool_keep_warm(); }   // a grid-only caller gets a warm pool too, not a cold one at every synchronisation
    int alloc(size_t bytes) { return cudaMallocAsync(&p, bytes ? bytes : 1, s) == cudaSuccess ? BATHY_OK : BATHY_ERR_CUDA; }
    ~DevBuf() { if (p) cudaFreeAsync(p, s); }
};

}  // namespace bathy

using namespace bathy;

extern "C" {

BATHY_API int interp_bilinear(const float* d_in, grid_geom_t in, float* d_out, grid_geom_t out, void* cuda_stream)
{
    if (!d_in || !d_out) return BATHY_ERR_NULL;
    int rc = check_in_geom(in);
    if (rc) return rc;
    rc = check_out_geom(out);
    if (rc) return rc;
    return launch_bilinear(d_in, in, d_out, out, static_cast<cudaStream_t>(cuda_stream));
}

BATHY_API int interp_catmull_rom(const float* d_in, grid_geom_t in, float* d_out, grid_geom_t out, void* cuda_stream)
{
    if (!d_in || !d_out) return BATHY_ERR_NULL;
    int rc = check_in_geom(in);
    if (rc) return rc;
    rc = check_out_geom(out);
    if (rc) return rc;
    return launch_catmull_rom(d_in, in, d_out, out, static_cast<cudaStream_t>(cuda_stream));
}

BATHY_API size_t interp_spline_workspace_bytes(grid_geom_t in, grid_geom_t out)
{
    if (check_in_geom(in) || check_out_geom(out)) return 0;
    return spline_workspace_bytes(in, out);
}

BATHY_API int interp_spline(const float* d_in, grid_geom_t in, float* d_out, grid_geom_t out,
                  void* d_workspace, size_t workspace_bytes, void* cuda_stream)
{
    if (!d_in || !d_out) return BATHY_ERR_NULL;
    int rc = check_in_geom(in);
    if (rc) return rc;
    rc = check_out_geom(out);
    if (rc) return rc;
    if (!d_workspace || workspace_bytes < spline_workspace_bytes(in, out)) return BATHY_ERR_WORKSPACE;
    if (reinterpret_cast<uintptr_t>(d_workspace) % 256 != 0) return BATHY_ERR_WORKSPACE;
    return launch_spline(d_in, in, d_out, out, d_workspace, static_cast<cudaStream_t>(cuda_stream), g_spline_path.load());
}

BATHY_API int krige_build_index(const float* d_x, const float* d_y, const float* d_z, int64_t n,
                      float cell_size, void* cuda_stream, krige_index_t** out_index)
{
    if (!d_x || !d_y || !d_z || !out_index) return BATHY_ERR_NULL;
    *out_index = nullptr;
    if (n < 1 || n > 0x7fffffffLL) return BATHY_ERR_SIZE;
    if (!(cell_size >= 0.0f) || !isfinite(cell_size)) return BATHY_ERR_GEOMETRY;
    return build_index(d_x, d_y, d_z, n, cell_size, static_cast<cudaStream_t>(cuda_stream), out_index);
}

BATHY_API int krige_predict(const krige_index_t* idx, grid_geom_t out, variogram_t vg, int32_t k,
                  float* d_zhat, int32_t* d_nbr_or_null, int64_t* d_failed_or_null, void* cuda_stream)
{
    if (!idx || idx->magic != kIndexMagic) return BATHY_ERR_INDEX;
    if (!d_zhat) return BATHY_ERR_NULL;
    int rc = check_out_geom(out);
    if (rc) return rc;
    rc = check_variogram(vg);
    if (rc) return rc;
    if (k < 1 || k > BATHY_MAX_K || (int64_t)k > idx->n) return BATHY_ERR_K;
    return launch_predict(idx, out, vg, k, d_zhat, nullptr, d_nbr_or_null, d_failed_or_null, nullptr,
                          static_cast<cudaStream_t>(cuda_stream), nullptr);
}

BATHY_API int krige_predict_ex(const krige_index_t* idx, grid_geom_t out, variogram_t vg, int32_t k,
                     float* d_zhat, const krige_outputs_t* outputs_or_null, void* cuda_stream)
{
    if (!idx || idx->magic != kIndexMagic) return BATHY_ERR_INDEX;
    if (!d_zhat) return BATHY_ERR_NULL;
    int rc = check_out_geom(out);
    if (rc) return rc;
    rc = check_variogram(vg);
    if (rc) return rc;
    if (k < 1 || k > BATHY_MAX_K || (int64_t)k > idx->n) return BATHY_ERR_K;
    krige_outputs_t o = {nullptr, nullptr, nullptr, nullptr};
    if (outputs_or_null) o = *outputs_or_null;
    return launch_predict(idx, out, vg, k, d_zhat, o.d_var, o.d_nbr, o.d_failed, o.d_illcond,
                          static_cast<cudaStream_t>(cuda_stream), nullptr);
}

BATHY_API int krige_predict_aniso(const krige_index_t* idx, grid_geom_t out, variogram_t vg, krige_aniso_t aniso, int32_t k,
                        float* d_zhat, const krige_outputs_t* outputs_or_null, void* cuda_stream)
{
    if (!idx || idx->magic != kIndexMagic) return BATHY_ERR_INDEX;
    if (!d_zhat) return BATHY_ERR_NULL;
    int rc = check_out_geom(out);
    if (rc) return rc;
    rc = check_variogram(vg);
    if (rc) return rc;
    if (!isfinite(aniso.angle_deg) || !(aniso.ratio > 0.0f) || aniso.ratio > 1.0f) return BATHY_ERR_VARIOGRAM;
    if (k < 1 || k > BATHY_MAX_K || (int64_t)k > idx->n) return BATHY_ERR_K;
    krige_outputs_t o = {nullptr, nullptr, nullptr, nullptr};
    if (outputs_or_null) o = *outputs_or_null;
    return launch_predict(idx, out, vg, k, d_zhat, o.d_var, o.d_nbr, o.d_failed, o.d_illcond,
                          static_cast<cudaStream_t>(cuda_stream), &aniso);
}

BATHY_API int interp_krige_window(const float* d_in, grid_geom_t g, krige_window_t win, variogram_t vg,
                        float* d_out, uint8_t* d_how_or_null, int64_t* d_failed_or_null, void* cuda_stream)
{
    if (!d_in || !d_out) return BATHY_ERR_NULL;
    int rc = check_in_geom(g);
    if (rc) return rc;
    rc = check_variogram(vg);
    if (rc) return rc;
    if (win.half < 1 || win.half > 3 || win.n_max < 1 || win.n_min < 1) return BATHY_ERR_K;
    return launch_krige_window(d_in, g, win.half, win.n_max, win.n_min, vg, d_out, d_how_or_null, d_failed_or_null,
                               static_cast<cudaStream_t>(cuda_stream));
}

// interp_krige_window with its scratch in a fixed device array of the library (krige_window.cu): for callers that
// may not allocate device memory while they run (bathy.h says who and why).  Same checks, then the size limit.
BATHY_API int interp_krige_window_noalloc(const float* d_in, grid_geom_t g, krige_window_t win, variogram_t vg,
                                float* d_out, uint8_t* d_how_or_null, int64_t* d_failed_or_null, void* cuda_stream)
{
    if (!d_in || !d_out) return BATHY_ERR_NULL;
    int rc = check_in_geom(g);
    if (rc) return rc;
    rc = check_variogram(vg);
    if (rc) return rc;
    if (win.half < 1 || win.half > 3 || win.n_max < 1 || win.n_min < 1) return BATHY_ERR_K;
    if ((long long)g.nx * g.ny > (long long)BATHY_NOALLOC_MAX_CELLS) return BATHY_ERR_SCRATCH;
    return launch_krige_window_noalloc(d_in, g, win.half, win.n_max, win.n_min, vg, d_out, d_how_or_null, d_failed_or_null,
                                       static_cast<cudaStream_t>(cuda_stream));
}

BATHY_API int krige_index_create(float xmin, float xmax, float ymin, float ymax, float cell_size, int64_t capacity,
                       void* cuda_stream, krige_index_t** out_index)
{
    if (!out_index) return BATHY_ERR_NULL;
    *out_index = nullptr;
    if (capacity < 1 || capacity > 0x7fffffffLL) return BATHY_ERR_SIZE;
    if (!isfinite(xmin) || !isfinite(xmax) || !isfinite(ymin) || !isfinite(ymax) || !(xmax >= xmin) || !(ymax >= ymin))
        return BATHY_ERR_GEOMETRY;
    if (!(cell_size >= 0.0f) || !isfinite(cell_size)) return BATHY_ERR_GEOMETRY;
    return create_index(xmin, xmax, ymin, ymax, cell_size, capacity, static_cast<cudaStream_t>(cuda_stream), out_index);
}

BATHY_API int krige_index_append(krige_index_t* idx, const float* d_x, const float* d_y, const float* d_z, int64_t n,
                       float* d_changed_bbox_or_null, void* cuda_stream)
{
    if (!idx || idx->magic != kIndexMagic) return BATHY_ERR_INDEX;
    if (!d_x || !d_y || !d_z) return BATHY_ERR_NULL;
    if (n < 1) return BATHY_ERR_SIZE;
    return append_index(idx, d_x, d_y, d_z, n, d_changed_bbox_or_null, static_cast<cudaStream_t>(cuda_stream));
}

BATHY_API void krige_free_index(krige_index_t* idx) { free_index(idx); }
BATHY_API void krige_free_index_async(krige_index_t* idx, void* cuda_stream) { free_index_async(idx, static_cast<cudaStream_t>(cuda_stream)); }

BATHY_API int krige_index_info(const krige_index_t* idx, int64_t* n, float* cell_size, int32_t* ncx, int32_t* ncy)
{
    if (!idx || idx->magic != kIndexMagic) return BATHY_ERR_INDEX;
    IndexHeader h;
    const int rc = index_header(idx, &h);                  // waits for the build / append to finish
    if (rc) return rc;
    if (n) *n = h.n;
    if (cell_size) *cell_size = h.cell;
    if (ncx) *ncx = h.ncx;
    if (ncy) *ncy = h.ncy;
    return h.status;                                       // BATHY_ERR_GEOMETRY: non-finite soundings
}

}  // extern "C"

namespace {

// The host-buffer forms: `wait` = synchronise the stream before returning (the plain forms), else
// everything (allocations, copies, kernels, releases) is only enqueued on the stream (`*_async`).
typedef int (*grid_launch_fn)(const float*, const grid_geom_t&, float*, const grid_geom_t&, cudaStream_t);

int gather_host(grid_launch_fn launch, const float* h_in, grid_geom_t in, float* h_out, grid_geom_t out, void* cuda_stream, bool wait)
{
    if (!h_in || !h_out) return BATHY_ERR_NULL;
    int rc = check_in_geom(in);
    if (rc) return rc;
    rc = check_out_geom(out);
    if (rc) return rc;
    cudaStream_t s = static_cast<cudaStream_t>(cuda_stream);
    const size_t nin = (size_t)in.nx * in.ny * sizeof(float), nout = (size_t)out.nx * out.ny * sizeof(float);
    DevBuf din(s), dout(s);
    if (din.alloc(nin) || dout.alloc(nout)) return BATHY_ERR_CUDA;
    BATHY_CUDA_TRY(cudaMemcpyAsync(din.p, h_in, nin, cudaMemcpyHostToDevice, s));
    rc = launch(static_cast<const float*>(din.p), in, static_cast<float*>(dout.p), out, s);
    if (rc) return rc;
    BATHY_CUDA_TRY(cudaMemcpyAsync(h_out, dout.p, nout, cudaMemcpyDeviceToHost, s));
    if (wait) BATHY_CUDA_TRY(cudaStreamSynchronize(s));
    return BATHY_OK;
}

int spline_host(const float* h_in, grid_geom_t in, float* h_out, grid_geom_t out, void* cuda_stream, bool wait)
{
    if (!h_in || !h_out) return BATHY_ERR_NULL;
    int rc = check_in_geom(in);
    if (rc) return rc;
    rc = check_out_geom(out);
    if (rc) return rc;
    cudaStream_t s = static_cast<cudaStream_t>(cuda_stream);
    const size_t nin = (size_t)in.nx * in.ny * sizeof(float), nout = (size_t)out.nx * out.ny * sizeof(float);
    DevBuf din(s), dout(s), ws(s);
    if (din.alloc(nin) || dout.alloc(nout) || ws.alloc(spline_workspace_bytes(in, out))) return BATHY_ERR_CUDA;
    BATHY_CUDA_TRY(cudaMemcpyAsync(din.p, h_in, nin, cudaMemcpyHostToDevice, s));
    rc = launch_spline(static_cast<const float*>(din.p), in, static_cast<float*>(dout.p), out, ws.p, s, g_spline_path.load());
    if (rc) return rc;
    BATHY_CUDA_TRY(cudaMemcpyAsync(h_out, dout.p, nout, cudaMemcpyDeviceToHost, s));
    if (wait) BATHY_CUDA_TRY(cudaStreamSynchronize(s));
    return BATHY_OK;
}

int krige_host_impl(const float* h_x, const float* h_y, const float* h_z, int64_t n, float cell_size,
                    grid_geom_t out, variogram_t vg, int32_t k, float* h_zhat, int64_t* h_failed_or_null,
                    void* cuda_stream, bool wait)
{
    if (!h_x || !h_y || !h_z || !h_zhat) return BATHY_ERR_NULL;
    if (n < 1 || n > 0x7fffffffLL) return BATHY_ERR_SIZE;
    if (!(cell_size >= 0.0f) || !isfinite(cell_size)) return BATHY_ERR_GEOMETRY;
    int rc = check_out_geom(out);
    if (rc) return rc;
    rc = check_variogram(vg);
    if (rc) return rc;
    if (k < 1 || k > BATHY_MAX_K || (int64_t)k > n) return BATHY_ERR_K;
    cudaStream_t s = static_cast<cudaStream_t>(cuda_stream);
    const size_t nb = (size_t)n * sizeof(float), nout = (size_t)out.nx * out.ny * sizeof(float);
    DevBuf dx(s), dy(s), dz(s), dout(s), dfail(s);
    if (dx.alloc(nb) || dy.alloc(nb) || dz.alloc(nb) || dout.alloc(nout) || dfail.alloc(sizeof(int64_t))) return BATHY_ERR_CUDA;
    BATHY_CUDA_TRY(cudaMemcpyAsync(dx.p, h_x, nb, cudaMemcpyHostToDevice, s));
    BATHY_CUDA_TRY(cudaMemcpyAsync(dy.p, h_y, nb, cudaMemcpyHostToDevice, s));
    BATHY_CUDA_TRY(cudaMemcpyAsync(dz.p, h_z, nb, cudaMemcpyHostToDevice, s));
    BATHY_CUDA_TRY(cudaMemsetAsync(dfail.p, 0, sizeof(int64_t), s));
    krige_index* idx = nullptr;
    rc = build_index(static_cast<const float*>(dx.p), static_cast<const float*>(dy.p), static_cast<const float*>(dz.p),
                     n, cell_size, s, &idx);
    if (rc) return rc;
    rc = launch_predict(idx, out, vg, k, static_cast<float*>(dout.p), nullptr, nullptr, static_cast<int64_t*>(dfail.p), nullptr, s, nullptr);
    if (rc == BATHY_OK) {
        cudaError_t e = cudaMemcpyAsync(h_zhat, dout.p, nout, cudaMemcpyDeviceToHost, s);
        if (e == cudaSuccess && h_failed_or_null)
            e = cudaMemcpyAsync(h_failed_or_null, dfail.p, sizeof(int64_t), cudaMemcpyDeviceToHost, s);
        if (e == cudaSuccess && wait) e = cudaStreamSynchronize(s);
        if (e != cudaSuccess) rc = BATHY_ERR_CUDA;
    }
    free_index_async(idx, s);
    return rc;
}

}  // namespace

extern "C" {

BATHY_API int interp_bilinear_host(const float* h_in, grid_geom_t in, float* h_out, grid_geom_t out, void* cuda_stream)
{ return gather_host(launch_bilinear, h_in, in, h_out, out, cuda_stream, true); }
BATHY_API int interp_bilinear_host_async(const float* h_in, grid_geom_t in, float* h_out, grid_geom_t out, void* cuda_stream)
{ return gather_host(launch_bilinear, h_in, in, h_out, out, cuda_stream, false); }
BATHY_API int interp_catmull_rom_host(const float* h_in, grid_geom_t in, float* h_out, grid_geom_t out, void* cuda_stream)
{ return gather_host(launch_catmull_rom, h_in, in, h_out, out, cuda_stream, true); }
BATHY_API int interp_catmull_rom_host_async(const float* h_in, grid_geom_t in, float* h_out, grid_geom_t out, void* cuda_stream)
{ return gather_host(launch_catmull_rom, h_in, in, h_out, out, cuda_stream, false); }
BATHY_API int interp_spline_host(const float* h_in, grid_geom_t in, float* h_out, grid_geom_t out, void* cuda_stream)
{ return spline_host(h_in, in, h_out, out, cuda_stream, true); }
BATHY_API int interp_spline_host_async(const float* h_in, grid_geom_t in, float* h_out, grid_geom_t out, void* cuda_stream)
{ return spline_host(h_in, in, h_out, out, cuda_stream, false); }
BATHY_API int krige_host(const float* h_x, const float* h_y, const float* h_z, int64_t n, float cell_size,
               grid_geom_t out, variogram_t vg, int32_t k, float* h_zhat, int64_t* h_failed_or_null,
               void* cuda_stream)
{ return krige_host_impl(h_x, h_y, h_z, n, cell_size, out, vg, k, h_zhat, h_failed_or_null, cuda_stream, true); }
BATHY_API int krige_host_async(const float* h_x, const float* h_y, const float* h_z, int64_t n, float cell_size,
               grid_geom_t out, variogram_t vg, int32_t k, float* h_zhat, int64_t* h_failed_or_null,
               void* cuda_stream)
{ return krige_host_impl(h_x, h_y, h_z, n, cell_size, out, vg, k, h_zhat, h_failed_or_null, cuda_stream, false); }

BATHY_API const char* bathy_strerror(int status)
{
    switch (status) {
        case BATHY_OK:            return "ok";
        case BATHY_ERR_NULL:      return "a required pointer is NULL";
        case BATHY_ERR_GEOMETRY:  return "invalid grid geometry or non-finite coordinates";
        case BATHY_ERR_K:         return "neighbour count k out of range";
        case BATHY_ERR_VARIOGRAM: return "invalid variogram parameters";
        case BATHY_ERR_WORKSPACE: return "workspace missing, misaligned or too small";
        case BATHY_ERR_CUDA:      return "CUDA runtime error (no device, out of memory or launch failure)";
        case BATHY_ERR_SIZE:      return "problem size out of range";
        case BATHY_ERR_INDEX:     return "invalid kriging index handle";
        case BATHY_ERR_SCRATCH:   return "grid larger than the fixed scratch of interp_krige_window_noalloc (BATHY_NOALLOC_MAX_CELLS = 4194304 cells): tile it or call interp_krige_window";
        default:                  return "unknown status";
    }
}

BATHY_API int bathy_set_spline_path(int path)
{
    if (path < 0 || path > 3) return BATHY_ERR_GEOMETRY;
    g_spline_path.store(path);
    g_bilinear_tma.store(path != 3, std::memory_order_relaxed);
    return BATHY_OK;
}

BATHY_API int64_t bathy_launch_count(void) { return g_launches.load(std::memory_order_relaxed); }

}  // extern "C"
