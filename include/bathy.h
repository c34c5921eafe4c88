/* bathy.h -- C ABI of libbathy.so: B200 (sm_100a) interpolation of sonar depth soundings onto a
 * regular grid by three methods -- bilinear, separable natural bicubic spline, ordinary kriging.
 *
 * The operations are those of "Towards Real-Time Interpolation for Enhanced AUV Deep Sea Mapping"
 * (arxiv 2505.22675), cited below as PAPER.md:Lnn, with the readings listed in DESIGN.md.
 *
 * Conventions (every entry point):
 *   - `d_*` arguments are DEVICE pointers owned by the caller; `h_*` arguments are HOST pointers.
 *     The library never allocates or frees caller buffers and never keeps a caller pointer after
 *     the call's work on `cuda_stream` has completed.
 *   - `cuda_stream` is a cudaStream_t passed as void* (NULL = the legacy default stream).  Device-
 *     pointer calls only ENQUEUE work on that stream and never synchronise the host (the two
 *     exceptions say so: krige_index_info and krige_free_index).  `*_host` calls copy host->device,
 *     run the same kernels and copy device->host on that stream and return after the stream has
 *     drained; `*_host_async` calls only enqueue.
 *   - Return value: 0 (BATHY_OK) or a negative bathy_status.  Argument errors are detected
 *     synchronously and nothing is launched.  No exceptions, no environment variables.  Global state:
 *     the launch counter, the spline path selector with the TMA-staging switch it drives (both atomic; profiling
 *     knobs, see bathy_set_spline_path), the fixed scratch array of interp_krige_window_noalloc, and per-DEVICE one-time setup (kernel attributes;
 *     the first index or host-buffer call on a device raises the release threshold of that device's default memory
 *     pool to 2 GiB so that stream-ordered scratch is recycled instead of returned to the driver).
 *     Calls on distinct streams are thread-safe, and one process may use several devices (the current
 *     device of the calling thread is used; an index belongs to the device it was built on).
 *   - A grid is row-major fp32 with leading dimension nx.  Node (i, j) -- i = row (y), j = column
 *     (x) -- sits at x = x0 + j*dx, y = y0 + i*dy.
 *   - There is no CPU fallback: without a CUDA device every compute call returns BATHY_ERR_CUDA.
 */
#ifndef BATHY_H
#define BATHY_H

#include <stddef.h>
#include <stdint.h>

#if defined(__GNUC__)
#define BATHY_API __attribute__((visibility("default")))
#else
#define BATHY_API
#endif

#ifdef __cplusplus
extern "C" {
#endif

typedef enum {
    BATHY_OK                = 0,
    BATHY_ERR_NULL          = -1,   /* a required pointer is NULL */
    BATHY_ERR_GEOMETRY      = -2,   /* input grid nx<2 or ny<2, output nx<1 or ny<1, dx<=0 or dy<=0, non-finite */
    BATHY_ERR_K             = -3,   /* k<1, k>BATHY_MAX_K or k>n */
    BATHY_ERR_VARIOGRAM     = -4,   /* range<=0, sill<=0, nugget<0, nugget>sill, unknown model, non-finite */
    BATHY_ERR_WORKSPACE     = -5,   /* workspace NULL or smaller than *_workspace_bytes() */
    BATHY_ERR_CUDA          = -6,   /* a CUDA runtime call failed (no device, out of memory, launch error) */
    BATHY_ERR_SIZE          = -7,   /* n<1 or n>2^31-1 soundings, or a grid with more than 2^31-1 nodes per row/column */
    BATHY_ERR_INDEX         = -8,   /* index handle NULL, not built by krige_build_index, or built on another device than the current one */
    BATHY_ERR_SCRATCH       = -9    /* interp_krige_window_noalloc: the grid has more than BATHY_NOALLOC_MAX_CELLS cells */
} bathy_status;

#define BATHY_MAX_K 64

/* Regular grid geometry ("a given cell structure of existing points ... inside a
 * larger grid"). */
typedef struct {
    int32_t nx, ny;
    float   x0, y0, dx, dy;
} grid_geom_t;

/* Variogram.  model 0 = exponential exactly as printed at L157,
 * gamma(h) = nugget + (sill-nugget)(1 - exp(-h/range)) (no factor 3); model 1 = spherical,
 * gamma(h) = nugget + (sill-nugget)(1.5 h/range - 0.5 (h/range)^3) for 0<h<range, sill beyond.
 * gamma(0) = 0 for both.  `sill` is the TOTAL sill (nugget included); nugget <= sill. */
typedef struct {
    int32_t model;
    float   range, sill, nugget;
} variogram_t;

#define BATHY_VGM_EXPONENTIAL 0
#define BATHY_VGM_SPHERICAL   1
/* SURVEY.md 8(f) NEXT-4 ("many variants ... can be easily implemented on top"): Gaussian,
 * gamma(h) = nugget + (sill-nugget)(1 - exp(-(h/range)^2)) in the same no-factor-3 convention as L157. */
#define BATHY_VGM_GAUSSIAN    2

/* Opaque, library-owned, immutable after build; may be shared by concurrent krige_predict calls. */
typedef struct krige_index krige_index_t;

/* ---------------------------------------------------------------------------------------------
 * interp_bilinear -- PAPER.md:L115-L134 (section III-A), formula at L132.
 * For every node (I, J) of `out`: u = (x - in.x0)/in.dx, v = (y - in.y0)/in.dy (float64 from the
 * fp32 fields); i = min(floor u, nx-2), t = u - i (same for j, s); result =
 * (1-t)(1-s) Q11 + t(1-s) Q21 + (1-t)s Q12 + t s Q22 with Q11 = in[j][i], Q21 = in[j][i+1],
 * Q12 = in[j+1][i], Q22 = in[j+1][i+1], evaluated in fp32.  Nodes outside the input extent
 * (u<0, u>nx-1, v<0, v>ny-1) are NaN; a NaN corner makes the node NaN (the paper's bilinear "has no
 * fallback", L182).
 * d_in  [in.ny * in.nx] fp32, read only.   d_out [out.ny * out.nx] fp32, fully overwritten.
 * d_in and d_out must not overlap. */
BATHY_API int interp_bilinear(const float* d_in, grid_geom_t in, float* d_out, grid_geom_t out, void* cuda_stream);

/* ---------------------------------------------------------------------------------------------
 * interp_catmull_rom -- the paper's own "cubic spline" (section III-B; SURVEY.md
 * 8(f) NEXT-1).  Interval location, extent and layout as interp_bilinear.  With P0..P3 the samples at
 * i-1, i, i+1, i+2 and t = u - i,
 *   C(t) = 1/2 (2 P1 + (-P0 + P2) t + (2 P0 - 5 P1 + 4 P2 - P3) t^2 + (-P0 + 3 P1 - 3 P2 + P3) t^3)
 * is applied in x on each of the 4 rows j-1 .. j+2 and then in y (L138).  A node with
 * one of its 16 neighbours outside the grid or NaN "falls back to a bilinear calculation" (L144, sense
 * fixed by L171): it gets the value of interp_bilinear (NaN if one of the 4 corners is NaN, L182).
 * d_in  [in.ny * in.nx] fp32, read only.   d_out [out.ny * out.nx] fp32, fully overwritten; no overlap. */
BATHY_API int interp_catmull_rom(const float* d_in, grid_geom_t in, float* d_out, grid_geom_t out, void* cuda_stream);

/* ---------------------------------------------------------------------------------------------
 * interp_spline -- separable natural bicubic spline (BASELINE.json north_star; DESIGN.md reading
 * D1: the paper's section III-B, uses the local Catmull-Rom cubic instead).
 * 1-D operator on uniform knots with spacing h: second derivatives M with M_0 = M_{n-1} = 0 and
 * M_{i-1} + 4 M_i + M_{i+1} = 6 (z_{i-1} - 2 z_i + z_{i+1}) / h^2 (batched tridiagonal solves);
 * S = A z_i + B z_{i+1} + ((A^3-A) M_i + (B^3-B) M_{i+1}) h^2/6, A = 1-t, B = t.  2-D = the tensor
 * product (rows in x, then columns in y).  Interval location, extent and NaN rules as bilinear.
 * Precondition: d_in holds no NaN (not checked).  With a NaN in d_in the result is undefined in the sense that it
 * depends on the implementation path: the NaN spreads through the tridiagonal solves that contain it -- the solve
 * windows of the fused tile kernel (about 11 knots either side), or the 256-knot segments (+ 32-knot halo) of the
 * global-solve path -- along its row and its column, and through everything evaluated from those knots; output
 * nodes further away are unaffected.
 * d_workspace: device scratch of at least interp_spline_workspace_bytes(in, out) bytes, 256-byte
 * aligned, contents undefined on return; may be reused by later calls on the same stream. */
BATHY_API size_t interp_spline_workspace_bytes(grid_geom_t in, grid_geom_t out);
BATHY_API int interp_spline(const float* d_in, grid_geom_t in, float* d_out, grid_geom_t out,
                  void* d_workspace, size_t workspace_bytes, void* cuda_stream);

/* ---------------------------------------------------------------------------------------------
 * krige_build_index -- uniform-grid binning of the soundings for the neighbour search that
 * replaces the paper's "nearest n valid candidate neighbors" helper: bounding box,
 * cell id per sounding, histogram, exclusive scan, stable scatter of (x, y, z, original index).
 * d_x, d_y, d_z [n] fp32 (SoA), n in [1, 2^31-1]; finite, no two soundings at identical (x, y)
 * (kriging with duplicates is singular -- such nodes come out NaN, see krige_predict).
 * cell_size: edge of a square cell in the units of x/y; 0 = automatic (about 8 soundings per cell).  A
 * performance knob only: results do not depend on it.  The library enlarges it when the cell grid would
 * exceed 4 cells per sounding or 2^26 cells.  The build orders the soundings of a cell by original index with a
 * rank count that is quadratic in the cell's population: fine at the ~8 soundings per cell of the automatic size
 * on survey-like data, slow when a caller's cell size (or extreme clustering) puts more than ~10^4 soundings into
 * one cell.
 * The soundings are copied into library-owned device memory: the caller may free d_x/d_y/d_z once
 * the stream reaches this point.  ENQUEUE ONLY: the bounding box never comes back to the host -- the
 * cell grid is sized by a kernel and lives in a device header that krige_predict reads.  Non-finite
 * coordinates therefore cannot be reported by this call: they mark the index unusable on the device,
 * krige_index_info then returns BATHY_ERR_GEOMETRY and every krige_predict node comes out NaN and is
 * counted in d_failed.  *out_index is released only by krige_free_index[_async]. */
BATHY_API int krige_build_index(const float* d_x, const float* d_y, const float* d_z, int64_t n,
                      float cell_size, void* cuda_stream, krige_index_t** out_index);

/* ---------------------------------------------------------------------------------------------
 * krige_predict -- ordinary kriging (section III-C) at every node of `out`.
 * Node coordinates are the fp32 values xq = fmaf(J, dx, x0), yq = fmaf(I, dy, y0).
 *   neighbours : the k soundings with the smallest (key, original index), key =
 *                fmaf(ddx, ddx, ddy*ddy) in fp32 with ddx = xq - x_i, ddy = yq - y_i;
 *   covariances: C_ij = sill - gamma(h_ij), c0_i = sill - gamma(h_0i);
 *   weights    : C lambda + mu 1 = c0, 1^T lambda = 1, the standard ordinary-kriging system
 *                (what PAPER.md:L159-L165 solves "using Gaussian elimination"), here by Cholesky
 *                of C and a Schur complement for mu;
 *   estimate   : z_hat = sum_i lambda_i z_i.
 * k in [1, min(BATHY_MAX_K, n)].
 * d_zhat            [out.ny * out.nx] fp32, fully overwritten.
 * d_nbr_or_null     [out.ny * out.nx * k] int32: original indices of the neighbours in ascending
 *                   (key, index) order (parity/debug output), or NULL.
 * d_failed_or_null  one int64 device counter, INCREMENTED by the number of nodes whose system was
 *                   not positive definite (duplicate soundings); those nodes are written NaN.
 *                   The caller zeroes it.  NULL = not counted.
 * Tiles (BASELINE.json config 5) are calls with a sub-geometry: x0/y0 shifted to the tile's first
 * node, nx/ny the tile size, d_zhat a tile buffer. */
BATHY_API int krige_predict(const krige_index_t* idx, grid_geom_t out, variogram_t vg, int32_t k,
                  float* d_zhat, int32_t* d_nbr_or_null, int64_t* d_failed_or_null, void* cuda_stream);

/* Releases an index once every kernel that reads it has finished.  BLOCKS the host: it waits for the stream of
 * the last build / append when every krige_predict[_ex] and append of this index was issued on that stream, and
 * for the whole device as soon as one of them went to any other stream (the library keeps track; the caller need
 * not).  Safe to call right after a krige_predict on any stream.  NULL is a no-op. */
BATHY_API void krige_free_index(krige_index_t* idx);

/* Stream-ordered release, no host synchronisation: the index memory returns to the device's memory
 * pool when `cuda_stream` reaches this point.  The caller guarantees that every krige_predict that
 * uses the index was issued on `cuda_stream` before this call (or is otherwise ordered before it).
 * The handle is invalid on return.  NULL is a no-op.  (Real-time tile loop: build, predict tiles,
 * release -- without ever stalling the host.) */
BATHY_API void krige_free_index_async(krige_index_t* idx, void* cuda_stream);

/* Introspection of an index: number of soundings, cell size used, cell-grid dimensions.  These live on
 * the device, so this call WAITS for the stream of the last build / append.  Returns BATHY_ERR_GEOMETRY
 * when the soundings held a non-finite coordinate. */
BATHY_API int krige_index_info(const krige_index_t* idx, int64_t* n, float* cell_size, int32_t* ncx, int32_t* ncy);

/* ---------------------------------------------------------------------------------------------
 * krige_predict_ex -- krige_predict with optional extra outputs.  All pointers
 * may be NULL; `outputs_or_null` == NULL is krige_predict without neighbour and failure outputs.
 *   d_var      [out.ny * out.nx] fp32: the ordinary-kriging variance
 *              sigma^2 = sum_i lambda_i gamma(h_0i) + mu   (mu: the Lagrange multiplier of the gamma-form
 *              system [Gamma 1; 1^T 0][lambda; mu] = [gamma0; 1], the standard form of PAPER.md:L159-L165),
 *              in the units of sill; 0 at a node that coincides with a sounding; NaN where the node failed.
 *   d_nbr, d_failed: as krige_predict.
 *   d_illcond  one int64 device counter, INCREMENTED by the number of nodes whose smallest Cholesky pivot
 *              of the sill-normalised covariance matrix fell below BATHY_ILLCOND_PIVOT (neighbours much
 *              closer to each other than the variogram range): their estimate is finite but the fp32
 *              factorisation has lost accuracy, relative error of the weights ~ k * 6e-8 / pivot
 *              (reading K-cond).  The caller zeroes it. */
typedef struct {
    float*   d_var;
    int32_t* d_nbr;
    int64_t* d_failed;
    int64_t* d_illcond;
} krige_outputs_t;
#define BATHY_ILLCOND_PIVOT 1e-3f
BATHY_API int krige_predict_ex(const krige_index_t* idx, grid_geom_t out, variogram_t vg, int32_t k,
                     float* d_zhat, const krige_outputs_t* outputs_or_null, void* cuda_stream);

/* ---------------------------------------------------------------------------------------------
 * krige_predict_aniso -- krige_predict_ex with a geometrically anisotropic variogram ("many
 * variants ... can be easily implemented on top"; reading Ani).  The lag between two
 * locations is measured in the axes of the anisotropy ellipse: with t = angle_deg (counter-clockwise from +x, the
 * direction of greatest continuity),
 *      u = cos(t) dx + sin(t) dy,   w = (-sin(t) dx + cos(t) dy) / ratio,   h = sqrt(u^2 + w^2),
 * and gamma(h) is the variogram `vg`, whose `range` is the range ALONG that direction; across it the same values are
 * reached at ratio times the distance.  ratio = (range across) / (range along) in (0, 1]; ratio = 1 is krige_predict_ex
 * whatever the angle.  Only the variogram sees this lag: the neighbours are the k nearest soundings by the plain
 * (key, index) order of krige_predict.  All outputs as krige_predict_ex.
 * Errors as krige_predict, plus BATHY_ERR_VARIOGRAM for a ratio outside (0, 1] or a non-finite angle. */
typedef struct {
    float angle_deg, ratio;
} krige_aniso_t;
BATHY_API int krige_predict_aniso(const krige_index_t* idx, grid_geom_t out, variogram_t vg, krige_aniso_t aniso, int32_t k,
                        float* d_zhat, const krige_outputs_t* outputs_or_null, void* cuda_stream);

/* ---------------------------------------------------------------------------------------------
 * interp_krige_window -- hole filling on a regular grid by ordinary kriging over a window of grid cells, the form
 * of kriging the paper measured: "the implementation in this study uses a 5x5 grid"
 * (PAPER.md:L163); cells removed at random are interpolated back (Grid B, L225-L234).
 *   - a valid (non-NaN) cell of d_in is copied to d_out;
 *   - a NaN cell (i, j) is estimated by ordinary kriging (as krige_predict: variogram, ordinary-kriging system,
 *     z_hat = sum lambda z) from the valid cells of the (2 half + 1)^2 window centred on it, clipped by the grid;
 *     if more than n_max are valid, the n_max with the smallest (key, window order) are used -- the paper's
 *     "nearest n valid candidate neighbors" (L179) -- key = fmaf(ddx, ddx, ddy*ddy) in fp32 with ddx = (float)dj * dx,
 *     ddy = (float)di * dy, window order = row-major over the window;
 *   - with fewer than n_min valid candidates the cell "falls back to bilinear interpolation" (L171, L180): the
 *     formula of L132 on the rectangle of its four diagonal neighbours (t = s = 1/2, i.e. their mean); NaN if one
 *     of them is NaN or outside the grid (bilinear has no fallback, L182).
 * win.half in [1, 3] (3x3, 5x5 = the paper's, 7x7); win.n_max >= 1 (values above the window size mean "all");
 * win.n_min >= 1.  d_in [g.ny * g.nx] fp32; d_out the same size, fully overwritten, no overlap with d_in.
 * d_how_or_null [g.ny * g.nx] uint8: 0 = valid cell copied, 1..48 = kriged from that many neighbours, 255 =
 * bilinear fallback.  d_how is written when the method is chosen, before the solve: how = 1..48 can accompany a NaN
 * depth when the system turned out singular (that hole is then counted in d_failed).
 * d_failed_or_null: one int64 device counter, INCREMENTED by the number of holes whose kriging system was not
 * positive definite (written NaN), as krige_predict.  It counts singular solves ONLY: a hole that stays NaN through
 * the bilinear fallback (how = 255 with a NaN or off-grid diagonal neighbour -- always the case on the border rows
 * and columns) is NOT counted; find those with how == 255 and a NaN depth.
 * Enqueue only (scratch comes from the stream's pool). */
typedef struct {
    int32_t half, n_max, n_min;
} krige_window_t;
BATHY_API int interp_krige_window(const float* d_in, grid_geom_t g, krige_window_t win, variogram_t vg,
                        float* d_out, uint8_t* d_how_or_null, int64_t* d_failed_or_null, void* cuda_stream);

/* ---------------------------------------------------------------------------------------------
 * interp_krige_window_noalloc -- interp_krige_window for callers that must not allocate device memory while they
 * run.  Same arguments, same operation, same kernels and the same results as interp_krige_window; the only
 * difference is where the scratch (the list of hole cells and its counter) lives: in a fixed array inside the
 * library's device image instead of memory drawn from the stream's pool.  The call issues no cudaMalloc, cudaFree,
 * cudaMallocAsync, cudaFreeAsync or any other allocating routine; d_in, d_out, d_how and d_failed are the
 * caller's, as everywhere in this header.
 *
 * Meant for: the vehicle's real-time mapping loop, which hands out its whole device-memory budget before the dive
 * and then may not ask the driver for more (an allocation in the middle of a survey line can fail, and cudaMalloc /
 * cudaFree stall every stream of the device while they run); host programs whose own allocator has reserved the
 * GPU, so that a driver allocation behind its back competes with it; and devices or driver configurations without
 * stream-ordered memory pools, where interp_krige_window itself returns BATHY_ERR_CUDA.
 *
 * Limit: g.nx * g.ny <= BATHY_NOALLOC_MAX_CELLS (2048 x 2048 cells); a larger grid is refused with
 * BATHY_ERR_SCRATCH before anything is enqueued -- tile the grid (overlapping the tiles by win.half cells), or use
 * interp_krige_window.  Cost: the array takes 16 MiB (4 bytes per cell + 256) of device memory on every GPU on
 * which this process loads the library's device code, until the process exits, used or not.
 *
 * First call on a device: looks up the array's device address (cudaGetSymbolAddress, with the calling thread's
 * current device) and sets the kernel attributes, once per device; later calls reuse both.  Make that first call
 * on each device during start-up, outside of any stream capture.
 *
 * Sharing: there is ONE array per device and every call on that device uses it.  Calls issued on the same stream
 * (or ordered by events) are safe -- each call resets the counter on its stream and rewrites the part of the list
 * it reads; nothing else of the previous call's contents matters.  Two calls whose work can overlap on the GPU
 * (different streams with no ordering between them, whether from one host thread or several) race on the list and
 * both results are undefined.  Each process and each device has its own copy.
 * Enqueue only; errors as interp_krige_window plus BATHY_ERR_SCRATCH. */
#define BATHY_NOALLOC_MAX_CELLS 4194304
BATHY_API int interp_krige_window_noalloc(const float* d_in, grid_geom_t g, krige_window_t win, variogram_t vg,
                                float* d_out, uint8_t* d_how_or_null, int64_t* d_failed_or_null, void* cuda_stream);

/* ---------------------------------------------------------------------------------------------
 * Streaming index (the paper's real-time onboard goal).
 * krige_index_create makes an EMPTY index over the caller's extent -- the planned survey area
 * [xmin, xmax] x [ymin, ymax]; soundings outside it are legal and are kept in the border cells -- with
 * room for `capacity` soundings; krige_index_append merges a batch of n soundings (the pings that just
 * arrived) into it.  The original index of a sounding is its position in the concatenation of all
 * appended batches.  create + append(A) + append(B) gives bit for bit the index of create + append(A|B),
 * hence identical neighbours and depths.  Both calls only enqueue work.  Appends and the krige_predict
 * calls that use the index must be ordered by the caller (same stream, or events): an append rewrites the
 * buffers the append before it read from.  Cost of one append: O(batch + cells of the grid in use + soundings
 * already held) -- the sorted arrays are re-merged, not O(capacity).  After an append only nodes within their k-th-neighbour
 * distance of the new soundings change: d_changed_bbox_or_null (4 floats on the device: xmin, xmax,
 * ymin, ymax of the batch) tells the caller which tiles to predict again.
 * Errors: BATHY_ERR_SIZE (capacity exceeded, n < 1), BATHY_ERR_INDEX (index not made by krige_index_create). */
BATHY_API int krige_index_create(float xmin, float xmax, float ymin, float ymax, float cell_size, int64_t capacity,
                       void* cuda_stream, krige_index_t** out_index);
BATHY_API int krige_index_append(krige_index_t* idx, const float* d_x, const float* d_y, const float* d_z, int64_t n,
                       float* d_changed_bbox_or_null, void* cuda_stream);

/* ---------------------------------------------------------------------------------------------
 * Host-buffer forms: the same operations for callers whose data lives in host memory.  Each
 * allocates device scratch, copies h_in (or h_x/h_y/h_z) to the device, runs the kernels of the
 * device-pointer form, copies the result back and waits for the stream.  Pinned host memory makes
 * the copies asynchronous and faster but is not required. */
BATHY_API int interp_bilinear_host(const float* h_in, grid_geom_t in, float* h_out, grid_geom_t out, void* cuda_stream);
BATHY_API int interp_spline_host(const float* h_in, grid_geom_t in, float* h_out, grid_geom_t out, void* cuda_stream);
BATHY_API int interp_catmull_rom_host(const float* h_in, grid_geom_t in, float* h_out, grid_geom_t out, void* cuda_stream);
BATHY_API int krige_host(const float* h_x, const float* h_y, const float* h_z, int64_t n, float cell_size,
               grid_geom_t out, variogram_t vg, int32_t k, float* h_zhat, int64_t* h_failed_or_null,
               void* cuda_stream);

/* The same three, ENQUEUED only: scratch allocation, copies, kernels and releases are all ordered on
 * `cuda_stream` and the call returns without waiting for them.  The host buffers must be
 * pinned (otherwise the copies fall back to synchronous staging) and must stay valid, and h_out /
 * h_zhat / *h_failed_or_null are defined, only after the caller has synchronised `cuda_stream`.
 * Issued on different streams, the copies of one call overlap the kernels and the opposite-direction
 * copies of another: the way to run the three methods of a survey step at PCIe speed
 * (bench.py's `e2e`).  Errors detected at enqueue time are returned; later ones surface at the
 * caller's synchronisation. */
BATHY_API int interp_bilinear_host_async(const float* h_in, grid_geom_t in, float* h_out, grid_geom_t out, void* cuda_stream);
BATHY_API int interp_spline_host_async(const float* h_in, grid_geom_t in, float* h_out, grid_geom_t out, void* cuda_stream);
BATHY_API int interp_catmull_rom_host_async(const float* h_in, grid_geom_t in, float* h_out, grid_geom_t out, void* cuda_stream);
BATHY_API int krige_host_async(const float* h_x, const float* h_y, const float* h_z, int64_t n, float cell_size,
               grid_geom_t out, variogram_t vg, int32_t k, float* h_zhat, int64_t* h_failed_or_null,
               void* cuda_stream);

/* Selects the implementation interp_spline uses (process-wide; for tests and profiling):
 * 0 = automatic (default): the fused single-pass tile kernel where it applies (up-sampling, input at
 *     least one solve window wide), else the global-solve path;
 * 1 = fused tile kernel only (BATHY_ERR_GEOMETRY where it does not apply);
 * 2 = global-solve path only (three batched full-length Thomas solves + gather evaluate);
 * 3 = fused tile kernel with the window staged by cp.async instead of the TMA box load (profiling A/B).  Side
 *     effect: path 3 ALSO turns the TMA staging of interp_bilinear and interp_catmull_rom off (they stage by cp.async
 *     instead, same results), and paths 0-2 turn it back on -- one process-wide atomic switch for all grid kernels.
 * Both compute the same natural bicubic spline; DESIGN.md "Spline window bound" gives the bound on
 * their difference (8.2e-7 x depth range per direction). */
BATHY_API int bathy_set_spline_path(int path);

/* FP32 ALU peak probe ("the builder measures an FMA-chain microbenchmark"): launches one kernel
 * in which every thread of `ctas_per_sm` (1..4) CTAs of 512 threads per SM runs 16 independent fused multiply-add
 * chains for `iters` iterations -- scalar FFMA (packed = 0) or packed fp32x2 FFMA2 (packed = 1) -- and writes the
 * number of floating-point operations the launch retires to *flop_out (host).  The caller times the launch with
 * CUDA events: flop / time is the measured peak the kriging roofline is reported against.  d_sink: one device
 * float (never written in practice).  Enqueue only. */
BATHY_API int bathy_probe_fp32(int32_t packed, int64_t iters, int32_t ctas_per_sm, float* d_sink, double* flop_out,
                     void* cuda_stream);

/* TMA probe: loads the 88 x 54 fp32 box whose first element is column x0, row y0 of the
 * [ny][nx] tensor d_in (nx and x0 multiples of 4, d_in 16-byte aligned; y0 is free) with ONE cp.async.bulk.tensor.2d into shared
 * memory and copies it to d_out [54 * 88]; elements outside the tensor arrive as zeros.  The committed reproduction
 * of whether TMA tensor loads work on the box.  Enqueue only; BATHY_ERR_CUDA if the tensor map cannot be encoded. */
BATHY_API int bathy_probe_tma(const float* d_in, int32_t nx, int32_t ny, int32_t x0, int32_t y0, float* d_out,
                    void* cuda_stream);

/* Static, never NULL. */
BATHY_API const char* bathy_strerror(int status);

/* Number of kernel launches the library has issued in this process (monotonic; for bench.py's
 * gpu_launches and tests). */
BATHY_API int64_t bathy_launch_count(void);

#ifdef __cplusplus
}
#endif
#endif /* BATHY_H */
