// spline.cu -- interp_spline: separable natural bicubic spline (
// DESIGN.md reading D1 -- the paper's own cubic, is Catmull-Rom).
//
// General path ("4-array form", any output geometry):
//   S1  Mx  = second derivatives along x of every input row      (batched tridiagonal solves)
//   S2  My  = second derivatives along y of every input column
//   S3  Mxy = second derivatives along y of every column of Mx   (== along x of the rows of My)
//   S4  S(x,y) = sum over the 4 cell corners of {z, Mx, My, Mxy} times the cubic blending weights.
// The tridiagonal matrix is the constant [1 4 1] (uniform knots), so the Thomas forward-sweep
// pivots c'_q = 1/(4 - c'_{q-1}) depend on q only and are shared by all systems: they are a 24-entry
// table (c' has converged to 2 - sqrt(3) in fp32 long before q = 24).  One thread per system.
#include "common.cuh"

namespace bathy {

namespace {

constexpr int kThreads = 256;

// c'_q of the [1 4 1] system, q = 0 is the first interior unknown: 1/4, 4/15, 15/56, ... -> 2 - sqrt(3)
__device__ __forceinline__ float thomas_cp(int q)
{
    constexpr float kCp[8] = {
        0.25f, 0.26666666666666666f, 0.26785714285714285f, 0.26794258373205743f,
        0.26794871794871794f, 0.26794915836482308f, 0.26794918998527245f, 0.26794919225551855f};
    return q < 8 ? kCp[q] : 0.26794919243112270f;
}

// The Thomas solves of the global path.  A 4096 x 4096 grid has only 4096 systems per direction -- 128 warps on
// 148 SMs, each walking a 4096-step recurrence with nothing to hide the memory latency behind (round 1: 2.1 ms
// per pass).  So every system is cut into SEGMENTS of kSegLen knots that are solved independently on a window
// that extends kSegHalo = 32 knots beyond the segment on either side, with M = 0 imposed at the window ends: the
// [1 4 1] inverse decays as 0.268^d, so the effect of that condition on the segment's own knots is below
// 0.268^32 = 5e-19 of |M| -- far under fp32 rounding (1.2e-7), i.e. the result IS the global solve to rounding
// (the fused tile kernel uses the same property with a halo of 11 and a stated 8.2e-7 bound).  A window end on the
// true end of the system is the natural condition itself.  Forward-sweep values d' of a segment's own knots go to
// M and are replaced by M in the backward sweep; those of the trailing halo stay in registers.
constexpr int kSegLen = 256;
constexpr int kSegHalo = 32;

// S2 / S3: ALONG Y, one thread per (column, segment): adjacent threads read adjacent addresses (coalesced).
// Knot q of column c is at z[q*ld + c]; M has the same layout.
// rhs_q = 6 (z_{q-1} - 2 z_q + z_{q+1}) / h^2 is formed as a difference of first differences.
constexpr int kColThreads = 128;

__global__ void __launch_bounds__(kColThreads)
thomas_col_kernel(const float* __restrict__ z, float* __restrict__ M, int n, int ncol, long long ld, float six_over_h2)
{
    const int c = blockIdx.x * kColThreads + threadIdx.x;
    if (c >= ncol) return;
    const int own0 = blockIdx.y * kSegLen, own1 = min(n, own0 + kSegLen);
    const int w0 = max(0, own0 - kSegHalo), w1 = min(n, own1 + kSegHalo);      // window [w0, w1): M = 0 at w0 and w1 - 1
    const float* zs = z + c;
    float* Ms = M + c;
    if (w0 == own0) Ms[(long long)w0 * ld] = 0.0f;
    if (w1 == own1) Ms[(long long)(w1 - 1) * ld] = 0.0f;
    if (w1 - w0 < 3) return;
    float zm = __ldg(zs + (long long)w0 * ld), z0 = __ldg(zs + (long long)(w0 + 1) * ld);
    float dprev = 0.0f;
    auto step = [&](int i) {                               // d'_q = (rhs_q - d'_{q-1}) c'_q, q counted from the window start
        const float zp = __ldg(zs + (long long)(i + 1) * ld);
        const float rhs = ((zp - z0) - (z0 - zm)) * six_over_h2;
        dprev = (rhs - dprev) * thomas_cp(i - w0 - 1);
        zm = z0;
        z0 = zp;
    };
    int i = w0 + 1;
    for (; i < own0; ++i) step(i);                         // leading halo: only the recurrence
#pragma unroll 8
    for (; i < min(own1, w1 - 1); ++i) { step(i); Ms[(long long)i * ld] = dprev; }   // own knots: d' -> M
    float dh[kSegHalo];                                    // trailing halo: d' stays in registers
#pragma unroll
    for (int h = 0; h < kSegHalo; ++h) {
        dh[h] = 0.0f;
        if (own1 + h < w1 - 1) { step(own1 + h); dh[h] = dprev; }
    }
    float mnext = 0.0f;                                    // M = 0 at the window end
#pragma unroll
    for (int h = kSegHalo - 1; h >= 0; --h)
        if (own1 + h < w1 - 1) mnext = fmaf(-thomas_cp(own1 + h - w0 - 1), mnext, dh[h]);
#pragma unroll 8
    for (int q = min(own1, w1 - 1) - 1; q >= max(own0, w0 + 1); --q) {   // M_q = d'_q - c'_q M_{q+1}
        mnext = fmaf(-thomas_cp(q - w0 - 1), mnext, Ms[(long long)q * ld]);
        Ms[(long long)q * ld] = mnext;
    }
}

// S1: ALONG X.  A thread per row would read addresses a whole row apart (uncoalesced: what made the round-1 x pass
// the slowest kernel of the path), so a warp owns 32 rows x one segment and walks the window in chunks of 32
// columns through a shared-memory tile: a chunk is read with lane = column (128 contiguous bytes per row),
// transposed in shared memory, and the recurrence runs with lane = row.  kSegLen and kSegHalo are multiples of 32:
// the leading halo is one chunk, the trailing halo one chunk whose d' stay in registers.
__global__ void __launch_bounds__(32)
thomas_row_kernel(const float* __restrict__ z, float* __restrict__ M, int n, int nrow, float six_over_h2)
{
    static_assert(kSegLen % 32 == 0 && kSegHalo == 32, "segments and halos are whole chunks");
    __shared__ float tile[32][33];
    const int lane = threadIdx.x;
    const int r0 = blockIdx.x * 32;
    const int rows = min(32, nrow - r0);
    const int own0 = blockIdx.y * kSegLen, own1 = min(n, own0 + kSegLen);
    const int w0 = max(0, own0 - kSegHalo), w1 = min(n, own1 + kSegHalo);
    const float* zb = z + (size_t)r0 * n;
    float* Mb = M + (size_t)r0 * n;
    const size_t myrow = (size_t)min(lane, rows - 1) * n;      // lane = row addressing (idle lanes shadow the last row, never store)
    const bool row_ok = lane < rows;
    if (row_ok && w0 == own0) Mb[myrow + w0] = 0.0f;
    if (row_ok && w1 == own1) Mb[myrow + w1 - 1] = 0.0f;
    if (w1 - w0 < 3) return;
    // chunk k of the window = columns w0 + 32 k ...; tile[r][j] <-> row r0 + r, column w0 + 32 k + j
    auto load_tile = [&](const float* src, int col0) {     // lane = column: coalesced rows
        const int col = col0 + lane;
#pragma unroll 8
        for (int rr = 0; rr < 32; ++rr) tile[rr][lane] = (rr < rows && col < w1) ? src[(size_t)rr * n + col] : 0.0f;
    };
    const int nchunk = (w1 - w0 + 31) / 32;
    float zm = 0.0f, z0 = 0.0f, dprev = 0.0f;
    float dh[32];                                          // d' of the last chunk swept (the trailing halo, in the end)
#pragma unroll
    for (int j = 0; j < 32; ++j) dh[j] = 0.0f;
    // ---- forward sweep, left to right.  The equation of knot i needs z_{i+1}: knot i is complete when column
    //      i + 1 arrives, so a chunk yields d' of the knots one column behind it
    for (int k = 0; k < nchunk; ++k) {
        const int col0 = w0 + 32 * k;
        load_tile(zb, col0);
        __syncwarp();
        float dcol[32];                                    // d' of knots col0 - 1 .. col0 + 30 of this lane's row
#pragma unroll
        for (int j = 0; j < 32; ++j) {
            const int q = col0 + j, i = q - 1;
            const float zp = tile[lane][j];
            float d = 0.0f;
            if (q < w1) {
                if (i >= w0 + 1 && i <= w1 - 2) {
                    const float rhs = ((zp - z0) - (z0 - zm)) * six_over_h2;
                    dprev = (rhs - dprev) * thomas_cp(i - w0 - 1);
                    d = dprev;
                }
                zm = z0;
                z0 = zp;
            }
            dcol[j] = d;
        }
        __syncwarp();
        // d' of OWN knots go to M (through the tile: lane = column stores); knots at or beyond own1 stay in dh
        if (row_ok && col0 - 1 >= own0 && col0 - 1 < own1 && col0 - 1 >= w0 + 1) Mb[myrow + col0 - 1] = dcol[0];
#pragma unroll
        for (int j = 1; j < 32; ++j) tile[lane][j - 1] = dcol[j];
        __syncwarp();
        {
            const int col = col0 + lane;                   // tile column `lane` now holds d' of knot col0 + lane (lane < 31)
            if (lane < 31 && col >= max(own0, w0 + 1) && col < min(own1, w1 - 1)) {
#pragma unroll 8
                for (int rr = 0; rr < 32; ++rr)
                    if (rr < rows) Mb[(size_t)rr * n + col] = tile[rr][lane];
            }
        }
        __syncwarp();
        if (col0 - 1 >= own1 - 1) {                        // (part of) the trailing halo: keep d' of knots col0-1 .. col0+30
#pragma unroll
            for (int j = 0; j < 32; ++j) dh[j] = dcol[j];
        }
    }
    __syncwarp();
    __threadfence_block();
    // ---- backward sweep: M = 0 at the window end; first through the trailing halo (registers: knots >= own1)
    float mnext = 0.0f;
    {
        const int base = w0 + 32 * (nchunk - 1) - 1;       // dh[j] is knot base + j (only if that chunk reached beyond own1)
#pragma unroll
        for (int j = 31; j >= 0; --j) {
            const int q = base + j;
            if (q >= own1 && q <= w1 - 2 && q >= w0 + 1) mnext = fmaf(-thomas_cp(q - w0 - 1), mnext, dh[j]);
        }
    }
    // (if the trailing halo spans two chunks' worth of knots -- it cannot: kSegHalo = 32 and chunks are aligned to w0,
    //  which is aligned to the segment grid unless w0 = 0; own1 - w0 is then a multiple of 32 as well)
    for (int k = (min(own1, w1 - 1) - 1 - w0) / 32; k >= 0 && w0 + 32 * k + 31 >= max(own0, w0 + 1); --k) {
        const int col0 = w0 + 32 * k;
        load_tile(Mb, col0);                               // the d' written above (own knots), lane = column
        __syncwarp();
        float mcol[32];
#pragma unroll
        for (int j = 31; j >= 0; --j) {
            const int q = col0 + j;
            float m = tile[lane][j];
            if (q >= max(own0, w0 + 1) && q < min(own1, w1 - 1)) {
                m = fmaf(-thomas_cp(q - w0 - 1), mnext, m);
                mnext = m;
            }
            mcol[j] = m;
        }
        __syncwarp();
#pragma unroll
        for (int j = 0; j < 32; ++j) tile[lane][j] = mcol[j];
        __syncwarp();
        {
            const int col = col0 + lane;
            if (col >= max(own0, w0 + 1) && col < min(own1, w1 - 1)) {
#pragma unroll 8
                for (int rr = 0; rr < 32; ++rr)
                    if (rr < rows) Mb[(size_t)rr * n + col] = tile[rr][lane];
            }
        }
        __syncwarp();
    }
}

// S4: a CTA owns kThreads output columns x kEvalRows output rows; a thread owns one column and marches down the
// rows.  The row entries (interval, s) are computed once per CTA; the x-direction splines X = S_x[z], Y = S_x[My] of
// the two bracketing knot rows live in registers and only the lower one is recomputed when the row enters the next
// interval (8 loads per interval instead of 16 per node), on values relative to a per-thread reference depth.
constexpr int kEvalRows = 64;

__global__ void __launch_bounds__(kThreads)
spline_eval_kernel(const float* __restrict__ z, const float* __restrict__ Mx, const float* __restrict__ My,
                   const float* __restrict__ Mxy, float* __restrict__ out, AxisMap ax, AxisMap ay,
                   float hx2_6, float hy2_6)
{
    __shared__ int2 s_row[kEvalRows];                      // (interval j or -1, float bits of s)
    const int I0 = blockIdx.y * kEvalRows;
    const int nrows = min(kEvalRows, ay.n_out - I0);
    if (threadIdx.x < kEvalRows) {
        float sv = 0.0f;
        const int j = (threadIdx.x < nrows) ? axis_locate(ay, I0 + threadIdx.x, &sv) : -1;
        s_row[threadIdx.x] = make_int2(j, __float_as_int(sv));
    }
    __syncthreads();
    const int J = blockIdx.x * kThreads + threadIdx.x;
    if (J >= ax.n_out) return;
    float t;
    const int i = axis_locate(ax, J, &t);
    const float A = 1.0f - t, B = t;
    const float Cx = (A * A * A - A) * hx2_6, Dx = (B * B * B - B) * hx2_6;
    const float qnan = __int_as_float(0x7fc00000);
    float zref = 0.0f, X0 = 0.0f, X1 = 0.0f, Y0 = 0.0f, Y1 = 0.0f;
    bool have_ref = false;
    int cur_j = -2;
    auto xspline = [&](int row, float& X, float& Y) {      // x-direction splines of knot row `row` at this column
        const size_t p = (size_t)row * ax.n_in + i;
        const float za = __ldg(z + p) - zref, zb = __ldg(z + p + 1) - zref;
        X = fmaf(A, za, fmaf(B, zb, fmaf(Cx, __ldg(Mx + p), Dx * __ldg(Mx + p + 1))));
        Y = fmaf(A, __ldg(My + p), fmaf(B, __ldg(My + p + 1), fmaf(Cx, __ldg(Mxy + p), Dx * __ldg(Mxy + p + 1))));
    };
    float* op = out + (size_t)I0 * ax.n_out + J;
    for (int r = 0; r < nrows; ++r, op += ax.n_out) {
        const int2 rw = s_row[r];
        const int j = rw.x;
        float f = qnan;
        if (i >= 0 && j >= 0) {
            if (j != cur_j) {
                if (!have_ref) { zref = __ldg(z + (size_t)j * ax.n_in + i); if (!(zref == zref)) zref = 0.0f; have_ref = true; }
                if (j == cur_j + 1) { X0 = X1; Y0 = Y1; } else xspline(j, X0, Y0);
                xspline(j + 1, X1, Y1);
                cur_j = j;
            }
            const float sv = __int_as_float(rw.y);
            const float As = 1.0f - sv;
            const float Cy = (As * As * As - As) * hy2_6, Dy = (sv * sv * sv - sv) * hy2_6;
            f = zref + fmaf(sv, X1 - X0, X0 + fmaf(Cy, Y0, Dy * Y1));
        }
        *op = f;
    }
}

}  // namespace

size_t spline_tiled_table_bytes(const grid_geom_t&, const grid_geom_t&);                                      // spline_tile.cu
int launch_spline_tiled(const float*, const grid_geom_t&, float*, const grid_geom_t&, void*, cudaStream_t, bool allow_tma);   // spline_tile.cu

// Workspace: the axis tables of the fused path, then the three second-derivative planes of the
// global-solve path.
size_t spline_workspace_bytes(const grid_geom_t& in, const grid_geom_t& out)
{
    const size_t n = (size_t)in.nx * (size_t)in.ny;
    const size_t one = (n * sizeof(float) + 255) / 256 * 256;
    return spline_tiled_table_bytes(in, out) + 3 * one;
}

int launch_spline(const float* d_in, const grid_geom_t& in, float* d_out, const grid_geom_t& out,
                  void* d_ws, cudaStream_t stream, int path)
{
    if (path != 2) {                                   // 0 = automatic, 1 / 3 = fused tiles only (3: no TMA), 2 = global solves only
        const int rc = launch_spline_tiled(d_in, in, d_out, out, d_ws, stream, path != 3);
        if (rc != 1) return rc;
        if (path == 1 || path == 3) return BATHY_ERR_GEOMETRY;
    }
    const AxisMap ax = axis_x(in, out), ay = axis_y(in, out);
    const size_t n = (size_t)in.nx * (size_t)in.ny;
    const size_t one = (n * sizeof(float) + 255) / 256 * 256;
    char* planes = static_cast<char*>(d_ws) + spline_tiled_table_bytes(in, out);
    float* Mx = reinterpret_cast<float*>(planes);
    float* My = reinterpret_cast<float*>(planes + one);
    float* Mxy = reinterpret_cast<float*>(planes + 2 * one);
    const float hx = in.dx, hy = in.dy;
    const float six_hx2 = (float)(6.0 / ((double)hx * (double)hx)), six_hy2 = (float)(6.0 / ((double)hy * (double)hy));
    // S1: rows (along x): a warp per 32 rows, transposed through shared memory
    const int segx = (in.nx + kSegLen - 1) / kSegLen, segy = (in.ny + kSegLen - 1) / kSegLen;
    if (segx > 65535 || segy > 65535) return BATHY_ERR_SIZE;
    thomas_row_kernel<<<dim3((in.ny + 31) / 32, segx), 32, 0, stream>>>(d_in, Mx, in.nx, in.ny, six_hx2);
    // S2: columns (along y): a thread per column, coalesced across threads
    thomas_col_kernel<<<dim3((in.nx + kColThreads - 1) / kColThreads, segy), kColThreads, 0, stream>>>(d_in, My, in.ny, in.nx, in.nx, six_hy2);
    // S3: columns of Mx
    thomas_col_kernel<<<dim3((in.nx + kColThreads - 1) / kColThreads, segy), kColThreads, 0, stream>>>(Mx, Mxy, in.ny, in.nx, in.nx, six_hy2);
    const long long bands = ((long long)out.ny + kEvalRows - 1) / kEvalRows;
    if (bands > 65535) return BATHY_ERR_SIZE;
    dim3 grid((out.nx + kThreads - 1) / kThreads, (unsigned)bands);
    spline_eval_kernel<<<grid, kThreads, 0, stream>>>(d_in, Mx, My, Mxy, d_out, ax, ay,
                                                      (float)((double)hx * hx / 6.0), (float)((double)hy * hy / 6.0));
    count_launch(4);
    return launch_status();
}

}  // namespace bathy
