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

// Thomas solve of nsys independent systems of n knots each; knot q of system s is at
// z[s*sys_stride + q*elem_stride]; M has the same layout.  M_0 = M_{n-1} = 0.
// rhs_q = 6 (z_{q-1} - 2 z_q + z_{q+1}) / h^2 is formed as a difference of first differences.
__global__ void __launch_bounds__(kThreads)
thomas_kernel(const float* __restrict__ z, float* __restrict__ M, int n, int nsys,
              long long elem_stride, long long sys_stride, float six_over_h2)
{
    const int s = blockIdx.x * kThreads + threadIdx.x;
    if (s >= nsys) return;
    const float* zs = z + (long long)s * sys_stride;
    float* Ms = M + (long long)s * sys_stride;
    Ms[0] = 0.0f;
    Ms[(long long)(n - 1) * elem_stride] = 0.0f;
    if (n < 3) return;
    float zm = zs[0], z0 = zs[elem_stride];
    float dprev = 0.0f;
    for (int i = 1; i <= n - 2; ++i) {                     // forward sweep: d'_q = (rhs_q - d'_{q-1}) c'_q
        const float zp = zs[(long long)(i + 1) * elem_stride];
        const float rhs = ((zp - z0) - (z0 - zm)) * six_over_h2;
        dprev = (rhs - dprev) * thomas_cp(i - 1);
        Ms[(long long)i * elem_stride] = dprev;
        zm = z0;
        z0 = zp;
    }
    float mnext = dprev;                                   // M_{n-2} = d'_{n-2}
    for (int i = n - 3; i >= 1; --i) {                     // back substitution: M_q = d'_q - c'_q M_{q+1}
        mnext = fmaf(-thomas_cp(i - 1), mnext, Ms[(long long)i * elem_stride]);
        Ms[(long long)i * elem_stride] = mnext;
    }
}

// S4: one thread per output column, marching over output rows.
__global__ void __launch_bounds__(kThreads)
spline_eval_kernel(const float* __restrict__ z, const float* __restrict__ Mx, const float* __restrict__ My,
                   const float* __restrict__ Mxy, float* __restrict__ out, AxisMap ax, AxisMap ay,
                   float hx2_6, float hy2_6)
{
    const int J = blockIdx.x * kThreads + threadIdx.x;
    if (J >= ax.n_out) return;
    float t, s;
    const int i = axis_locate(ax, J, &t);
    const float A = 1.0f - t, B = t;
    const float Cx = (A * A * A - A) * hx2_6, Dx = (B * B * B - B) * hx2_6;
    const float qnan = __int_as_float(0x7fc00000);
    for (int I = blockIdx.y; I < ay.n_out; I += gridDim.y) {
        const int j = axis_locate(ay, I, &s);
        float f = qnan;
        if (i >= 0 && j >= 0) {
            const size_t p0 = (size_t)j * ax.n_in + i, p1 = p0 + ax.n_in;
            const float zref = __ldg(z + p0);
            // x-spline of the two bracketing rows (values relative to zref) ...
            const float X0 = fmaf(B, __ldg(z + p0 + 1) - zref, fmaf(Cx, __ldg(Mx + p0), Dx * __ldg(Mx + p0 + 1)));
            const float z01 = __ldg(z + p1) - zref;
            const float X1 = z01 + fmaf(B, (__ldg(z + p1 + 1) - zref) - z01, fmaf(Cx, __ldg(Mx + p1), Dx * __ldg(Mx + p1 + 1)));
            // ... and of their second derivatives in y
            const float Y0 = fmaf(A, __ldg(My + p0), fmaf(B, __ldg(My + p0 + 1), fmaf(Cx, __ldg(Mxy + p0), Dx * __ldg(Mxy + p0 + 1))));
            const float Y1 = fmaf(A, __ldg(My + p1), fmaf(B, __ldg(My + p1 + 1), fmaf(Cx, __ldg(Mxy + p1), Dx * __ldg(Mxy + p1 + 1))));
            const float As = 1.0f - s, Bs = s;
            const float Cy = (As * As * As - As) * hy2_6, Dy = (Bs * Bs * Bs - Bs) * hy2_6;
            f = zref + fmaf(Bs, X1 - X0, X0 + fmaf(Cy, Y0, Dy * Y1));
        }
        out[(size_t)I * ax.n_out + J] = f;
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
    // S1: rows (along x): system = row, elements contiguous
    thomas_kernel<<<(in.ny + kThreads - 1) / kThreads, kThreads, 0, stream>>>(d_in, Mx, in.nx, in.ny, 1, in.nx, six_hx2);
    // S2: columns (along y): system = column, coalesced across threads
    thomas_kernel<<<(in.nx + kThreads - 1) / kThreads, kThreads, 0, stream>>>(d_in, My, in.ny, in.nx, in.nx, 1, six_hy2);
    // S3: columns of Mx
    thomas_kernel<<<(in.nx + kThreads - 1) / kThreads, kThreads, 0, stream>>>(Mx, Mxy, in.ny, in.nx, in.nx, 1, six_hy2);
    dim3 grid((out.nx + kThreads - 1) / kThreads, out.ny < 65535 ? out.ny : 65535);
    spline_eval_kernel<<<grid, kThreads, 0, stream>>>(d_in, Mx, My, Mxy, d_out, ax, ay,
                                                      (float)((double)hx * hx / 6.0), (float)((double)hy * hy / 6.0));
    count_launch(4);
    return launch_status();
}

}  // namespace bathy
