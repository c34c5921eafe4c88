// bilinear.cu -- interp_bilinear (formula at L132).
//
// HBM-bound: the output write stream is 80-94 % of the bytes.  One CTA owns a TW x TH output tile.
// It stages the covering input tile (+1 sample halo) in shared memory, minus a tile reference
// depth z_ref so that the fp32 arithmetic runs on small numbers (|z| ~ 5000 m, ulp 4.9e-4 m), and
// every thread marches down TH output rows for CPT columns that are lane-contiguous (column =
// tile_x0 + e*THREADS + tid), so that every store instruction of a warp writes 128 contiguous
// bytes whatever the alignment of the output row (nx_out = 8191 and 4093 are odd, so rows are not
// 16-byte aligned and float4 stores would need a per-row shift that breaks the row-to-row reuse).
// The horizontal interpolants H(j, column) are computed once per input row and reused for all
// output rows that fall between input rows j and j+1.
#include "common.cuh"

namespace bathy {

namespace {

constexpr int kThreads = 256;

template <int CPT, int TH>
__global__ void __launch_bounds__(kThreads)
bilinear_tiled_kernel(const float* __restrict__ in, float* __restrict__ out,
                      AxisMap ax, AxisMap ay, int fw_cap, int fh_cap)
{
    constexpr int TW = CPT * kThreads;
    extern __shared__ float s_tile[];                 // [fh][fw] input samples minus z_ref
    __shared__ int   s_rowj[TH];                      // input row of each output row (-1: outside)
    __shared__ float s_rows[TH];                      // local coordinate s of each output row
    __shared__ int   s_bounds[4];                     // i_lo, i_hi, j_lo, j_hi (sample indices)

    const int tid = threadIdx.x;
    const int J0 = blockIdx.x * TW;
    const int I0 = blockIdx.y * TH;
    const int Jlast = min(J0 + TW, ax.n_out) - 1;
    const int Ilast = min(I0 + TH, ay.n_out) - 1;

    if (tid == 0) s_bounds[0] = axis_clamped(ax, J0);
    if (tid == 1) s_bounds[1] = axis_clamped(ax, Jlast) + 1;
    if (tid == 2) s_bounds[2] = axis_clamped(ay, I0);
    if (tid == 3) s_bounds[3] = axis_clamped(ay, Ilast) + 1;
    if (tid >= 32 && tid < 32 + TH) {
        float s;
        int r = tid - 32;
        int j = (I0 + r <= Ilast) ? axis_locate(ay, I0 + r, &s) : -1;
        s_rowj[r] = j;
        s_rows[r] = (j < 0) ? 0.0f : s;
    }
    // this thread's columns
    int   ci[CPT];
    float ct[CPT];
#pragma unroll
    for (int e = 0; e < CPT; ++e) {
        int J = J0 + e * kThreads + tid;
        ci[e] = (J <= Jlast) ? axis_locate(ax, J, &ct[e]) : -1;
        if (ci[e] < 0) ct[e] = 0.0f;
    }
    __syncthreads();
    const int i_lo = s_bounds[0], i_hi = s_bounds[1], j_lo = s_bounds[2], j_hi = s_bounds[3];
    const int fw = i_hi - i_lo + 1, fh = j_hi - j_lo + 1;
    (void)fw_cap; (void)fh_cap;

    float zref = __ldg(in + (size_t)j_lo * ax.n_in + i_lo);
    if (!isfinite(zref)) zref = 0.0f;
    {
        const int warp = tid >> 5, lane = tid & 31;
        for (int r = warp; r < fh; r += kThreads / 32) {
            const float* src = in + (size_t)(j_lo + r) * ax.n_in + i_lo;
            float* dst = s_tile + r * fw;
            for (int c = lane; c < fw; c += 32) dst[c] = __ldg(src + c) - zref;
        }
    }
    __syncthreads();

#pragma unroll
    for (int e = 0; e < CPT; ++e) ci[e] = (ci[e] < 0) ? -1 : ci[e] - i_lo;

    float hlo[CPT], hhi[CPT];
#pragma unroll
    for (int e = 0; e < CPT; ++e) hlo[e] = hhi[e] = 0.0f;
    int cur_j = -2;
    const float qnan = __int_as_float(0x7fc00000);
    for (int r = 0; r < TH; ++r) {
        const int I = I0 + r;
        if (I > Ilast) break;
        const int j = s_rowj[r];
        const float s = s_rows[r];
        if (j >= 0 && j != cur_j) {                    // CTA-uniform branch: a new input row pair
            const float* row0 = s_tile + (j - j_lo) * fw;
            const float* row1 = row0 + fw;
            const bool step = (j == cur_j + 1);        // the old upper row is the new lower row
#pragma unroll
            for (int e = 0; e < CPT; ++e) {
                const int c = max(ci[e], 0);
                hlo[e] = step ? hhi[e] : fmaf(ct[e], row0[c + 1] - row0[c], row0[c]);
                hhi[e] = fmaf(ct[e], row1[c + 1] - row1[c], row1[c]);
            }
            cur_j = j;
        }
        float* orow = out + (size_t)I * ax.n_out;
#pragma unroll
        for (int e = 0; e < CPT; ++e) {
            const int J = J0 + e * kThreads + tid;
            if (J <= Jlast) {
                float f = fmaf(s, hhi[e] - hlo[e], hlo[e]) + zref;
                if (ci[e] < 0 || j < 0) f = qnan;
                orow[J] = f;
            }
        }
    }
}

// Any geometry (including strong down-sampling, where a tile's input footprint does not fit in
// shared memory): one thread per output node, corners through the read-only path.
__global__ void __launch_bounds__(kThreads)
bilinear_gather_kernel(const float* __restrict__ in, float* __restrict__ out, AxisMap ax, AxisMap ay)
{
    const int J = blockIdx.x * kThreads + threadIdx.x;
    if (J >= ax.n_out) return;
    float t, s;
    const int i = axis_locate(ax, J, &t);
    for (int I = blockIdx.y; I < ay.n_out; I += gridDim.y) {
        const int j = axis_locate(ay, I, &s);
        float f = __int_as_float(0x7fc00000);
        if (i >= 0 && j >= 0) {
            const float* p = in + (size_t)j * ax.n_in + i;
            const float q11 = __ldg(p), q21 = __ldg(p + 1), q12 = __ldg(p + ax.n_in), q22 = __ldg(p + ax.n_in + 1);
            const float lo = fmaf(t, q21 - q11, q11);
            const float hi = fmaf(t, q22 - q12, q12);
            f = fmaf(s, hi - lo, lo);
        }
        out[(size_t)I * ax.n_out + J] = f;
    }
}

}  // namespace

int launch_bilinear(const float* d_in, const grid_geom_t& in, float* d_out, const grid_geom_t& out,
                    cudaStream_t stream)
{
    const AxisMap ax = axis_x(in, out), ay = axis_y(in, out);
    constexpr int CPT = 2, TH = 16, TW = CPT * kThreads;
    const long long fw = footprint_bound(ax, TW), fh = footprint_bound(ay, TH);
    const long long smem = fw * fh * (long long)sizeof(float);
    if (smem <= 160 * 1024 && (out.ny + TH - 1) / TH <= 65535) {
        static bool attr_set = false;
        if (!attr_set) {
            BATHY_CUDA_TRY(cudaFuncSetAttribute(bilinear_tiled_kernel<CPT, TH>,
                                                cudaFuncAttributeMaxDynamicSharedMemorySize, 160 * 1024));
            attr_set = true;
        }
        dim3 grid((out.nx + TW - 1) / TW, (out.ny + TH - 1) / TH);
        bilinear_tiled_kernel<CPT, TH><<<grid, kThreads, (size_t)smem, stream>>>(d_in, d_out, ax, ay, (int)fw, (int)fh);
    } else {
        dim3 grid((out.nx + kThreads - 1) / kThreads, out.ny < 65535 ? out.ny : 65535);
        bilinear_gather_kernel<<<grid, kThreads, 0, stream>>>(d_in, d_out, ax, ay);
    }
    count_launch();
    return launch_status();
}

}  // namespace bathy
