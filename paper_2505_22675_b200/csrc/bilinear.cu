// bilinear.cu -- interp_bilinear (formula at L132).
//
// HBM-bound (the output write stream is 80-94 % of the bytes) -- and, at ~1e12 nodes/s, issue-bound
// unless a node costs fewer than ~10 instructions.  One CTA owns a TW x TH output tile.  It stages
// the covering input tile (+1 sample halo) in shared memory, minus a tile reference depth z_ref so
// that the fp32 arithmetic runs on small numbers (|z| ~ 5000 m, ulp 4.9e-4 m).  A thread owns CPT
// columns that are lane-contiguous inside its warp (column = tile_x0 + warp*32*CPT + e*32 + lane),
// so every store instruction of a warp writes 128 contiguous bytes whatever the alignment of the
// output row (nx_out = 8191 and 4093 are odd: rows are not 16-byte aligned, and a per-row shift to
// float4 alignment would break the row-to-row register reuse below).  The thread marches down the TH
// rows: the horizontal interpolants of the two bracketing input rows live in registers and are
// recomputed only when the output row enters a new input interval, so a node costs half a packed FMA,
// half a packed add (z_ref, added last) and one store plus its share of the per-row and per-interval work.
#include "common.cuh"
#include "tma.cuh"
#include <string.h>

namespace bathy {

namespace {

constexpr int kThreads = 256;

constexpr int kBoxW = 64;                            // columns of one TMA box of the footprint

// TMA = true (input rows 16-byte aligned): the footprint arrives as ceil(width / 64) TMA boxes of 64 columns x box_h
// rows (cp.async.bulk.tensor.2d: one elected thread, no per-thread address arithmetic, no LSU wavefronts), box b at
// s_tile + b * box_h * 64; sample (row r, column c) of the footprint sits at (c / 64) * box_h * 64 + r * 64 + c % 64.
// TMA = false: cp.async into [fh][pitch] (common.cuh stage_footprint).
template <int CPT, int TH, bool TMA>
__global__ void __launch_bounds__(kThreads)
bilinear_tiled_kernel(const float* __restrict__ in, float* __restrict__ out, AxisMap ax, AxisMap ay,
                      const __grid_constant__ CUtensorMap tmap, int box_h)
{
    constexpr int TW = CPT * kThreads;
    extern __shared__ __align__(128) float s_tile[];  // raw input samples of the tile's footprint
    __shared__ __align__(8) unsigned long long s_bar; // mbarrier of the TMA loads
    __shared__ int2  s_row[TH];                       // (input row j or -1, float bits of s) per output row
    __shared__ int   s_bounds[4];                     // i_lo, i_hi, j_lo, j_hi (sample indices)

    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int J0 = blockIdx.x * TW;
    const int I0 = blockIdx.y * TH;
    const int Jlast = min(J0 + TW, ax.n_out) - 1;
    const int Ilast = min(I0 + TH, ay.n_out) - 1;
    const int nrows = Ilast - I0 + 1;

    if (tid == 0) s_bounds[0] = axis_clamped(ax, J0);
    if (tid == 1) s_bounds[1] = axis_clamped(ax, Jlast) + 1;
    if (tid == 2) s_bounds[2] = axis_clamped(ay, I0);
    if (tid == 3) s_bounds[3] = axis_clamped(ay, Ilast) + 1;
    if (tid >= 32 && tid < 32 + TH) {
        float s = 0.0f;
        const int r = tid - 32;
        const int j = (r < nrows) ? axis_locate(ay, I0 + r, &s) : -1;
        s_row[r] = make_int2(j, __float_as_int(j < 0 ? 0.0f : s));
    }
    __syncthreads();
    const int i_lo = s_bounds[0], i_hi = s_bounds[1], j_lo = s_bounds[2], j_hi = s_bounds[3];
    const int fw = i_hi - i_lo + 1, fh = j_hi - j_lo + 1;

    // The footprint goes global -> shared by cp.async, all of it in flight at once (16-byte vectors
    // from the aligned column at or before i_lo when the rows are 16-byte aligned); the double-precision
    // column maps below are computed while it streams in.
    const int offx = i_lo & 3;
    const int pitch = TMA ? kBoxW : stage_pitch(fw);  // floats between consecutive footprint rows
    const unsigned bar = (unsigned)__cvta_generic_to_shared(&s_bar);
    if (TMA) {
        if (tid == 0) {
            const int nb = (offx + fw + kBoxW - 1) / kBoxW;
            const unsigned box_bytes = (unsigned)(box_h * kBoxW * sizeof(float));
            mbar_init(bar, 1);
            mbar_expect(bar, box_bytes * nb);
            for (int b = 0; b < nb; ++b)
                tma_issue_2d((unsigned)__cvta_generic_to_shared(s_tile) + b * box_bytes, &tmap, (i_lo & ~3) + b * kBoxW, j_lo, bar);
        }
    } else {
        stage_footprint(in, ax.n_in, i_lo, j_lo, fw, fh, s_tile, tid, kThreads);
        asm volatile("cp.async.commit_group;" ::: "memory");
    }
    float zref = __ldg(in + (size_t)j_lo * ax.n_in + i_lo);
    if (!isfinite(zref)) zref = 0.0f;

    // this thread's columns: interval index and local coordinate
    const int Jt = J0 + warp * (32 * CPT) + lane;     // column of e = 0
    int   ci[CPT];
    float ct[CPT];
#pragma unroll
    for (int e = 0; e < CPT; ++e) {
        const int J = Jt + 32 * e;
        ct[e] = 0.0f;
        ci[e] = (J <= Jlast) ? axis_locate(ax, J, &ct[e]) : -1;
    }
    if (TMA) {
        __syncthreads();                                  // the barrier is initialised
        mbar_wait(bar, 0);                                // the footprint has landed
    } else {
        asm volatile("cp.async.wait_group 0;" ::: "memory");
        __syncthreads();
    }

    const float qnan = __int_as_float(0x7fc00000);
    static_assert(CPT % 2 == 0, "columns are processed as fp32x2 pairs");
    bool cok[CPT];                                    // column is inside the tile (store predicate)
    float cz[CPT];                                    // z_ref, or NaN for a column outside the input extent
    int   cofl[CPT], cofr[CPT];                       // offsets of the interval's left / right sample from the start of its footprint row
#pragma unroll
    for (int e = 0; e < CPT; ++e) {
        cok[e] = (Jt + 32 * e) <= Jlast;
        cz[e] = (ci[e] < 0) ? qnan : zref;
        const int c = max(ci[e] - i_lo, 0) + offx;
        if (TMA) {
            const int bs = box_h * kBoxW;
            cofl[e] = (c / kBoxW) * bs + (c % kBoxW);
            cofr[e] = ((c + 1) / kBoxW) * bs + ((c + 1) % kBoxW);
        } else {
            cofl[e] = c;
            cofr[e] = c + 1;
        }
    }

    // Two columns to a 64-bit register pair: a node is half a packed FMA (FFMA2) and a store.
    u64 hlo2[CPT / 2], hd2[CPT / 2];                  // lower interpolant (relative to z_ref) and (upper - lower)
#pragma unroll
    for (int p = 0; p < CPT / 2; ++p) hlo2[p] = hd2[p] = pack2(0.0f, 0.0f);
    int cur_j = -2;
    float* orow = out + (size_t)I0 * ax.n_out + Jt;
    // interval change: the horizontal interpolants of input row `row` at this thread's columns, on
    // (sample - z_ref) so that the arithmetic runs on small numbers (|z| ~ 5000 m, ulp 4.9e-4 m),
    // two columns at a time in packed arithmetic
    const u64 nzref2 = pack2(-zref, -zref), neg1 = pack2(-1.0f, -1.0f);
    const u64 ct2[CPT / 2] = {pack2(ct[0], ct[1]), pack2(ct[2], ct[3])};
    const u64 cz2[CPT / 2] = {pack2(cz[0], cz[1]), pack2(cz[2], cz[3])};
    static_assert(CPT == 4, "column pairs are written out for CPT = 4");
    auto hrow = [&](const float* row, u64* h2) {
#pragma unroll
        for (int p = 0; p < CPT / 2; ++p) {
            const u64 l = pack2(row[cofl[2 * p]], row[cofl[2 * p + 1]]), r = pack2(row[cofr[2 * p]], row[cofr[2 * p + 1]]);
            h2[p] = ffma2(ct2[p], ffma2(l, neg1, r), fadd2(l, nzref2));
        }
    };
    u64 hhi2[CPT / 2] = {pack2(0.0f, 0.0f), pack2(0.0f, 0.0f)};
    // interior tile (CTA-uniform): every column inside the tile, every row inside the input extent
    const bool full = (J0 + TW - 1 <= Jlast) && s_row[0].x >= 0 && s_row[nrows - 1].x >= 0;
    int2 rw_next = s_row[0];
    for (int r = 0; r < nrows; ++r, orow += ax.n_out) {
        const int2 rw = rw_next;
        rw_next = s_row[min(r + 1, TH - 1)];          // the next row's entry is in flight while this row is stored
        const int j = rw.x;
        const float s = __int_as_float(rw.y);
        if (!full && j < 0) {                          // CTA-uniform: row outside the input extent
#pragma unroll
            for (int e = 0; e < CPT; ++e) if (cok[e]) orow[32 * e] = qnan;
            continue;
        }
        if (j != cur_j) {                              // CTA-uniform: a new input row pair
            const float* row0 = s_tile + (j - j_lo) * pitch;
            u64 lo2[CPT / 2];
            if (j == cur_j + 1) {                      // the old upper row is the new lower row
#pragma unroll
                for (int p = 0; p < CPT / 2; ++p) lo2[p] = hhi2[p];
            } else {
                hrow(row0, lo2);
            }
            hrow(row0 + pitch, hhi2);
#pragma unroll
            for (int p = 0; p < CPT / 2; ++p) {
                hd2[p] = ffma2(lo2[p], neg1, hhi2[p]);
                hlo2[p] = lo2[p];
            }
            cur_j = j;
        }
        const u64 s2 = pack2(s, s);
        if (full) {
#pragma unroll
            for (int p = 0; p < CPT / 2; ++p) {
                // z_ref is added LAST: the only rounding at full magnitude (0.5 ulp of the depth)
                const u64 o = fadd2(ffma2(s2, hd2[p], hlo2[p]), cz2[p]);
                orow[64 * p] = lo_of(o);
                orow[64 * p + 32] = hi_of(o);
            }
        } else {
#pragma unroll
            for (int p = 0; p < CPT / 2; ++p) {
                const u64 o = fadd2(ffma2(s2, hd2[p], hlo2[p]), cz2[p]);
                if (cok[2 * p]) orow[64 * p] = lo_of(o);
                if (cok[2 * p + 1]) orow[64 * p + 32] = hi_of(o);
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
            // on differences to q11, which is added last: one rounding at full magnitude
            const float a = q21 - q11, b = q12 - q11, c = q22 - q11;
            const float lo = t * a;
            const float hi = fmaf(t, c - b, b);
            f = q11 + fmaf(s, hi - lo, lo);
        }
        out[(size_t)I * ax.n_out + J] = f;
    }
}

}  // namespace

std::atomic<bool> g_bilinear_tma{true};   // A/B switch (bathy_set_spline_path(3) turns the TMA staging of the grid kernels off)

int launch_bilinear(const float* d_in, const grid_geom_t& in, float* d_out, const grid_geom_t& out,
                    cudaStream_t stream)
{
    const AxisMap ax = axis_x(in, out), ay = axis_y(in, out);
    constexpr int CPT = 4, TH = 32, TW = CPT * kThreads;
    const long long fw = footprint_bound(ax, TW), fh = footprint_bound(ay, TH);
    long long smem = ((fw + 6) & ~3LL) * fh * (long long)sizeof(float);
    // TMA staging when the input rows are 16-byte aligned and the box fits (box height <= 256): the footprint as
    // boxes of 64 columns x fh rows
    CUtensorMap tmap;
    memset(&tmap, 0, sizeof(tmap));
    const long long nbox = (fw + 3 + kBoxW - 1) / kBoxW;
    const long long smem_tma = nbox * fh * kBoxW * (long long)sizeof(float);
    bool use_tma = g_bilinear_tma.load(std::memory_order_relaxed) && (reinterpret_cast<uintptr_t>(d_in) & 15) == 0 && (in.nx & 3) == 0 && fh <= 256 &&
                   smem_tma <= 160 * 1024 && in.nx >= kBoxW;
    if (use_tma) use_tma = tensor_map_2d(&tmap, d_in, in.nx, in.ny, kBoxW, (int)fh) == BATHY_OK;
    if (use_tma) smem = smem_tma;
    if (smem <= 160 * 1024 && (out.ny + TH - 1) / TH <= 65535) {
        static DeviceOnce once;
        const int rc = once_per_device(once, []() -> int {
            BATHY_CUDA_TRY(cudaFuncSetAttribute(bilinear_tiled_kernel<CPT, TH, true>,
                                                cudaFuncAttributeMaxDynamicSharedMemorySize, 160 * 1024));
            BATHY_CUDA_TRY(cudaFuncSetAttribute(bilinear_tiled_kernel<CPT, TH, false>,
                                                cudaFuncAttributeMaxDynamicSharedMemorySize, 160 * 1024));
            return (int)BATHY_OK;
        });
        if (rc) return rc;
        dim3 grid((out.nx + TW - 1) / TW, (out.ny + TH - 1) / TH);
        if (use_tma) bilinear_tiled_kernel<CPT, TH, true><<<grid, kThreads, (size_t)smem, stream>>>(d_in, d_out, ax, ay, tmap, (int)fh);
        else         bilinear_tiled_kernel<CPT, TH, false><<<grid, kThreads, (size_t)smem, stream>>>(d_in, d_out, ax, ay, tmap, 0);
    } else {
        dim3 grid((out.nx + kThreads - 1) / kThreads, out.ny < 65535 ? out.ny : 65535);
        bilinear_gather_kernel<<<grid, kThreads, 0, stream>>>(d_in, d_out, ax, ay);
    }
    count_launch();
    return launch_status();
}

}  // namespace bathy
