// catmull_rom.cu -- interp_catmull_rom: the paper's own "cubic spline" (formula at
// L140).  4 x 4 neighbours, x on each of the 4 rows, then y; a node with one of
// its 16 neighbours outside the grid or NaN falls back to bilinear (sense fixed by L171;
// DESIGN.md readings CR1-CR3).
//
// Same skeleton as bilinear.cu: one CTA owns a TW x TH output tile, stages the covering input
// footprint (+2 samples of halo) in shared memory by cp.async, a thread owns CPT lane-contiguous
// columns and marches down the rows.  Per column it keeps, for the 4 input rows j-1 .. j+2 around the
// current row interval, the x-direction cubic X and the x-direction linear interpolant L (for the
// fallback), all on (sample - z_ref).  When the output row enters the next interval the window of
// rows shifts by one and ONE new row is evaluated (4 shared loads, 6 FMA); a node then costs the
// 4-term y cubic, the 1-term y lerp and a select.
// The printed polynomial is evaluated as weights w_k(t) (they sum to 1, so subtracting z_ref is exact
// algebra):  w0 = (-t + 2t^2 - t^3)/2, w1 = (2 - 5t^2 + 3t^3)/2, w2 = (t + 4t^2 - 3t^3)/2,
// w3 = (-t^2 + t^3)/2.
#include "common.cuh"
#include "tma.cuh"
#include <string.h>

namespace bathy {

namespace {

constexpr int kThreads = 256;

__device__ __forceinline__ float4 cr_weights(float t)
{
    const float t2 = t * t, t3 = t2 * t;
    return make_float4(0.5f * (-t + 2.0f * t2 - t3), 0.5f * (2.0f - 5.0f * t2 + 3.0f * t3),
                       0.5f * (t + 4.0f * t2 - 3.0f * t3), 0.5f * (-t2 + t3));
}

constexpr int kBoxW = 64;                            // columns of one TMA box of the footprint (layout: see bilinear.cu)

template <int CPT, int TH, bool TMA>
__global__ void __launch_bounds__(kThreads, 3)
catmull_rom_tiled_kernel(const float* __restrict__ in, float* __restrict__ out, AxisMap ax, AxisMap ay,
                         const __grid_constant__ CUtensorMap tmap, int box_h)
{
    constexpr int TW = CPT * kThreads;
    extern __shared__ __align__(128) float s_tile[];  // raw input samples of the tile's footprint
    __shared__ __align__(8) unsigned long long s_bar; // mbarrier of the TMA loads
    __shared__ float4 s_wy[TH];                       // y weights of the output row
    __shared__ int2   s_row[TH];                      // (input row j or -1, float bits of s) per output row
    __shared__ int    s_bounds[4];                    // i_lo, i_hi, j_lo, j_hi (interval bounds of the tile)

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
        s_wy[r] = cr_weights(j < 0 ? 0.0f : s);
    }
    __syncthreads();
    // footprint: the intervals' samples plus one more sample on every side, clipped to the grid
    const int fi0 = max(s_bounds[0] - 1, 0), fi1 = min(s_bounds[1] + 1, ax.n_in - 1);
    const int fj0 = max(s_bounds[2] - 1, 0), fj1 = min(s_bounds[3] + 1, ay.n_in - 1);
    const int fw = fi1 - fi0 + 1, fh = fj1 - fj0 + 1;

    const int offx = fi0 & 3;
    const int pitch = TMA ? kBoxW : stage_pitch(fw);  // floats between consecutive footprint rows
    const int bs = box_h * kBoxW;                     // floats between consecutive boxes
    const unsigned bar = (unsigned)__cvta_generic_to_shared(&s_bar);
    if (TMA) {
        if (tid == 0) {
            const int nb = (offx + fw + kBoxW - 1) / kBoxW;
            const unsigned box_bytes = (unsigned)(bs * sizeof(float));
            mbar_init(bar, 1);
            mbar_expect(bar, box_bytes * nb);
            for (int b = 0; b < nb; ++b)
                tma_issue_2d((unsigned)__cvta_generic_to_shared(s_tile) + b * box_bytes, &tmap, (fi0 & ~3) + b * kBoxW, fj0, bar);
        }
    } else {
        stage_footprint(in, ax.n_in, fi0, fj0, fw, fh, s_tile, tid, kThreads);
        asm volatile("cp.async.commit_group;" ::: "memory");
    }
    // byte offset of footprint column c (counted from the aligned start) inside a footprint row
    auto boff = [&](int c) { return TMA ? 4u * (unsigned)((c / kBoxW) * bs + (c % kBoxW)) : 4u * (unsigned)c; };
    float zref = __ldg(in + (size_t)fj0 * ax.n_in + fi0);
    if (!isfinite(zref)) zref = 0.0f;

    // this thread's columns
    const int Jt = J0 + warp * (32 * CPT) + lane;     // column of e = 0
    bool cok[CPT], c4ok[CPT];                         // column inside the tile / has its 4 x neighbours in the grid
    float ct[CPT], cnan[CPT];
    float cw0[CPT], cw2[CPT], cw3[CPT];               // x weights of P0, P2, P3 (P1's is 1 minus their sum)
    unsigned o1[CPT], o0[CPT], o2[CPT], o3[CPT];      // byte offsets of P1, P0, P2, P3 in a footprint row (P0 and P3 clamped
                                                      // into the footprint): a shared-memory address is one add
    const float qnan = __int_as_float(0x7fc00000);
#pragma unroll
    for (int e = 0; e < CPT; ++e) {
        const int J = Jt + 32 * e;
        cok[e] = J <= Jlast;
        ct[e] = 0.0f;
        const int i = cok[e] ? axis_locate(ax, J, &ct[e]) : -1;
        cnan[e] = (i < 0) ? qnan : 0.0f;
        const int ic = (i < 0) ? fi0 : i;             // a column outside the extent still reads inside the footprint
        c4ok[e] = (i >= 1) && (i + 2 <= ax.n_in - 1);
        const float4 w = cr_weights(ct[e]);
        cw0[e] = w.x; cw2[e] = w.z; cw3[e] = w.w;
        const int c1 = min(max(ic, fi0), fi1 - 1) - fi0 + offx;
        o1[e] = boff(c1);
        o2[e] = boff(c1 + 1);
        o0[e] = (c1 - 1 >= offx) ? boff(c1 - 1) : o1[e];
        o3[e] = (c1 + 2 <= fi1 - fi0 + offx) ? boff(c1 + 2) : o2[e];
    }
    const unsigned tile_sa = (unsigned)__cvta_generic_to_shared(s_tile);
    auto lds = [](unsigned a) { float v; asm volatile("ld.shared.f32 %0, [%1];" : "=f"(v) : "r"(a) : "memory"); return v; };
    if (TMA) {
        __syncthreads();                                  // the barrier is initialised
        mbar_wait(bar, 0);                                // the footprint has landed
    } else {
        asm volatile("cp.async.wait_group 0;" ::: "memory");
        __syncthreads();
    }

    // x cubic of input row jrow at this thread's columns, on (sample - z_ref), two columns to a pair.  With
    // w1 = 1 - w0 - w2 - w3 the cubic is P1 + w0 (P0 - P1) + w2 (P2 - P1) + w3 (P3 - P1): differences of
    // neighbouring samples, no weight ever multiplies a 5000 m depth.  A column that lacks one of its 4 x
    // neighbours subtracts NaN instead of z_ref, a row outside the grid is NaN: X is NaN exactly when one
    // of the row's 4 neighbours is missing.
    static_assert(CPT == 4, "column pairs are written out for CPT = 4");
    float zrc[CPT];
#pragma unroll
    for (int e = 0; e < CPT; ++e) zrc[e] = c4ok[e] ? zref : qnan;
    const u64 w0x[CPT / 2] = {pack2(cw0[0], cw0[1]), pack2(cw0[2], cw0[3])};
    const u64 w2x[CPT / 2] = {pack2(cw2[0], cw2[1]), pack2(cw2[2], cw2[3])};
    const u64 w3x[CPT / 2] = {pack2(cw3[0], cw3[1]), pack2(cw3[2], cw3[3])};
    const u64 nzr[CPT / 2] = {pack2(-zrc[0], -zrc[1]), pack2(-zrc[2], -zrc[3])};
    const u64 neg1 = pack2(-1.0f, -1.0f);
    // returns true (warp-uniform) when some column of the warp got a NaN in this row
    auto row_eval = [&](int jrow, u64* X2) -> bool {
        if (jrow < 0 || jrow > ay.n_in - 1) {          // CTA-uniform
            X2[0] = X2[1] = pack2(qnan, qnan);
            return true;
        }
        const unsigned row = tile_sa + 4u * (unsigned)((jrow - fj0) * pitch);
#pragma unroll
        for (int p = 0; p < CPT / 2; ++p) {
            const unsigned qa = row + o1[2 * p], qb = row + o1[2 * p + 1];
            const u64 p1 = pack2(lds(qa), lds(qb));
            const u64 np1 = fmul2(p1, neg1);
            const u64 d0 = fadd2(pack2(lds(row + o0[2 * p]), lds(row + o0[2 * p + 1])), np1);
            const u64 d2 = fadd2(pack2(lds(row + o2[2 * p]), lds(row + o2[2 * p + 1])), np1);
            const u64 d3 = fadd2(pack2(lds(row + o3[2 * p]), lds(row + o3[2 * p + 1])), np1);
            X2[p] = ffma2(w3x[p], d3, ffma2(w2x[p], d2, ffma2(w0x[p], d0, fadd2(p1, nzr[p]))));
        }
        const u64 t = fadd2(X2[0], X2[1]);
        const float u = lo_of(t) + hi_of(t);
        return __any_sync(0xffffffffu, u != u);
    };
    // x lerp of input row jrow (always inside the grid) for the bilinear fallback
    auto row_lerp = [&](int jrow, float* L) {
        const unsigned row = tile_sa + 4u * (unsigned)((jrow - fj0) * pitch);
#pragma unroll
        for (int e = 0; e < CPT; ++e) {
            const float p1 = lds(row + o1[e]);
            L[e] = fmaf(ct[e], lds(row + o2[e]) - p1, p1 - zref);
        }
    };

    u64 X[4][CPT / 2];                                // x cubics of rows j-1 .. j+2
    // what a node of the current row interval evaluates:  out = wy . Xu + (Lu1 + s Ld) + zc, where a column
    // that can use the cubic has Lu1 = Ld = 0 and a column that falls back to bilinear has Xu = 0 (the choice
    // is per column and interval, not per node: the cubic is NaN exactly when one of the 16 neighbours is
    // missing, whatever the y weights).  `plain`: every column of the warp uses the cubic (the usual case).
    u64 Xu[4][CPT / 2], Lu1[CPT / 2], Ld[CPT / 2];
    const u64 zc2[CPT / 2] = {pack2(zref + cnan[0], zref + cnan[1]), pack2(zref + cnan[2], zref + cnan[3])};
#pragma unroll
    for (int p = 0; p < CPT / 2; ++p) {
        Lu1[p] = Ld[p] = pack2(0.0f, 0.0f);
#pragma unroll
        for (int b = 0; b < 4; ++b) X[b][p] = Xu[b][p] = pack2(0.0f, 0.0f);
    }
    bool plain = true;
    bool bad[4] = {true, true, true, true};           // warp-uniform: row b of the window has a NaN somewhere in the warp
    int cur_j = -5;
    float* orow = out + (size_t)I0 * ax.n_out + Jt;
    for (int r = 0; r < nrows; ++r, orow += ax.n_out) {
        const int2 rw = s_row[r];
        const int j = rw.x;
        if (j < 0) {                                   // CTA-uniform: row outside the input extent
#pragma unroll
            for (int e = 0; e < CPT; ++e) if (cok[e]) orow[32 * e] = qnan;
            continue;
        }
        if (j != cur_j) {                              // CTA-uniform: the window of 4 input rows moves
            if (j == cur_j + 1) {
#pragma unroll
                for (int b = 0; b < 3; ++b) { X[b][0] = X[b + 1][0]; X[b][1] = X[b + 1][1]; bad[b] = bad[b + 1]; }
                bad[3] = row_eval(j + 2, X[3]);
            } else {
#pragma unroll
                for (int b = 0; b < 4; ++b) bad[b] = row_eval(j - 1 + b, X[b]);
            }
            cur_j = j;
            plain = !(bad[0] || bad[1] || bad[2] || bad[3]);
            if (!plain) {                              // somewhere in the warp a column falls back to bilinear
                const u64 sum0 = fadd2(fadd2(X[0][0], X[1][0]), fadd2(X[2][0], X[3][0]));
                const u64 sum1 = fadd2(fadd2(X[0][1], X[1][1]), fadd2(X[2][1], X[3][1]));
                const float sm[CPT] = {lo_of(sum0), hi_of(sum0), lo_of(sum1), hi_of(sum1)};
                bool use[CPT];
#pragma unroll
                for (int e = 0; e < CPT; ++e) use[e] = sm[e] == sm[e];  // no NaN among the column's 4 row cubics
                float l1[CPT], l2[CPT];
                row_lerp(j, l1);
                row_lerp(j + 1, l2);
#pragma unroll
                for (int p = 0; p < CPT / 2; ++p) {
                    const bool ua = use[2 * p], ub = use[2 * p + 1];
#pragma unroll
                    for (int b = 0; b < 4; ++b)
                        Xu[b][p] = pack2(ua ? lo_of(X[b][p]) : 0.0f, ub ? hi_of(X[b][p]) : 0.0f);
                    Lu1[p] = pack2(ua ? 0.0f : l1[2 * p], ub ? 0.0f : l1[2 * p + 1]);
                    Ld[p] = pack2(ua ? 0.0f : l2[2 * p] - l1[2 * p], ub ? 0.0f : l2[2 * p + 1] - l1[2 * p + 1]);
                }
            }
        }
        const float4 wy = s_wy[r];
        const u64 w0 = pack2(wy.x, wy.x), w1 = pack2(wy.y, wy.y), w2 = pack2(wy.z, wy.z), w3 = pack2(wy.w, wy.w);
        if (plain) {
#pragma unroll
            for (int p = 0; p < CPT / 2; ++p) {
                u64 o = ffma2(w1, X[1][p], fmul2(w0, X[0][p]));
                o = ffma2(w2, X[2][p], o);
                o = ffma2(w3, X[3][p], o);
                o = fadd2(o, zc2[p]);
                if (cok[2 * p]) orow[64 * p] = lo_of(o);
                if (cok[2 * p + 1]) orow[64 * p + 32] = hi_of(o);
            }
        } else {
            const float s = __int_as_float(rw.y);
            const u64 s2 = pack2(s, s);
#pragma unroll
            for (int p = 0; p < CPT / 2; ++p) {
                u64 o = ffma2(s2, Ld[p], Lu1[p]);
                o = ffma2(w0, Xu[0][p], o);
                o = ffma2(w1, Xu[1][p], o);
                o = ffma2(w2, Xu[2][p], o);
                o = ffma2(w3, Xu[3][p], o);
                o = fadd2(o, zc2[p]);
                if (cok[2 * p]) orow[64 * p] = lo_of(o);
                if (cok[2 * p + 1]) orow[64 * p + 32] = hi_of(o);
            }
        }
    }
}

// Any geometry (including strong down-sampling, where a tile's input footprint does not fit in
// shared memory): one thread per output node, the 16 neighbours through the read-only path.
__global__ void __launch_bounds__(kThreads)
catmull_rom_gather_kernel(const float* __restrict__ in, float* __restrict__ out, AxisMap ax, AxisMap ay)
{
    const int J = blockIdx.x * kThreads + threadIdx.x;
    if (J >= ax.n_out) return;
    float t, s;
    const int i = axis_locate(ax, J, &t);
    const float4 wx = cr_weights(t);
    const bool c4ok = (i >= 1) && (i + 2 <= ax.n_in - 1);
    for (int I = blockIdx.y; I < ay.n_out; I += gridDim.y) {
        const int j = axis_locate(ay, I, &s);
        float f = __int_as_float(0x7fc00000);
        if (i >= 0 && j >= 0) {
            const float* p = in + (size_t)j * ax.n_in + i;
            const float zref = __ldg(p);
            const float q11 = __ldg(p) - zref, q21 = __ldg(p + 1) - zref;
            const float q12 = __ldg(p + ax.n_in) - zref, q22 = __ldg(p + ax.n_in + 1) - zref;
            const float lo = fmaf(t, q21 - q11, q11), hi = fmaf(t, q22 - q12, q12);
            f = fmaf(s, hi - lo, lo);                              // the bilinear fallback (NaN if a corner is NaN)
            const bool zok = zref == zref;
            if (zok && c4ok && j >= 1 && j + 2 <= ay.n_in - 1) {
                const float4 wy = cr_weights(s);
                const float wyv[4] = {wy.x, wy.y, wy.z, wy.w};
                float cub = 0.0f;
#pragma unroll
                for (int b = 0; b < 4; ++b) {
                    const float* r = p + (ptrdiff_t)(b - 1) * ax.n_in - 1;
                    const float x = fmaf(wx.w, __ldg(r + 3) - zref, fmaf(wx.z, __ldg(r + 2) - zref,
                                    fmaf(wx.y, __ldg(r + 1) - zref, wx.x * (__ldg(r) - zref))));
                    cub = fmaf(wyv[b], x, cub);
                }
                if (cub == cub) f = cub;                           // NaN: one of the 16 neighbours is NaN
            }
            f += zref;
        }
        out[(size_t)I * ax.n_out + J] = f;
    }
}

}  // namespace

extern std::atomic<bool> g_bilinear_tma;    // bilinear.cu

int launch_catmull_rom(const float* d_in, const grid_geom_t& in, float* d_out, const grid_geom_t& out,
                       cudaStream_t stream)
{
    const AxisMap ax = axis_x(in, out), ay = axis_y(in, out);
    constexpr int CPT = 4, TH = 32, TW = CPT * kThreads;
    const long long fw = footprint_bound(ax, TW) + 2, fh = footprint_bound(ay, TH) + 2;
    long long smem = ((fw + 6) & ~3LL) * fh * (long long)sizeof(float);
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
            BATHY_CUDA_TRY(cudaFuncSetAttribute(catmull_rom_tiled_kernel<CPT, TH, true>,
                                                cudaFuncAttributeMaxDynamicSharedMemorySize, 160 * 1024));
            BATHY_CUDA_TRY(cudaFuncSetAttribute(catmull_rom_tiled_kernel<CPT, TH, false>,
                                                cudaFuncAttributeMaxDynamicSharedMemorySize, 160 * 1024));
            return (int)BATHY_OK;
        });
        if (rc) return rc;
        dim3 grid((out.nx + TW - 1) / TW, (out.ny + TH - 1) / TH);
        if (use_tma) catmull_rom_tiled_kernel<CPT, TH, true><<<grid, kThreads, (size_t)smem, stream>>>(d_in, d_out, ax, ay, tmap, (int)fh);
        else         catmull_rom_tiled_kernel<CPT, TH, false><<<grid, kThreads, (size_t)smem, stream>>>(d_in, d_out, ax, ay, tmap, 0);
    } else {
        dim3 grid((out.nx + kThreads - 1) / kThreads, out.ny < 65535 ? out.ny : 65535);
        catmull_rom_gather_kernel<<<grid, kThreads, 0, stream>>>(d_in, d_out, ax, ay);
    }
    count_launch();
    return launch_status();
}

}  // namespace bathy
