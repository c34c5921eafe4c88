// spline_tile.cu -- interp_spline, fused single-pass path (SURVEY.md 8(a) rows S1-S4 in ONE kernel).
//
// The natural-spline second derivatives solve the constant tridiagonal system [1 4 1] (uniform
// knots).  Its inverse decays as (2 - sqrt 3)^|i-j| = 0.268^d, so the solve is numerically LOCAL:
// a Thomas solve of the WINDOWED system that extends H knots beyond the knots a tile needs, with the
// natural condition M = 0 imposed at the window ends, differs from the global solve by at most
// 0.268^H times the true M at the window end.  In the spline value that enters with a factor
// <= 2 * 0.385, and |M h^2/6| <= 2 * range for any data, hence
//     |S_window - S_global| <= 1.6 * 0.268^H * range   per solve direction,
// = 8.2e-7 * range at H = 11 for ANY input (white noise of full amplitude; smooth terrain is orders below).
// A window end that coincides with the true end of the grid is exact.
//
// One CTA owns TXI x TYI input cells and every output node inside them:
//   load   the (TXI+1+2H) x (TYI+1+2H) window of z (minus a reference depth) into shared memory;
//   S2     one thread per window column: Thomas along y, d' held in REGISTERS (fully unrolled),
//          keeps My on the TYI+1 knot rows the tile needs;
//   S1,S3  one thread per knot row: Thomas along x of z (-> Mx) and of My (-> Mxy);
//   S4     a thread owns output columns (lane-contiguous: a warp stores 128 contiguous bytes) and
//          marches down the tile's output rows; the x-direction splines X = S_x[z], Y = S_x[My] of
//          the two bracketing knot rows live in registers, a node is 3 FMA + 1 add + 1 store.
// All M are stored scaled by h^2/6 (M' = M h^2/6 solves [1 4 1] M' = second difference of z), so
// the grid spacing drops out of the arithmetic.
// HBM traffic: the input once (window halos are L2 hits), the output once = the compulsory bytes.
#include <type_traits>
#include <string.h>

#include "common.cuh"
#include "tma.cuh"

namespace bathy {

namespace {

constexpr int kTileThreads = 128;

// c'_q of the [1 4 1] Thomas forward sweep, q = 0 is the first unknown after an M = 0 end:
// 1/4, 4/15, 15/56, ... -> 2 - sqrt(3) (converged in fp32 from q = 8 on).
__device__ __forceinline__ constexpr float cp141(int q)
{
    constexpr float kCp[8] = {
        0.25f, 0.26666666666666666f, 0.26785714285714285f, 0.26794258373205743f,
        0.26794871794871794f, 0.26794915836482308f, 0.26794918998527245f, 0.26794919225551855f};
    return q < 8 ? kCp[q] : 0.26794919243112270f;
}

template <int TXI_, int TYI_, int H_>
struct TileShape {
    static constexpr int TXI = TXI_, TYI = TYI_, H = H_;
    static constexpr int WX = TXI + 1 + 2 * H;        // window knots along x
    static constexpr int WY = TYI + 1 + 2 * H;
    static constexpr int NXI = TXI + 1, NYI = TYI + 1;  // knots the tile's cells touch
    static constexpr int PZ = WX | 1;                  // odd pitches: a thread per row is bank-conflict free
    static constexpr int PA = (WX + 3 + 3) / 4 * 4;    // pitch of the raw window: 16-byte rows for cp.async, room for the
                                                       // 0..3 columns between the aligned start and the window start
    static constexpr int PQ = NXI;                     // pitch of the knot records Q = (z, Mx', My', Mxy'), in float4
    static constexpr int front_floats = (4 * NYI * PQ > WY * PA) ? 4 * NYI * PQ : WY * PA;   // max(knot records, raw window)
    static constexpr int PSK = (16 - (NYI * PZ) % 32 + 32) % 32;   // skew of the second plane: the two planes of a
                                                       // knot row sit 16 banks apart (x sweeps, below)
    static constexpr size_t data_bytes = (sizeof(float) * ((size_t)front_floats + 2 * (size_t)NYI * PZ + PSK) + 15) / 16 * 16;
    static constexpr size_t smem_bytes = data_bytes + 16;             // + the mbarrier of the TMA window load
    static_assert(WX <= kTileThreads && 2 * NYI <= kTileThreads && NYI <= 32, "tile shape");
};

// Smallest J in [0, n_out] whose clamped interval index is >= i0 (axis_clamped is monotone in J).
__device__ int first_node_ge(const AxisMap& m, int i0)
{
    if (i0 <= 0) return 0;
    const double g = ((m.i0 + (double)i0 * m.id) - m.o0) / m.od;
    int J = (g >= (double)m.n_out) ? m.n_out : (g <= 0.0 ? 0 : (int)ceil(g));
    while (J > 0 && axis_clamped(m, J - 1) >= i0) --J;
    while (J < m.n_out && axis_clamped(m, J) < i0) ++J;
    return J;
}

// Thomas solve of one windowed system of N knots; rd(q) returns knot q (relative to z_ref), st(k, v, m)
// receives, for the kept knots k = q - k0 in [0, nk), the knot value v and M' = M h^2/6, with M' = 0
// at both window ends.
// Formulation: M' = z - 6 w, where w solves [1 4 1] w = z on the interior knots with w = z/6 at the
// two ends (substitute M'_q = z_q - 6 w_q into M'_{q-1} + 4 M'_q + M'_{q+1} = z_{q-1} - 2 z_q + z_{q+1}).
// The sweeps run on e_q = d'_q / c'_q and wt_q = w_q / c'_q, which makes each of them ONE dependent
// FMA per knot:   e_q = rhs_q - c'_{q-1} e_{q-1},   wt_q = e_q - c'_{q+1} wt_{q+1},   M'_q = z_q - 6 c'_q wt_q.
// e lives in registers (everything is unrolled; c'_q are compile-time constants).
// STATIC: k0 and nk are the compile-time K0, NK (interior tiles), so the store predicates fold.
template <int N, bool STATIC, int K0, int NK, class Rd, class St>
__device__ __forceinline__ void thomas_window(Rd rd, St st, int k0_rt, int nk_rt)
{
    static_assert(N >= 6, "window too short");
    const int k0 = STATIC ? K0 : k0_rt, nk = STATIC ? NK : nk_rt;
    // Four passes so that the two serial sweeps are pure register chains (one dependent FMA per knot)
    // and every shared-memory access sits in a pass without dependencies, all loads in flight at once.
    float e[N];
#pragma unroll
    for (int q = 0; q < N; ++q) e[q] = rd(q);                          // pass 1: the knots
    // interior tiles keep the knots they will write out in registers (a second read of shared memory
    // costs wavefronts of the unit that bounds the kernel); edge tiles read them again in pass 4
    constexpr int NV = STATIC ? NK : 1;
    float vk[NV];
    if (STATIC) {
#pragma unroll
        for (int k = 0; k < NV; ++k) vk[k] = e[K0 + k];
    }
    e[1] = fmaf(-1.0f / 6.0f, e[0], e[1]);                             // pass 2: forward sweep, e_q in place
#pragma unroll
    for (int q = 2; q <= N - 3; ++q) e[q] = fmaf(-cp141(q - 2), e[q - 1], e[q]);
    e[N - 2] = fmaf(-cp141(N - 4), e[N - 3], fmaf(-1.0f / 6.0f, e[N - 1], e[N - 2]));
#pragma unroll
    for (int q = N - 3; q >= 1; --q) e[q] = fmaf(-cp141(q), e[q + 1], e[q]);   // pass 3: backward sweep, wt_q in place
    // pass 4: M'_q = z_q - 6 c'_q wt_q on the kept knots.  Where the knot is read again, reads and writes
    // go in groups of 8: the compiler cannot prove that the stores do not alias the knots, so a store
    // between two loads would serialise them (one shared-memory latency per knot: this was 20 % of the
    // kernel's warp time).
    if (STATIC) {
        static_assert(!STATIC || (K0 >= 1 && K0 + NK <= N - 1), "kept knots are interior knots of the window");
#pragma unroll
        for (int k = NV - 1; k >= 0; --k) {
            const int q = K0 + k;
            st(k, vk[k], fmaf(-6.0f * cp141(q - 1), e[q], vk[k]));
        }
        return;
    }
    if (N - 1 - k0 >= 0 && N - 1 - k0 < nk) st(N - 1 - k0, rd(N - 1), 0.0f);
    constexpr int B = 8;
#pragma unroll
    for (int qb = N - 2; qb >= 1; qb -= B) {
        float v[B];
#pragma unroll
        for (int g = 0; g < B; ++g) {
            const int q = qb - g, k = q - k0;
            v[g] = (q >= 1 && k >= 0 && k < nk) ? rd(q) : 0.0f;
        }
#pragma unroll
        for (int g = 0; g < B; ++g) {
            const int q = qb - g, k = q - k0;
            if (q >= 1 && k >= 0 && k < nk) st(k, v[g], fmaf(-6.0f * cp141(q >= 1 ? q - 1 : 0), e[q >= 1 ? q : 0], v[g]));
        }
    }
    if (k0 == 0) st(0, rd(0), 0.0f);
}

// Per-axis tables of the output->input map, computed once per call in float64 exactly as the
// definition (readings B1/B2) so that the tile kernel does no double-precision arithmetic:
//   rowtab[n] = (interval index or -1 as int bits, t, C(t) = ((1-t)^2 - 1)(1-t), D(t) = (t^2 - 1) t)
//   colw[n]   = (1-t, C(t), t, D(t)), coli[n] = interval index or -1
//   tb[b]     = first output node whose (clamped) interval is >= b * tile cells; tb[nb] = n_out
//   rfirst[j] = first output row whose (clamped) interval is >= j, j = 0 .. ny_in.
__global__ void __launch_bounds__(256)
spline_tables_kernel(AxisMap ax, AxisMap ay, float4* __restrict__ colw, float4* __restrict__ rowtab,
                     int* __restrict__ tbx, int* __restrict__ tby, int* __restrict__ rfirst, int* __restrict__ coli,
                     int nbx, int nby, int txi, int tyi)
{
    // the tile kernel is launched with programmatic stream serialisation: its CTAs may start (and load
    // their windows) while this grid still runs; they wait (griddepcontrol.wait) before reading a table
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
    int n = blockIdx.x * 256 + threadIdx.x;
    if (n < ax.n_out + ay.n_out) {
        const bool isx = n < ax.n_out;
        const AxisMap& m = isx ? ax : ay;
        const int J = isx ? n : n - ax.n_out;
        float t;
        const int i = axis_locate(m, J, &t);
        const float a = 1.0f - t;
        const float C = (a * a - 1.0f) * a, D = (t * t - 1.0f) * t;
        if (isx) {
            // columns: the blending weights as two fp32x2 operands (1-t, C), (t, D), NaN outside the input
            // extent (reading B4: the node then comes out NaN without a test in the tile kernel)
            const float qn = __int_as_float(0x7fc00000);
            colw[J] = (i < 0) ? make_float4(qn, qn, qn, qn) : make_float4(a, C, t, D);
            coli[J] = i;
        } else {
            rowtab[J] = make_float4(__int_as_float(i), t, C, D);
        }
        return;
    }
    n -= ax.n_out + ay.n_out;
    if (n <= nbx) { tbx[n] = (n == nbx) ? ax.n_out : first_node_ge(ax, n * txi); return; }
    n -= nbx + 1;
    if (n <= nby) { tby[n] = (n == nby) ? ay.n_out : first_node_ge(ay, n * tyi); return; }
    n -= nby + 1;
    if (n <= ay.n_in) rfirst[n] = (n >= ay.n_in - 1) ? ay.n_out : first_node_ge(ay, n);
}

template <class S>
__global__ void __launch_bounds__(kTileThreads, 4)
spline_tile_kernel(const float* __restrict__ in, float* __restrict__ out, AxisMap ax, AxisMap ay,
                   const float4* __restrict__ colw, const float4* __restrict__ rowtab,
                   const int* __restrict__ tbx, const int* __restrict__ tby, const int* __restrict__ rfirst,
                   const int* __restrict__ coli, int nbx, int n_tiles, int pf_dist,
                   const __grid_constant__ CUtensorMap tmap, int use_tma)
{
    constexpr int TXI = S::TXI, TYI = S::TYI, H = S::H, WX = S::WX, WY = S::WY;
    constexpr int NXI = S::NXI, NYI = S::NYI, PZ = S::PZ, PA = S::PA, PQ = S::PQ;
    constexpr int NW = kTileThreads / 32;
    extern __shared__ __align__(128) unsigned char s_raw[];
    // The raw window is dead once the y sweep has run, the knot records are born after it: they share
    // the front of the buffer (55 KB per CTA: four CTAs per SM).
    float4* s_q = reinterpret_cast<float4*>(s_raw);                       // [NYI][PQ] knot records (z, Mx', My', Mxy')
    float* s_zbuf = reinterpret_cast<float*>(s_raw);                      // [WY][PA] raw window
    float* s_zf = reinterpret_cast<float*>(s_raw) + S::front_floats;      // [NYI][PZ] z - zref on the tile's knot rows
    float* s_my = s_zf + NYI * PZ + S::PSK;                               // [NYI][PZ] My' on the tile's knot rows

    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const bool vec_ok = (reinterpret_cast<uintptr_t>(in) & 15) == 0 && (ax.n_in & 3) == 0;

    // Window of tile `tile` -> buffer `buf`: raw depths, whole 16-byte vectors from the aligned column
    // at or before the window start, global -> shared without passing through registers (cp.async).
    auto issue_load = [&](int tile, int buf) {
        const int bx = tile % nbx, by = tile / nbx;
        const int w0x = min(max(bx * TXI - H, 0), ax.n_in - WX);          // window origin (host guarantees n_in >= W)
        const int w0y = min(max(by * TYI - H, 0), ay.n_in - WY);
        const int ax0 = w0x & ~3, offx = w0x - ax0;
        float* dstz = s_zbuf + buf * (WY * PA);
        if (vec_ok) {
            // a warp takes whole window rows, a lane one 16-byte vector of the row: everything that
            // depends on the column is computed once, a row costs one address add and one cp.async
            constexpr int VPR = PA / 4;
            static_assert(VPR <= 32, "a window row is at most 32 vectors");
            const int col = ax0 + 4 * lane;
            const int bytes = max(0, min(16, (ax.n_in - col) * 4));      // past the row end: zero fill
            const float* src = in + (size_t)(w0y + warp) * ax.n_in + min(col, ax.n_in - 4);
            unsigned dst = (unsigned)__cvta_generic_to_shared(dstz + warp * PA + 4 * lane);
            if (lane < VPR) {
#pragma unroll 4
                for (int r = warp; r < WY; r += NW) {
                    asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;" :: "r"(dst), "l"(src), "r"(bytes) : "memory");
                    src += (size_t)NW * ax.n_in;
                    dst += NW * PA * 4;
                }
            }
        } else {
            for (int v = tid; v < WY * WX; v += kTileThreads) {
                const int r = v / WX, c = v - r * WX;
                dstz[r * PA + offx + c] = __ldg(in + (size_t)(w0y + r) * ax.n_in + w0x + c);
            }
        }
    };

    {
        const int tile = blockIdx.x;
        const int bxt = tile % nbx, byt = tile / nbx;
        const int i0 = bxt * TXI, j0 = byt * TYI;                         // first cell of the tile
        const int w0x = min(max(i0 - H, 0), ax.n_in - WX);
        const int w0y = min(max(j0 - H, 0), ay.n_in - WY);
        const int kx0 = i0 - w0x, ky0 = j0 - w0y;                         // tile knot 0 in window coordinates
        const int nkx = min(NXI, ax.n_in - i0), nky = min(NYI, ay.n_in - j0);   // knots present (last tile may be short)
        // The window goes global -> shared in ONE TMA box load (cp.async.bulk.tensor.2d: no LSU wavefronts, no
        // per-thread address arithmetic) when the input rows are 16-byte aligned; the box starts at the aligned
        // column at or before the window start (profiles/r2_tma_probe.md), columns past the row end arrive as
        // zeros.  Otherwise by cp.async / plain loads.
        const unsigned bar = (unsigned)__cvta_generic_to_shared(s_raw + S::data_bytes);
        if (use_tma) {
            if (tid == 0) {
                mbar_init(bar, 1);
                tma_load_2d((unsigned)__cvta_generic_to_shared(s_zbuf), &tmap, w0x & ~3, w0y, bar, (unsigned)(WY * PA * sizeof(float)));
            }
        } else {
            issue_load(tile, 0);
            asm volatile("cp.async.commit_group;" ::: "memory");
        }
        {
            // L2 prefetch of the window of the tile that starts one wave of CTAs later: its cp.async
            // then finds the rows in L2 instead of waiting for HBM at the head of the CTA
            const int pt = tile + pf_dist;
            if (pt < n_tiles) {
                const int pbx = pt % nbx, pby = pt / nbx;
                const int px = min(max(pbx * TXI - H, 0), ax.n_in - WX) & ~31;          // 128-byte lines
                const int py = min(max(pby * TYI - H, 0), ay.n_in - WY);
                constexpr int LPR = (WX + 31 + 31) / 32;                               // lines per window row
                for (int v = tid; v < WY * LPR; v += kTileThreads) {
                    const int r = v / LPR, c = px + (v - r * LPR) * 32;
                    if (c < ax.n_in) asm volatile("prefetch.global.L2 [%0];" :: "l"(in + (size_t)(py + r) * ax.n_in + c));
                }
            }
        }
        asm volatile("griddepcontrol.wait;" ::: "memory");               // the tables of this call are complete
        // The first table reads behind the wait go through ld_behind_wait, NOT __ldg: a non-coherent load
        // (LDG.CONSTANT) promises data that nobody writes while this grid runs, so ptxas is free to schedule it --
        // and every load whose address depends on it -- above the wait, where the tables kernel may not have
        // written the entry yet (it did: the first wave of CTAs then ran on whatever the workspace held before).
        // Every other table read of this kernel takes its address from these six values and so stays behind them.
        auto ld_behind_wait = [](const int* p) {
            int v;
            asm volatile("ld.global.ca.s32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
            return v;
        };
        const int Jbeg = ld_behind_wait(tbx + bxt), Jend = ld_behind_wait(tbx + bxt + 1);   // output nodes of the tile
        const int Ibeg = ld_behind_wait(tby + byt), Iend = ld_behind_wait(tby + byt + 1);
        const int offx = w0x & 3;
        const float* s_z = s_zbuf;
        // the warp's band: knot intervals [kja, kjb) of the tile = output rows [rb, re) (rfirst[j]: first
        // output row whose interval is >= j)
        constexpr int TI = (TYI + NW - 1) / NW;                           // knot intervals per warp
        const int kja = warp * TI, kjb = min(min(kja + TI, TYI), nky - 1);
        const int rb = min(max(ld_behind_wait(rfirst + min(j0 + kja, ay.n_in)), Ibeg), Iend);
        const int re = (kjb > kja) ? min(max(ld_behind_wait(rfirst + min(j0 + kjb, ay.n_in)), Ibeg), Iend) : rb;
        if (use_tma) {
            __syncthreads();                                             // the barrier is initialised
            mbar_wait(bar, 0);                                           // the window has landed
        } else {
            asm volatile("cp.async.wait_group 0;" ::: "memory");         // the window has landed
            __syncthreads();
        }
        float zref = s_z[offx];                                           // the window's first sample
        if (!isfinite(zref)) zref = 0.0f;
        // the table entries the evaluate stage starts with: into L1 now, two stages ahead of their use
        for (int i = rb + lane; i < re; i += 32) asm volatile("prefetch.global.L1 [%0];" :: "l"(rowtab + i));
#pragma unroll
        for (int e = 0; e < 4; ++e) {
            const int J = Jbeg + lane + 32 * e;
            if (J < Jend) {
                asm volatile("prefetch.global.L1 [%0];" :: "l"(colw + J));
                asm volatile("prefetch.global.L1 [%0];" :: "l"(coli + J));
            }
        }

        // ---- S2: Thomas along y of every window column (one thread per column): z - zref and My' on the
        //      tile's knot rows, into odd-pitch planes that the row-wise solves read without bank conflicts
        const bool inner_y = (ky0 == H) && (nky == NYI), inner_x = (kx0 == H) && (nkx == NXI);   // CTA-uniform
        if (tid < WX) {
            const float* col = s_z + offx + tid;
            auto rd = [&](int q) { return col[q * PA] - zref; };
            auto st = [&](int k, float v, float m) { s_zf[k * PZ + tid] = v; s_my[k * PZ + tid] = m; };
            if (inner_y) thomas_window<WY, true, H, NYI>(rd, st, 0, 0);
            else         thomas_window<WY, false, 0, 0>(rd, st, ky0, nky);
        }
        __syncthreads();

        // ---- S1: Mx' = Thomas along x of z on the knot rows (warp 0 -> Q.xy = (z, Mx'));
        //      S3: Mxy' = Thomas along x of My' (warp 1 -> Q.zw = (My', Mxy'))
        if (inner_x) {
            // interior tile: every warp works; the row's
            // knots are solved as two overlapping windows of HW = TXI/2 + 1 + 2H knots (the same
            // 0.268^H bound applies where the halves meet), so the serial chains are 55 instead of 87 long
            constexpr int HL = TXI / 2 + 1;                               // knots kept by the left half
            constexpr int HW = HL + 2 * H;                                // window of a half
            // A warp takes one half and 16 knot rows, both planes: lanes 0-7 / 8-15 are plane 0 / 1 of
            // rows 0-7, lanes 16-31 the same of rows 8-15.  A half-warp then writes 8 records' (z, Mx')
            // and (My', Mxy') halves = 16 different 8-byte bank pairs: the STS.64 are conflict-free
            // (a warp of one plane writes 4-way conflicting: this was a tenth of the kernel's
            // shared-memory wavefronts, the unit that bounds it), and so are the loads (plane skew PSK).
            const int plane = (lane >> 3) & 1, half = warp >> 1;
            const int krow = 16 * (warp & 1) + (lane & 7) + 8 * (lane >> 4);
            if (krow < nky) {
                const float* row = (plane == 0 ? s_zf : s_my) + krow * PZ + (half ? WX - HW : 0);
                static_assert(WX - HW == HL - 1 && NXI - HL == HL - 1, "the halves share one instantiation");
                float2* dst = reinterpret_cast<float2*>(s_q + krow * PQ + (half ? HL - 1 : 0)) + plane;
                auto rd = [&](int q) { return row[q]; };
                // left: window knots [0, HW), kept = tile knots [0, HL) = window [H, H + HL)
                // right: window knots [WX - HW, WX), window [H, H + HL) = tile knots [HL - 1, NXI): the same
                // code (one instantiation, half the instructions); its first knot is the left half's last
                auto st = [&](int k, float v, float m) { if (k > 0 || half == 0) dst[2 * k] = make_float2(v, m); };
                thomas_window<HW, true, H, HL>(rd, st, 0, 0);
            }
        } else if (warp < 2 && lane < nky) {
            const float* row = (warp == 0 ? s_zf : s_my) + lane * PZ;
            float2* dst = reinterpret_cast<float2*>(s_q + lane * PQ) + warp;
            auto rd = [&](int q) { return row[q]; };
            auto st = [&](int k, float v, float m) { dst[2 * k] = make_float2(v, m); };
            thomas_window<WX, false, 0, 0>(rd, st, kx0, nkx);
        }
        __syncthreads();

        // ---- S4: evaluate.  A warp owns a band of knot intervals (rows of cells) and, per pass, 128
        //      columns (a thread: 4 columns 32 apart, so every store instruction of a warp writes 128
        //      contiguous bytes).  Per knot row and column the x-direction splines X = S_x[z], Y = S_x[My']
        //      are two LDS.128 and four packed fp32x2 operations; per node the y-direction blend is three
        //      packed FMAs for two columns.  The row loop of an interval has no data-dependent branch.
        const float qnan = __int_as_float(0x7fc00000);
        const u64 neg1 = pack2(-1.0f, -1.0f), zref2 = pack2(zref, zref);
        const bool oob_rows = (byt == 0 || (byt + 1) * TYI >= ay.n_in - 1) && Ibeg < Iend &&
            (__float_as_int(__ldg(rowtab + Ibeg).x) < 0 || __float_as_int(__ldg(rowtab + Iend - 1).x) < 0);
        if (oob_rows) {
            // rows of the tile outside the input extent (reading B4): NaN
            for (int I = Ibeg + warp; I < Iend; I += NW)
                if (__float_as_int(__ldg(rowtab + I).x) < 0)
                    for (int J = Jbeg + lane; J < Jend; J += 32) out[(size_t)I * ax.n_out + J] = qnan;
        }
        // the row entries (j, s, Cy, Dy) of this warp's band go to shared memory once (the planes of the
        // sweeps are dead): a global load per row would expose an L2 round trip in every interval
        constexpr int RT_CAP = (2 * NYI * PZ) / (4 * NW);                 // float4 entries per warp
        float4* s_rt = reinterpret_cast<float4*>(s_zf) + warp * RT_CAP;
        // (a band longer than the buffer -- up-sampling factors above ~40 -- goes through it in chunks)
        for (int cb = rb; cb < re; cb += RT_CAP) {
        const int ce = min(cb + RT_CAP, re);
        __syncwarp();
        for (int i = lane; i < ce - cb; i += 32) s_rt[i] = __ldg(rowtab + cb + i);
        __syncwarp();
        for (int Jp = Jbeg; Jp < Jend; Jp += 128) {
            const int Jt = Jp + lane;                  // column of e = 0; e-th column is 32 e further
            bool cok[4];
            u64 wl[4], wh[4];                          // blending weights (1-t, C(t)) and (t, D(t)) of the column
            unsigned qc[4];                            // left knot record of the column's interval, knot row 0 of the tile
#pragma unroll
            for (int e = 0; e < 4; ++e) {
                const int J = Jt + 32 * e;
                cok[e] = J < Jend;
                // the weights arrive as 64-bit pairs (NaN pairs outside the input extent): no repacking
                const ulonglong2 cw = cok[e] ? __ldg(reinterpret_cast<const ulonglong2*>(colw + J)) : make_ulonglong2(0ull, 0ull);
                const int i = cok[e] ? __ldg(coli + J) : -1;
                wl[e] = cw.x;
                wh[e] = cw.y;
                qc[e] = (unsigned)__cvta_generic_to_shared(s_q + max(i - i0, 0));
            }
            // x-direction splines of knot row kj at this thread's 4 columns, paired by column:
            // X2[p] = (X[2p], X[2p+1])
            auto knot_row = [&](int kj, u64* X2, u64* Y2) {
                float xv[4], yv[4];
                const unsigned ro = (unsigned)(kj * (PQ * 16));
#pragma unroll
                for (int e = 0; e < 4; ++e) {
                    u64 Lx, Ly, Rx, Ry;                // (z, Mx'), (My', Mxy') of the interval's two knots
                    asm volatile("ld.shared.v2.b64 {%0, %1}, [%2];" : "=l"(Lx), "=l"(Ly) : "r"(qc[e] + ro) : "memory");
                    asm volatile("ld.shared.v2.b64 {%0, %1}, [%2+16];" : "=l"(Rx), "=l"(Ry) : "r"(qc[e] + ro) : "memory");
                    const u64 ux = ffma2(Rx, wh[e], fmul2(Lx, wl[e]));
                    const u64 uy = ffma2(Ry, wh[e], fmul2(Ly, wl[e]));
                    xv[e] = lo_of(ux) + hi_of(ux);
                    yv[e] = lo_of(uy) + hi_of(uy);
                }
                X2[0] = pack2(xv[0], xv[1]); X2[1] = pack2(xv[2], xv[3]);
                Y2[0] = pack2(yv[0], yv[1]); Y2[1] = pack2(yv[2], yv[3]);
            };
            u64 X0[2], X1[2], Xd[2], Y0[2], Y1[2];
#pragma unroll
            for (int p = 0; p < 2; ++p) X0[p] = X1[p] = Xd[p] = Y0[p] = Y1[p] = pack2(0.0f, 0.0f);
            const bool full = !oob_rows && (Jp + 128 <= Jend);        // warp-uniform
            // Row-driven: the band's output rows in order; a row whose knot interval differs from the one
            // before it (warp-uniform test) first moves the two knot rows on.  With up-sampling factor 2
            // there are only two rows per interval, so nothing is set up per interval beyond that.
            auto band = [&](auto full_c) {
                constexpr bool FULL = decltype(full_c)::value;
                int curj = -2;
                unsigned rtp = (unsigned)__cvta_generic_to_shared(s_rt);
                float* op = out + (size_t)cb * ax.n_out + Jt;
                auto lds_row = [&](unsigned addr) {
                    float4 rc;                                            // (j, s, Cy, Dy); j < 0: outside the extent
                    asm volatile("ld.shared.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(rc.x), "=f"(rc.y), "=f"(rc.z), "=f"(rc.w) : "r"(addr) : "memory");
                    return rc;
                };
                auto one_row = [&](const float4 rc) {
                    const int jr = __float_as_int(rc.x);
                    const bool rv = FULL || jr >= 0;
                    if (jr != curj && rv) {
                        const int kj = jr - j0;
                        if (jr != curj + 1) knot_row(kj, X1, Y1);         // first interval of the band only
#pragma unroll
                        for (int p = 0; p < 2; ++p) { X0[p] = X1[p]; Y0[p] = Y1[p]; }
                        knot_row(kj + 1, X1, Y1);
#pragma unroll
                        for (int p = 0; p < 2; ++p) Xd[p] = ffma2(X0[p], neg1, X1[p]);
                        curj = jr;
                    }
                    const u64 s2 = pack2(rc.y, rc.y), cy2 = pack2(rc.z, rc.z), dy2 = pack2(rc.w, rc.w);
#pragma unroll
                    for (int p = 0; p < 2; ++p) {
                        u64 o = ffma2(s2, Xd[p], X0[p]);
                        o = ffma2(cy2, Y0[p], o);
                        o = ffma2(dy2, Y1[p], o);
                        o = fadd2(o, zref2);
                        if (FULL || (cok[2 * p] && rv)) op[64 * p] = lo_of(o);
                        if (FULL || (cok[2 * p + 1] && rv)) op[64 * p + 32] = hi_of(o);
                    }
                    op += ax.n_out;
                };
                // two rows per trip, both row entries in flight before the first is used
                int r = cb;
#pragma unroll 1
                for (; r + 1 < ce; r += 2, rtp += 32) {
                    const float4 ra = lds_row(rtp), rb2 = lds_row(rtp + 16);
                    one_row(ra);
                    one_row(rb2);
                }
                if (r < ce) one_row(lds_row(rtp));
            };
            if (full) band(std::true_type{}); else band(std::false_type{});
        }
        }
    }
}

template <class S>
int launch_tile(const float* d_in, float* d_out, const AxisMap& ax, const AxisMap& ay, void* d_ws, cudaStream_t stream, bool allow_tma)
{
    static DeviceOnce once;
    const int rc_attr = once_per_device(once, []() -> int {
        BATHY_CUDA_TRY(cudaFuncSetAttribute(spline_tile_kernel<S>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                            (int)S::smem_bytes));
        return (int)BATHY_OK;
    });
    if (rc_attr) return rc_attr;
    dim3 grid((ax.n_in - 1 + S::TXI - 1) / S::TXI, (ay.n_in - 1 + S::TYI - 1) / S::TYI);
    float4* colw = static_cast<float4*>(d_ws);
    float4* rowtab = colw + ax.n_out;
    int* tbx = reinterpret_cast<int*>(rowtab + ay.n_out);
    int* tby = tbx + grid.x + 1;
    int* rfirst = tby + grid.y + 1;
    int* coli = rfirst + ay.n_in + 1;
    const long long items = (long long)ax.n_out + ay.n_out + grid.x + grid.y + 2 + ay.n_in + 1;
    spline_tables_kernel<<<(unsigned)((items + 255) / 256), 256, 0, stream>>>(ax, ay, colw, rowtab, tbx, tby, rfirst, coli,
                                                                              (int)grid.x, (int)grid.y, S::TXI, S::TYI);
    const long long n_tiles = (long long)grid.x * grid.y;
    if (n_tiles > 0x7fffffffLL) return 1;
    const unsigned ctas = (unsigned)n_tiles;
    CUtensorMap tmap;
    memset(&tmap, 0, sizeof(tmap));
    int use_tma = 0;
    if (allow_tma && (reinterpret_cast<uintptr_t>(d_in) & 15) == 0 && (ax.n_in & 3) == 0)
        use_tma = tensor_map_2d(&tmap, d_in, ax.n_in, ay.n_in, S::PA, S::WY) == BATHY_OK ? 1 : 0;
    {
        cudaLaunchConfig_t cfg = {};
        cfg.gridDim = dim3(ctas);
        cfg.blockDim = dim3(kTileThreads);
        cfg.dynamicSmemBytes = S::smem_bytes;
        cfg.stream = stream;
        cudaLaunchAttribute attr[1];
        attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
        attr[0].val.programmaticStreamSerializationAllowed = 1;
        cfg.attrs = attr;
        cfg.numAttrs = 1;
        BATHY_CUDA_TRY(cudaLaunchKernelEx(&cfg, spline_tile_kernel<S>, d_in, d_out, ax, ay, (const float4*)colw, (const float4*)rowtab,
                                          (const int*)tbx, (const int*)tby, (const int*)rfirst, (const int*)coli,
                                          (int)grid.x, (int)n_tiles, 4 * kSMs /* CTAs resident at once */, tmap, use_tma));
    }
    count_launch(2);
    return launch_status();
}

}  // namespace

// Returns 1 when the geometry is not served by the fused path (the caller falls back to the
// global-solve path), else the launch status.
// Bytes of the axis tables at the start of the workspace (an upper bound over both tile shapes).
size_t spline_tiled_table_bytes(const grid_geom_t& in, const grid_geom_t& out)
{
    const size_t b = 16 * ((size_t)out.nx + (size_t)out.ny) + 4 * ((size_t)in.nx + 2 * (size_t)in.ny + (size_t)out.nx + 8);
    return (b + 255) / 256 * 256;
}

int launch_spline_tiled(const float* d_in, const grid_geom_t& in, float* d_out, const grid_geom_t& out,
                        void* d_ws, cudaStream_t stream, bool allow_tma)
{
    const AxisMap ax = axis_x(in, out), ay = axis_y(in, out);
    // up-sampling (or 1:1) only: a tile must produce at least about as many nodes as it reads knots
    if (!(out.dx <= in.dx) || !(out.dy <= in.dy)) return 1;
    using Big = TileShape<64, 31, 11>;
    using Small = TileShape<16, 16, 11>;
    if (in.nx >= Big::WX && in.ny >= Big::WY) {
        if ((in.ny - 1 + Big::TYI - 1) / Big::TYI > 65535) return 1;
        return launch_tile<Big>(d_in, d_out, ax, ay, d_ws, stream, allow_tma);
    }
    if (in.nx >= Small::WX && in.ny >= Small::WY) return launch_tile<Small>(d_in, d_out, ax, ay, d_ws, stream, allow_tma);
    return 1;
}

}  // namespace bathy
