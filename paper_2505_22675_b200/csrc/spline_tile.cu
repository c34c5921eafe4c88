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
#include "common.cuh"

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
    static constexpr int PQ = NXI;                     // pitch of the knot records Q = (z, My', Mx', Mxy'), in float4
    static constexpr int RCAP = 160;                   // output rows per table chunk
    static constexpr size_t smem_bytes =
        sizeof(float) * ((size_t)WY * PA + (size_t)NYI * PZ) + sizeof(float4) * ((size_t)NYI * PQ + RCAP);
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

// Thomas solve of one windowed system of N knots read with `stride` from `src` (values relative to
// z_ref).  Result M' = M h^2/6 with M' = 0 at both window ends; knots [k0, k0 + nk) go to
// dst[0 .. nk) with stride `dstride`.
// Formulation: M' = z - 6 w, where w solves [1 4 1] w = z on the interior knots with w = z/6 at the
// two ends (substitute M'_q = z_q - 6 w_q into M'_{q-1} + 4 M'_q + M'_{q+1} = z_{q-1} - 2 z_q + z_{q+1}).
// The sweeps run on e_q = d'_q / c'_q and wt_q = w_q / c'_q, which makes each of them ONE dependent
// FMA per knot:   e_q = rhs_q - c'_{q-1} e_{q-1},   wt_q = e_q - c'_{q+1} wt_{q+1},   M'_q = z_q - 6 c'_q wt_q.
// e lives in registers (everything is unrolled; c'_q are compile-time constants).
// STATIC: k0 and nk are the compile-time K0, NK (interior tiles), so the store predicates fold.
// COPY: the source value of every kept knot is stored too, at dst[k * dstride - 2] (the knot record
// Q = (z, My', Mx', Mxy') is filled by the two x-direction solves: z and Mx' by one, My' and Mxy' by
// the other).
// FIX: the source holds raw depths; the forward sweep (which reads every knot exactly once)
// subtracts zref and writes the difference back, so that everything later reads small numbers.
template <int N, bool STATIC, int K0, int NK, bool COPY, bool FIX>
__device__ __forceinline__ void thomas_window(float* __restrict__ src, int stride,
                                              float* __restrict__ dst, int dstride, int k0_rt, int nk_rt, float zref)
{
    static_assert(N >= 6, "window too short");
    const int k0 = STATIC ? K0 : k0_rt, nk = STATIC ? NK : nk_rt;
    auto rd = [&](int q) {
        float v = src[q * stride];
        if (FIX) { v -= zref; src[q * stride] = v; }
        return v;
    };
    float e[N];
    {
        const float v0 = rd(0);
        e[1] = fmaf(-1.0f / 6.0f, v0, rd(1));
    }
#pragma unroll
    for (int q = 2; q <= N - 3; ++q) e[q] = fmaf(-cp141(q - 2), e[q - 1], rd(q));
    {
        const float vl = rd(N - 1);
        e[N - 2] = fmaf(-cp141(N - 4), e[N - 3], fmaf(-1.0f / 6.0f, vl, rd(N - 2)));
    }
    if (N - 1 - k0 >= 0 && N - 1 - k0 < nk) {
        dst[(N - 1 - k0) * dstride] = 0.0f;
        if (COPY) dst[(N - 1 - k0) * dstride - 2] = src[(N - 1) * stride];
    }
    float wt = e[N - 2];
    {
        const int k = N - 2 - k0;
        if (k >= 0 && k < nk) {
            const float v = src[(N - 2) * stride];
            dst[k * dstride] = fmaf(-6.0f * cp141(N - 3), wt, v);
            if (COPY) dst[k * dstride - 2] = v;
        }
    }
#pragma unroll
    for (int q = N - 3; q >= 1; --q) {
        wt = fmaf(-cp141(q), wt, e[q]);
        const int k = q - k0;
        if (k >= 0 && k < nk) {
            const float v = src[q * stride];
            dst[k * dstride] = fmaf(-6.0f * cp141(q - 1), wt, v);
            if (COPY) dst[k * dstride - 2] = v;
        }
    }
    if (k0 == 0) {
        dst[0] = 0.0f;
        if (COPY) dst[-2] = src[0];
    }
}

// Per-axis tables of the output->input map, computed once per call in float64 exactly as the
// definition (readings B1/B2) so that the tile kernel does no double-precision arithmetic:
//   tab[n]  = (interval index or -1 as int bits, t, C(t) = ((1-t)^2 - 1)(1-t), D(t) = (t^2 - 1) t)
//   tb[b]   = first output node whose (clamped) interval is >= b * tile cells; tb[nb] = n_out.
__global__ void __launch_bounds__(256)
spline_tables_kernel(AxisMap ax, AxisMap ay, float4* __restrict__ coltab, float4* __restrict__ rowtab,
                     int* __restrict__ tbx, int* __restrict__ tby, int nbx, int nby, int txi, int tyi)
{
    int n = blockIdx.x * 256 + threadIdx.x;
    if (n < ax.n_out + ay.n_out) {
        const bool isx = n < ax.n_out;
        const AxisMap& m = isx ? ax : ay;
        const int J = isx ? n : n - ax.n_out;
        float t;
        const int i = axis_locate(m, J, &t);
        const float a = 1.0f - t;
        (isx ? coltab : rowtab)[J] = make_float4(__int_as_float(i), t, (a * a - 1.0f) * a, (t * t - 1.0f) * t);
        return;
    }
    n -= ax.n_out + ay.n_out;
    if (n <= nbx) { tbx[n] = (n == nbx) ? ax.n_out : first_node_ge(ax, n * txi); return; }
    n -= nbx + 1;
    if (n <= nby) tby[n] = (n == nby) ? ay.n_out : first_node_ge(ay, n * tyi);
}

template <class S>
__global__ void __launch_bounds__(kTileThreads)
spline_tile_kernel(const float* __restrict__ in, float* __restrict__ out, AxisMap ax, AxisMap ay,
                   const float4* __restrict__ coltab, const float4* __restrict__ rowtab,
                   const int* __restrict__ tbx, const int* __restrict__ tby)
{
    constexpr int TXI = S::TXI, TYI = S::TYI, H = S::H, WX = S::WX, WY = S::WY;
    constexpr int NXI = S::NXI, NYI = S::NYI, PZ = S::PZ, PA = S::PA, PQ = S::PQ, RCAP = S::RCAP;
    constexpr int NW = kTileThreads / 32;
    extern __shared__ __align__(16) unsigned char s_raw[];
    float4* s_rowtab = reinterpret_cast<float4*>(s_raw);                 // (j bits, s, Cy, Dy) per output row
    float4* s_q = s_rowtab + RCAP;                                        // [NYI][PQ] knot records (z, My', Mx', Mxy')
    float* s_z = reinterpret_cast<float*>(s_q + NYI * PQ);                // [WY][PA] window: raw z, then z - zref
    float* s_my = s_z + WY * PA;                                          // [NYI][PZ] My' on the tile's knot rows

    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int i0 = blockIdx.x * TXI, j0 = blockIdx.y * TYI;               // first cell of the tile
    const int w0x = min(max(i0 - H, 0), ax.n_in - WX);                    // window origin (host guarantees n_in >= W)
    const int w0y = min(max(j0 - H, 0), ay.n_in - WY);
    const int kx0 = i0 - w0x, ky0 = j0 - w0y;                             // tile knot 0 in window coordinates
    const int nkx = min(NXI, ax.n_in - i0), nky = min(NYI, ay.n_in - j0); // knots present (last tile may be short)

    const int Jbeg = __ldg(tbx + blockIdx.x), Jend = __ldg(tbx + blockIdx.x + 1);   // output nodes of the tile
    const int Ibeg = __ldg(tby + blockIdx.y), Iend = __ldg(tby + blockIdx.y + 1);

    // ---- load the window: raw depths, whole 16-byte vectors from the aligned column at or before the
    //      window start, global -> shared without passing through registers (cp.async)
    const int ax0 = w0x & ~3, offx = w0x - ax0;
    if ((reinterpret_cast<uintptr_t>(in) & 15) == 0 && (ax.n_in & 3) == 0) {
        constexpr int VPR = PA / 4;
        for (int v = tid; v < WY * VPR; v += kTileThreads) {
            const int r = v / VPR, c4 = (v - r * VPR) * 4;
            const int col = ax0 + c4;
            const int bytes = max(0, min(16, (ax.n_in - col) * 4));      // past the row end: zero fill
            const float* src = in + (size_t)(w0y + r) * ax.n_in + min(col, ax.n_in - 4);
            const unsigned dst = (unsigned)__cvta_generic_to_shared(s_z + r * PA + c4);
            asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;" :: "r"(dst), "l"(src), "r"(bytes) : "memory");
        }
        asm volatile("cp.async.commit_group;" ::: "memory");
        asm volatile("cp.async.wait_group 0;" ::: "memory");
    } else {
        for (int v = tid; v < WY * WX; v += kTileThreads) {
            const int r = v / WX, c = v - r * WX;
            s_z[r * PA + offx + c] = __ldg(in + (size_t)(w0y + r) * ax.n_in + w0x + c);
        }
    }
    __syncthreads();
    float zref = s_z[offx];
    if (!isfinite(zref)) zref = 0.0f;
    __syncthreads();                                   // everybody has zref before the first column is rewritten

    // ---- S2: My' = Thomas along y of every window column, kept on the tile's knot rows
    const bool inner_y = (ky0 == H) && (nky == NYI), inner_x = (kx0 == H) && (nkx == NXI);   // CTA-uniform
    if (tid < WX) {
        if (inner_y) thomas_window<WY, true, H, NYI, false, true>(s_z + offx + tid, PA, s_my + tid, PZ, 0, 0, zref);
        else         thomas_window<WY, false, 0, 0, false, true>(s_z + offx + tid, PA, s_my + tid, PZ, ky0, nky, zref);
    }
    __syncthreads();

    // ---- S1: Mx' = Thomas along x of z on the knot rows (warp 0, fills Q.x, Q.z);
    //      S3: Mxy' = Thomas along x of My' (warp 1, fills Q.y, Q.w)
    if (warp < 2 && lane < nky) {
        float* src = warp == 0 ? s_z + (ky0 + lane) * PA + offx : s_my + lane * PZ;
        float* dst = reinterpret_cast<float*>(s_q + lane * PQ) + 2 + warp;
        if (inner_x) thomas_window<WX, true, H, NXI, true, false>(src, 1, dst, 4, 0, 0, 0.0f);
        else         thomas_window<WX, false, 0, 0, true, false>(src, 1, dst, 4, kx0, nkx, 0.0f);
    }

    // ---- S4: evaluate.  A warp owns a band of consecutive output rows and, per pass, 128 columns
    //      (a thread: 4 columns 32 apart, so every store instruction of a warp writes 128 contiguous
    //      bytes).  Per knot row and column the x-direction splines of z and My' come out of two
    //      LDS.128 and four packed fp32x2 FMAs as the pair (X, Y); per node the y-direction blend is
    //      three packed FMAs for two columns.
    const float qnan = __int_as_float(0x7fc00000);
    const u64 neg1 = pack2(-1.0f, -1.0f), zref2 = pack2(zref, zref);
    for (int Ic = Ibeg; Ic < Iend; Ic += RCAP) {
        const int nrows = min(RCAP, Iend - Ic);
        __syncthreads();                               // chains done / previous chunk's table no longer read
        for (int r = tid; r < nrows; r += kTileThreads) s_rowtab[r] = __ldg(rowtab + Ic + r);
        __syncthreads();
        const int r0 = (nrows * warp) / NW, r1 = (nrows * (warp + 1)) / NW;
        for (int Jp = Jbeg; Jp < Jend; Jp += 128) {
            const int Jt = Jp + lane;                  // column of e = 0; e-th column is 32 e further
            if (Jt >= Jend) continue;
            bool cok[4];
            float t[4], Cx[4], Dx[4], cnan[4];
            const float4* qc[4];                       // left knot record of the column's interval, knot row 0 of the tile
#pragma unroll
            for (int e = 0; e < 4; ++e) {
                const int J = Jt + 32 * e;
                cok[e] = J < Jend;
                const float4 ct = cok[e] ? __ldg(coltab + J) : make_float4(__int_as_float(-1), 0.0f, 0.0f, 0.0f);
                const int i = __float_as_int(ct.x);
                t[e] = ct.y; Cx[e] = ct.z; Dx[e] = ct.w;
                cnan[e] = (i < 0 && cok[e]) ? qnan : 0.0f;   // outside the input extent
                const int ic = (i < 0) ? i0 : i;
                qc[e] = s_q + (ic - i0);
            }
            // x-direction splines (X, Y) = S_x[z], S_x[My'] of knot row kj at this thread's 4 columns,
            // re-paired by column: X2[p] = (X[2p], X[2p+1])
            auto knot_row = [&](int kj, u64* X2, u64* Y2) {
                float xv[4], yv[4];
#pragma unroll
                for (int e = 0; e < 4; ++e) {
                    const ulonglong2 L = *reinterpret_cast<const ulonglong2*>(qc[e] + kj * PQ);
                    const ulonglong2 Hh = *reinterpret_cast<const ulonglong2*>(qc[e] + kj * PQ + 1);
                    u64 xy = ffma2(pack2(t[e], t[e]), ffma2(L.x, neg1, Hh.x), L.x);
                    xy = ffma2(pack2(Cx[e], Cx[e]), L.y, xy);
                    xy = ffma2(pack2(Dx[e], Dx[e]), Hh.y, xy);
                    xv[e] = lo_of(xy); yv[e] = hi_of(xy);
                }
                X2[0] = pack2(xv[0], xv[1]); X2[1] = pack2(xv[2], xv[3]);
                Y2[0] = pack2(yv[0], yv[1]); Y2[1] = pack2(yv[2], yv[3]);
            };
            u64 X0[2], X1[2], Xd[2], Y0[2], Y1[2];
#pragma unroll
            for (int p = 0; p < 2; ++p) X0[p] = X1[p] = Xd[p] = Y0[p] = Y1[p] = pack2(0.0f, 0.0f);
            const u64 cn2[2] = {pack2(cnan[0], cnan[1]), pack2(cnan[2], cnan[3])};
            int cur_j = -2;
            float* op = out + (size_t)(Ic + r0) * ax.n_out + Jt;
            for (int r = r0; r < r1; ++r, op += ax.n_out) {
                const float4 rw = s_rowtab[r];
                const int j = __float_as_int(rw.x);
                if (j != cur_j) {                      // warp-uniform: a new pair of knot rows
                    if (j < 0) {                       // row outside the input extent: NaN through X0
#pragma unroll
                        for (int p = 0; p < 2; ++p) { X0[p] = pack2(qnan, qnan); Xd[p] = Y0[p] = Y1[p] = pack2(0.0f, 0.0f); }
                    } else {
                        const int kj = j - j0;
                        if (j == cur_j + 1) {
#pragma unroll
                            for (int p = 0; p < 2; ++p) { X0[p] = X1[p]; Y0[p] = Y1[p]; }
                        } else {
                            knot_row(kj, X0, Y0);
                        }
                        knot_row(kj + 1, X1, Y1);
#pragma unroll
                        for (int p = 0; p < 2; ++p) {
                            Xd[p] = ffma2(X0[p], neg1, X1[p]);
                            X0[p] = fadd2(X0[p], cn2[p]);
                        }
                    }
                    cur_j = (j < 0) ? -3 : j;          // a NaN row never serves as "previous interval"
                }
                const u64 s2 = pack2(rw.y, rw.y), cy2 = pack2(rw.z, rw.z), dy2 = pack2(rw.w, rw.w);
#pragma unroll
                for (int p = 0; p < 2; ++p) {
                    u64 o = ffma2(s2, Xd[p], X0[p]);
                    o = ffma2(cy2, Y0[p], o);
                    o = ffma2(dy2, Y1[p], o);
                    o = fadd2(o, zref2);
                    if (cok[2 * p]) op[64 * p] = lo_of(o);
                    if (cok[2 * p + 1]) op[64 * p + 32] = hi_of(o);
                }
            }
        }
    }
}

template <class S>
int launch_tile(const float* d_in, float* d_out, const AxisMap& ax, const AxisMap& ay, void* d_ws, cudaStream_t stream)
{
    static bool attr_set = false;
    if (!attr_set) {
        BATHY_CUDA_TRY(cudaFuncSetAttribute(spline_tile_kernel<S>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                            (int)S::smem_bytes));
        attr_set = true;
    }
    dim3 grid((ax.n_in - 1 + S::TXI - 1) / S::TXI, (ay.n_in - 1 + S::TYI - 1) / S::TYI);
    float4* coltab = static_cast<float4*>(d_ws);
    float4* rowtab = coltab + ax.n_out;
    int* tbx = reinterpret_cast<int*>(rowtab + ay.n_out);
    int* tby = tbx + grid.x + 1;
    const long long items = (long long)ax.n_out + ay.n_out + grid.x + grid.y + 2;
    spline_tables_kernel<<<(unsigned)((items + 255) / 256), 256, 0, stream>>>(ax, ay, coltab, rowtab, tbx, tby,
                                                                              (int)grid.x, (int)grid.y, S::TXI, S::TYI);
    spline_tile_kernel<S><<<grid, kTileThreads, S::smem_bytes, stream>>>(d_in, d_out, ax, ay, coltab, rowtab, tbx, tby);
    count_launch(2);
    return launch_status();
}

}  // namespace

// Returns 1 when the geometry is not served by the fused path (the caller falls back to the
// global-solve path), else the launch status.
// Bytes of the axis tables at the start of the workspace (an upper bound over both tile shapes).
size_t spline_tiled_table_bytes(const grid_geom_t& in, const grid_geom_t& out)
{
    const size_t b = 16 * ((size_t)out.nx + (size_t)out.ny) + 4 * ((size_t)in.nx + (size_t)in.ny + 4);
    return (b + 255) / 256 * 256;
}

int launch_spline_tiled(const float* d_in, const grid_geom_t& in, float* d_out, const grid_geom_t& out,
                        void* d_ws, cudaStream_t stream)
{
    const AxisMap ax = axis_x(in, out), ay = axis_y(in, out);
    // up-sampling (or 1:1) only: a tile must produce at least about as many nodes as it reads knots
    if (!(out.dx <= in.dx) || !(out.dy <= in.dy)) return 1;
    using Big = TileShape<64, 31, 11>;
    using Small = TileShape<16, 16, 11>;
    if (in.nx >= Big::WX && in.ny >= Big::WY) {
        if ((in.ny - 1 + Big::TYI - 1) / Big::TYI > 65535) return 1;
        return launch_tile<Big>(d_in, d_out, ax, ay, d_ws, stream);
    }
    if (in.nx >= Small::WX && in.ny >= Small::WY) return launch_tile<Small>(d_in, d_out, ax, ay, d_ws, stream);
    return 1;
}

}  // namespace bathy
