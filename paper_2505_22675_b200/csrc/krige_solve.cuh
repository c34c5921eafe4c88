// krige_solve.cuh -- K3-K5 of ordinary kriging for a batch of nodes whose neighbour lists
// sit in shared memory: covariance build, Cholesky of C, Schur step for the Lagrange multiplier, estimate.
// Shared by krige_predict.cu (scattered soundings, kNN) and krige_window.cu (grid-window hole filling).
#pragma once
#include "common.cuh"

namespace bathy {

constexpr unsigned kFull = 0xffffffffu;
constexpr float kPivEps = 1e-6f;                 // smallest accepted Cholesky pivot (sill = 1)

// What the solve needs to know about the variogram and where its results go.
struct SolveParams {
    float cpn;          // (sill - nugget) / sill : partial sill of the covariance normalised to sill = 1
    float lc;           // log2(cpn)                                   (exponential, Gaussian)
    float c05, c15;     // 0.5 cpn, -1.5 cpn                           (spherical)
    float s_coord;      // coordinate scale of the solve: log2(e)/a (exponential), sqrt(log2 e)/a (Gaussian), 1/a (spherical)
    float sill;         // kriging variance is reported in the units of sill
    float* zhat;
    float* var;         // kriging variance (or NULL)
    unsigned long long* failed;
    unsigned long long* illcond;
};

inline void set_variogram(SolveParams& p, const variogram_t& vg)
{
    const double cpn = ((double)vg.sill - (double)vg.nugget) / (double)vg.sill;
    p.cpn = (float)cpn;
    p.lc = cpn > 0.0 ? (float)log2(cpn) : -INFINITY;
    p.c05 = (float)(0.5 * cpn);
    p.c15 = (float)(-1.5 * cpn);
    p.s_coord = (vg.model == BATHY_VGM_EXPONENTIAL) ? (float)(1.4426950408889634 / (double)vg.range)
              : (vg.model == BATHY_VGM_GAUSSIAN)    ? (float)(sqrt(1.4426950408889634) / (double)vg.range)
                                                    : (float)(1.0 / (double)vg.range);
    p.sill = vg.sill;
}

template <int K, int G>
struct Shape {
    static constexpr int R = K / G;             // rows of C per lane
    static constexpr int NB = 32 / G;           // nodes solved by a warp at once
    static constexpr int CAP = (K <= 32) ? 256 : 512;          // shared candidate list
    static constexpr int WARPS = 8;                            // warps per CTA
    // CTAs per SM (registers: 128 per thread at K <= 32, 255 at K = 64).  Two CTAs of 8 warps instead of one of 16:
    // each CTA walks the long unrolled solve code together (instruction cache), but the two are in different
    // phases -- one searches (integer / shared-memory work) while the other solves (FMA work).  Measured on
    // config 4: 4.88 -> 4.68 ms; four CTAs of 4 warps 4.91 ms; at K = 64 two CTAs of 4 warps 7.2 against 5.8 ms.
    static constexpr int CTAS = (K <= 32) ? 2 : 1;           // warps per CTA: one CTA per SM (registers)
    static constexpr int NQ = CAP / 32;
    static constexpr int XYS = K + 4;           // float stride of a node's coordinate lists (bank skew)
    // float stride of a node's column buffer: = G (mod 32), so that the NB x G lanes of a warp, each
    // storing one entry of its node's column, hit 32 different banks (K + 4 gave 2-way conflicts)
    static constexpr int CBS = K + ((G - K) % 32 + 32) % 32;
    static constexpr bool ILV = (K > 32);       // lane <-> (node, row group) mapping of the solve, see solve_batch
    static constexpr int NBLP = 33;             // pitch of the per-lane uint16 lists: 16.5 words, so that one lane's
                                                // column (the gather before the solve) spreads over all banks
};

template <int K, int G>
struct __align__(16) SolveSmem {
    using S = Shape<K, G>;
    float4   rhs[2][S::NB];                     // (rhs_z, rhs_1, rhs_c, pivot) of row 0, per node (slot [1])
    float    colbuf[2][S::NB][S::CBS];          // -(column j of L), per node (double buffered)
    float    nb_x[S::NB][S::XYS];               // neighbour coordinates, scaled, relative to the block centre
    float    nb_y[S::NB][S::XYS];
    float    nb_z[S::NB][K];                    // neighbour depths
};

__device__ __forceinline__ float rsqrt_approx(float v)
{
    float r;
    asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(v));
    return r;
}

__device__ __forceinline__ float ex2_approx(float v)
{
    float r;
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(v));
    return r;
}


// Two covariances at once, normalised to sill = 1, from squared distances in SCALED coordinates (h2 > 0):
// exponential C = cpn exp(-h/a) = 2^(log2 cpn - h log2(e)/a) (no factor 3);
// spherical   C = cpn (1 - 1.5 q + 0.5 q^3), q = min(h/a, 1);  Gaussian C = cpn exp(-(h/a)^2) (NEXT-4).  h2 == 0 gives NaN (0 * inf): two
// soundings at one place make the system singular and the node fails (reading K-dup).
// The distance and polynomial arithmetic is packed fp32x2; the two rsqrt and the two ex2 go to the
// MUFU pipe one by one.
template <int MODEL>
__device__ __forceinline__ u64 cov2_scaled(u64 h2, const SolveParams& p)
{
    const u64 rs2 = pack2(rsqrt_approx(lo_of(h2)), rsqrt_approx(hi_of(h2)));
    const u64 q2 = fmul2(h2, rs2);                         // scaled distances
    if (MODEL == BATHY_VGM_EXPONENTIAL) {
        const u64 a2 = ffma2(q2, pack2(-1.0f, -1.0f), pack2(p.lc, p.lc));
        return pack2(ex2_approx(lo_of(a2)), ex2_approx(hi_of(a2)));
    } else if (MODEL == BATHY_VGM_GAUSSIAN) {
        // C = cpn exp(-(h/a)^2) = 2^(log2 cpn - q^2), coordinates pre-scaled by sqrt(log2 e)/a; q = h2 rsqrt(h2)
        // rather than h2 itself so that h2 == 0 (duplicate soundings) still gives NaN
        const u64 a2 = ffma2(fmul2(q2, pack2(-1.0f, -1.0f)), q2, pack2(p.lc, p.lc));
        return pack2(ex2_approx(lo_of(a2)), ex2_approx(hi_of(a2)));
    } else {
        float qa, qb;
        asm("min.NaN.f32 %0, %1, %2;" : "=f"(qa) : "f"(lo_of(q2)), "f"(1.0f));   // NaN (h2 == 0) survives
        asm("min.NaN.f32 %0, %1, %2;" : "=f"(qb) : "f"(hi_of(q2)), "f"(1.0f));
        const u64 q = pack2(qa, qb);
        const u64 pp = ffma2(fmul2(q, q), pack2(p.c05, p.c05), pack2(p.c15, p.c15));
        return ffma2(q, pp, pack2(p.cpn, p.cpn));
    }
}

// K3-K5 for the NB nodes whose neighbour lists (scaled coordinates relative to the block centre,
// depths) sit in ws.nb_x, ws.nb_y, ws.nb_z.  Lane (nd, g) = (lane / G, lane % G) holds rows g, g+G, ...
// (at k = 64 the nodes are interleaved instead, (nd, g) = (lane % NB, lane / NB).  Measured: k = 64 6.07 ->
// 5.98 ms per 1 M nodes; at k = 32 the broadcast column loads get slower, 5.55 -> 6.02 ms)
// of node nd, two columns to a 64-bit register pair.  Rows at or beyond k are pad soundings placed
// far away from everything (covariance exactly 0): they decouple as identity rows with zero
// right-hand sides.
template <int K, int G, int MODEL, bool EX>
__device__ __forceinline__ void solve_batch(const SolveParams& p, SolveSmem<K, G>& ws, int lane,
                                            float xs, float ys, bool node_ok, long long node, int k)
{
    using S = Shape<K, G>;
    constexpr int R = S::R;
    static_assert(G % 2 == 0 && K % 4 == 0, "column pairs must not straddle a row block");
    const int nd = S::ILV ? lane % S::NB : lane / G, g = S::ILV ? lane / S::NB : lane % G;
    const float zref = ws.nb_z[nd][0];

    u64 A2[R][K / 2];                // A2[t][q] = (A[t][2q], A[t][2q+1]): row g + G t (only 2q < (t+1) G is live)
    u64 yz1[R];                      // right-hand sides (z - z_ref, 1) of the row
    float yc[R];                     // right-hand side c0 of the row
    float xr[R], yr[R];
#pragma unroll
    for (int t = 0; t < R; ++t) {
        const int r = g + G * t;
        xr[t] = ws.nb_x[nd][r]; yr[t] = ws.nb_y[nd][r];
        const float ddx = xs - xr[t], ddy = ys - yr[t];
        const float h2 = fmaf(ddx, ddx, ddy * ddy);
        const float c0 = lo_of(cov2_scaled<MODEL>(pack2(h2, h2), p));
        yc[t] = (h2 > 0.0f) ? c0 : 1.0f;                   // gamma(0) = 0: a node on a datum sees the full sill
        yz1[t] = pack2(ws.nb_z[nd][r] - zref, (r < k) ? 1.0f : 0.0f);
    }
    // K3: block-lower triangle of C, two columns at a time in packed fp32x2 arithmetic
    const u64 neg1 = pack2(-1.0f, -1.0f);
#pragma unroll
    for (int q = 0; q < K / 2; ++q) {
        const u64 cx2 = *reinterpret_cast<const u64*>(&ws.nb_x[nd][2 * q]);    // x of columns 2q, 2q+1
        const u64 cy2 = *reinterpret_cast<const u64*>(&ws.nb_y[nd][2 * q]);
#pragma unroll
        for (int t = (2 * q) / G; t < R; ++t) {
            const u64 dx2 = ffma2(cx2, neg1, pack2(xr[t], xr[t]));
            const u64 dy2 = ffma2(cy2, neg1, pack2(yr[t], yr[t]));
            u64 c2 = cov2_scaled<MODEL>(ffma2(dx2, dx2, fmul2(dy2, dy2)), p);
            if (t == (2 * q) / G) {                        // the diagonal: sill
                const float ca = (g == (2 * q) % G) ? 1.0f : lo_of(c2);
                const float cb = (g == (2 * q + 1) % G) ? 1.0f : hi_of(c2);
                c2 = pack2(ca, cb);
            }
            A2[t][q] = c2;
        }
    }

    // K4: right-looking Cholesky, column by column; the three right-hand sides are forward-substituted
    // on the way and their four dot products (the Schur step, K5) accumulate as the y_j appear.
    // Row j's owner hands P_j = (rhs_z, rhs_1, rhs_c, pivot) of its row to the lanes of its node -- final
    // once column j-1 has been applied, which it can do for its own row before anybody else has seen
    // that column -- in the same phase as column j-1 itself, by four shuffles: one __syncwarp per
    // column, and the rsqrt of the next pivot overlaps the trailing update.  (Row 0 goes through
    // ws.rhs once: replacing that by shuffles too changes nothing at k = 32 and costs 2 % at k = 64,
    // where the kernel is at the register limit.)
    float pmin = 1.0f;               // smallest pivot (a NaN pivot poisons every later column and the estimate)
    u64 dots_c = pack2(0.0f, 0.0f);  // (y_c.y_z, y_c.y_1)
    u64 dots_1 = pack2(0.0f, 0.0f);  // (y_1.y_z, y_1.y_1)
    float dcc = 0.0f;                // y_c.y_c (kriging variance)
    if (g == 0) ws.rhs[1][nd] = make_float4(lo_of(yz1[0]), hi_of(yz1[0]), yc[0], lo_of(A2[0][0]));
    __syncwarp();
    ulonglong2 P = *reinterpret_cast<const ulonglong2*>(&ws.rhs[1][nd]);
#pragma unroll
    for (int j = 0; j < K; ++j) {
        const int tj = j / G, gj = j % G, buf = j & 1;
        const float piv = hi_of(P.y);
        pmin = fminf(pmin, piv);
        const float inv = rsqrt_approx(piv);
        const u64 yj = pack2(lo_of(P.x) * inv, hi_of(P.x) * inv);      // (y_z, y_1) of column j
        const float ycj = lo_of(P.y) * inv, y1j = hi_of(yj);
        dots_c = ffma2(pack2(ycj, ycj), yj, dots_c);
        dots_1 = ffma2(pack2(y1j, y1j), yj, dots_1);
        if (EX) dcc = fmaf(ycj, ycj, dcc);
        float nLr[R];
#pragma unroll
        for (int t = tj; t < R; ++t) {
            const float a = (j & 1) ? hi_of(A2[t][j / 2]) : lo_of(A2[t][j / 2]);
            float sc = inv;
            if (t == tj) sc = (g > gj) ? inv : 0.0f;       // rows <= j of the diagonal block are finished
            const float l = a * sc;
            ws.colbuf[buf][nd][g + G * t] = l;
            nLr[t] = -l;
            yz1[t] = ffma2(pack2(nLr[t], nLr[t]), yj, yz1[t]);
            yc[t] = fmaf(nLr[t], ycj, yc[t]);
        }
        if (j + 1 < K) {                                   // P_{j+1}: row j+1 with column j applied
            const int t1 = (j + 1) / G, g1 = (j + 1) % G;
            const float a1 = ((j + 1) & 1) ? hi_of(A2[t1][(j + 1) / 2]) : lo_of(A2[t1][(j + 1) / 2]);
            const float pv = fmaf(nLr[t1], -nLr[t1], a1);
            // from the row's owner to the lanes of its node: four shuffles (a 16-byte store by the 4
            // owners, one per quarter-warp, plus the load back cost 6 shared-memory wavefronts)
            const int owner = S::ILV ? (lane % S::NB) + S::NB * g1 : (lane & ~(G - 1)) | g1;
            P.x = __shfl_sync(kFull, yz1[t1], owner);
            P.y = pack2(__shfl_sync(kFull, yc[t1], owner), __shfl_sync(kFull, pv, owner));
        }
        __syncwarp();
#pragma unroll
        for (int m4 = (j + 1) / 4; m4 < K / 4; ++m4) {
            const ulonglong2 L4 = *reinterpret_cast<const ulonglong2*>(&ws.colbuf[buf][nd][4 * m4]);
#pragma unroll
            for (int e = 0; e < 2; ++e) {
                const int q = 2 * m4 + e;                  // columns 2q, 2q+1
                if (2 * q + 1 > j) {
                    const u64 Lq = e ? L4.y : L4.x;
#pragma unroll
                    for (int t = ((2 * q) / G > tj ? (2 * q) / G : tj); t < R; ++t)
                        A2[t][q] = ffma2(pack2(nLr[t], nLr[t]), Lq, A2[t][q]);
                }
            }
        }
    }

    if (g == 0 && node_ok) {
        const float dcz = lo_of(dots_c), d1c = hi_of(dots_c), d1z = lo_of(dots_1), d11 = hi_of(dots_1);
        const float mu = (d1c - 1.0f) / d11;
        float est = zref + (dcz - mu * d1z);
        // kriging variance (sill = 1): 1 - c0^T C^-1 c0 + mu (1^T C^-1 c0 - 1) = 1 - y_c.y_c + mu^2 (y_1.y_1)
        float var = EX ? p.sill * ((1.0f - dcc) + mu * mu * d11) : 0.0f;
        if (!(pmin > kPivEps) || !(est == est)) {
            est = var = __int_as_float(0x7fc00000);
            if (p.failed) atomicAdd(p.failed, 1ull);
        } else if (EX && p.illcond && pmin < BATHY_ILLCOND_PIVOT) {
            atomicAdd(p.illcond, 1ull);
        }
        p.zhat[node] = est;
        if (EX && p.var) p.var[node] = var;
    }
}

}  // namespace bathy
