// krige_predict.cu -- ordinary kriging at every node of the output grid (
// SURVEY.md 8(a) rows K2-K5).
//
// One warp owns a BW x BH = 8 x 4 block of output nodes, lane l <-> node (l % 8, l / 8).
//   K2  search, in two levels:
//       pilot    the warp finds a key bound T such that at least k soundings lie within sqrt(T) of the
//                block centre c (cell-grid scan + bisection on the key bits).  By the triangle
//                inequality the k-th key of node q is then at most hi_q = (sqrt(T) + |q - c|)^2.
//       gather   every sounding closer than sqrt(T) + max|q - c| to the block rectangle is copied once
//                into shared memory (the candidate list all 32 nodes share; ~5 soundings per node).
//       select   ONE THREAD PER NODE: pass 1 histograms the fp32 keys (reading K2: the defined
//                expression) of the shared candidates into 32 buckets that are uniform in key over
//                [0, hi_q] (private column of a shared-memory histogram); a scan finds the bucket b*
//                that holds the k-th key; pass 2 takes every candidate below b* and lists the few in
//                b*, among which the (key, index) ranking picks the rest -- exact, ties by index.
//                No cross-lane traffic: a node's selection costs ~1/32 warp instruction per thread
//                instruction, instead of a warp-wide bisection per node.
//       A candidate list that does not fit splits the block into half blocks (down to single nodes).
//   K3-K5 solve: G lanes per node (32/G nodes per warp at once), rows of C dealt cyclically to the
//       lanes and held in REGISTERS as fp32x2 pairs (fully unrolled right-looking Cholesky, FFMA2
//       trailing update); column j of L is published through a double-buffered shared-memory column
//       and read back as broadcast LDS.128.
//       The three right-hand sides c0, 1 and z ride along as forward substitutions, and
//           z_hat = y_z.y_c - mu * (y_z.y_1),   mu = (y_1.y_c - 1) / (y_1.y_1),   y_b = L^-1 b
//       gives the Lagrange/Schur step without any back substitution or explicit weights.
//       Covariances are built from coordinates relative to the block centre, pre-scaled by
//       log2(e)/a (exponential) or 1/a (spherical), two pairs per packed fp32x2 operation.
//   Tensor cores are not used: the factorisation is a k x k problem with a serial pivot chain.
#include "krige_index.cuh"
#include "krige_solve.cuh"

namespace bathy {

namespace {

constexpr int BW = 8, BH = 4;                    // node block of a warp
constexpr int kBuckets = 32;                     // key histogram of the per-node selection
constexpr int kCrit = 16;                        // listed candidates of the critical bucket

// The cell grid of the index, read from its DEVICE header at kernel start (the host never sees it:
// krige_build_index only enqueues) and kept in shared memory; r0 / rmax are derived from it there.
struct GridInfo {
    float xmin, ymin, inv_cell, cell;
    int ncx, ncy;
    float r0;           // first pilot radius
    float rmax;         // radius that certainly covers every sounding from any node of this call
    int bad;            // the index is unusable (non-finite soundings, or fewer than k of them): every node fails
};

struct PredictParams : SolveParams {
    const float4* pts;
    const int32_t* cell_start;
    const IndexHeader* hdr;
    float r0_factor;    // first pilot radius / mean sounding spacing: the radius that holds ~1.5 k soundings
    int nx, ny;
    float x0, y0, dx, dy;
    int k;
    int32_t* nbr;
    int nbx, nby;       // blocks per row / column of blocks
    int chain;          // consecutive blocks walked by one warp
    long long n_blocks;
    // Coordinate map of the solve (block-relative fp32 coordinates -> the scaled coordinates the covariances are built
    // from): (u, w) = (m00 dx + m01 dy, m10 dx + m11 dy).  Isotropic: s_coord times the identity.  Geometric anisotropy
    // (krige_predict_aniso; reading Ani): s_coord * diag(1, 1/ratio) * rotation by -angle.  s_pad = the map's
    // largest stretch (s_coord / ratio): what the far-away pad soundings are placed with.
    float m00, m01, m10, m11, s_pad;
    int aniso;          // the map is not the identity: the launch takes the EX instantiation (the only one that applies it)
};

// The map, as ONE expression used for neighbours and nodes alike: a node that coincides with a sounding gets the
// same (u, w) bit for bit and sees h2 == 0 exactly.  With m01 = m10 = 0 the fused multiply-adds add an exact zero:
// the isotropic coordinates are bit-identical to s_coord * dx, s_coord * dy.
// Only the EX instantiations of the kernel (extra outputs, anisotropy) carry the two extra multiply-adds per stored
// coordinate; the plain krige_predict kernels keep the bare scaling (measured: the general map in every kernel cost
// 0.9 % on config 4).
template <bool EX>
__device__ __forceinline__ float2 map_coord(const PredictParams& p, float dx, float dy)
{
    if (EX) return make_float2(__fmaf_rn(p.m01, dy, __fmul_rn(p.m00, dx)), __fmaf_rn(p.m10, dx, __fmul_rn(p.m11, dy)));
    return make_float2(__fmul_rn(dx, p.s_coord), __fmul_rn(dy, p.s_coord));
}

// A warp's shared memory: the solve's part (krige_solve.cuh) followed by the search's.
template <int K, int G>
struct __align__(16) WarpSmem : SolveSmem<K, G> {
    using S = Shape<K, G>;
    float    cx[S::CAP];                        // candidates: coordinates as given (fp32), as two planes so
    float    cy[S::CAP];                        //             that two candidates load as one fp32x2 pair
    float    cz[S::CAP];                        //             depth (pilot: key bits)
    int32_t  cid[S::CAP];                       //             original index
    uint16_t hist[kBuckets + 1][32];            // per-lane key histogram (column = lane)
    uint16_t nbl[K][S::NBLP];                   // per-lane neighbour list: candidate slots
    uint16_t crit[kCrit][32];                   // per-lane candidates of the critical bucket (the last row is a dump slot)
};

// Reading K2: key = fmaf(ddx, ddx, ddy*ddy) in fp32, ddx = xq - x_i, ddy = yq - y_i.
__device__ __forceinline__ float knn_key(float xq, float yq, float x, float y)
{
    const float ddx = __fsub_rn(xq, x), ddy = __fsub_rn(yq, y);
    return __fmaf_rn(ddx, ddx, __fmul_rn(ddy, ddy));
}

// ---------------------------------------------------------------------------------------------
// Cell-grid scan: calls f(in_range, pt, n_so_far) for every sounding of the cells that overlap
// [xlo, xhi] x [ylo, yhi], 32 soundings at a time (one per lane); f returns the keep predicate and
// the scan compacts the kept ones: store(slot, pt) is called with consecutive slots.  Returns the
// number kept (it may exceed `cap`, in which case the stores beyond cap were skipped).
template <class Keep, class Store>
__device__ __forceinline__ int scan_cells(const PredictParams& p, const GridInfo& gi, int lane, float xlo, float xhi, float ylo, float yhi,
                                          int cap, Keep keep_fn, Store store_fn)
{
    const float slack = 2e-3f * gi.cell;                   // cell_of() rounding slack
    const int ncx = gi.ncx;
    const int cx0 = cell_of(xlo - slack, gi.xmin, gi.inv_cell, ncx), cx1 = cell_of(xhi + slack, gi.xmin, gi.inv_cell, ncx);
    const int cy0 = cell_of(ylo - slack, gi.ymin, gi.inv_cell, gi.ncy), cy1 = cell_of(yhi + slack, gi.ymin, gi.inv_cell, gi.ncy);
    int n = 0;
    for (int cyb = cy0; cyb <= cy1; cyb += 32) {
        const int cy = cyb + lane;
        int seg_s = 0, seg_e = 0;
        if (cy <= cy1) {
            seg_s = __ldg(p.cell_start + (size_t)cy * ncx + cx0);
            seg_e = __ldg(p.cell_start + (size_t)cy * ncx + cx1 + 1);
        }
        const int rows = min(32, cy1 - cyb + 1);
        for (int rr = 0; rr < rows; ++rr) {
            const int s = __shfl_sync(kFull, seg_s, rr), e = __shfl_sync(kFull, seg_e, rr);
            for (int base = s; base < e; base += 32) {
                const int pos = base + lane;
                float4 pt = make_float4(0.0f, 0.0f, 0.0f, 0.0f);
                bool keep = false;
                if (pos < e) {
                    pt = __ldg(p.pts + pos);
                    keep = keep_fn(pt);
                }
                const unsigned m = __ballot_sync(kFull, keep);
                const int off = n + __popc(m & ((1u << lane) - 1u));
                if (keep && off < cap) store_fn(off, pt);
                n += __popc(m);
            }
        }
    }
    return n;
}

// K2 pilot: a key bound T with at least k soundings within sqrt(T) of (cx, cy) and not many more.
// `r` is the radius to try first and returns the radius that worked.  Returns a negative value for
// degenerate input (more than CAP soundings at one distance).
template <int K, int G>
__device__ __forceinline__ float pilot(const PredictParams& p, const GridInfo& gi, WarpSmem<K, G>& ws, int lane, float cx, float cy, float& r)
{
    using S = Shape<K, G>;
    const int k = p.k;
    uint32_t* keys = reinterpret_cast<uint32_t*>(ws.cz);
    float r_low = 0.0f, r_high = INFINITY;
    int n = 0;
    uint32_t key_hi = 0;
    bool found = false;
    for (int it = 0; it < 96; ++it) {
        key_hi = __float_as_uint(fminf(r * r * 1.00001f, 3.0e38f));
        n = scan_cells(p, gi, lane, cx - r, cx + r, cy - r, cy + r, S::CAP,
                       [&](const float4& pt) { return __float_as_uint(knn_key(cx, cy, pt.x, pt.y)) <= key_hi; },
                       [&](int slot, const float4& pt) { keys[slot] = __float_as_uint(knn_key(cx, cy, pt.x, pt.y)); });
        if (n < k) {
            if (r >= gi.rmax) break;                       // cannot happen for k <= n
            r_low = r;
            r = isinf(r_high) ? fminf(r * 1.5f, gi.rmax) : 0.5f * (r_low + r_high);
        } else if (n > S::CAP) {
            r_high = r;
            r = 0.5f * (r_low + r_high);
        } else { found = true; break; }
    }
    __syncwarp();
    if (!found) return -1.0f;
    // tighten: T = the smallest value of a fixed grid (fp32 patterns whose low 16 bits are all ones:
    // 0.8 % steps) with at least k keys at or below it.  It depends on the soundings and the centre
    // only -- not on the radius the scan happened to use -- so a block gives the same candidate
    // list, hence bit-identical depths, whatever call, tile or launch shape it is part of.
    uint32_t ck[S::NQ];
#pragma unroll
    for (int q = 0; q < S::NQ; ++q) {
        const int c = lane + 32 * q;
        ck[q] = (c < n) ? keys[c] : 0xffffffffu;
    }
    uint32_t lo = 0, hi = key_hi >> 16;
    while (lo < hi) {
        const uint32_t mid = lo + ((hi - lo) >> 1);
        const uint32_t v = (mid << 16) | 0xffffu;
        int c = 0;
#pragma unroll
        for (int q = 0; q < S::NQ; ++q) c += (ck[q] <= v) ? 1 : 0;
        c = (int)__reduce_add_sync(kFull, (unsigned)c);
        if (c >= k) hi = mid; else lo = mid + 1;
    }
    hi = (hi << 16) | 0xffffu;
    __syncwarp();
    return __uint_as_float(hi);
}

// Bucket of a key in the per-lane histogram: round(key * scale) through the 1.5 * 2^23 magic
// constant (no F2I).  Monotone non-decreasing in key, which is all the selection needs.
__device__ __forceinline__ int bucket_of(float key, float scale)
{
    return __float_as_int(fmaf(key, scale, 12582912.0f)) - 0x4B400000;
}

// K2 select, one thread per node: the k candidates with the smallest (key, original index) among
// the n_c shared candidates, all of them known to have key <= hi (hi < 0: lane idle).  Fills the
// lane's column of ws.nbl with candidate slots.  Returns false if fewer than k candidates qualify
// (cannot happen when hi is a valid bound).
template <int K, int G>
__device__ __forceinline__ bool select_per_lane(const PredictParams& p, WarpSmem<K, G>& ws, int lane, int n_c,
                                                float xq, float yq, float hi)
{
    const int k = p.k;
    const float scale = (float)kBuckets / fmaxf(hi, 1e-30f);
#pragma unroll
    for (int b = 0; b <= kBuckets; ++b) ws.hist[b][lane] = (uint16_t)0;
    // pass 1: histogram of the keys
    // Two candidates at a time in packed fp32x2 arithmetic: every operation is the round-to-nearest
    // operation of reading K2 (x*(-1) + xq is exactly xq - x), so the keys are bit-identical to knn_key.
    // (The caller pads an odd list with a candidate at infinity: its key is +inf.)
    const u64 xq2 = pack2(xq, xq), yq2 = pack2(yq, yq), neg1 = pack2(-1.0f, -1.0f);
    const u64 sc2 = pack2(scale, scale), mg2 = pack2(12582912.0f, 12582912.0f);
    // keys and buckets of the candidate pair (X, Y) = (cx[c..c+1], cy[c..c+1])
    auto keys2 = [&](u64 X, u64 Y, float& k0, float& k1, int& b0, int& b1) {
        const u64 dx = ffma2(X, neg1, xq2), dy = ffma2(Y, neg1, yq2);
        const u64 kk = ffma2(dx, dx, fmul2(dy, dy));
        const u64 bb = ffma2(kk, sc2, mg2);
        k0 = lo_of(kk); k1 = hi_of(kk);
        b0 = __float_as_int(lo_of(bb)) - 0x4B400000; b1 = __float_as_int(hi_of(bb)) - 0x4B400000;
    };
    auto ldpair = [&](int c, u64& X, u64& Y) {
        X = *reinterpret_cast<const u64*>(&ws.cx[c]); Y = *reinterpret_cast<const u64*>(&ws.cy[c]);
    };
    // Both passes are software-pipelined by hand: the next pair's coordinates are loaded BEFORE this pair's
    // shared-memory stores (the compiler does not move a load above a store it cannot prove disjoint, and the
    // loop would otherwise pay a full shared-memory round trip per pair), and the two histogram counters of a pair
    // are read together.  (Reading one pair past the list is harmless: the arrays are followed by others.)
    {
        u64 X, Y;
        ldpair(0, X, Y);
#pragma unroll 4
        for (int c = 0; c < n_c; c += 2) {
            u64 Xn, Yn;
            ldpair(c + 2, Xn, Yn);
            float k0, k1; int b0, b1;
            keys2(X, Y, k0, k1, b0, b1);
            const bool in0 = k0 <= hi, in1 = k1 <= hi;
            const int s0 = in0 ? b0 : 0, s1 = in1 ? b1 : 0;                // out of range: a harmless read of bucket 0
            const unsigned h0 = ws.hist[s0][lane], h1 = ws.hist[s1][lane];
            if (in0) ws.hist[s0][lane] = (uint16_t)(h0 + 1u);
            if (in1) ws.hist[s1][lane] = (uint16_t)(((in0 && s1 == s0) ? h0 + 1u : h1) + 1u);
            X = Xn; Y = Yn;
        }
    }
    // the bucket that holds the k-th key
    int bstar = kBuckets + 1, below = 0, cum = 0;
#pragma unroll
    for (int b = 0; b <= kBuckets; ++b) {
        const int h = (int)ws.hist[b][lane];
        if (bstar > kBuckets && cum + h >= k) { bstar = b; below = cum; }
        cum += h;
    }
    if (hi < 0.0f) return true;
    if (bstar > kBuckets) return false;
    // pass 2: everything below the critical bucket is a neighbour; the critical bucket is listed
    int cnt = 0, ncrit = 0;
    {
        u64 X, Y;
        ldpair(0, X, Y);
#pragma unroll 4
        for (int c = 0; c < n_c; c += 2) {
            u64 Xn, Yn;
            ldpair(c + 2, Xn, Yn);
            float k0, k1; int b0, b1;
            keys2(X, Y, k0, k1, b0, b1);
            // branch-free: the slot is written unconditionally and only kept (the counter advanced) when the candidate
            // qualifies -- the next candidate overwrites it otherwise.  cnt <= below < k, so nbl[cnt] is inside the list;
            // the last row of the critical list is its dump slot: the list holds at most kCrit - 1 candidates.
            const bool t0 = b0 < bstar, c0 = (b0 == bstar) && (k0 <= hi);       // (b < bstar <= 32 implies key < hi)
            ws.nbl[cnt][lane] = (uint16_t)c;
            ws.crit[min(ncrit, kCrit - 1)][lane] = (uint16_t)c;
            cnt += t0 ? 1 : 0; ncrit += c0 ? 1 : 0;
            const bool t1 = b1 < bstar, c1 = (b1 == bstar) && (k1 <= hi);
            ws.nbl[cnt][lane] = (uint16_t)(c + 1);
            ws.crit[min(ncrit, kCrit - 1)][lane] = (uint16_t)(c + 1);
            cnt += t1 ? 1 : 0; ncrit += c1 ? 1 : 0;
            X = Xn; Y = Yn;
        }
    }
    const int need = k - below;                            // >= 1 candidates of the critical bucket
    if (ncrit < kCrit) {
        for (int e = 0; e < ncrit; ++e) {                  // rank by (key, index) inside the bucket
            const int ce = ws.crit[e][lane];
            const float2 xe = make_float2(ws.cx[ce], ws.cy[ce]);
            const uint32_t ke = __float_as_uint(knn_key(xq, yq, xe.x, xe.y));
            const int32_t ie = ws.cid[ce];
            int rank = 0;
            for (int f = 0; f < ncrit; ++f) {
                const int cf = ws.crit[f][lane];
                const float2 xf = make_float2(ws.cx[cf], ws.cy[cf]);
                const uint32_t kf = __float_as_uint(knn_key(xq, yq, xf.x, xf.y));
                const int32_t jf = ws.cid[cf];
                rank += (kf < ke || (kf == ke && jf < ie)) ? 1 : 0;
            }
            if (rank < need) { ws.nbl[cnt][lane] = (uint16_t)ce; ++cnt; }
        }
    } else {
        // the list overflowed (many ties): take the `need` smallest (key, index) of the bucket one by one
        uint32_t lk = 0; int32_t li = -1;                  // last taken
        for (int t = 0; t < need; ++t) {
            uint32_t bk = 0xffffffffu; int32_t bi = 0x7fffffff; int bc = -1;
            for (int c = 0; c < n_c; ++c) {
                const float2 xy = make_float2(ws.cx[c], ws.cy[c]);
                const float key = knn_key(xq, yq, xy.x, xy.y);
                if (!(key <= hi) || bucket_of(key, scale) != bstar) continue;
                const uint32_t kc = __float_as_uint(key);
                const int32_t ic = ws.cid[c];
                const bool after = (kc > lk) || (kc == lk && ic > li);
                const bool better = (kc < bk) || (kc == bk && ic < bi);
                if (after && better) { bk = kc; bi = ic; bc = c; }
            }
            if (bc < 0) return false;
            ws.nbl[cnt][lane] = (uint16_t)bc; ++cnt;
            lk = bk; li = bi;
        }
    }
    return cnt == k;
}

// Parity/debug output, one thread per node: neighbours in ascending (key, index) order.
template <int K, int G>
__device__ __forceinline__ void write_sorted_nbr(const PredictParams& p, WarpSmem<K, G>& ws, int lane,
                                                 float xq, float yq, long long node)
{
    const int k = p.k;
    for (int e = 0; e < k; ++e) {
        const int ce = ws.nbl[e][lane];
        const float2 xe = make_float2(ws.cx[ce], ws.cy[ce]);
        const uint32_t ke = __float_as_uint(knn_key(xq, yq, xe.x, xe.y));
        const int32_t ie = ws.cid[ce];
        int rank = 0;
        for (int f = 0; f < k; ++f) {
            const int cf = ws.nbl[f][lane];
            const float2 xf = make_float2(ws.cx[cf], ws.cy[cf]);
            const uint32_t kf = __float_as_uint(knn_key(xq, yq, xf.x, xf.y));
            const int32_t jf = ws.cid[cf];
            rank += (kf < ke || (kf == ke && jf < ie)) ? 1 : 0;
        }
        p.nbr[node * k + rank] = ie;
    }
}

// EX: the krige_predict_ex outputs (kriging variance, ill-conditioning counter) are compiled in
template <int K, int G, int MODEL, bool EX>
__global__ void __launch_bounds__(Shape<K, G>::WARPS * 32, Shape<K, G>::CTAS)
krige_predict_kernel(const PredictParams p)
{
    using S = Shape<K, G>;
    extern __shared__ __align__(16) unsigned char s_raw[];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    WarpSmem<K, G>& ws = reinterpret_cast<WarpSmem<K, G>*>(s_raw)[warp];
    const long long wid = (long long)blockIdx.x * S::WARPS + warp;
    const long long b0 = wid * p.chain;
    const long long b1 = min(b0 + (long long)p.chain, p.n_blocks);
    const int k = p.k;
    const float qnan = __int_as_float(0x7fc00000);
    __shared__ GridInfo gi;
    if (threadIdx.x == 0) {
        const IndexHeader h = *p.hdr;
        gi.xmin = h.xmin; gi.ymin = h.ymin; gi.inv_cell = h.inv_cell; gi.cell = h.cell; gi.ncx = h.ncx; gi.ncy = h.ncy;
        // farthest any node of this call can be from any sounding: covers the union of both extents
        const double bx1 = (double)h.xmin + (double)h.ncx * h.cell, by1 = (double)h.ymin + (double)h.ncy * h.cell;
        const double bx0 = fmin((double)h.xmin, (double)h.bb[0]), by0 = fmin((double)h.ymin, (double)h.bb[2]);
        const double gx1 = (double)p.x0 + (double)(p.nx - 1) * p.dx, gy1 = (double)p.y0 + (double)(p.ny - 1) * p.dy;
        const double lox = fmin(bx0, fmin((double)p.x0, gx1)), hix = fmax(fmax(bx1, (double)h.bb[1]), fmax((double)p.x0, gx1));
        const double loy = fmin(by0, fmin((double)p.y0, gy1)), hiy = fmax(fmax(by1, (double)h.bb[3]), fmax((double)p.y0, gy1));
        float rmax = (float)(1.01 * ((hix - lox) + (hiy - loy)) + 1.0);
        float r0 = h.step_hint * p.r0_factor;              // the radius that holds ~1.5 k soundings at the mean density
        if (!(r0 > 0.0f) || !isfinite(r0)) r0 = rmax;
        if (r0 > rmax) r0 = rmax;
        gi.r0 = r0; gi.rmax = rmax;
        gi.bad = (h.status != BATHY_OK) || (h.n < k) || !isfinite(rmax);
    }
    __syncthreads();
    if (gi.bad) {                                          // CTA-uniform: every node of the call fails
        for (long long blk = b0; blk < b1; ++blk) {
            const int bj = (int)(blk % p.nbx), bi = (int)(blk / p.nbx);
            const int J = bj * BW + (lane & (BW - 1)), I = bi * BH + (lane / BW);
            if (J < p.nx && I < p.ny) {
                p.zhat[(long long)I * p.nx + J] = qnan;
                if (p.var) p.var[(long long)I * p.nx + J] = qnan;
                if (p.failed) atomicAdd(p.failed, 1ull);
            }
        }
        return;
    }
    float rho = gi.r0;                                     // pilot radius to try first

#pragma unroll 1
    for (int it = 0; it < p.chain; ++it) {
        const long long blk = b0 + it;
        // One CTA barrier per block, between its search and its solves: the warps of the CTA then run
        // the (long, fully unrolled) solve code side by side and share its instruction-cache lines.
        bool synced = false;
        if (blk >= b1) { __syncthreads(); continue; }
        const int bj = (int)(blk % p.nbx), bi = (int)(blk / p.nbx);
        const int J = bj * BW + (lane & (BW - 1)), I = bi * BH + (lane / BW);
        const bool valid = (J < p.nx) && (I < p.ny);
        const float xq = __fmaf_rn((float)J, p.dx, p.x0), yq = __fmaf_rn((float)I, p.dy, p.y0);
        const long long node = (long long)I * p.nx + J;

        int nsub = 1;                                      // the block is searched as nsub groups of 32/nsub lanes
#pragma unroll 1
        for (int s = 0; s < nsub;) {
            const int sz = 32 / nsub, l0 = s * sz;
            int jx0, jx1, iy0, iy1;                        // the group's nodes inside the block
            if (sz >= BW) { jx0 = 0; jx1 = BW - 1; iy0 = l0 / BW; iy1 = (l0 + sz - 1) / BW; }
            else          { iy0 = iy1 = l0 / BW; jx0 = l0 % BW; jx1 = jx0 + sz - 1; }
            const int Jlo = bj * BW + jx0, Jhi = min(bj * BW + jx1, p.nx - 1);
            const int Ilo = bi * BH + iy0, Ihi = min(bi * BH + iy1, p.ny - 1);
            if (Jlo > p.nx - 1 || Ilo > p.ny - 1) { ++s; continue; }       // no node of the grid in this group
            const bool in_group = valid && lane >= l0 && lane < l0 + sz;
            const float xlo = __fmaf_rn((float)Jlo, p.dx, p.x0), xhi = __fmaf_rn((float)Jhi, p.dx, p.x0);
            const float ylo = __fmaf_rn((float)Ilo, p.dy, p.y0), yhi = __fmaf_rn((float)Ihi, p.dy, p.y0);
            const float cx = 0.5f * (xlo + xhi), cy = 0.5f * (ylo + yhi);
            // every bound below is inflated by far more than the fp32 rounding of the expressions in it
            // (4 ulp of the largest coordinate: centre, half extents and distances are each a few roundings)
            const float slack = 5e-7f * fmaxf(fmaxf(fabsf(xlo), fabsf(xhi)), fmaxf(fabsf(ylo), fabsf(yhi))) + 1e-30f;
            const float ex = 0.5f * (xhi - xlo) + slack, ey = 0.5f * (yhi - ylo) + slack;
            const float dmax = sqrtf(ex * ex + ey * ey) * 1.00001f;

            __syncwarp();
            const float T = pilot<K, G>(p, gi, ws, lane, cx, cy, rho);
            bool group_ok = T >= 0.0f;
            int n_c = 0;
            float sT = 0.0f;
            if (group_ok) {
                sT = sqrtf(T) * 1.00001f;
                rho = sT * 1.1f + slack;
                const float Rb = (sT + dmax) * 1.0001f + slack;
                const float Rb2 = Rb * Rb;
                n_c = scan_cells(p, gi, lane, cx - ex - Rb, cx + ex + Rb, cy - ey - Rb, cy + ey + Rb, S::CAP,
                                 [&](const float4& pt) {
                                     const float ax = fmaxf(fabsf(pt.x - cx) - ex, 0.0f), ay = fmaxf(fabsf(pt.y - cy) - ey, 0.0f);
                                     return fmaf(ax, ax, ay * ay) <= Rb2;
                                 },
                                 [&](int slot, const float4& pt) {
                                     ws.cx[slot] = pt.x;
                                     ws.cy[slot] = pt.y;
                                     ws.cz[slot] = pt.z;
                                     ws.cid[slot] = __float_as_int(pt.w);
                                 });
                __syncwarp();
                if (n_c > S::CAP) {
                    if (sz > 1) { nsub *= 2; s *= 2; continue; }           // split the group and search again
                    group_ok = false;                                      // a single node: degenerate input
                } else if ((n_c & 1) && lane == 0) {
                    ws.cx[n_c] = INFINITY;                                 // pad to a whole pair: key = +inf
                    ws.cy[n_c] = INFINITY;
                }
                __syncwarp();
            } else {
                rho = gi.r0;
            }
            bool lane_ok = false;
            if (group_ok) {
                float hi = -1.0f;
                if (in_group) {
                    const float ddx = xq - cx, ddy = yq - cy;
                    const float h = sT + (sqrtf(fmaf(ddx, ddx, ddy * ddy)) * 1.00001f + slack);
                    hi = h * h * 1.00001f;
                }
                lane_ok = select_per_lane<K, G>(p, ws, lane, n_c, xq, yq, hi) && in_group;
            }
            if (in_group && !lane_ok) {                    // degenerate input: the node fails
                p.zhat[node] = qnan;
                if (p.var) p.var[node] = qnan;
                if (p.failed) atomicAdd(p.failed, 1ull);
            }
            __syncwarp();
            if (p.nbr && lane_ok) write_sorted_nbr<K, G>(p, ws, lane, xq, yq, node);

            // K3-K5, NB nodes at a time
            if (!synced) { __syncthreads(); synced = true; }
            const unsigned solvable = __ballot_sync(kFull, lane_ok);
            const float padbase = 2.0f * (ex + ey + (sT + dmax) * 1.0001f + slack) * p.s_pad + 300.0f;
#pragma unroll 1
            for (int bb = l0 / S::NB; bb * S::NB < l0 + sz; ++bb) {
                if (((solvable >> (bb * S::NB)) & ((S::NB == 32) ? 0xffffffffu : ((1u << S::NB) - 1u))) == 0u) continue;
                for (int e = lane; e < S::NB * K; e += 32) {
                    const int nd = e / K, m = e % K, sl = bb * S::NB + nd;
                    const bool node_live = (solvable >> sl) & 1u;
                    float2 xy = make_float2(padbase + 300.0f * (float)m, 0.0f);
                    float z = 0.0f;
                    if (node_live) {
                        const int c = ws.nbl[m < k ? m : 0][sl];
                        z = ws.cz[c];
                        if (m < k) {
                            const float2 o = make_float2(ws.cx[c], ws.cy[c]);
                            xy = map_coord<EX>(p, o.x - cx, o.y - cy);
                        }
                    }
                    ws.nb_x[nd][m] = xy.x;
                    ws.nb_y[nd][m] = xy.y;
                    ws.nb_z[nd][m] = z;
                }
                __syncwarp();
                const int src = bb * S::NB + (S::ILV ? lane % S::NB : lane / G);   // the lane whose node this lane helps to solve
                const int Js = bj * BW + (src & (BW - 1)), Is = bi * BH + (src / BW);
                // map_coord rounds every product and sum on its own (no contraction into the subtractions of the
                // solve), so that a node on a datum sees h2 == 0 exactly (same expression as the neighbour's coordinates)
                const float2 qs = map_coord<EX>(p, __fmaf_rn((float)Js, p.dx, p.x0) - cx, __fmaf_rn((float)Is, p.dy, p.y0) - cy);
                solve_batch<K, G, MODEL, EX>(p, ws, lane, qs.x, qs.y, (solvable >> src) & 1u, (long long)Is * p.nx + Js, k);
                __syncwarp();
            }
            ++s;
        }
        if (!synced) __syncthreads();
    }
}

template <int K, int G, int MODEL, bool EX>
int launch_one(const PredictParams& p, unsigned ctas, size_t smem, cudaStream_t stream)
{
    static DeviceOnce once;
    const int rc = once_per_device(once, [smem]() -> int {
        BATHY_CUDA_TRY(cudaFuncSetAttribute(krige_predict_kernel<K, G, MODEL, EX>,
                                            cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        return (int)BATHY_OK;
    });
    if (rc) return rc;
    krige_predict_kernel<K, G, MODEL, EX><<<ctas, Shape<K, G>::WARPS * 32, smem, stream>>>(p);
    count_launch();
    return launch_status();
}

template <int K, int G>
int launch_shape(const PredictParams& p, int model, cudaStream_t stream)
{
    const long long warps = (p.n_blocks + p.chain - 1) / p.chain;
    constexpr int kWarpsPerCta = Shape<K, G>::WARPS;
    const long long ctas = (warps + kWarpsPerCta - 1) / kWarpsPerCta;
    if (ctas > 0x7fffffffLL) return BATHY_ERR_SIZE;
    const size_t smem = sizeof(WarpSmem<K, G>) * kWarpsPerCta;
    const bool ex = p.var != nullptr || p.illcond != nullptr || p.aniso != 0;
    const unsigned n = (unsigned)ctas;
    switch (model * 2 + (ex ? 1 : 0)) {
        case BATHY_VGM_EXPONENTIAL * 2:     return launch_one<K, G, BATHY_VGM_EXPONENTIAL, false>(p, n, smem, stream);
        case BATHY_VGM_EXPONENTIAL * 2 + 1: return launch_one<K, G, BATHY_VGM_EXPONENTIAL, true>(p, n, smem, stream);
        case BATHY_VGM_SPHERICAL * 2:       return launch_one<K, G, BATHY_VGM_SPHERICAL, false>(p, n, smem, stream);
        case BATHY_VGM_SPHERICAL * 2 + 1:   return launch_one<K, G, BATHY_VGM_SPHERICAL, true>(p, n, smem, stream);
        case BATHY_VGM_GAUSSIAN * 2:        return launch_one<K, G, BATHY_VGM_GAUSSIAN, false>(p, n, smem, stream);
        default:                            return launch_one<K, G, BATHY_VGM_GAUSSIAN, true>(p, n, smem, stream);
    }
}

}  // namespace

int launch_predict(const krige_index* idx, const grid_geom_t& out, const variogram_t& vg, int k,
                   float* d_zhat, float* d_var, int32_t* d_nbr, int64_t* d_failed, int64_t* d_illcond, cudaStream_t stream,
                   const krige_aniso_t* aniso)
{
    if (!index_on_current_device(idx)) return BATHY_ERR_INDEX;
    if (stream != idx->stream) __atomic_store_n(&const_cast<krige_index*>(idx)->used_elsewhere, 1, __ATOMIC_RELEASE);
    PredictParams p;
    p.pts = idx->d_pts;
    p.cell_start = idx->d_cell_start;
    p.hdr = idx->d_hdr;
    p.nx = out.nx; p.ny = out.ny; p.x0 = out.x0; p.y0 = out.y0; p.dx = out.dx; p.dy = out.dy;
    p.k = k;
    set_variogram(p, vg);
    p.m00 = p.m11 = p.s_pad = p.s_coord;
    p.m01 = p.m10 = 0.0f;
    p.aniso = aniso ? 1 : 0;
    if (aniso) {
        const double t = (double)aniso->angle_deg * (3.141592653589793 / 180.0), sc = (double)p.s_coord, r = (double)aniso->ratio;
        p.m00 = (float)(sc * cos(t));      p.m01 = (float)(sc * sin(t));
        p.m10 = (float)(-sc * sin(t) / r); p.m11 = (float)(sc * cos(t) / r);
        p.s_pad = (float)(sc / r);
    }
    p.r0_factor = (float)sqrt(1.5 * (double)k / 3.141592653589793);
    p.zhat = d_zhat;
    p.var = d_var;
    p.nbr = d_nbr;
    p.failed = reinterpret_cast<unsigned long long*>(d_failed);
    p.illcond = reinterpret_cast<unsigned long long*>(d_illcond);
    p.nbx = (out.nx + BW - 1) / BW;
    p.nby = (out.ny + BH - 1) / BH;
    p.n_blocks = (long long)p.nbx * p.nby;
    {
        // one block per warp: the hardware CTA scheduler balances the uneven sounding density best
        // (measured: 5.91 ms with 1 block per warp, 5.99 ms with 8, 6.80 ms with 16 on config 4);
        // longer chains only where the grid would exceed the CTA-count limit
        const long long per = p.n_blocks / (0x7fffffffLL / 2) + 1;
        p.chain = (int)per;
    }
    if (k <= 8)  return launch_shape<8, 8>(p, vg.model, stream);
    if (k <= 16) return launch_shape<16, 8>(p, vg.model, stream);
    if (k <= 32) return launch_shape<32, 8>(p, vg.model, stream);
    return launch_shape<64, 16>(p, vg.model, stream);
}

}  // namespace bathy
