// krige_predict.cu -- ordinary kriging at every node of the output grid (
// SURVEY.md 8(a) rows K2-K5).
//
// One warp walks a strip of consecutive nodes of one output row.
//   K2  search: the warp collects, from the uniform cell grid, every sounding whose fp32 key
//       (squared distance, the defined expression of reading K2) is <= an upper bound of the k-th
//       key, then finds the exact k-th (key, index) by bisection on the key bits (ties: bisection
//       on the index) with warp vote/reduce counts.  The bound for the next node of the strip is
//       (r_k + node spacing)^2 by the triangle inequality, so only a thin annulus is ever in doubt.
//   K3-K5 solve: G lanes per node (32/G nodes per warp at once), rows of C dealt cyclically to the
//       lanes and held in REGISTERS (fully unrolled right-looking Cholesky); column j of L is
//       published through a small shared-memory buffer and read back as broadcast float4.  The
//       three right-hand sides c0, 1 and z ride along as forward substitutions, and
//           z_hat = y_z.y_c - mu * (y_z.y_1),   mu = (y_1.y_c - 1) / (y_1.y_1),   y_b = L^-1 b
//       gives the Lagrange/Schur step without any back substitution or explicit weights.
//   Tensor cores are not used: the factorisation is a k x k problem with a serial pivot chain.
#include "krige_index.cuh"

namespace bathy {

namespace {

constexpr int kWarpsPerCta = 4;
constexpr unsigned kFull = 0xffffffffu;

struct PredictParams {
    const float4* pts;
    const int32_t* cell_start;
    float xmin, ymin, inv_cell, cell;
    int ncx, ncy;
    int nx, ny;
    float x0, y0, dx, dy;
    int k;
    float cpn;          // (sill - nugget) / sill : partial sill of the covariance normalised to sill = 1
    float inv_range;    // 1 / a
    float exp_scale;    // -log2(e) / a
    float r0;           // first search radius of a strip
    float rmax;         // radius that certainly covers every sounding from any node of this call
    float* zhat;
    int32_t* nbr;
    unsigned long long* failed;
    int strip_len, strips_per_row;
    long long n_strips;
};

template <int K, int G>
struct Shape {
    static constexpr int R = K / G;             // rows of C per lane
    static constexpr int NB = 32 / G;           // nodes solved by a warp at once
    static constexpr int CMAX = (4 * K > 128) ? 4 * K : 128;   // candidate buffer
    static constexpr int NQ = CMAX / 32;
    static constexpr int XYS = K + 4;           // float2 stride of a node's coordinate list (bank skew)
    static constexpr int CBS = K + 4;           // float stride of a node's column buffer (bank skew)
};

template <int K, int G>
struct __align__(16) WarpSmem {
    using S = Shape<K, G>;
    float4   rhs[S::NB];                        // y_c, y_1, y_z of the current column, per node
    float    colbuf[S::NB][S::CBS];             // column j of L, per node
    float2   nb_xy[S::NB][S::XYS];              // neighbour coordinates
    float    nb_z[S::NB][K];                    // neighbour depths
    int32_t  nb_idx[S::NB][K];                  // neighbour original indices
    uint32_t cand_key[S::CMAX];
    int32_t  cand_idx[S::CMAX];
    int32_t  cand_pos[S::CMAX];
};

// Reading K2: key = fmaf(ddx, ddx, ddy*ddy) in fp32, ddx = xq - x_i, ddy = yq - y_i.
__device__ __forceinline__ float knn_key(float xq, float yq, float x, float y)
{
    const float ddx = __fsub_rn(xq, x), ddy = __fsub_rn(yq, y);
    return __fmaf_rn(ddx, ddx, __fmul_rn(ddy, ddy));
}

// Covariance normalised to sill = 1: C(h) = 1 - gamma(h)/sill.  gamma(0) = 0 -> C(0) = 1.
template <int MODEL>
__device__ __forceinline__ float cov_of_h2(float h2, const PredictParams& p)
{
    const float h = h2 * rsqrtf(h2);                       // NaN at h2 == 0, replaced below
    float c;
    if (MODEL == BATHY_VGM_EXPONENTIAL) {
        c = p.cpn * exp2f(h * p.exp_scale);                // exp(-h/a), no factor 3
    } else {
        const float q = h * p.inv_range;
        c = (q < 1.0f) ? p.cpn * fmaf(q, fmaf(0.5f * q, q, -1.5f), 1.0f) : 0.0f;
    }
    return (h2 > 0.0f) ? c : 1.0f;
}

// ---------------------------------------------------------------------------------------------
// K2: collect every sounding with key bits <= key_hi inside the square of half-width r around the
// node into the warp's candidate buffer, in index (cell-scan) order.  Returns the number found
// (it may exceed CMAX, in which case the buffer is incomplete).
template <int K, int G>
__device__ __forceinline__ int collect(const PredictParams& p, WarpSmem<K, G>& ws, int lane,
                                       float xq, float yq, float r, uint32_t key_hi)
{
    using S = Shape<K, G>;
    const float rs = r + 2e-3f * p.cell;                   // cell_of() rounding slack
    const int cx0 = cell_of(xq - rs, p.xmin, p.inv_cell, p.ncx), cx1 = cell_of(xq + rs, p.xmin, p.inv_cell, p.ncx);
    const int cy0 = cell_of(yq - rs, p.ymin, p.inv_cell, p.ncy), cy1 = cell_of(yq + rs, p.ymin, p.inv_cell, p.ncy);
    int n_c = 0;
    for (int cyb = cy0; cyb <= cy1; cyb += 32) {
        const int cy = cyb + lane;
        int seg_s = 0, seg_e = 0;
        if (cy <= cy1) {
            seg_s = __ldg(p.cell_start + (size_t)cy * p.ncx + cx0);
            seg_e = __ldg(p.cell_start + (size_t)cy * p.ncx + cx1 + 1);
        }
        const int rows = min(32, cy1 - cyb + 1);
        for (int rr = 0; rr < rows; ++rr) {
            const int s = __shfl_sync(kFull, seg_s, rr), e = __shfl_sync(kFull, seg_e, rr);
            for (int base = s; base < e; base += 32) {
                const int pos = base + lane;
                bool keep = false;
                uint32_t kb = 0;
                int32_t id = 0;
                if (pos < e) {
                    const float4 pt = __ldg(p.pts + pos);
                    kb = __float_as_uint(knn_key(xq, yq, pt.x, pt.y));
                    id = __float_as_int(pt.w);
                    keep = kb <= key_hi;
                }
                const unsigned m = __ballot_sync(kFull, keep);
                const int off = n_c + __popc(m & ((1u << lane) - 1u));
                if (keep && off < S::CMAX) {
                    ws.cand_key[off] = kb;
                    ws.cand_idx[off] = id;
                    ws.cand_pos[off] = pos;
                }
                n_c += __popc(m);
            }
        }
    }
    return n_c;
}

// K2: exact selection of the k smallest (key, index) among the n_c buffered candidates and
// transfer of their (x, y, z, index) into neighbour slot `slot`.  Returns the k-th key bits
// through *kth_key.  lo_hint: a value believed to satisfy count(key < lo_hint) < k (0 = none).
template <int K, int G>
__device__ __forceinline__ void select_k(const PredictParams& p, WarpSmem<K, G>& ws, int lane, int slot,
                                         int n_c, uint32_t lo_hint, uint32_t key_hi, uint32_t* kth_key)
{
    using S = Shape<K, G>;
    const int k = p.k;
    uint32_t ck[S::NQ];
#pragma unroll
    for (int q = 0; q < S::NQ; ++q) {
        const int c = lane + 32 * q;
        ck[q] = (c < n_c) ? ws.cand_key[c] : 0xffffffffu;
    }
    auto count_le = [&](uint32_t v) {
        int c = 0;
#pragma unroll
        for (int q = 0; q < S::NQ; ++q) c += (ck[q] <= v) ? 1 : 0;
        return (int)__reduce_add_sync(kFull, (unsigned)c);
    };
    uint32_t lo = lo_hint, hi = key_hi, tau = 0;
    if (lo > 0 && count_le(lo - 1) >= k) lo = 0;           // the hint was not a lower bound
    int cnt;
    // invariant: count(key <= hi) >= k, count(key <= lo-1) < k
    while (true) {
        const uint32_t mid = lo + ((hi - lo) >> 1);
        cnt = count_le(mid);
        if (cnt == k) { tau = mid; break; }
        if (cnt > k) hi = mid; else lo = mid + 1;
        if (lo == hi) { tau = lo; cnt = count_le(tau); break; }
    }
    int32_t idx_max = 0x7fffffff;                          // ties on the k-th key: lowest indices win
    if (cnt != k) {
        int32_t ci[S::NQ];
        int below = 0;
#pragma unroll
        for (int q = 0; q < S::NQ; ++q) {
            const int c = lane + 32 * q;
            ci[q] = (c < n_c && ck[q] == tau) ? ws.cand_idx[c] : 0x7fffffff;   // 0x7fffffff is never a valid index (n <= 2^31-1)
            below += (ck[q] < tau) ? 1 : 0;
        }
        const int want = k - (int)__reduce_add_sync(kFull, (unsigned)below);
        int32_t ilo = 0, ihi = 0x7ffffffe;
        while (true) {
            const int32_t mid = ilo + ((ihi - ilo) >> 1);
            int c = 0;
#pragma unroll
            for (int q = 0; q < S::NQ; ++q) c += (ci[q] <= mid) ? 1 : 0;
            c = (int)__reduce_add_sync(kFull, (unsigned)c);
            if (c == want) { idx_max = mid; break; }
            if (c > want) ihi = mid; else ilo = mid + 1;
            if (ilo == ihi) { idx_max = ilo; break; }
        }
    }
    // transfer, preserving index (scan) order
    int n_sel = 0;
    uint32_t kmax = 0;
#pragma unroll
    for (int q = 0; q < S::NQ; ++q) {
        if (32 * q < n_c) {                                // warp-uniform
            const int c = lane + 32 * q;
            bool sel = false;
            int32_t id = 0;
            if (c < n_c) {
                id = ws.cand_idx[c];
                sel = (ck[q] < tau) || (ck[q] == tau && id <= idx_max);
            }
            const unsigned m = __ballot_sync(kFull, sel);
            const int off = n_sel + __popc(m & ((1u << lane) - 1u));
            if (sel) {
                const float4 pt = __ldg(p.pts + ws.cand_pos[c]);
                ws.nb_xy[slot][off] = make_float2(pt.x, pt.y);
                ws.nb_z[slot][off] = pt.z;
                ws.nb_idx[slot][off] = id;
                kmax = max(kmax, ck[q]);
            }
            n_sel += __popc(m);
        }
    }
    *kth_key = __reduce_max_sync(kFull, kmax);
}

// Parity/debug output: neighbours in ascending (key, index) order.
template <int K, int G>
__device__ __forceinline__ void write_sorted_nbr(const PredictParams& p, WarpSmem<K, G>& ws, int lane, int slot,
                                                 float xq, float yq, long long node)
{
    const int k = p.k;
    for (int e = lane; e < k; e += 32) {
        const float2 me = ws.nb_xy[slot][e];
        const uint32_t mk = __float_as_uint(knn_key(xq, yq, me.x, me.y));
        const int32_t mi = ws.nb_idx[slot][e];
        int rank = 0;
        for (int f = 0; f < k; ++f) {
            const float2 o = ws.nb_xy[slot][f];
            const uint32_t ok = __float_as_uint(knn_key(xq, yq, o.x, o.y));
            const int32_t oi = ws.nb_idx[slot][f];
            rank += (ok < mk || (ok == mk && oi < mi)) ? 1 : 0;
        }
        p.nbr[node * k + rank] = mi;
    }
}

// ---------------------------------------------------------------------------------------------
// K3-K5 for the NB nodes whose neighbour lists sit in the warp's shared memory.
template <int K, int G, int MODEL>
__device__ __forceinline__ void solve_nodes(const PredictParams& p, WarpSmem<K, G>& ws, int lane,
                                            float xq, float yq, bool node_valid, long long node)
{
    using S = Shape<K, G>;
    constexpr int R = S::R;
    const int nd = lane / G, g = lane % G;
    const int k = p.k;
    const float zref = ws.nb_z[nd][0];

    float A[R][K];                   // A[t][m]: row g + G t, column m <= row (registers; only m < (t+1)G live)
    float yc[R], y1[R], yz[R];
    float xr[R], yr[R];
#pragma unroll
    for (int t = 0; t < R; ++t) {
        const int r = g + G * t;
        const float2 c = ws.nb_xy[nd][r];
        xr[t] = c.x; yr[t] = c.y;
        const bool live = r < k;
        const float ddx = xq - c.x, ddy = yq - c.y;
        yc[t] = live ? cov_of_h2<MODEL>(fmaf(ddx, ddx, ddy * ddy), p) : 0.0f;
        y1[t] = live ? 1.0f : 0.0f;
        yz[t] = live ? ws.nb_z[nd][r] - zref : 0.0f;
    }
    // K3: lower triangle of C (rows beyond k are identity rows: they decouple and carry zero rhs)
#pragma unroll
    for (int m = 0; m < K; ++m) {
        const float2 cm = ws.nb_xy[nd][m];
#pragma unroll
        for (int t = m / G; t < R; ++t) {
            const int r = g + G * t;
            const float ddx = xr[t] - cm.x, ddy = yr[t] - cm.y;
            float c = cov_of_h2<MODEL>(fmaf(ddx, ddx, ddy * ddy), p);
            if (r == m) c = 1.0f;
            if (r >= k || m >= k) c = (r == m) ? 1.0f : 0.0f;
            A[t][m] = c;
        }
    }
    __syncwarp();

    // K4: right-looking Cholesky, column by column; rhs vectors forward-substituted on the way
    bool ok = true;
#pragma unroll
    for (int j = 0; j < K; ++j) {
        constexpr int dummy = 0; (void)dummy;
        const int tj = j / G, gj = j % G;
        const float piv = __shfl_sync(kFull, A[tj][j], gj, G);
        ok = ok && (piv > 1e-6f);
        const float inv = rsqrtf(piv);
        float Lr[R];
#pragma unroll
        for (int t = tj; t < R; ++t) {
            const int r = g + G * t;
            Lr[t] = (r > j) ? A[t][j] * inv : 0.0f;
            ws.colbuf[nd][r] = Lr[t];
        }
        if (g == gj) ws.rhs[nd] = make_float4(yc[tj] * inv, y1[tj] * inv, yz[tj] * inv, 0.0f);
        __syncwarp();
        const float4 yj = ws.rhs[nd];
#pragma unroll
        for (int t = tj; t < R; ++t) {
            if (t == tj && g == gj) { yc[t] = yj.x; y1[t] = yj.y; yz[t] = yj.z; }
            yc[t] = fmaf(-Lr[t], yj.x, yc[t]);
            y1[t] = fmaf(-Lr[t], yj.y, y1[t]);
            yz[t] = fmaf(-Lr[t], yj.z, yz[t]);
        }
#pragma unroll
        for (int m4 = (j + 1) / 4; m4 < K / 4; ++m4) {
            const float4 L4 = *reinterpret_cast<const float4*>(&ws.colbuf[nd][4 * m4]);
            const float Lm[4] = {L4.x, L4.y, L4.z, L4.w};
#pragma unroll
            for (int e = 0; e < 4; ++e) {
                const int m = 4 * m4 + e;
                if (m > j) {
#pragma unroll
                    for (int t = (m / G > tj ? m / G : tj); t < R; ++t) A[t][m] = fmaf(-Lr[t], Lm[e], A[t][m]);
                }
            }
        }
        __syncwarp();
    }

    // K5 with the Schur step: four dot products over the G lanes of the node
    float dcz = 0.0f, d1c = 0.0f, d11 = 0.0f, d1z = 0.0f;
#pragma unroll
    for (int t = 0; t < R; ++t) {
        dcz = fmaf(yc[t], yz[t], dcz);
        d1c = fmaf(y1[t], yc[t], d1c);
        d11 = fmaf(y1[t], y1[t], d11);
        d1z = fmaf(y1[t], yz[t], d1z);
    }
#pragma unroll
    for (int o = G / 2; o > 0; o >>= 1) {
        dcz += __shfl_xor_sync(kFull, dcz, o);
        d1c += __shfl_xor_sync(kFull, d1c, o);
        d11 += __shfl_xor_sync(kFull, d11, o);
        d1z += __shfl_xor_sync(kFull, d1z, o);
    }
    if (g == 0 && node_valid) {
        const float mu = (d1c - 1.0f) / d11;
        float est = zref + (dcz - mu * d1z);
        if (!ok) {
            est = __int_as_float(0x7fc00000);
            if (p.failed) atomicAdd(p.failed, 1ull);
        }
        p.zhat[node] = est;
    }
}

template <int K, int G, int MODEL>
__global__ void __launch_bounds__(kWarpsPerCta * 32)
krige_predict_kernel(const PredictParams p)
{
    using S = Shape<K, G>;
    __shared__ WarpSmem<K, G> s_ws[kWarpsPerCta];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    WarpSmem<K, G>& ws = s_ws[warp];
    const long long sid = (long long)blockIdx.x * kWarpsPerCta + warp;
    if (sid >= p.n_strips) return;
    const int I = (int)(sid / p.strips_per_row);
    const int Jbeg = (int)(sid % p.strips_per_row) * p.strip_len;
    const int Jend = min(Jbeg + p.strip_len, p.nx);
    const float yq = __fmaf_rn((float)I, p.dy, p.y0);
    const int k = p.k;

    float r = p.r0;                    // search radius to try
    uint32_t lo_hint = 0;
    float xprev = 0.0f;
    bool have_prev = false;
    float rk_prev = 0.0f;

    for (int Jb = Jbeg; Jb < Jend; Jb += S::NB) {
        float my_xq = 0.0f;            // node of this lane's group
        bool my_valid = false;
#pragma unroll 1
        for (int s = 0; s < S::NB; ++s) {
            const int J = Jb + s;
            if (J >= Jend) break;                                   // warp-uniform
            const float xq = __fmaf_rn((float)J, p.dx, p.x0);
            if (lane / G == s) { my_xq = xq; my_valid = true; }
            if (have_prev) {
                const float step = fabsf(xq - xprev);
                const float rhi = (rk_prev + step) * 1.00001f + 1e-30f;
                const float rlo = fmaxf(rk_prev - step, 0.0f) * 0.99999f;
                r = rhi;
                lo_hint = __float_as_uint(rlo * rlo * 0.99999f);
            }
            float r_low = 0.0f, r_high = INFINITY;
            int n_c = 0;
            uint32_t key_hi = 0;
            bool found = false;
            for (int it = 0; it < 96; ++it) {
                const float kh = r * r * 1.00001f;
                key_hi = __float_as_uint(fminf(kh, 3.0e38f));
                n_c = collect<K, G>(p, ws, lane, xq, yq, r, key_hi);
                if (n_c < k) {
                    if (r >= p.rmax) break;                         // cannot happen for k <= n
                    r_low = r;
                    r = isinf(r_high) ? fminf(r * 1.5f, p.rmax) : 0.5f * (r_low + r_high);
                    lo_hint = 0;
                } else if (n_c > S::CMAX) {
                    r_high = r;
                    r = 0.5f * (r_low + r_high);
                } else { found = true; break; }
            }
            __syncwarp();
            uint32_t kth = 0;
            if (found) {
                select_k<K, G>(p, ws, lane, s, n_c, lo_hint, key_hi, &kth);
            } else {
                // degenerate input (more than CMAX-k soundings at one distance): mark the node failed
                for (int e = lane; e < K; e += 32) { ws.nb_xy[s][e] = make_float2(xq, yq); ws.nb_z[s][e] = 0.0f; ws.nb_idx[s][e] = -1; }
            }
            // pad the coordinate list so that the solve can read K entries
            for (int e = k + lane; e < K; e += 32) { ws.nb_xy[s][e] = make_float2(0.0f, 0.0f); ws.nb_z[s][e] = 0.0f; ws.nb_idx[s][e] = -1; }
            __syncwarp();
            if (p.nbr && found) write_sorted_nbr<K, G>(p, ws, lane, s, xq, yq, (long long)I * p.nx + J);
            rk_prev = sqrtf(__uint_as_float(kth));
            have_prev = found;
            xprev = xq;
            if (!found) { r = p.r0; lo_hint = 0; }
        }
        __syncwarp();
        const int Jmine = Jb + lane / G;
        solve_nodes<K, G, MODEL>(p, ws, lane, my_xq, yq, my_valid && Jmine < Jend, (long long)I * p.nx + Jmine);
        __syncwarp();
    }
}

template <int K, int G>
int launch_shape(const PredictParams& p, int model, cudaStream_t stream)
{
    const long long ctas = (p.n_strips + kWarpsPerCta - 1) / kWarpsPerCta;
    if (ctas > 0x7fffffffLL) return BATHY_ERR_SIZE;
    if (model == BATHY_VGM_EXPONENTIAL)
        krige_predict_kernel<K, G, BATHY_VGM_EXPONENTIAL><<<(unsigned)ctas, kWarpsPerCta * 32, 0, stream>>>(p);
    else
        krige_predict_kernel<K, G, BATHY_VGM_SPHERICAL><<<(unsigned)ctas, kWarpsPerCta * 32, 0, stream>>>(p);
    count_launch();
    return launch_status();
}

}  // namespace

int launch_predict(const krige_index* idx, const grid_geom_t& out, const variogram_t& vg, int k,
                   float* d_zhat, int32_t* d_nbr, int64_t* d_failed, cudaStream_t stream)
{
    PredictParams p;
    p.pts = idx->d_pts;
    p.cell_start = idx->d_cell_start;
    p.xmin = idx->xmin; p.ymin = idx->ymin; p.inv_cell = idx->inv_cell; p.cell = idx->cell;
    p.ncx = idx->ncx; p.ncy = idx->ncy;
    p.nx = out.nx; p.ny = out.ny; p.x0 = out.x0; p.y0 = out.y0; p.dx = out.dx; p.dy = out.dy;
    p.k = k;
    p.cpn = (float)(((double)vg.sill - (double)vg.nugget) / (double)vg.sill);
    p.inv_range = (float)(1.0 / (double)vg.range);
    p.exp_scale = (float)(-1.4426950408889634 / (double)vg.range);
    // first radius of a strip: the radius that holds ~1.5 k soundings at the mean density
    p.r0 = (float)((double)idx->step_hint * sqrt(1.5 * (double)k / 3.141592653589793));
    {
        // farthest any node of this call can be from any sounding: covers the union of both extents
        const double bx1 = (double)idx->xmin + (double)idx->ncx * idx->cell, by1 = (double)idx->ymin + (double)idx->ncy * idx->cell;
        const double gx1 = (double)out.x0 + (double)(out.nx - 1) * out.dx, gy1 = (double)out.y0 + (double)(out.ny - 1) * out.dy;
        const double lox = fmin((double)idx->xmin, fmin((double)out.x0, gx1)), hix = fmax(bx1, fmax((double)out.x0, gx1));
        const double loy = fmin((double)idx->ymin, fmin((double)out.y0, gy1)), hiy = fmax(by1, fmax((double)out.y0, gy1));
        p.rmax = (float)(1.01 * ((hix - lox) + (hiy - loy)) + 1.0);
        if (!(p.r0 > 0.0f) || !isfinite(p.r0)) p.r0 = p.rmax;
        if (p.r0 > p.rmax) p.r0 = p.rmax;
    }
    p.zhat = d_zhat;
    p.nbr = d_nbr;
    p.failed = reinterpret_cast<unsigned long long*>(d_failed);
    p.strip_len = 32;
    p.strips_per_row = (out.nx + p.strip_len - 1) / p.strip_len;
    p.n_strips = (long long)p.strips_per_row * out.ny;
    if (k <= 8)  return launch_shape<8, 8>(p, vg.model, stream);
    if (k <= 16) return launch_shape<16, 8>(p, vg.model, stream);
    if (k <= 32) return launch_shape<32, 8>(p, vg.model, stream);
    return launch_shape<64, 32>(p, vg.model, stream);
}

}  // namespace bathy
