/* oracle/oracle.c -- TEST INFRASTRUCTURE, NOT PRODUCT.
 *
 * Plain, slow, float64 CPU statement of what the hot path computes, written from the paper
 * (/root/reference/PAPER.md, cited as PAPER.md:Lnn) and the readings in DESIGN.md "Readings of
 * the paper".  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
 * legs may build, load or call this file.  It shares NO code, header, table or constant with
 * paper_2505_22675_b200/csrc (the CUDA path): every struct is re-declared here.
 *
 * Every function is the definition (or the paper's algorithm) written out, one step per line,
 * no blocking, no fusion, no reordering.  OpenMP appears only on the outermost per-node loop.
 * Build:  gcc -O2 -ffp-contract=off -fno-fast-math -fopenmp -shared -fPIC oracle.c -o liboracle.so -lm
 *
 * Pins (tests/test_oracle_*.py, -m "not gpu"): planes, 2.375, knots, S(0.5)=0.6875, S(1.5)=2.2,
 * 0.47265625, M=(0,18/7,-30/7,18/7,0), scipy CubicSpline(natural), two-point closed form
 * lambda1=0.748755187238, equilateral 1/3, constants, sum(lambda)=1, exactness at data, brute-force
 * kNN vs bucket kNN, LU vs numpy.linalg.solve; Catmull-Rom: C(0)=P1, C(1)=P2, C(1/2)=(-P0+9P1+9P2-P3)/16,
 * quadratics reproduced, NaN/edge fallback = bilinear; kriging variance: two-point closed form 0.148703758152,
 * zero at data, sill (1 + 1/k) for the local mean, C-form LAPACK; Gaussian variogram gamma(a); geometric anisotropy
 * (tests/test_oracle_aniso.py): lags by hand (3-4-5, the sense of the angle), two-point closed form 0.29421281, equal
 * weights at d along / ratio x d across, ratio 1 = isotropic, isotropic weights and kriging of points transformed
 * beforehand, neighbours unchanged.  No function here is "parity unpinned" against
 * mathematics; nothing is pinned against the paper's own tables (they need GEBCO).
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

/* Regular grid: node (i,j), i = row (y), j = column (x); x = x0 + j*dx, y = y0 + i*dy;
 * data row-major with leading dimension nx. */
typedef struct { int32_t nx, ny; float x0, y0, dx, dy; } ora_geom;

/* Variogram: model 0 = exponential exactly as PAPER.md:L157 (no factor 3), 1 = spherical
 * (textbook), 2 = Gaussian (textbook, same no-factor-3 convention).
 * sill is the TOTAL sill; c_p = sill - nugget.  gamma(0) = 0 exactly. */
typedef struct { int32_t model; double range, sill, nugget; } ora_vgm;

int oracle_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

void oracle_set_num_threads(int n)
{
#ifdef _OPENMP
    if (n > 0) omp_set_num_threads(n);
#else
    (void)n;
#endif
}

/* ------------------------------------------------------------------ interval location (B1, B2)
 * u = (x - in.x0)/in.dx in float64 from the fp32 geometry fields.  Out of extent -> -1 (B4).
 * i = min(max(floor(u),0), n-2), t = u - i; so the last node (u = n-1) gives i = n-2, t = 1. */
static int locate(double u, int n, double *t)
{
    if (!(u >= 0.0) || !(u <= (double)(n - 1))) return -1;
    int i = (int)floor(u);
    if (i > n - 2) i = n - 2;
    if (i < 0) i = 0;
    *t = u - (double)i;
    return i;
}

static double node_u(const ora_geom *in, const ora_geom *out, int J)
{
    double x = (double)out->x0 + (double)J * (double)out->dx;
    return (x - (double)in->x0) / (double)in->dx;
}

static double node_v(const ora_geom *in, const ora_geom *out, int I)
{
    double y = (double)out->y0 + (double)I * (double)out->dy;
    return (y - (double)in->y0) / (double)in->dy;
}

/* ------------------------------------------------------------------ bilinear
 * f = [(x2-x)(y2-y)Q11 + (x-x1)(y2-y)Q21 + (x2-x)(y-y1)Q12 + (x-x1)(y-y1)Q22]/((x2-x1)(y2-y1))
 * (eq. at) with t = (x-x1)/(x2-x1), s = (y-y1)/(y2-y1).
 * All four corners are always read and multiplied: a NaN corner gives NaN even with weight 0. */
int oracle_bilinear(const float *in, const ora_geom *gi, const ora_geom *go, double *out)
{
    if (!in || !out || gi->nx < 2 || gi->ny < 2 || go->nx < 1 || go->ny < 1) return -1;
    if (!(gi->dx > 0.0f) || !(gi->dy > 0.0f)) return -1;
    #pragma omp parallel for schedule(static)
    for (int I = 0; I < go->ny; ++I) {
        double s;
        int j = locate(node_v(gi, go, I), gi->ny, &s);
        for (int J = 0; J < go->nx; ++J) {
            double t;
            int i = locate(node_u(gi, go, J), gi->nx, &t);
            double f = NAN;
            if (i >= 0 && j >= 0) {
                double Q11 = in[(size_t)j * gi->nx + i];
                double Q21 = in[(size_t)j * gi->nx + i + 1];
                double Q12 = in[(size_t)(j + 1) * gi->nx + i];
                double Q22 = in[(size_t)(j + 1) * gi->nx + i + 1];
                f = (1.0 - t) * (1.0 - s) * Q11 + t * (1.0 - s) * Q21
                  + (1.0 - t) * s * Q12 + t * s * Q22;
            }
            out[(size_t)I * go->nx + J] = f;
        }
    }
    return 0;
}

/* ------------------------------------------------------------------ Catmull-Rom cubic
 * (the paper's own "cubic spline", readings CR1-CR3).
 * C(t) = 1/2 (2 P1 + (-P0 + P2) t + (2 P0 - 5 P1 + 4 P2 - P3) t^2 + (-P0 + 3 P1 - 3 P2 + P3) t^3)
 * (eq. at), P0..P3 the samples at i-1, i, i+1, i+2, t = u - i. */
static double catmull_rom(double P0, double P1, double P2, double P3, double t)
{
    return 0.5 * (2.0 * P1 + (-P0 + P2) * t + (2.0 * P0 - 5.0 * P1 + 4.0 * P2 - P3) * t * t
                  + (-P0 + 3.0 * P1 - 3.0 * P2 + P3) * t * t * t);
}

/* "first interpolates in x on each of 4 rows, and then in y".  Interval location as
 * bilinear (B1, B2, B4).  CR2/CR3: if any of the 16 neighbours lies outside the grid or is NaN the node
 * "falls back to a bilinear calculation" (sense fixed by L171), i.e. the value of
 * oracle_bilinear at that node (NaN if one of its 4 corners is NaN: bilinear has no fallback, L182). */
int oracle_catmull_rom(const float *in, const ora_geom *gi, const ora_geom *go, double *out)
{
    if (!in || !out || gi->nx < 2 || gi->ny < 2 || go->nx < 1 || go->ny < 1) return -1;
    if (!(gi->dx > 0.0f) || !(gi->dy > 0.0f)) return -1;
    #pragma omp parallel for schedule(static)
    for (int I = 0; I < go->ny; ++I) {
        double s;
        int j = locate(node_v(gi, go, I), gi->ny, &s);
        for (int J = 0; J < go->nx; ++J) {
            double t;
            int i = locate(node_u(gi, go, J), gi->nx, &t);
            double f = NAN;
            if (i >= 0 && j >= 0) {
                int all16 = (i - 1 >= 0) && (i + 2 <= gi->nx - 1) && (j - 1 >= 0) && (j + 2 <= gi->ny - 1);
                double R[4];
                if (all16) {
                    for (int b = 0; b < 4 && all16; ++b) {
                        const float *row = in + (size_t)(j - 1 + b) * gi->nx + (i - 1);
                        for (int a = 0; a < 4; ++a) if (isnan(row[a])) all16 = 0;
                        R[b] = catmull_rom(row[0], row[1], row[2], row[3], t);
                    }
                }
                if (all16) {
                    f = catmull_rom(R[0], R[1], R[2], R[3], s);
                } else {
                    double Q11 = in[(size_t)j * gi->nx + i];
                    double Q21 = in[(size_t)j * gi->nx + i + 1];
                    double Q12 = in[(size_t)(j + 1) * gi->nx + i];
                    double Q22 = in[(size_t)(j + 1) * gi->nx + i + 1];
                    f = (1.0 - t) * (1.0 - s) * Q11 + t * (1.0 - s) * Q21
                      + (1.0 - t) * s * Q12 + t * s * Q22;
                }
            }
            out[(size_t)I * go->nx + J] = f;
        }
    }
    return 0;
}

/* ------------------------------------------------------------------ natural cubic spline, 1-D
 * DESIGN.md reading D1 (BASELINE.json north_star; the paper's own cubic, is
 * Catmull-Rom and is a different operator).  Uniform knots, spacing h.  Unknown second
 * derivatives M: M_0 = M_{n-1} = 0, interior rows  M_{i-1} + 4 M_i + M_{i+1} = 6 (z_{i-1} - 2 z_i
 * + z_{i+1}) / h^2.  Solved by the Thomas algorithm (strictly diagonally dominant: no pivoting).
 * z and M are strided so that the same routine serves rows and columns. */
int oracle_spline_second_derivs(const double *z, int n, long zs, double h, double *M, long ms)
{
    if (n < 2) return -1;
    for (int i = 0; i < n; ++i) M[(long)i * ms] = 0.0;
    if (n < 3) return 0;                      /* n = 2: M == 0, the spline is the chord */
    int m = n - 2;                            /* unknowns M_1 .. M_{n-2} */
    double *cp = (double *)malloc(sizeof(double) * (size_t)m);
    double *dp = (double *)malloc(sizeof(double) * (size_t)m);
    if (!cp || !dp) { free(cp); free(dp); return -2; }
    for (int q = 0; q < m; ++q) {
        int i = q + 1;
        double rhs = 6.0 * (z[(long)(i - 1) * zs] - 2.0 * z[(long)i * zs] + z[(long)(i + 1) * zs]) / (h * h);
        if (q == 0) {
            cp[q] = 1.0 / 4.0;
            dp[q] = rhs / 4.0;
        } else {
            double den = 4.0 - cp[q - 1];
            cp[q] = 1.0 / den;
            dp[q] = (rhs - dp[q - 1]) / den;
        }
    }
    M[(long)m * ms] = dp[m - 1];
    for (int q = m - 2; q >= 0; --q)
        M[(long)(q + 1) * ms] = dp[q] - cp[q] * M[(long)(q + 2) * ms];
    free(cp);
    free(dp);
    return 0;
}

/* S on interval i at local coordinate t in [0,1]:  A = 1-t, B = t,
 * S = A z_i + B z_{i+1} + ((A^3 - A) M_i + (B^3 - B) M_{i+1}) h^2 / 6. */
double oracle_spline_eval(const double *z, long zs, const double *M, long ms, double h, int i, double t)
{
    double A = 1.0 - t, B = t;
    return A * z[(long)i * zs] + B * z[(long)(i + 1) * zs]
         + ((A * A * A - A) * M[(long)i * ms] + (B * B * B - B) * M[(long)(i + 1) * ms]) * (h * h) / 6.0;
}

/* 1-D convenience for the pins: knots at 0,h,2h,...; evaluates at nq abscissae u (in knot units). */
int oracle_spline1d(const double *z, int n, double h, const double *u, int nq, double *out, double *M_out)
{
    double *M = (double *)malloc(sizeof(double) * (size_t)(n > 0 ? n : 1));
    if (!M) return -2;
    int rc = oracle_spline_second_derivs(z, n, 1, h, M, 1);
    if (rc) { free(M); return rc; }
    for (int q = 0; q < nq; ++q) {
        double t;
        int i = locate(u[q], n, &t);
        out[q] = (i < 0) ? NAN : oracle_spline_eval(z, 1, M, 1, h, i, t);
    }
    if (M_out) memcpy(M_out, M, sizeof(double) * (size_t)n);
    free(M);
    return 0;
}

/* 2-D: spline every input row in x, evaluate at all output x -> T[ny_in x nx_out]; then spline
 * every column of T in y and evaluate at all output y (reading S3).  Out-of-extent -> NaN.
 * Precondition: no NaN in the input (not checked). */
int oracle_spline(const float *in, const ora_geom *gi, const ora_geom *go, double *out)
{
    if (!in || !out || gi->nx < 2 || gi->ny < 2 || go->nx < 1 || go->ny < 1) return -1;
    if (!(gi->dx > 0.0f) || !(gi->dy > 0.0f)) return -1;
    const int nxi = gi->nx, nyi = gi->ny, nxo = go->nx, nyo = go->ny;
    const double hx = (double)gi->dx, hy = (double)gi->dy;
    double *T = (double *)malloc(sizeof(double) * (size_t)nyi * (size_t)nxo);
    if (!T) return -2;
    int fail = 0;
    #pragma omp parallel
    {
        double *zr = (double *)malloc(sizeof(double) * (size_t)(nxi > nyi ? nxi : nyi));
        double *Mr = (double *)malloc(sizeof(double) * (size_t)(nxi > nyi ? nxi : nyi));
        if (!zr || !Mr) {
            #pragma omp atomic write
            fail = 1;
        } else {
            #pragma omp for schedule(static)
            for (int r = 0; r < nyi; ++r) {                         /* pass 1: rows, along x */
                for (int c = 0; c < nxi; ++c) zr[c] = (double)in[(size_t)r * nxi + c];
                oracle_spline_second_derivs(zr, nxi, 1, hx, Mr, 1);
                for (int J = 0; J < nxo; ++J) {
                    double t;
                    int i = locate(node_u(gi, go, J), nxi, &t);
                    T[(size_t)r * nxo + J] = (i < 0) ? NAN : oracle_spline_eval(zr, 1, Mr, 1, hx, i, t);
                }
            }
            #pragma omp for schedule(static)
            for (int J = 0; J < nxo; ++J) {                         /* pass 2: columns, along y */
                double tdummy;
                int bad = locate(node_u(gi, go, J), nxi, &tdummy) < 0;   /* column out of x extent */
                if (!bad) {
                    for (int r = 0; r < nyi; ++r) zr[r] = T[(size_t)r * nxo + J];
                    oracle_spline_second_derivs(zr, nyi, 1, hy, Mr, 1);
                }
                for (int I = 0; I < nyo; ++I) {
                    double s;
                    int j = locate(node_v(gi, go, I), nyi, &s);
                    out[(size_t)I * nxo + J] = (bad || j < 0) ? NAN : oracle_spline_eval(zr, 1, Mr, 1, hy, j, s);
                }
            }
        }
        free(zr);
        free(Mr);
    }
    free(T);
    return fail ? -2 : 0;
}

/* ================================================================== ordinary kriging
 * PAPER.md:L146-L171 (section III-C).  Readings K1-K5 in DESIGN.md. */

/* K1: output node coordinates are the fp32 values fmaf((float)J, dx, x0), fmaf((float)I, dy, y0). */
void oracle_node_coords(const ora_geom *g, float *xq, float *yq)
{
    for (int I = 0; I < g->ny; ++I)
        for (int J = 0; J < g->nx; ++J) {
            xq[(size_t)I * g->nx + J] = fmaf((float)J, g->dx, g->x0);
            yq[(size_t)I * g->nx + J] = fmaf((float)I, g->dy, g->y0);
        }
}

/* K2: the selection key is a DEFINED fp32 expression: ddx = xq - xi, ddy = yq - yi (fp32
 * subtractions), key = fmaf(ddx, ddx, ddy*ddy) with ddy*ddy an fp32 product, round-to-nearest.
 * (Compiled with -ffp-contract=off so the product below is not fused by the compiler.) */
float oracle_knn_key(float xq, float yq, float xi, float yi)
{
    volatile float ddx = xq - xi;
    volatile float ddy = yq - yi;
    volatile float p = ddy * ddy;
    return fmaf(ddx, ddx, p);
}

/* insert (key, idx) into the ascending (key, idx) list of at most k entries */
static void knn_insert(float *bk, int32_t *bi, int *cnt, int k, float key, int32_t idx)
{
    int c = *cnt;
    if (c == k) {
        if (!(key < bk[k - 1] || (key == bk[k - 1] && idx < bi[k - 1]))) return;
        c = k - 1;
    }
    int p = c;
    while (p > 0 && (key < bk[p - 1] || (key == bk[p - 1] && idx < bi[p - 1]))) {
        bk[p] = bk[p - 1];
        bi[p] = bi[p - 1];
        --p;
    }
    bk[p] = key;
    bi[p] = idx;
    *cnt = c + 1;
}

/* Brute force: the k soundings with the smallest (key, original index), ascending.  The definition. */
int oracle_knn_brute(const float *x, const float *y, int64_t n, float xq, float yq, int k,
                     int32_t *idx_out, float *key_out)
{
    if (k < 1 || k > n || k > 4096) return -1;
    float bk[4096];
    int32_t bi[4096];
    int cnt = 0;
    for (int64_t i = 0; i < n; ++i)
        knn_insert(bk, bi, &cnt, k, oracle_knn_key(xq, yq, x[i], y[i]), (int32_t)i);
    for (int q = 0; q < k; ++q) {
        idx_out[q] = bi[q];
        if (key_out) key_out[q] = bk[q];
    }
    return 0;
}

/* Bucket-grid search for large inputs: an independent float64 uniform grid that collects
 * candidates ring by ring and re-ranks them by the fp32 key.  It stops once k candidates have
 * key < (r_safe^2)(1 - 1e-6), r_safe = the distance every unvisited point is at least away; the
 * 1e-6 margin dominates the <= 3*2^-24 relative rounding of the fp32 key, so no unvisited point
 * can enter the top k, ties included.  Validated against oracle_knn_brute in the tests. */
typedef struct {
    double xmin, ymin, cell;
    int ncx, ncy;
    int64_t n;
    int64_t *start;      /* [ncx*ncy + 1] */
    int32_t *order;      /* point ids sorted by bucket, ascending id inside a bucket */
} ora_buckets;

ora_buckets *oracle_buckets_build(const float *x, const float *y, int64_t n, double cell)
{
    if (n < 1 || !(cell > 0.0)) return NULL;
    ora_buckets *b = (ora_buckets *)calloc(1, sizeof(ora_buckets));
    double xmin = x[0], xmax = x[0], ymin = y[0], ymax = y[0];
    for (int64_t i = 1; i < n; ++i) {
        if (x[i] < xmin) xmin = x[i];
        if (x[i] > xmax) xmax = x[i];
        if (y[i] < ymin) ymin = y[i];
        if (y[i] > ymax) ymax = y[i];
    }
    b->xmin = xmin; b->ymin = ymin; b->cell = cell; b->n = n;
    b->ncx = (int)floor((xmax - xmin) / cell) + 1;
    b->ncy = (int)floor((ymax - ymin) / cell) + 1;
    size_t nc = (size_t)b->ncx * (size_t)b->ncy;
    b->start = (int64_t *)calloc(nc + 1, sizeof(int64_t));
    b->order = (int32_t *)malloc(sizeof(int32_t) * (size_t)n);
    for (int64_t i = 0; i < n; ++i) {
        int cx = (int)floor(((double)x[i] - xmin) / cell), cy = (int)floor(((double)y[i] - ymin) / cell);
        b->start[(size_t)cy * b->ncx + cx + 1]++;
    }
    for (size_t c = 0; c < nc; ++c) b->start[c + 1] += b->start[c];
    int64_t *fill = (int64_t *)malloc(sizeof(int64_t) * nc);
    memcpy(fill, b->start, sizeof(int64_t) * nc);
    for (int64_t i = 0; i < n; ++i) {
        int cx = (int)floor(((double)x[i] - xmin) / cell), cy = (int)floor(((double)y[i] - ymin) / cell);
        b->order[fill[(size_t)cy * b->ncx + cx]++] = (int32_t)i;
    }
    free(fill);
    return b;
}

void oracle_buckets_free(ora_buckets *b)
{
    if (!b) return;
    free(b->start);
    free(b->order);
    free(b);
}

int oracle_knn_buckets(const ora_buckets *b, const float *x, const float *y, float xq, float yq, int k,
                       int32_t *idx_out, float *key_out)
{
    if (!b || k < 1 || k > b->n || k > 4096) return -1;
    float bk[4096];
    int32_t bi[4096];
    int cnt = 0;
    /* the query's (clamped) bucket; a query outside the bounding box starts from the nearest one */
    double fx = ((double)xq - b->xmin) / b->cell, fy = ((double)yq - b->ymin) / b->cell;
    int qx = (int)floor(fx), qy = (int)floor(fy);
    if (qx < 0) qx = 0;
    if (qx > b->ncx - 1) qx = b->ncx - 1;
    if (qy < 0) qy = 0;
    if (qy > b->ncy - 1) qy = b->ncy - 1;
    int rmax = (b->ncx > b->ncy ? b->ncx : b->ncy);
    for (int r = 0; r <= rmax; ++r) {
        for (int cy = qy - r; cy <= qy + r; ++cy) {
            if (cy < 0 || cy >= b->ncy) continue;
            for (int cx = qx - r; cx <= qx + r; ++cx) {
                if (cx < 0 || cx >= b->ncx) continue;
                if (cy != qy - r && cy != qy + r && cx != qx - r && cx != qx + r) continue;  /* ring only */
                size_t c = (size_t)cy * b->ncx + cx;
                for (int64_t p = b->start[c]; p < b->start[c + 1]; ++p) {
                    int32_t i = b->order[p];
                    knn_insert(bk, bi, &cnt, k, oracle_knn_key(xq, yq, x[i], y[i]), i);
                }
            }
        }
        /* every unvisited bucket lies outside the square of buckets [qx-r, qx+r] x [qy-r, qy+r];
         * the distance from the query to the outside of that square (where it is not clipped by
         * the edge of the bucket grid, beyond which there are no points) is r_safe */
        double r_safe = INFINITY, d;
        if (qx - r > 0)           { d = (double)xq - (b->xmin + (double)(qx - r) * b->cell);     if (d < r_safe) r_safe = d; }
        if (qx + r < b->ncx - 1)  { d = (b->xmin + (double)(qx + r + 1) * b->cell) - (double)xq; if (d < r_safe) r_safe = d; }
        if (qy - r > 0)           { d = (double)yq - (b->ymin + (double)(qy - r) * b->cell);     if (d < r_safe) r_safe = d; }
        if (qy + r < b->ncy - 1)  { d = (b->ymin + (double)(qy + r + 1) * b->cell) - (double)yq; if (d < r_safe) r_safe = d; }
        if (r_safe == INFINITY) break;                       /* the whole grid has been visited */
        if (r_safe > 0.0 && cnt == k && (double)bk[k - 1] < r_safe * r_safe * (1.0 - 1e-6)) break;
    }
    if (cnt < k) return -1;
    for (int q = 0; q < k; ++q) {
        idx_out[q] = bi[q];
        if (key_out) key_out[q] = bk[q];
    }
    return 0;
}

/* K3: variogram.  Exponential exactly as printed at PAPER.md:L157, gamma(h) = C0 (1 - exp(-h/a)),
 * extended by a nugget the textbook way: gamma(h) = nugget + c_p (1 - exp(-h/a)), c_p = sill -
 * nugget, for h > 0.  Spherical (textbook): nugget + c_p (1.5 h/a - 0.5 (h/a)^3) for 0 < h < a,
 * sill for h >= a.  Gaussian (textbook, NEXT-4): nugget + c_p (1 - exp(-(h/a)^2)).  gamma(0) = 0 exactly
 * for all three. */
double oracle_variogram(const ora_vgm *v, double h)
{
    if (h == 0.0) return 0.0;
    double cp = v->sill - v->nugget;
    if (v->model == 0) return v->nugget + cp * (1.0 - exp(-h / v->range));
    if (v->model == 2) return v->nugget + cp * (1.0 - exp(-(h / v->range) * (h / v->range)));
    if (h >= v->range) return v->sill;
    double q = h / v->range;
    return v->nugget + cp * (1.5 * q - 0.5 * q * q * q);
}

/* Geometric anisotropy of the variogram ("many variants ... can be easily
 * implemented on top"; the textbook form, e.g. Cressie, the paper's ref [4]; reading Ani).  The lag vector
 * (dx, dy) between two locations is expressed in the axes of the anisotropy ellipse -- u along the direction of
 * greatest continuity, angle_deg counter-clockwise from +x, w across it -- and the across component is stretched by
 * 1 / ratio, ratio = (range across) / (range along) in (0, 1]:
 *      u =  cos(t) dx + sin(t) dy,   w = (-sin(t) dx + cos(t) dy) / ratio,   h = sqrt(u^2 + w^2),
 * so that gamma(h) with the variogram's `range` is the variogram along the major axis and reaches the same value
 * at `ratio` times the distance across it.  a == NULL: the isotropic lag sqrt(dx^2 + dy^2), exactly as before.
 * Only the variogram sees this lag: the neighbours are still the k nearest in plain Euclidean distance (K2). */
typedef struct { double angle_deg, ratio; } ora_aniso;

double oracle_aniso_lag(const ora_aniso *a, double dx, double dy)
{
    if (!a) return sqrt(dx * dx + dy * dy);
    double t = a->angle_deg * (3.14159265358979323846 / 180.0);
    double u = cos(t) * dx + sin(t) * dy;
    double w = (-sin(t) * dx + cos(t) * dy) / a->ratio;
    return sqrt(u * u + w * w);
}

/* Dense LU with partial pivoting ("Gaussian elimination") of the n x n row-major
 * system A x = b, in place.  Returns -1 when a pivot is smaller in magnitude than tiny. */
int oracle_lu_solve(double *A, double *b, int n, double tiny)
{
    for (int c = 0; c < n; ++c) {
        int p = c;
        double best = fabs(A[(size_t)c * n + c]);
        for (int r = c + 1; r < n; ++r)
            if (fabs(A[(size_t)r * n + c]) > best) { best = fabs(A[(size_t)r * n + c]); p = r; }
        if (!(best >= tiny)) return -1;
        if (p != c) {
            for (int q = 0; q < n; ++q) { double tmp = A[(size_t)c * n + q]; A[(size_t)c * n + q] = A[(size_t)p * n + q]; A[(size_t)p * n + q] = tmp; }
            double tb = b[c]; b[c] = b[p]; b[p] = tb;
        }
        for (int r = c + 1; r < n; ++r) {
            double f = A[(size_t)r * n + c] / A[(size_t)c * n + c];
            A[(size_t)r * n + c] = 0.0;
            for (int q = c + 1; q < n; ++q) A[(size_t)r * n + q] -= f * A[(size_t)c * n + q];
            b[r] -= f * b[c];
        }
    }
    for (int r = n - 1; r >= 0; --r) {
        double s = b[r];
        for (int q = r + 1; q < n; ++q) s -= A[(size_t)r * n + q] * b[q];
        b[r] = s / A[(size_t)r * n + r];
    }
    return 0;
}

/* K4: ordinary-kriging weights in the gamma form (the standard form of the system the paper
 * prints garbled at PAPER.md:L161-L165, reading D3):
 *      [ Gamma  1 ] [ lambda ]   [ gamma0 ]
 *      [ 1^T    0 ] [   mu   ] = [   1    ],   Gamma_ij = gamma(|p_i - p_j|), gamma0_i = gamma(|q - p_i|)
 * h in float64 from the (fp32-valued) coordinates.  lambda[k], *mu out.  -1 if singular. */
static int ok_weights_impl(const double *px, const double *py, int k, double xq, double yq,
                           const ora_vgm *v, const ora_aniso *a, double *lambda, double *mu)
{
    int n = k + 1;
    double *A = (double *)malloc(sizeof(double) * (size_t)n * (size_t)n);
    double *b = (double *)malloc(sizeof(double) * (size_t)n);
    if (!A || !b) { free(A); free(b); return -2; }
    for (int i = 0; i < k; ++i) {
        for (int j = 0; j < k; ++j) {
            double dx = px[i] - px[j], dy = py[i] - py[j];
            A[(size_t)i * n + j] = oracle_variogram(v, oracle_aniso_lag(a, dx, dy));
        }
        A[(size_t)i * n + k] = 1.0;
        A[(size_t)k * n + i] = 1.0;
        double dx = xq - px[i], dy = yq - py[i];
        b[i] = oracle_variogram(v, oracle_aniso_lag(a, dx, dy));
    }
    A[(size_t)k * n + k] = 0.0;
    b[k] = 1.0;
    int rc = oracle_lu_solve(A, b, n, 1e-12 * v->sill);
    if (rc == 0) {
        for (int i = 0; i < k; ++i) lambda[i] = b[i];
        if (mu) *mu = b[k];
    }
    free(A);
    free(b);
    return rc;
}

int oracle_ok_weights(const double *px, const double *py, int k, double xq, double yq,
                      const ora_vgm *v, double *lambda, double *mu)
{
    return ok_weights_impl(px, py, k, xq, yq, v, NULL, lambda, mu);
}

/* The same system with the anisotropic lag in Gamma and gamma0 (NEXT-4).  ratio outside (0, 1]: -3. */
int oracle_ok_weights_aniso(const double *px, const double *py, int k, double xq, double yq,
                            const ora_vgm *v, const ora_aniso *a, double *lambda, double *mu)
{
    if (!a || !(a->ratio > 0.0) || a->ratio > 1.0 || !isfinite(a->angle_deg)) return -3;
    return ok_weights_impl(px, py, k, xq, yq, v, a, lambda, mu);
}

/* K1-K5 for a list of query points (fp32 coordinates): neighbours (K2), weights (K3, K4) and
 * z_hat = sum lambda_i z_i (K5).  buckets == NULL -> brute-force search.
 * nbr_out [nq*k] (or NULL) receives original indices in ascending (key, index) order;
 * lambda_out [nq*k] (or NULL) the weights in the same order.  A singular node gets NaN.
 * Returns the number of singular nodes, or a negative error. */
static int64_t krige_points_impl(const float *x, const float *y, const float *z, int64_t n,
                            const ora_buckets *buckets,
                            const float *xq, const float *yq, int64_t nq,
                            const ora_vgm *v, const ora_aniso *a, int k,
                            double *zhat, int32_t *nbr_out, double *lambda_out, double *var_out)
{
    if (!x || !y || !z || !xq || !yq || !zhat || k < 1 || k > n || k > 4096) return -1;
    if (a && (!(a->ratio > 0.0) || a->ratio > 1.0 || !isfinite(a->angle_deg))) return -1;
    if (!(v->range > 0.0) || !(v->sill > 0.0) || v->nugget < 0.0 || v->nugget > v->sill) return -1;
    if (v->model != 0 && v->model != 1 && v->model != 2) return -1;
    int64_t failed = 0;
    #pragma omp parallel for schedule(dynamic, 64) reduction(+:failed)
    for (int64_t q = 0; q < nq; ++q) {
        int32_t idx[4096];
        double px[4096], py[4096], lam[4096];
        int rc = buckets ? oracle_knn_buckets(buckets, x, y, xq[q], yq[q], k, idx, NULL)
                         : oracle_knn_brute(x, y, n, xq[q], yq[q], k, idx, NULL);
        double est = NAN, var = NAN, mu = 0.0;
        if (rc == 0) {
            for (int i = 0; i < k; ++i) { px[i] = (double)x[idx[i]]; py[i] = (double)y[idx[i]]; }
            rc = ok_weights_impl(px, py, k, (double)xq[q], (double)yq[q], v, a, lam, &mu);
        }
        if (rc == 0) {
            est = 0.0;
            for (int i = 0; i < k; ++i) est += lam[i] * (double)z[idx[i]];
            /* ordinary-kriging variance (textbook, e.g. Cressie, the paper's ref [4]):
             * sigma^2 = sum_i lambda_i gamma(|q - p_i|) + mu, mu the Lagrange multiplier of the gamma form */
            var = mu;
            for (int i = 0; i < k; ++i) {
                double dx = (double)xq[q] - px[i], dy = (double)yq[q] - py[i];
                var += lam[i] * oracle_variogram(v, oracle_aniso_lag(a, dx, dy));
            }
        } else {
            failed += 1;
            for (int i = 0; i < k; ++i) lam[i] = NAN;
        }
        zhat[q] = est;
        if (var_out) var_out[q] = var;
        if (nbr_out) for (int i = 0; i < k; ++i) nbr_out[q * k + i] = idx[i];
        if (lambda_out) for (int i = 0; i < k; ++i) lambda_out[q * k + i] = lam[i];
    }
    return failed;
}

int64_t oracle_krige_points(const float *x, const float *y, const float *z, int64_t n,
                            const ora_buckets *buckets,
                            const float *xq, const float *yq, int64_t nq,
                            const ora_vgm *v, int k,
                            double *zhat, int32_t *nbr_out, double *lambda_out)
{
    return krige_points_impl(x, y, z, n, buckets, xq, yq, nq, v, NULL, k, zhat, nbr_out, lambda_out, NULL);
}

/* The same with the kriging variance sigma^2 in var_out [nq]. */
int64_t oracle_krige_points_var(const float *x, const float *y, const float *z, int64_t n,
                                const ora_buckets *buckets,
                                const float *xq, const float *yq, int64_t nq,
                                const ora_vgm *v, int k,
                                double *zhat, double *var_out, int32_t *nbr_out)
{
    return krige_points_impl(x, y, z, n, buckets, xq, yq, nq, v, NULL, k, zhat, nbr_out, NULL, var_out);
}

/* The same with a geometrically anisotropic variogram (NEXT-4): neighbours by plain distance (K2), lags of the
 * variogram by oracle_aniso_lag.  var_out, nbr_out, lambda_out may be NULL. */
int64_t oracle_krige_points_aniso(const float *x, const float *y, const float *z, int64_t n,
                                  const ora_buckets *buckets,
                                  const float *xq, const float *yq, int64_t nq,
                                  const ora_vgm *v, const ora_aniso *a, int k,
                                  double *zhat, double *var_out, int32_t *nbr_out, double *lambda_out)
{
    if (!a) return -1;
    return krige_points_impl(x, y, z, n, buckets, xq, yq, nq, v, a, k, zhat, nbr_out, lambda_out, var_out);
}

/* ================================================================== grid-window kriging (hole filling)
 * SURVEY.md 8(f) NEXT-2; PAPER.md:L163 ("the implementation in this study uses a 5x5 grid"), L171 and L180
 * (fallback to bilinear "if enough valid candidate neighbors are not found"), L179 (helper that finds "the
 * nearest n valid candidate neighbors"), L225-L234 (Grid B: cells removed at random from a regular grid are
 * interpolated back).  Readings W1-W4 of DESIGN.md:
 *  W1  a valid (non-NaN) cell is copied; a NaN cell (a hole) at row i, column j is estimated by ordinary kriging
 *      (K3-K5 above, gamma-form LU) from valid cells of the (2 half + 1)^2 window centred on it, clipped by the grid;
 *  W2  "nearest n valid": the n_max candidates with the smallest (key, window order), key = fmaf(ddx, ddx, ddy*ddy)
 *      in fp32 with ddx = (float)dj * dx, ddy = (float)di * dy (fp32 products; dj, di the lattice offsets), window
 *      order = row-major over the window; neighbours are used in window order;
 *  W3  fewer than n_min valid candidates -> the bilinear fallback;
 *  W4  bilinear at a hole = the formula of PAPER.md:L132 on the rectangle spanned by columns j-1, j+1 and rows i-1,
 *      i+1, which the hole sits in the middle of (t = s = 1/2): the mean of the four diagonal neighbours, NaN if
 *      one of them is NaN or outside the grid (bilinear has no fallback, L182).
 * how [ny*nx] (or NULL): 0 = valid cell copied, 1..64 = kriged from that many neighbours, 255 = bilinear fallback.
 * A singular system gives NaN (counted in the return value). */
int64_t oracle_krige_window(const float *in, const ora_geom *g, int half, int n_max, int n_min, const ora_vgm *v,
                            double *out, uint8_t *how)
{
    if (!in || !out || g->nx < 2 || g->ny < 2 || half < 1 || half > 3 || n_max < 1 || n_max > 64 || n_min < 1) return -1;
    if (!(g->dx > 0.0f) || !(g->dy > 0.0f)) return -1;
    const int nx = g->nx, ny = g->ny, side = 2 * half + 1;
    int64_t failed = 0;
    #pragma omp parallel for schedule(dynamic, 8) reduction(+:failed)
    for (int i = 0; i < ny; ++i) {
        for (int j = 0; j < nx; ++j) {
            const size_t at = (size_t)i * nx + j;
            if (!isnan(in[at])) { out[at] = (double)in[at]; if (how) how[at] = 0; continue; }
            /* W1: valid cells of the clipped window, in window (row-major) order */
            int ci[64], cj[64], m = 0;
            float key[64];
            for (int a = -half; a <= half; ++a)
                for (int b = -half; b <= half; ++b) {
                    int ii = i + a, jj = j + b;
                    if ((a == 0 && b == 0) || ii < 0 || ii >= ny || jj < 0 || jj >= nx) continue;
                    if (isnan(in[(size_t)ii * nx + jj])) continue;
                    volatile float ddx = (float)b * g->dx;
                    volatile float ddy = (float)a * g->dy;
                    volatile float pr = ddy * ddy;
                    ci[m] = ii; cj[m] = jj; key[m] = fmaf(ddx, ddx, pr); ++m;
                }
            (void)side;
            /* W2: keep the n_max nearest by (key, window order) */
            int keep[64], k = 0;
            for (int e = 0; e < m; ++e) {
                int rank = 0;
                for (int f = 0; f < m; ++f) rank += (key[f] < key[e] || (key[f] == key[e] && f < e));
                if (rank < n_max) keep[k++] = e;
            }
            if (k < n_min) {
                /* W3 + W4: bilinear on the rectangle of the diagonal neighbours, t = s = 1/2 */
                double f = NAN;
                if (i - 1 >= 0 && i + 1 < ny && j - 1 >= 0 && j + 1 < nx) {
                    double Q11 = in[(size_t)(i - 1) * nx + j - 1], Q21 = in[(size_t)(i - 1) * nx + j + 1];
                    double Q12 = in[(size_t)(i + 1) * nx + j - 1], Q22 = in[(size_t)(i + 1) * nx + j + 1];
                    double t = 0.5, s = 0.5;
                    f = (1.0 - t) * (1.0 - s) * Q11 + t * (1.0 - s) * Q21 + (1.0 - t) * s * Q12 + t * s * Q22;
                }
                out[at] = f;
                if (how) how[at] = 255;
                continue;
            }
            double px[64], py[64], lam[64];
            for (int e = 0; e < k; ++e) {
                px[e] = (double)g->x0 + (double)cj[keep[e]] * (double)g->dx;
                py[e] = (double)g->y0 + (double)ci[keep[e]] * (double)g->dy;
            }
            double xq = (double)g->x0 + (double)j * (double)g->dx, yq = (double)g->y0 + (double)i * (double)g->dy;
            double est = NAN;
            if (oracle_ok_weights(px, py, k, xq, yq, v, lam, NULL) == 0) {
                est = 0.0;
                for (int e = 0; e < k; ++e) est += lam[e] * (double)in[(size_t)ci[keep[e]] * nx + cj[keep[e]]];
            } else {
                failed += 1;
            }
            out[at] = est;
            if (how) how[at] = (uint8_t)k;
        }
    }
    return failed;
}
