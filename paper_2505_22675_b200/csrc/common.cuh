// common.cuh -- shared plumbing of libbathy.so (CUDA path only; the oracle shares nothing with this).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <math.h>
#include <atomic>
#include "../../include/bathy.h"

namespace bathy {

constexpr int kSMs = 148;            // B200: 2 dies x 74 SMs

void count_launch(int n = 1);        // api.cu: backs bathy_launch_count()

#define BATHY_CUDA_TRY(expr)                         \
    do {                                             \
        cudaError_t e__ = (expr);                    \
        if (e__ != cudaSuccess) { cudaGetLastError(); return BATHY_ERR_CUDA; } /* (clears the non-sticky error) */ \
    } while (0)

// Runs `f` (a cudaFuncSetAttribute sequence) once per CUDA DEVICE of this process: function attributes
// are per device, so a process-wide flag would leave the second device of a process without them.
// Thread-safe; a racing first call runs f twice, which is harmless.
struct DeviceOnce { std::atomic<unsigned long long> mask{0}; };
template <class F>
inline int once_per_device(DeviceOnce& o, F f)
{
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return BATHY_ERR_CUDA;
    const unsigned long long bit = 1ull << (dev & 63);
    if (dev < 64 && (o.mask.load(std::memory_order_acquire) & bit)) return BATHY_OK;
    const int rc = f();
    if (rc == BATHY_OK && dev < 64) o.mask.fetch_or(bit, std::memory_order_release);
    return rc;
}

inline int launch_status() { return cudaGetLastError() == cudaSuccess ? BATHY_OK : BATHY_ERR_CUDA; }

inline bool finite_f(float v) { return isfinite(v); }

inline int check_in_geom(const grid_geom_t& g)
{
    if (g.nx < 2 || g.ny < 2) return BATHY_ERR_GEOMETRY;
    if (!finite_f(g.x0) || !finite_f(g.y0) || !finite_f(g.dx) || !finite_f(g.dy)) return BATHY_ERR_GEOMETRY;
    if (!(g.dx > 0.0f) || !(g.dy > 0.0f)) return BATHY_ERR_GEOMETRY;
    return BATHY_OK;
}

inline int check_out_geom(const grid_geom_t& g)
{
    if (g.nx < 1 || g.ny < 1) return BATHY_ERR_GEOMETRY;
    if (!finite_f(g.x0) || !finite_f(g.y0) || !finite_f(g.dx) || !finite_f(g.dy)) return BATHY_ERR_GEOMETRY;
    if (!(g.dx > 0.0f) || !(g.dy > 0.0f)) return BATHY_ERR_GEOMETRY;
    return BATHY_OK;
}

// One axis of the output->input index map (readings B1/B2): u = ((o0 + J*od) - i0) / id in float64
// from the fp32 geometry fields, each operation rounded separately (no contraction) so that the
// interval decision is taken in the same precision as the definition.
struct AxisMap {
    double o0, od, i0, id;
    int n_in, n_out;
};

inline AxisMap axis_x(const grid_geom_t& in, const grid_geom_t& out)
{
    return AxisMap{(double)out.x0, (double)out.dx, (double)in.x0, (double)in.dx, in.nx, out.nx};
}
inline AxisMap axis_y(const grid_geom_t& in, const grid_geom_t& out)
{
    return AxisMap{(double)out.y0, (double)out.dy, (double)in.y0, (double)in.dy, in.ny, out.ny};
}

__device__ __forceinline__ double axis_u(const AxisMap& m, int J)
{
    double x = __dadd_rn(m.o0, __dmul_rn((double)J, m.od));
    return __ddiv_rn(__dsub_rn(x, m.i0), m.id);
}

// Interval index (or -1 when the node is outside the input extent) and local coordinate t.
__device__ __forceinline__ int axis_locate(const AxisMap& m, int J, float* t)
{
    double u = axis_u(m, J);
    if (!(u >= 0.0) || !(u <= (double)(m.n_in - 1))) { *t = 0.0f; return -1; }
    int i = (int)floor(u);
    i = min(i, m.n_in - 2);
    i = max(i, 0);
    *t = (float)(u - (double)i);
    return i;
}

// Interval index clamped into [0, n_in-2] whatever u is (footprint bounds of a tile).
__device__ __forceinline__ int axis_clamped(const AxisMap& m, int J)
{
    double u = axis_u(m, J);
    if (!(u >= 0.0)) return 0;
    if (u >= (double)(m.n_in - 1)) return m.n_in - 2;
    return min((int)floor(u), m.n_in - 2);
}

// Host-side bound on the input footprint (in samples) of `n_nodes` consecutive output nodes.
inline long long footprint_bound(const AxisMap& m, int n_nodes)
{
    double span = (double)(n_nodes - 1) * m.od / m.id;
    if (!(span < 1e9)) return (long long)2e9;
    return (long long)floor(span) + 3;        // floor(u_last) - floor(u_first) <= floor(span)+1, +1 sample, +1 slack
}


// Stages rows [j0, j0 + fh) x columns [i0, i0 + fw) of the row-major input (leading dimension n_in) in shared
// memory by cp.async, ALL of it in flight at once; the caller commits / waits.  Row r of the footprint starts at
// s_tile + r * pitch + offx, where pitch = stage_pitch(fw) and offx = i0 & 3: with 16-byte aligned input rows the
// copy runs in whole 16-byte vectors from the aligned column at or before i0 (columns past the row end are zero
// filled), else element by element.  Shared by the bilinear and Catmull-Rom tile kernels.
__host__ __device__ __forceinline__ int stage_pitch(int fw) { return (fw + 6) & ~3; }   // >= (i0 & 3) + fw, a multiple of 4

__device__ __forceinline__ void stage_footprint(const float* __restrict__ in, int n_in, int i0, int j0, int fw, int fh,
                                                float* s_tile, int tid, int nthreads)
{
    const int a_lo = i0 & ~3, offx = i0 - a_lo;
    const int pitch = stage_pitch(fw);
    if ((reinterpret_cast<uintptr_t>(in) & 15) == 0 && (n_in & 3) == 0) {
        const int vpr = pitch >> 2;
        for (int v = tid; v < fh * vpr; v += nthreads) {
            const int r = v / vpr, c4 = (v - r * vpr) << 2;
            const int col = a_lo + c4;
            const int bytes = max(0, min(16, (n_in - col) * 4));         // past the row end: zero fill
            const float* src = in + (size_t)(j0 + r) * n_in + min(col, n_in - 4);
            const unsigned dst = (unsigned)__cvta_generic_to_shared(s_tile + r * pitch + c4);
            asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;" :: "r"(dst), "l"(src), "r"(bytes) : "memory");
        }
    } else {
        for (int v = tid; v < fh * fw; v += nthreads) {
            const int r = v / fw, c = v - r * fw;
            const unsigned dst = (unsigned)__cvta_generic_to_shared(s_tile + r * pitch + offx + c);
            asm volatile("cp.async.ca.shared.global [%0], [%1], 4;" :: "r"(dst), "l"(in + (size_t)(j0 + r) * n_in + i0 + c) : "memory");
        }
    }
}

// ---------------------------------------------------------------------------------------------
// Packed fp32x2 arithmetic of sm_100 (SASS FFMA2 / FMUL2 / FADD2): one issue slot, two fp32
// operations.  A pair lives in a 64-bit register; a scalar operand packed as (a, a) is folded by
// ptxas into the broadcast operand form.
typedef unsigned long long u64;
__device__ __forceinline__ u64 pack2(float lo, float hi)
{
    u64 r;
    asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(lo), "f"(hi));
    return r;
}
__device__ __forceinline__ float lo_of(u64 v)
{
    float lo;
    float hi __attribute__((unused));
    asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(v));
    return lo;
}
__device__ __forceinline__ float hi_of(u64 v)
{
    float lo __attribute__((unused));
    float hi;
    asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(v));
    return hi;
}
__device__ __forceinline__ u64 ffma2(u64 a, u64 b, u64 c)
{
    u64 d;
    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(d) : "l"(a), "l"(b), "l"(c));
    return d;
}
__device__ __forceinline__ u64 fmul2(u64 a, u64 b)
{
    u64 d;
    asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b));
    return d;
}
__device__ __forceinline__ u64 fadd2(u64 a, u64 b)
{
    u64 d;
    asm("add.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b));
    return d;
}

}  // namespace bathy
