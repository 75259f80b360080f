// Device-side helpers shared by the demons kernels (sm_100a).  Product code: nothing here is
// shared with oracle/.
#pragma once

#include <cuda_runtime.h>
#include <stdint.h>

namespace demons {

struct Dims {
    int nx, ny, nz;
};

__host__ __device__ __forceinline__ size_t nvox(const Dims& d) {
    return (size_t)d.nx * (size_t)d.ny * (size_t)d.nz;
}

constexpr int LHIST = 16;  // power of two >= 11 (lag of 10 iterations)

// Per-registration control block in the workspace (one per pair of a batch): block ticket of the metric
// reduction, statistics row cursor and the state of the device-side stopping rule.
struct Control {
    unsigned int ticket;       // block-completion counter, left at 0 by the last block
    unsigned int row_counter;  // next row of the statistics buffer
    unsigned int level_iter;   // iterations executed on the current level
    int stop_force;            // set when the stopping rule fires; force kernels then skip
    int stop_smooth;           // set by the first skipped force kernel; smoothing then skips
    int pad0[11];
    int lvalid[LHIST];         // l_n defined (sum|u| > 0)
    double lhist[LHIST];       // ring of relative norms l_n of this level
    int iters_done[8];         // per level, copied from level_iter when the level ends
    int pad1[56];
};
static_assert(sizeof(Control) == 512, "control block layout");

// Where the three metrics of one warp_force pass go (S6 of the hot path).
// Per-block partials in double, fixed-order final sum by the last block to finish: the result
// does not depend on scheduling.  Pair b of a batched launch uses ctl[b], partials + b * 5 * stride and
// out + b * out_stride.
struct MetricSink {
    double* partials;   // [pairs][5][stride] block partials
    Control* ctl;       // [pairs]
    double* out;        // nullptr: metrics not wanted
    size_t out_stride;  // doubles between the outputs of consecutive pairs
    int stride;         // capacity of one partial row (>= number of blocks per pair)
    int driver;         // 1 inside demons_register: rows advance, the stopping rule runs, stop flags are honoured
    double eps;         // stopping rule threshold (<= 0: off)
    int defer;          // 1: force blocks only store their partials; k_metrics_final sums and publishes them
    unsigned nblocks;   // k_metrics_final only: block partials per pair written by the force kernel before it
};

__device__ __forceinline__ float lerpf(float a, float b, float t) { return fmaf(t, b - a, a); }

// One axis of O2 (reading A11): p = x + u clamped to [0, n-1], i0 = floor(p), f = p - i0,
// i1 = min(i0 + 1, n - 1).
//  * The split is taken on u, not on x + u: floor(x + u) = x + floor(u) for integer x and
//    u - floor(u) is exact in fp32, so no bits of the fraction are lost to the magnitude of x.
//  * floor without the conversion unit: for |u| <= 2^21, t = u + 1.5*2^23 ROUNDED DOWN (add.rm) has
//    ulp 1, so t - 1.5*2^23 = floor(u) exactly and the low mantissa bits of t are that integer.
// floor_split returns i = x + floor(u) (unclamped) and f = u - floor(u).
__device__ __forceinline__ int floor_split(int x, float u, float& f) {
    u = fminf(fmaxf(u, -2097152.f), 2097152.f);
    const float t = __fadd_rd(u, 12582912.f);
    f = u - (t - 12582912.f);
    return __float_as_int(t) - 0x4B400000 + x;
}

// Generic form: the clamp is taken on the two indices.  When p is outside [0, n-1] both become the
// same edge voxel and lerp(a, a, f) = a exactly, which is what clamping p does.
__device__ __forceinline__ void split_axis(int x, float u, int n, int& i0, int& i1, float& f) {
    const int i = floor_split(x, u, f);
    i0 = min(max(i, 0), n - 1);
    i1 = min(max(i + 1, 0), n - 1);
}

// Software trilinear sample of I at (x + ux, y + uy, z + uz): PAPER.md L179-181 ("our own
// trilinear interpolation function").  Interpolates along x, then y, then z.  32-bit offsets
// (volumes have fewer than 2^29 voxels, checked by demons_create).
__device__ __forceinline__ float trilinear(const float* __restrict__ I, const Dims& d, int x, int y,
                                           int z, float ux, float uy, float uz) {
    int x0, x1, y0, y1, z0, z1;
    float fx, fy, fz;
    split_axis(x, ux, d.nx, x0, x1, fx);
    split_axis(y, uy, d.ny, y0, y1, fy);
    split_axis(z, uz, d.nz, z0, z1, fz);
    const int zo0 = z0 * d.ny, zo1 = z1 * d.ny;
    const int r00 = (zo0 + y0) * d.nx, r10 = (zo0 + y1) * d.nx;
    const int r01 = (zo1 + y0) * d.nx, r11 = (zo1 + y1) * d.nx;
    const float c000 = __ldg(I + (unsigned)(r00 + x0)), c100 = __ldg(I + (unsigned)(r00 + x1));
    const float c010 = __ldg(I + (unsigned)(r10 + x0)), c110 = __ldg(I + (unsigned)(r10 + x1));
    const float c001 = __ldg(I + (unsigned)(r01 + x0)), c101 = __ldg(I + (unsigned)(r01 + x1));
    const float c011 = __ldg(I + (unsigned)(r11 + x0)), c111 = __ldg(I + (unsigned)(r11 + x1));
    const float a00 = lerpf(c000, c100, fx), a10 = lerpf(c010, c110, fx);
    const float a01 = lerpf(c001, c101, fx), a11 = lerpf(c011, c111, fx);
    const float b0 = lerpf(a00, a10, fy), b1 = lerpf(a01, a11, fy);
    return lerpf(b0, b1, fz);
}

// ---- cell form of the same sample (the fast kernels) --------------------------------------------
// The 2x2x2 cell is addressed by ONE offset o (its low corner); the other seven values sit at fixed
// distances (+1, +nx, +nx*ny), so a lane issues its eight loads from one base with no per-load
// index arithmetic and no branch.  The clamp of O2 is folded into (index, fraction):
//     i < 0      ->  cell 0,     f = 0   (the sample is voxel 0)
//     i > n - 2  ->  cell n - 2, f = 1   (the sample is voxel n - 1)
// lerp1 is exact at both ends (t = 0 -> a, t = 1 -> b), so these reproduce the clamped sample bit for
// bit -- with fma(t, b - a, a) the t = 1 case returns a + (b - a) != b and identical volumes would no
// longer give exactly zero force at the high faces (pin P1).  lerp1 costs one more rounding per level.
// Needs n >= 2 on every axis (the launchers send degenerate volumes elsewhere).
__device__ __forceinline__ float lerp1(float a, float b, float t) { return fmaf(t, b, fmaf(-t, a, a)); }

__device__ __forceinline__ void clamp_cell_axis(int& i, float& f, int n) {
    f = i < 0 ? 0.f : f;
    f = i > n - 2 ? 1.f : f;
    i = min(max(i, 0), n - 2);
}

// Cells of NV voxels (xs[j], y, z) of one lane.  The clamp arithmetic of an axis is skipped when no
// lane of the warp needs it (warp-uniform tests; only pure ALU code sits under the branches).
template <int NV>
__device__ __forceinline__ void make_cells(const Dims& d, const int (&xs)[NV], int y, int z, const float (&ux)[NV],
                                           const float (&uy)[NV], const float (&uz)[NV], unsigned (&o)[NV],
                                           float (&fx)[NV], float (&fy)[NV], float (&fz)[NV]) {
    int ix[NV], iy[NV], iz[NV];
    bool inx = true, iny = true, inz = true;
#pragma unroll
    for (int j = 0; j < NV; ++j) {
        ix[j] = floor_split(xs[j], ux[j], fx[j]);
        iy[j] = floor_split(y, uy[j], fy[j]);
        iz[j] = floor_split(z, uz[j], fz[j]);
        inx = inx && (unsigned)ix[j] < (unsigned)(d.nx - 1);
        iny = iny && (unsigned)iy[j] < (unsigned)(d.ny - 1);
        inz = inz && (unsigned)iz[j] < (unsigned)(d.nz - 1);
    }
    // one vote per axis: a warp that spans a row end nearly always needs the x clamp, rarely the others
    const unsigned mask = __activemask();
    if (!__all_sync(mask, inx)) {
#pragma unroll
        for (int j = 0; j < NV; ++j) clamp_cell_axis(ix[j], fx[j], d.nx);
    }
    if (!__all_sync(mask, iny)) {
#pragma unroll
        for (int j = 0; j < NV; ++j) clamp_cell_axis(iy[j], fy[j], d.ny);
    }
    if (!__all_sync(mask, inz)) {
#pragma unroll
        for (int j = 0; j < NV; ++j) clamp_cell_axis(iz[j], fz[j], d.nz);
    }
#pragma unroll
    for (int j = 0; j < NV; ++j) o[j] = (unsigned)((iz[j] * d.ny + iy[j]) * d.nx + ix[j]);
}

// The eight loads of a cell, issued back to back (x fastest).
__device__ __forceinline__ void load_cell(const float* __restrict__ I, const Dims& d, unsigned o, float (&c)[8]) {
    const unsigned o01 = o + (unsigned)(d.nx * d.ny);
    const float* r00 = I + o;
    const float* r10 = I + (o + (unsigned)d.nx);
    const float* r01 = I + o01;
    const float* r11 = I + (o01 + (unsigned)d.nx);
    c[0] = __ldg(r00), c[1] = __ldg(r00 + 1), c[2] = __ldg(r10), c[3] = __ldg(r10 + 1);
    c[4] = __ldg(r01), c[5] = __ldg(r01 + 1), c[6] = __ldg(r11), c[7] = __ldg(r11 + 1);
}

// Interpolation along x, then y, then z (O2).  The two z planes go through the x and y lerps as packed
// f32x2 pairs (FFMA2 on sm_100): 8 instructions instead of 14, the same roundings as 7 scalar lerp1.
__device__ __forceinline__ float2 lerp1x2(float2 a, float2 b, float t) {
    const float2 t2 = make_float2(t, t), nt2 = make_float2(-t, -t);
    return __ffma2_rn(t2, b, __ffma2_rn(nt2, a, a));
}
__device__ __forceinline__ float lerp_cell(const float (&c)[8], float fx, float fy, float fz) {
    const float2 x0 = lerp1x2(make_float2(c[0], c[4]), make_float2(c[1], c[5]), fx);  // (a00, a01)
    const float2 x1 = lerp1x2(make_float2(c[2], c[6]), make_float2(c[3], c[7]), fx);  // (a10, a11)
    const float2 yb = lerp1x2(x0, x1, fy);                                            // (b0, b1)
    return lerp1(yb.x, yb.y, fz);
}

// VEC consecutive floats along x: one 128-bit access when VEC == 4.
template <int VEC>
__device__ __forceinline__ void load_vec(const float* __restrict__ p, float (&v)[VEC]) {
    if constexpr (VEC == 4) {
        const float4 t = __ldg(reinterpret_cast<const float4*>(p));
        v[0] = t.x;
        v[1] = t.y;
        v[2] = t.z;
        v[3] = t.w;
    } else {
#pragma unroll
        for (int j = 0; j < VEC; ++j) v[j] = __ldg(p + j);
    }
}

template <int VEC>
__device__ __forceinline__ void store_vec(float* __restrict__ p, const float (&v)[VEC]) {
    if constexpr (VEC == 4) {
        *reinterpret_cast<float4*>(p) = make_float4(v[0], v[1], v[2], v[3]);
    } else {
#pragma unroll
        for (int j = 0; j < VEC; ++j) p[j] = v[j];
    }
}

// Centre values and central-difference gradient (O1: g_c = (I(x+e_c) - I(x-e_c))/2, indices
// clamped; reading A7) of VEC consecutive voxels starting at (x0, y, z).
template <int VEC>
__device__ __forceinline__ void centre_and_gradient(const float* __restrict__ I, const Dims& d, int x0,
                                                    int y, int z, float (&c)[VEC], float (&gx)[VEC],
                                                    float (&gy)[VEC], float (&gz)[VEC]) {
    const int plane = d.nx * d.ny;
    const int row = z * plane + y * d.nx;
    float ym[VEC], yp[VEC], zm[VEC], zp[VEC];
    load_vec<VEC>(I + (unsigned)(row + x0), c);
    const float xm = __ldg(I + (unsigned)(row + max(x0 - 1, 0)));
    const float xp = __ldg(I + (unsigned)(row + min(x0 + VEC, d.nx - 1)));
    load_vec<VEC>(I + (unsigned)(row + x0 - (y > 0 ? d.nx : 0)), ym);
    load_vec<VEC>(I + (unsigned)(row + x0 + (y < d.ny - 1 ? d.nx : 0)), yp);
    load_vec<VEC>(I + (unsigned)(row + x0 - (z > 0 ? plane : 0)), zm);
    load_vec<VEC>(I + (unsigned)(row + x0 + (z < d.nz - 1 ? plane : 0)), zp);
#pragma unroll
    for (int j = 0; j < VEC; ++j) {
        const float l = j > 0 ? c[j - 1] : xm;
        const float r = j < VEC - 1 ? c[j + 1] : xp;
        gx[j] = 0.5f * (r - l);
        gy[j] = 0.5f * (yp[j] - ym[j]);
        gz[j] = 0.5f * (zp[j] - zm[j]);
    }
}

// sqrt on the special-function unit (relative error ~2^-22); used for the metrics only.
__device__ __forceinline__ float fast_sqrt(float x) {
    float r;
    asm("sqrt.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x));
    return r;
}

// q(num, den) = den > 1e-9 ? num/den : 0 -- the zero guard of reading A6.
__device__ __forceinline__ float guarded_div(float num, float den) {
    return den > 1e-9f ? __fdividef(num, den) : 0.f;
}

__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
    return v;
}

__device__ __forceinline__ double warp_max(double v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v = fmax(v, __shfl_down_sync(0xffffffffu, v, o));
    return v;
}

// Fixed-order sum (max for the last NMAX) of the `nblocks` block partials of NV quantities; the totals end up in v of
// thread 0.  Must be called by every thread of the block.
template <int NV, int NMAX = 0>
__device__ __forceinline__ void final_sum(double (&v)[NV], const double* partials, int stride, unsigned int nblocks) {
    __shared__ double fs[NV][32];
    const int tid = threadIdx.x + blockDim.x * (threadIdx.y + blockDim.y * threadIdx.z);
    const int nthreads = blockDim.x * blockDim.y * blockDim.z;
    const int lane = tid & 31, wid = tid >> 5, nwarps = (nthreads + 31) >> 5;
#pragma unroll
    for (int i = 0; i < NV; ++i) {
        const bool is_max = i >= NV - NMAX;
        double r = is_max ? -1.0e300 : 0.0;
        const volatile double* p = partials + (size_t)i * stride;
        for (unsigned int b = tid; b < nblocks; b += nthreads) r = is_max ? fmax(r, p[b]) : r + p[b];
        r = is_max ? warp_max(r) : warp_sum(r);
        if (lane == 0) fs[i][wid] = r;
    }
    __syncthreads();
    if (wid == 0) {
#pragma unroll
        for (int i = 0; i < NV; ++i) {
            const bool is_max = i >= NV - NMAX;
            double q = lane < nwarps ? fs[i][lane] : (is_max ? -1.0e300 : 0.0);
            q = is_max ? warp_max(q) : warp_sum(q);
            v[i] = q;
        }
    }
}

// Block-wide reduction of NV doubles and publication of the block partial, nothing else: the deferred form, summed
// later by k_metrics_final (no fence, no ticket: the kernel boundary orders the partials).
template <int NV>
__device__ __forceinline__ void block_reduce_store(double (&v)[NV], double* partials, int stride, unsigned int bid) {
    __shared__ double sm[NV][32];
    const int tid = threadIdx.x + blockDim.x * (threadIdx.y + blockDim.y * threadIdx.z);
    const int nthreads = blockDim.x * blockDim.y * blockDim.z;
    const int lane = tid & 31, wid = tid >> 5, nwarps = (nthreads + 31) >> 5;
#pragma unroll
    for (int i = 0; i < NV; ++i) {
        const double r = warp_sum(v[i]);
        if (lane == 0) sm[i][wid] = r;
    }
    __syncthreads();
    if (wid == 0) {
#pragma unroll
        for (int i = 0; i < NV; ++i) {
            double r = lane < nwarps ? sm[i][lane] : 0.0;
            r = warp_sum(r);
            if (lane == 0) partials[(size_t)i * stride + bid] = r;
        }
    }
}

// Block-wide reduction of NV doubles (sum; the last NMAX of them by max), publication of the
// block partial, and the fixed-order final reduction by the last block to arrive (of the `nblocks` that
// share this ticket; `bid` = this block's index among them).  Returns true in thread 0 of the last block,
// with the totals in v.  Must be called by every thread.
template <int NV, int NMAX = 0>
__device__ __forceinline__ bool block_reduce_publish(double (&v)[NV], double* partials, int stride,
                                                     unsigned int* ticket, unsigned int bid, unsigned int nblocks) {
    __shared__ double sm[NV][32];
    __shared__ int s_last;
    const int tid = threadIdx.x + blockDim.x * (threadIdx.y + blockDim.y * threadIdx.z);
    const int nthreads = blockDim.x * blockDim.y * blockDim.z;
    const int lane = tid & 31, wid = tid >> 5, nwarps = (nthreads + 31) >> 5;
#pragma unroll
    for (int i = 0; i < NV; ++i) {
        const double r = i >= NV - NMAX ? warp_max(v[i]) : warp_sum(v[i]);
        if (lane == 0) sm[i][wid] = r;
    }
    __syncthreads();
    if (wid == 0) {
#pragma unroll
        for (int i = 0; i < NV; ++i) {
            double r = lane < nwarps ? sm[i][lane] : (i >= NV - NMAX ? -1.0e300 : 0.0);
            r = i >= NV - NMAX ? warp_max(r) : warp_sum(r);
            if (lane == 0) partials[(size_t)i * stride + bid] = r;
        }
        if (lane == 0) {
            __threadfence();
            const unsigned int t = atomicAdd(ticket, 1u);
            s_last = (t == nblocks - 1u);
        }
    }
    __syncthreads();
    if (!s_last) return false;
    __threadfence();
    final_sum<NV, NMAX>(v, partials, stride, nblocks);
    if (tid == 0) *ticket = 0u;
    return tid == 0;
}

}  // namespace demons
