// Evaluation reductions: the final SSD of O8 (one extra warp after the last iteration) and the
// inverse-consistency error of BASELINE.json config 4, e(x) = |u_f(x) + u_b(x + u_f(x))|_2.
// Warp-shuffle block reductions in double, fixed-order final sum (deterministic).
#include "kernels.h"

namespace demons {

namespace {

constexpr int RB = 256;

__global__ void __launch_bounds__(RB) k_ssd(const float* __restrict__ S, const float* __restrict__ M,
                                            const float* __restrict__ u, const float* __restrict__ ub,
                                            const Dims d, double* out, double* partials, int stride,
                                            unsigned int* ticket) {
    const size_t N = nvox(d);
    const size_t plane = (size_t)d.nx * d.ny;
    double acc[1] = {0.0};
    for (size_t i = (size_t)blockIdx.x * RB + threadIdx.x; i < N; i += (size_t)gridDim.x * RB) {
        const int z = (int)(i / plane);
        const int r = (int)(i - (size_t)z * plane);
        const int y = r / d.nx, x = r - y * d.nx;
        const float mw = trilinear(M, d, x, y, z, u[i], u[N + i], u[2 * N + i]);
        const float s = ub != nullptr ? trilinear(S, d, x, y, z, ub[i], ub[N + i], ub[2 * N + i]) : __ldg(S + i);
        const float dd = mw - s;
        acc[0] += (double)(dd * dd);
    }
    if (block_reduce_publish<1>(acc, partials, stride, ticket, blockIdx.x, gridDim.x)) out[0] = acc[0];
}

__global__ void __launch_bounds__(RB) k_ic_error(const float* __restrict__ uf, const float* __restrict__ ub,
                                                 const Dims d, double* out, double* partials, int stride,
                                                 unsigned int* ticket) {
    const size_t N = nvox(d);
    const size_t plane = (size_t)d.nx * d.ny;
    double acc[2] = {0.0, 0.0};  // sum e, max e
    for (size_t i = (size_t)blockIdx.x * RB + threadIdx.x; i < N; i += (size_t)gridDim.x * RB) {
        const int z = (int)(i / plane);
        const int r = (int)(i - (size_t)z * plane);
        const int y = r / d.nx, x = r - y * d.nx;
        const float ax = uf[i], ay = uf[N + i], az = uf[2 * N + i];
        const float ex = ax + trilinear(ub, d, x, y, z, ax, ay, az);
        const float ey = ay + trilinear(ub + N, d, x, y, z, ax, ay, az);
        const float ez = az + trilinear(ub + 2 * N, d, x, y, z, ax, ay, az);
        const double e = (double)sqrtf(fmaf(ex, ex, fmaf(ey, ey, ez * ez)));
        acc[0] += e;
        acc[1] = fmax(acc[1], e);
    }
    if (block_reduce_publish<2, 1>(acc, partials, stride, ticket, blockIdx.x, gridDim.x)) {
        out[0] = acc[0] / (double)N;
        out[1] = acc[1];
    }
}

// Correlation coefficient of a = warp(M,u) and b = S (variant 5: warp(S,ub)), PAPER.md L234 (the
// similarity measure the paper compares its relative-norm rule with).  One pass: the five raw sums
// in double (products of fp32 values are exact in double; with |I| ~ 1e3 and N ~ 1e7 the
// cancellation in  sum ab - sum a sum b / N  leaves ~1e-10 relative), closed in the last block.
__global__ void __launch_bounds__(RB) k_cc(const float* __restrict__ S, const float* __restrict__ M,
                                           const float* __restrict__ u, const float* __restrict__ ub,
                                           const Dims d, double* out, double* partials, int stride,
                                           unsigned int* ticket) {
    const size_t N = nvox(d);
    const size_t plane = (size_t)d.nx * d.ny;
    double acc[5] = {0.0, 0.0, 0.0, 0.0, 0.0};  // sum a, sum b, sum aa, sum bb, sum ab
    for (size_t i = (size_t)blockIdx.x * RB + threadIdx.x; i < N; i += (size_t)gridDim.x * RB) {
        const int z = (int)(i / plane);
        const int r = (int)(i - (size_t)z * plane);
        const int y = r / d.nx, x = r - y * d.nx;
        const double a = (double)trilinear(M, d, x, y, z, u[i], u[N + i], u[2 * N + i]);
        const double b =
            (double)(ub != nullptr ? trilinear(S, d, x, y, z, ub[i], ub[N + i], ub[2 * N + i]) : __ldg(S + i));
        acc[0] += a;
        acc[1] += b;
        acc[2] += a * a;
        acc[3] += b * b;
        acc[4] += a * b;
    }
    if (block_reduce_publish<5>(acc, partials, stride, ticket, blockIdx.x, gridDim.x)) {
        const double n = (double)N;
        const double saa = acc[2] - acc[0] * acc[0] / n, sbb = acc[3] - acc[1] * acc[1] / n;
        const double sab = acc[4] - acc[0] * acc[1] / n;
        // a constant image has variance 0 up to the rounding of the sums: 1e-12 of the raw moment
        const bool flat = saa <= 1e-12 * acc[2] || sbb <= 1e-12 * acc[3];
        out[0] = flat ? 0.0 : sab / sqrt(saa * sbb);
    }
}

// PAPER.md L222 (Sec. 3.2): three-dimensional Euclidean error at feature points.  One thread per
// point: the field sampled trilinearly (clamped) at an arbitrary position, minus the expected
// displacement, scaled to mm.
__global__ void __launch_bounds__(RB) k_point_error(const float* __restrict__ u, const Dims d, float sx, float sy,
                                                    float sz, int n, const float* __restrict__ pts,
                                                    const float* __restrict__ expect, double* __restrict__ err) {
    const int i = blockIdx.x * RB + threadIdx.x;
    if (i >= n) return;
    const size_t N = nvox(d);
    const float px = pts[3 * i], py = pts[3 * i + 1], pz = pts[3 * i + 2];
    // trilinear() takes an integer voxel plus a displacement: split the position that way
    const int x = (int)floorf(fminf(fmaxf(px, -1.0e6f), 1.0e6f)), y = (int)floorf(fminf(fmaxf(py, -1.0e6f), 1.0e6f)),
              z = (int)floorf(fminf(fmaxf(pz, -1.0e6f), 1.0e6f));
    const float fx = fminf(fmaxf(px, -1.0e6f), 1.0e6f) - (float)x, fy = fminf(fmaxf(py, -1.0e6f), 1.0e6f) - (float)y,
                fz = fminf(fmaxf(pz, -1.0e6f), 1.0e6f) - (float)z;
    const float ex = (trilinear(u, d, x, y, z, fx, fy, fz) - expect[3 * i]) * sx;
    const float ey = (trilinear(u + N, d, x, y, z, fx, fy, fz) - expect[3 * i + 1]) * sy;
    const float ez = (trilinear(u + 2 * N, d, x, y, z, fx, fy, fz) - expect[3 * i + 2]) * sz;
    err[i] = sqrt((double)ex * ex + (double)ey * ey + (double)ez * ez);
}

int reduce_blocks(const Dims& d, int stride) {
    const size_t N = nvox(d);
    size_t b = (N + RB - 1) / RB;
    const size_t cap = (size_t)sm_count() * 8;
    if (b > cap) b = cap;
    if (b > (size_t)stride) b = stride;
    return b < 1 ? 1 : (int)b;
}

}  // namespace

int launch_ssd(const Dims& d, const float* S, const float* M, const float* u, const float* ub, double* out,
               const ReduceScratch& rs, cudaStream_t st) {
    k_ssd<<<reduce_blocks(d, rs.stride), RB, 0, st>>>(S, M, u, ub, d, out, rs.partials, rs.stride, rs.ticket);
    return cudaPeekAtLastError() == cudaSuccess ? 1 : -1;
}

int launch_ic_error(const Dims& d, const float* uf, const float* ub, double* out, const ReduceScratch& rs,
                    cudaStream_t st) {
    k_ic_error<<<reduce_blocks(d, rs.stride), RB, 0, st>>>(uf, ub, d, out, rs.partials, rs.stride, rs.ticket);
    return cudaPeekAtLastError() == cudaSuccess ? 1 : -1;
}

int launch_cc(const Dims& d, const float* S, const float* M, const float* u, const float* ub, double* out,
              const ReduceScratch& rs, cudaStream_t st) {
    k_cc<<<reduce_blocks(d, rs.stride), RB, 0, st>>>(S, M, u, ub, d, out, rs.partials, rs.stride, rs.ticket);
    return cudaPeekAtLastError() == cudaSuccess ? 1 : -1;
}

int launch_point_error(const Dims& d, const float spacing[3], const float* u, int n, const float* points,
                       const float* expect, double* err, cudaStream_t st) {
    k_point_error<<<(n + RB - 1) / RB, RB, 0, st>>>(u, d, spacing[0], spacing[1], spacing[2], n, points, expect, err);
    return cudaPeekAtLastError() == cudaSuccess ? 1 : -1;
}

}  // namespace demons
