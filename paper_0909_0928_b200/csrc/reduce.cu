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
    if (block_reduce_publish<1>(acc, partials, stride, ticket)) out[0] = acc[0];
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
    if (block_reduce_publish<2, 1>(acc, partials, stride, ticket)) {
        out[0] = acc[0] / (double)N;
        out[1] = acc[1];
    }
}

int reduce_blocks(const Dims& d, int stride) {
    const size_t N = nvox(d);
    size_t b = (N + RB - 1) / RB;
    const size_t cap = 148 * 8;
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

}  // namespace demons
