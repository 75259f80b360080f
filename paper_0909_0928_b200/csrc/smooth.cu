// S5 of the demons hot path: separable 3D Gaussian smoothing of the displacement field
// ("Gaussian filter to smooth the displacement field", L175 "separable ... we can
// perform the convolution in the x, y, and z directions independently"), radius R = ceil(3 sigma),
// normalised taps, clamped borders (reading A9).
//
// This file holds the separable fallback (any radius, any dims, any alignment): one launch per
// axis.  The TMA-fed single-pass kernel for the common case lives in smooth_tma.cu.
#include "kernels.h"

namespace demons {

int launch_smooth_tma(const SmoothArgs& a, cudaStream_t st);  // smooth_tma.cu; 0 = not applicable

namespace {

struct Taps {
    float w[33];
};

// out(i) = sum_{k=-R..R} w_|k| in(clamp(i + k)) along AXIS; one thread per element, threads span x
// so every tap is a coalesced row access (the strided y/z neighbours come from L1/L2).
// blockIdx.z = m * nz + z: volume m of the launch lives at in + m * in_stride and goes to out + m * out_stride
// (all components of all pairs in the x pass; one component of every pair in the y and z passes).
template <int AXIS>
__global__ void __launch_bounds__(256) k_smooth_axis(const float* __restrict__ in, const size_t in_stride,
                                                     float* __restrict__ out, const size_t out_stride, const Dims d,
                                                     const int R, const Taps t, const Control* __restrict__ ctl,
                                                     const int vols_per_pair) {
    const int m = blockIdx.z / d.nz, z = blockIdx.z - m * d.nz;
    if (ctl != nullptr && *reinterpret_cast<const volatile int*>(&ctl[m / vols_per_pair].stop_smooth) != 0) return;
    const int x = blockIdx.x * blockDim.x + threadIdx.x;
    const int y = blockIdx.y * blockDim.y + threadIdx.y;
    if (x >= d.nx || y >= d.ny) return;
    const size_t plane = (size_t)d.nx * d.ny;
    const float* src = in + (size_t)m * in_stride;
    const int n = AXIS == 0 ? d.nx : (AXIS == 1 ? d.ny : d.nz);
    const int c = AXIS == 0 ? x : (AXIS == 1 ? y : z);
    const size_t stride = AXIS == 0 ? 1 : (AXIS == 1 ? (size_t)d.nx : plane);
    const size_t base = (size_t)z * plane + (size_t)y * d.nx + x - (size_t)c * stride;
    float acc = t.w[0] * __ldg(src + base + (size_t)c * stride);
    for (int k = 1; k <= R; ++k) {
        const float a = __ldg(src + base + (size_t)max(c - k, 0) * stride);
        const float b = __ldg(src + base + (size_t)min(c + k, n - 1) * stride);
        acc = fmaf(t.w[k], a + b, acc);
    }
    out[(size_t)m * out_stride + (size_t)z * plane + (size_t)y * d.nx + x] = acc;
}

}  // namespace

int launch_smooth(const SmoothArgs& a, cudaStream_t st) {
    if (!a.force_generic) {
        const int n = launch_smooth_tma(a, st);
        if (n != 0) return n;
    }
    const int cpp = a.comps_per_pair > 0 ? a.comps_per_pair : a.ncomp;
    Taps t;
    for (int k = 0; k < 33; ++k) t.w[k] = k <= a.R ? a.w[k] : 0.f;
    const dim3 block(128, 2);
    const size_t N = nvox(a.d);
    const int pairs = a.ncomp / cpp;
    if (a.ncomp % cpp != 0 || (long long)a.d.nz * a.ncomp > 65535) return -1;
    int launches = 0;
    // x for all components of all pairs at once (in -> out); then, component by component of every pair,
    // y (out -> tmp, [pairs][N]) and z (tmp -> out)
    {
        const dim3 grid((a.d.nx + 127) / 128, (a.d.ny + 1) / 2, (unsigned)(a.d.nz * a.ncomp));
        k_smooth_axis<0><<<grid, block, 0, st>>>(a.in, N, a.out, N, a.d, a.R, t, a.ctl, cpp);
        ++launches;
    }
    for (int c = 0; c < cpp; ++c) {
        const dim3 grid((a.d.nx + 127) / 128, (a.d.ny + 1) / 2, (unsigned)(a.d.nz * pairs));
        k_smooth_axis<1><<<grid, block, 0, st>>>(a.out + c * N, (size_t)cpp * N, a.tmp, N, a.d, a.R, t, a.ctl, 1);
        k_smooth_axis<2><<<grid, block, 0, st>>>(a.tmp, N, a.out + c * N, (size_t)cpp * N, a.d, a.R, t, a.ctl, 1);
        launches += 2;
    }
    if (cudaPeekAtLastError() != cudaSuccess) return -1;
    return launches;
}

}  // namespace demons
