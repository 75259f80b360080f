// S5 of the demons hot path: separable 3D Gaussian smoothing of the displacement field
// ("Gaussian filter to smooth the displacement field", L175 "separable ... we can
// perform the convolution in the x, y, and z directions independently"), radius R = ceil(3 sigma),
// normalised taps, clamped borders (reading A9).
//
// This file holds the separable fallback (any radius, any dims, any alignment): one launch per
// axis.  The fused single-pass kernel for the common case lives in smooth_fused.cu.
#include "kernels.h"

namespace demons {

int launch_smooth_tma(const SmoothArgs& a, cudaStream_t st);    // smooth_tma.cu; 0 = not applicable
int launch_smooth_fused(const SmoothArgs& a, cudaStream_t st);  // smooth_fused.cu; 0 = not applicable

namespace {

struct Taps {
    float w[33];
};

// out(i) = sum_{k=-R..R} w_|k| in(clamp(i + k)) along AXIS; one thread per element, threads span x
// so every tap is a coalesced row access (the strided y/z neighbours come from L1/L2).
template <int AXIS>
__global__ void __launch_bounds__(256) k_smooth_axis(const float* __restrict__ in, float* __restrict__ out,
                                                     const Dims d, const int R, const Taps t,
                                                     const int* __restrict__ skip) {
    if (skip != nullptr && *reinterpret_cast<const volatile int*>(skip) != 0) return;
    const int x = blockIdx.x * blockDim.x + threadIdx.x;
    const int y = blockIdx.y * blockDim.y + threadIdx.y;
    if (x >= d.nx || y >= d.ny) return;
    const size_t plane = (size_t)d.nx * d.ny;
    // blockIdx.z runs over (component, z)
    const int z = blockIdx.z % d.nz;
    const size_t comp_off = (size_t)(blockIdx.z / d.nz) * plane * d.nz;
    const float* src = in + comp_off;
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
    out[comp_off + (size_t)z * plane + (size_t)y * d.nx + x] = acc;
}

}  // namespace

int launch_smooth(const SmoothArgs& a, cudaStream_t st) {
    if (!a.force_generic) {
        int n = a.no_tma ? 0 : launch_smooth_tma(a, st);
        if (n != 0) return n;
        n = launch_smooth_fused(a, st);
        if (n != 0) return n;
    }
    Taps t;
    for (int k = 0; k < 33; ++k) t.w[k] = k <= a.R ? a.w[k] : 0.f;
    const dim3 block(128, 2);
    const size_t N = nvox(a.d);
    int launches = 0;
    // x for all components at once (in -> out), then per component y (out -> tmp), z (tmp -> out)
    {
        const long long gz = (long long)a.d.nz * a.ncomp;
        if (gz > 65535) return -1;
        const dim3 grid((a.d.nx + 127) / 128, (a.d.ny + 1) / 2, (unsigned)gz);
        k_smooth_axis<0><<<grid, block, 0, st>>>(a.in, a.out, a.d, a.R, t, a.skip);
        ++launches;
    }
    for (int c = 0; c < a.ncomp; ++c) {
        const dim3 grid((a.d.nx + 127) / 128, (a.d.ny + 1) / 2, a.d.nz);
        k_smooth_axis<1><<<grid, block, 0, st>>>(a.out + c * N, a.tmp, a.d, a.R, t, a.skip);
        k_smooth_axis<2><<<grid, block, 0, st>>>(a.tmp, a.out + c * N, a.d, a.R, t, a.skip);
        launches += 2;
    }
    if (cudaPeekAtLastError() != cudaSuccess) return -1;
    return launches;
}

}  // namespace demons
