// S7 / S8 of the demons hot path: the multi-scale pyramid of PAPER.md L123-125 ("both static image
// and moving images are down-sampled ... The final displacement vectors obtained at the coarse
// level are upsampled and serve as initial displacement vectors at a finer scale").
#include "kernels.h"

namespace demons {

namespace {

// O6: coarse(i,j,k) = mean of the 2x2x2 fine voxels {2i, min(2i+1, n-1)} x ...; n_c = ceil(n_f/2)
// (2x2x2 averaging per BASELINE.json config 3; odd tail counted twice, reading A12).
__global__ void __launch_bounds__(256) k_restrict(const float* __restrict__ fine, float* __restrict__ coarse,
                                                  const Dims fd, const Dims cd) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    const int j = blockIdx.y * blockDim.y + threadIdx.y;
    const int k = blockIdx.z;
    if (i >= cd.nx || j >= cd.ny) return;
    const int x0 = 2 * i, x1 = min(2 * i + 1, fd.nx - 1);
    const int y0 = 2 * j, y1 = min(2 * j + 1, fd.ny - 1);
    const int z0 = 2 * k, z1 = min(2 * k + 1, fd.nz - 1);
    const size_t plane = (size_t)fd.nx * fd.ny;
    const float* p00 = fine + z0 * plane + (size_t)y0 * fd.nx;
    const float* p10 = fine + z0 * plane + (size_t)y1 * fd.nx;
    const float* p01 = fine + z1 * plane + (size_t)y0 * fd.nx;
    const float* p11 = fine + z1 * plane + (size_t)y1 * fd.nx;
    const float a = __ldg(p00 + x0) + __ldg(p00 + x1) + __ldg(p10 + x0) + __ldg(p10 + x1);
    const float b = __ldg(p01 + x0) + __ldg(p01 + x1) + __ldg(p11 + x0) + __ldg(p11 + x1);
    coarse[((size_t)k * cd.ny + j) * cd.nx + i] = 0.125f * (a + b);
}

// O7: fine voxel x sits at coarse coordinate (x - 0.5)/2, clamped to [0, n_c - 1];
// u_f = 2 * trilinear(u_c) per component (factor 2: PAPER.md L123-125; alignment: reading A12).
__device__ __forceinline__ void coarse_axis(int x, int nc, int& i0, int& i1, float& f) {
    float p = 0.5f * ((float)x - 0.5f);
    p = fminf(fmaxf(p, 0.f), (float)(nc - 1));
    const float fl = floorf(p);
    i0 = (int)fl;
    f = p - fl;
    i1 = min(i0 + 1, nc - 1);
}

__global__ void __launch_bounds__(256) k_prolong(const float* __restrict__ uc, float* __restrict__ uf,
                                                 const Dims cd, const Dims fd) {
    const int x = blockIdx.x * blockDim.x + threadIdx.x;
    const int y = blockIdx.y * blockDim.y + threadIdx.y;
    const int z = blockIdx.z;
    if (x >= fd.nx || y >= fd.ny) return;
    int x0, x1, y0, y1, z0, z1;
    float fx, fy, fz;
    coarse_axis(x, cd.nx, x0, x1, fx);
    coarse_axis(y, cd.ny, y0, y1, fy);
    coarse_axis(z, cd.nz, z0, z1, fz);
    const size_t Nc = nvox(cd), Nf = nvox(fd);
    const size_t o00 = ((size_t)z0 * cd.ny + y0) * cd.nx, o10 = ((size_t)z0 * cd.ny + y1) * cd.nx;
    const size_t o01 = ((size_t)z1 * cd.ny + y0) * cd.nx, o11 = ((size_t)z1 * cd.ny + y1) * cd.nx;
    const size_t of = ((size_t)z * fd.ny + y) * fd.nx + x;
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        const float* I = uc + c * Nc;
        const float a00 = lerpf(__ldg(I + o00 + x0), __ldg(I + o00 + x1), fx);
        const float a10 = lerpf(__ldg(I + o10 + x0), __ldg(I + o10 + x1), fx);
        const float a01 = lerpf(__ldg(I + o01 + x0), __ldg(I + o01 + x1), fx);
        const float a11 = lerpf(__ldg(I + o11 + x0), __ldg(I + o11 + x1), fx);
        const float b0 = lerpf(a00, a10, fy), b1 = lerpf(a01, a11, fy);
        uf[c * Nf + of] = 2.f * lerpf(b0, b1, fz);
    }
}

}  // namespace

int launch_restrict(const Dims& fd, const float* in, float* out, cudaStream_t st) {
    const Dims cd{(fd.nx + 1) / 2, (fd.ny + 1) / 2, (fd.nz + 1) / 2};
    const dim3 block(64, 4);
    const dim3 grid((cd.nx + 63) / 64, (cd.ny + 3) / 4, cd.nz);
    k_restrict<<<grid, block, 0, st>>>(in, out, fd, cd);
    return cudaPeekAtLastError() == cudaSuccess ? 1 : -1;
}

int launch_prolong(const Dims& cd, const float* uc, const Dims& fd, float* uf, cudaStream_t st) {
    const dim3 block(128, 2);
    const dim3 grid((fd.nx + 127) / 128, (fd.ny + 1) / 2, fd.nz);
    k_prolong<<<grid, block, 0, st>>>(uc, uf, cd, fd);
    return cudaPeekAtLastError() == cudaSuccess ? 1 : -1;
}

}  // namespace demons
