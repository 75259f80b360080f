// S7 / S8 of the demons hot path: the multi-scale pyramid of PAPER.md L123-125 ("both static image
// and moving images are down-sampled ... The final displacement vectors obtained at the coarse
// level are upsampled and serve as initial displacement vectors at a finer scale").
#include "kernels.h"

namespace demons {

namespace {

// O6: coarse(i,j,k) = mean of the 2x2x2 fine voxels {2i, min(2i+1, n-1)} x ...; n_c = ceil(n_f/2)
// (2x2x2 averaging per BASELINE.json config 3; odd tail counted twice, reading A12).
// blockIdx.z = pair * cd.nz + k (a batch of images in one launch).
__global__ void __launch_bounds__(256) k_restrict(const float* __restrict__ fine, float* __restrict__ coarse,
                                                  const Dims fd, const Dims cd, const size_t in_stride,
                                                  const size_t out_stride) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    const int j = blockIdx.y * blockDim.y + threadIdx.y;
    const int pair = blockIdx.z / cd.nz, k = blockIdx.z - pair * cd.nz;
    if (i >= cd.nx || j >= cd.ny) return;
    fine += (size_t)pair * in_stride;
    coarse += (size_t)pair * out_stride;
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
// One thread per coarse CELL (i..i+1, j..j+1, k..k+1), i in [-1, n_c - 1]: the up to 2x2x2 fine voxels
// x in {2i+1, 2i+2} x ... interpolate inside that one cell with the weights 1/4 (x = 2i+1) and 3/4
// (x = 2i+2), so the 8 coarse values of a component are loaded once for 8 outputs.  At the faces the
// clamp makes both cell corners the same voxel (i = -1 -> voxel 0, i = n_c - 1 -> voxel n_c - 1), which is
// exactly what clamping the coarse coordinate does.  Interpolation order x, y, z as in O2.
__global__ void __launch_bounds__(256) k_prolong(const float* __restrict__ uc, float* __restrict__ uf,
                                                 const Dims cd, const Dims fd) {
    const int i = (int)(blockIdx.x * blockDim.x + threadIdx.x) - 1;
    const int j = (int)(blockIdx.y * blockDim.y + threadIdx.y) - 1;
    const int b = blockIdx.z / (cd.nz + 1);  // blockIdx.z = pair * (cd.nz + 1) + (k + 1)
    const int k = (int)(blockIdx.z - b * (cd.nz + 1)) - 1;
    if (i >= cd.nx || j >= cd.ny) return;
    uc += (size_t)b * 3 * nvox(cd);
    uf += (size_t)b * 3 * nvox(fd);
    const int x0 = max(i, 0), x1 = min(i + 1, cd.nx - 1);
    const int y0 = max(j, 0), y1 = min(j + 1, cd.ny - 1);
    const int z0 = max(k, 0), z1 = min(k + 1, cd.nz - 1);
    const unsigned Nc = (unsigned)nvox(cd), Nf = (unsigned)nvox(fd);
    const unsigned o00 = (unsigned)((z0 * cd.ny + y0) * cd.nx), o10 = (unsigned)((z0 * cd.ny + y1) * cd.nx);
    const unsigned o01 = (unsigned)((z1 * cd.ny + y0) * cd.nx), o11 = (unsigned)((z1 * cd.ny + y1) * cd.nx);
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        const float* I = uc + c * Nc;
        const float c000 = __ldg(I + o00 + x0), c100 = __ldg(I + o00 + x1), c010 = __ldg(I + o10 + x0),
                    c110 = __ldg(I + o10 + x1), c001 = __ldg(I + o01 + x0), c101 = __ldg(I + o01 + x1),
                    c011 = __ldg(I + o11 + x0), c111 = __ldg(I + o11 + x1);
#pragma unroll
        for (int dz = 1; dz <= 2; ++dz) {
            const int z = 2 * k + dz;
            if (z < 0 || z >= fd.nz) continue;
            const float fz = dz == 1 ? 0.25f : 0.75f;
#pragma unroll
            for (int dy = 1; dy <= 2; ++dy) {
                const int y = 2 * j + dy;
                if (y < 0 || y >= fd.ny) continue;
                const float fy = dy == 1 ? 0.25f : 0.75f;
#pragma unroll
                for (int dx = 1; dx <= 2; ++dx) {
                    const int x = 2 * i + dx;
                    if (x < 0 || x >= fd.nx) continue;
                    const float fx = dx == 1 ? 0.25f : 0.75f;
                    const float a00 = lerpf(c000, c100, fx), a10 = lerpf(c010, c110, fx);
                    const float a01 = lerpf(c001, c101, fx), a11 = lerpf(c011, c111, fx);
                    const float b0 = lerpf(a00, a10, fy), b1 = lerpf(a01, a11, fy);
                    uf[c * Nf + (unsigned)((z * fd.ny + y) * fd.nx + x)] = 2.f * lerpf(b0, b1, fz);
                }
            }
        }
    }
}

}  // namespace

int launch_restrict(const Dims& fd, const float* in, size_t in_stride, float* out, size_t out_stride, int nb,
                    cudaStream_t st) {
    const Dims cd{(fd.nx + 1) / 2, (fd.ny + 1) / 2, (fd.nz + 1) / 2};
    if ((long long)cd.nz * nb > 65535) return -1;
    const dim3 block(64, 4);
    const dim3 grid((cd.nx + 63) / 64, (cd.ny + 3) / 4, cd.nz * nb);
    k_restrict<<<grid, block, 0, st>>>(in, out, fd, cd, in_stride, out_stride);
    return cudaPeekAtLastError() == cudaSuccess ? 1 : -1;
}

int launch_prolong(const Dims& cd, const float* uc, const Dims& fd, float* uf, int nb, cudaStream_t st) {
    if ((long long)(cd.nz + 1) * nb > 65535) return -1;
    const dim3 block(64, 4);
    const dim3 grid((cd.nx + 1 + 63) / 64, (cd.ny + 1 + 3) / 4, (cd.nz + 1) * nb);  // cells: i, j, k in [-1, n_c - 1]
    k_prolong<<<grid, block, 0, st>>>(uc, uf, cd, fd);
    return cudaPeekAtLastError() == cudaSuccess ? 1 : -1;
}

}  // namespace demons
