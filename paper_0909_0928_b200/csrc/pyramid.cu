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

// The same for fine rows that are a whole number of float4s: a thread averages 4 x 2 x 2 fine voxels into TWO coarse
// voxels (four 128-bit loads, one 64-bit store); the sums are taken in the order of k_restrict, hence the same bits.
__global__ void __launch_bounds__(256) k_restrict_v4(const float* __restrict__ fine, float* __restrict__ coarse,
                                                     const Dims fd, const Dims cd, const size_t in_stride,
                                                     const size_t out_stride) {
    const int i2 = blockIdx.x * blockDim.x + threadIdx.x;  // pair of coarse voxels (2 i2, 2 i2 + 1)
    const int j = blockIdx.y * blockDim.y + threadIdx.y;
    const int pair = blockIdx.z / cd.nz, k = blockIdx.z - pair * cd.nz;
    if (4 * i2 >= fd.nx || j >= cd.ny) return;
    fine += (size_t)pair * in_stride;
    coarse += (size_t)pair * out_stride;
    const int y0 = 2 * j, y1 = min(2 * j + 1, fd.ny - 1);
    const int z0 = 2 * k, z1 = min(2 * k + 1, fd.nz - 1);
    const size_t plane = (size_t)fd.nx * fd.ny;
    const float4 p00 = __ldg(reinterpret_cast<const float4*>(fine + z0 * plane + (size_t)y0 * fd.nx + 4 * i2));
    const float4 p10 = __ldg(reinterpret_cast<const float4*>(fine + z0 * plane + (size_t)y1 * fd.nx + 4 * i2));
    const float4 p01 = __ldg(reinterpret_cast<const float4*>(fine + z1 * plane + (size_t)y0 * fd.nx + 4 * i2));
    const float4 p11 = __ldg(reinterpret_cast<const float4*>(fine + z1 * plane + (size_t)y1 * fd.nx + 4 * i2));
    const float a0 = p00.x + p00.y + p10.x + p10.y, b0 = p01.x + p01.y + p11.x + p11.y;
    const float a1 = p00.z + p00.w + p10.z + p10.w, b1 = p01.z + p01.w + p11.z + p11.w;
    *reinterpret_cast<float2*>(coarse + ((size_t)k * cd.ny + j) * cd.nx + 2 * i2) = make_float2(0.125f * (a0 + b0), 0.125f * (a1 + b1));
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

// The same prolongation for fine rows that are a whole number of float4s: one thread per (4 fine voxels along x) x
// (2 fine rows) x (2 fine planes) of a coarse cell row pair / plane pair.  Fine x = 4i + e sits in the coarse cells
// (2i-1, 2i) [f = 3/4], (2i, 2i+1) [1/4], (2i, 2i+1) [3/4], (2i+1, 2i+2) [1/4]: four coarse values per row feed four
// outputs, the stores are 128-bit and coalesced (the scalar form stores with stride 2).  Same arithmetic per output
// as k_prolong (x, then y, then z; lerpf), hence the same bits.
__global__ void __launch_bounds__(256) k_prolong_v4(const float* __restrict__ uc, float* __restrict__ uf,
                                                    const Dims cd, const Dims fd) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;               // fine float4 index along x
    const int j = (int)(blockIdx.y * blockDim.y + threadIdx.y) - 1;    // coarse cell row pair (j, j+1)
    const int b = blockIdx.z / (cd.nz + 1);
    const int k = (int)(blockIdx.z - b * (cd.nz + 1)) - 1;             // coarse plane pair (k, k+1)
    if (4 * i >= fd.nx || j >= cd.ny) return;
    uc += (size_t)b * 3 * nvox(cd);
    uf += (size_t)b * 3 * nvox(fd);
    const int y0 = max(j, 0), y1 = min(j + 1, cd.ny - 1);
    const int z0 = max(k, 0), z1 = min(k + 1, cd.nz - 1);
    int xc[4];
#pragma unroll
    for (int t = 0; t < 4; ++t) xc[t] = min(max(2 * i - 1 + t, 0), cd.nx - 1);
    const unsigned Nc = (unsigned)nvox(cd), Nf = (unsigned)nvox(fd);
    const unsigned row[4] = {(unsigned)((z0 * cd.ny + y0) * cd.nx), (unsigned)((z0 * cd.ny + y1) * cd.nx),
                             (unsigned)((z1 * cd.ny + y0) * cd.nx), (unsigned)((z1 * cd.ny + y1) * cd.nx)};
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        const float* I = uc + c * Nc;
        float a[4][4];  // [row: (z0,y0), (z0,y1), (z1,y0), (z1,y1)][e]: interpolated along x
#pragma unroll
        for (int r = 0; r < 4; ++r) {
            const float c0 = __ldg(I + row[r] + xc[0]), c1 = __ldg(I + row[r] + xc[1]), c2 = __ldg(I + row[r] + xc[2]),
                        c3 = __ldg(I + row[r] + xc[3]);
            a[r][0] = lerpf(c0, c1, 0.75f);
            a[r][1] = lerpf(c1, c2, 0.25f);
            a[r][2] = lerpf(c1, c2, 0.75f);
            a[r][3] = lerpf(c2, c3, 0.25f);
        }
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
                float o[4];
#pragma unroll
                for (int e = 0; e < 4; ++e) {
                    const float b0 = lerpf(a[0][e], a[1][e], fy), b1 = lerpf(a[2][e], a[3][e], fy);
                    o[e] = 2.f * lerpf(b0, b1, fz);
                }
                *reinterpret_cast<float4*>(uf + c * Nf + (unsigned)((z * fd.ny + y) * fd.nx + 4 * i)) =
                    make_float4(o[0], o[1], o[2], o[3]);
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
    if (fd.nx % 4 == 0 && (reinterpret_cast<uintptr_t>(in) & 15u) == 0 && (reinterpret_cast<uintptr_t>(out) & 7u) == 0 &&
        (nb == 1 || (in_stride % 4 == 0 && out_stride % 2 == 0))) {
        const dim3 grid((fd.nx / 4 + 63) / 64, (cd.ny + 3) / 4, cd.nz * nb);
        k_restrict_v4<<<grid, block, 0, st>>>(in, out, fd, cd, in_stride, out_stride);
        return cudaPeekAtLastError() == cudaSuccess ? 1 : -1;
    }
    const dim3 grid((cd.nx + 63) / 64, (cd.ny + 3) / 4, cd.nz * nb);
    k_restrict<<<grid, block, 0, st>>>(in, out, fd, cd, in_stride, out_stride);
    return cudaPeekAtLastError() == cudaSuccess ? 1 : -1;
}

int launch_prolong(const Dims& cd, const float* uc, const Dims& fd, float* uf, int nb, cudaStream_t st) {
    if ((long long)(cd.nz + 1) * nb > 65535) return -1;
    const dim3 block(64, 4);
    if (fd.nx % 4 == 0 && (reinterpret_cast<uintptr_t>(uf) & 15u) == 0) {  // 128-bit rows (every pair: 3 N_f floats apart)
        const dim3 grid((fd.nx / 4 + 63) / 64, (cd.ny + 1 + 3) / 4, (cd.nz + 1) * nb);
        k_prolong_v4<<<grid, block, 0, st>>>(uc, uf, cd, fd);
        return cudaPeekAtLastError() == cudaSuccess ? 1 : -1;
    }
    const dim3 grid((cd.nx + 1 + 63) / 64, (cd.ny + 1 + 3) / 4, (cd.nz + 1) * nb);  // cells: i, j, k in [-1, n_c - 1]
    k_prolong<<<grid, block, 0, st>>>(uc, uf, cd, fd);
    return cudaPeekAtLastError() == cudaSuccess ? 1 : -1;
}

}  // namespace demons
