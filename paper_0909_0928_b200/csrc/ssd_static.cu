// demons_ssd_static: the SSD of demons_ssd for callers who cannot hand the library any device memory.
//
// Every other compute entry point needs a workspace, and a workspace is a device allocation somebody has to make.
// Some users of this library are not in a position to make one: a quality-assurance hook that a planning system calls
// with device pointers to two CT volumes and a field and that must not change the process's memory footprint; a plug-in
// running under a host application that owns the whole device memory budget through its own pool and forbids
// cudaMalloc in plug-ins; code inside a time-critical loop, where cudaMalloc / cudaFree stall every stream of the
// device while the allocator runs.  Such a caller can still ask "how well does this field match these two images?"
// (PAPER.md L145 / L234: the similarity the stopping-rule study looks at; reading O8), because the only scratch that
// sum needs -- one double per thread block and a counter -- fits in a small array that is part of the library image.
//
// The array below is that scratch.  It lives in the module's global memory on every device that loads libdemons.so
// (SSD_STATIC_BYTES per device, held until the process exits).  Host code may not pass the symbol `g_ssd_scratch` to a
// kernel: on the host that name is only a handle.  The device address is asked for once per device with
// cudaGetSymbolAddress while that device is current, cached, and handed to the kernel as an ordinary pointer.
#include "../../include/demons.h"

#include <cstdarg>
#include <cstdio>
#include <mutex>

#include "kernels.h"

namespace demons {

namespace {

constexpr int SB = 256;                                    // threads per block
constexpr int SSD_STATIC_PER_THREAD = 16;                  // voxels per thread
constexpr int SSD_STATIC_TILE = SB * SSD_STATIC_PER_THREAD;  // voxels per block: 4096
constexpr int SSD_STATIC_SLOTS = (int)(DEMONS_SSD_STATIC_MAX_VOXELS / SSD_STATIC_TILE);  // block partials: 16384
constexpr size_t SSD_STATIC_BYTES = (size_t)SSD_STATIC_SLOTS * sizeof(double) + 256;     // + the counter's line
static_assert((size_t)SSD_STATIC_SLOTS * SSD_STATIC_TILE == DEMONS_SSD_STATIC_MAX_VOXELS, "limit = slots x tile");

// [SSD_STATIC_SLOTS] doubles (block partials), then one unsigned int (arrival counter) on a line of its own.
static __device__ __align__(256) unsigned char g_ssd_scratch[SSD_STATIC_BYTES];

// Same per-voxel arithmetic as k_ssd (reduce.cu): software trilinear of M (and of S for the two-field form), fp32
// difference, squared in fp32, summed in double.  What differs is the partition: block b owns the 4096 consecutive
// voxels [b * 4096, (b + 1) * 4096) whatever the GPU, so the number of partials follows from the volume alone (and is
// what the size limit bounds), and the fixed-order final sum gives the same bits on every device.
__global__ void __launch_bounds__(SB) k_ssd_static(const float* __restrict__ S, const float* __restrict__ M,
                                                   const float* __restrict__ u, const float* __restrict__ ub,
                                                   const Dims d, double* __restrict__ out, double* partials,
                                                   unsigned int* ticket) {
    const size_t N = nvox(d);
    const size_t plane = (size_t)d.nx * d.ny;
    const size_t base = (size_t)blockIdx.x * SSD_STATIC_TILE + threadIdx.x;
    double acc[1] = {0.0};
#pragma unroll 4
    for (int k = 0; k < SSD_STATIC_PER_THREAD; ++k) {
        const size_t i = base + (size_t)k * SB;
        if (i >= N) break;
        const int z = (int)(i / plane);
        const int r = (int)(i - (size_t)z * plane);
        const int y = r / d.nx, x = r - y * d.nx;
        const float mw = trilinear(M, d, x, y, z, u[i], u[N + i], u[2 * N + i]);
        const float s = ub != nullptr ? trilinear(S, d, x, y, z, ub[i], ub[N + i], ub[2 * N + i]) : __ldg(S + i);
        const float dd = mw - s;
        acc[0] += (double)(dd * dd);
    }
    if (block_reduce_publish<1>(acc, partials, SSD_STATIC_SLOTS, ticket, blockIdx.x, gridDim.x)) out[0] = acc[0];
}

// Device address of g_ssd_scratch per device ordinal; filled on the first call made with that device current.
constexpr int MAX_DEVICES = 64;
std::mutex g_setup_mutex;
unsigned char* g_scratch_addr[MAX_DEVICES] = {};

int fail_static(int code, const char* fmt, ...) {
    char buf[512];
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(buf, sizeof buf, fmt, ap);
    va_end(ap);
    set_last_error(buf);
    return code;
}

}  // namespace

}  // namespace demons

using namespace demons;

extern "C" int demons_ssd_static(const int dims[3], const float* d_static, const float* d_moving, const float* d_u,
                                 const float* d_ub, double* d_out, void* stream) {
    if (!dims) return fail_static(DEMONS_E_ARG, "dims is NULL");
    for (int c = 0; c < 3; ++c)
        if (dims[c] < 1 || dims[c] > 16384) return fail_static(DEMONS_E_ARG, "bad dims");
    if (!d_static || !d_moving || !d_u || !d_out) return fail_static(DEMONS_E_ARG, "NULL pointer");
    const Dims d{dims[0], dims[1], dims[2]};
    const size_t N = nvox(d);
    if (N > (size_t)DEMONS_SSD_STATIC_MAX_VOXELS)
        return fail_static(DEMONS_E_UNSUPPORTED,
                           "demons_ssd_static: %d x %d x %d = %zu voxels is more than the built-in scratch array serves "
                           "(DEMONS_SSD_STATIC_MAX_VOXELS = %zu); use demons_ssd with a workspace",
                           d.nx, d.ny, d.nz, N, (size_t)DEMONS_SSD_STATIC_MAX_VOXELS);

    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return fail_static(DEMONS_E_CUDA, "cudaGetDevice failed: %s", cudaGetErrorString(e));
    if (dev < 0 || dev >= MAX_DEVICES) return fail_static(DEMONS_E_UNSUPPORTED, "device ordinal %d out of range", dev);
    unsigned char* scratch = nullptr;
    {
        // Set-up, once per device, with that device current: turn the host-side handle into the device address.
        std::lock_guard<std::mutex> lock(g_setup_mutex);
        if (!g_scratch_addr[dev]) {
            void* p = nullptr;
            e = cudaGetSymbolAddress(&p, g_ssd_scratch);
            if (e != cudaSuccess || !p)
                return fail_static(DEMONS_E_CUDA, "cudaGetSymbolAddress(g_ssd_scratch) failed on device %d: %s", dev,
                                   cudaGetErrorString(e));
            g_scratch_addr[dev] = static_cast<unsigned char*>(p);
        }
        scratch = g_scratch_addr[dev];
    }
    double* partials = reinterpret_cast<double*>(scratch);
    unsigned int* ticket = reinterpret_cast<unsigned int*>(scratch + (size_t)SSD_STATIC_SLOTS * sizeof(double));

    cudaStream_t st = static_cast<cudaStream_t>(stream);
    // The array keeps whatever the last call left.  The partials are all overwritten before they are read; the arrival
    // counter is the one thing that must start at zero, also after a call that died half-way.
    e = cudaMemsetAsync(ticket, 0, sizeof(unsigned int), st);
    if (e != cudaSuccess) return fail_static(DEMONS_E_CUDA, "cudaMemsetAsync failed: %s", cudaGetErrorString(e));
    const unsigned int blocks = (unsigned int)((N + SSD_STATIC_TILE - 1) / SSD_STATIC_TILE);
    k_ssd_static<<<blocks, SB, 0, st>>>(d_static, d_moving, d_u, d_ub, d, d_out, partials, ticket);
    e = cudaPeekAtLastError();
    if (e != cudaSuccess) {
        cudaGetLastError();
        return fail_static(DEMONS_E_CUDA, "ssd_static launch failed: %s", cudaGetErrorString(e));
    }
    return DEMONS_OK;
}
