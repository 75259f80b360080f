// S5, fast path: the whole separable Gaussian (reading A9) in ONE pass over the
// field -- 4 B read + 4 B written per element of compulsory HBM traffic instead of 3 x (4 + 4).
//
// A CTA owns an (x, y) tile and marches along z:
//   y pass  in registers: a thread owns float4 columns of K consecutive rows and loads the K + 2R
//           rows it needs (128-bit, coalesced along x; the overlap between row groups hits L1);
//   x pass  through shared memory: the y-smoothed float4s of the tile (+ one halo float4 group per
//           side per 4 taps) are exchanged once per plane, one barrier per plane (double buffer);
//   z pass  in registers: a ring of the last 2R + 1 xy-smoothed planes, statically indexed by
//           unrolling the march by the ring length.
// Borders replicate the edge value on every axis (clamp), as the oracle's index clamp does.
// The paper staged all three passes through shared memory with one kernel per axis (L175, GTX 285);
// here only the x exchange touches shared memory and HBM sees the field once.
#include "kernels.h"

namespace demons {

namespace {

struct Taps {
    float w[12];
};

template <int R>
struct FusedCfg {
    static constexpr int NH = (R + 3) / 4;  // halo float4 groups per side
    static constexpr int L = 2 * R + 1;     // ring length
};

// GX: float4 groups per tile row (tile width 4 GX), RG: row groups, K: rows per thread.
template <int R, int K, int GX, int RG>
__global__ void __launch_bounds__((GX + 2 * FusedCfg<R>::NH) * RG)
    k_smooth_fused(const float* __restrict__ in, float* __restrict__ out, const Dims d, const int zc,
                   const int tiles_x, const Taps t, const int* __restrict__ skip) {
    constexpr int NH = FusedCfg<R>::NH;
    constexpr int L = FusedCfg<R>::L;
    constexpr int GW = GX + 2 * NH;  // float4 groups per shared row
    constexpr int TY = RG * K;
    __shared__ float4 xs[2][TY][GW];

    if (skip != nullptr && *reinterpret_cast<const volatile int*>(skip) != 0) return;

    const int gx = threadIdx.x, rg = threadIdx.y;
    const int tile_x = blockIdx.x % tiles_x, tile_y = blockIdx.x / tiles_x;
    const int x0 = tile_x * GX * 4, y0 = tile_y * TY;
    const int z_start = blockIdx.y * zc;
    const int nplanes = min(zc, d.nz - z_start);  // output planes of this CTA
    const size_t plane = (size_t)d.nx * d.ny;
    const float* src = in + (size_t)blockIdx.z * plane * d.nz;
    float* dst = out + (size_t)blockIdx.z * plane * d.nz;

    const int xg = x0 + 4 * (gx - NH);            // first x of this thread's float4
    const int xg_c = min(max(xg, 0), d.nx - 4);   // where it is loaded from
    const bool owner = gx >= NH && gx < NH + GX && xg < d.nx;
    int rowoff[K + 2 * R];
#pragma unroll
    for (int i = 0; i < K + 2 * R; ++i) {
        const int y = min(max(y0 + rg * K - R + i, 0), d.ny - 1);
        rowoff[i] = y * d.nx + xg_c;
    }

    float4 v[K + 2 * R];
    auto load_plane = [&](int p) {  // p-th plane of the march = volume plane z_start - R + p, clamped
        const int z = min(max(z_start - R + p, 0), d.nz - 1);
        const float* base = src + (size_t)z * plane;
#pragma unroll
        for (int i = 0; i < K + 2 * R; ++i) v[i] = __ldg(reinterpret_cast<const float4*>(base + rowoff[i]));
    };

    float4 ring[L][K];
    const int P = nplanes + 2 * R;
    load_plane(0);
    for (int pg = 0; pg < P; pg += L) {
#pragma unroll
        for (int s = 0; s < L; ++s) {
            const int p = pg + s;
            if (p < P) {  // uniform over the CTA
                // ---- y pass (registers) ----
                float4 ys[K];
#pragma unroll
                for (int j = 0; j < K; ++j) {
                    float4 a = v[j + R];
                    a.x *= t.w[0];
                    a.y *= t.w[0];
                    a.z *= t.w[0];
                    a.w *= t.w[0];
#pragma unroll
                    for (int k = 1; k <= R; ++k) {
                        const float4 lo = v[j + R - k], hi = v[j + R + k];
                        a.x = fmaf(t.w[k], lo.x + hi.x, a.x);
                        a.y = fmaf(t.w[k], lo.y + hi.y, a.y);
                        a.z = fmaf(t.w[k], lo.z + hi.z, a.z);
                        a.w = fmaf(t.w[k], lo.w + hi.w, a.w);
                    }
                    if (xg < 0) a = make_float4(a.x, a.x, a.x, a.x);          // left of the volume
                    if (xg >= d.nx) a = make_float4(a.w, a.w, a.w, a.w);      // right of the volume
                    ys[j] = a;
                    xs[p & 1][rg * K + j][gx] = a;
                }
                if (p + 1 < P) load_plane(p + 1);  // in flight during the x and z passes
                __syncthreads();
                if (owner) {
                    // ---- x pass (shared-memory exchange) ----
#pragma unroll
                    for (int j = 0; j < K; ++j) {
                        float a[4 * (2 * NH + 1)];
#pragma unroll
                        for (int h = 0; h < 2 * NH + 1; ++h) {
                            const float4 q = h == NH ? ys[j] : xs[p & 1][rg * K + j][gx - NH + h];
                            a[4 * h + 0] = q.x;
                            a[4 * h + 1] = q.y;
                            a[4 * h + 2] = q.z;
                            a[4 * h + 3] = q.w;
                        }
                        float o[4];
#pragma unroll
                        for (int e = 0; e < 4; ++e) {
                            float acc = t.w[0] * a[4 * NH + e];
#pragma unroll
                            for (int k = 1; k <= R; ++k) acc = fmaf(t.w[k], a[4 * NH + e - k] + a[4 * NH + e + k], acc);
                            o[e] = acc;
                        }
                        ring[s][j] = make_float4(o[0], o[1], o[2], o[3]);
                    }
                    // ---- z pass (register ring) ----
                    if (p >= 2 * R) {
                        const int z = z_start + p - 2 * R;
#pragma unroll
                        for (int j = 0; j < K; ++j) {
                            const int y = y0 + rg * K + j;
                            float4 c = ring[(s - R + L) % L][j];
                            c.x *= t.w[0];
                            c.y *= t.w[0];
                            c.z *= t.w[0];
                            c.w *= t.w[0];
#pragma unroll
                            for (int k = 1; k <= R; ++k) {
                                const float4 lo = ring[(s - R - k + 2 * L) % L][j], hi = ring[(s - R + k + L) % L][j];
                                c.x = fmaf(t.w[k], lo.x + hi.x, c.x);
                                c.y = fmaf(t.w[k], lo.y + hi.y, c.y);
                                c.z = fmaf(t.w[k], lo.z + hi.z, c.z);
                                c.w = fmaf(t.w[k], lo.w + hi.w, c.w);
                            }
                            if (y < d.ny)
                                *reinterpret_cast<float4*>(dst + (size_t)z * plane + (size_t)y * d.nx + xg) = c;
                        }
                    }
                }
            }
        }
    }
}

bool aligned16(const void* p) { return (reinterpret_cast<uintptr_t>(p) & 15u) == 0; }

template <int R, int K, int GX, int RG>
int launch_cfg(const SmoothArgs& a, int zc, cudaStream_t st) {
    constexpr int NH = FusedCfg<R>::NH;
    const int tiles_x = (a.d.nx + GX * 4 - 1) / (GX * 4);
    const int tiles_y = (a.d.ny + RG * K - 1) / (RG * K);
    const int chunks = (a.d.nz + zc - 1) / zc;
    if (chunks > 65535 || a.ncomp > 65535) return 0;
    Taps t;
    for (int k = 0; k < 12; ++k) t.w[k] = k <= a.R ? a.w[k] : 0.f;
    const dim3 grid(tiles_x * tiles_y, chunks, a.ncomp);
    const dim3 block(GX + 2 * NH, RG);
    k_smooth_fused<R, K, GX, RG><<<grid, block, 0, st>>>(a.in, a.out, a.d, zc, tiles_x, t, a.skip);
    return cudaPeekAtLastError() == cudaSuccess ? 1 : -1;
}

// z-chunk: long enough to amortise the 2R warm-up planes, short enough to fill the 148 SMs.
int pick_zc(const SmoothArgs& a, int tile_w, int tile_h, int ctas_wanted) {
    const long long tiles = (long long)((a.d.nx + tile_w - 1) / tile_w) * ((a.d.ny + tile_h - 1) / tile_h) * a.ncomp;
    long long chunks = (ctas_wanted + tiles - 1) / tiles;
    if (chunks < 1) chunks = 1;
    int zc = (int)((a.d.nz + chunks - 1) / chunks);
    const int zmin = 4 * a.R < 8 ? 8 : 4 * a.R;
    if (zc < zmin) zc = zmin;
    if (zc > a.d.nz) zc = a.d.nz;
    return zc;
}

}  // namespace

// Returns launches (1), 0 if the fast path does not apply, -1 on a launch error.
int launch_smooth_fused(const SmoothArgs& a, cudaStream_t st) {
    if (a.d.nx % 4 != 0 || a.d.nx < 4 || !aligned16(a.in) || !aligned16(a.out)) return 0;
    if (a.R < 1 || a.R > 6) return 0;  // wider filters: the separable fallback
    const int zc = a.zc_override > 0 ? a.zc_override : pick_zc(a, 64, 16, 148 * 6);
    switch (a.R) {
    case 1: return launch_cfg<1, 2, 16, 8>(a, zc, st);
    case 2: return launch_cfg<2, 2, 16, 8>(a, zc, st);
    case 3: return launch_cfg<3, 2, 16, 8>(a, zc, st);
    case 4: return launch_cfg<4, 2, 16, 8>(a, zc, st);
    case 5: return launch_cfg<5, 1, 16, 16>(a, zc, st);
    case 6: return launch_cfg<6, 1, 16, 16>(a, zc, st);
    default: return 0;
    }
}

}  // namespace demons
