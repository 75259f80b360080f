// S5, B200 fast path: the whole separable Gaussian (reading A9) in ONE pass
// over the field, fed by TMA.
//
// A CTA owns a 128-wide (x) by TY-high (y) tile and marches along z.  Per plane:
//   * one elected thread issues a 4D `cp.async.bulk.tensor` (TMA) load of the tile plus its
//     y/x halo into a STAGES-deep shared-memory ring, completion on an mbarrier -- no load
//     instructions, no address arithmetic, no registers spent on prefetch;
//   * y pass in registers from shared memory (a thread owns one float4 column of K rows and reads
//     the K + 2R rows it needs), packed f32x2 arithmetic (FFMA2 / FADD2 on sm_100);
//   * x pass through a small shared-memory exchange of the y-smoothed float4s; the halo columns
//     of the tile are y-smoothed by a few lanes of one extra warp (which also issues the TMA);
//   * z pass in registers: a ring of the last 2R + 1 xy-smoothed planes, statically indexed by
//     unrolling the march by the ring length; 128-bit coalesced stores.
// Borders replicate the edge value (index clamp) on every axis, exactly as the oracle's clamp:
// TMA zero-fills outside the volume, and those cells are never read -- rows / column groups are
// clamped when the shared-memory addresses are formed.
// HBM sees every element once in and once out (8 B / element); the paper's design was one
// kernel per axis through shared memory (L175), i.e. 24 B / element.
// R >= 5 (one CTA per SM): work is split evenly over ONE wave of CTAs (round 2): the columns (tile, component) are laid end to end on a
// virtual z axis, each preceded by its 2R warm-up planes, and CTA i takes the i-th equal share of that axis -- a
// run of planes that may end one column and begin the next.  Equal z chunks cost  waves x (planes + 2R)  and left
// half of the last wave idle at 256x256x100; the shares cost  total / slots + 2R  (70.2 -> 66.5 us there, 381 -> 346 us
// at 512x512x160).  R <= 4 keeps equal chunks: with three CTAs per SM the even split gains 1.5 % standalone, and it
// loses the reuse of the y halo rows between neighbouring tiles in L2 (204 -> 282 us at 512x512x160).
// The march runs DOWN the z axis by default (`rev`): the force kernels march up, so the planes they
// wrote last are read first while they are still in L2, and the planes written last here are the
// ones the next force kernel reads first.  The taps are symmetric: the result is bit-identical.
#include <algorithm>
#include <atomic>

#include "kernels.h"
#include "tma.cuh"

namespace demons {

namespace {

struct Taps {
    float w[8];
};

using tma::mbar_expect_tx;
using tma::mbar_init;
using tma::mbar_wait;

struct F4 {  // a float4 as two packed pairs
    float2 a, b;
};
__device__ __forceinline__ F4 ld_f4(const float* p) {
    const float4 q = *reinterpret_cast<const float4*>(p);
    F4 r;
    r.a = make_float2(q.x, q.y);
    r.b = make_float2(q.z, q.w);
    return r;
}

template <int R, int K, int RG, int STAGES, int PAIR = 1>
struct Cfg {
    static constexpr int NH = (R + 3) / 4;      // halo float4 groups per side
    static constexpr int L = 2 * R + 1;         // ring length
    static constexpr int GX = 32;               // owner float4 groups per row (one warp wide)
    // groups per shared row: owners, halos and one group of padding -- without it the rows of consecutive row
    // groups (K rows apart) start on the same banks and the halo warp's loads conflict 8 ways (24 % of the
    // shared-memory wavefronts at R = 6; 39.6 -> 38.6 us at R = 3, 75.2 -> 71.6 us at R = 6, bit-identical)
    static constexpr int GW = GX + 2 * NH + 1;
    static constexpr int TY = RG * K;           // output rows per tile
    static constexpr int ROWS = TY + 2 * R;     // rows per loaded plane
    static constexpr int BOXW = 4 * GW;         // floats per loaded row
    static constexpr int STAGE_BYTES = (ROWS * BOXW * 4 + 127) / 128 * 128;
    static constexpr int LR = PAIR == 2 ? L + 1 : L;  // ring slots (even when planes go in pairs)
    static constexpr int XS_BYTES = 2 * PAIR * TY * GW * 16;
    static constexpr int THREADS = 32 * (RG + 1);
    static constexpr int SMEM = STAGES * STAGE_BYTES + XS_BYTES + STAGES * 8 + 128;
    static_assert(2 * NH * RG <= 32, "halo jobs must fit one warp");
    static_assert(TY >= R, "tile must be at least R rows high");
    static_assert(PAIR == 1 || (PAIR == 2 && STAGES % 2 == 0), "pairs need an even number of stages");
};

template <int R, int K, int RG, int STAGES, int MINB, int PAIR, int XP, int BAL>
__global__ void __launch_bounds__(32 * (RG + 1), MINB)
    k_smooth_tma(const __grid_constant__ CUtensorMap tmap, float* __restrict__ out, const Dims d, const int zc,
                 const int tiles_x, const Taps t, const Control* __restrict__ ctl, const int comps_per_pair, const int rev, const int tiles, const int ncols) {
    using C = Cfg<R, K, RG, STAGES, PAIR>;
    constexpr int LR = C::LR;
    constexpr int NH = C::NH, L = C::L, GX = C::GX, GW = C::GW, TY = C::TY, BOXW = C::BOXW;
    extern __shared__ __align__(1024) unsigned char smem[];
    float4* xs = reinterpret_cast<float4*>(smem + STAGES * C::STAGE_BYTES);  // [2][TY][GW]
    uint64_t* full = reinterpret_cast<uint64_t*>(smem + STAGES * C::STAGE_BYTES + C::XS_BYTES);

    if constexpr (!BAL) {
        // the stopping rule of this component's pair has fired: nothing to do
        if (ctl != nullptr && *reinterpret_cast<const volatile int*>(&ctl[blockIdx.z / comps_per_pair].stop_smooth) != 0) return;
    }

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const bool halo_warp = warp == RG;
    const size_t plane = (size_t)d.nx * d.ny;
    const bool issuer = halo_warp && lane == 0;

    // BAL: this CTA's share [va, vb) of the virtual axis -- column c occupies [c W, (c + 1) W), W = nz + 2R, and position
    // c W + 2R + z is output plane z of that column.  Otherwise: grid (tile, z chunk, component), one segment per CTA
    // (this loop runs once and folds away).
    const int W = d.nz + 2 * R;
    int col_first = 0, col_last = 0, off_a = 0, off_b = 0;
    if constexpr (BAL) {
        const long long V = (long long)ncols * W;
        const long long va = V * blockIdx.x / gridDim.x, vb = V * (blockIdx.x + 1) / gridDim.x;
        col_first = (int)(va / W), col_last = (int)((vb - 1) / W);
        off_a = (int)(va - (long long)col_first * W), off_b = (int)(vb - (long long)col_last * W);
    }
    bool bars_live = false;

    // one segment: planes [z_start, z_start + nplanes) of column (tile, comp), warm-up included
    auto segment = [&](const int z_start, const int nplanes, const int comp, const int tile) {
    if (nplanes <= 0) return;  // the share ends inside the warm-up prefix of this column
    // the stopping rule of this component's pair has fired: nothing to do
    if (BAL && ctl != nullptr && *reinterpret_cast<const volatile int*>(&ctl[comp / comps_per_pair].stop_smooth) != 0) return;
    const int tile_x = tile % tiles_x, tile_y = tile / tiles_x;
    const int x0 = tile_x * GX * 4, y0 = tile_y * TY;
    const int P = nplanes + 2 * R;

    // role of this thread: which float4 group (g) of which row group (rg)
    int g, rg;
    bool active;
    if (!halo_warp) {
        g = lane + NH;
        rg = warp;
        active = true;
    } else {
        rg = lane / (2 * NH);
        const int h = lane % (2 * NH);
        g = h < NH ? h : GX + h;  // left groups 0..NH-1, right groups GX+NH..GX+2NH-1
        active = lane < 2 * NH * RG;
        if (!active) rg = 0;
    }
    const int xg = x0 + 4 * (g - NH);
    const int xg_c = min(max(xg, 0), d.nx - 4);
    const int gc = (xg_c - (x0 - 4 * NH)) >> 2;  // group actually read (clamp = replicate)
    const bool owner = !halo_warp && xg < d.nx;
    const bool outside = xg < 0 || xg >= d.nx;
    int rowoff[K + 2 * R];
#pragma unroll
    for (int i = 0; i < K + 2 * R; ++i) {
        const int y = min(max(y0 + rg * K - R + i, 0), d.ny - 1);
        rowoff[i] = (y - (y0 - R)) * BOXW + 4 * gc;
    }
    float2 w2[R + 1];
#pragma unroll
    for (int k = 0; k <= R; ++k) w2[k] = make_float2(t.w[k], t.w[k]);

    auto issue = [&](int p) {  // plane p of the march -> stage p % STAGES
        const int s = p % STAGES;
        const int z = min(max(rev ? z_start + nplanes - 1 + R - p : z_start - R + p, 0), d.nz - 1);
        mbar_expect_tx(&full[s], (uint32_t)(C::ROWS * BOXW * 4));
        tma::load_4d(smem + s * C::STAGE_BYTES, &tmap, &full[s], x0 - 4 * NH, y0 - R, z, comp);
    };
    // a segment starts with fresh barriers (phase 0), so that stage and parity of plane p stay p % STAGES and
    // (p / STAGES) & 1; the __syncthreads also keeps a fast warp out of the exchange buffer the slow ones still read
    if constexpr (BAL) __syncthreads();
    if (issuer) {
#pragma unroll
        for (int s = 0; s < STAGES; ++s) {
            if (BAL && bars_live) tma::mbar_inval(&full[s]);
            mbar_init(&full[s], 1);
        }
        tma::mbar_fence_init();
    }
    bars_live = true;
    __syncthreads();
    if (issuer) {
        for (int p = 0; p < STAGES && p < P; ++p) issue(p);
    }

    float* dst = out + (size_t)comp * plane * d.nz + (size_t)(y0 + rg * K) * d.nx + xg;
    F4 ring[LR][K];
    auto xrow_of = [&](int p) { return xs + ((((p / PAIR) & 1) * PAIR + (p % PAIR)) * TY + rg * K) * GW; };
    // ---- y pass of plane p: registers, packed f32x2; the y-smoothed float4s also go to the exchange buffer
    auto ypass = [&](int p, F4 (&ys)[K], float4* xrow) {
        const int stage = p % STAGES;
        mbar_wait(&full[stage], (uint32_t)((p / STAGES) & 1));
        const float* raw = reinterpret_cast<const float*>(smem + stage * C::STAGE_BYTES);
        if (active) {
            F4 v[K + 2 * R];
#pragma unroll
            for (int i = 0; i < K + 2 * R; ++i) v[i] = ld_f4(raw + rowoff[i]);
#pragma unroll
            for (int j = 0; j < K; ++j) {
                float2 a = __fmul2_rn(w2[0], v[j + R].a), b = __fmul2_rn(w2[0], v[j + R].b);
#pragma unroll
                for (int k = 1; k <= R; ++k) {
                    a = __ffma2_rn(w2[k], __fadd2_rn(v[j + R - k].a, v[j + R + k].a), a);
                    b = __ffma2_rn(w2[k], __fadd2_rn(v[j + R - k].b, v[j + R + k].b), b);
                }
                if (outside) {  // rare: halo lanes / ragged tiles at the volume border
                    if (xg < 0) {  // left of the volume: replicate x = 0
                        a = make_float2(a.x, a.x);
                        b = a;
                    } else {  // right of the volume: replicate x = nx - 1
                        b = make_float2(b.y, b.y);
                        a = b;
                    }
                }
                ys[j].a = a;
                ys[j].b = b;
                if constexpr (!XP) xrow[j * GW + g] = make_float4(a.x, a.y, b.x, b.y);
            }
            if constexpr (XP) {  // rows 2jp and 2jp + 1 interleaved element by element: (r0 x0, r1 x0, r0 x1, r1 x1), (.. x2, x3)
#pragma unroll
                for (int jp = 0; jp < K / 2; ++jp) {
                    const F4 &r0 = ys[2 * jp], &r1 = ys[2 * jp + 1];
                    xrow[(2 * jp) * GW + g] = make_float4(r0.a.x, r1.a.x, r0.a.y, r1.a.y);
                    xrow[(2 * jp + 1) * GW + g] = make_float4(r0.b.x, r1.b.x, r0.b.y, r1.b.y);
                }
            }
        }
    };
    // ---- x and z pass, ROW-PAIR form (XP; R >= 5).  Element e of the x window is the float2 (row 2jp, row 2jp + 1) at
    // one x, so every tap is an aligned register pair and the whole x pass is packed f32x2 (half the instructions of
    // the scalar pass; the y pass wrote the exchange rows interleaved that way).  The ring and the z pass carry the
    // same pairs; the rows are separated again at the store.
    auto xzpass_xp = [&](int p, int sl, const F4 (&ys)[K], const float4* xrow) {
        static_assert(!XP || K % 2 == 0, "row pairs");
        float4 q[K][2 * NH];  // the neighbours' y-smoothed float4s of this thread's exchange rows
#pragma unroll
        for (int r = 0; r < K; ++r)
#pragma unroll
            for (int h = 0; h < 2 * NH; ++h) q[r][h] = xrow[r * GW + g - NH + (h < NH ? h : h + 1)];
#pragma unroll
        for (int jp = 0; jp < K / 2; ++jp) {
            float2 a[4 * (2 * NH + 1)];
#pragma unroll
            for (int h = 0; h < 2 * NH + 1; ++h) {
                if (h == NH) {
                    const F4 &r0 = ys[2 * jp], &r1 = ys[2 * jp + 1];
                    a[4 * h + 0] = make_float2(r0.a.x, r1.a.x);
                    a[4 * h + 1] = make_float2(r0.a.y, r1.a.y);
                    a[4 * h + 2] = make_float2(r0.b.x, r1.b.x);
                    a[4 * h + 3] = make_float2(r0.b.y, r1.b.y);
                } else {
                    const float4 q0 = q[2 * jp][h < NH ? h : h - 1], q1 = q[2 * jp + 1][h < NH ? h : h - 1];
                    a[4 * h + 0] = make_float2(q0.x, q0.y);
                    a[4 * h + 1] = make_float2(q0.z, q0.w);
                    a[4 * h + 2] = make_float2(q1.x, q1.y);
                    a[4 * h + 3] = make_float2(q1.z, q1.w);
                }
            }
            float2 o[4];
#pragma unroll
            for (int e = 0; e < 4; ++e) {
                float2 acc = __fmul2_rn(w2[0], a[4 * NH + e]);
#pragma unroll
                for (int k = 1; k <= R; ++k) acc = __ffma2_rn(w2[k], __fadd2_rn(a[4 * NH + e - k], a[4 * NH + e + k]), acc);
                o[e] = acc;
            }
            ring[sl][2 * jp].a = o[0];  // (x0, x1) of the row pair
            ring[sl][2 * jp].b = o[1];
            ring[sl][2 * jp + 1].a = o[2];  // (x2, x3)
            ring[sl][2 * jp + 1].b = o[3];
        }
        if (p >= 2 * R) {
            float* orow = dst + (size_t)(rev ? z_start + nplanes - 1 - (p - 2 * R) : z_start + p - 2 * R) * plane;
            F4 zo[K];
#pragma unroll
            for (int j = 0; j < K; ++j) {
                const F4& c = ring[(sl - R + LR) % LR][j];
                float2 a = __fmul2_rn(w2[0], c.a), b = __fmul2_rn(w2[0], c.b);
#pragma unroll
                for (int k = 1; k <= R; ++k) {
                    const F4& lo = ring[(sl - R - k + 2 * LR) % LR][j];
                    const F4& hi = ring[(sl - R + k + LR) % LR][j];
                    a = __ffma2_rn(w2[k], __fadd2_rn(lo.a, hi.a), a);
                    b = __ffma2_rn(w2[k], __fadd2_rn(lo.b, hi.b), b);
                }
                zo[j].a = a;
                zo[j].b = b;
            }
#pragma unroll
            for (int j = 0; j < K; ++j) {  // .x = even row, .y = odd row
                const F4 &lo = zo[j & ~1], &hi = zo[j | 1];
                const float4 v = (j & 1) ? make_float4(lo.a.y, lo.b.y, hi.a.y, hi.b.y) : make_float4(lo.a.x, lo.b.x, hi.a.x, hi.b.x);
                if (y0 + rg * K + j < d.ny) *reinterpret_cast<float4*>(orow + (size_t)j * d.nx) = v;
            }
        }
    };
    // ---- x pass of plane p into ring slot sl (neighbours' float4s from the exchange buffer), then the
    // z pass of the plane R behind it (register ring, packed f32x2) and its store
    auto xzpass_scalar = [&](int p, int sl, const F4 (&ys)[K], const float4* xrow) {
#pragma unroll
        for (int j = 0; j < K; ++j) {
            float a[4 * (2 * NH + 1)];
#pragma unroll
            for (int h = 0; h < 2 * NH + 1; ++h) {
                if (h == NH) {
                    a[4 * h + 0] = ys[j].a.x;
                    a[4 * h + 1] = ys[j].a.y;
                    a[4 * h + 2] = ys[j].b.x;
                    a[4 * h + 3] = ys[j].b.y;
                } else {
                    const float4 q = xrow[j * GW + g - NH + h];
                    a[4 * h + 0] = q.x;
                    a[4 * h + 1] = q.y;
                    a[4 * h + 2] = q.z;
                    a[4 * h + 3] = q.w;
                }
            }
            float o[4];
#pragma unroll
            for (int e = 0; e < 4; ++e) {
                float acc = t.w[0] * a[4 * NH + e];
#pragma unroll
                for (int k = 1; k <= R; ++k) acc = fmaf(t.w[k], a[4 * NH + e - k] + a[4 * NH + e + k], acc);
                o[e] = acc;
            }
            ring[sl][j].a = make_float2(o[0], o[1]);
            ring[sl][j].b = make_float2(o[2], o[3]);
        }
        if (p >= 2 * R) {
            float* orow = dst + (size_t)(rev ? z_start + nplanes - 1 - (p - 2 * R) : z_start + p - 2 * R) * plane;
#pragma unroll
            for (int j = 0; j < K; ++j) {
                const F4& c = ring[(sl - R + LR) % LR][j];
                float2 a = __fmul2_rn(w2[0], c.a), b = __fmul2_rn(w2[0], c.b);
#pragma unroll
                for (int k = 1; k <= R; ++k) {
                    const F4& lo = ring[(sl - R - k + 2 * LR) % LR][j];
                    const F4& hi = ring[(sl - R + k + LR) % LR][j];
                    a = __ffma2_rn(w2[k], __fadd2_rn(lo.a, hi.a), a);
                    b = __ffma2_rn(w2[k], __fadd2_rn(lo.b, hi.b), b);
                }
                if (y0 + rg * K + j < d.ny)
                    *reinterpret_cast<float4*>(orow + (size_t)j * d.nx) = make_float4(a.x, a.y, b.x, b.y);
            }
        }
    };
    if constexpr (PAIR == 1) {
        for (int pg = 0; pg < P; pg += LR) {
#pragma unroll
            for (int s = 0; s < LR; ++s) {
                const int p = pg + s;
                if (p < P) {  // uniform over the CTA
                    float4* xrow = xrow_of(p);
                    F4 ys[K];
                    ypass(p, ys, xrow);
                    __syncthreads();  // xs complete; every warp is done reading this raw stage
                    if (issuer && p + STAGES < P) issue(p + STAGES);
                    if (owner) {
                        if constexpr (XP) xzpass_xp(p, s, ys, xrow);
                        else xzpass_scalar(p, s, ys, xrow);
                    }
                }
            }
        }
    } else {
        // Two planes per barrier: half the block-wide synchronisations and twice the independent
        // arithmetic between them.
        for (int pg = 0; pg < P; pg += LR) {
#pragma unroll
            for (int s2 = 0; s2 < LR / 2; ++s2) {
                const int p0 = pg + 2 * s2;
                if (p0 < P) {  // uniform over the CTA
                    const bool two = p0 + 1 < P;
                    float4* xr0 = xrow_of(p0);
                    float4* xr1 = xrow_of(p0 + 1);
                    F4 ys0[K], ys1[K];
                    ypass(p0, ys0, xr0);
                    if (two) ypass(p0 + 1, ys1, xr1);
                    __syncthreads();
                    if (issuer) {
                        if (p0 + STAGES < P) issue(p0 + STAGES);
                        if (p0 + 1 + STAGES < P) issue(p0 + 1 + STAGES);
                    }
                    if (owner) {
                        xzpass_scalar(p0, 2 * s2, ys0, xr0);
                        if (two) xzpass_scalar(p0 + 1, 2 * s2 + 1, ys1, xr1);
                    }
                }
            }
        }
    }
    };  // segment
    if constexpr (BAL) {
        for (int col = col_first; col <= col_last; ++col) {
            const int z_start = col == col_first ? max(off_a - 2 * R, 0) : 0;
            const int z_end = col == col_last ? min(off_b - 2 * R, d.nz) : d.nz;
            segment(z_start, z_end - z_start, col / tiles, col % tiles);
        }
    } else {
        segment(blockIdx.y * zc, min(zc, d.nz - (int)blockIdx.y * zc), blockIdx.z, blockIdx.x);
    }
}

// Planes per CTA: the number of z chunks that minimises  waves x (planes per chunk + 2R warm-up + start-up).  Small
// volumes end up with very short chunks (2-3 planes behind 2R warm-up planes): the machine is mostly empty there and
// the length of the march counts, not the number of CTAs (64x64x25: 9.4 -> 9.2 us per iteration with chunks of 2
// instead of 7 planes; start-up and drain dominate at that size).
int pick_zc(const SmoothArgs& a, int tile_w, int tile_h, int slots) {
    const long long tiles = (long long)((a.d.nx + tile_w - 1) / tile_w) * ((a.d.ny + tile_h - 1) / tile_h) * a.ncomp;
    int best_zc = a.d.nz;
    double best = 1e300;
    for (int chunks = 1; chunks <= a.d.nz; ++chunks) {
        const int zc = (a.d.nz + chunks - 1) / chunks;
        const long long ctas = tiles * ((a.d.nz + zc - 1) / zc);
        const double waves = (double)((ctas + slots - 1) / slots);
        const double cost = waves * (zc + 2 * a.R + 2);
        if (cost < best - 1e-9) {
            best = cost;
            best_zc = zc;
        }
    }
    return best_zc;
}

template <int R, int K, int RG, int STAGES, int MINB, int PAIR = 1, int XP = 0, int BAL = 0>
int launch_cfg(const SmoothArgs& a, int slots, cudaStream_t st) {
    using C = Cfg<R, K, RG, STAGES, PAIR>;
    const Dims d = a.d;
    alignas(64) CUtensorMap map;
    const unsigned long long gdim[4] = {(unsigned long long)d.nx, (unsigned long long)d.ny, (unsigned long long)d.nz,
                                        (unsigned long long)a.ncomp};
    const unsigned box[4] = {(unsigned)C::BOXW, (unsigned)C::ROWS, 1u, 1u};
    if (!tma::encode_f32(&map, a.in, 4, gdim, box)) return 0;
    // per device: the attribute belongs to the device's copy of the kernel.  Atomic flags: two host threads may get
    // here together; setting the attribute twice is harmless, a torn flag is not.
    static std::atomic<bool> attr_set[64] = {};
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= 64) return 0;
    if (!attr_set[dev].load(std::memory_order_acquire)) {
        if (cudaFuncSetAttribute(k_smooth_tma<R, K, RG, STAGES, MINB, PAIR, XP, BAL>, cudaFuncAttributeMaxDynamicSharedMemorySize, C::SMEM) !=
            cudaSuccess) {
            cudaGetLastError();
            return 0;  // refused: not applicable here, the caller falls back to the separable passes
        }
        cudaFuncSetAttribute(k_smooth_tma<R, K, RG, STAGES, MINB, PAIR, XP, BAL>, cudaFuncAttributePreferredSharedMemoryCarveout, 100);
        attr_set[dev].store(true, std::memory_order_release);
    }
    const int tiles_x = (d.nx + C::GX * 4 - 1) / (C::GX * 4);
    const int tiles_y = (d.ny + C::TY - 1) / C::TY;
    const long long ncols = (long long)tiles_x * tiles_y * a.ncomp;
    if (ncols * (d.nz + 2 * R) >= (1ll << 31)) return 0;
    dim3 grid;
    int zc = 0;
    if constexpr (BAL) {
        // one wave of equal shares; a share is never shorter than the 2R + 2 planes of a warm-up
        grid = dim3((unsigned)std::max(1ll, std::min((long long)slots, ncols * (d.nz + 2 * R) / (2 * R + 2))));
    } else {
        zc = pick_zc(a, C::GX * 4, C::TY, slots);
        const int chunks = (d.nz + zc - 1) / zc;
        if (chunks > 65535 || a.ncomp > 65535) return 0;
        grid = dim3(tiles_x * tiles_y, chunks, a.ncomp);
    }
    Taps t;
    for (int k = 0; k < 8; ++k) t.w[k] = k <= a.R ? a.w[k] : 0.f;
    k_smooth_tma<R, K, RG, STAGES, MINB, PAIR, XP, BAL><<<grid, C::THREADS, C::SMEM, st>>>(
        map, a.out, d, zc, tiles_x, t, a.ctl, a.comps_per_pair > 0 ? a.comps_per_pair : a.ncomp,
        a.ascending ? 0 : 1, tiles_x * tiles_y, (int)ncols);
    return cudaPeekAtLastError() == cudaSuccess ? 1 : -1;
}

bool aligned16(const void* p) { return (reinterpret_cast<uintptr_t>(p) & 15u) == 0; }

}  // namespace

// Returns launches (1), 0 if this path does not apply (caller falls back), -1 on a launch error.
int launch_smooth_tma(const SmoothArgs& a, cudaStream_t st) {
    if (a.d.nx % 4 != 0 || a.d.nx < 4 || !aligned16(a.in) || !aligned16(a.out)) return 0;
    if (a.R < 1 || a.R > 6) return 0;
    // CTAs per SM of the configuration picked below (its launch bounds): the grid is one wave of them
    int per_sm = 3;
    if (a.R == 4) per_sm = 2;
    if (a.R > 4) per_sm = 1;
    const int slots = sm_count() * per_sm;
    // two planes per barrier where the registers allow it: 39.6 against 41.8 us at sigma 1 (R = 3),
    // 50.0 against 51.9 us at sigma 1.3 (R = 4), 256x256x100; no difference at R <= 2
    switch (a.R) {
    case 1: return launch_cfg<1, 2, 4, 4, 3, 2>(a, slots, st);
    case 2: return launch_cfg<2, 2, 4, 4, 3, 2>(a, slots, st);
    case 3: return launch_cfg<3, 2, 4, 4, 3, 2>(a, slots, st);
    case 4: return launch_cfg<4, 2, 4, 4, 2, 2>(a, slots, st);
    case 5: return launch_cfg<5, 2, 8, 4, 1, 1, 1, 1>(a, slots, st);
    case 6: return launch_cfg<6, 2, 8, 4, 1, 1, 1, 1>(a, slots, st);
    default: return 0;
    }
}

}  // namespace demons
