// S1-S4 and S6 of the demons hot path: trilinear warp, central-difference gradients, the per-voxel
// force of Eq.(1)-(6), the additive update u' = u - F and the three metrics of
// PAPER.md L145, hand-written for sm_100a.
//
// Variants 0-1 (gradients of the fixed level images only): ONE kernel -- the warped intensity
// lives in a register, grad S (and grad M0) are recomputed from a 6-point stencil whose re-reads
// hit L1/L2, so the compulsory HBM traffic is u (12 B) + S (4 B) + M (4 B) in, u' (12 B) out.
// Variants 2-5 need the gradient of the WARPED image (reading A8), i.e. the warped values of the
// six neighbours: the warped image is materialised once (k_warp_lc) and then stencilled
// (k_force_active) instead of gathering 7x per voxel, which would be instruction-bound.
//
// The gathering passes are the lane-consecutive kernels (k_force_fixed_lc, k_warp_lc: one 2x2x2 cell
// offset per sample, no branch between the loads of a plane); k_force_active (no gathers) is float4 per
// lane.  Volumes with an axis of length 1, where a 2x2x2 cell does not exist, take the one-voxel-per-thread
// kernels k_force_fixed / k_warp (generic index-clamped sampler).
//
// Every kernel carries a pair index in blockIdx.z (blockIdx.z = pair * chunks + z-chunk): a batch of
// independent registrations runs as ONE launch per kernel, so that the small pyramid levels fill the GPU.
#include <mutex>

#include "kernels.h"

namespace demons {

namespace {

constexpr int BX = 32;  // threads along x
constexpr int BY = 8;   // threads along y (the lane-consecutive kernels may be launched with 4..8 rows)

__device__ __forceinline__ bool skip_pass(const MetricSink& s, unsigned b) {
    // eps <= 0: the rule is off and the flag can never be set -- no load (an L2 round trip before the first useful one)
    if (s.driver && s.eps > 0.0 && *reinterpret_cast<volatile int*>(&s.ctl[b].stop_force) != 0) {
        s.ctl[b].stop_smooth = 1;
        return true;
    }
    return false;
}

// Thread 0 of the last block of pair b: write {SSD, sum|F|, sum|u|}, advance the row, apply the stopping
// rule  l_n = sum|F| / sum|u|;  stop after the first n >= 10 with |l_n - l_{n-10}| <= eps.
__device__ __forceinline__ void publish_metrics_at(const double (&v)[3], const MetricSink& s, unsigned b, unsigned row,
                                                   unsigned n) {
    Control& c = s.ctl[b];
    double* o = s.out + (size_t)b * s.out_stride + 3 * (size_t)row;
    o[0] = v[0];
    o[1] = v[1];
    o[2] = v[2];
    if (s.driver) {
        c.row_counter = row + 1u;
        const int valid = v[2] > 0.0;
        const double l = valid ? v[1] / v[2] : 0.0;
        c.lhist[n & (LHIST - 1)] = l;
        c.lvalid[n & (LHIST - 1)] = valid;
        if (s.eps > 0.0 && n >= 10u && valid && c.lvalid[(n - 10u) & (LHIST - 1)] &&
            fabs(l - c.lhist[(n - 10u) & (LHIST - 1)]) <= s.eps)
            c.stop_force = 1;
        c.level_iter = n + 1u;
    }
}
__device__ __forceinline__ void publish_metrics(const double (&v)[3], const MetricSink& s, unsigned b) {
    publish_metrics_at(v, s, b, s.driver ? s.ctl[b].row_counter : 0u, s.driver ? s.ctl[b].level_iter : 0u);
}

// Block-wide reduction of the three metrics of pair b and their publication by the last block of the pair.
__device__ __forceinline__ void reduce_metrics(double (&acc)[3], const MetricSink& s, unsigned b, unsigned chunk,
                                               unsigned chunks) {
    if (s.out == nullptr) return;
    const unsigned bid = blockIdx.x + gridDim.x * (blockIdx.y + gridDim.y * chunk);
    const unsigned nblocks = gridDim.x * gridDim.y * chunks;
    if (s.defer) {
        // inside a registration: the fence, the ticket and the last block's final sum were 4.8 of the 47 us of the
        // fused pass at 256x256x100 (the tail of the kernel); k_metrics_final does them beside the smoothing kernel
        block_reduce_store<3>(acc, s.partials + (size_t)b * 5 * s.stride, s.stride, bid);
        return;
    }
    if (block_reduce_publish<3>(acc, s.partials + (size_t)b * 5 * s.stride, s.stride, &s.ctl[b].ticket, bid, nblocks))
        publish_metrics(acc, s, b);
}

// Deferred metrics (MetricSink::defer): one block per pair sums the block partials of the force kernel that has
// just finished, in a fixed order, writes the statistics row and applies the stopping rule.  Runs on a side branch
// of the iteration, beside the smoothing kernel; the next force kernel waits for both.
__global__ void __launch_bounds__(256) k_metrics_final(const MetricSink s) {
    const unsigned b = blockIdx.x;
    // the force pass of this iteration was skipped (the rule fired earlier): nothing was written
    if (s.driver && s.eps > 0.0 && *reinterpret_cast<volatile int*>(&s.ctl[b].stop_smooth) != 0) return;
    // the cursors are read before the sum, not behind its barriers: one L2 round trip for everything this block loads
    unsigned row = 0u, n = 0u;
    if (threadIdx.x == 0 && s.driver) {
        row = *reinterpret_cast<volatile unsigned*>(&s.ctl[b].row_counter);
        n = *reinterpret_cast<volatile unsigned*>(&s.ctl[b].level_iter);
    }
    double v[3];
    final_sum<3>(v, s.partials + (size_t)b * 5 * s.stride, s.stride, s.nblocks);
    if (threadIdx.x == 0) publish_metrics_at(v, s, b, row, n);
}

// Eq.(1): F = q(d, d^2 + |g|^2) g, with alpha^2 d^2 for Eq.(5).  Returns the scalar factor.
__device__ __forceinline__ float demons_factor(float d, float a2, float gx, float gy, float gz) {
    const float g2 = fmaf(gx, gx, fmaf(gy, gy, gz * gz));
    return guarded_div(d, fmaf(a2 * d, d, g2));
}

struct KParams {
    Dims d;
    float alpha2;
    const float* S;
    const float* M;
    const float* u_in;
    float* u_out;
    const float* ub_in;
    float* ub_out;
    float* Mw;
    float* Sw;
    const float* gm2;  // variant 1: |grad M|^2 of the level, [N]
    MetricSink sink;
    cudaTextureObject_t texM;
    unsigned img_stride;  // floats between the images of consecutive pairs
    int zper;             // consecutive planes per block
    int chunks;           // z chunks per pair; blockIdx.z = pair * chunks + chunk
    // z-slab form (SLAB kernels): the fields and warped images are a slab of d.nz planes that starts at plane zoff of
    // the images, which are whole volumes of gnz planes; only planes [mz0, mz1) of the slab count in the metrics
    int zoff, gnz, mz0, mz1;
};

// Pair b of a batched launch: every pointer moves to that pair's data.
__device__ __forceinline__ void select_pair(KParams& p, unsigned b) {
    const size_t N = nvox(p.d);
    p.S += (size_t)b * p.img_stride;
    p.M += (size_t)b * p.img_stride;
    p.u_in += (size_t)b * 3 * N;
    p.u_out += (size_t)b * 3 * N;
    if (p.ub_in) p.ub_in += (size_t)b * 3 * N;
    if (p.ub_out) p.ub_out += (size_t)b * 3 * N;
    if (p.Mw) p.Mw += (size_t)b * N;
    if (p.Sw) p.Sw += (size_t)b * N;
    if (p.gm2) p.gm2 += (size_t)b * N;
}

// ---- variants 0, 1, generic form (one voxel per thread, index-clamped sampler): volumes with an axis of
// length 1 only ---------------------------------------------------------------------------------------
template <int VARIANT>
__global__ void __launch_bounds__(BX* BY) k_force_fixed(const KParams p0) {
    constexpr int VEC = 1;
    const unsigned b = blockIdx.z / (unsigned)p0.chunks, cz = blockIdx.z - b * (unsigned)p0.chunks;
    if (skip_pass(p0.sink, b)) return;
    KParams p = p0;
    select_pair(p, b);
    const Dims d = p.d;
    const unsigned N = (unsigned)nvox(d);
    const int x0 = (blockIdx.x * BX + threadIdx.x) * VEC;
    const int y = blockIdx.y * BY + threadIdx.y;
    const bool active = x0 < d.nx && y < d.ny;
    double acc[3] = {0.0, 0.0, 0.0};
    if (active) {
        // the field of the next plane is fetched while this plane's gathers and arithmetic run
        const int zb = (int)cz * p.zper, ze = min(d.nz, zb + p.zper);
        const unsigned plane = (unsigned)(d.nx * d.ny);
        unsigned i0 = (unsigned)((zb * d.ny + y) * d.nx + x0);
        float nux[VEC], nuy[VEC], nuz[VEC];
        load_vec<VEC>(p.u_in + i0, nux);
        load_vec<VEC>(p.u_in + N + i0, nuy);
        load_vec<VEC>(p.u_in + 2 * N + i0, nuz);
        for (int z = zb; z < ze; ++z, i0 += plane) {
            float ux[VEC], uy[VEC], uz[VEC];
#pragma unroll
            for (int j = 0; j < VEC; ++j) {
                ux[j] = nux[j];
                uy[j] = nuy[j];
                uz[j] = nuz[j];
            }
            if (z + 1 < ze) {
                load_vec<VEC>(p.u_in + i0 + plane, nux);
                load_vec<VEC>(p.u_in + N + i0 + plane, nuy);
                load_vec<VEC>(p.u_in + 2 * N + i0 + plane, nuz);
            }
            float mw[VEC];
#pragma unroll
            for (int j = 0; j < VEC; ++j) mw[j] = trilinear(p.M, d, x0 + j, y, z, ux[j], uy[j], uz[j]);
            float s[VEC], gx[VEC], gy[VEC], gz[VEC];
            centre_and_gradient<VEC>(p.S, d, x0, y, z, s, gx, gy, gz);
            float k[VEC];
            if constexpr (VARIANT == 0) {
#pragma unroll
                for (int j = 0; j < VEC; ++j) k[j] = demons_factor(mw[j] - s[j], 1.f, gx[j], gy[j], gz[j]);
            } else {
                // Eq.(2): 4 d |gS| |gM0| / ((2 d^2 + |gS|^2 + |gM0|^2)(|gS|^2 + |gM0|^2)); gM0 =
                // gradient of the UNWARPED level moving image at the grid point (reading A4).
                float m0[VEC], hx[VEC], hy[VEC], hz[VEC];
                centre_and_gradient<VEC>(p.M, d, x0, y, z, m0, hx, hy, hz);
#pragma unroll
                for (int j = 0; j < VEC; ++j) {
                    const float dd = mw[j] - s[j];
                    const float s2 = fmaf(gx[j], gx[j], fmaf(gy[j], gy[j], gz[j] * gz[j]));
                    const float m2 = fmaf(hx[j], hx[j], fmaf(hy[j], hy[j], hz[j] * hz[j]));
                    const float num = 4.f * dd * fast_sqrt(s2 * m2);  // |gS| |gM0| with one square root
                    const float den = (fmaf(2.f * dd, dd, s2 + m2)) * (s2 + m2);
                    k[j] = guarded_div(num, den);
                }
            }
            float ox[VEC], oy[VEC], oz[VEC];
            float ssd = 0.f, sf = 0.f, su = 0.f;
#pragma unroll
            for (int j = 0; j < VEC; ++j) {
                const float dd = mw[j] - s[j];
                const float fx = k[j] * gx[j], fy = k[j] * gy[j], fz = k[j] * gz[j];
                ox[j] = ux[j] - fx;
                oy[j] = uy[j] - fy;
                oz[j] = uz[j] - fz;
                ssd = fmaf(dd, dd, ssd);
                sf += fast_sqrt(fmaf(fx, fx, fmaf(fy, fy, fz * fz)));
                su += fast_sqrt(fmaf(ux[j], ux[j], fmaf(uy[j], uy[j], uz[j] * uz[j])));
            }
            store_vec<VEC>(p.u_out + i0, ox);
            store_vec<VEC>(p.u_out + N + i0, oy);
            store_vec<VEC>(p.u_out + 2 * N + i0, oz);
            acc[0] += (double)ssd;
            acc[1] += (double)sf;
            acc[2] += (double)su;
        }
    }
    reduce_metrics(acc, p.sink, b, cz, (unsigned)p.chunks);
}

// ---- lane-consecutive kernels (the fast path) --------------------------------------------------
// A warp owns a 32*XPT-wide stretch of one row; lane l owns the voxels x = xb + 32 j.  Every access
// of a warp is then to 32 consecutive floats: the eight gathers of a voxel touch one or two
// 128-byte lines per warp instead of the five that a float4-per-lane assignment touches (the L1
// data pipe, not HBM, bounded that kernel).  All addresses of a row are (one 64-bit base) +
// (128 j bytes), so the j loop costs no address arithmetic.  Per plane a lane issues, back to
// back and with no branch in between, the field of the NEXT plane (register prefetch), the
// stencil of S, and the 8 XPT gathers of M; it waits for memory once.  The centre value of S
// rolls through registers along the z march.  FULL: nx is a multiple of 32*XPT (no ragged tail).
template <int XPT, bool FULL>
struct LcRow {
    bool ok[XPT];  // voxel j exists
    int dl0;       // 1 if voxel 0 has a left neighbour (x > 0); voxels j >= 1 always have one
    int dr[XPT];   // 1 if voxel j has a right neighbour (x < nx - 1)
    __device__ __forceinline__ LcRow(int xb, int nx) {
        dl0 = xb > 0;
#pragma unroll
        for (int j = 0; j < XPT; ++j) {
            ok[j] = FULL || xb + 32 * j < nx;
            dr[j] = (FULL && j < XPT - 1) ? 1 : (xb + 32 * j < nx - 1);
        }
    }
};

// Raw stencil of I at the XPT voxels of a lane on plane z: x-1, x+1, y-1, y+1, z+1 (the values of
// planes z-1 and z are already in registers).  Loads only; gradient_from_stencil does the math
// after the gathers have been issued.
template <int XPT>
struct Stencil {
    float xl[XPT], xr[XPT], ym[XPT], yp[XPT], zp[XPT];
};

template <int XPT, bool FULL>
__device__ __forceinline__ void load_stencil(const float* __restrict__ I, const LcRow<XPT, FULL>& r, unsigned row,
                                             unsigned dym, unsigned dyp, unsigned dzp, Stencil<XPT>& s) {
    const float* pc = I + row;
    const float* pl = I + (row - (unsigned)r.dl0);
    const float* pym = I + (row - dym);
    const float* pyp = I + (row + dyp);
    const float* pzp = I + (row + dzp);
#pragma unroll
    for (int j = 0; j < XPT; ++j) {
        if (FULL || r.ok[j]) {
            s.xl[j] = j == 0 ? __ldg(pl) : __ldg(pc + 32 * j - 1);
            s.xr[j] = (FULL && j < XPT - 1) ? __ldg(pc + 32 * j + 1) : __ldg(pc + 32 * j + r.dr[j]);
            s.ym[j] = __ldg(pym + 32 * j);
            s.yp[j] = __ldg(pyp + 32 * j);
            s.zp[j] = __ldg(pzp + 32 * j);
        } else {
            s.xl[j] = s.xr[j] = s.ym[j] = s.yp[j] = s.zp[j] = 0.f;
        }
    }
}

// Everything a lane needs to finish one plane: the field, the raw stencil(s) and the gathered cells.
template <int VARIANT, int XPT>
struct PlaneRegs {
    float ux[XPT], uy[XPT], uz[XPT];
    Stencil<XPT> ss;
    float m2[VARIANT == 1 ? XPT : 1];  // variant 1: |grad M0|^2 at the grid point (precomputed per level)
    float c[XPT][8], fx[XPT], fy[XPT], fz[XPT];
};

// One plane per iteration: issue() puts every load of the plane in flight (the field of the NEXT
// plane, the stencil, the 8 XPT gathers), finish() does the arithmetic and the stores.
// The stencil loads sit under a condition that is always true but opaque to the compiler (`rt`):
// the basic-block boundary keeps ptxas from merging the three load groups into one 64-load burst
// that it then schedules behind the cell arithmetic.  Measured at 256x256x100: 56.3 us with the
// boundary, 64.3 us without (the same instructions, a different order).
// BATCH = false is the single-registration launch (blockIdx.z is the z chunk, every pointer stays a kernel
// parameter): the pair offsets of a batch cost registers that the 128-register configuration does not have.
// SLAB = true: one rank's share of a z-slab decomposition (see KParams): every image access (the gather from M, the
// stencil of S, |grad M|^2) is in global planes z + zoff with the clamps of the whole volume; the field is local.
template <int VARIANT, int XPT, bool FULL, bool TEX, int MINB, bool BATCH, bool SLAB = false>
__global__ void __launch_bounds__(BX* BY, MINB) k_force_fixed_lc(const KParams p0) {
    const unsigned b = BATCH ? blockIdx.z / (unsigned)p0.chunks : 0u;
    const unsigned cz = BATCH ? blockIdx.z - b * (unsigned)p0.chunks : blockIdx.z;
    if (skip_pass(p0.sink, b)) return;
    KParams p = p0;
    if constexpr (BATCH) select_pair(p, b);
    const Dims d = p.d;
    const unsigned N = (unsigned)nvox(d);
    const int xb = blockIdx.x * (32 * XPT) + threadIdx.x;
    const int y = blockIdx.y * blockDim.y + threadIdx.y;
    double acc[3] = {0.0, 0.0, 0.0};
    if (xb < d.nx && y < d.ny) {
        const LcRow<XPT, FULL> r(xb, d.nx);
        int xs[XPT];  // a voxel past the ragged end samples the last voxel of the row (never stored)
#pragma unroll
        for (int j = 0; j < XPT; ++j) xs[j] = (FULL || r.ok[j]) ? xb + 32 * j : d.nx - 1;
        const int zb = (int)cz * p.zper, ze = min(d.nz, zb + p.zper);
        const unsigned plane = (unsigned)(d.nx * d.ny);
        const unsigned row0 = (unsigned)((zb * d.ny + y) * d.nx + xb);
        const int zoff = SLAB ? p.zoff : 0;                               // image plane of field plane 0
        const Dims dg = SLAB ? Dims{d.nx, d.ny, p.gnz} : d;               // dims of the images
        const unsigned rowS0 = row0 + (unsigned)zoff * plane;             // the same voxel in the images
        const unsigned dym = y > 0 ? (unsigned)d.nx : 0u, dyp = y < d.ny - 1 ? (unsigned)d.nx : 0u;
        float nux[XPT], nuy[XPT], nuz[XPT];  // field of the plane after the one being issued
        float sm[XPT], sc[XPT];  // centre values of S on planes z-1 and z

        const bool rt = p.zper > 0;  // always true; opaque to the compiler (see above)
        auto load_u = [&](unsigned row) {
            const float *q0 = p.u_in + row, *q1 = p.u_in + (N + row), *q2 = p.u_in + (2 * N + row);
#pragma unroll
            for (int j = 0; j < XPT; ++j) {
                const bool ok = FULL || r.ok[j];
                nux[j] = ok ? __ldg(q0 + 32 * j) : 0.f;
                nuy[j] = ok ? __ldg(q1 + 32 * j) : 0.f;
                nuz[j] = ok ? __ldg(q2 + 32 * j) : 0.f;
            }
        };
        // issue every load of plane z into q (its field is in nu*), then start fetching the field of z + 1
        auto issue = [&](PlaneRegs<VARIANT, XPT>& q, int z) {
            const unsigned row = row0 + (unsigned)(z - zb) * plane;
#pragma unroll
            for (int j = 0; j < XPT; ++j) {
                q.ux[j] = nux[j];
                q.uy[j] = nuy[j];
                q.uz[j] = nuz[j];
            }
            const unsigned rowS = rowS0 + (unsigned)(z - zb) * plane;
            const unsigned dzp = z + zoff < dg.nz - 1 ? plane : 0u;
            if (z + 1 < ze) load_u(row + plane);
            if (rt) {
                load_stencil<XPT, FULL>(p.S, r, rowS, dym, dyp, dzp, q.ss);
                if constexpr (VARIANT == 1) {
                    const float* pg = p.gm2 + rowS;
#pragma unroll
                    for (int j = 0; j < XPT; ++j) q.m2[j] = (FULL || r.ok[j]) ? __ldg(pg + 32 * j) : 0.f;
                }
            }
            if constexpr (!TEX) {
                unsigned o[XPT];
                make_cells<XPT>(dg, xs, y, z + zoff, q.ux, q.uy, q.uz, o, q.fx, q.fy, q.fz);
#pragma unroll
                for (int j = 0; j < XPT; ++j) load_cell(p.M, dg, o[j], q.c[j]);
            }
        };
        auto finish = [&](PlaneRegs<VARIANT, XPT>& q, int z) {
            const unsigned row = row0 + (unsigned)(z - zb) * plane;
            float* o0 = p.u_out + row;
            float* o1 = p.u_out + (N + row);
            float* o2 = p.u_out + (2 * N + row);
            float ssd = 0.f, sf = 0.f, su = 0.f;
            const bool counted = !SLAB || (z >= p.mz0 && z < p.mz1);  // halo planes of a slab belong to a neighbour
#pragma unroll
            for (int j = 0; j < XPT; ++j) {
                float mw;
                if constexpr (TEX)
                    mw = tex3D<float>(p.texM, xs[j] + q.ux[j] + 0.5f, y + q.uy[j] + 0.5f, z + q.uz[j] + 0.5f);
                else
                    mw = lerp_cell(q.c[j], q.fx[j], q.fy[j], q.fz[j]);
                const float gx = 0.5f * (q.ss.xr[j] - q.ss.xl[j]), gy = 0.5f * (q.ss.yp[j] - q.ss.ym[j]),
                            gz = 0.5f * (q.ss.zp[j] - sm[j]);
                const float dd = mw - sc[j];
                const float g2 = fmaf(gx, gx, fmaf(gy, gy, gz * gz));
                sm[j] = sc[j];
                sc[j] = q.ss.zp[j];
                float k;
                if constexpr (VARIANT == 0) {
                    k = guarded_div(dd, fmaf(dd, dd, g2));  // Eq.(1)
                } else {
                    // Eq.(2) needs only |gM0|, the gradient magnitude of the UNWARPED level moving image at the grid
                    // point (reading A4): fixed for the level, so it is read from a precomputed volume
                    const float m2 = q.m2[j];
                    const float num = 4.f * dd * fast_sqrt(g2 * m2);  // |gS| |gM0| with one square root
                    const float den = (fmaf(2.f * dd, dd, g2 + m2)) * (g2 + m2);
                    k = guarded_div(num, den);
                }
                if (FULL || r.ok[j]) {
                    o0[32 * j] = fmaf(-k, gx, q.ux[j]);
                    o1[32 * j] = fmaf(-k, gy, q.uy[j]);
                    o2[32 * j] = fmaf(-k, gz, q.uz[j]);
                    ssd = fmaf(dd, dd, ssd);
                    sf = fmaf(fabsf(k), fast_sqrt(g2), sf);  // |F| = |k| |gS|
                    su += fast_sqrt(fmaf(q.ux[j], q.ux[j], fmaf(q.uy[j], q.uy[j], q.uz[j] * q.uz[j])));
                }
            }
            if (counted) {
                acc[0] += (double)ssd;
                acc[1] += (double)sf;
                acc[2] += (double)su;
            }
        };

        load_u(row0);
        {
            const float *qs = p.S + rowS0, *qsm = p.S + (rowS0 - (zb + zoff > 0 ? plane : 0u));
#pragma unroll
            for (int j = 0; j < XPT; ++j) {
                const bool ok = FULL || r.ok[j];
                sc[j] = ok ? __ldg(qs + 32 * j) : 0.f;
                sm[j] = ok ? __ldg(qsm + 32 * j) : 0.f;
            }
        }
        PlaneRegs<VARIANT, XPT> q;
        for (int z = zb; z < ze; ++z) {
            issue(q, z);
            finish(q, z);
        }
    }
    reduce_metrics(acc, p.sink, b, cz, (unsigned)p.chunks);
}

// |grad M|^2 of a level image (central differences, clamped; O1), once per level for variant 1.
__global__ void __launch_bounds__(256) k_grad_mag2(const float* __restrict__ I, float* __restrict__ out, const Dims d,
                                                   const size_t img_stride, const int z0, const int zn) {
    const int x = blockIdx.x * 64 + threadIdx.x, y = blockIdx.y * 4 + threadIdx.y;
    const int b = blockIdx.z / zn, z = z0 + (int)(blockIdx.z - b * zn);  // blockIdx.z = pair * zn + (z - z0)
    if (x >= d.nx || y >= d.ny) return;
    I += (size_t)b * img_stride;
    out += (size_t)b * nvox(d);
    const unsigned plane = (unsigned)(d.nx * d.ny), i = (unsigned)((z * d.ny + y) * d.nx + x);
    const float gx = 0.5f * (__ldg(I + i + (x < d.nx - 1)) - __ldg(I + i - (x > 0)));
    const float gy = 0.5f * (__ldg(I + i + (y < d.ny - 1 ? d.nx : 0)) - __ldg(I + i - (y > 0 ? d.nx : 0)));
    const float gz = 0.5f * (__ldg(I + i + (z < d.nz - 1 ? plane : 0u)) - __ldg(I + i - (z > 0 ? plane : 0u)));
    out[i] = fmaf(gx, gx, fmaf(gy, gy, gz * gz));
}

// The same for rows that are a whole number of float4s: a thread owns one float4 of a row and marches along z with
// the planes z-1, z, z+1 rolling through registers (one 128-bit load of new data per plane; the y neighbours and the
// two x edge values come from L1).  Same arithmetic per voxel as k_grad_mag2.
__global__ void __launch_bounds__(256) k_grad_mag2_v4(const float* __restrict__ I, float* __restrict__ out, const Dims d,
                                                      const size_t img_stride, const int zper, const int chunks,
                                                      const int z0, const int zn) {
    const int x0 = 4 * (blockIdx.x * 32 + threadIdx.x), y = blockIdx.y * 8 + threadIdx.y;
    const int b = blockIdx.z / chunks, cz = blockIdx.z - b * chunks;
    if (x0 >= d.nx || y >= d.ny) return;
    I += (size_t)b * img_stride;
    out += (size_t)b * nvox(d);
    const unsigned plane = (unsigned)(d.nx * d.ny);
    const int zb = z0 + cz * zper, ze = min(z0 + zn, zb + zper);  // planes [z0, z0 + zn) of the volume
    unsigned i = (unsigned)((zb * d.ny + y) * d.nx + x0);
    const unsigned dym = y > 0 ? (unsigned)d.nx : 0u, dyp = y < d.ny - 1 ? (unsigned)d.nx : 0u;
    const unsigned dxm = x0 > 0 ? 1u : 0u, dxp = x0 + 4 < d.nx ? 4u : 3u;
    float4 lo = __ldg(reinterpret_cast<const float4*>(I + i - (zb > 0 ? plane : 0u)));
    float4 c = __ldg(reinterpret_cast<const float4*>(I + i));
    for (int z = zb; z < ze; ++z, i += plane) {
        const float4 hi = __ldg(reinterpret_cast<const float4*>(I + i + (z < d.nz - 1 ? plane : 0u)));
        const float4 ym = __ldg(reinterpret_cast<const float4*>(I + i - dym)), yp = __ldg(reinterpret_cast<const float4*>(I + i + dyp));
        const float xl = __ldg(I + i - dxm), xr = __ldg(I + i + dxp);
        const float cv[6] = {xl, c.x, c.y, c.z, c.w, xr};
        const float ymv[4] = {ym.x, ym.y, ym.z, ym.w}, ypv[4] = {yp.x, yp.y, yp.z, yp.w};
        const float lov[4] = {lo.x, lo.y, lo.z, lo.w}, hiv[4] = {hi.x, hi.y, hi.z, hi.w};
        float o[4];
#pragma unroll
        for (int e = 0; e < 4; ++e) {
            const float gx = 0.5f * (cv[e + 2] - cv[e]), gy = 0.5f * (ypv[e] - ymv[e]), gz = 0.5f * (hiv[e] - lov[e]);
            o[e] = fmaf(gx, gx, fmaf(gy, gy, gz * gz));
        }
        *reinterpret_cast<float4*>(out + i) = make_float4(o[0], o[1], o[2], o[3]);
        lo = c;
        c = hi;
    }
}

// Pass 1 of variants 2-5 in the same layout: Mw = warp(M, u)  (variant 5 also Sw = warp(S, ub)).
// IC: 0 = variants 2-4; 1 = variant 5 with two stored fields; 2 = variant 5 in the one-field form, where
// u_b = -u_f exactly (pin P10: from a zero start negation commutes with every operation of the iteration),
// so S is warped by the negated registers of u and the second field is never read.
template <int XPT, bool FULL, int IC, bool TEX, bool SLAB = false>
__global__ void __launch_bounds__(BX* BY) k_warp_lc(const KParams p0) {
    const unsigned b = blockIdx.z / (unsigned)p0.chunks, cz = blockIdx.z - b * (unsigned)p0.chunks;
    if (skip_pass(p0.sink, b)) return;
    KParams p = p0;
    select_pair(p, b);
    const Dims d = p.d;
    const unsigned N = (unsigned)nvox(d);
    const int xb = blockIdx.x * (32 * XPT) + threadIdx.x;
    const int y = blockIdx.y * blockDim.y + threadIdx.y;
    if (xb >= d.nx || y >= d.ny) return;
    const LcRow<XPT, FULL> r(xb, d.nx);
    int xs[XPT];
#pragma unroll
    for (int j = 0; j < XPT; ++j) xs[j] = (FULL || r.ok[j]) ? xb + 32 * j : d.nx - 1;
    const int zb = (int)cz * p.zper, ze = min(d.nz, zb + p.zper);
    const unsigned plane = (unsigned)(d.nx * d.ny);
    unsigned row = (unsigned)((zb * d.ny + y) * d.nx + xb);
    const int zoff = SLAB ? p.zoff : 0;                  // image plane of field plane 0 (z-slab form)
    const Dims dg = SLAB ? Dims{d.nx, d.ny, p.gnz} : d;  // dims of the images
    constexpr int NF = IC == 1 ? 2 : 1;  // fields loaded: u (warps M), u_b (warps S)
    constexpr int NW = IC != 0 ? 2 : 1;  // images warped
    float nux[NF][XPT], nuy[NF][XPT], nuz[NF][XPT];  // the field(s) of the next plane (register prefetch)
    auto load_u = [&](unsigned rw) {
#pragma unroll
        for (int f = 0; f < NF; ++f) {
            const float* u = f == 0 ? p.u_in : p.ub_in;
            const float *q0 = u + rw, *q1 = u + (N + rw), *q2 = u + (2 * N + rw);
#pragma unroll
            for (int j = 0; j < XPT; ++j) {
                const bool ok = FULL || r.ok[j];
                nux[f][j] = ok ? __ldg(q0 + 32 * j) : 0.f;
                nuy[f][j] = ok ? __ldg(q1 + 32 * j) : 0.f;
                nuz[f][j] = ok ? __ldg(q2 + 32 * j) : 0.f;
            }
        }
    };
    load_u(row);
    for (int z = zb; z < ze; ++z, row += plane) {
        float ux[NW][XPT], uy[NW][XPT], uz[NW][XPT];
#pragma unroll
        for (int f = 0; f < NW; ++f)
#pragma unroll
            for (int j = 0; j < XPT; ++j) {
                const bool neg = IC == 2 && f == 1;
                ux[f][j] = neg ? -nux[0][j] : nux[f < NF ? f : 0][j];
                uy[f][j] = neg ? -nuy[0][j] : nuy[f < NF ? f : 0][j];
                uz[f][j] = neg ? -nuz[0][j] : nuz[f < NF ? f : 0][j];
            }
        if (z + 1 < ze) load_u(row + plane);
#pragma unroll
        for (int f = 0; f < NW; ++f) {
            const float* I = f == 0 ? p.M : p.S;
            float* out = (f == 0 ? p.Mw : p.Sw) + row;
            float v[XPT];
            if (TEX && f == 0) {
#pragma unroll
                for (int j = 0; j < XPT; ++j)
                    v[j] = tex3D<float>(p.texM, xs[j] + ux[f][j] + 0.5f, y + uy[f][j] + 0.5f, z + uz[f][j] + 0.5f);
            } else {
                unsigned o[XPT];
                float fx[XPT], fy[XPT], fz[XPT], c[XPT][8];
                make_cells<XPT>(dg, xs, y, z + zoff, ux[f], uy[f], uz[f], o, fx, fy, fz);
#pragma unroll
                for (int j = 0; j < XPT; ++j) load_cell(I, dg, o[j], c[j]);
#pragma unroll
                for (int j = 0; j < XPT; ++j) v[j] = lerp_cell(c[j], fx[j], fy[j], fz[j]);
            }
#pragma unroll
            for (int j = 0; j < XPT; ++j)
                if (FULL || r.ok[j]) out[32 * j] = v[j];
        }
    }
}

// ---- variants 2-5, pass 1, generic form (volumes with an axis of length 1) ---------------------
template <int IC>
__global__ void __launch_bounds__(BX* BY) k_warp(const KParams p0) {
    const unsigned b = blockIdx.z / (unsigned)p0.chunks, cz = blockIdx.z - b * (unsigned)p0.chunks;
    if (skip_pass(p0.sink, b)) return;
    KParams p = p0;
    select_pair(p, b);
    const Dims d = p.d;
    const unsigned N = (unsigned)nvox(d);
    const int x = blockIdx.x * BX + threadIdx.x;
    const int y = blockIdx.y * BY + threadIdx.y;
    if (x >= d.nx || y >= d.ny) return;
    for (int z = (int)cz * p.zper; z < min(d.nz, (int)(cz + 1) * p.zper); ++z) {
        const unsigned i = (unsigned)((z * d.ny + y) * d.nx + x);
        const float ux = __ldg(p.u_in + i), uy = __ldg(p.u_in + N + i), uz = __ldg(p.u_in + 2 * N + i);
        p.Mw[i] = trilinear(p.M, d, x, y, z, ux, uy, uz);
        if constexpr (IC == 1)
            p.Sw[i] = trilinear(p.S, d, x, y, z, __ldg(p.ub_in + i), __ldg(p.ub_in + N + i), __ldg(p.ub_in + 2 * N + i));
        if constexpr (IC == 2) p.Sw[i] = trilinear(p.S, d, x, y, z, -ux, -uy, -uz);
    }
}

// ---- variants 2-5, pass 2: gradient of the warped image(s), force, update ---------------------
// ONEF (variant 5 only): the one-field form -- u_b' = u_b + F = -(u - F) = -u' exactly, so it is not stored.
// SLAB: the stencils of the warped images are local to the slab (its outermost planes are halo and are discarded by
// the caller); the static image is a whole volume, indexed in global planes.
template <int VARIANT, int VEC, bool ONEF = false, bool SLAB = false>
__global__ void __launch_bounds__(BX* BY) k_force_active(const KParams p0) {
    const unsigned b = blockIdx.z / (unsigned)p0.chunks, cz = blockIdx.z - b * (unsigned)p0.chunks;
    if (skip_pass(p0.sink, b)) return;
    KParams p = p0;
    select_pair(p, b);
    const Dims d = p.d;
    const unsigned N = (unsigned)nvox(d);
    const int x0 = (blockIdx.x * BX + threadIdx.x) * VEC;
    const int y = blockIdx.y * BY + threadIdx.y;
    const bool active = x0 < d.nx && y < d.ny;
    double acc[3] = {0.0, 0.0, 0.0};
    if (active) {
        for (int z = (int)cz * p.zper; z < min(d.nz, (int)(cz + 1) * p.zper); ++z) {
            const unsigned i0 = (unsigned)((z * d.ny + y) * d.nx + x0);
            const int zoff = SLAB ? p.zoff : 0;
            const Dims dg = SLAB ? Dims{d.nx, d.ny, p.gnz} : d;
            const bool counted = !SLAB || (z >= p.mz0 && z < p.mz1);
            float mw[VEC], ax[VEC], ay[VEC], az[VEC];  // warped moving image and its gradient
            centre_and_gradient<VEC>(p.Mw, d, x0, y, z, mw, ax, ay, az);
            float fx[VEC], fy[VEC], fz[VEC], dd[VEC];
            if constexpr (VARIANT == 2) {  // Eq.(3)
                float s[VEC];
                load_vec<VEC>(p.S + (i0 + (unsigned)zoff * (unsigned)(d.nx * d.ny)), s);
#pragma unroll
                for (int j = 0; j < VEC; ++j) {
                    dd[j] = mw[j] - s[j];
                    const float k = demons_factor(dd[j], 1.f, ax[j], ay[j], az[j]);
                    fx[j] = k * ax[j];
                    fy[j] = k * ay[j];
                    fz[j] = k * az[j];
                }
            } else if constexpr (VARIANT == 3 || VARIANT == 4) {  // Eq.(4), Eq.(5)
                float s[VEC], gx[VEC], gy[VEC], gz[VEC];
                centre_and_gradient<VEC>(p.S, dg, x0, y, z + zoff, s, gx, gy, gz);
                const float a2 = VARIANT == 4 ? p.alpha2 : 1.f;
#pragma unroll
                for (int j = 0; j < VEC; ++j) {
                    dd[j] = mw[j] - s[j];
                    const float k1 = demons_factor(dd[j], a2, gx[j], gy[j], gz[j]);
                    const float k2 = demons_factor(dd[j], a2, ax[j], ay[j], az[j]);
                    fx[j] = fmaf(k1, gx[j], k2 * ax[j]);
                    fy[j] = fmaf(k1, gy[j], k2 * ay[j]);
                    fz[j] = fmaf(k1, gz[j], k2 * az[j]);
                }
            } else {  // Eq.(6): G = grad Mw + grad Sw, d = Mw - Sw
                float sw[VEC], gx[VEC], gy[VEC], gz[VEC];
                centre_and_gradient<VEC>(p.Sw, d, x0, y, z, sw, gx, gy, gz);
#pragma unroll
                for (int j = 0; j < VEC; ++j) {
                    dd[j] = mw[j] - sw[j];
                    const float Gx = ax[j] + gx[j], Gy = ay[j] + gy[j], Gz = az[j] + gz[j];
                    const float k = demons_factor(dd[j], 1.f, Gx, Gy, Gz);
                    fx[j] = k * Gx;
                    fy[j] = k * Gy;
                    fz[j] = k * Gz;
                }
            }
            float ux[VEC], uy[VEC], uz[VEC];
            load_vec<VEC>(p.u_in + i0, ux);
            load_vec<VEC>(p.u_in + N + i0, uy);
            load_vec<VEC>(p.u_in + 2 * N + i0, uz);
            float ssd = 0.f, sf = 0.f, su = 0.f;
#pragma unroll
            for (int j = 0; j < VEC; ++j) {
                ssd = fmaf(dd[j], dd[j], ssd);
                sf += fast_sqrt(fmaf(fx[j], fx[j], fmaf(fy[j], fy[j], fz[j] * fz[j])));
                su += fast_sqrt(fmaf(ux[j], ux[j], fmaf(uy[j], uy[j], uz[j] * uz[j])));
                ux[j] -= fx[j];
                uy[j] -= fy[j];
                uz[j] -= fz[j];
            }
            store_vec<VEC>(p.u_out + i0, ux);
            store_vec<VEC>(p.u_out + N + i0, uy);
            store_vec<VEC>(p.u_out + 2 * N + i0, uz);
            if constexpr (VARIANT == 5 && !ONEF) {  // O4: the static side moves by +F
                load_vec<VEC>(p.ub_in + i0, ux);
                load_vec<VEC>(p.ub_in + N + i0, uy);
                load_vec<VEC>(p.ub_in + 2 * N + i0, uz);
#pragma unroll
                for (int j = 0; j < VEC; ++j) {
                    ux[j] += fx[j];
                    uy[j] += fy[j];
                    uz[j] += fz[j];
                }
                store_vec<VEC>(p.ub_out + i0, ux);
                store_vec<VEC>(p.ub_out + N + i0, uy);
                store_vec<VEC>(p.ub_out + 2 * N + i0, uz);
            }
            if (counted) {
                acc[0] += (double)ssd;
                acc[1] += (double)sf;
                acc[2] += (double)su;
            }
        }
    }
    reduce_metrics(acc, p.sink, b, cz, (unsigned)p.chunks);
}

// out = -in (the backward field of variant 5 on exit from the one-field form)
__global__ void __launch_bounds__(256) k_negate(const float* __restrict__ in, float* __restrict__ out, const size_t n) {
    for (size_t i = (size_t)blockIdx.x * 256 + threadIdx.x; i < n; i += (size_t)gridDim.x * 256) out[i] = -in[i];
}

bool aligned16(const void* p) { return p == nullptr || (reinterpret_cast<uintptr_t>(p) & 15u) == 0; }

constexpr int ZPER = 4;  // planes per block of the generic kernels

// Block shape of a marching kernel: rows per block (4..8 warps) and planes per block, chosen to
// minimise  (waves of blocks) x (rows per block) x (planes per chunk + 2 planes of ring warm-up),
// i.e. the work of the busiest SM.  One wave of long marches beats many short blocks (59 against 65 us
// at 256x256x100), and a wave that fills every slot beats one that leaves SMs half empty: 8-row blocks
// give 256 blocks for 296 slots there, 7-row blocks give exactly 296.  A batch multiplies the blocks of
// every candidate by the number of pairs.
struct Shape {
    int by, zper;
};

template <typename K>
Shape pick_shape(K kernel, int tiles_x, int ny, int nz, int nb, long long max_blocks_per_pair, int by_min, int by_max) {
    Shape best{by_max, nz};
    long long best_cost = -1;
    for (int by = by_max; by >= by_min; --by) {
        int per_sm = 0;
        if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kernel, BX * by, 0) != cudaSuccess || per_sm < 1) {
            cudaGetLastError();
            per_sm = 1;
        }
        const long long slots = (long long)sm_count() * per_sm, xy = (long long)tiles_x * ((ny + by - 1) / by);
        for (int chunks = 1; chunks <= nz; ++chunks) {
            const int zper = (nz + chunks - 1) / chunks;
            const long long per_pair = xy * ((nz + zper - 1) / zper);
            if (per_pair > max_blocks_per_pair) continue;  // more blocks than the metric partials have room for
            if (per_pair * nb > 65535LL * xy) continue;     // gridDim.z limit
            const long long cost = ((per_pair * nb + slots - 1) / slots) * by * per_sm * (zper + 2);
            if (best_cost < 0 || cost < best_cost) {
                best_cost = cost;
                best = Shape{by, zper};
            }
        }
    }
    return best;
}

KParams make_params(const ForceArgs& a) {
    KParams p{};
    p.d = a.d;
    p.alpha2 = a.alpha2;
    p.S = a.S;
    p.M = a.M;
    p.u_in = a.u_in;
    p.u_out = a.u_out;
    p.ub_in = a.ub_in;
    p.ub_out = a.ub_out;
    p.Mw = a.Mw;
    p.Sw = a.Sw;
    p.gm2 = a.variant == 1 ? a.Mw : nullptr;  // variants 0-1 do not materialise Mw: the buffer holds |grad M|^2
    p.sink = a.sink;
    p.texM = a.texM;
    p.img_stride = (unsigned)a.img_stride;
    p.zoff = a.slab ? a.zoff : 0;
    p.gnz = a.slab ? a.gnz : a.d.nz;
    p.mz0 = a.slab ? a.mz0 : 0;
    p.mz1 = a.slab ? a.mz1 : a.d.nz;
    return p;
}

long long blocks_cap(const ForceArgs& a) {
    const long long cap = force_partial_blocks(a.d);
    return a.sink.stride > 0 && a.sink.stride < cap ? a.sink.stride : cap;
}

// The lane-consecutive kernels for the passes that gather; the stencil-only force pass of variants 2-5 is
// float4 per lane when 128-bit access applies.
template <int XPT, bool FULL, bool TEX, int MINB>
int launch_lc(const ForceArgs& a, bool vec4, cudaStream_t st) {
    const int tiles_x = (a.d.nx + 32 * XPT - 1) / (32 * XPT);
    KParams p = make_params(a);
    auto run = [&](auto kernel) {
        const Shape sh = pick_shape(kernel, tiles_x, a.d.ny, a.d.nz, a.nb, blocks_cap(a), 4, BY);
        p.zper = sh.zper;
        p.chunks = (a.d.nz + sh.zper - 1) / sh.zper;
        const dim3 grid(tiles_x, (a.d.ny + sh.by - 1) / sh.by, p.chunks * a.nb);
        if (a.metric_blocks && a.variant <= 1) *a.metric_blocks = (int)(grid.x * grid.y) * p.chunks;
        // The gathered image is re-read by every iteration and is the one stream whose misses sit on the
        // critical path (the gathers): an access-policy window asks L2 to keep it (persisting) while the
        // field streams through.  At 256x256x100 the fused pass goes from 54 to 49.7 us.
        cudaLaunchConfig_t cfg{};
        cfg.gridDim = grid;
        cfg.blockDim = dim3(BX, sh.by);
        cfg.stream = st;
        cudaLaunchAttribute attr[1];
        if (a.l2_bytes > 0) {
            attr[0].id = cudaLaunchAttributeAccessPolicyWindow;
            attr[0].val.accessPolicyWindow.base_ptr = const_cast<void*>(a.l2_ptr);
            attr[0].val.accessPolicyWindow.num_bytes = a.l2_bytes;
            attr[0].val.accessPolicyWindow.hitRatio = a.l2_ratio;
            attr[0].val.accessPolicyWindow.hitProp = cudaAccessPropertyPersisting;
            attr[0].val.accessPolicyWindow.missProp = cudaAccessPropertyStreaming;
            cfg.attrs = attr;
            cfg.numAttrs = 1;
        }
        cudaLaunchKernelEx(&cfg, kernel, p);
    };
    constexpr bool S = !TEX;  // the z-slab instantiations exist for the software sampler only
    if (a.variant == 0) {
        if (a.slab) run(k_force_fixed_lc<0, XPT, FULL, TEX, MINB, false, S>);
        else if (a.nb == 1) run(k_force_fixed_lc<0, XPT, FULL, TEX, MINB, false>);
        else run(k_force_fixed_lc<0, XPT, FULL, TEX, MINB, true>);
        return 1;
    }
    if (a.variant == 1) {
        if (a.slab) run(k_force_fixed_lc<1, XPT, FULL, TEX, MINB, false, S>);
        else if (a.nb == 1) run(k_force_fixed_lc<1, XPT, FULL, TEX, MINB, false>);
        else run(k_force_fixed_lc<1, XPT, FULL, TEX, MINB, true>);
        return 1;
    }
    if (a.slab) {
        if (a.variant == 5 && a.one_field) run(k_warp_lc<XPT, FULL, 2, TEX, S>);
        else if (a.variant == 5) run(k_warp_lc<XPT, FULL, 1, TEX, S>);
        else run(k_warp_lc<XPT, FULL, 0, TEX, S>);
    } else if (a.variant == 5 && a.one_field) run(k_warp_lc<XPT, FULL, 2, TEX>);
    else if (a.variant == 5) run(k_warp_lc<XPT, FULL, 1, TEX>);
    else run(k_warp_lc<XPT, FULL, 0, TEX>);
    if (a.ev_mid) cudaEventRecord(a.ev_mid, st);
    // the stencil pass marches too: same one-wave sizing, 8-row blocks (its float4 tiles are fixed)
    auto run_active = [&](auto kernel) {
        const int vec = vec4 ? 4 : 1;
        const int tx = (a.d.nx + BX * vec - 1) / (BX * vec);
        const Shape sh = pick_shape(kernel, tx, a.d.ny, a.d.nz, a.nb, blocks_cap(a), BY, BY);
        p.zper = sh.zper;
        p.chunks = (a.d.nz + sh.zper - 1) / sh.zper;
        if (a.metric_blocks) *a.metric_blocks = tx * ((a.d.ny + BY - 1) / BY) * p.chunks;
        kernel<<<dim3(tx, (a.d.ny + BY - 1) / BY, p.chunks * a.nb), dim3(BX, BY), 0, st>>>(p);
    };
    if (a.slab) {
        switch (a.variant) {
        case 2: if (vec4) run_active(k_force_active<2, 4, false, true>); else run_active(k_force_active<2, 1, false, true>); break;
        case 3: if (vec4) run_active(k_force_active<3, 4, false, true>); else run_active(k_force_active<3, 1, false, true>); break;
        case 4: if (vec4) run_active(k_force_active<4, 4, false, true>); else run_active(k_force_active<4, 1, false, true>); break;
        case 5:
            if (a.one_field) {
                if (vec4) run_active(k_force_active<5, 4, true, true>); else run_active(k_force_active<5, 1, true, true>);
            } else {
                if (vec4) run_active(k_force_active<5, 4, false, true>); else run_active(k_force_active<5, 1, false, true>);
            }
            break;
        default: return -1;
        }
        return 2;
    }
    switch (a.variant) {
    case 2: if (vec4) run_active(k_force_active<2, 4>); else run_active(k_force_active<2, 1>); break;
    case 3: if (vec4) run_active(k_force_active<3, 4>); else run_active(k_force_active<3, 1>); break;
    case 4: if (vec4) run_active(k_force_active<4, 4>); else run_active(k_force_active<4, 1>); break;
    case 5:
        if (a.one_field) {
            if (vec4) run_active(k_force_active<5, 4, true>); else run_active(k_force_active<5, 1, true>);
        } else {
            if (vec4) run_active(k_force_active<5, 4>); else run_active(k_force_active<5, 1>);
        }
        break;
    default: return -1;
    }
    return 2;
}

// Voxels per lane by row length; 128 registers / 2 blocks per SM for the 128-wide tiles, 80 / 3
// for the narrower ones (the coarse pyramid levels).
template <bool TEX>
int launch_lc_x(const ForceArgs& a, bool vec4, cudaStream_t st) {
    const int xpt = a.d.nx <= 32 ? 1 : a.d.nx <= 64 ? 2 : 4;
    if (a.d.nx % (32 * xpt) == 0) {
        if (xpt == 1) return launch_lc<1, true, TEX, 3>(a, vec4, st);
        if (xpt == 2) return launch_lc<2, true, TEX, 3>(a, vec4, st);
        return launch_lc<4, true, TEX, 2>(a, vec4, st);
    }
    if (xpt == 1) return launch_lc<1, false, TEX, 3>(a, vec4, st);
    if (xpt == 2) return launch_lc<2, false, TEX, 3>(a, vec4, st);
    return launch_lc<4, false, TEX, 2>(a, vec4, st);
}

// Volumes with an axis of length 1: one voxel per thread, ZPER planes per block.
int launch_generic(const ForceArgs& a, cudaStream_t st) {
    KParams p = make_params(a);
    p.zper = ZPER;
    p.chunks = (a.d.nz + ZPER - 1) / ZPER;
    const dim3 block(BX, BY), grid((a.d.nx + BX - 1) / BX, (a.d.ny + BY - 1) / BY, p.chunks * a.nb);
    if (a.metric_blocks) *a.metric_blocks = (int)(grid.x * grid.y) * p.chunks;
    switch (a.variant) {
    case 0: k_force_fixed<0><<<grid, block, 0, st>>>(p); return 1;
    case 1: k_force_fixed<1><<<grid, block, 0, st>>>(p); return 1;
    default: break;
    }
    if (a.variant == 5 && a.one_field) k_warp<2><<<grid, block, 0, st>>>(p);
    else if (a.variant == 5) k_warp<1><<<grid, block, 0, st>>>(p);
    else k_warp<0><<<grid, block, 0, st>>>(p);
    if (a.ev_mid) cudaEventRecord(a.ev_mid, st);
    switch (a.variant) {
    case 2: k_force_active<2, 1><<<grid, block, 0, st>>>(p); break;
    case 3: k_force_active<3, 1><<<grid, block, 0, st>>>(p); break;
    case 4: k_force_active<4, 1><<<grid, block, 0, st>>>(p); break;
    case 5:
        if (a.one_field) k_force_active<5, 1, true><<<grid, block, 0, st>>>(p);
        else k_force_active<5, 1><<<grid, block, 0, st>>>(p);
        break;
    default: return -1;
    }
    return 2;
}

struct DeviceProps {
    int sms = 0;
    size_t window = 0, persist = 0;
    bool known = false;
};

const DeviceProps& device_props() {
    static DeviceProps props[64];
    static std::mutex props_mutex;  // host threads driving different contexts share this table
    std::lock_guard<std::mutex> lock(props_mutex);
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= 64) {
        cudaGetLastError();
        dev = 0;
    }
    DeviceProps& q = props[dev];
    if (!q.known) {
        int v = 0;
        q.sms = cudaDeviceGetAttribute(&v, cudaDevAttrMultiProcessorCount, dev) == cudaSuccess && v > 0 ? v : 148;
        q.window = cudaDeviceGetAttribute(&v, cudaDevAttrMaxAccessPolicyWindowSize, dev) == cudaSuccess && v > 0 ? (size_t)v : 0;
        q.persist = cudaDeviceGetAttribute(&v, cudaDevAttrMaxPersistingL2CacheSize, dev) == cudaSuccess && v > 0 ? (size_t)v : 0;
        cudaGetLastError();
        q.known = true;
    }
    return q;
}

}  // namespace

int sm_count() { return device_props().sms; }
size_t max_policy_window() { return device_props().window; }
size_t max_persisting_l2() { return device_props().persist; }

int force_partial_blocks(const Dims& d) {
    // the largest grid any force kernel uses per pair: 32-voxel tiles, 4-row blocks and single planes
    // (pick_shape takes short marches only on small volumes, where the launch would otherwise not fill the
    // GPU), capped; the generic kernels use 8-row blocks of ZPER planes
    const long long gx = (d.nx + BX - 1) / BX, gy = (d.ny + 3) / 4, gz = d.nz;
    const long long generic = gx * ((d.ny + BY - 1) / BY) * ((d.nz + ZPER - 1) / ZPER);
    long long n = gx * gy * gz;
    if (n > 65536) n = 65536;
    return (int)(n > generic ? n : generic);
}

int launch_grad_mag2(const Dims& d, const float* I, size_t img_stride, float* out, int nb, cudaStream_t st, int z0,
                     int zn) {
    if (zn < 0) zn = d.nz - z0;  // default: every plane
    if (z0 < 0 || zn < 1 || z0 + zn > d.nz) return -1;
    if (d.nx % 4 == 0 && aligned16(I) && aligned16(out) && (nb == 1 || img_stride % 4 == 0)) {
        // enough z chunks for about four blocks per SM
        const long long xy = (long long)((d.nx / 4 + 31) / 32) * ((d.ny + 7) / 8) * nb;
        long long chunks = (4LL * sm_count() + xy - 1) / xy;
        if (chunks > zn) chunks = zn;
        if (chunks < 1) chunks = 1;
        const int zper = (int)((zn + chunks - 1) / chunks);
        chunks = (zn + zper - 1) / zper;
        if (chunks * nb <= 65535) {
            const dim3 grid((d.nx / 4 + 31) / 32, (d.ny + 7) / 8, (unsigned)(chunks * nb));
            k_grad_mag2_v4<<<grid, dim3(32, 8), 0, st>>>(I, out, d, img_stride, zper, (int)chunks, z0, zn);
            return cudaPeekAtLastError() == cudaSuccess ? 1 : -1;
        }
    }
    if ((long long)zn * nb > 65535) return -1;
    const dim3 grid((d.nx + 63) / 64, (d.ny + 3) / 4, zn * nb);
    k_grad_mag2<<<grid, dim3(64, 4), 0, st>>>(I, out, d, img_stride, z0, zn);
    return cudaPeekAtLastError() == cudaSuccess ? 1 : -1;
}

int launch_negate(const float* in, float* out, size_t n, cudaStream_t st) {
    size_t blocks = (n + 255) / 256;
    if (blocks > (size_t)sm_count() * 16) blocks = (size_t)sm_count() * 16;
    k_negate<<<(unsigned)(blocks < 1 ? 1 : blocks), 256, 0, st>>>(in, out, n);
    return cudaPeekAtLastError() == cudaSuccess ? 1 : -1;
}

int launch_metrics_final(const MetricSink& sink, int nb, cudaStream_t st) {
    k_metrics_final<<<nb, 256, 0, st>>>(sink);
    return cudaPeekAtLastError() == cudaSuccess ? 1 : -1;
}

int launch_warp_force(const ForceArgs& a, cudaStream_t st) {
    if (a.nb < 1 || (a.texM != 0 && a.nb != 1)) return -1;
    if (a.slab && (a.nb != 1 || a.texM != 0 || a.d.nx < 2 || a.d.ny < 2 || a.d.nz < 2 || a.gnz < 2)) return -1;
    const bool vec4 = (a.d.nx % 4 == 0) && aligned16(a.S) && aligned16(a.M) && aligned16(a.u_in) &&
                      aligned16(a.u_out) && aligned16(a.ub_in) && aligned16(a.ub_out) && aligned16(a.Mw) &&
                      aligned16(a.Sw) && (a.nb == 1 || (a.img_stride % 4 == 0 && nvox(a.d) % 4 == 0));
    const bool cells_ok = a.d.nx >= 2 && a.d.ny >= 2 && a.d.nz >= 2;  // make_cells needs a 2x2x2 cell
    int n;
    if (!cells_ok) n = launch_generic(a, st);
    else n = a.texM != 0 ? launch_lc_x<true>(a, vec4, st) : launch_lc_x<false>(a, vec4, st);
    if (cudaPeekAtLastError() != cudaSuccess) return -1;
    return n;
}

}  // namespace demons
