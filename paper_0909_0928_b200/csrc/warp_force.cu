// S1-S4 and S6 of the demons hot path: trilinear warp, central-difference gradients, the per-voxel
// force of Eq.(1)-(6), the additive update u' = u - F and the three metrics of
// PAPER.md L145, hand-written for sm_100a.
//
// Variants 0-1 (gradients of the fixed level images only): ONE kernel -- the warped intensity
// lives in a register, grad S (and grad M0) are recomputed from a 6-point stencil whose re-reads
// hit L1/L2, so the compulsory HBM traffic is u (12 B) + S (4 B) + M (4 B) in, u' (12 B) out.
// Variants 2-5 need the gradient of the WARPED image (reading A8), i.e. the warped values of the
// six neighbours: the warped image is materialised once (k_warp) and then stencilled
// (k_force_active) instead of gathering 7x per voxel, which would be instruction-bound.
#include "kernels.h"

namespace demons {

namespace {

constexpr int BX = 32;  // threads along x (each owns VEC consecutive voxels)
constexpr int BY = 8;   // threads along y

__device__ __forceinline__ bool skip_pass(const MetricSink& s) {
    if (s.stop_force != nullptr && *reinterpret_cast<volatile int*>(s.stop_force) != 0) {
        if (s.stop_smooth != nullptr) *s.stop_smooth = 1;
        return true;
    }
    return false;
}

// Thread 0 of the last block: write {SSD, sum|F|, sum|u|}, advance the row, apply the stopping
// rule  l_n = sum|F| / sum|u|;  stop after the first n >= 10 with |l_n - l_{n-10}| <= eps.
__device__ __forceinline__ void publish_metrics(const double (&v)[3], const MetricSink& s) {
    const unsigned int row = s.row_counter ? *s.row_counter : 0u;
    double* o = s.out + 3 * (size_t)row;
    o[0] = v[0];
    o[1] = v[1];
    o[2] = v[2];
    if (s.row_counter) *s.row_counter = row + 1u;
    if (s.level_iter) {
        const unsigned int n = *s.level_iter;
        const int valid = v[2] > 0.0;
        const double l = valid ? v[1] / v[2] : 0.0;
        s.lhist[n & (LHIST - 1)] = l;
        s.lvalid[n & (LHIST - 1)] = valid;
        if (s.eps > 0.0 && n >= 10u && valid && s.lvalid[(n - 10u) & (LHIST - 1)] &&
            fabs(l - s.lhist[(n - 10u) & (LHIST - 1)]) <= s.eps)
            *s.stop_force = 1;
        *s.level_iter = n + 1u;
    }
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
    MetricSink sink;
    cudaTextureObject_t texM;
    int zper;  // consecutive planes per block
};

// ---- variants 0, 1: fused warp + gradient + force + update ------------------------------------
template <int VARIANT, int VEC, bool TEX>
__global__ void __launch_bounds__(BX* BY) k_force_fixed(const KParams p) {
    if (skip_pass(p.sink)) return;
    const Dims d = p.d;
    const unsigned N = (unsigned)nvox(d);
    const int x0 = (blockIdx.x * BX + threadIdx.x) * VEC;
    const int y = blockIdx.y * BY + threadIdx.y;
    const bool active = x0 < d.nx && y < d.ny;
    double acc[3] = {0.0, 0.0, 0.0};
    if (active) {
        // the field of the next plane is fetched while this plane's gathers and arithmetic run
        const int zb = blockIdx.z * p.zper, ze = min(d.nz, zb + p.zper);
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
            for (int j = 0; j < VEC; ++j) {
                if constexpr (TEX)
                    mw[j] = tex3D<float>(p.texM, x0 + j + ux[j] + 0.5f, y + uy[j] + 0.5f, z + uz[j] + 0.5f);
                else
                    mw[j] = trilinear(p.M, d, x0 + j, y, z, ux[j], uy[j], uz[j]);
            }
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
                    const float num = 4.f * dd * fast_sqrt(s2) * fast_sqrt(m2);
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
    if (p.sink.out != nullptr) {
        if (block_reduce_publish<3>(acc, p.sink.partials, p.sink.stride, p.sink.ticket))
            publish_metrics(acc, p.sink);
    }
}

// ---- variants 2-5, pass 1: Mw = warp(M, u)  (variant 5 also Sw = warp(S, ub)) -----------------
template <int VEC, bool IC, bool TEX>
__global__ void __launch_bounds__(BX* BY) k_warp(const KParams p) {
    if (skip_pass(p.sink)) return;
    const Dims d = p.d;
    const unsigned N = (unsigned)nvox(d);
    const int x0 = (blockIdx.x * BX + threadIdx.x) * VEC;
    const int y = blockIdx.y * BY + threadIdx.y;
    if (x0 >= d.nx || y >= d.ny) return;
    for (int z = blockIdx.z * p.zper; z < min(d.nz, (int)(blockIdx.z + 1) * p.zper); ++z) {
        const unsigned i0 = (unsigned)((z * d.ny + y) * d.nx + x0);
        float ux[VEC], uy[VEC], uz[VEC], o[VEC];
        load_vec<VEC>(p.u_in + i0, ux);
        load_vec<VEC>(p.u_in + N + i0, uy);
        load_vec<VEC>(p.u_in + 2 * N + i0, uz);
#pragma unroll
        for (int j = 0; j < VEC; ++j) {
            if constexpr (TEX)
                o[j] = tex3D<float>(p.texM, x0 + j + ux[j] + 0.5f, y + uy[j] + 0.5f, z + uz[j] + 0.5f);
            else
                o[j] = trilinear(p.M, d, x0 + j, y, z, ux[j], uy[j], uz[j]);
        }
        store_vec<VEC>(p.Mw + i0, o);
        if constexpr (IC) {
            load_vec<VEC>(p.ub_in + i0, ux);
            load_vec<VEC>(p.ub_in + N + i0, uy);
            load_vec<VEC>(p.ub_in + 2 * N + i0, uz);
#pragma unroll
            for (int j = 0; j < VEC; ++j) o[j] = trilinear(p.S, d, x0 + j, y, z, ux[j], uy[j], uz[j]);
            store_vec<VEC>(p.Sw + i0, o);
        }
    }
}

// ---- variants 2-5, pass 2: gradient of the warped image(s), force, update ---------------------
template <int VARIANT, int VEC>
__global__ void __launch_bounds__(BX* BY) k_force_active(const KParams p) {
    if (skip_pass(p.sink)) return;
    const Dims d = p.d;
    const unsigned N = (unsigned)nvox(d);
    const int x0 = (blockIdx.x * BX + threadIdx.x) * VEC;
    const int y = blockIdx.y * BY + threadIdx.y;
    const bool active = x0 < d.nx && y < d.ny;
    double acc[3] = {0.0, 0.0, 0.0};
    if (active) {
        for (int z = blockIdx.z * p.zper; z < min(d.nz, (int)(blockIdx.z + 1) * p.zper); ++z) {
            const unsigned i0 = (unsigned)((z * d.ny + y) * d.nx + x0);
            float mw[VEC], ax[VEC], ay[VEC], az[VEC];  // warped moving image and its gradient
            centre_and_gradient<VEC>(p.Mw, d, x0, y, z, mw, ax, ay, az);
            float fx[VEC], fy[VEC], fz[VEC], dd[VEC];
            if constexpr (VARIANT == 2) {  // Eq.(3)
                float s[VEC];
                load_vec<VEC>(p.S + i0, s);
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
                centre_and_gradient<VEC>(p.S, d, x0, y, z, s, gx, gy, gz);
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
            if constexpr (VARIANT == 5) {  // O4: the static side moves by +F
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
            acc[0] += (double)ssd;
            acc[1] += (double)sf;
            acc[2] += (double)su;
        }
    }
    if (p.sink.out != nullptr) {
        if (block_reduce_publish<3>(acc, p.sink.partials, p.sink.stride, p.sink.ticket))
            publish_metrics(acc, p.sink);
    }
}

bool aligned16(const void* p) { return p == nullptr || (reinterpret_cast<uintptr_t>(p) & 15u) == 0; }

constexpr int ZPER = 4;  // planes per block: amortises the block reduction, keeps z neighbours in L1

dim3 force_grid(const Dims& d, int vec, int zper = ZPER) {
    const int gx = (d.nx + BX * vec - 1) / (BX * vec);
    const int gy = (d.ny + BY - 1) / BY;
    const int gz = (d.nz + zper - 1) / zper;
    return dim3(gx, gy, gz);
}

template <int VEC, bool TEX>
int launch_t(const ForceArgs& a, const KParams& p, cudaStream_t st) {
    const dim3 block(BX, BY);
    const dim3 grid = force_grid(a.d, VEC, p.zper);
    switch (a.variant) {
    case 0: k_force_fixed<0, VEC, TEX><<<grid, block, 0, st>>>(p); return 1;
    case 1: k_force_fixed<1, VEC, TEX><<<grid, block, 0, st>>>(p); return 1;
    case 2:
        k_warp<VEC, false, TEX><<<grid, block, 0, st>>>(p);
        if (a.ev_mid) cudaEventRecord(a.ev_mid, st);
        k_force_active<2, VEC><<<grid, block, 0, st>>>(p);
        return 2;
    case 3:
        k_warp<VEC, false, TEX><<<grid, block, 0, st>>>(p);
        if (a.ev_mid) cudaEventRecord(a.ev_mid, st);
        k_force_active<3, VEC><<<grid, block, 0, st>>>(p);
        return 2;
    case 4:
        k_warp<VEC, false, TEX><<<grid, block, 0, st>>>(p);
        if (a.ev_mid) cudaEventRecord(a.ev_mid, st);
        k_force_active<4, VEC><<<grid, block, 0, st>>>(p);
        return 2;
    case 5:
        k_warp<VEC, true, TEX><<<grid, block, 0, st>>>(p);
        if (a.ev_mid) cudaEventRecord(a.ev_mid, st);
        k_force_active<5, VEC><<<grid, block, 0, st>>>(p);
        return 2;
    default: return -1;
    }
}

}  // namespace

int force_partial_blocks(const Dims& d) {
    // the scalar grid is the larger of the two
    const dim3 g = force_grid(d, 1);
    return (int)(g.x * g.y * g.z);
}

int launch_warp_force(const ForceArgs& a, cudaStream_t st) {
    KParams p;
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
    p.sink = a.sink;
    p.texM = a.texM;
    // planes per block: at least ZPER (never more blocks than force_partial_blocks() promised),
    // more on large volumes so that ~1800 blocks remain (L1 reuse along z, fewer block reductions)
    {
        const dim3 g = force_grid(a.d, 1, 1);
        const long long per_plane4 = (long long)((a.d.nx + BX * 4 - 1) / (BX * 4)) * g.y;
        int zper = (int)((per_plane4 * a.d.nz + 1799) / 1800);
        if (zper < ZPER) zper = ZPER;
        if (zper > 32) zper = 32;
        p.zper = a.zper >= ZPER ? a.zper : zper;
    }
    const bool vec4 = !a.force_scalar && (a.d.nx % 4 == 0) && aligned16(a.S) && aligned16(a.M) && aligned16(a.u_in) &&
                      aligned16(a.u_out) && aligned16(a.ub_in) && aligned16(a.ub_out) &&
                      aligned16(a.Mw) && aligned16(a.Sw);
    int n;
    if (a.texM != 0)
        n = vec4 ? launch_t<4, true>(a, p, st) : launch_t<1, true>(a, p, st);
    else
        n = vec4 ? launch_t<4, false>(a, p, st) : launch_t<1, false>(a, p, st);
    if (cudaPeekAtLastError() != cudaSuccess) return -1;
    return n;
}

}  // namespace demons
