// Host-side launchers of the demons kernels.  Internal to the library (not part of the C ABI).
#pragma once

#include "common.cuh"

namespace demons {

struct ForceArgs {
    Dims d;
    int variant;
    float alpha2;        // alpha^2 (variant 4; 1 for variant 3)
    const float* S;      // static image of the level
    const float* M;      // moving image of the level
    const float* u_in;   // [3][N]
    float* u_out;        // [3][N], u_in - F
    const float* ub_in;  // variant 5
    float* ub_out;       // variant 5
    float* Mw;           // workspace, [N]: warped moving image (variants 2-5)
    float* Sw;           // workspace, [N]: warped static image (variant 5)
    MetricSink sink;
    cudaTextureObject_t texM;  // 0 = software trilinear (default)
    cudaEvent_t ev_mid;        // nullable: recorded between the warp and the force kernel (profiling)
    int zper;                  // > 0: planes per block (tuning); 0 = default
    int tune;                  // kernel-layout selector (tuning experiments; 0 = default)
    size_t l2_persist_bytes;   // > 0: the gathering kernels ask L2 to keep up to this many bytes of M resident
    int force_scalar;          // 1 = take the one-voxel-per-thread kernels even when 128-bit access applies
};

// True when the moving image starts right behind the static one (at most one alignment gap): one
// L2 access-policy window can then cover both.
inline bool images_adjacent(const float* S, const float* M, size_t n) {
    return S != nullptr && M > S && (size_t)((const char*)M - (const char*)S) <= n * sizeof(float) + 4096;
}

// S1-S4 (+S6).  Returns the number of kernels launched, or -1 with cudaGetLastError() set.
int launch_warp_force(const ForceArgs& a, cudaStream_t stream);

// Variant 1, once per level (and per standalone demons_warp_force call): a.Mw <- |grad M|^2, which
// launch_warp_force then reads instead of stencilling M (Eq.(2) uses only the magnitude of grad M0).
int launch_grad_mag2(const Dims& d, const float* I, float* out, cudaStream_t stream);

// Number of per-block partial slots launch_warp_force may use for dims d.
int force_partial_blocks(const Dims& d);

struct SmoothArgs {
    Dims d;
    const float* in;   // [ncomp][N]
    float* out;        // [ncomp][N]
    float* tmp;        // workspace [N] (separable fallback only)
    int ncomp;
    int R;             // radius
    float w[33];       // w[k], k = 0..R
    const int* skip;   // nullable device flag: non-zero = do nothing
    int force_generic; // 1 = always use the three separable passes
    int zc_override;   // > 0: planes per CTA of the fused kernel (tuning)
    int no_tma;        // 1 = skip the TMA kernel (use the LDG-fed fused kernel)
    int tune;          // kernel-configuration selector (tuning experiments; 0 = default)
    int ascending;     // 1 = the fused kernel marches z upwards (default 0: downwards, see smooth_tma.cu)
};
int launch_smooth(const SmoothArgs& a, cudaStream_t stream);

int launch_restrict(const Dims& fine, const float* in, float* out, cudaStream_t stream);
int launch_prolong(const Dims& coarse, const float* uc, const Dims& fine, float* uf, cudaStream_t stream);

struct ReduceScratch {
    double* partials;
    unsigned int* ticket;
    int stride;
};
int launch_ssd(const Dims& d, const float* S, const float* M, const float* u, const float* ub,
               double* out, const ReduceScratch& rs, cudaStream_t stream);
int launch_ic_error(const Dims& d, const float* uf, const float* ub, double* out,
                    const ReduceScratch& rs, cudaStream_t stream);
int launch_cc(const Dims& d, const float* S, const float* M, const float* u, const float* ub, double* out,
              const ReduceScratch& rs, cudaStream_t stream);
int launch_point_error(const Dims& d, const float spacing[3], const float* u, int n, const float* points,
                       const float* expect, double* err, cudaStream_t stream);

}  // namespace demons
