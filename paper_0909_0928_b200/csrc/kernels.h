// Host-side launchers of the demons kernels.  Internal to the library (not part of the C ABI).
//
// Batched launches: every launcher takes `nb` pairs laid out back to back -- images [nb][N] (stride
// img_stride floats, so that the S and M of a pair may be interleaved), fields [nb][3][N], warped images
// [nb][N] -- and carries the pair index in the grid, so that small pyramid levels of several independent
// registrations fill the machine with one launch.  nb = 1 is the single-registration case.
#pragma once

#include "common.cuh"

namespace demons {

struct ForceArgs {
    Dims d;
    int variant;
    float alpha2;        // alpha^2 (variant 4; 1 for variant 3)
    int nb;              // pairs in this launch (>= 1)
    size_t img_stride;   // floats between the S (and between the M) of consecutive pairs
    const float* S;      // static image of the level
    const float* M;      // moving image of the level
    const float* u_in;   // [nb][3][N]
    float* u_out;        // [nb][3][N], u_in - F
    const float* ub_in;  // variant 5, two-field form; nullptr with one_field
    float* ub_out;       // variant 5, two-field form; nullptr with one_field
    int one_field;       // variant 5 with u_b = -u_f held implicitly (pin P10): only u is read and written
    float* Mw;           // workspace, [nb][N]: warped moving image (variants 2-5); |grad M|^2 for variant 1
    float* Sw;           // workspace, [nb][N]: warped static image (variant 5)
    MetricSink sink;
    cudaTextureObject_t texM;  // 0 = software trilinear (default); nb must be 1 otherwise
    cudaEvent_t ev_mid;        // nullable: recorded between the warp and the force kernel (profiling)
    int* metric_blocks;        // nullable out: block partials per pair the pass wrote (sink.nblocks of k_metrics_final)
    // z-slab form (one rank of a z-slab decomposition): d is the local slab (fields, warped images), which starts at
    // plane zoff of the images; S and M are whole volumes of gnz planes; planes [mz0, mz1) of the slab count in the
    // metrics.  nb must be 1, texM 0.
    int slab, zoff, gnz, mz0, mz1;
    // L2 access-policy window of the gathering kernels (persisting); l2_bytes == 0: none
    const void* l2_ptr;
    size_t l2_bytes;
    float l2_ratio;
};

// S1-S4 (+S6).  Returns the number of kernels launched, or -1 with cudaGetLastError() set.
int launch_warp_force(const ForceArgs& a, cudaStream_t stream);

// Deferred metrics (sink.defer = 1 in the ForceArgs of the pass before): sums the block partials of every pair of the
// launch (sink.nblocks of them per pair) and publishes them (row, stopping rule).  One launch, nb blocks.
int launch_metrics_final(const MetricSink& sink, int nb, cudaStream_t stream);

// Variant 1, once per level (and per standalone demons_warp_force call): out <- |grad I|^2, [nb][N], which
// launch_warp_force then reads instead of stencilling M (Eq.(2) uses only the magnitude of grad M0).
// Planes [z0, z0 + zn) of the volume only (zn < 0: all of them).
int launch_grad_mag2(const Dims& d, const float* I, size_t img_stride, float* out, int nb, cudaStream_t stream,
                     int z0 = 0, int zn = -1);

// out[nb][3][N] = -in: the backward field of variant 5 on exit from the one-field form (u_b = -u_f, P10).
int launch_negate(const float* in, float* out, size_t n, cudaStream_t stream);

// Number of per-block partial slots launch_warp_force may use per pair for dims d.
int force_partial_blocks(const Dims& d);

struct SmoothArgs {
    Dims d;
    const float* in;     // [ncomp][N]
    float* out;          // [ncomp][N]
    float* tmp;          // workspace [pairs][N] (separable fallback only)
    int ncomp;           // components in this launch (pairs x components per pair)
    int comps_per_pair;  // component c belongs to pair c / comps_per_pair
    int R;               // radius
    float w[33];         // w[k], k = 0..R
    const Control* ctl;  // nullable, [pairs]: ctl[pair].stop_smooth != 0 = do nothing for that pair
    int force_generic;   // 1 = always use the three separable passes
    int ascending;       // 1 = the fused kernel marches z upwards (default 0: downwards, see smooth_tma.cu)
};
int launch_smooth(const SmoothArgs& a, cudaStream_t stream);

// images [nb][N_fine] (stride in_stride) -> [nb][N_coarse] (stride out_stride)
int launch_restrict(const Dims& fine, const float* in, size_t in_stride, float* out, size_t out_stride, int nb,
                    cudaStream_t stream);
// fields [nb][3][N_coarse] -> [nb][3][N_fine]
int launch_prolong(const Dims& coarse, const float* uc, const Dims& fine, float* uf, int nb, cudaStream_t stream);

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

// Stores `msg` as this thread's demons_last_error() text (for entry points that live outside demons_api.cu).
void set_last_error(const char* msg);

// Per-device properties, cached per device ordinal (a process may drive several devices).
int sm_count();
size_t max_policy_window();
size_t max_persisting_l2();

}  // namespace demons
