/* include/demons.h -- C ABI of the B200-native demons deformable-registration library.
 *
 * Method: Gu et al., "Implementation and evaluation of various demons deformable image
 * registration algorithms on GPU" (arxiv/paper_0909_0928).  "PAPER.md L<n>" below is line n of
 * the paper text; "reading Xn" refers to the ambiguity ledger in DESIGN.md.
 *
 * Conventions shared by every entry point
 * ---------------------------------------
 *  - All d_* pointers are DEVICE pointers (CUDA global memory of the current device), all h_*
 *    pointers are HOST pointers.  The library never allocates device memory: the caller owns
 *    every buffer and the workspace (demons_set_workspace), and they must stay alive until the
 *    work enqueued on `stream` has completed.
 *  - dims = {nx, ny, nz}.  A scalar volume is float32, flat index x + nx*(y + ny*z)
 *    (Sec. 2.5: "x as rows, y as columns, z as frames" -- x is unit stride).
 *  - A displacement field is float32, planar: component c (0 = x, 1 = y, 2 = z) starts at
 *    base + c*nx*ny*nz.  Units are voxels of the level the field lives on (reading C3).
 *  - Direction (reading C1): warp(I,u)(x) = trilinear(I, x + u(x)); the update is u <- u - F
 *    with F exactly as printed in Eq.(1)-(6), d = Mw - S.
 *  - `stream` is a cudaStream_t passed as void* (NULL = the legacy default stream).  Calls
 *    enqueue work on it and return without synchronising unless stated otherwise.
 *  - Every function returns a DEMONS_* status; nothing throws, aborts or exits.  On failure
 *    demons_last_error() returns a thread-local description.  There is no CPU fallback: with no
 *    usable CUDA device every compute entry point returns DEMONS_E_CUDA.
 *  - ONE DEVICE-WIDE SIDE EFFECT, on by default: with the "l2_persist" option (default 1) the first call that gathers
 *    from a moving image raises the device limit cudaLimitPersistingL2CacheSize to that image's size (other users of
 *    the device see a smaller non-persisting L2 while lines are pinned); demons_destroy resets the persisting lines
 *    and restores the limit it found.  demons_set_option(ctx, "l2_persist", 0) before the first compute call leaves
 *    the device untouched (the fused pass is then ~10 % slower at 256x256x100).  Details under demons_set_option.
 *  - Host threads: entry points may be called from several host threads as long as each context is used by one
 *    thread at a time; the library's per-device one-time set-up is synchronised, the error string is per thread.
 *  - Buffers that are 16-byte aligned with nx % 4 == 0 take the fast kernels (TMA-fed smoothing, 128-bit
 *    rows in the stencil pass; the gathering passes use lane-consecutive 32-bit accesses, one 128-byte
 *    line per warp); anything else takes scalar kernels with identical results.
 */
#ifndef DEMONS_H
#define DEMONS_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct demons_ctx demons_ctx;

/* Variant k = the paper's "Method k+1" (Table 2). */
enum {
    DEMONS_PASSIVE = 0,            /* Eq.(1):  d gS / (d^2 + |gS|^2)                       */
    DEMONS_EVOLVED_PASSIVE = 1,    /* Eq.(2), PAPER.md L64 (readings A3, A4), gS and gM0 fixed           */
    DEMONS_ACTIVE = 2,             /* Eq.(3):  d gMw / (d^2 + |gMw|^2), gMw = grad(warp M) */
    DEMONS_DOUBLE = 3,             /* Eq.(4):  Eq.(1) + Eq.(3)                             */
    DEMONS_ADJUSTED_DOUBLE = 4,    /* Eq.(5), PAPER.md L93 (reading A5): alpha^2 d^2 in both denominators*/
    DEMONS_INVERSE_CONSISTENT = 5  /* Eq.(6): G = gMw + gSw, d = Mw - Sw                  */
};

enum {
    DEMONS_OK = 0,
    DEMONS_E_ARG = -1,         /* NULL / out-of-range / inconsistent argument                 */
    DEMONS_E_CUDA = -2,        /* a CUDA runtime call failed (no device, launch failure, ...) */
    DEMONS_E_WORKSPACE = -3,   /* workspace missing or too small for this call                */
    DEMONS_E_UNSUPPORTED = -4  /* valid request this build cannot serve (e.g. sigma too large) */
};

/* Largest Gaussian radius R = ceil(3 sigma) the smoothing kernels accept. */
#define DEMONS_MAX_RADIUS 32
/* Largest number of pyramid levels. */
#define DEMONS_MAX_LEVELS 8
/* Capacity of the per-iteration statistics buffer inside the workspace (rows of 3 doubles, per pair). */
#define DEMONS_MAX_STATS_ROWS 16384
/* Largest batch of demons_register_batch. */
#define DEMONS_MAX_BATCH 64

/* ---- context ---------------------------------------------------------------------------
 * demons_create: host-only, no CUDA call.  dims = finest-level volume size (each >= 1),
 * spacing in mm (> 0; stored, used only by callers that report errors in mm, reading C3),
 * variant in [0,5], alpha > 0 (used by variant 4 only), sigma > 0 in voxels
 * with ceil(3 sigma) <= DEMONS_MAX_RADIUS ("Gaussian filter of unit standard deviation",
 * PAPER.md L175; sigma is an argument per BASELINE.json north_star).
 * The context holds host-side state only (parameters, workspace partition, cached CUDA graphs). */
int demons_create(demons_ctx** out, const int dims[3], const float spacing[3], int variant,
                  float alpha, float sigma);
void demons_destroy(demons_ctx* ctx);

/* Bytes of device workspace needed by every entry point below for volumes up to the context's
 * dims and a pyramid of `levels` (1..DEMONS_MAX_LEVELS).  Includes the device staging buffers
 * of demons_register_host.  Returns 0 on bad arguments. */
size_t demons_workspace_bytes(const demons_ctx* ctx, int levels);
/* The same for demons_register_batch with up to `nbatch` pairs (1..DEMONS_MAX_BATCH); a workspace of this
 * size also serves every single-registration entry point. */
size_t demons_workspace_bytes_batch(const demons_ctx* ctx, int levels, int nbatch);
/* d_ws: device pointer, 256-byte aligned, `bytes` >= demons_workspace_bytes(ctx, levels) for
 * the `levels` later passed to demons_register.  The library zeroes its counters on `stream`
 * lazily at first use.  The caller keeps ownership. */
int demons_set_workspace(demons_ctx* ctx, void* d_ws, size_t bytes);

/* Pyramid geometry (reading A12 / O6): level 0 = finest = ctx dims, level l+1 = ceil(level l / 2). */
int demons_level_dims(const demons_ctx* ctx, int level, int out_dims[3]);

/* Number of kernel launches this context has enqueued so far (graph replays count their nodes). */
long long demons_launch_count(const demons_ctx* ctx);

/* "profile" option: after a demons_register call made with the option on, the summed device time
 * (ms, CUDA events on the caller's stream) and the number of timed groups per kernel class:
 * [0] force kernels (fused warp+force+update, or the force pass of variants 2-5), [1] the warp
 * pass of variants 2-5, [2] smoothing, [3] pyramid (restrict + prolong).
 * With "profile" = 2 the registration keeps replaying its level graphs, and ONE iteration in the middle of every
 * replayed chunk of 20 carries three event-record nodes (before the force kernel(s), between force and smoothing,
 * after the smoothing kernel(s)): [0] is then the time from the first to the second (variants 2-5: warp pass and
 * force pass together), [2] from the second to the third, each summed over the replays (groups = replays); [1] is
 * an EMPTY bracket in this mode -- a fourth record node directly behind the third -- i.e. what one record node adds
 * to each of the two intervals; the host reads the events after every replay (one stream synchronise per 20 iterations), [3] is not
 * timed.  These are the durations of the kernels as the run executes them -- warm L2, neighbours in flight. */
int demons_get_profile(const demons_ctx* ctx, double h_ms[4], long long h_launch_groups[4]);

/* Named integer options.  "graphs" (default 1): replay the per-level iteration through a CUDA
 * graph.  "texture" (default 0): S9, sample the moving image through the texture unit with
 * hardware linear filtering (PAPER.md L181 reports its precision as insufficient; measured
 * option only -- fails parity by design).  "generic_smooth" (default 0): always use
 * the three separable smoothing passes instead of the fused kernel.  "profile" (default 0): 1 = time
 * every kernel class with events inside demons_register (disables graphs, adds a final
 * synchronise; see demons_get_profile); 2 = time one iteration per replayed graph chunk from inside the graph.  "zero_start" (default 0): a single-level registration starts
 * from a zero field set on the device; d_u / h_u (and u_back) are then outputs only and
 * demons_register_host does not upload them.  "l2_persist" (default 1): the kernels that gather from the
 * moving image launch with an access-policy window that asks L2 to keep that image resident
 * (persisting) while the field streams through; for this the library RAISES the device-wide limit
 * cudaLimitPersistingL2CacheSize to the size of the moving image on the first call that needs it (images
 * larger than the device's maximum set-aside are left alone), and demons_destroy resets the persisting
 * lines (cudaCtxResetPersistingL2Cache) and restores the limit it found.  If d_moving starts directly behind
 * d_static in memory (one allocation holding both, as the workspace's own pyramid levels and host-staging
 * buffers do) the window covers the static image as well.  Set the option to 0 to leave the device limit
 * alone.  "ic_one_field" (default 1): variant 5 started from zero fields (every multi-level call, and single
 * levels under "zero_start") iterates on the forward field alone and writes u_back = -u once on exit; the two
 * fields are exact negatives of each other at every iteration (negation commutes with every operation of the
 * iteration), so the result is bit-identical to iterating on both (0 = always iterate on both).
 * Unknown name -> DEMONS_E_ARG. */
int demons_set_option(demons_ctx* ctx, const char* name, int value);

/* ---- full registration (PAPER.md L123-125 multi-scale, L145 stopping rule; O9/O10) ---------
 * d_static, d_moving: finest-level volumes.  d_u: field of the moving image, [3][N];
 * levels == 1: in = initial field, out = result; levels > 1: ignored on input (the coarsest
 * level starts from zero), out = result.  d_u_back: variant 5 only (the field applied to the
 * static image), same rule; must be NULL for the other variants.
 * h_iters_per_level[levels], coarse -> fine, each >= 0, sum <= DEMONS_MAX_STATS_ROWS.
 * eps <= 0: run exactly the given counts.  eps > 0: per level, stop after the first iteration
 * n >= 10 with |l_n - l_{n-10}| <= eps, l_n = sum|F| / sum|u| (reading A13);
 * tested on the device, no host round trip.
 * h_stats (nullable): [sum iters][3] doubles = {SSD, sum|F|_2, sum|u|_2} per executed iteration
 * in execution order, evaluated with the state before that iteration's update (reading O8); rows
 * of skipped iterations are zero.  h_iters_done (nullable): [levels] iterations executed.
 * If h_stats or h_iters_done is non-NULL the call synchronises `stream` before returning. */
int demons_register(demons_ctx* ctx, const float* d_static, const float* d_moving, float* d_u,
                    float* d_u_back, int levels, const int* h_iters_per_level, double eps,
                    double* h_stats, int* h_iters_done, void* stream);

/* A batch of `nbatch` INDEPENDENT registrations of equally sized pairs in one call (many
 * registrations per patient course; Table 2: five cases x six methods).  Layouts: d_static and
 * d_moving [nbatch][N], d_u (and d_u_back) [nbatch][3][N], contiguous; h_stats (nullable)
 * [nbatch][sum iters][3]; h_iters_done (nullable) [nbatch][levels].  Pyramid levels too small to fill the
 * GPU run several pairs per kernel launch (the pair index rides in the grid); large levels run pair by
 * pair, so that one pair's images stay resident in L2.  Each pair stops on its own when eps > 0.  The
 * field of every pair is bit-identical to what demons_register gives for that pair alone; the statistics
 * agree to rounding (the block partition of the reduction differs).  Needs a workspace of
 * demons_workspace_bytes_batch(ctx, levels, nbatch).  The "texture" option serves nbatch == 1 only. */
int demons_register_batch(demons_ctx* ctx, int nbatch, const float* d_static, const float* d_moving, float* d_u,
                          float* d_u_back, int levels, const int* h_iters_per_level, double eps,
                          double* h_stats, int* h_iters_done, void* stream);

/* Same as demons_register, with HOST buffers: copies h_static/h_moving (and, for levels == 1, h_u / h_u_back) to
 * staging buffers inside the workspace, registers, copies the field(s) back, synchronises.
 * Pinned host memory makes the copies asynchronous on `stream`; pageable memory also works. */
int demons_register_host(demons_ctx* ctx, const float* h_static, const float* h_moving, float* h_u,
                         float* h_u_back, int levels, const int* h_iters_per_level, double eps,
                         double* h_stats, int* h_iters_done, void* stream);

/* A QUEUE of n registrations of equally sized pairs from host buffers (the paper's use case: many registrations per
 * patient course), run one after another on `stream` exactly as demons_register_host runs each of them,
 * with two staging slots in the workspace: the upload of pair k + 1 and the download of field k - 1 ride on two internal
 * streams beside registration k, so that the PCIe transfers (8 B/voxel up, 12 B/voxel down per registration) cost no
 * GPU time except for the first upload and the last download.  h_static, h_moving, h_u (and h_u_back, variant 5; NULL
 * otherwise) are arrays of n HOST pointers; the same buffer may appear several times (downloads are ordered).  Pinned
 * host memory is what makes the overlap possible; pageable memory works and serialises.  h_stats (nullable)
 * [n][sum iters][3], h_iters_done (nullable) [n][levels].  Results are bit-identical to n demons_register_host calls.
 * Needs a workspace of demons_workspace_bytes_queue(ctx, levels) (the single-registration workspace plus the second
 * staging slot); synchronises before returning. */
size_t demons_workspace_bytes_queue(const demons_ctx* ctx, int levels);
int demons_register_host_queue(demons_ctx* ctx, int n, const float* const* h_static, const float* const* h_moving,
                               float* const* h_u, float* const* h_u_back, int levels, const int* h_iters_per_level,
                               double eps, double* h_stats, int* h_iters_done, void* stream);

/* ---- per-kernel entry points (one pass each, what the parity tests and the sweep call) -------
 * All take explicit dims (nx*ny*nz must not exceed the context's finest volume).
 *
 * demons_warp_force: S1-S4 + S6 of the hot path -- Mw = warp(M, u_in) (software
 * trilinear, L181), central-difference gradients (reading A7/A8), F per the context's variant
 * (Eq.(1)-(6)), d_u_out = d_u_in - F, UNSMOOTHED.  Variant 5 also needs d_ub_in / d_ub_out
 * (ub_out = ub_in + F); they must be NULL otherwise.  d_u_out must not alias any input.
 * d_metrics (nullable): 3 doubles on the device = {SSD, sum|F|_2, sum|u_in|_2}. */
int demons_warp_force(demons_ctx* ctx, const int dims[3], const float* d_static,
                      const float* d_moving, const float* d_u_in, float* d_u_out,
                      const float* d_ub_in, float* d_ub_out, double* d_metrics, void* stream);

/* demons_warp_force_slab: the same pass for ONE RANK of a z-slab decomposition (volumes of
 * 512x512x256 and up, one slab of planes per GPU).  dims = the WHOLE volume; d_static and d_moving are whole
 * volumes (replicated on every rank, so that the gather of PAPER.md L179 never leaves the device); the fields are
 * the rank's slab only: planes [z_begin, z_begin + z_count) of the volume, [3][z_count*ny*nx], own planes plus
 * halo planes.  Every image access uses global planes and the clamps of the whole volume; gradients of the warped
 * images (variants 2-5) are taken inside the slab, so the OUTERMOST plane of a slab side that is not a face of the
 * volume comes out wrong and must be halo.  With R = ceil(3 sigma), a halo of R + 1 planes per interior side makes
 * [warp_force_slab ; demons_smooth on the slab] exact on the own planes; the caller then refreshes the halos from
 * the neighbours' own planes (paper_0909_0928_b200/slabs.py: torch.distributed send/recv, one exchange per
 * iteration).  d_metrics (nullable): the three sums over planes [own_begin, own_begin + own_count) of the SLAB
 * (local indices), to be added over the ranks.  Variant 5 with d_ub_in = d_ub_out = NULL is the one-field form: the
 * caller holds u_b = -u_f (exact from a zero start, "ic_one_field") and S is warped by -u_f.
 * The context must have been created with the whole volume's dims;
 * z_count >= 2.  The "texture" option is not served. */
int demons_warp_force_slab(demons_ctx* ctx, const int dims[3], int z_begin, int z_count, int own_begin, int own_count,
                           const float* d_static, const float* d_moving, const float* d_u_in, float* d_u_out,
                           const float* d_ub_in, float* d_ub_out, double* d_metrics, void* stream);

/* demons_smooth: S5 -- separable Gaussian of `ncomp` planar components, radius R = ceil(3 sigma),
 * normalised taps, clamped borders (reading A9).  d_in != d_out. */
int demons_smooth(demons_ctx* ctx, const int dims[3], const float* d_in, float* d_out, int ncomp,
                  float sigma, void* stream);

/* demons_restrict: S7 -- 2x2x2 box average to ceil(fine/2) ("down-sampled";
 * reading A12).  d_coarse holds prod(ceil(fine_dims/2)) floats. */
int demons_restrict(demons_ctx* ctx, const int fine_dims[3], const float* d_fine, float* d_coarse,
                    void* stream);

/* demons_prolong: S8 -- u_fine(x) = 2 * trilinear(u_coarse, clamp((x - 0.5)/2)), three planar
 * components (one coarse voxel of motion = 2 fine voxels; reading A12). */
int demons_prolong(demons_ctx* ctx, const int coarse_dims[3], const float* d_u_coarse,
                   const int fine_dims[3], float* d_u_fine, void* stream);

/* demons_ssd: the final SSD of O8 -- sum (warp(M,u) - S)^2, variant 5: sum (warp(M,u) -
 * warp(S,ub))^2 (d_ub NULL otherwise).  d_out: 1 double on the device. */
int demons_ssd(demons_ctx* ctx, const int dims[3], const float* d_static, const float* d_moving,
               const float* d_u, const float* d_ub, double* d_out, void* stream);

/* demons_ic_error: BASELINE.json config 4 -- e(x) = |u_f(x) + u_b(x + u_f(x))|_2, u_b sampled
 * trilinearly with clamping (reading A14).  d_out: 2 doubles on the device = {mean e, max e}. */
int demons_ic_error(demons_ctx* ctx, const int dims[3], const float* d_uf, const float* d_ub,
                    double* d_out, void* stream);

/* demons_cc: correlation coefficient between the deformed moving image and the static image,
 *   CC = sum (a - mean a)(b - mean b) / sqrt( sum (a - mean a)^2 sum (b - mean b)^2 ),
 * a = warp(M,u), b = S (variant 5: b = warp(S,ub), d_ub NULL otherwise) -- the similarity measure
 * PAPER.md L234 (Sec. 3.3) compares the relative-norm stopping rule with.  0 if either image is
 * constant.  d_out: 1 double on the device. */
int demons_cc(demons_ctx* ctx, const int dims[3], const float* d_static, const float* d_moving,
              const float* d_u, const float* d_ub, double* d_out, void* stream);

/* demons_point_error: the landmark evaluation of PAPER.md L222 (Sec. 3.2, "three-dimensional
 * Euclidean distance").  d_points: [n][3] positions (x, y, z) in voxels of `dims`, any real value
 * (clamped to the volume); d_expect: [n][3] expected displacement at those points in voxels;
 * d_err: [n] doubles on the device = | (u(p_i) - expect_i) * spacing |_2 in mm, u sampled
 * trilinearly, spacing = the context's.  n_points == 0 is a no-op. */
int demons_point_error(demons_ctx* ctx, const int dims[3], const float* d_u, int n_points,
                       const float* d_points, const float* d_expect, double* d_err, void* stream);

/* ---- the one entry point that needs no workspace and allocates nothing ------------------------------------
 * demons_ssd_static computes what demons_ssd computes -- sum (warp(M,u) - S)^2, or with d_ub != NULL the two-field
 * form sum (warp(M,u) - warp(S,ub))^2 of variant 5 (reading O8) -- for callers who cannot
 * give the library device memory of their own: a plug-in inside an application that owns the device's memory
 * budget and forbids cudaMalloc, a checking hook that must leave the process's footprint as it found it, a
 * time-critical loop in which an allocator call would stall every stream of the device.  It takes no context:
 * inputs and the one output double are the caller's, everything else it needs is a scratch array compiled into the
 * library (128 KiB + 256 B of global memory on every GPU that loads libdemons.so, held until the process ends).
 * The call makes no cudaMalloc / cudaFree and uses no allocating library routine; it enqueues one 4-byte
 * memset and one kernel on `stream` and returns without synchronising.
 *  - Limit: nx*ny*nz <= DEMONS_SSD_STATIC_MAX_VOXELS (one scratch slot per 4096 voxels).  Anything larger is
 *    refused with DEMONS_E_UNSUPPORTED and a message that names both numbers; use demons_ssd then.
 *  - First call on a device: looks up the scratch array's device address (once per device, with that device
 *    current, kept for the life of the process).  Make that first call outside any stream capture.
 *  - All calls on a device share the one array.  Two calls whose kernels may run at the same time (different
 *    streams, or host threads that do not order their work) overwrite each other's partial sums and give wrong
 *    results: order them on one stream or with events.  Back-to-back calls on one stream are fine; each call
 *    re-zeroes the only word that must start at zero.
 *  - Result: agrees with demons_ssd to rounding of a double sum (the block partition differs: here it depends on
 *    the volume only, so the same inputs give the same bits on any GPU).
 * d_static, d_moving: [N] floats; d_u (d_ub): [3][N] floats; d_out: 1 double; all DEVICE pointers. */
#define DEMONS_SSD_STATIC_MAX_VOXELS 67108864 /* 2^26 = 512 x 512 x 256 */
int demons_ssd_static(const int dims[3], const float* d_static, const float* d_moving, const float* d_u,
                      const float* d_ub, double* d_out, void* stream);

/* Thread-local description of the last failure on this thread ("" if none). */
const char* demons_last_error(void);

#ifdef __cplusplus
}
#endif
#endif /* DEMONS_H */
