/* oracle/demons_oracle.h -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, single-threaded CPU restatement of the demons iteration of
 * Gu et al. (arxiv/paper_0909_0928), written from PAPER.md and the readings listed in
 * DESIGN.md.  It shares no code with the CUDA path and the CUDA path never calls it.
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
 * legs may load this library.
 *
 * Conventions:
 *   - volume: float32, flat index x + nx*(y + ny*z)          (Sec. 2.5)
 *   - field : float32, planar [3][nz][ny][nx], comp 0 = x, in voxels of its level
 *   - warp(I,u)(x) = trilinear(I, x + u(x)); update u <- u - F (reading C1)
 *   - every per-voxel evaluation in double from float32 inputs, rounded once on store;
 *     reductions in double.
 *
 * Parity pins (tests/test_oracle_pins.py): every function below is pinned by closed
 * forms, library routines or invariants EXCEPT the value of the whole trajectory of
 * oracle_register on a given pair, which nothing in the paper fixes: parity unpinned
 * for the trajectory itself (it is held by the pins of each step plus the invariants
 * P1, P2b, P10, P12, P13, P14 on the whole loop).
 */
#ifndef DEMONS_ORACLE_H
#define DEMONS_ORACLE_H

#ifdef __cplusplus
extern "C" {
#endif

/* Method numbering: PAPER.md L284 (Table 2 caption) "Methods 1-6", here 0-based. */
enum {
    ORACLE_PASSIVE = 0,            /* Eq.(1)  */
    ORACLE_EVOLVED_PASSIVE = 1,    /* Eq.(2)  */
    ORACLE_ACTIVE = 2,             /* Eq.(3)  */
    ORACLE_DOUBLE = 3,             /* Eq.(4)  */
    ORACLE_ADJUSTED_DOUBLE = 4,    /* Eq.(5)  */
    ORACLE_INVERSE_CONSISTENT = 5  /* Eq.(6) */
};

/* O1: central differences, clamped indices. g is [3][N]. */
void oracle_gradient(const float* I, const int dims[3], float* g);

/* O2: out(x) = trilinear(I, clamp(x + u(x))). */
void oracle_warp(const float* I, const float* u, const int dims[3], float* out);

/* O3: one voxel of Eq.(1)-(6). Unused gradient arguments may be NULL. */
void oracle_force_voxel(int variant, double alpha, double d, const double gS[3], const double gM0[3],
                        const double gMw[3], const double gSw[3], double F[3]);

/* O5: Gaussian taps w[0..R] (w[k] = w[-k]); returns R = ceil(3 sigma), or -1 if cap < R+1. */
int oracle_gauss_taps(double sigma, float* w, int cap);

/* O5: separable smoothing x then y then z of ncomp planar components. in != out. */
void oracle_smooth(const float* in, float* out, const int dims[3], int ncomp, double sigma);

/* O6: 2x2x2 box average, coarse dims = ceil(fine/2), odd tail counted twice. */
void oracle_coarse_dims(const int fine[3], int coarse[3]);
void oracle_restrict(const float* fine, const int fine_dims[3], float* coarse);

/* O7: u_fine(x) = 2 * trilinear(u_coarse, clamp((x - 0.5)/2)), 3 planar components. */
void oracle_prolong(const float* uc, const int coarse_dims[3], const int fine_dims[3], float* uf);

/* O2+O1+O3+O4+O8: one un-smoothed demons update.
 * u_out = u_in - F; variant 5 also ub_out = ub_in + F (NULL otherwise).
 * gS / gM0 are the fixed level gradients ([3][N], may be NULL when the variant does not use
 * them, see oracle_variant_needs). metrics (nullable) = {SSD, sum|F|, sum|u_in|}. */
void oracle_warp_force(int variant, double alpha, const int dims[3], const float* S, const float* M,
                       const float* gS, const float* gM0, const float* u_in, float* u_out,
                       const float* ub_in, float* ub_out, double metrics[3]);

/* O9 (+O10 when eps > 0): full multi-level registration.
 * u: in = initial field when levels == 1 (ignored and zeroed when levels > 1), out = final.
 * ub: variant 5 only, same rule. iters: per level, coarse -> fine. stats (nullable):
 * [sum(iters)][3] rows in execution order. iters_done (nullable): per level. Returns 0 or -1. */
int oracle_register(int variant, double alpha, double sigma, const int dims[3], const float* S,
                    const float* M, float* u, float* ub, int levels, const int* iters, double eps,
                    double* stats, int* iters_done);

/* SSD between warp(M,u) and S (variant 5: warp(M,u) and warp(S,ub)). */
double oracle_final_ssd(int variant, const int dims[3], const float* S, const float* M,
                        const float* u, const float* ub);

/* BASELINE.json config 4: e(x) = | u_f(x) + u_b(x + u_f(x)) |, u_b sampled trilinearly, clamped. */
void oracle_ic_error(const float* uf, const float* ub, const int dims[3], double* mean, double* max);

/* Correlation coefficient of warp(M,u) and S (variant 5: warp(S,ub)). */
double oracle_cc(int variant, const int dims[3], const float* S, const float* M, const float* u,
                 const float* ub);

/* 3D Euclidean error in mm of the field sampled at n points against expected
 * displacements; points / expect: [n][3] in voxels, err: [n]. */
void oracle_point_error(const float* u, const int dims[3], const double spacing[3], int n,
                        const float* points, const float* expect, double* err);

#ifdef __cplusplus
}
#endif
#endif
