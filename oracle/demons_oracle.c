/* oracle/demons_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT (see demons_oracle.h).
 *
 * Plain nested loops, one thread, double arithmetic per voxel, float32 storage between
 * steps.  Steps follow the paper's order (Sec. 2.5: interpolation kernel,
 * gradient kernel, displacement kernel, low-pass filter kernel, comparison kernel).
 * No blocking, no fusion, no vectorisation.  "reading" = a point the paper leaves open,
 * resolved in DESIGN.md.
 */
#include "demons_oracle.h"

#include <math.h>
#include <stdlib.h>
#include <string.h>

static size_t vox(int x, int y, int z, const int dims[3]) {
    return (size_t)x + (size_t)dims[0] * ((size_t)y + (size_t)dims[1] * (size_t)z);
}

static int clampi(int i, int lo, int hi) { return i < lo ? lo : (i > hi ? hi : i); }

static size_t nvox(const int dims[3]) { return (size_t)dims[0] * (size_t)dims[1] * (size_t)dims[2]; }

/* ---- O1 gradient -------------------------------------------------------------------
 * g_c(x) = ( I(x + e_c) - I(x - e_c) ) / 2, indices clamped to the volume.
 * Paper: "gradient mask"; central differences per BASELINE.json
 * north_star; clamped border is a reading (A7). */
void oracle_gradient(const float* I, const int dims[3], float* g) {
    const size_t N = nvox(dims);
    for (int z = 0; z < dims[2]; ++z)
        for (int y = 0; y < dims[1]; ++y)
            for (int x = 0; x < dims[0]; ++x) {
                const size_t i = vox(x, y, z, dims);
                const double xp = I[vox(clampi(x + 1, 0, dims[0] - 1), y, z, dims)];
                const double xm = I[vox(clampi(x - 1, 0, dims[0] - 1), y, z, dims)];
                const double yp = I[vox(x, clampi(y + 1, 0, dims[1] - 1), z, dims)];
                const double ym = I[vox(x, clampi(y - 1, 0, dims[1] - 1), z, dims)];
                const double zp = I[vox(x, y, clampi(z + 1, 0, dims[2] - 1), dims)];
                const double zm = I[vox(x, y, clampi(z - 1, 0, dims[2] - 1), dims)];
                g[0 * N + i] = (float)(0.5 * (xp - xm));
                g[1 * N + i] = (float)(0.5 * (yp - ym));
                g[2 * N + i] = (float)(0.5 * (zp - zm));
            }
}

/* ---- O2 trilinear sample -----------------------------------------------------------
 * Software trilinear (Sec. 2.5).  p clamped to [0, n-1] per axis
 * (reading A11), i0 = floor(p), f = p - i0, i1 = min(i0 + 1, n - 1);
 * lerp(a, b, t) = a + t (b - a) along x, then y, then z. */
static double lerp(double a, double b, double t) { return a + t * (b - a); }

static double sample_trilinear(const float* I, const int dims[3], double px, double py, double pz) {
    double p[3] = {px, py, pz};
    int i0[3], i1[3];
    double f[3];
    for (int c = 0; c < 3; ++c) {
        double q = p[c];
        const double hi = (double)(dims[c] - 1);
        if (q < 0.0) q = 0.0;
        if (q > hi) q = hi;
        const double fl = floor(q);
        i0[c] = (int)fl;
        f[c] = q - fl;
        i1[c] = i0[c] + 1 > dims[c] - 1 ? dims[c] - 1 : i0[c] + 1;
    }
    const double c000 = I[vox(i0[0], i0[1], i0[2], dims)], c100 = I[vox(i1[0], i0[1], i0[2], dims)];
    const double c010 = I[vox(i0[0], i1[1], i0[2], dims)], c110 = I[vox(i1[0], i1[1], i0[2], dims)];
    const double c001 = I[vox(i0[0], i0[1], i1[2], dims)], c101 = I[vox(i1[0], i0[1], i1[2], dims)];
    const double c011 = I[vox(i0[0], i1[1], i1[2], dims)], c111 = I[vox(i1[0], i1[1], i1[2], dims)];
    const double a00 = lerp(c000, c100, f[0]), a10 = lerp(c010, c110, f[0]);
    const double a01 = lerp(c001, c101, f[0]), a11 = lerp(c011, c111, f[0]);
    const double b0 = lerp(a00, a10, f[1]), b1 = lerp(a01, a11, f[1]);
    return lerp(b0, b1, f[2]);
}

/* warp(I,u)(x) = trilinear(I, x + u(x))  (reading C1: pull-back, "x + u") */
void oracle_warp(const float* I, const float* u, const int dims[3], float* out) {
    const size_t N = nvox(dims);
    for (int z = 0; z < dims[2]; ++z)
        for (int y = 0; y < dims[1]; ++y)
            for (int x = 0; x < dims[0]; ++x) {
                const size_t i = vox(x, y, z, dims);
                out[i] = (float)sample_trilinear(I, dims, (double)x + (double)u[i],
                                                 (double)y + (double)u[N + i], (double)z + (double)u[2 * N + i]);
            }
}

/* ---- O3 force ----------------------------------------------------------------------
 * q(num, den) = den > 1e-9 ? num / den : 0  (zero guard, reading A6). */
static double guarded(double num, double den) { return den > 1e-9 ? num / den : 0.0; }

static double norm2(const double g[3]) { return g[0] * g[0] + g[1] * g[1] + g[2] * g[2]; }

void oracle_force_voxel(int variant, double alpha, double d, const double gS[3], const double gM0[3],
                        const double gMw[3], const double gSw[3], double F[3]) {
    F[0] = F[1] = F[2] = 0.0;
    switch (variant) {
    case ORACLE_PASSIVE: { /* Eq.(1): d gS / (d^2 + |gS|^2) */
        const double k = guarded(d, d * d + norm2(gS));
        for (int c = 0; c < 3; ++c) F[c] = k * gS[c];
        break;
    }
    case ORACLE_EVOLVED_PASSIVE: { /* Eq.(2), garbles repaired (readings A3, A4):
        4 d gS |gS| |gM0| / ( [2 d^2 + |gS|^2 + |gM0|^2] (|gS|^2 + |gM0|^2) ) */
        const double s2 = norm2(gS), m2 = norm2(gM0);
        const double k = guarded(4.0 * d * sqrt(s2) * sqrt(m2), (2.0 * d * d + s2 + m2) * (s2 + m2));
        for (int c = 0; c < 3; ++c) F[c] = k * gS[c];
        break;
    }
    case ORACLE_ACTIVE: { /* Eq.(3): d gMw / (d^2 + |gMw|^2) */
        const double k = guarded(d, d * d + norm2(gMw));
        for (int c = 0; c < 3; ++c) F[c] = k * gMw[c];
        break;
    }
    case ORACLE_DOUBLE: { /* Eq.(4): Eq.(1) + Eq.(3), each term guarded */
        const double k1 = guarded(d, d * d + norm2(gS));
        const double k2 = guarded(d, d * d + norm2(gMw));
        for (int c = 0; c < 3; ++c) F[c] = k1 * gS[c] + k2 * gMw[c];
        break;
    }
    case ORACLE_ADJUSTED_DOUBLE: { /* Eq.(5), second denominator squared (A5) */
        const double a2d2 = alpha * alpha * d * d;
        const double k1 = guarded(d, a2d2 + norm2(gS));
        const double k2 = guarded(d, a2d2 + norm2(gMw));
        for (int c = 0; c < 3; ++c) F[c] = k1 * gS[c] + k2 * gMw[c];
        break;
    }
    case ORACLE_INVERSE_CONSISTENT: { /* Eq.(6): d G / (d^2 + |G|^2), G = gMw + gSw */
        double G[3];
        for (int c = 0; c < 3; ++c) G[c] = gMw[c] + gSw[c];
        const double k = guarded(d, d * d + norm2(G));
        for (int c = 0; c < 3; ++c) F[c] = k * G[c];
        break;
    }
    default: break;
    }
}

/* ---- O5 Gaussian smoothing ---------------------------------------------------------
 * "Gaussian filter of unit standard deviation", separable.  R = ceil(3 sigma),
 * w_k = exp(-k^2 / 2 sigma^2) / sum_j exp(-j^2 / 2 sigma^2), in double, stored float32;
 * out(i) = sum_{k=-R..R} w_k in(clamp(i + k))   (reading A9). */
int oracle_gauss_taps(double sigma, float* w, int cap) {
    const int R = (int)ceil(3.0 * sigma);
    if (cap < R + 1) return -1;
    double sum = 0.0;
    for (int k = -R; k <= R; ++k) sum += exp(-(double)(k * k) / (2.0 * sigma * sigma));
    for (int k = 0; k <= R; ++k) w[k] = (float)(exp(-(double)(k * k) / (2.0 * sigma * sigma)) / sum);
    return R;
}

static void smooth_axis(const float* in, float* out, const int dims[3], int axis, const float* w, int R) {
    for (int z = 0; z < dims[2]; ++z)
        for (int y = 0; y < dims[1]; ++y)
            for (int x = 0; x < dims[0]; ++x) {
                int p[3] = {x, y, z};
                const int centre = p[axis];
                double acc = 0.0;
                for (int k = -R; k <= R; ++k) {
                    p[axis] = clampi(centre + k, 0, dims[axis] - 1);
                    acc += (double)w[k < 0 ? -k : k] * (double)in[vox(p[0], p[1], p[2], dims)];
                }
                out[vox(x, y, z, dims)] = (float)acc;
            }
}

void oracle_smooth(const float* in, float* out, const int dims[3], int ncomp, double sigma) {
    const size_t N = nvox(dims);
    float w[64];
    const int R = oracle_gauss_taps(sigma, w, 64);
    if (R < 0) return;
    float* tmp = (float*)malloc(N * sizeof(float));
    for (int c = 0; c < ncomp; ++c) {
        smooth_axis(in + c * N, out + c * N, dims, 0, w, R); /* x: in  -> out */
        smooth_axis(out + c * N, tmp, dims, 1, w, R);        /* y: out -> tmp */
        smooth_axis(tmp, out + c * N, dims, 2, w, R);        /* z: tmp -> out */
    }
    free(tmp);
}

/* ---- O6 restriction ----------------------------------------------------------------
 * "down-sampled"; 2x2x2 averaging per BASELINE.json config 3; n_c = ceil(n_f/2),
 * on an odd axis the last fine voxel is averaged with itself (reading A12). */
void oracle_coarse_dims(const int fine[3], int coarse[3]) {
    for (int c = 0; c < 3; ++c) coarse[c] = (fine[c] + 1) / 2;
}

void oracle_restrict(const float* fine, const int fd[3], float* coarse) {
    int cd[3];
    oracle_coarse_dims(fd, cd);
    for (int k = 0; k < cd[2]; ++k)
        for (int j = 0; j < cd[1]; ++j)
            for (int i = 0; i < cd[0]; ++i) {
                double acc = 0.0;
                for (int dz = 0; dz < 2; ++dz)
                    for (int dy = 0; dy < 2; ++dy)
                        for (int dx = 0; dx < 2; ++dx) {
                            const int x = clampi(2 * i + dx, 0, fd[0] - 1);
                            const int y = clampi(2 * j + dy, 0, fd[1] - 1);
                            const int z = clampi(2 * k + dz, 0, fd[2] - 1);
                            acc += (double)fine[vox(x, y, z, fd)];
                        }
                coarse[vox(i, j, k, cd)] = (float)(acc / 8.0);
            }
}

/* ---- O7 prolongation ---------------------------------------------------------------
 * "upsampled"; one coarse voxel of motion = 2 fine voxels.  Cell-centred
 * alignment: fine x sits at coarse (x - 0.5)/2, clamped (reading A12). */
void oracle_prolong(const float* uc, const int cd[3], const int fd[3], float* uf) {
    const size_t Nc = nvox(cd), Nf = nvox(fd);
    for (int c = 0; c < 3; ++c)
        for (int z = 0; z < fd[2]; ++z)
            for (int y = 0; y < fd[1]; ++y)
                for (int x = 0; x < fd[0]; ++x) {
                    const double v = sample_trilinear(uc + c * Nc, cd, ((double)x - 0.5) / 2.0,
                                                      ((double)y - 0.5) / 2.0, ((double)z - 0.5) / 2.0);
                    uf[c * Nf + vox(x, y, z, fd)] = (float)(2.0 * v);
                }
}

/* ---- one un-smoothed update: O2 -> O1 -> O3 -> O4, metrics O8 -------------------------
 * Order of the paper's kernels: interpolation, gradient, displacement.
 *   Mw = warp(M, u)                      (all variants)
 *   Sw = warp(S, ub)                     (variant 5)
 *   gMw = grad(Mw)  (variants 2-5; "gradient of the iteratively updated moving image", L75; A8)
 *   gSw = grad(Sw)  (variant 5)
 *   d = Mw - S      (variant 5: Mw - Sw)
 *   F per Eq.(1)-(6); u_out = u_in - F; variant 5: ub_out = ub_in + F (O4; C1, A14)
 *   metrics, state before the update: SSD = sum d^2, D = sum |F|_2, U = sum |u_in|_2 */
void oracle_warp_force(int variant, double alpha, const int dims[3], const float* S, const float* M,
                       const float* gS, const float* gM0, const float* u_in, float* u_out,
                       const float* ub_in, float* ub_out, double metrics[3]) {
    const size_t N = nvox(dims);
    const int needs_gMw = variant >= ORACLE_ACTIVE;
    const int ic = variant == ORACLE_INVERSE_CONSISTENT;
    float* Mw = (float*)malloc(N * sizeof(float));
    float* Sw = ic ? (float*)malloc(N * sizeof(float)) : NULL;
    float* gMw = needs_gMw ? (float*)malloc(3 * N * sizeof(float)) : NULL;
    float* gSw = ic ? (float*)malloc(3 * N * sizeof(float)) : NULL;

    oracle_warp(M, u_in, dims, Mw);
    if (ic) oracle_warp(S, ub_in, dims, Sw);
    if (needs_gMw) oracle_gradient(Mw, dims, gMw);
    if (ic) oracle_gradient(Sw, dims, gSw);

    double ssd = 0.0, sumF = 0.0, sumU = 0.0;
    for (size_t i = 0; i < N; ++i) {
        const double d = (double)Mw[i] - (double)(ic ? Sw[i] : S[i]);
        double a[3] = {0, 0, 0}, b[3] = {0, 0, 0}, c[3] = {0, 0, 0}, e[3] = {0, 0, 0}, F[3];
        for (int k = 0; k < 3; ++k) {
            if (gS) a[k] = gS[k * N + i];
            if (gM0) b[k] = gM0[k * N + i];
            if (gMw) c[k] = gMw[k * N + i];
            if (gSw) e[k] = gSw[k * N + i];
        }
        oracle_force_voxel(variant, alpha, d, a, b, c, e, F);
        double un = 0.0;
        for (int k = 0; k < 3; ++k) {
            const double uk = (double)u_in[k * N + i];
            un += uk * uk;
            u_out[k * N + i] = (float)(uk - F[k]);
            if (ic) ub_out[k * N + i] = (float)((double)ub_in[k * N + i] + F[k]);
        }
        ssd += d * d;
        sumF += sqrt(F[0] * F[0] + F[1] * F[1] + F[2] * F[2]);
        sumU += sqrt(un);
    }
    if (metrics) {
        metrics[0] = ssd;
        metrics[1] = sumF;
        metrics[2] = sumU;
    }
    free(Mw);
    free(Sw);
    free(gMw);
    free(gSw);
}

/* ---- O9 driver, O10 stopping rule ------------------------------------------------------
 * Multi-scale: PAPER.md L123-125 (coarse -> fine, up-sampled field is the next initial
 * field).  Per level: fixed gradients once ("only needs to be computed once"),
 * then iterations of [warp_force ; smooth the total field] (reading C2).
 * Stopping: l_n = D_n / U_n; stop after the first iteration n >= 10 with
 * |l_n - l_{n-10}| <= eps, both defined (U > 0)  (reading A13).  eps <= 0: fixed counts. */
int oracle_register(int variant, double alpha, double sigma, const int dims[3], const float* S,
                    const float* M, float* u, float* ub, int levels, const int* iters, double eps,
                    double* stats, int* iters_done) {
    if (levels < 1 || levels > 16) return -1;
    const int ic = variant == ORACLE_INVERSE_CONSISTENT;
    if (ic && !ub) return -1;
    int ld[16][3];
    float* Sl[16];
    float* Ml[16];
    /* level 0 = finest here; pyramids by O6, images only, no pre-blur (reading A15) */
    memcpy(ld[0], dims, sizeof(int) * 3);
    Sl[0] = (float*)S;
    Ml[0] = (float*)M;
    for (int l = 1; l < levels; ++l) {
        oracle_coarse_dims(ld[l - 1], ld[l]);
        Sl[l] = (float*)malloc(nvox(ld[l]) * sizeof(float));
        Ml[l] = (float*)malloc(nvox(ld[l]) * sizeof(float));
        oracle_restrict(Sl[l - 1], ld[l - 1], Sl[l]);
        oracle_restrict(Ml[l - 1], ld[l - 1], Ml[l]);
    }
    const size_t Nfine = nvox(dims);
    float* cur = (float*)malloc(3 * Nfine * sizeof(float));   /* u on the current level */
    float* curb = ic ? (float*)malloc(3 * Nfine * sizeof(float)) : NULL;
    float* upd = (float*)malloc(3 * Nfine * sizeof(float));   /* un-smoothed update */
    float* updb = ic ? (float*)malloc(3 * Nfine * sizeof(float)) : NULL;
    const size_t Ncoarsest = nvox(ld[levels - 1]);
    if (levels == 1) {
        memcpy(cur, u, 3 * Nfine * sizeof(float));
        if (ic) memcpy(curb, ub, 3 * Nfine * sizeof(float));
    } else {
        memset(cur, 0, 3 * Ncoarsest * sizeof(float));
        if (ic) memset(curb, 0, 3 * Ncoarsest * sizeof(float));
    }
    size_t row = 0;
    for (int step = 0; step < levels; ++step) {
        const int l = levels - 1 - step; /* coarse -> fine */
        const int* d3 = ld[l];
        const size_t N = nvox(d3);
        const int needs_gS = variant == ORACLE_PASSIVE || variant == ORACLE_EVOLVED_PASSIVE ||
                             variant == ORACLE_DOUBLE || variant == ORACLE_ADJUSTED_DOUBLE;
        const int needs_gM0 = variant == ORACLE_EVOLVED_PASSIVE;
        float* gS = needs_gS ? (float*)malloc(3 * N * sizeof(float)) : NULL;
        float* gM0 = needs_gM0 ? (float*)malloc(3 * N * sizeof(float)) : NULL;
        if (gS) oracle_gradient(Sl[l], d3, gS);
        if (gM0) oracle_gradient(Ml[l], d3, gM0);
        double lhist[4096];
        int lvalid[4096];
        int n = 0;
        for (; n < iters[step]; ++n) {
            double m[3];
            oracle_warp_force(variant, alpha, d3, Sl[l], Ml[l], gS, gM0, cur, upd, curb, updb, m);
            oracle_smooth(upd, cur, d3, 3, sigma);
            if (ic) oracle_smooth(updb, curb, d3, 3, sigma);
            if (stats) {
                stats[3 * row + 0] = m[0];
                stats[3 * row + 1] = m[1];
                stats[3 * row + 2] = m[2];
            }
            ++row;
            if (eps > 0.0 && n < 4096) {
                lvalid[n] = m[2] > 0.0;
                lhist[n] = lvalid[n] ? m[1] / m[2] : 0.0;
                if (n >= 10 && lvalid[n] && lvalid[n - 10] && fabs(lhist[n] - lhist[n - 10]) <= eps) {
                    ++n;
                    break;
                }
            }
        }
        if (iters_done) iters_done[step] = n;
        free(gS);
        free(gM0);
        if (l > 0) {
            oracle_prolong(cur, d3, ld[l - 1], upd);
            memcpy(cur, upd, 3 * nvox(ld[l - 1]) * sizeof(float));
            if (ic) {
                oracle_prolong(curb, d3, ld[l - 1], updb);
                memcpy(curb, updb, 3 * nvox(ld[l - 1]) * sizeof(float));
            }
        }
    }
    memcpy(u, cur, 3 * Nfine * sizeof(float));
    if (ic) memcpy(ub, curb, 3 * Nfine * sizeof(float));
    for (int l = 1; l < levels; ++l) {
        free(Sl[l]);
        free(Ml[l]);
    }
    free(cur);
    free(curb);
    free(upd);
    free(updb);
    return 0;
}

/* final SSD: one extra warp after the last iteration (O8) */
double oracle_final_ssd(int variant, const int dims[3], const float* S, const float* M,
                        const float* u, const float* ub) {
    const size_t N = nvox(dims);
    const int ic = variant == ORACLE_INVERSE_CONSISTENT;
    float* Mw = (float*)malloc(N * sizeof(float));
    float* Sw = ic ? (float*)malloc(N * sizeof(float)) : NULL;
    oracle_warp(M, u, dims, Mw);
    if (ic) oracle_warp(S, ub, dims, Sw);
    double ssd = 0.0;
    for (size_t i = 0; i < N; ++i) {
        const double d = (double)Mw[i] - (double)(ic ? Sw[i] : S[i]);
        ssd += d * d;
    }
    free(Mw);
    free(Sw);
    return ssd;
}

/* BASELINE.json config 4: inverse-consistency error |u_f(x) + u_b(x + u_f(x))|. */
void oracle_ic_error(const float* uf, const float* ub, const int dims[3], double* mean, double* max) {
    const size_t N = nvox(dims);
    double sum = 0.0, mx = 0.0;
    for (int z = 0; z < dims[2]; ++z)
        for (int y = 0; y < dims[1]; ++y)
            for (int x = 0; x < dims[0]; ++x) {
                const size_t i = vox(x, y, z, dims);
                const double px = x + (double)uf[i], py = y + (double)uf[N + i], pz = z + (double)uf[2 * N + i];
                double e2 = 0.0;
                for (int c = 0; c < 3; ++c) {
                    const double s = (double)uf[c * N + i] + sample_trilinear(ub + c * N, dims, px, py, pz);
                    e2 += s * s;
                }
                const double e = sqrt(e2);
                sum += e;
                if (e > mx) mx = e;
            }
    *mean = sum / (double)N;
    *max = mx;
}

/* Correlation coefficient between the deformed moving image and the static image (PAPER.md L234,
 * Sec. 3.3: the "commonly used" similarity measure the paper compares its relative norm with):
 *   CC = sum (a - mean a)(b - mean b) / sqrt( sum (a - mean a)^2  sum (b - mean b)^2 ),
 * a = warp(M,u), b = S (variant 5: b = warp(S,ub)).  Two passes (means first), all in double.
 * Returns 0 when either image is constant. */
double oracle_cc(int variant, const int dims[3], const float* S, const float* M, const float* u,
                 const float* ub) {
    const size_t N = nvox(dims);
    const int ic = variant == ORACLE_INVERSE_CONSISTENT;
    float* Mw = (float*)malloc(N * sizeof(float));
    float* Sw = ic ? (float*)malloc(N * sizeof(float)) : NULL;
    oracle_warp(M, u, dims, Mw);
    if (ic) oracle_warp(S, ub, dims, Sw);
    const float* b = ic ? Sw : S;
    double ma = 0.0, mb = 0.0;
    for (size_t i = 0; i < N; ++i) {
        ma += (double)Mw[i];
        mb += (double)b[i];
    }
    ma /= (double)N;
    mb /= (double)N;
    double sab = 0.0, saa = 0.0, sbb = 0.0;
    for (size_t i = 0; i < N; ++i) {
        const double da = (double)Mw[i] - ma, db = (double)b[i] - mb;
        sab += da * db;
        saa += da * da;
        sbb += db * db;
    }
    free(Mw);
    free(Sw);
    return (saa > 0.0 && sbb > 0.0) ? sab / sqrt(saa * sbb) : 0.0;
}

/* Landmark-style evaluation (Sec. 3.2: "three-dimensional Euclidean distance" at
 * feature points): for each point p_i (voxel coordinates, any real position) sample the field
 * trilinearly (clamped, O2) and return  err_i = | (u(p_i) - expect_i) * spacing |_2  in mm.
 * points, expect: [n][3] (x, y, z); err: [n]. */
void oracle_point_error(const float* u, const int dims[3], const double spacing[3], int n,
                        const float* points, const float* expect, double* err) {
    const size_t N = nvox(dims);
    for (int i = 0; i < n; ++i) {
        double e2 = 0.0;
        for (int c = 0; c < 3; ++c) {
            const double v = sample_trilinear(u + c * N, dims, (double)points[3 * i], (double)points[3 * i + 1],
                                              (double)points[3 * i + 2]);
            const double d = (v - (double)expect[3 * i + c]) * spacing[c];
            e2 += d * d;
        }
        err[i] = sqrt(e2);
    }
}
