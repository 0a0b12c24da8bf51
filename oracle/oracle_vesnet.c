/*
 * oracle_vesnet.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, obviously-correct CPU statement of what the far-field path of
 * VesNet (arxiv/paper_2606_25569) computes.  Only tests/, __graft_entry__.smoke()
 * and bench.py's cpu_baseline / --impl reference legs may build, load or call this
 * file.  It shares no code, header, table or constant with the CUDA path under
 * paper_2606_25569_b200/csrc/, and neither side includes the other.
 *
 * What it states (citations are PAPER.md lines):
 *
 *   single-layer integral        S[X,f](x) = int_gamma G(x - X) f(X) ds(X)           PAPER.md:129-131 (eq 2.8)
 *   2-D Stokeslet                G(r) = 1/(4 pi mu) ( -log|r| I + r (x) r / |r|^2 )   PAPER.md:133-136 (eq 2.9;
 *                                the extracted text prints "+log|r|" and drops I -- DESIGN.md reading A1,
 *                                pinned by the S[n] = 0 identity in tests/test_oracle_pins.py)
 *   far-field quadrature         trapezoid rule in alpha, ds = |X_alpha| dalpha      PAPER.md:173 (sec 2.2.2)
 *   who contributes              every point of every OTHER vesicle; the target's
 *                                own vesicle is a separate (self) term               PAPER.md:140-144 (eq 2.10), 425 (Alg. 4 l.3)
 *   "done without any approximation", O((MN)^2)
 *   spectral derivative          X(alpha) = sum_k Xhat_k e^{ik alpha},
 *                                d/ds = |dX/dalpha|^-1 d/dalpha                      PAPER.md:161-169 (sec 2.2.1)
 *   near field of a point        distance to the vesicle <= arclength spacing
 *   near vesicles masked out of the direct sum, same mask returned                   PAPER.md:329 (sec 4.1), 426 (Alg. 4 l.4)
 *   free targets (all vesicles contribute)                                           eq 2.8 summed over every vesicle
 *   elastic force                f = -kappa_b X_ssss + (sigma X_s)_s                 PAPER.md:123 (eq 2.7)
 *   redistribution               6x upsampling, arclength, search, linear interp.    PAPER.md:331-335 (sec 4.2)
 *
 * Arithmetic: every term and every accumulator is `long double` (x87 80-bit on
 * x86-64; >= fp64 everywhere), loops are in the order the definition is written,
 * no blocking, no reordering, no fused contraction (-ffp-contract=off), one
 * multiplication by 1/(4 pi mu) at the end.  OpenMP splits the outermost target
 * loop only.
 *
 * Pins (tests/test_oracle_pins.py, tests/golden/): closed form of one point
 * Stokeslet, S[n] = 0 outside a closed circle / ellipse, closed form for a
 * constant density on a circle, scaling / adjoint identities, brute-force
 * symmetric pair sums, equivariances, circle / ellipse weights and the elliptic
 * integral perimeter, numpy.fft for the derivative; near mask against a brute-force
 * definition; elastic force against circle / warped-circle / ellipse closed forms,
 * zero net force and a numpy FFT route; redistribution against its fixed point, a
 * warped circle and a numpy FFT / interp route.  Nothing here is "parity unpinned".
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef long double ld;

static const ld ORACLE_PI = 3.141592653589793238462643383279502884L;

int oracle_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/* One target (vesicle v, coordinates x) against every point of every other
 * vesicle: eq 2.8 / 2.9 with the trapezoid weights W, written term by term. */
static void farfield_one_target(const double *X, const double *F, const double *W,
                                int64_t nves, int64_t npts, int64_t v,
                                ld xt, ld yt, const unsigned char *skip_ves,
                                ld *ux, ld *uy)
{
    ld sx = 0.0L, sy = 0.0L;
    for (int64_t vp = 0; vp < nves; ++vp) {
        if (vp == v) continue;                       /* own vesicle: self term, not ours (eq 2.10) */
        if (skip_ves && skip_ves[vp]) continue;      /* near vesicle masked out     */
        for (int64_t j = 0; j < npts; ++j) {
            const int64_t s = vp * npts + j;
            const ld rx = xt - (ld)X[2 * s + 0];
            const ld ry = yt - (ld)X[2 * s + 1];
            const ld r2 = rx * rx + ry * ry;
            const ld gx = (ld)F[2 * s + 0] * (ld)W[s];   /* f_j w_j */
            const ld gy = (ld)F[2 * s + 1] * (ld)W[s];
            const ld mlog = -0.5L * logl(r2);            /* -log|r| */
            const ld rdotg = rx * gx + ry * gy;
            sx += mlog * gx + (rdotg / r2) * rx;         /* (-log|r| I + r r^T/|r|^2) g */
            sy += mlog * gy + (rdotg / r2) * ry;
        }
    }
    *ux = sx;
    *uy = sy;
}

/* U[v,i,:] for every point of every vesicle.  X,F,U: [nves,npts,2]; W: [nves,npts]. */
int oracle_farfield(const double *X, const double *F, const double *W,
                    int64_t nves, int64_t npts, double mu, double *U)
{
    if (!X || !F || !W || !U || nves < 1 || npts < 1 || !(mu > 0.0)) return 1;
    const ld scale = 1.0L / (4.0L * ORACLE_PI * (ld)mu);
    const int64_t P = nves * npts;
#pragma omp parallel for schedule(dynamic, 16)
    for (int64_t t = 0; t < P; ++t) {
        ld ux, uy;
        farfield_one_target(X, F, W, nves, npts, t / npts,
                            (ld)X[2 * t + 0], (ld)X[2 * t + 1], NULL, &ux, &uy);
        U[2 * t + 0] = (double)(scale * ux);
        U[2 * t + 1] = (double)(scale * uy);
    }
    return 0;
}

/* Same definition, only for the listed targets (flat point indices idx[0..nidx)).
 * Used where a full evaluation would take hours (8,000 vesicles). Usub: [nidx,2]. */
int oracle_farfield_subset(const double *X, const double *F, const double *W,
                           int64_t nves, int64_t npts, double mu,
                           const int64_t *idx, int64_t nidx, double *Usub)
{
    if (!X || !F || !W || !Usub || !idx || nves < 1 || npts < 1 || !(mu > 0.0)) return 1;
    const ld scale = 1.0L / (4.0L * ORACLE_PI * (ld)mu);
    const int64_t P = nves * npts;
    for (int64_t q = 0; q < nidx; ++q)
        if (idx[q] < 0 || idx[q] >= P) return 1;
#pragma omp parallel for schedule(dynamic, 16)
    for (int64_t q = 0; q < nidx; ++q) {
        const int64_t t = idx[q];
        ld ux, uy;
        farfield_one_target(X, F, W, nves, npts, t / npts,
                            (ld)X[2 * t + 0], (ld)X[2 * t + 1], NULL, &ux, &uy);
        Usub[2 * q + 0] = (double)(scale * ux);
        Usub[2 * q + 1] = (double)(scale * uy);
    }
    return 0;
}

/* Free targets (not on any membrane): velocity induced at xt[nt,2] by ALL vesicles
 * (eq 2.8 summed over every gamma_i, trapezoid rule).  Ut: [nt,2]. */
int oracle_farfield_targets(const double *X, const double *F, const double *W,
                            int64_t nves, int64_t npts, double mu,
                            const double *xt, int64_t nt, double *Ut)
{
    if (!X || !F || !W || !Ut || !xt || nves < 1 || npts < 1 || nt < 0 || !(mu > 0.0)) return 1;
    const ld scale = 1.0L / (4.0L * ORACLE_PI * (ld)mu);
#pragma omp parallel for schedule(dynamic, 16)
    for (int64_t q = 0; q < nt; ++q) {
        ld ux, uy;
        farfield_one_target(X, F, W, nves, npts, -1,
                            (ld)xt[2 * q + 0], (ld)xt[2 * q + 1], NULL, &ux, &uy);
        Ut[2 * q + 0] = (double)(scale * ux);
        Ut[2 * q + 1] = (double)(scale * uy);
    }
    return 0;
}

/* W[v,j] = (2 pi / N) |dX_v/dalpha (alpha_j)|,  alpha_j = 2 pi j / N.
 * The derivative is the definition written out: forward DFT,
 * multiply mode k by i k, inverse DFT.  Modes k = -floor((N-1)/2) .. floor((N-1)/2);
 * for even N the unmatched k = N/2 mode is dropped (reading A4).
 * Also returns the derivative itself when dX != NULL ([nves,npts,2]). */
int oracle_weights(const double *X, int64_t nves, int64_t npts, double *W, double *dX)
{
    if (!X || !W || nves < 1 || npts < 1) return 1;
    const int64_t N = npts;
    const int64_t kmax = (N - 1) / 2;
    ld *ctab = (ld *)malloc(sizeof(ld) * (size_t)N);
    ld *stab = (ld *)malloc(sizeof(ld) * (size_t)N);
    if (!ctab || !stab) { free(ctab); free(stab); return 2; }
    for (int64_t m = 0; m < N; ++m) {               /* cos, sin of 2 pi m / N */
        ctab[m] = cosl(2.0L * ORACLE_PI * (ld)m / (ld)N);
        stab[m] = sinl(2.0L * ORACLE_PI * (ld)m / (ld)N);
    }
    int fail = 0;
#pragma omp parallel for schedule(static)
    for (int64_t v = 0; v < nves; ++v) {
        const double *Xv = X + 2 * v * N;
        const int64_t nk = 2 * kmax + 1;
        /* Xhat_k = (1/N) sum_m X_m e^{-i k alpha_m},  k = -kmax..kmax  (both components) */
        ld *coef = (ld *)malloc(sizeof(ld) * 4 * (size_t)(nk > 0 ? nk : 1));
        if (!coef) { fail = 1; continue; }
        for (int64_t k = -kmax; k <= kmax; ++k) {
            ld cre_x = 0.0L, cim_x = 0.0L, cre_y = 0.0L, cim_y = 0.0L;
            for (int64_t m = 0; m < N; ++m) {
                int64_t a = (k * m) % N; if (a < 0) a += N;
                const ld c = ctab[a], s = stab[a];
                cre_x += (ld)Xv[2 * m + 0] * c;  cim_x -= (ld)Xv[2 * m + 0] * s;
                cre_y += (ld)Xv[2 * m + 1] * c;  cim_y -= (ld)Xv[2 * m + 1] * s;
            }
            ld *q = coef + 4 * (k + kmax);
            q[0] = cre_x / (ld)N; q[1] = cim_x / (ld)N; q[2] = cre_y / (ld)N; q[3] = cim_y / (ld)N;
        }
        /* dX/dalpha (alpha_j) = sum_k (i k Xhat_k) e^{i k alpha_j}  (real part; the sum is real) */
        for (int64_t j = 0; j < N; ++j) {
            ld dx = 0.0L, dy = 0.0L;
            for (int64_t k = -kmax; k <= kmax; ++k) {
                const ld *q = coef + 4 * (k + kmax);
                int64_t b = (k * j) % N; if (b < 0) b += N;
                const ld c = ctab[b], s = stab[b];
                dx += (ld)k * (-q[1] * c - q[0] * s);
                dy += (ld)k * (-q[3] * c - q[2] * s);
            }
            W[v * N + j] = (double)((2.0L * ORACLE_PI / (ld)N) * sqrtl(dx * dx + dy * dy));
            if (dX) { dX[2 * (v * N + j) + 0] = (double)dx; dX[2 * (v * N + j) + 1] = (double)dy; }
        }
        free(coef);
    }
    if (fail) { free(ctab); free(stab); return 2; }
    free(ctab); free(stab);
    return 0;
}

/* Near-field mask (PAPER.md:144, 248, 426 FindNearFieldPoints): near[t, vp] = 1 when
 * vp != ves(t) and min_j |x_t - X[vp,j]| <= h[vp]; h[vp] = the arclength spacing of
 * vesicle vp, taken as its largest trapezoid weight (reading N1).
 * near: [nves*npts, nves] bytes. */
int oracle_near_mask(const double *X, const double *W, int64_t nves, int64_t npts,
                     unsigned char *near)
{
    if (!X || !W || !near || nves < 1 || npts < 1) return 1;
    const int64_t P = nves * npts;
#pragma omp parallel for schedule(dynamic, 16)
    for (int64_t t = 0; t < P; ++t) {
        const int64_t v = t / npts;
        for (int64_t vp = 0; vp < nves; ++vp) {
            unsigned char flag = 0;
            if (vp != v) {
                ld h = 0.0L;
                for (int64_t j = 0; j < npts; ++j)
                    if ((ld)W[vp * npts + j] > h) h = (ld)W[vp * npts + j];
                ld dmin2 = INFINITY;
                for (int64_t j = 0; j < npts; ++j) {
                    const ld rx = (ld)X[2 * t + 0] - (ld)X[2 * (vp * npts + j) + 0];
                    const ld ry = (ld)X[2 * t + 1] - (ld)X[2 * (vp * npts + j) + 1];
                    const ld d2 = rx * rx + ry * ry;
                    if (d2 < dmin2) dmin2 = d2;
                }
                flag = (dmin2 <= h * h) ? 1 : 0;
            }
            near[t * nves + vp] = flag;
        }
    }
    return 0;
}

/* The paper's DirectSingleLayerIntegral: the direct sum with the
 * contribution of near vesicles (given mask near[t,vp]) set to zero. */
int oracle_farfield_masked(const double *X, const double *F, const double *W,
                           int64_t nves, int64_t npts, double mu,
                           const unsigned char *near, double *U)
{
    if (!X || !F || !W || !U || !near || nves < 1 || npts < 1 || !(mu > 0.0)) return 1;
    const ld scale = 1.0L / (4.0L * ORACLE_PI * (ld)mu);
    const int64_t P = nves * npts;
#pragma omp parallel for schedule(dynamic, 16)
    for (int64_t t = 0; t < P; ++t) {
        ld ux, uy;
        farfield_one_target(X, F, W, nves, npts, t / npts,
                            (ld)X[2 * t + 0], (ld)X[2 * t + 1], near + t * nves, &ux, &uy);
        U[2 * t + 0] = (double)(scale * ux);
        U[2 * t + 1] = (double)(scale * uy);
    }
    return 0;
}

/* Rows idx[0..nidx) of the near mask only (same definition; for suspensions whose full
 * [P, nves] mask would not fit).  near: [nidx, nves] bytes. */
int oracle_near_mask_subset(const double *X, const double *W, int64_t nves, int64_t npts,
                            const int64_t *idx, int64_t nidx, unsigned char *near)
{
    if (!X || !W || !near || !idx || nves < 1 || npts < 1 || nidx < 0) return 1;
    const int64_t P = nves * npts;
    for (int64_t q = 0; q < nidx; ++q)
        if (idx[q] < 0 || idx[q] >= P) return 1;
#pragma omp parallel for schedule(dynamic, 16)
    for (int64_t q = 0; q < nidx; ++q) {
        const int64_t t = idx[q];
        const int64_t v = t / npts;
        for (int64_t vp = 0; vp < nves; ++vp) {
            unsigned char flag = 0;
            if (vp != v) {
                ld h = 0.0L;
                for (int64_t j = 0; j < npts; ++j)
                    if ((ld)W[vp * npts + j] > h) h = (ld)W[vp * npts + j];
                ld dmin2 = INFINITY;
                for (int64_t j = 0; j < npts; ++j) {
                    const ld rx = (ld)X[2 * t + 0] - (ld)X[2 * (vp * npts + j) + 0];
                    const ld ry = (ld)X[2 * t + 1] - (ld)X[2 * (vp * npts + j) + 1];
                    const ld d2 = rx * rx + ry * ry;
                    if (d2 < dmin2) dmin2 = d2;
                }
                flag = (dmin2 <= h * h) ? 1 : 0;
            }
            near[q * nves + vp] = flag;
        }
    }
    return 0;
}

/* The masked direct sum at the listed targets only; near: [nidx, nves] rows for those targets. */
int oracle_farfield_masked_subset(const double *X, const double *F, const double *W,
                                  int64_t nves, int64_t npts, double mu,
                                  const int64_t *idx, int64_t nidx,
                                  const unsigned char *near, double *Usub)
{
    if (!X || !F || !W || !Usub || !near || !idx || nves < 1 || npts < 1 || !(mu > 0.0)) return 1;
    const ld scale = 1.0L / (4.0L * ORACLE_PI * (ld)mu);
    const int64_t P = nves * npts;
    for (int64_t q = 0; q < nidx; ++q)
        if (idx[q] < 0 || idx[q] >= P) return 1;
#pragma omp parallel for schedule(dynamic, 16)
    for (int64_t q = 0; q < nidx; ++q) {
        const int64_t t = idx[q];
        ld ux, uy;
        farfield_one_target(X, F, W, nves, npts, t / npts,
                            (ld)X[2 * t + 0], (ld)X[2 * t + 1], near + q * nves, &ux, &uy);
        Usub[2 * q + 0] = (double)(scale * ux);
        Usub[2 * q + 1] = (double)(scale * uy);
    }
    return 0;
}

/* ---------------------------------------------------------------------------------------------
 * Row f-2: the elastic membrane force (PAPER.md:123 eq 2.7, :319 Fig. 5b)
 *
 *     f = -kappa_b X_ssss + (sigma X_s)_s ,      d/ds = |dX/dalpha|^-1 d/dalpha
 *
 * with every d/dalpha the Fourier derivative written out as in oracle_weights (forward DFT,
 * multiply by i k, inverse DFT, unmatched k = N/2 mode dropped -- DESIGN.md reading A4) and the
 * four arclength derivatives applied one after the other (reading E1: no filtering, no
 * de-aliasing; the paper is silent).  kappa_b is one scalar, sigma a value per point. */
static void fourier_derivative(const ld *f, int64_t N, const ld *ctab, const ld *stab, ld *df)
{
    const int64_t kmax = (N - 1) / 2;
    for (int64_t j = 0; j < N; ++j) df[j] = 0.0L;
    for (int64_t k = -kmax; k <= kmax; ++k) {
        ld cre = 0.0L, cim = 0.0L;                        /* fhat_k = (1/N) sum_m f_m e^{-i k alpha_m} */
        for (int64_t m = 0; m < N; ++m) {
            int64_t a = (k * m) % N; if (a < 0) a += N;
            cre += f[m] * ctab[a];
            cim -= f[m] * stab[a];
        }
        cre /= (ld)N; cim /= (ld)N;
        for (int64_t j = 0; j < N; ++j) {                 /* + Re( i k fhat_k e^{i k alpha_j} ) */
            int64_t b = (k * j) % N; if (b < 0) b += N;
            df[j] += (ld)k * (-cim * ctab[b] - cre * stab[b]);
        }
    }
}

int oracle_elastic_force(const double *X, const double *sigma, int64_t nves, int64_t npts,
                         double kappa_b, double *F)
{
    if (!X || !sigma || !F || nves < 1 || npts < 1) return 1;
    const int64_t N = npts;
    ld *ctab = (ld *)malloc(sizeof(ld) * (size_t)N);
    ld *stab = (ld *)malloc(sizeof(ld) * (size_t)N);
    if (!ctab || !stab) { free(ctab); free(stab); return 2; }
    for (int64_t m = 0; m < N; ++m) {
        ctab[m] = cosl(2.0L * ORACLE_PI * (ld)m / (ld)N);
        stab[m] = sinl(2.0L * ORACLE_PI * (ld)m / (ld)N);
    }
    int fail = 0;
#pragma omp parallel for schedule(dynamic, 1)
    for (int64_t v = 0; v < nves; ++v) {
        ld *w = (ld *)malloc(sizeof(ld) * 9 * (size_t)N);
        if (!w) { fail = 1; continue; }
        ld *x = w, *y = w + N, *dx = w + 2 * N, *dy = w + 3 * N, *sa = w + 4 * N;
        ld *xs = w + 5 * N, *ys = w + 6 * N, *tx = w + 7 * N, *ty = w + 8 * N;
        for (int64_t j = 0; j < N; ++j) { x[j] = (ld)X[2 * (v * N + j)]; y[j] = (ld)X[2 * (v * N + j) + 1]; }
        fourier_derivative(x, N, ctab, stab, dx);
        fourier_derivative(y, N, ctab, stab, dy);
        for (int64_t j = 0; j < N; ++j) {
            sa[j] = sqrtl(dx[j] * dx[j] + dy[j] * dy[j]);                 /* |dX/dalpha| */
            xs[j] = dx[j] / sa[j]; ys[j] = dy[j] / sa[j];                 /* X_s */
        }
        /* (sigma X_s)_s */
        for (int64_t j = 0; j < N; ++j) { x[j] = (ld)sigma[v * N + j] * xs[j]; y[j] = (ld)sigma[v * N + j] * ys[j]; }
        fourier_derivative(x, N, ctab, stab, tx);
        fourier_derivative(y, N, ctab, stab, ty);
        for (int64_t j = 0; j < N; ++j) { tx[j] /= sa[j]; ty[j] /= sa[j]; }
        /* X_ss, X_sss, X_ssss: three more arclength derivatives of X_s */
        for (int64_t j = 0; j < N; ++j) { x[j] = xs[j]; y[j] = ys[j]; }
        for (int rep = 0; rep < 3; ++rep) {
            fourier_derivative(x, N, ctab, stab, dx);
            fourier_derivative(y, N, ctab, stab, dy);
            for (int64_t j = 0; j < N; ++j) { x[j] = dx[j] / sa[j]; y[j] = dy[j] / sa[j]; }
        }
        for (int64_t j = 0; j < N; ++j) {
            F[2 * (v * N + j) + 0] = (double)(-(ld)kappa_b * x[j] + tx[j]);
            F[2 * (v * N + j) + 1] = (double)(-(ld)kappa_b * y[j] + ty[j]);
        }
        free(w);
    }
    free(ctab); free(stab);
    return fail ? 2 : 0;
}

/* ---------------------------------------------------------------------------------------------
 * Row f-3: redistributing the points of a vesicle equally in arclength (sec 4.2).
 * Step by step, in the paper's order, with DESIGN.md readings R1-R5 where the text is silent:
 *   1. "we first upsample the membrane points by a factor of 6": trigonometric interpolation of X
 *      to M = 6 N nodes alpha'_m = 2 pi m / M (an even N keeps its k = N/2 mode as cos(N alpha/2), so
 *      the interpolant passes through the data; R1).
 *   2. "we compute arclength {l_k}": sa_m = |dX/dalpha (alpha'_m)| (Fourier derivative, reading A4),
 *      l(alpha) = int_0^alpha sa by integrating the Fourier series of sa on the fine grid term by
 *      term, its k = M/2 mode dropped (R2: "the FFT in computing arclength").  l_M = L = 2 pi mean(sa).
 *   3. "build a piece-wise linear interpolant, and then infer the corresponding alpha~_k for the
 *      equispaced arclength": targets l~_k = k L / N, k = 0 .. N-1 (point 0 stays where it is; R3);
 *      "a search in the increasing arclength sequence to locate the interval containing the target
 *      arclength, then interpolate based on the two endpoints of the interval": the first m with
 *      l_{m+1} > l~_k, theta = (l~_k - l_m)/(l_{m+1} - l_m), and the new point is the same linear
 *      interpolation of the two upsampled points, Xnew_k = Xup_m + theta (Xup_{m+1} - Xup_m)   (R4).
 * Xnew: [nves, npts, 2]. */
int oracle_redistribute(const double *X, int64_t nves, int64_t npts, double *Xnew)
{
    if (!X || !Xnew || nves < 1 || npts < 1) return 1;
    const int64_t N = npts, M = 6 * npts, K = (N - 1) / 2;
    ld *cM = (ld *)malloc(sizeof(ld) * (size_t)M), *sM = (ld *)malloc(sizeof(ld) * (size_t)M);
    ld *cN = (ld *)malloc(sizeof(ld) * (size_t)N), *sN = (ld *)malloc(sizeof(ld) * (size_t)N);
    if (!cM || !sM || !cN || !sN) { free(cM); free(sM); free(cN); free(sN); return 2; }
    for (int64_t m = 0; m < M; ++m) { cM[m] = cosl(2.0L * ORACLE_PI * (ld)m / (ld)M); sM[m] = sinl(2.0L * ORACLE_PI * (ld)m / (ld)M); }
    for (int64_t m = 0; m < N; ++m) { cN[m] = cosl(2.0L * ORACLE_PI * (ld)m / (ld)N); sN[m] = sinl(2.0L * ORACLE_PI * (ld)m / (ld)N); }
    int fail = 0;
#pragma omp parallel for schedule(dynamic, 1)
    for (int64_t v = 0; v < nves; ++v) {
        const double *Xv = X + 2 * v * N;
        ld *w = (ld *)malloc(sizeof(ld) * (size_t)(4 * (2 * K + 1) + 2 + 4 * M + 1 + 2 * M));
        if (!w) { fail = 1; continue; }
        ld *coef = w;                                   /* (re_x, im_x, re_y, im_y) for k = -K..K */
        ld *nyq = w + 4 * (2 * K + 1);                  /* k = N/2 coefficient of x, y (even N)   */
        ld *xu = nyq + 2, *yu = xu + M, *sa = yu + M, *l = sa + M;   /* l has M + 1 entries */
        ld *p = l + M + 1, *q = p + M;                  /* Fourier coefficients of sa             */
        /* 1. coefficients of X, then the interpolant and its derivative on the fine grid */
        for (int64_t k = -K; k <= K; ++k) {
            ld rx = 0.0L, ix = 0.0L, ry = 0.0L, iy = 0.0L;
            for (int64_t j = 0; j < N; ++j) {
                int64_t a = (k * j) % N; if (a < 0) a += N;
                rx += (ld)Xv[2 * j] * cN[a];     ix -= (ld)Xv[2 * j] * sN[a];
                ry += (ld)Xv[2 * j + 1] * cN[a]; iy -= (ld)Xv[2 * j + 1] * sN[a];
            }
            ld *c = coef + 4 * (k + K);
            c[0] = rx / (ld)N; c[1] = ix / (ld)N; c[2] = ry / (ld)N; c[3] = iy / (ld)N;
        }
        nyq[0] = nyq[1] = 0.0L;
        if (N % 2 == 0) {
            for (int64_t j = 0; j < N; ++j) {
                const ld sgn = (j % 2) ? -1.0L : 1.0L;
                nyq[0] += sgn * (ld)Xv[2 * j]; nyq[1] += sgn * (ld)Xv[2 * j + 1];
            }
            nyq[0] /= (ld)N; nyq[1] /= (ld)N;
        }
        for (int64_t m = 0; m < M; ++m) {
            ld x = 0.0L, y = 0.0L, dx = 0.0L, dy = 0.0L;
            for (int64_t k = -K; k <= K; ++k) {
                const ld *c = coef + 4 * (k + K);
                int64_t a = (k * m) % M; if (a < 0) a += M;
                x += c[0] * cM[a] - c[1] * sM[a];
                y += c[2] * cM[a] - c[3] * sM[a];
                dx += (ld)k * (-c[1] * cM[a] - c[0] * sM[a]);
                dy += (ld)k * (-c[3] * cM[a] - c[2] * sM[a]);
            }
            if (N % 2 == 0) {                                   /* cos(N alpha'/2) = cos(2 pi (N/2) m / M) */
                const int64_t a = ((N / 2) * m) % M;
                x += nyq[0] * cM[a]; y += nyq[1] * cM[a];
            }
            xu[m] = x; yu[m] = y;
            sa[m] = sqrtl(dx * dx + dy * dy);
        }
        /* 2. arclength at the fine nodes by term-by-term integration of the Fourier series of sa */
        ld s0 = 0.0L;
        for (int64_t m = 0; m < M; ++m) s0 += sa[m];
        s0 /= (ld)M;
        for (int64_t k = 1; k <= M / 2 - 1; ++k) {              /* shat_k = p_k + i q_k */
            ld pr = 0.0L, qi = 0.0L;
            for (int64_t m = 0; m < M; ++m) {
                const int64_t a = (k * m) % M;
                pr += sa[m] * cM[a]; qi -= sa[m] * sM[a];
            }
            p[k] = pr / (ld)M; q[k] = qi / (ld)M;
        }
        for (int64_t m = 0; m < M; ++m) {
            ld acc = s0 * (2.0L * ORACLE_PI * (ld)m / (ld)M);
            for (int64_t k = 1; k <= M / 2 - 1; ++k) {
                const int64_t a = (k * m) % M;
                acc += 2.0L * (p[k] * sM[a] - q[k] * (1.0L - cM[a])) / (ld)k;
            }
            l[m] = acc;
        }
        const ld L = 2.0L * ORACLE_PI * s0;
        l[M] = L;
        /* 3. search + linear interpolation */
        for (int64_t k = 0; k < N; ++k) {
            const ld lt = (ld)k * L / (ld)N;
            int64_t m = 0;
            while (m < M - 1 && !(l[m + 1] > lt)) ++m;
            const ld theta = (lt - l[m]) / (l[m + 1] - l[m]);
            const int64_t m1 = (m + 1) % M;
            Xnew[2 * (v * N + k) + 0] = (double)(xu[m] + theta * (xu[m1] - xu[m]));
            Xnew[2 * (v * N + k) + 1] = (double)(yu[m] + theta * (yu[m1] - yu[m]));
        }
        free(w);
    }
    free(cM); free(sM); free(cN); free(sN);
    return fail ? 2 : 0;
}
