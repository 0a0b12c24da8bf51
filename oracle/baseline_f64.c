/*
 * baseline_f64.c -- TEST / BENCH INFRASTRUCTURE, NOT THE PRODUCT, and NOT the parity oracle.
 *
 * The same direct sum as oracle_vesnet.c's farfield_one_target (PAPER.md:129-136 eqs 2.8/2.9, :173 trapezoid
 * rule, own vesicle excluded), written in plain `double` so that a compiler may vectorise it: the CPU SPEED
 * baseline bench.py reports beside the long-double oracle's (`cpu_baseline.fast_double`).  The long-double
 * oracle is the right code to check against and the wrong code to time (x87, scalar logl); this file is the
 * opposite.  Built with -O3 -march=native -ffast-math -fopenmp (libmvec's vector log where available).
 * Pinned to the long-double oracle at 1e-13 relative L2 in tests/test_oracle_pins.py; nothing is ever
 * compared with the CUDA path through it.  Shares no code with csrc/.
 */
#include <math.h>
#include <stdint.h>
#ifdef _OPENMP
#include <omp.h>
#endif

int baseline_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/* U at the flat point indices idx[0..nidx): every point of every OTHER vesicle contributes. Usub: [nidx,2]. */
int baseline_farfield_subset(const double *X, const double *F, const double *W, int64_t nves, int64_t npts,
                             double mu, const int64_t *idx, int64_t nidx, double *Usub)
{
    if (!X || !F || !W || !Usub || !idx || nves < 1 || npts < 1 || !(mu > 0.0)) return 1;
    const double scale = 1.0 / (4.0 * 3.14159265358979323846 * mu);
    const int64_t P = nves * npts;
    for (int64_t q = 0; q < nidx; ++q)
        if (idx[q] < 0 || idx[q] >= P) return 1;
#pragma omp parallel for schedule(dynamic, 16)
    for (int64_t q = 0; q < nidx; ++q) {
        const int64_t t = idx[q], v = t / npts;
        const double xt = X[2 * t + 0], yt = X[2 * t + 1];
        double sx = 0.0, sy = 0.0;
        for (int64_t vp = 0; vp < nves; ++vp) {
            if (vp == v) continue;
            const double *Xs = X + 2 * vp * npts, *Fs = F + 2 * vp * npts, *Ws = W + vp * npts;
            double px = 0.0, py = 0.0;
#pragma omp simd reduction(+ : px, py)
            for (int64_t j = 0; j < npts; ++j) {
                const double rx = xt - Xs[2 * j + 0], ry = yt - Xs[2 * j + 1];
                const double r2 = rx * rx + ry * ry;
                const double gx = Fs[2 * j + 0] * Ws[j], gy = Fs[2 * j + 1] * Ws[j];
                const double ml = -0.5 * log(r2);
                const double qd = (rx * gx + ry * gy) / r2;
                px += ml * gx + qd * rx;
                py += ml * gy + qd * ry;
            }
            sx += px;
            sy += py;
        }
        Usub[2 * q + 0] = scale * sx;
        Usub[2 * q + 1] = scale * sy;
    }
    return 0;
}
