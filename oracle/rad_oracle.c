/*
 * rad_oracle.c -- CPU ORACLE (test infrastructure, not product; see rad_oracle.h).
 *
 * Literal loop nest of the paper's expanded radiation integral:
 *   eqs. (3)-(5) f_x, f_y, f_z
 *   eq.  (6)     g
 *   eq.  (7)     phase
 *   eq.  (1)     e^2/4pi^2 |int|^2
 *   eqs. (8)-(9) omega -> omega*      PAPER.md:50-56   (spin-0 = substitution model)
 *   eqs. (10)-(12) BCK, I and J       PAPER.md:62-68   (spin-1/2)
 *   sum over sections / particles
 * Quadrature: composite trapezoid on the given t_k (reading Q1;
 * the paper only says "points in time").
 * Outside [t_0, t_{N-1}] the acceleration is zero, no boundary terms (Q2).
 * Output in units of e^2, 1/4pi^2 included (Q7).
 *
 * Every quantity is converted to RAD_REAL on load and every operation is done
 * in RAD_REAL.  No fast-math, no blocking, no reordering; one grid point at a
 * time, samples in ascending k.
 */
#include "rad_oracle.h"

#include <math.h>
#include <stddef.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#if defined(RAD_ORACLE_QUAD)
#include <quadmath.h>
typedef __float128 real;
#define R_SIN(x) sinq(x)
#define R_COS(x) cosq(x)
#define R_DIGITS 113
#define R_PI M_PIq
#elif defined(RAD_ORACLE_DOUBLE)
typedef double real;
#define R_SIN(x) sin(x)
#define R_COS(x) cos(x)
#define R_DIGITS 53
#define R_PI 3.14159265358979323846
#else
typedef long double real;
#define R_SIN(x) sinl(x)
#define R_COS(x) cosl(x)
#define R_DIGITS 64
#define R_PI 3.14159265358979323846264338327950288L
#endif

int rad_oracle_real_digits(void) { return R_DIGITS; }

int rad_oracle_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/* Trapezoid weight of sample k on the (possibly non-uniform) abscissae t[0..n-1]. */
static real trapezoid_weight(const double *t, int64_t n, int64_t k)
{
    const real half = (real)0.5;
    if (k == 0) return ((real)t[1] - (real)t[0]) * half;
    if (k == n - 1) return ((real)t[n - 1] - (real)t[n - 2]) * half;
    return ((real)t[k + 1] - (real)t[k - 1]) * half;
}

/*
 * The eight quadrature sums of one point: A_x, A_y, A_z (eq. 1 / eq. 11 with
 * eqs. 3-7) and J (eq. 12, leading order), each complex, at phase frequency w_ph.
 */
static void point_sums(int64_t n,
                       const double *t, const double *dz, const double *x, const double *y,
                       const double *vx, const double *vy, const double *dvz,
                       const double *ax, const double *ay, const double *az,
                       const double *gamma,
                       real w_ph, real n_x, real n_y, real sums[8])
{
    const real half = (real)0.5, one = (real)1, two = (real)2;
    const real theta2 = n_x * n_x + n_y * n_y;
    real Axr = 0, Axi = 0, Ayr = 0, Ayi = 0, Azr = 0, Azi = 0, Jr = 0, Ji = 0;

    for (int64_t k = 0; k < n; ++k) {
        const real tk = t[k], dzk = dz[k], xk = x[k], yk = y[k];
        const real vxk = vx[k], vyk = vy[k], dvzk = dvz[k];
        const real axk = ax[k], ayk = ay[k], azk = az[k], gk = gamma[k];

        const real a = one / (two * gk * gk);                 /* 1/(2 gamma^2) */
        const real D = -theta2 * half - dvzk + a;             /* round bracket of eqs. 3-5 */
        const real q = a + theta2 * half - dvzk - n_x * vxk - n_y * vyk;
        const real g = one / (q * q);                         /* eq. 6 */

        const real fx = ((azk + n_y * ayk) * (n_x - vxk)
                         - (n_y * (n_y - vyk) + D) * axk) * g;                    /* eq. 3 */
        const real fy = ((azk + n_x * axk) * (n_y - vyk)
                         - (n_x * (n_x - vxk) + D) * ayk) * g;                    /* eq. 4 */
        const real fz = (D * (n_x * axk + n_y * ayk)
                         - (n_x * (n_x - vxk) + n_y * (n_y - vyk)) * azk) * g;    /* eq. 5 */
        const real h = (n_x * axk + n_y * ayk + azk) * g;     /* eq. 12 integrand, leading order */

        const real psi = (a + theta2 * half) * tk - dzk - n_x * xk - n_y * yk;   /* eq. 7 / omega */
        const real phi = w_ph * psi;
        const real c = R_COS(phi), s = R_SIN(phi);
        const real w = trapezoid_weight(t, n, k);

        Axr += w * fx * c;  Axi += w * fx * s;
        Ayr += w * fy * c;  Ayi += w * fy * s;
        Azr += w * fz * c;  Azi += w * fz * s;
        Jr  += w * h  * c;  Ji  += w * h  * s;
    }
    sums[0] = Axr; sums[1] = Axi; sums[2] = Ayr; sums[3] = Ayi;
    sums[4] = Azr; sums[5] = Azi; sums[6] = Jr;  sums[7] = Ji;
}

/* d2I/domega dOmega (units of e^2) of one point from its quadrature sums. */
static real point_value(const real sums[8], int model, real u, real gamma0)
{
    const real half = (real)0.5, one = (real)1, two = (real)2, four = (real)4;
    const real S = sums[0] * sums[0] + sums[1] * sums[1]
                 + sums[2] * sums[2] + sums[3] * sums[3]
                 + sums[4] * sums[4] + sums[5] * sums[5];
    const real J2 = sums[6] * sums[6] + sums[7] * sums[7];
    const real norm = one / (four * R_PI * R_PI);
    if (model == RAD_ORACLE_CLASSICAL) return S * norm;                   /* eq. 1 */
    if (model == RAD_ORACLE_SPIN0) return (one - u) * S * norm;          /* eq. 9: omega/omega* = 1-u */
    /* eq. 10: (E*^2+E^2)/2E^2 = (1+(1-u)^2)/2,  omega^2/(2 E^2 gamma^2) = u^2/(2 gamma^2) */
    return ((one + (one - u) * (one - u)) * half * S
            + u * u / (two * gamma0 * gamma0) * J2) * norm;
}

static int check_args(int64_t n, int64_t npts, const double *omega, int model, double lam)
{
    if (n < 2 || npts < 0) return -1;
    if (model < 0 || model > 2) return -1;
    if (model != RAD_ORACLE_CLASSICAL)
        for (int64_t i = 0; i < npts; ++i)
            if (!(omega[i] * lam < 1.0)) return -1;
    return 0;
}

int rad_oracle_points(int64_t n,
                      const double *t, const double *dz, const double *x, const double *y,
                      const double *vx, const double *vy, const double *dvz,
                      const double *ax, const double *ay, const double *az,
                      const double *gamma,
                      int64_t npts, const double *omega, const double *nx, const double *ny,
                      int model, double hbarc_over_E,
                      double *out, double *amp)
{
    if (!t || !dz || !x || !y || !vx || !vy || !dvz || !ax || !ay || !az || !gamma) return -1;
    if (npts > 0 && (!omega || !nx || !ny || !out)) return -1;
    if (check_args(n, npts, omega, model, hbarc_over_E)) return -1;

#pragma omp parallel for schedule(dynamic, 1)
    for (int64_t i = 0; i < npts; ++i) {
        const real one = (real)1;
        const real w = omega[i];
        real u = 0, w_ph = w;
        if (model != RAD_ORACLE_CLASSICAL) {
            u = w * (real)hbarc_over_E;                       /* hbar omega / E */
            w_ph = w / (one - u);                             /* omega* */
        }
        real sums[8];
        point_sums(n, t, dz, x, y, vx, vy, dvz, ax, ay, az, gamma,
                   w_ph, (real)nx[i], (real)ny[i], sums);
        out[i] = (double)point_value(sums, model, u, (real)gamma[0]);
        if (amp)
            for (int c = 0; c < 8; ++c) amp[8 * i + c] = (double)sums[c];
    }
    return 0;
}

int rad_oracle_ensemble_points(int32_t count, int64_t stride, const int64_t *n,
                               const double *t, const double *dz, const double *x, const double *y,
                               const double *vx, const double *vy, const double *dvz,
                               const double *ax, const double *ay, const double *az,
                               const double *gamma,
                               int64_t npts, const double *omega, const double *nx, const double *ny,
                               int model, const double *hbarc_over_E, int accumulate,
                               double *out)
{
    if (count < 0 || !n) return -1;
    if (!t || !dz || !x || !y || !vx || !vy || !dvz || !ax || !ay || !az || !gamma) return -1;
    if (npts > 0 && (!omega || !nx || !ny || !out)) return -1;
    if (model != RAD_ORACLE_CLASSICAL && !hbarc_over_E) return -1;
    for (int32_t p = 0; p < count; ++p) {
        if (n[p] > stride) return -1;
        if (check_args(n[p], npts, omega, model, hbarc_over_E ? hbarc_over_E[p] : 0.0)) return -1;
    }

#pragma omp parallel for schedule(dynamic, 1)
    for (int64_t i = 0; i < npts; ++i) {
        const real one = (real)1;
        const real w = omega[i];
        real total = accumulate ? (real)out[i] : (real)0;
        for (int32_t p = 0; p < count; ++p) {                 /* p ascending */
            const int64_t o = (int64_t)p * stride;
            real u = 0, w_ph = w;
            if (model != RAD_ORACLE_CLASSICAL) {
                u = w * (real)hbarc_over_E[p];
                w_ph = w / (one - u);
            }
            real sums[8];
            point_sums(n[p], t + o, dz + o, x + o, y + o, vx + o, vy + o, dvz + o,
                       ax + o, ay + o, az + o, gamma + o,
                       w_ph, (real)nx[i], (real)ny[i], sums);
            total += point_value(sums, model, u, (real)gamma[o]);
        }
        out[i] = (double)total;
    }
    return 0;
}
