/*
 * rad_oracle.h -- CPU ORACLE for the radiation integral of arXiv 1910.10391.
 *
 * TEST INFRASTRUCTURE, NOT PRODUCT.  Only tests/, __graft_entry__.smoke() and
 * bench.py's cpu_baseline / --impl reference legs may build, load or call this.
 * It shares no code, header, table or constant with the CUDA path under
 * paper_1910_10391_b200/csrc/ and include/rad.h; neither includes the other.
 *
 * What it computes: the quadrature sum of the paper's small-angle expanded
 * radiation integral, eqs. (3)-(7), for a list of
 * (omega, n_x, n_y) points over one sampled trajectory, in the classical
 * (eq. 1), substitution / spin-0 (eqs. 8-9) and
 * BCK / spin-1/2 (eqs. 10-12) variants, plus the sum over
 * trajectories / sections.  Plain loop nest, paper order,
 * no blocking, no reordering.  Arithmetic type RAD_REAL (default long double;
 * the same source is built with double for the timed CPU baseline and with
 * __float128 to check that long double is itself accurate enough).
 *
 * Parity pins (tests/test_oracle_pins.py): P1 straight line, P2 transversality,
 * P3 per-angle Parseval, P4 harmonic positions, P5 weak-undulator closed form,
 * P6 brute force of the unexpanded eqs. (1)-(2), P7 variant identities,
 * P8 J by parts, P9 quantum synchrotron (Baier-Katkov) limit, P10 independent numpy re-implementation,
 * symmetries (shifts, mirror, axis swap), Q1 (the trapezoid weights, end weights
 * included: exact closed forms for linear and quadratic integrands on ragged
 * abscissae), Q6 (gamma_k sample-wise in the integrand, gamma[0] in eq. 10's J
 * coefficient).  Every function of this file has at least one such pin.
 */
#ifndef RAD_ORACLE_H
#define RAD_ORACLE_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

enum { RAD_ORACLE_CLASSICAL = 0, RAD_ORACLE_SPIN0 = 1, RAD_ORACLE_SPIN_HALF = 2 };

/*
 * One trajectory, npts points.  All pointers are HOST arrays of doubles.
 *   t, dz, x, y, vx, vy, dvz, ax, ay, az, gamma : length n  (n >= 2)
 *   omega, nx, ny                               : length npts
 *   model        : RAD_ORACLE_*
 *   hbarc_over_E : Lambda = hbar c / E in the unit of t (ignored if classical)
 *   out          : length npts, d2I/(d omega d Omega) in units of e^2
 *   amp          : NULL, or length 8*npts: Re,Im of A_x, A_y, A_z, J per point
 *                  (the raw quadrature sums before |.|^2; for the pins)
 * Returns 0, or -1 on invalid arguments (n < 2, u = omega*Lambda >= 1, NULLs).
 */
int rad_oracle_points(int64_t n,
                      const double *t, const double *dz, const double *x, const double *y,
                      const double *vx, const double *vy, const double *dvz,
                      const double *ax, const double *ay, const double *az,
                      const double *gamma,
                      int64_t npts, const double *omega, const double *nx, const double *ny,
                      int model, double hbarc_over_E,
                      double *out, double *amp);

/*
 * Ensemble: sum over `count` trajectories, p ascending.
 * Row p of each of the 11 arrays starts at p*stride and has n[p] samples.
 * hbarc_over_E: per trajectory (length count), may be NULL if classical.
 * accumulate != 0 adds to out instead of overwriting it.
 */
int rad_oracle_ensemble_points(int32_t count, int64_t stride, const int64_t *n,
                               const double *t, const double *dz, const double *x, const double *y,
                               const double *vx, const double *vy, const double *dvz,
                               const double *ax, const double *ay, const double *az,
                               const double *gamma,
                               int64_t npts, const double *omega, const double *nx, const double *ny,
                               int model, const double *hbarc_over_E, int accumulate,
                               double *out);

/* Bits in the significand of RAD_REAL (53, 64 or 113) and threads OpenMP will use. */
int rad_oracle_real_digits(void);
int rad_oracle_threads(void);

#ifdef __cplusplus
}
#endif
#endif
