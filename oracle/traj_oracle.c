/*
 * traj_oracle.c -- CPU ORACLE for the synthetic-well trajectory generator (test infrastructure, not
 * product; same rules as rad_oracle.h: only tests/, smoke() and bench.py's CPU legs may use it, and it
 * shares nothing with the CUDA path).
 *
 * What it computes: `count` independent particles in a static transverse well,
 * integrated with the fixed-step velocity-Verlet scheme of the workload recipe, and the
 * longitudinal bookkeeping the radiation integral needs, all in long double, step by step:
 *
 *   a_k = A(r_k);  v_h = v_k + (dt/2) a_k;  r_{k+1} = r_k + dt v_h;  v_{k+1} = v_h + (dt/2) A(r_{k+1})
 *   well 0 (planar cosine):   A_x = -kappa sin(2 pi x / L),  A_y = 0
 *   well 1 (axial, exp):      A   = -kappa (r / |r|) exp(-|r| / L),  A(0) = 0
 *   t_k = k dt
 *   dvz_k = -(vx_k^2 + vy_k^2)/2                         leading-order relation, PAPER.md:28 (north_star)
 *   dz_k  = dz_{k-1} + (dvz_k + dvz_{k-1}) dt / 2,  dz_0 = 0   (dz = z - beta0 t)
 *   az_k  = -(vx_k ax_k + vy_k ay_k)                      d(dvz)/dt
 *   gamma_k = gamma
 *
 * The paper's own solver (RK45 + Doyle-Turner potentials + Monte-Carlo scattering)
 * needs tables that are not available; "many particle trajectories evaluated in parallel on the GPU" is
 * its stated outlook.
 * Pins (tests/test_traj_oracle.py): free particle, harmonic-limit period, energy conservation O(dt^2),
 * angular-momentum conservation in the axial well, time-reversal.
 */
#include <math.h>
#include <stdint.h>

typedef long double real;

static void accel(int well, real kappa, real L, real x, real y, real *ax, real *ay)
{
    if (well == 0) {
        *ax = -kappa * sinl(2.0L * 3.14159265358979323846264338327950288L * x / L);
        *ay = 0;
    } else {
        const real r = sqrtl(x * x + y * y);
        if (r == 0) { *ax = 0; *ay = 0; return; }
        const real s = -kappa * expl(-r / L) / r;
        *ax = s * x;
        *ay = s * y;
    }
}

/* Arrays t..gam: [count][stride] doubles, row p = particle p, first n entries written.  Returns 0 / -1. */
int traj_oracle_generate(int well, double kappa, double L, double gamma, double dt,
                         int32_t count, int64_t n, int64_t stride,
                         const double *x0, const double *y0, const double *vx0, const double *vy0,
                         double *t, double *dz, double *x, double *y, double *vx, double *vy,
                         double *dvz, double *ax, double *ay, double *az, double *gam)
{
    if (well < 0 || well > 1 || count < 1 || n < 2 || stride < n || !(dt > 0) || !(L > 0)) return -1;
#pragma omp parallel for schedule(dynamic, 1)
    for (int32_t p = 0; p < count; ++p) {
        const int64_t o = (int64_t)p * stride;
        const real h = dt;
        real rx = x0[p], ry = y0[p], wx = vx0[p], wy = vy0[p], a_x, a_y;
        real dzk = 0, dvz_prev = 0;
        accel(well, kappa, L, rx, ry, &a_x, &a_y);
        for (int64_t k = 0; k < n; ++k) {
            const real dvzk = -(wx * wx + wy * wy) / 2;
            if (k > 0) dzk += (dvzk + dvz_prev) * h / 2;
            dvz_prev = dvzk;
            t[o + k] = (double)(h * (real)k);
            x[o + k] = (double)rx;  y[o + k] = (double)ry;
            vx[o + k] = (double)wx; vy[o + k] = (double)wy;
            ax[o + k] = (double)a_x; ay[o + k] = (double)a_y;
            dvz[o + k] = (double)dvzk; dz[o + k] = (double)dzk;
            az[o + k] = (double)(-(wx * a_x + wy * a_y));
            gam[o + k] = gamma;
            const real hx = wx + h / 2 * a_x, hy = wy + h / 2 * a_y;
            rx += h * hx; ry += h * hy;
            accel(well, kappa, L, rx, ry, &a_x, &a_y);
            wx = hx + h / 2 * a_x; wy = hy + h / 2 * a_y;
        }
    }
    return 0;
}
