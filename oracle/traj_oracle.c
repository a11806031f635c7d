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
 *   well 2 (planar harmonic well with multiple-scattering kicks, the recipe of configs 2 and 4; kappa = w_p^2):
 *       exact rotation of (x, u = vx / w_p) by w_p dt, then Gaussian kicks of standard deviation sigma:
 *         x_{k+1} = c x_k + s u_k,  u_{k+1} = c u_k - s x_k + (sigma / w_p) xi1_{k+1},  vy_{k+1} = vy_k + sigma xi2_{k+1}
 *         ax_k = -w_p^2 x_k + sigma xi1_k / dt,  ay_k = sigma xi2_k / dt  (xi_0 = 0),  y = cumulative trapezoid of vy
 *       xi1, xi2 of (particle p, step k): Box-Muller of the two uniforms (r + 1/2) 2^-32 made from the first two
 *       words of Philox4x32-10 (Salmon et al., SC'11) with counter (k, 0, p, 0) and key (seed low, seed high) --
 *       a counter-based generator, so that the CUDA path can draw the same numbers without sharing code.
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

/* Philox4x32-10: ten rounds of two 32 x 32 -> 64 multiplies and a key bump. */
static void philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4])
{
    uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3], k0 = key[0], k1 = key[1];
    for (int r = 0; r < 10; ++r) {
        const uint64_t p0 = (uint64_t)0xD2511F53u * c0, p1 = (uint64_t)0xCD9E8D57u * c2;
        const uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ k0, n1 = (uint32_t)p1;
        const uint32_t n2 = (uint32_t)(p0 >> 32) ^ c3 ^ k1, n3 = (uint32_t)p0;
        c0 = n0; c1 = n1; c2 = n2; c3 = n3;
        k0 += 0x9E3779B9u; k1 += 0xBB67AE85u;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

/* for the known-answer pin */
void traj_oracle_philox(const uint32_t *ctr, const uint32_t *key, uint32_t *out) { philox4x32_10(ctr, key, out); }

/* the two standard normals of (particle p, step k) */
static void kick_normals(uint64_t seed, int32_t p, int64_t k, real *xi1, real *xi2)
{
    const uint32_t ctr[4] = {(uint32_t)k, (uint32_t)((uint64_t)k >> 32), (uint32_t)p, 0u};
    const uint32_t key[2] = {(uint32_t)seed, (uint32_t)(seed >> 32)};
    uint32_t r[4];
    philox4x32_10(ctr, key, r);
    const real two32 = 4294967296.0L;
    const real u1 = ((real)r[0] + 0.5L) / two32, u2 = ((real)r[1] + 0.5L) / two32;
    const real rho = sqrtl(-2.0L * logl(u1)), ang = 2.0L * 3.14159265358979323846264338327950288L * u2;
    *xi1 = rho * cosl(ang);
    *xi2 = rho * sinl(ang);
}

/* for the statistical pin: normals of particle p, steps 0..n-1 */
void traj_oracle_normals(uint64_t seed, int32_t p, int64_t n, double *xi1, double *xi2)
{
    for (int64_t k = 0; k < n; ++k) {
        real a, b;
        kick_normals(seed, p, k, &a, &b);
        xi1[k] = (double)a; xi2[k] = (double)b;
    }
}

/* Arrays t..gam: [count][stride] doubles, row p = particle p, first n entries written.  Returns 0 / -1. */
int traj_oracle_generate(int well, double kappa, double L, double gamma, double dt, double sigma, uint64_t seed,
                         int32_t count, int64_t n, int64_t stride,
                         const double *x0, const double *y0, const double *vx0, const double *vy0,
                         double *t, double *dz, double *x, double *y, double *vx, double *vy,
                         double *dvz, double *ax, double *ay, double *az, double *gam)
{
    if (well < 0 || well > 2 || count < 1 || n < 2 || stride < n || !(dt > 0) || !(L > 0)) return -1;
#pragma omp parallel for schedule(dynamic, 1)
    for (int32_t p = 0; p < count; ++p) {
        const int64_t o = (int64_t)p * stride;
        const real h = dt;
        real rx = x0[p], ry = y0[p], wx = vx0[p], wy = vy0[p], a_x, a_y;
        real dzk = 0, dvz_prev = 0;
        if (well == 2) {                               /* harmonic rotation + scattering kicks */
            const real wp = sqrtl((real)kappa), cs = cosl(wp * h), sn = sinl(wp * h);
            real u = wx / wp, vy_prev = wy, xi1 = 0, xi2 = 0;
            for (int64_t k = 0; k < n; ++k) {
                const real vxk = u * wp;
                const real dvzk = -(vxk * vxk + wy * wy) / 2;
                if (k > 0) { dzk += (dvzk + dvz_prev) * h / 2; ry += (wy + vy_prev) * h / 2; }
                dvz_prev = dvzk; vy_prev = wy;
                a_x = -(real)kappa * rx + (real)sigma * xi1 / h;
                a_y = (real)sigma * xi2 / h;
                t[o + k] = (double)(h * (real)k);
                x[o + k] = (double)rx;  y[o + k] = (double)ry;
                vx[o + k] = (double)vxk; vy[o + k] = (double)wy;
                ax[o + k] = (double)a_x; ay[o + k] = (double)a_y;
                dvz[o + k] = (double)dvzk; dz[o + k] = (double)dzk;
                az[o + k] = (double)(-(vxk * a_x + wy * a_y));
                gam[o + k] = gamma;
                kick_normals(seed, p, k + 1, &xi1, &xi2);
                const real xn = cs * rx + sn * u;
                u = cs * u - sn * rx + (real)sigma / wp * xi1;
                rx = xn;
                wy += (real)sigma * xi2;
            }
            continue;
        }
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
