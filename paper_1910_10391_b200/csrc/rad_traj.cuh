// rad_traj.cuh -- trajectories of many particles in a static synthetic well, generated on the device
// (the paper's outlook "many particle trajectories evaluated in parallel on the GPU",
// PAPER.md:233).  Fixed-step velocity Verlet, the scheme of the workload recipe, plus the
// leading-order longitudinal bookkeeping the radiation integral needs:
//   dvz = -(vx^2 + vy^2)/2,  dz = cumulative trapezoid of dvz,  az = -(vx ax + vy ay),  t = k dt.
// One thread per particle (the time loop is a recurrence); the arrays it writes feed rad_ensemble_sum
// without a host round trip.  CUDA path only; the CPU oracle (oracle/traj_oracle.c) shares nothing with it.
#pragma once

namespace rad {

struct TrajOut { double *t, *dz, *x, *y, *vx, *vy, *dvz, *ax, *ay, *az, *gamma; };

template <int WELL>
__device__ __forceinline__ void well_accel(double kappa, double L, double x, double y, double &ax, double &ay) {
    if (WELL == 0) {                                  // planar cosine well: v'_x = -kappa sin(2 pi x / L)
        ax = -kappa * sinpi(2.0 * (x / L));
        ay = 0.0;
    } else {                                          // axial well: v'_perp = -kappa r^ exp(-r / L)
        const double r = sqrt(x * x + y * y);
        if (r == 0.0) { ax = 0.0; ay = 0.0; return; }
        const double s = -kappa * exp(-r / L) / r;
        ax = s * x;
        ay = s * y;
    }
}

template <int WELL>
__global__ void __launch_bounds__(128)
rad_traj_kernel(double kappa, double L, double gamma, double dt, int count, int64_t n, int64_t stride,
                const double *x0, const double *y0, const double *vx0, const double *vy0, TrajOut o) {
    const int p = blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= count) return;
    const int64_t base = (int64_t)p * stride;
    double rx = x0[p], ry = y0[p], wx = vx0[p], wy = vy0[p], a_x, a_y;
    double dzk = 0.0, dvz_prev = 0.0;
    const double hh = 0.5 * dt;
    well_accel<WELL>(kappa, L, rx, ry, a_x, a_y);
    for (int64_t k = 0; k < n; ++k) {
        const double dvzk = -0.5 * (wx * wx + wy * wy);
        if (k > 0) dzk += (dvzk + dvz_prev) * hh;
        dvz_prev = dvzk;
        const int64_t i = base + k;
        o.t[i] = dt * (double)k;
        o.x[i] = rx;   o.y[i] = ry;
        o.vx[i] = wx;  o.vy[i] = wy;
        o.ax[i] = a_x; o.ay[i] = a_y;
        o.dvz[i] = dvzk; o.dz[i] = dzk;
        o.az[i] = -(wx * a_x + wy * a_y);
        o.gamma[i] = gamma;
        const double hx = wx + hh * a_x, hy = wy + hh * a_y;      // half kick
        rx += dt * hx; ry += dt * hy;                            // drift
        well_accel<WELL>(kappa, L, rx, ry, a_x, a_y);
        wx = hx + hh * a_x; wy = hy + hh * a_y;                  // half kick
    }
}

}  // namespace rad
