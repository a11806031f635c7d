// rad_traj.cuh -- trajectories of many particles in a static synthetic well, generated on the device
// (the paper's outlook "many particle trajectories evaluated in parallel on the GPU",
// PAPER.md:233).  Fixed-step velocity Verlet, the scheme of the workload recipe, plus the
// leading-order longitudinal bookkeeping the radiation integral needs:
//   dvz = -(vx^2 + vy^2)/2,  dz = cumulative trapezoid of dvz,  az = -(vx ax + vy ay),  t = k dt.
// One thread per particle (the time loop is a recurrence), one warp per CTA, stores staged through shared memory
// and written transposed (TrajStage); the arrays it writes feed rad_ensemble_sum without a host round trip.  CUDA path only; the CPU oracle (oracle/traj_oracle.c) shares nothing with it.
#pragma once

namespace rad {

struct TrajOut { double *t, *dz, *x, *y, *vx, *vy, *dvz, *ax, *ay, *az, *gamma; };

// Stores of the time loop.  One thread per particle writes 11 doubles per step into 11 arrays whose rows lie `stride`
// apart: written directly, every store instruction of a warp touches 32 different 32-byte sectors with 8 bytes each
// (measured: 22-25 ms for 2000 particles x 20 000 steps in all three wells alike -- the stores, not the arithmetic).
// Here a CTA is ONE warp; it collects TRAJ_T steps of its 32 particles in shared memory and then writes them
// transposed: a half-warp writes 16 consecutive steps of one particle = 128 contiguous bytes, so a store instruction
// touches two lines instead of 32 sectors (16 x fewer requests, 4 x fewer sectors).
constexpr int TRAJ_T = 16;                       // steps per flush
constexpr int TRAJ_PAD = 33;                     // row pitch of the staging buffer (conflict-free column reads)
struct TrajStage {
    double (*buf)[TRAJ_T][TRAJ_PAD];             // [11][TRAJ_T][TRAJ_PAD] in shared memory
    double *arr[11];
    int lane, p0, count;
    int64_t stride;
    __device__ __forceinline__ void put(int a, int s, double v) { buf[a][s][lane] = v; }
    // write steps [k0, k0 + nsteps) of the CTA's particles (nsteps <= TRAJ_T), all lanes take part
    __device__ __forceinline__ void flush(int64_t k0, int nsteps) {
        __syncwarp();
        const int s = lane & (TRAJ_T - 1), half = lane >> 4;
        const int64_t first = (int64_t)(p0 + half) * stride + k0 + s;     // element of particle p0 + half; + 2 stride per row
        const int rows = s < nsteps ? min(16, (count - p0 - half + 1) / 2) : 0;   // particles p0 + half + 2 r < count
#pragma unroll 1
        for (int a = 0; a < 11; ++a) {
            double *dst = arr[a] + first;
            const double *src = &buf[a][s][half];
#pragma unroll 4
            for (int r = 0; r < rows; ++r, dst += 2 * stride, src += 2) *dst = *src;
        }
        __syncwarp();
    }
};
#define RAD_TRAJ_STAGE(o)                                                                     \
    __shared__ double stage_buf[11][TRAJ_T][TRAJ_PAD];                                        \
    TrajStage W;                                                                              \
    W.buf = stage_buf;                                                                        \
    W.arr[0] = o.t; W.arr[1] = o.dz; W.arr[2] = o.x; W.arr[3] = o.y; W.arr[4] = o.vx; W.arr[5] = o.vy;   \
    W.arr[6] = o.dvz; W.arr[7] = o.ax; W.arr[8] = o.ay; W.arr[9] = o.az; W.arr[10] = o.gamma;            \
    W.lane = threadIdx.x; W.p0 = blockIdx.x * 32; W.count = count; W.stride = stride;

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

// Philox4x32-10 (Salmon, Moraes, Dror, Shaw, SC'11): counter-based, so particle p / step k draw the same
// numbers wherever and in whatever order they are evaluated.
__device__ __forceinline__ uint2 philox4x32_10_first2(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3,
                                                      uint32_t k0, uint32_t k1) {
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        const uint32_t h0 = __umulhi(0xD2511F53u, c0), l0 = 0xD2511F53u * c0;
        const uint32_t h1 = __umulhi(0xCD9E8D57u, c2), l1 = 0xCD9E8D57u * c2;
        const uint32_t n0 = h1 ^ c1 ^ k0, n2 = h0 ^ c3 ^ k1;
        c0 = n0; c1 = l1; c2 = n2; c3 = l0;
        k0 += 0x9E3779B9u; k1 += 0xBB67AE85u;
    }
    return make_uint2(c0, c1);
}

// the two standard normals of (particle p, step k): Box-Muller of (r + 1/2) 2^-32
__device__ __forceinline__ void kick_normals(uint64_t seed, int p, int64_t k, double &xi1, double &xi2) {
    const uint2 r = philox4x32_10_first2((uint32_t)k, (uint32_t)((uint64_t)k >> 32), (uint32_t)p, 0u,
                                         (uint32_t)seed, (uint32_t)(seed >> 32));
    const double u1 = ((double)r.x + 0.5) * 0x1p-32, u2 = ((double)r.y + 0.5) * 0x1p-32;
    const double rho = sqrt(-2.0 * log(u1));
    double sn, cs;
    sincospi(2.0 * u2, &sn, &cs);
    xi1 = rho * cs;
    xi2 = rho * sn;
}

// planar harmonic well (kappa = w_p^2) with Gaussian multiple-scattering kicks of standard deviation sigma on
// v_x, v_y after every step: exact rotation of (x, v_x / w_p) by w_p dt, then the kick (recipe of configs 2, 4)
__global__ void __launch_bounds__(32)
rad_traj_ms_kernel(double kappa, double gamma, double dt, double sigma, uint64_t seed, int count, int64_t n,
                   int64_t stride, const double *x0, const double *y0, const double *vx0, const double *vy0,
                   TrajOut o) {
    RAD_TRAJ_STAGE(o)
    const int p = min(blockIdx.x * 32 + (int)threadIdx.x, count - 1);     // (lanes beyond count repeat the last particle; never stored)
    const double wp = sqrt(kappa), hh = 0.5 * dt;
    double sn, cs;
    sincos(wp * dt, &sn, &cs);
    double rx = x0[p], ry = y0[p], u = vx0[p] / wp, wy = vy0[p];
    double dzk = 0.0, dvz_prev = 0.0, vy_prev = wy, xi1 = 0.0, xi2 = 0.0;
    for (int64_t k = 0; k < n; ++k) {
        const double vxk = u * wp;
        const double dvzk = -0.5 * (vxk * vxk + wy * wy);
        if (k > 0) { dzk += (dvzk + dvz_prev) * hh; ry += (wy + vy_prev) * hh; }
        dvz_prev = dvzk; vy_prev = wy;
        const double a_x = -kappa * rx + sigma * xi1 / dt, a_y = sigma * xi2 / dt;
        const int sl = (int)(k & (TRAJ_T - 1));
        W.put(0, sl, dt * (double)k);
        W.put(2, sl, rx);    W.put(3, sl, ry);
        W.put(4, sl, vxk);   W.put(5, sl, wy);
        W.put(7, sl, a_x);   W.put(8, sl, a_y);
        W.put(6, sl, dvzk);  W.put(1, sl, dzk);
        W.put(9, sl, -(vxk * a_x + wy * a_y));
        W.put(10, sl, gamma);
        if (sl == TRAJ_T - 1 || k == n - 1) W.flush(k - sl, sl + 1);
        kick_normals(seed, p, k + 1, xi1, xi2);
        const double xn = cs * rx + sn * u;
        u = cs * u - sn * rx + sigma / wp * xi1;
        rx = xn;
        wy += sigma * xi2;
    }
}

template <int WELL>
__global__ void __launch_bounds__(32)
rad_traj_kernel(double kappa, double L, double gamma, double dt, int count, int64_t n, int64_t stride,
                const double *x0, const double *y0, const double *vx0, const double *vy0, TrajOut o) {
    RAD_TRAJ_STAGE(o)
    const int p = min(blockIdx.x * 32 + (int)threadIdx.x, count - 1);     // (lanes beyond count repeat the last particle; never stored)
    double rx = x0[p], ry = y0[p], wx = vx0[p], wy = vy0[p], a_x, a_y;
    double dzk = 0.0, dvz_prev = 0.0;
    const double hh = 0.5 * dt;
    well_accel<WELL>(kappa, L, rx, ry, a_x, a_y);
    for (int64_t k = 0; k < n; ++k) {
        const double dvzk = -0.5 * (wx * wx + wy * wy);
        if (k > 0) dzk += (dvzk + dvz_prev) * hh;
        dvz_prev = dvzk;
        const int sl = (int)(k & (TRAJ_T - 1));
        W.put(0, sl, dt * (double)k);
        W.put(2, sl, rx);   W.put(3, sl, ry);
        W.put(4, sl, wx);   W.put(5, sl, wy);
        W.put(7, sl, a_x);  W.put(8, sl, a_y);
        W.put(6, sl, dvzk); W.put(1, sl, dzk);
        W.put(9, sl, -(wx * a_x + wy * a_y));
        W.put(10, sl, gamma);
        if (sl == TRAJ_T - 1 || k == n - 1) W.flush(k - sl, sl + 1);
        const double hx = wx + hh * a_x, hy = wy + hh * a_y;      // half kick
        rx += dt * hx; ry += dt * hy;                            // drift
        well_accel<WELL>(kappa, L, rx, ry, a_x, a_y);
        wx = hx + hh * a_x; wy = hy + hh * a_y;                  // half kick
    }
}

}  // namespace rad
