// rad.cu -- sm_100a FP64 kernels and the C ABI of include/rad.h.
//
// Hot path:
//   rad_pack_kernel      a0/a1  caller SoA -> chunk records (trapezoid weights folded into the
//                               accelerations, 1/(2 gamma^2) - dvz, chunk-relative phase terms,
//                               double-double chunk base)                 PAPER.md:34-46 (eqs. 3-7)
//   rad_main_kernel      a0-a5  one CTA per tile of 128 (angle, omega-group) threads x W omegas;
//                               trajectory chunks staged by TMA bulk copies into a 3-stage
//                               shared-memory ring; per-thread complex accumulation;
//                               epilogue |A|^2 with the variant's coefficients
//                                                          PAPER.md:23 (eq. 1), :56 (eq. 9), :62-68 (eqs. 10-12)
//   rad_finalize_kernel  a6/a7  ordered reduction of time-split amplitudes / trajectory-split
//                               spectra
//   rad_angular_sum_kernel      sum of the cube over angles
//   rad_sep_kernel (rad_sep.cuh) a0-a7 again for tensor grids that fill its tiles (the default path): the phasor of
//                               eq. (7) factorised into T(omega, n_x) Y(omega, n_y), warp-specialised CTAs in
//                               thread-block cluster pairs that share a table through distributed shared memory
//   rad_fused_kernel (rad_fused.cuh) a0-a6 in ONE cooperative launch for one short trajectory on a small grid
//   rad_ang_final_*_kernel      second pass of the angular spectrum formed in the main kernels' epilogue (no cube)
//   (launch planning: rad_plan.h)
//   rad_sum_cubes_kernel        ordered sum of partial cubes (ensemble shards)
//   rad_traj_kernel (rad_traj.cuh)  synthetic-well trajectories on the device
#include <atomic>
#include <cmath>
#include <cstdio>
#include <cstring>
#include <new>
#include <vector>

#include <cuda_runtime.h>

#include "../../include/rad.h"
#include "rad_device.cuh"
#include "rad_plan.h"

namespace rad {

#ifndef RAD_W
#define RAD_W 8
#endif
#ifndef RAD_DEG
#define RAD_DEG 5            // polynomial set of sincos_coeffs.h: 5 = LO (1e-13, default), 6 = HI (2e-16)
#endif
constexpr int TPB = 128;     // threads per CTA: one (angle, omega-group) each
constexpr int W = RAD_W;     // omegas per thread (register tile)
constexpr int STAGES = 3;    // shared-memory ring depth
constexpr int SMEM_WT = W * TPB * 16;            // per-thread omega*/2pi double-doubles, parked in smem
constexpr int SMEM_BYTES = STAGES * CHUNK_BYTES + SMEM_WT + STAGES * 8;

struct MainParams {
    const double *packed;     // [count][cpt][CHUNK_DBL]
    const int64_t *n_dev;     // samples per trajectory (device) or nullptr -> n_single
    const double *lam_dev;    // hbar c / E per trajectory (device) or nullptr -> lam_single
    int64_t n_single;
    double lam_single;
    int count, cpt;
    const double *omega, *thx, *thy;
    int n_omega, n_thx, n_thy;
    int model, mode, p_slices, t_slices, accumulate;
    double *out;              // first element of this launch's part of the cube
    int out_nx;               // row stride of the cube (n_thx of the whole grid)
    int64_t out_plane;        // omega stride of the cube (n_thx * n_thy of the whole grid)
    double *partial;
    int64_t t_pad;            // tiles * TPB
    // direct kernel on the L-shaped rest of the angle plane (the separable kernel took [0, l_x0) x [0, l_y0));
    // l_x0 < 0: the whole tensor grid.  n_thx, n_thy are the whole plane's in that case.
    int l_x0, l_y0;
    // angular spectrum (MODE_DIRECT only): per-(CTA, omega slot) sums over the CTA's angles instead of the cube
    int ang, ang_groups;      // ang_groups: omega groups a CTA of the direct kernel can span
    double cut2;              // theta_cut^2, <= 0: no mask
    double *ang_partial;
    int cl;                   // separable kernel: 2 = launched as cluster pairs that share the T table, else 1
};

// Angles a launch of the direct kernel covers, and the (i_x, i_y) of its a-th angle.
__host__ __device__ __forceinline__ int angle_count(int n_thx, int n_thy, int l_x0, int l_y0) {
    return l_x0 < 0 ? n_thx * n_thy : (n_thx - l_x0) * n_thy + l_x0 * (n_thy - l_y0);
}
__device__ __forceinline__ void angle_of(const MainParams &P, int a, int &ix, int &iy) {
    if (P.l_x0 < 0) { ix = a % P.n_thx; iy = a / P.n_thx; return; }
    const int rx = P.n_thx - P.l_x0, n1 = rx * P.n_thy;
    if (a < n1) { ix = P.l_x0 + a % rx; iy = a / rx; }              // columns right of the interior, all rows
    else { const int j = a - n1; ix = j % P.l_x0; iy = P.l_y0 + j / P.l_x0; }   // rows above it, interior columns
}

}  // namespace rad
#include "rad_sep.cuh"
#include "rad_traj.cuh"
namespace rad {

// ------------------------------------------------------------------------------ pack (a0, a1)
// P0 = t/(2 gamma^2) - dz as a double-double
__device__ __forceinline__ dd phase_offset_dd(double gamma, double t, double dz, double &a_hi) {
    dd g2 = two_prod(gamma, gamma);
    dd den = {2.0 * g2.hi, 2.0 * g2.lo};
    dd a = d_div_dd(1.0, den);                      // 1/(2 gamma^2)
    a_hi = a.hi;
    dd at = dd_mul_d(a, t);
    dd s = two_sum(at.hi, -dz);
    return fast_two_sum(s.hi, s.lo + at.lo);
}

__device__ __forceinline__ void pack_one(const rad_traj_batch &b, const int64_t *n_dev, int64_t n_single,
                                         const int64_t *off_dev, int cpt, double *packed, int p, int64_t slot);

__global__ void __launch_bounds__(256)
rad_pack_kernel(rad_traj_batch b, const int64_t *n_dev, int64_t n_single, const int64_t *off_dev, int cpt,
                double *packed) {
    const int64_t slot = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (slot >= (int64_t)cpt * CH) return;
    for (int p = blockIdx.y; p < b.count; p += gridDim.y)           // gridDim.y <= 65535 trajectories at a time
        pack_one(b, n_dev, n_single, off_dev, cpt, packed, p, slot);
}

__device__ __forceinline__ void pack_one(const rad_traj_batch &b, const int64_t *n_dev, int64_t n_single,
                                         const int64_t *off_dev, int cpt, double *packed, int p, int64_t slot) {
    const int64_t n = n_dev ? n_dev[p] : n_single;
    const int c = (int)(slot / CH), i = (int)(slot % CH);
    const int64_t c0 = (int64_t)c * CH;
    if (c0 >= n) return;                              // chunk never read
    const int64_t o = off_dev ? off_dev[p] : (int64_t)p * b.stride;     // first sample of trajectory / section p
    const int nvalid = (int)min((int64_t)CH, n - c0);
    const int64_t kb = c0 + min(CH / 2, nvalid - 1);  // base sample of the chunk
    double *chunk = packed + ((int64_t)p * cpt + c) * CHUNK_DBL;

    double ab;
    const dd P0b = phase_offset_dd(b.gamma[o + kb], b.t[o + kb], b.dz[o + kb], ab);
    if (i == 0) {
        chunk[0] = P0b.hi; chunk[1] = P0b.lo;
        chunk[2] = b.t[o + kb]; chunk[3] = b.x[o + kb]; chunk[4] = b.y[o + kb];
        chunk[5] = b.gamma[o]; chunk[6] = 0.0; chunk[7] = 0.0;
    }
    double *rec = chunk + HDR + i * REC;
    const int64_t k = c0 + i;
    if (k >= n) {                                     // zero-weight padding, q = 1
        rec[0] = 1.0;
#pragma unroll
        for (int j = 1; j < REC; ++j) rec[j] = 0.0;
        return;
    }
    const double tk = b.t[o + k];
    const double w = 0.5 * (b.t[o + min(k + 1, n - 1)] - b.t[o + max(k - 1, (int64_t)0)]);
    double ak;
    const dd P0k = phase_offset_dd(b.gamma[o + k], tk, b.dz[o + k], ak);
    const dd dP = dd_add(P0k, dd_neg(P0b));
    rec[0] = ak - b.dvz[o + k];
    rec[1] = b.vx[o + k];
    rec[2] = b.vy[o + k];
    rec[3] = w * b.ax[o + k];
    rec[4] = w * b.ay[o + k];
    rec[5] = w * b.az[o + k];
    rec[6] = dP.hi + dP.lo;
    rec[7] = tk - b.t[o + kb];
    rec[8] = b.x[o + k] - b.x[o + kb];
    rec[9] = b.y[o + k] - b.y[o + kb];
}

// ------------------------------------------------------------------------------ epilogue (a5)
// d2I/dw dOmega (units of e^2) from A_x, A_y (and J); A_z = -(n_x A_x + n_y A_y) is the
// transversality identity of eqs. (3)-(5).
template <int NC>
__device__ __forceinline__ double spectrum_value(const double (&acc)[NC], double nx, double ny,
                                                 int model, double u, double gamma0) {
    const double INV_4PI2 = 0.025330295910584442860969;   // 1/(4 pi^2)
    // imaginary accumulators hold Im/sqrt(2) (see phasor_turns): their squares count twice
    const double azr = -(nx * acc[0] + ny * acc[2]);
    const double azi = -(nx * acc[1] + ny * acc[3]);
    const double S = acc[0] * acc[0] + acc[2] * acc[2] + azr * azr
                   + 2.0 * (acc[1] * acc[1] + acc[3] * acc[3] + azi * azi);
    if (!(u < 1.0)) return __longlong_as_double(0x7ff8000000000000LL);   // no final state: NaN
    if (model == RAD_CLASSICAL) return S * INV_4PI2;
    const double e = 1.0 - u;
    if (model == RAD_SPIN0) return e * S * INV_4PI2;
    double J2 = 0.0;
    if (NC == 6) J2 = acc[4] * acc[4] + 2.0 * acc[5] * acc[5];
    return (0.5 * (1.0 + e * e) * S + u * u / (2.0 * gamma0 * gamma0) * J2) * INV_4PI2;
}

// ------------------------------------------------------------------------------ shared pieces of the direct kernels
// Chunk base phase in turns, per omega, reduced to [-1/2, 1/2] (a3, the exact part):
// psi_b = P0_b + theta^2/2 t_b - n_x x_b - n_y y_b as a double-double, times omega*/2pi (double-double, parked
// in shared memory at wt[j * stride]).  Returns gamma[0] of the trajectory (header slot 5).
__device__ __forceinline__ double chunk_base_phase(const double *ck, dd h, double nx, double ny,
                                                   const double2 *wt, int stride, double (&p0)[W]) {
    const double2 h01 = *reinterpret_cast<const double2 *>(ck);
    const double2 h23 = *reinterpret_cast<const double2 *>(ck + 2);
    const double2 h45 = *reinterpret_cast<const double2 *>(ck + 4);
    dd psi = {h01.x, h01.y};                               // P0_b
    psi = dd_add(psi, dd_mul_d(h, h23.x));                 // + theta^2/2 * t_b
    psi = dd_add(psi, dd_neg(two_prod(nx, h23.y)));        // - n_x x_b
    psi = dd_add(psi, dd_neg(two_prod(ny, h45.x)));        // - n_y y_b
#pragma unroll
    for (int j = 0; j < W; ++j) {
        const double2 w = wt[j * stride];
        p0[j] = dd_frac(dd_mul(dd{w.x, w.y}, psi));
    }
    return h45.y;
}

// One sample record against one angle and W omegas: a2 (integrand geometry, eqs. 3, 4, 6, 12), a3 (phase and
// phasor), a4 (complex accumulation).
template <int NC, int DEG>
__device__ __forceinline__ void accumulate_sample(const double *rec, double nx, double ny, double hhi,
                                                  const double (&wh)[W], const double (&p0)[W],
                                                  double (&acc)[W][NC]) {
    const double2 r01 = *reinterpret_cast<const double2 *>(rec);       // D0, vx
    const double2 r23 = *reinterpret_cast<const double2 *>(rec + 2);   // vy, w ax
    const double2 r45 = *reinterpret_cast<const double2 *>(rec + 4);   // w ay, w az
    const double2 r67 = *reinterpret_cast<const double2 *>(rec + 6);   // dP0, dt
    const double2 r89 = *reinterpret_cast<const double2 *>(rec + 8);   // dx, dy
    // a2: integrand geometry, independent of omega (eqs. 3, 4, 6, 12)
    const double D = r01.x - hhi;                  // round bracket of eqs. 3-5
    const double ux = nx - r01.y, uy = ny - r23.x;
    const double bx = fma(ny, uy, D);              // n_y(n_y - v_y) + D
    const double by = fma(nx, ux, D);              // n_x(n_x - v_x) + D
    const double q = fma(nx, ux, bx);              // eq. 6 denominator
    const double g = inv_square(q);
    const double s1 = fma(ny, r45.x, r45.y);       // w(az + n_y ay)
    const double s2 = fma(nx, r23.y, r45.y);       // w(az + n_x ax)
    const double fx = fma(s1, ux, -(bx * r23.y)) * g;      // eq. 3 (times w)
    const double fy = fma(s2, uy, -(by * r45.x)) * g;      // eq. 4 (times w)
    double hj = 0.0;
    if (NC == 6) hj = fma(nx, r23.y, s1) * g;      // eq. 12 integrand (times w)
    // eq. 7 relative to the chunk base
    const double dpsi = fma(-ny, r89.y, fma(-nx, r89.x, fma(hhi, r67.y, r67.x)));
#pragma unroll
    for (int j = 0; j < W; ++j) {
        double cs, sn;
        phasor_turns<DEG>(fma(wh[j], dpsi, p0[j]), cs, sn);            // a3 (sn = sin/sqrt2)
        acc[j][0] = fma(fx, cs, acc[j][0]);                              // a4
        acc[j][1] = fma(fx, sn, acc[j][1]);
        acc[j][2] = fma(fy, cs, acc[j][2]);
        acc[j][3] = fma(fy, sn, acc[j][3]);
        if (NC == 6) {
            acc[j][4] = fma(hj, cs, acc[j][4]);
            acc[j][5] = fma(hj, sn, acc[j][5]);
        }
    }
}

// theta^2 / 2 as a double-double
__device__ __forceinline__ dd half_theta2_dd(double nx, double ny) {
    dd xx = two_prod(nx, nx), yy = two_prod(ny, ny);
    dd s = two_sum(xx.hi, yy.hi);
    s = fast_two_sum(s.hi, s.lo + (xx.lo + yy.lo));
    return {0.5 * s.hi, 0.5 * s.lo};
}

// ------------------------------------------------------------------------------ main (a0-a5)
// NC = number of real accumulators per omega: 4 (A_x, A_y) or 6 (+ J, spin-1/2).
// GEN: the general instantiation -- angles on the L-shaped rest of a two-part plan and / or the angular-spectrum
// epilogue.  The plain one (cube on a whole tensor grid) is what the BASELINE configs run; the extra index
// arithmetic of the general one costs it registers (255 + spills with 6 accumulators per omega: -30 % measured).
template <int NC, int DEG, bool GEN>
__global__ void __launch_bounds__(TPB, 1)
rad_main_kernel(const MainParams P) {
    extern __shared__ __align__(128) unsigned char smem_raw[];
    double *ring = reinterpret_cast<double *>(smem_raw);
    double2 *wt_sm = reinterpret_cast<double2 *>(smem_raw + STAGES * CHUNK_BYTES);   // [W][TPB]
    uint64_t *bars = reinterpret_cast<uint64_t *>(smem_raw + STAGES * CHUNK_BYTES + SMEM_WT);
    const int tid = threadIdx.x;

    // ---- this thread's grid coordinates: flattened (omega-group, angle), angle fastest
    const int A = angle_count(P.n_thx, P.n_thy, P.l_x0, P.l_y0);
    const int n_wg = (P.n_omega + W - 1) / W;
    const int64_t T = (int64_t)n_wg * A;
    const int64_t gid = (int64_t)blockIdx.x * TPB + tid;
    const int64_t gc = min(gid, T - 1);
    const int wg = (int)(gc / A), a = (int)(gc % A);
    double nx, ny;
    {
        int ix = a % P.n_thx, iy = a / P.n_thx;
        if (GEN) angle_of(P, a, ix, iy);
        nx = P.thx[ix]; ny = P.thy[iy];
    }
    const dd h = half_theta2_dd(nx, ny);               // theta^2 / 2, double-double
    auto omega_of = [&](int j) { return P.omega[min(wg * W + j, P.n_omega - 1)]; };

    // ---- this CTA's slice of the (trajectory, chunk) axis
    const int slice = blockIdx.y;
    int p_begin, p_end, ts = 0;
    if (P.mode == MODE_TSPLIT) { p_begin = slice / P.t_slices; p_end = p_begin + 1; ts = slice % P.t_slices; }
    else { p_begin = (int)((int64_t)slice * P.count / P.p_slices);
           p_end = (int)((int64_t)(slice + 1) * P.count / P.p_slices); }

    auto chunk_range = [&](int p, int &c0, int &c1) {
        const int64_t n = P.n_dev ? P.n_dev[p] : P.n_single;
        const int nch = (int)((n + CH - 1) / CH);
        if (P.mode == MODE_TSPLIT) { c0 = (int)((int64_t)ts * nch / P.t_slices);
                                     c1 = (int)((int64_t)(ts + 1) * nch / P.t_slices); }
        else { c0 = 0; c1 = nch; }
    };

    if (tid == 0) {
        for (int s = 0; s < STAGES; ++s) mbar_init(&bars[s], 1);
        mbar_fence_init();
    }
    __syncthreads();

    // producer cursor (thread 0 only): next chunk to request
    int pp = p_begin, pc = 0, pc1 = 0;
    uint32_t issued = 0;
    if (tid == 0 && pp < p_end) chunk_range(pp, pc, pc1);
    auto produce = [&]() {                            // request one more chunk if any is left
        while (pp < p_end && pc >= pc1) {             // move on to the next trajectory
            ++pp;
            if (pp < p_end) chunk_range(pp, pc, pc1);
        }
        if (pp >= p_end) return;
        const int s = issued % STAGES;
        mbar_expect_tx(&bars[s], CHUNK_BYTES);
        tma_load_1d(ring + (size_t)s * CHUNK_DBL,
                    P.packed + ((int64_t)pp * P.cpt + pc) * CHUNK_DBL, CHUNK_BYTES, &bars[s]);
        ++pc;
        ++issued;
    };
    if (tid == 0)
        for (int s = 0; s < STAGES; ++s) produce();

    uint32_t it = 0;                                  // chunks consumed so far by this CTA
    double S_sum[W];
#pragma unroll
    for (int j = 0; j < W; ++j) S_sum[j] = 0.0;

    for (int p = p_begin; p < p_end; ++p) {
        // ---- per-trajectory constants: omega* / 2 pi as a double-double, u = hbar omega / E
        const double lam = P.lam_dev ? P.lam_dev[p] : P.lam_single;
        // (kept in shared memory: only the high words are needed inside the sample loop)
        double wh[W];
#pragma unroll
        for (int j = 0; j < W; ++j) {
            const double om = omega_of(j);
            dd u = two_prod(om, lam);
            dd d = two_sum(1.0, -u.hi);
            d = fast_two_sum(d.hi, d.lo - u.lo);      // 1 - u
            dd wst = d_div_dd(om, d);                 // omega* = omega / (1 - u)
            dd wt = dd_mul(wst, dd{INV_2PI_HI, INV_2PI_LO});
            wt_sm[j * TPB + tid] = make_double2(wt.hi, wt.lo);
            wh[j] = wt.hi;
        }
        double acc[W][NC];
#pragma unroll
        for (int j = 0; j < W; ++j)
#pragma unroll
            for (int c = 0; c < NC; ++c) acc[j][c] = 0.0;
        double gamma0 = 1.0;

        int c0, c1;
        chunk_range(p, c0, c1);
        for (int c = c0; c < c1; ++c, ++it) {
            const int s = it % STAGES;
            mbar_wait(&bars[s], (it / STAGES) & 1);
            const double *ck = ring + (size_t)s * CHUNK_DBL;

            // ---- chunk base phase in turns, per omega, reduced to [-1/2, 1/2]  (a3, exact part)
            double p0[W];
            gamma0 = chunk_base_phase(ck, h, nx, ny, wt_sm + tid, TPB, p0);

            // ---- samples of the chunk
            const double *rec = ck + HDR;
#pragma unroll 1
            for (int k = 0; k < CH; ++k, rec += REC) {
                accumulate_sample<NC, DEG>(rec, nx, ny, h.hi, wh, p0, acc);
            }
            __syncthreads();                          // every thread is done with stage s
            if (tid == 0) produce();
        }

        // ---- end of this trajectory (or of this time slice of it)
        if (P.mode == MODE_TSPLIT) {
            double *dst = P.partial + (int64_t)slice * NC * W * P.t_pad + gid;
#pragma unroll
            for (int c = 0; c < NC; ++c)
#pragma unroll
                for (int j = 0; j < W; ++j) dst[(int64_t)(c * W + j) * P.t_pad] = acc[j][c];
        } else {
#pragma unroll
            for (int j = 0; j < W; ++j)
                S_sum[j] += spectrum_value<NC>(acc[j], nx, ny, P.model, omega_of(j) * lam, gamma0);
        }
    }

    if (P.mode == MODE_PSLICE) {
        double *dst = P.partial + (int64_t)slice * W * P.t_pad + gid;
#pragma unroll
        for (int j = 0; j < W; ++j) dst[(int64_t)j * P.t_pad] = S_sum[j];
    } else if (GEN && P.ang && P.mode == MODE_DIRECT) {
        // ---- angular spectrum: sum of this CTA's angles per omega, in thread order (N1)
        __syncthreads();                              // the ring is free: every chunk has been consumed
        double *red = ring;                           // [TPB][W]
        const bool inside = gid < T && (P.cut2 <= 0.0 || fma(nx, nx, ny * ny) <= P.cut2);
#pragma unroll
        for (int j = 0; j < W; ++j) red[tid * W + j] = inside ? S_sum[j] : 0.0;
        __syncthreads();
        const int64_t g0 = (int64_t)blockIdx.x * TPB;
        const int wg_first = (int)(g0 / A);
        for (int slot = tid; slot < P.ang_groups * W; slot += TPB) {
            const int g = slot / W, j = slot % W;
            const int64_t lo = max(g0, (int64_t)(wg_first + g) * A), hi = min(g0 + TPB, (int64_t)(wg_first + g + 1) * A);
            double sum = 0.0;
            for (int64_t t = lo; t < hi; ++t) sum += red[(int)(t - g0) * W + j];
            P.ang_partial[((int64_t)blockIdx.x * P.ang_groups + g) * W + j] = sum;
        }
    } else if (P.mode == MODE_DIRECT && gid < T) {
        int ix = a % P.n_thx, iy = a / P.n_thx;       // (recomputed: not kept in registers across the time loop)
        if (GEN) angle_of(P, a, ix, iy);
#pragma unroll
        for (int j = 0; j < W; ++j) {
            const int iw = wg * W + j;
            if (iw < P.n_omega) {
                double *o = P.out + iw * P.out_plane + (int64_t)iy * P.out_nx + ix;
                *o = P.accumulate ? *o + S_sum[j] : S_sum[j];
            }
        }
    }
}

// angular spectrum, second pass for the direct kernel: spec[i_w] (+)= d_solid * sum over the tiles that hold
// omega group i_w / W, in ascending tile order.  One CTA per omega: 256 threads sum contiguous blocks of tiles,
// thread 0 adds the 256 block sums in order (fixed order: deterministic).
__global__ void __launch_bounds__(256)
rad_ang_final_direct_kernel(const double *partial, int A, int groups, int n_omega, double d_solid, int accumulate,
                            double *spec) {
    __shared__ double red[256];
    const int iw = blockIdx.x, wg = iw / W, j = iw % W;
    const int64_t t_lo = (int64_t)wg * A / TPB, t_hi = ((int64_t)(wg + 1) * A - 1) / TPB + 1;    // tiles [t_lo, t_hi)
    const int64_t per = (t_hi - t_lo + 255) / 256;
    double s = 0.0;
    for (int64_t t = t_lo + threadIdx.x * per; t < min(t_hi, t_lo + (threadIdx.x + 1) * per); ++t) {
        const int g = wg - (int)(t * TPB / A);
        s += partial[(t * groups + g) * W + j];
    }
    red[threadIdx.x] = s;
    __syncthreads();
    if (threadIdx.x == 0) {
        double tot = 0.0;
        for (int k = 0; k < 256; ++k) tot += red[k];
        tot *= d_solid;
        spec[iw] = accumulate ? spec[iw] + tot : tot;
    }
}

// ------------------------------------------------------------------------------ finalize (a6, a7)
template <int NC>
__global__ void __launch_bounds__(TPB)
rad_finalize_kernel(const MainParams P) {
    const int A = angle_count(P.n_thx, P.n_thy, P.l_x0, P.l_y0);
    const int n_wg = (P.n_omega + W - 1) / W;
    const int64_t T = (int64_t)n_wg * A;
    const int64_t gid = (int64_t)blockIdx.x * TPB + threadIdx.x;
    if (gid >= T) return;
    const int wg = (int)(gid / A), a = (int)(gid % A);
    int ix, iy;
    angle_of(P, a, ix, iy);
    const double nx = P.thx[ix], ny = P.thy[iy];
    {                                                 // gridDim.y = W: one omega of the register tile per CTA row
        const int j = blockIdx.y;
        const int iw = wg * W + j;
        if (iw >= P.n_omega) return;
        const double om = P.omega[iw];
        double total = 0.0;
        if (P.mode == MODE_PSLICE) {
            for (int s = 0; s < P.p_slices; ++s)                       // slices ascending
                total += P.partial[((int64_t)s * W + j) * P.t_pad + gid];
        } else {
            for (int p = 0; p < P.count; ++p) {                        // trajectories ascending
                double acc[NC];
#pragma unroll
                for (int c = 0; c < NC; ++c) acc[c] = 0.0;
                for (int s = 0; s < P.t_slices; ++s) {                 // time slices ascending
                    const double *src = P.partial + (int64_t)(p * P.t_slices + s) * NC * W * P.t_pad + gid;
#pragma unroll
                    for (int c = 0; c < NC; ++c) acc[c] += src[(int64_t)(c * W + j) * P.t_pad];
                }
                const double lam = P.lam_dev ? P.lam_dev[p] : P.lam_single;
                const double gamma0 = P.packed[(int64_t)p * P.cpt * CHUNK_DBL + 5];
                total += spectrum_value<NC>(acc, nx, ny, P.model, om * lam, gamma0);
            }
        }
        double *o = P.out + iw * P.out_plane + (int64_t)iy * P.out_nx + ix;
        *o = P.accumulate ? *o + total : total;
    }
}

}  // namespace rad
#include "rad_fused.cuh"
namespace rad {

// ------------------------------------------------------------------------------ angular sum
// one CTA per omega; fixed-order tree reduction in shared memory (deterministic)
__global__ void __launch_bounds__(256)
rad_angular_sum_kernel(const double *cube, const double *thx, const double *thy, int n_thx, int n_thy,
                       double d_solid, double cut2, double *spec) {
    __shared__ double red[256];
    const int A = n_thx * n_thy;
    const double *src = cube + (int64_t)blockIdx.x * A;
    double s = 0.0;
    for (int a = threadIdx.x; a < A; a += 256) {
        const double nx = thx[a % n_thx], ny = thy[a / n_thx];
        if (cut2 <= 0.0 || nx * nx + ny * ny <= cut2) s += src[a];
    }
    red[threadIdx.x] = s;
    __syncthreads();
    for (int st = 128; st > 0; st >>= 1) {
        if (threadIdx.x < st) red[threadIdx.x] += red[threadIdx.x + st];
        __syncthreads();
    }
    if (threadIdx.x == 0) spec[blockIdx.x] = red[0] * d_solid;
}

// ------------------------------------------------------------------------------ number spectrum
// dN/dw = (dI/dw) / (hbar w), PAPER.md:50-56 (eq. 8 is stated for the number spectrum)
__global__ void __launch_bounds__(256)
rad_number_spectrum_kernel(const double *spec, const double *omega, int n, double hbar_c, double *number) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) number[i] = spec[i] / (hbar_c * omega[i]);
}

// ------------------------------------------------------------------------------ ordered cube sum
// out[m] (+)= cubes[0][m] + cubes[1][m] + ... in ascending index order (a7 across shards)
__global__ void __launch_bounds__(256)
rad_sum_cubes_kernel(const double *cubes, int count, int64_t m, int accumulate, double *out) {
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= m) return;
    double s = accumulate ? out[i] : 0.0;
    for (int c = 0; c < count; ++c) s += cubes[(int64_t)c * m + i];
    out[i] = s;
}

// ------------------------------------------------------------------------------ FP64 peak probe
__global__ void __launch_bounds__(256)
rad_fma_peak_kernel(double *sink, int iters, double a, double b) {
    double x[16];
#pragma unroll
    for (int i = 0; i < 16; ++i) x[i] = 1.0 + 1e-9 * (threadIdx.x + i);
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int r = 0; r < 8; ++r)
#pragma unroll
            for (int i = 0; i < 16; ++i) x[i] = fma(x[i], a, x[(i + 1) & 15]);   // two register operands + one: no bank stall
    }
    double s = 0.0;
#pragma unroll
    for (int i = 0; i < 16; ++i) s += x[i];
    if (s == 12345.678) sink[0] = s;      // never true; keeps the chains alive
}

// =============================================================================== host side
static std::atomic<int64_t> g_launches{0};
static thread_local char g_err[256] = "no CUDA error recorded";

static int cuda_fail(cudaError_t e, const char *what) {
    snprintf(g_err, sizeof g_err, "%s: %s", what, cudaGetErrorString(e));
    return RAD_ECUDA;
}
#define CK(call)                                              \
    do {                                                      \
        cudaError_t e_ = (call);                              \
        if (e_ != cudaSuccess) return cuda_fail(e_, #call);   \
    } while (0)

// ---- per-device facts and one-time setup, keyed by the current device (one process may drive several GPUs)
constexpr int MAX_DEV = 64;
struct DeviceState {
    std::atomic<int> sms{0};
    std::atomic<int> fused_resident[2];               // co-resident CTAs of rad_fused_kernel<4>, <6>; 0 = not asked yet
    std::atomic<unsigned> attr_done{0};               // bit per kernel whose dynamic shared-memory limit is set
    std::atomic<int> pool_done{0};
};
static DeviceState g_dev[MAX_DEV];

static int current_device() {
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess) { cudaGetLastError(); return -1; }
    return dev >= 0 && dev < MAX_DEV ? dev : -1;
}

static int sm_count() {
    const int dev = current_device();
    if (dev < 0) return 0;
    int n = g_dev[dev].sms.load();
    if (n == 0) {
        if (cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) { cudaGetLastError(); n = 0; }
        g_dev[dev].sms.store(n);
    }
    return n;
}

template <typename K>
static cudaError_t ensure_smem(K kernel, int bit, int bytes) {
    const int dev = current_device();
    if (dev < 0) return cudaErrorNoDevice;
    if (g_dev[dev].attr_done.load() & (1u << bit)) return cudaSuccess;
    const cudaError_t e = cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes);
    if (e == cudaSuccess) g_dev[dev].attr_done.fetch_or(1u << bit);
    return e;
}

// CTAs of the fused kernel the current device holds at once (0: no device / error -> the planner assumes 4 per SM)
template <int NC>
static int fused_resident() {
    const int dev = current_device();
    if (dev < 0) return 0;
    std::atomic<int> &slot = g_dev[dev].fused_resident[NC == 6];
    int v = slot.load();
    if (v == 0) {
        int per_sm = 0;
        int per_sm_gen = 0;                          // (the smaller of the two instantiations: one number plans both)
        if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, rad_fused_kernel<NC, RAD_DEG, false>, FUSED_TPB, FUSED_SMEM)
                != cudaSuccess
            || cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm_gen, rad_fused_kernel<NC, RAD_DEG, true>, FUSED_TPB,
                                                             FUSED_SMEM) != cudaSuccess) { cudaGetLastError(); per_sm = 0; }
        per_sm = std::min(per_sm, per_sm_gen);
        v = per_sm * sm_count();
        slot.store(v > 0 ? v : -1);
    }
    return v > 0 ? v : 0;
}
static int fused_resident_for(int nc) {
    const int v = nc == 6 ? fused_resident<6>() : fused_resident<4>();
    return v > 0 ? v : 4 * 148;                       // no device: plan as for a B200
}

// ---- per-call timing (rad_options.profile)
}  // namespace rad
struct rad_profile {
    cudaEvent_t ev[4];
    bool have_reduce;
};
namespace rad {
static void prof_mark(rad_profile *pr, int i, cudaStream_t st) {
    if (!pr) return;
    cudaEventRecord(pr->ev[i], st);
    if (i == 0) pr->have_reduce = false;
    if (i == 3) pr->have_reduce = true;
}

// Scratch taken from the stream-ordered pool goes back in stream order on every exit path.
struct PoolScratch {
    void *p = nullptr;
    cudaStream_t st = nullptr;
    ~PoolScratch() { if (p) cudaFreeAsync(p, st); }
};
static cudaError_t pool_alloc(void **p, size_t bytes, cudaStream_t st) {
    // keep freed scratch cached in the device's stream-ordered pool: with the default release threshold (0)
    // every synchronisation hands it back to the driver and the next call pays a fresh allocation
    // (measured: 3x slower steps on cfg 2)
    const int dev = current_device();
    if (dev >= 0 && !g_dev[dev].pool_done.exchange(1)) {
        cudaMemPool_t pool;
        if (cudaDeviceGetDefaultMemPool(&pool, dev) == cudaSuccess) {
            uint64_t keep = UINT64_MAX;
            cudaMemPoolSetAttribute(pool, cudaMemPoolAttrReleaseThreshold, &keep);
        }
        cudaGetLastError();
    }
    return cudaMallocAsync(p, bytes, st);
}

static bool grid_ok(const rad_grid *g) {
    return g && g->n_omega > 0 && g->n_thx > 0 && g->n_thy > 0 && g->omega && g->thx && g->thy;
}
static bool aligned8(const void *p) { return (reinterpret_cast<uintptr_t>(p) & 7) == 0; }
static int kernel_option(const rad_options *opt) { return opt ? opt->kernel : 0; }

static CallPlan plan_for(int count, int64_t n_max, int n_omega, int n_thx, int n_thy, int nc, int kernel, bool angular) {
    return plan_call(count, n_max, n_omega, n_thx, n_thy, nc, kernel, angular, sm_count(), fused_resident_for(nc));
}

template <int NC, int DEG>
static cudaError_t launch_main(const MainParams &mp, dim3 grid, cudaStream_t st) {
    if (mp.ang || mp.l_x0 >= 0) {
        const cudaError_t a = ensure_smem(rad_main_kernel<NC, DEG, true>, NC == 6 ? 5 : 4, SMEM_BYTES);
        if (a != cudaSuccess) return a;
        rad_main_kernel<NC, DEG, true><<<grid, TPB, SMEM_BYTES, st>>>(mp);
    } else {
        const cudaError_t a = ensure_smem(rad_main_kernel<NC, DEG, false>, NC == 6 ? 1 : 0, SMEM_BYTES);
        if (a != cudaSuccess) return a;
        rad_main_kernel<NC, DEG, false><<<grid, TPB, SMEM_BYTES, st>>>(mp);
    }
    ++g_launches;
    return cudaGetLastError();
}

template <int NC, int WY>
static cudaError_t launch_sep(const MainParams &mp, dim3 grid, cudaStream_t st) {
    if (mp.cl >= 2) {         // cluster pairs along the y (omega) tiles: thread-block clusters of 2 CTAs on neighbouring SMs
        constexpr int CLW = NC == 4 ? 3 : 2;          // (pairs along omega exist for 4 accumulators per point only)
        const bool along_w = mp.cl == 3 && NC == 4;
        const cudaError_t a = along_w ? ensure_smem(rad_sep_kernel<NC, WY, CLW>, 8, SepShape<NC, WY>::SMEM)
                                      : ensure_smem(rad_sep_kernel<NC, WY, 2>, NC == 6 ? 7 : 6, SepShape<NC, WY>::SMEM);
        if (a != cudaSuccess) return a;
        cudaLaunchConfig_t cfg = {};
        cfg.gridDim = grid; cfg.blockDim = dim3(SepRegs<NC>::THREADS); cfg.dynamicSmemBytes = SepShape<NC, WY>::SMEM;
        cfg.stream = st;
        cudaLaunchAttribute at[1];
        at[0].id = cudaLaunchAttributeClusterDimension;
        at[0].val.clusterDim.x = 2; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
        cfg.attrs = at; cfg.numAttrs = 1;
        ++g_launches;
        return along_w ? cudaLaunchKernelEx(&cfg, rad_sep_kernel<NC, WY, CLW>, mp)
                       : cudaLaunchKernelEx(&cfg, rad_sep_kernel<NC, WY, 2>, mp);
    }
    const cudaError_t a = ensure_smem(rad_sep_kernel<NC, WY, 1>, NC == 6 ? 3 : 2, SepShape<NC, WY>::SMEM);
    if (a != cudaSuccess) return a;
    rad_sep_kernel<NC, WY, 1><<<grid, SepRegs<NC>::THREADS, SepShape<NC, WY>::SMEM, st>>>(mp);
    ++g_launches;
    return cudaGetLastError();
}

template <int NC>
static cudaError_t launch_fused(FusedParams &fp, cudaStream_t st) {
    void *args[] = {&fp};
    const void *fn = fp.l_x0 >= 0 ? reinterpret_cast<const void *>(rad_fused_kernel<NC, RAD_DEG, true>)
                                  : reinterpret_cast<const void *>(rad_fused_kernel<NC, RAD_DEG, false>);
    const cudaError_t e = cudaLaunchCooperativeKernel(fn, dim3(fp.tiles, fp.slices), dim3(FUSED_TPB), args, FUSED_SMEM, st);
    ++g_launches;
    return e;
}

// Everything: pack, main, ordered reduction.  All device pointers; n_host / lam_host are host arrays.
// off_host (optional): first sample of each trajectory inside the arrays (sections of one long trajectory);
// NULL: row p starts at p * stride.  ang != nullptr: the angular spectrum instead of the cube (the caller has
// checked that the plan is one part in MODE_DIRECT).
struct AngularOut { double d_solid, cut2; double *spectrum; };

static int run_batch(const rad_traj_batch *b, const int64_t *n_host, const int64_t *off_host, const rad_grid *g,
                     int model, const double *lam_host, int accumulate, double *out, const AngularOut *ang,
                     void *workspace, size_t workspace_bytes, const rad_options *opt, cudaStream_t st) {
    if (!b || b->count < 1 || !n_host || !grid_ok(g) || (!out && !ang)) return RAD_EINVAL;
    if (model < RAD_CLASSICAL || model > RAD_SPIN_HALF) return RAD_EINVAL;
    if (model != RAD_CLASSICAL && !lam_host) return RAD_EINVAL;
    const int kopt = kernel_option(opt);
    if (kopt < RAD_KERNEL_AUTO || kopt > RAD_KERNEL_FUSED || (opt && opt->reserved != 0)) return RAD_EINVAL;
    const double *arrs[11] = {b->t, b->dz, b->x, b->y, b->vx, b->vy, b->dvz, b->ax, b->ay, b->az, b->gamma};
    for (const double *p : arrs)
        if (!p || !aligned8(p)) return RAD_EINVAL;
    if ((out && !aligned8(out)) || !aligned8(g->omega) || !aligned8(g->thx) || !aligned8(g->thy)) return RAD_EINVAL;
    int64_t n_max = 0;
    for (int p = 0; p < b->count; ++p) {
        if (n_host[p] < 2 || n_host[p] > b->stride) return RAD_EINVAL;
        if (off_host && (off_host[p] < 0 || off_host[p] + n_host[p] > b->stride)) return RAD_EINVAL;
        n_max = std::max(n_max, n_host[p]);
        if (model != RAD_CLASSICAL && !(lam_host[p] >= 0.0)) return RAD_EDOMAIN;
    }
    const int nc = model == RAD_SPIN_HALF ? 6 : 4;
    const CallPlan cp = plan_for(b->count, n_max, g->n_omega, g->n_thx, g->n_thy, nc, kopt, ang != nullptr);
    if (kopt == RAD_KERNEL_FUSED && !cp.fused) return RAD_EINVAL;
    // (a single section of a sectioned trajectory is one trajectory that starts at off_host[0]: the fused kernel
    // takes it like any other.  The plan of a fused call overlays the partial amplitudes on the packed buffer it does
    // not need, so a fused plan must never fall through to the multi-launch path below.)
    const bool fused = cp.fused;
    if (ang && !(cp.nparts == 1 && cp.part[0].plan.mode == MODE_DIRECT)) return RAD_EINVAL;
    if (workspace && (reinterpret_cast<uintptr_t>(workspace) & 255)) return RAD_EINVAL;
    if (workspace && workspace_bytes < cp.total) return RAD_ENOSPACE;
    PoolScratch pool;
    char *ws = static_cast<char *>(workspace);
    if (!ws) {
        void *pnew = nullptr;
        CK(pool_alloc(&pnew, cp.total, st));
        ws = static_cast<char *>(pnew);
        pool.p = pnew; pool.st = st;
    }
    rad_profile *prof = opt ? opt->profile : nullptr;

    if (fused) {              // ---- one cooperative launch does rows a0-a6 (rad_fused.cuh)
        FusedParams fp{};
        const int64_t o = off_host ? off_host[0] : 0;
        fp.tr = rad_traj{n_host[0], b->t + o, b->dz + o, b->x + o, b->y + o, b->vx + o, b->vy + o, b->dvz + o,
                         b->ax + o, b->ay + o, b->az + o, b->gamma + o};
        fp.lam = model == RAD_CLASSICAL ? 0.0 : lam_host[0];
        fp.omega = g->omega; fp.thx = g->thx; fp.thy = g->thy;
        fp.n_omega = g->n_omega; fp.n_thx = g->n_thx; fp.n_thy = g->n_thy;
        fp.model = model; fp.accumulate = accumulate ? 1 : 0;
        fp.tiles = cp.fused_tiles; fp.slices = cp.fused_slices;
        fp.partial = reinterpret_cast<double *>(ws + cp.part[0].off_partial);
        fp.out = out; fp.l_x0 = -1; fp.l_y0 = -1;
        prof_mark(prof, 0, st);
        prof_mark(prof, 1, st);
        const cudaError_t e = nc == 6 ? launch_fused<6>(fp, st) : launch_fused<4>(fp, st);
        if (e != cudaSuccess) return cuda_fail(e, "rad_fused_kernel");
        prof_mark(prof, 2, st);
        return RAD_OK;
    }

    double *packed = reinterpret_cast<double *>(ws + cp.off_packed);
    int64_t *n_dev = nullptr;
    double *lam_dev = nullptr;
    int64_t *off_dev = nullptr;
    if (off_host) {
        off_dev = reinterpret_cast<int64_t *>(ws + cp.off_start);
        CK(cudaMemcpyAsync(off_dev, off_host, (size_t)b->count * sizeof(int64_t), cudaMemcpyHostToDevice, st));
    }
    if (b->count > 1) {
        n_dev = reinterpret_cast<int64_t *>(ws + cp.off_n);
        CK(cudaMemcpyAsync(n_dev, n_host, (size_t)b->count * sizeof(int64_t), cudaMemcpyHostToDevice, st));
        if (model != RAD_CLASSICAL) {
            lam_dev = reinterpret_cast<double *>(ws + cp.off_lam);
            CK(cudaMemcpyAsync(lam_dev, lam_host, (size_t)b->count * sizeof(double), cudaMemcpyHostToDevice, st));
        }
    }
    prof_mark(prof, 0, st);
    {   // a0/a1: pack
        dim3 grid((unsigned)(((int64_t)cp.cpt * CH + 255) / 256), (unsigned)std::min(b->count, 65535));
        rad_pack_kernel<<<grid, 256, 0, st>>>(*b, n_dev, n_host[0], off_dev, cp.cpt, packed);
        ++g_launches;
        CK(cudaGetLastError());
    }
    prof_mark(prof, 1, st);
    MainParams mps[2];
    for (int i = 0; i < cp.nparts; ++i) {             // main kernels of all parts first, then their reductions
        const Part &pt = cp.part[i];
        const Plan &pl = pt.plan;
        MainParams &mp = mps[i];
        mp = MainParams{};
        mp.packed = packed; mp.n_dev = n_dev; mp.lam_dev = lam_dev;
        mp.n_single = n_host[0];
        mp.lam_single = model == RAD_CLASSICAL ? 0.0 : lam_host[0];
        mp.count = b->count; mp.cpt = cp.cpt;
        mp.omega = g->omega; mp.thx = g->thx; mp.thy = g->thy;
        mp.n_omega = g->n_omega; mp.n_thx = pt.n_thx; mp.n_thy = pt.n_thy;
        mp.model = model; mp.mode = pl.mode; mp.p_slices = pl.p_slices; mp.t_slices = pl.t_slices;
        mp.accumulate = accumulate ? 1 : 0;
        mp.out = out; mp.out_nx = g->n_thx; mp.out_plane = (int64_t)g->n_thx * g->n_thy;
        mp.partial = reinterpret_cast<double *>(ws + pt.off_partial);
        mp.t_pad = pl.t_pad;
        mp.l_x0 = pt.l_x0; mp.l_y0 = pt.l_y0;
        mp.cl = pt.cl;
        if (ang) {
            mp.ang = 1; mp.cut2 = ang->cut2;
            mp.ang_groups = std::min((g->n_omega + W - 1) / W, (TPB + pt.angles - 1) / pt.angles + 1);
            mp.ang_partial = reinterpret_cast<double *>(ws + cp.off_ang);
        }
        if (pt.f_tiles > 0) {                         // the rest of a two-part plan through the fused single-launch kernel
            const int64_t o = off_host ? off_host[0] : 0;
            FusedParams fp{};
            fp.tr = rad_traj{n_host[0], b->t + o, b->dz + o, b->x + o, b->y + o, b->vx + o, b->vy + o, b->dvz + o,
                             b->ax + o, b->ay + o, b->az + o, b->gamma + o};
            fp.lam = mp.lam_single;
            fp.omega = g->omega; fp.thx = g->thx; fp.thy = g->thy;
            fp.n_omega = g->n_omega; fp.n_thx = pt.n_thx; fp.n_thy = pt.n_thy;
            fp.model = model; fp.accumulate = accumulate ? 1 : 0;
            fp.tiles = pt.f_tiles; fp.slices = pt.f_slices;
            fp.partial = mp.partial;
            fp.out = out; fp.l_x0 = pt.l_x0; fp.l_y0 = pt.l_y0; fp.out_nx = g->n_thx;
            fp.out_plane = (int64_t)g->n_thx * g->n_thy;
            const cudaError_t ef = nc == 6 ? launch_fused<6>(fp, st) : launch_fused<4>(fp, st);
            if (ef != cudaSuccess) return cuda_fail(ef, "rad_fused_kernel");
            continue;
        }
        dim3 grid((unsigned)pl.tiles, (unsigned)pl.slices());
        cudaError_t e;
        if (pt.kernel == K_SEP) e = nc == 6 ? launch_sep<6, 2>(mp, grid, st) : launch_sep<4, 4>(mp, grid, st);
        else e = nc == 6 ? launch_main<6, RAD_DEG>(mp, grid, st) : launch_main<4, RAD_DEG>(mp, grid, st);
        if (e != cudaSuccess) return cuda_fail(e, pt.kernel == K_SEP ? "rad_sep_kernel" : "rad_main_kernel");
    }
    prof_mark(prof, 2, st);
    bool reduced = false;
    for (int i = 0; i < cp.nparts; ++i) {
        const Part &pt = cp.part[i];
        const Plan &pl = pt.plan;
        const MainParams &mp = mps[i];
        if (ang) {
            if (pt.kernel == K_SEP) {
                const int wy = nc == 6 ? 2 : 4;
                const int angle_tiles = ((pt.n_thx + 15) / 16) * ((pt.n_thy + 4 * wy - 1) / (4 * wy));
                rad_ang_final_sep_kernel<<<g->n_omega, 256, 0, st>>>(mp.ang_partial, angle_tiles, g->n_omega,
                                                                     ang->d_solid, 0, ang->spectrum);
            } else {
                rad_ang_final_direct_kernel<<<g->n_omega, 256, 0, st>>>(mp.ang_partial, pt.angles, mp.ang_groups,
                                                                        g->n_omega, ang->d_solid, 0, ang->spectrum);
            }
            ++g_launches;
            CK(cudaGetLastError());
            reduced = true;
        } else if (pl.mode != MODE_DIRECT && pt.f_tiles == 0) {
            if (pt.kernel == K_SEP) {
                if (nc == 6) rad_sep_finalize_kernel<6, 2><<<dim3(pl.tiles, 8), SEP_CONS, 0, st>>>(mp);
                else rad_sep_finalize_kernel<4, 4><<<dim3(pl.tiles, 16), SEP_CONS, 0, st>>>(mp);
            } else {
                if (nc == 6) rad_finalize_kernel<6><<<dim3(pl.tiles, W), TPB, 0, st>>>(mp);
                else rad_finalize_kernel<4><<<dim3(pl.tiles, W), TPB, 0, st>>>(mp);
            }
            ++g_launches;
            CK(cudaGetLastError());
            reduced = true;
        }
    }
    if (reduced) prof_mark(prof, 3, st);
    return RAD_OK;
}

static int run_single(const rad_traj *t, const rad_grid *g, int model, double lam, double *out,
                      void *ws, size_t ws_bytes, const rad_options *opt, cudaStream_t st) {
    if (!t) return RAD_EINVAL;
    rad_traj_batch b{1, t->n, nullptr, t->t, t->dz, t->x, t->y, t->vx, t->vy, t->dvz,
                     t->ax, t->ay, t->az, t->gamma};
    const int64_t n = t->n;
    return run_batch(&b, &n, nullptr, g, model, &lam, 0, out, nullptr, ws, ws_bytes, opt, st);
}

}  // namespace rad

// =============================================================================== C ABI
using namespace rad;

extern "C" {

int rad_classical(const rad_traj *traj, const rad_grid *grid, double *out,
                  void *workspace, size_t workspace_bytes, const rad_options *opt, void *cuda_stream) {
    return run_single(traj, grid, RAD_CLASSICAL, 0.0, out, workspace, workspace_bytes, opt,
                      static_cast<cudaStream_t>(cuda_stream));
}

int rad_semiclassical(const rad_traj *traj, const rad_grid *grid, int spin, double hbarc_over_E,
                      double *out, void *workspace, size_t workspace_bytes, const rad_options *opt,
                      void *cuda_stream) {
    if (spin != 0 && spin != 1) return RAD_EINVAL;
    if (!(hbarc_over_E >= 0.0)) return RAD_EDOMAIN;
    return run_single(traj, grid, spin == 0 ? RAD_SPIN0 : RAD_SPIN_HALF, hbarc_over_E, out,
                      workspace, workspace_bytes, opt, static_cast<cudaStream_t>(cuda_stream));
}

int rad_ensemble_sum(const rad_traj_batch *batch, const rad_grid *grid, rad_model model,
                     const double *hbarc_over_E, int accumulate, double *out,
                     void *workspace, size_t workspace_bytes, const rad_options *opt, void *cuda_stream) {
    if (!batch) return RAD_EINVAL;
    return run_batch(batch, batch->n, nullptr, grid, (int)model, hbarc_over_E, accumulate, out, nullptr,
                     workspace, workspace_bytes, opt, static_cast<cudaStream_t>(cuda_stream));
}

int rad_sections_sum(const rad_traj *traj, int32_t n_sections, const int64_t *start, const rad_grid *grid,
                     rad_model model, const double *hbarc_over_E, int accumulate, double *out,
                     void *workspace, size_t workspace_bytes, const rad_options *opt, void *cuda_stream) {
    if (!traj || !start || n_sections < 1) return RAD_EINVAL;
    std::vector<int64_t> n(n_sections), off(n_sections);
    for (int s = 0; s < n_sections; ++s) {            // section s = samples start[s] .. start[s+1], both included
        if (start[s] < 0 || start[s + 1] <= start[s] || start[s + 1] > traj->n - 1) return RAD_EINVAL;
        off[s] = start[s];
        n[s] = start[s + 1] - start[s] + 1;
    }
    rad_traj_batch b{n_sections, traj->n, n.data(), traj->t, traj->dz, traj->x, traj->y, traj->vx, traj->vy,
                     traj->dvz, traj->ax, traj->ay, traj->az, traj->gamma};
    return run_batch(&b, n.data(), off.data(), grid, (int)model, hbarc_over_E, accumulate, out, nullptr,
                     workspace, workspace_bytes, opt, static_cast<cudaStream_t>(cuda_stream));
}

int rad_sections_check(int32_t n_sections, const double *t_start, const double *gamma0,
                       const double *hbarc_over_E, double omega_min, int32_t *short_sections, int32_t cap) {
    if (n_sections < 1 || !t_start || !gamma0 || cap < 0 || (cap > 0 && !short_sections)) return RAD_EINVAL;
    if (!(omega_min > 0.0)) return RAD_EDOMAIN;
    int found = 0;
    for (int s = 0; s < n_sections; ++s) {
        if (!(t_start[s + 1] > t_start[s])) return RAD_EINVAL;
        const double lf = rad_formation_length(gamma0[s], omega_min, hbarc_over_E ? hbarc_over_E[s] : 0.0);
        if (lf < 0.0) return RAD_EDOMAIN;
        if (t_start[s + 1] - t_start[s] <= lf) {      // c = 1: a time span is a length
            if (found < cap) short_sections[found] = s;
            ++found;
        }
    }
    return found;
}

int rad_angular_sum(const double *cube, const rad_grid *grid, double d_solid_angle, double theta_cut,
                    double *spectrum, void *cuda_stream) {
    if (!cube || !spectrum || !grid_ok(grid)) return RAD_EINVAL;
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    rad_angular_sum_kernel<<<grid->n_omega, 256, 0, st>>>(
        cube, grid->thx, grid->thy, grid->n_thx, grid->n_thy, d_solid_angle,
        theta_cut > 0.0 ? theta_cut * theta_cut : 0.0, spectrum);
    ++g_launches;
    CK(cudaGetLastError());
    return RAD_OK;
}

int rad_number_spectrum(const double *spectrum, const double *omega, int32_t n, double hbar_c, double *number,
                        void *cuda_stream) {
    if (!spectrum || !omega || !number || n < 1) return RAD_EINVAL;
    if (!(hbar_c > 0.0)) return RAD_EDOMAIN;
    rad_number_spectrum_kernel<<<(n + 255) / 256, 256, 0, static_cast<cudaStream_t>(cuda_stream)>>>(
        spectrum, omega, n, hbar_c, number);
    ++g_launches;
    CK(cudaGetLastError());
    return RAD_OK;
}

// Does the angular spectrum of this call come straight out of the main kernel's epilogue?
static bool angular_is_fused(const CallPlan &cp) { return cp.nparts == 1 && cp.part[0].plan.mode == MODE_DIRECT && !cp.fused; }

static size_t angular_workspace(int count, int64_t n_max, int n_omega, int n_thx, int n_thy) {
    size_t need = 0;
    bool all_fused = true;
    for (int kernel = 0; kernel <= 2; ++kernel)
        for (int nc = 4; nc <= 6; nc += 2) {
            const CallPlan cp = plan_for(count, n_max, n_omega, n_thx, n_thy, nc, kernel, true);
            if (angular_is_fused(cp)) need = std::max(need, cp.total);
            else all_fused = false;
        }
    if (!all_fused)           // cube path (grids of fewer than 8 tiles per SM): the call's own workspace + the cube
        need = std::max(need, align_up(rad_workspace_bytes(count, n_max, n_omega, n_thx, n_thy), 256)
                                  + align_up((size_t)n_omega * n_thx * n_thy * 8, 256));
    return need;
}

size_t rad_angular_spectrum_workspace_bytes(int32_t count, int64_t n_max, int32_t n_omega, int32_t n_thx,
                                            int32_t n_thy) {
    if (count < 1 || n_max < 2 || n_omega < 1 || n_thx < 1 || n_thy < 1) return 0;
    return angular_workspace(count, n_max, n_omega, n_thx, n_thy);
}

int rad_angular_spectrum(const rad_traj_batch *batch, const rad_grid *grid, rad_model model,
                         const double *hbarc_over_E, double d_solid_angle, double theta_cut, double *spectrum,
                         void *workspace, size_t workspace_bytes, const rad_options *opt, void *cuda_stream) {
    if (!batch || !grid_ok(grid) || !spectrum || !workspace) return RAD_EINVAL;
    if (reinterpret_cast<uintptr_t>(workspace) & 255) return RAD_EINVAL;
    if (model < RAD_CLASSICAL || model > RAD_SPIN_HALF) return RAD_EINVAL;
    int64_t n_max = 0;
    if (!batch->n || batch->count < 1) return RAD_EINVAL;
    for (int p = 0; p < batch->count; ++p) n_max = std::max(n_max, batch->n[p]);
    if (n_max < 2) return RAD_EINVAL;
    const int kopt = kernel_option(opt);
    if (kopt < RAD_KERNEL_AUTO || kopt > RAD_KERNEL_SEPARABLE) return RAD_EINVAL;
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    const int nc = model == RAD_SPIN_HALF ? 6 : 4;
    const double cut2 = theta_cut > 0.0 ? theta_cut * theta_cut : 0.0;
    const CallPlan cp = plan_for(batch->count, n_max, grid->n_omega, grid->n_thx, grid->n_thy, nc, kopt, true);
    if (angular_is_fused(cp)) {                       // no cube: sums formed in the main kernel's epilogue
        if (workspace_bytes < cp.total) return RAD_ENOSPACE;
        const AngularOut ang{d_solid_angle, cut2, spectrum};
        return run_batch(batch, batch->n, nullptr, grid, (int)model, hbarc_over_E, 0, nullptr, &ang,
                         workspace, workspace_bytes, opt, st);
    }
    // small grid (fewer than 8 tiles per SM, i.e. a cube below 40 MB): the cube inside the workspace, then its sum
    const size_t inner = align_up(rad_workspace_bytes(batch->count, n_max, grid->n_omega, grid->n_thx, grid->n_thy), 256);
    const size_t cube_bytes = align_up((size_t)grid->n_omega * grid->n_thx * grid->n_thy * 8, 256);
    if (workspace_bytes < inner + cube_bytes) return RAD_ENOSPACE;
    double *cube = reinterpret_cast<double *>(static_cast<char *>(workspace) + inner);
    const int rc = run_batch(batch, batch->n, nullptr, grid, (int)model, hbarc_over_E, 0, cube, nullptr,
                             workspace, inner, opt, st);
    if (rc != RAD_OK) return rc;
    return rad_angular_sum(cube, grid, d_solid_angle, theta_cut, spectrum, cuda_stream);
}

int rad_generate_trajectories(rad_well well, double kappa, double length, double gamma, double dt,
                              double sigma, uint64_t seed, int32_t count, int64_t n, int64_t stride,
                              const double *x0, const double *y0, const double *vx0, const double *vy0,
                              const rad_traj_buffers *out, void *cuda_stream) {
    if (!out || !x0 || !y0 || !vx0 || !vy0 || count < 1 || n < 2 || stride < n) return RAD_EINVAL;
    if (well != RAD_WELL_COSINE && well != RAD_WELL_AXIAL_EXP && well != RAD_WELL_HARMONIC_MS) return RAD_EINVAL;
    if (!(dt > 0.0) || !(length > 0.0) || !(gamma >= 1.0) || !(sigma >= 0.0)) return RAD_EDOMAIN;
    if (well == RAD_WELL_HARMONIC_MS && !(kappa > 0.0)) return RAD_EDOMAIN;
    double *arrs[11] = {out->t, out->dz, out->x, out->y, out->vx, out->vy, out->dvz, out->ax, out->ay, out->az,
                        out->gamma};
    for (double *p : arrs)
        if (!p || !aligned8(p)) return RAD_EINVAL;
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    const TrajOut o{out->t, out->dz, out->x, out->y, out->vx, out->vy, out->dvz, out->ax, out->ay, out->az, out->gamma};
    const unsigned blocks = (unsigned)((count + 31) / 32);            // one warp per CTA (rad_traj.cuh TrajStage)
    if (well == RAD_WELL_HARMONIC_MS)
        rad_traj_ms_kernel<<<blocks, 32, 0, st>>>(kappa, gamma, dt, sigma, seed, count, n, stride, x0, y0, vx0, vy0, o);
    else if (well == RAD_WELL_COSINE)
        rad_traj_kernel<0><<<blocks, 32, 0, st>>>(kappa, length, gamma, dt, count, n, stride, x0, y0, vx0, vy0, o);
    else
        rad_traj_kernel<1><<<blocks, 32, 0, st>>>(kappa, length, gamma, dt, count, n, stride, x0, y0, vx0, vy0, o);
    ++g_launches;
    CK(cudaGetLastError());
    return RAD_OK;
}

int rad_sum_cubes(const double *cubes, int32_t count, int64_t m, int accumulate, double *out,
                  void *cuda_stream) {
    if (!cubes || !out || count < 1 || m < 1 || !aligned8(cubes) || !aligned8(out)) return RAD_EINVAL;
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    rad_sum_cubes_kernel<<<(unsigned)((m + 255) / 256), 256, 0, st>>>(cubes, count, m, accumulate ? 1 : 0, out);
    ++g_launches;
    CK(cudaGetLastError());
    return RAD_OK;
}

size_t rad_workspace_bytes(int32_t count, int64_t n_max, int32_t n_omega, int32_t n_thx, int32_t n_thy) {
    if (count < 1 || n_max < 2 || n_omega < 1 || n_thx < 1 || n_thy < 1) return 0;
    size_t need = 0;                                   // whichever kernel and variant the call ends up using
    for (int kernel = 0; kernel <= 3; ++kernel)
        for (int nc = 4; nc <= 6; nc += 2)
            need = std::max(need, plan_for(count, n_max, n_omega, n_thx, n_thy, nc, kernel, false).total);
    return need;
}

// ---- host-buffer variants: H2D once, compute, D2H once
int rad_ensemble_sum_host(const rad_traj_batch *b, const rad_grid *g, rad_model model,
                          const double *hbarc_over_E, int accumulate, double *out, const rad_options *opt,
                          void *cuda_stream) {
    if (!b || b->count < 1 || !b->n || !grid_ok(g) || !out) return RAD_EINVAL;
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    const size_t row = (size_t)b->stride, tot = row * b->count;
    const size_t M = (size_t)g->n_omega * g->n_thx * g->n_thy;
    const size_t ng = (size_t)g->n_omega + g->n_thx + g->n_thy;
    const double *src[11] = {b->t, b->dz, b->x, b->y, b->vx, b->vy, b->dvz, b->ax, b->ay, b->az, b->gamma};
    for (const double *p : src)
        if (!p) return RAD_EINVAL;
    double *dev = nullptr;
    CK(pool_alloc(reinterpret_cast<void **>(&dev), (11 * tot + ng + M) * sizeof(double), st));
    PoolScratch pool;
    pool.p = dev; pool.st = st;
    // Arrays that follow one another in host memory (a caller that keeps its SoA block -- and the grid behind it -- in
    // one allocation) go over in ONE copy: the device layout is the same sequence t, dz, ..., gamma, omega, thx, thy,
    // and for a small problem every separate copy costs more than its bytes (config 1: 14 copies ~ 85 us against a
    // 47 us kernel).
    const double *d[11];
    double *gw = dev + 11 * tot, *gx = gw + g->n_omega, *gy = gx + g->n_thx, *dout = gy + g->n_thy;
    {
        const double *hsrc[14];
        size_t cnt[14], off[14];
        for (int i = 0; i < 11; ++i) { hsrc[i] = src[i]; cnt[i] = tot; off[i] = i * tot; d[i] = dev + i * tot; }
        hsrc[11] = g->omega; cnt[11] = g->n_omega; off[11] = 11 * tot;
        hsrc[12] = g->thx;   cnt[12] = g->n_thx;   off[12] = off[11] + g->n_omega;
        hsrc[13] = g->thy;   cnt[13] = g->n_thy;   off[13] = off[12] + g->n_thx;
        for (int i = 0; i < 14;) {
            int j = i;
            size_t run = cnt[i];
            while (j + 1 < 14 && hsrc[j + 1] == hsrc[j] + cnt[j]) { ++j; run += cnt[j]; }
            CK(cudaMemcpyAsync(dev + off[i], hsrc[i], run * sizeof(double), cudaMemcpyHostToDevice, st));
            i = j + 1;
        }
    }
    if (accumulate) CK(cudaMemcpyAsync(dout, out, M * sizeof(double), cudaMemcpyHostToDevice, st));
    rad_traj_batch db{b->count, b->stride, b->n, d[0], d[1], d[2], d[3], d[4], d[5], d[6], d[7], d[8], d[9], d[10]};
    rad_grid dg{g->n_omega, g->n_thx, g->n_thy, gw, gx, gy};
    int rc = run_batch(&db, b->n, nullptr, &dg, (int)model, hbarc_over_E, accumulate, dout, nullptr, nullptr, 0, opt, st);
    if (rc == RAD_OK) {
        cudaError_t e = cudaMemcpyAsync(out, dout, M * sizeof(double), cudaMemcpyDeviceToHost, st);
        if (e != cudaSuccess) rc = cuda_fail(e, "D2H");
    }
    cudaFreeAsync(dev, st);
    pool.p = nullptr;
    cudaError_t e = cudaStreamSynchronize(st);
    if (rc == RAD_OK && e != cudaSuccess) rc = cuda_fail(e, "cudaStreamSynchronize");
    return rc;
}

int rad_eval_host(const rad_traj *t, const rad_grid *g, rad_model model, double hbarc_over_E,
                  double *out, const rad_options *opt, void *cuda_stream) {
    if (!t) return RAD_EINVAL;
    if (model != RAD_CLASSICAL && !(hbarc_over_E >= 0.0)) return RAD_EDOMAIN;
    const int64_t n = t->n;
    rad_traj_batch b{1, t->n, &n, t->t, t->dz, t->x, t->y, t->vx, t->vy, t->dvz, t->ax, t->ay, t->az, t->gamma};
    return rad_ensemble_sum_host(&b, g, model, &hbarc_over_E, 0, out, opt, cuda_stream);
}

double rad_measure_fp64_peak(double millis, void *cuda_stream) {
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    const int sms = sm_count();
    if (sms <= 0) return -1.0;
    double *sink = nullptr;
    if (cudaMalloc(reinterpret_cast<void **>(&sink), 8) != cudaSuccess) return -1.0;
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0); cudaEventCreate(&e1);
    const int blocks = sms * 8, threads = 256;
    auto run = [&](int iters) -> float {
        cudaEventRecord(e0, st);
        rad_fma_peak_kernel<<<blocks, threads, 0, st>>>(sink, iters, -0.4999, 1e-7);
        ++g_launches;
        cudaEventRecord(e1, st);
        cudaEventSynchronize(e1);
        float ms = 0.f;
        cudaEventElapsedTime(&ms, e0, e1);
        return ms;
    };
    run(64);                                           // warm-up
    int iters = 512;
    float ms = run(iters);
    if (ms > 0.f && millis > ms) {                     // scale to the requested duration
        iters = (int)std::min(1e8, iters * (millis / ms));
        ms = run(iters);
    }
    const double flops = 2.0 * 16 * 8 * (double)iters * blocks * threads;
    cudaEventDestroy(e0); cudaEventDestroy(e1);
    cudaFree(sink);
    if (cudaGetLastError() != cudaSuccess || ms <= 0.f) return -1.0;
    return flops / (ms * 1e-3);
}

int64_t rad_launch_count(void) { return g_launches.load(); }

static int kernel_code(const CallPlan &cp) { return cp.fused ? 3 : cp.part[0].kernel == K_SEP ? 2 : 1; }

int rad_plan_kernel(int32_t count, int64_t n_max, int32_t n_omega, int32_t n_thx, int32_t n_thy,
                    rad_model model, int32_t kernel) {
    if (count < 1 || n_max < 2 || n_omega < 1 || n_thx < 1 || n_thy < 1) return RAD_EINVAL;
    if (model < RAD_CLASSICAL || model > RAD_SPIN_HALF || kernel < 0 || kernel > 3) return RAD_EINVAL;
    const int nc = model == RAD_SPIN_HALF ? 6 : 4;
    const CallPlan cp = plan_for(count, n_max, n_omega, n_thx, n_thy, nc, kernel, false);
    if (kernel == 3 && !cp.fused) return RAD_EINVAL;
    return kernel_code(cp);
}

double rad_formation_length(double gamma, double omega, double hbarc_over_E) {
    const double u = omega * hbarc_over_E;            // hbar omega / E
    if (!(gamma >= 1.0) || !(omega > 0.0) || !(u >= 0.0) || !(u < 1.0)) return -1.0;
    return 2.0 * gamma * gamma * (1.0 - u) / omega;   // l_f = 2 gamma^2 (E - w) / (E w)
}

int rad_plan_describe(int32_t count, int64_t n_max, int32_t n_omega, int32_t n_thx, int32_t n_thy, rad_model model,
                      int32_t kernel, int32_t *plan) {
    if (!plan || count < 1 || n_max < 2 || n_omega < 1 || n_thx < 1 || n_thy < 1) return RAD_EINVAL;
    if (model < RAD_CLASSICAL || model > RAD_SPIN_HALF || kernel < 0 || kernel > 3) return RAD_EINVAL;
    const int nc = model == RAD_SPIN_HALF ? 6 : 4;
    const CallPlan cp = plan_for(count, n_max, n_omega, n_thx, n_thy, nc, kernel, false);
    if (kernel == 3 && !cp.fused) return RAD_EINVAL;
    const Plan &pl = cp.part[0].plan;
    plan[0] = kernel_code(cp);
    plan[1] = cp.fused ? MODE_TSPLIT : pl.mode;
    plan[2] = cp.fused ? cp.fused_tiles : pl.tiles;
    plan[3] = cp.fused ? cp.fused_slices : pl.slices();
    plan[4] = cp.fused ? cp.fused_slices : pl.t_slices;
    plan[5] = cp.cpt;
    plan[6] = cp.fused ? 1 : cp.nparts;
    plan[7] = !cp.fused && cp.nparts == 2 ? cp.part[0].n_thx : 0;
    plan[8] = !cp.fused && cp.nparts == 2 ? cp.part[0].n_thy : 0;
    plan[9] = cp.launches();
    plan[10] = cp.fused ? 1 : cp.part[0].cl;
    return RAD_OK;
}

rad_profile *rad_profile_create(void) {
    rad_profile *p = new (std::nothrow) rad_profile{};
    if (!p) return nullptr;
    for (int i = 0; i < 4; ++i)
        if (cudaEventCreate(&p->ev[i]) != cudaSuccess) {
            cudaGetLastError();
            for (int k = 0; k < i; ++k) cudaEventDestroy(p->ev[k]);
            delete p;
            return nullptr;
        }
    return p;
}

void rad_profile_destroy(rad_profile *p) {
    if (!p) return;
    for (auto &e : p->ev) cudaEventDestroy(e);
    delete p;
}

int rad_profile_read(rad_profile *p, float *ms) {
    if (!p || !ms) return RAD_EINVAL;
    CK(cudaEventSynchronize(p->ev[p->have_reduce ? 3 : 2]));
    CK(cudaEventElapsedTime(&ms[0], p->ev[0], p->ev[1]));
    CK(cudaEventElapsedTime(&ms[1], p->ev[1], p->ev[2]));
    ms[2] = 0.f;
    if (p->have_reduce) CK(cudaEventElapsedTime(&ms[2], p->ev[2], p->ev[3]));
    return RAD_OK;
}

// ---- the entry point that allocates nothing (include/rad.h rad_eval_static)
// Scratch of the single-trajectory path (packed chunk records, partial amplitudes / spectra of a split plan) in a
// file-scope device array instead of caller or pool memory: every GPU that loads this library holds these bytes until
// the process exits.  In host code `g_static_scratch` is a host-side stand-in for the symbol, NOT a device address:
// the address the kernels get comes from cudaGetSymbolAddress, asked once per device with that device current.
constexpr size_t STATIC_SCRATCH_BYTES = (size_t)16 << 20;
static __device__ __align__(256) unsigned char g_static_scratch[STATIC_SCRATCH_BYTES];
static std::atomic<void *> g_static_scratch_ptr[rad::MAX_DEV];          // per device; nullptr = not asked yet

static int static_scratch_address(void **ptr) {
    const int dev = rad::current_device();
    if (dev < 0) return rad::cuda_fail(cudaErrorNoDevice, "rad_eval_static");
    void *p = g_static_scratch_ptr[dev].load();
    if (!p) {
        const cudaError_t e = cudaGetSymbolAddress(&p, g_static_scratch);
        if (e != cudaSuccess) return rad::cuda_fail(e, "cudaGetSymbolAddress(g_static_scratch)");
        g_static_scratch_ptr[dev].store(p);
    }
    *ptr = p;
    return RAD_OK;
}

size_t rad_static_scratch_bytes(void) { return STATIC_SCRATCH_BYTES; }

int rad_eval_static(const rad_traj *traj, const rad_grid *grid, rad_model model, double hbarc_over_E, double *out,
                    const rad_options *opt, void *cuda_stream) {
    if (!traj || traj->n < 2 || !grid_ok(grid) || !out) return RAD_EINVAL;
    if (model < RAD_CLASSICAL || model > RAD_SPIN_HALF) return RAD_EINVAL;
    if (model != RAD_CLASSICAL && !(hbarc_over_E >= 0.0)) return RAD_EDOMAIN;
    const int kopt = kernel_option(opt);
    if (kopt < RAD_KERNEL_AUTO || kopt > RAD_KERNEL_FUSED || (opt && opt->reserved != 0)) return RAD_EINVAL;
    const int nc = model == RAD_SPIN_HALF ? 6 : 4;
    const CallPlan cp = plan_for(1, traj->n, grid->n_omega, grid->n_thx, grid->n_thy, nc, kopt, false);
    if (cp.total > STATIC_SCRATCH_BYTES) return RAD_ETOOBIG;          // (same plan, hence same size, as run_batch computes)
    void *scratch = nullptr;
    const int rc = static_scratch_address(&scratch);
    if (rc != RAD_OK) return rc;
    // the existing single-trajectory path with the static array as its caller workspace: with a workspace it enqueues
    // kernels only (no cudaMalloc / cudaMallocAsync / cudaFree, no host copy, no synchronisation)
    return run_single(traj, grid, (int)model, model == RAD_CLASSICAL ? 0.0 : hbarc_over_E, out, scratch,
                      STATIC_SCRATCH_BYTES, opt, static_cast<cudaStream_t>(cuda_stream));
}

const char *rad_strerror(int code) {
    switch (code) {
        case RAD_OK: return "ok";
        case RAD_EINVAL: return "invalid argument";
        case RAD_EDOMAIN: return "parameter outside the method's domain";
        case RAD_ECUDA: return g_err;
        case RAD_ENOSPACE: return "workspace too small (see rad_workspace_bytes)";
        case RAD_ETOOBIG: return "problem needs more scratch than the library's static scratch array holds "
                                 "(rad_static_scratch_bytes; use rad_classical / rad_semiclassical with a workspace)";
        default: return "unknown status";
    }
}

}  // extern "C"
