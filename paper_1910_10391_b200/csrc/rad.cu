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
//   rad_sep_kernel (rad_sep.cuh) a0-a7 again for tensor grids that fill its tiles: the phasor of eq. (7)
//                               factorised into T(omega, n_x) Y(omega, n_y), warp-specialised CTA
//   rad_sum_cubes_kernel        ordered sum of partial cubes (ensemble shards)
//   rad_traj_kernel (rad_traj.cuh)  synthetic-well trajectories on the device
#include <atomic>
#include <cmath>
#include <cstdio>
#include <cstring>
#include <mutex>
#include <vector>

#include <cuda_runtime.h>

#include "../../include/rad.h"
#include "rad_device.cuh"

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

enum Mode : int { MODE_DIRECT = 0, MODE_PSLICE = 1, MODE_TSPLIT = 2 };

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
    double *out;
    double *partial;
    int64_t t_pad;            // tiles * TPB
};

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

__global__ void __launch_bounds__(256)
rad_pack_kernel(rad_traj_batch b, const int64_t *n_dev, int64_t n_single, const int64_t *off_dev, int cpt,
                double *packed) {
    const int p = blockIdx.y;
    const int64_t slot = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (slot >= (int64_t)cpt * CH) return;
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

// ------------------------------------------------------------------------------ main (a0-a5)
// NC = number of real accumulators per omega: 4 (A_x, A_y) or 6 (+ J, spin-1/2).
template <int NC, int DEG>
__global__ void __launch_bounds__(TPB, 1)
rad_main_kernel(const MainParams P) {
    extern __shared__ __align__(128) unsigned char smem_raw[];
    double *ring = reinterpret_cast<double *>(smem_raw);
    double2 *wt_sm = reinterpret_cast<double2 *>(smem_raw + STAGES * CHUNK_BYTES);   // [W][TPB]
    uint64_t *bars = reinterpret_cast<uint64_t *>(smem_raw + STAGES * CHUNK_BYTES + SMEM_WT);
    const int tid = threadIdx.x;

    // ---- this thread's grid coordinates: flattened (omega-group, angle), angle fastest
    const int A = P.n_thx * P.n_thy;
    const int n_wg = (P.n_omega + W - 1) / W;
    const int64_t T = (int64_t)n_wg * A;
    const int64_t gid = (int64_t)blockIdx.x * TPB + tid;
    const int64_t gc = min(gid, T - 1);
    const int wg = (int)(gc / A), a = (int)(gc % A);
    const double nx = P.thx[a % P.n_thx], ny = P.thy[a / P.n_thx];
    dd h;                                             // theta^2 / 2, double-double
    {
        dd xx = two_prod(nx, nx), yy = two_prod(ny, ny);
        dd s = two_sum(xx.hi, yy.hi);
        s = fast_two_sum(s.hi, s.lo + (xx.lo + yy.lo));
        h = {0.5 * s.hi, 0.5 * s.lo};
    }
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
            {
                const double2 h01 = *reinterpret_cast<const double2 *>(ck);
                const double2 h23 = *reinterpret_cast<const double2 *>(ck + 2);
                const double2 h45 = *reinterpret_cast<const double2 *>(ck + 4);
                gamma0 = h45.y;
                dd psi = {h01.x, h01.y};                               // P0_b
                psi = dd_add(psi, dd_mul_d(h, h23.x));                 // + theta^2/2 * t_b
                psi = dd_add(psi, dd_neg(two_prod(nx, h23.y)));        // - n_x x_b
                psi = dd_add(psi, dd_neg(two_prod(ny, h45.x)));        // - n_y y_b
#pragma unroll
                for (int j = 0; j < W; ++j) {
                    const double2 wt = wt_sm[j * TPB + tid];
                    p0[j] = dd_frac(dd_mul(dd{wt.x, wt.y}, psi));
                }
            }

            // ---- samples of the chunk
            const double *rec = ck + HDR;
#pragma unroll 1
            for (int k = 0; k < CH; ++k, rec += REC) {
                const double2 r01 = *reinterpret_cast<const double2 *>(rec);       // D0, vx
                const double2 r23 = *reinterpret_cast<const double2 *>(rec + 2);   // vy, w ax
                const double2 r45 = *reinterpret_cast<const double2 *>(rec + 4);   // w ay, w az
                const double2 r67 = *reinterpret_cast<const double2 *>(rec + 6);   // dP0, dt
                const double2 r89 = *reinterpret_cast<const double2 *>(rec + 8);   // dx, dy
                // a2: integrand geometry, independent of omega (eqs. 3, 4, 6, 12)
                const double D = r01.x - h.hi;                 // round bracket of eqs. 3-5
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
                const double dpsi = fma(-ny, r89.y, fma(-nx, r89.x, fma(h.hi, r67.y, r67.x)));
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
    } else if (P.mode == MODE_DIRECT && gid < T) {
#pragma unroll
        for (int j = 0; j < W; ++j) {
            const int iw = wg * W + j;
            if (iw < P.n_omega) {
                double *o = P.out + (int64_t)iw * A + a;
                *o = P.accumulate ? *o + S_sum[j] : S_sum[j];
            }
        }
    }
}

// ------------------------------------------------------------------------------ finalize (a6, a7)
template <int NC>
__global__ void __launch_bounds__(TPB)
rad_finalize_kernel(const MainParams P) {
    const int A = P.n_thx * P.n_thy;
    const int n_wg = (P.n_omega + W - 1) / W;
    const int64_t T = (int64_t)n_wg * A;
    const int64_t gid = (int64_t)blockIdx.x * TPB + threadIdx.x;
    if (gid >= T) return;
    const int wg = (int)(gid / A), a = (int)(gid % A);
    const double nx = P.thx[a % P.n_thx], ny = P.thy[a / P.n_thx];
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
        double *o = P.out + (int64_t)iw * A + a;
        *o = P.accumulate ? *o + total : total;
    }
}

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

// Optional per-kernel timing of the last call (bench.py's roofline needs the main kernel's own
// duration): events recorded on the caller's stream around pack / main / finalize.
static std::atomic<int> g_prof{0};
static cudaEvent_t g_ev[4];
static bool g_ev_ready = false, g_ev_have_finalize = false;
static std::mutex g_ev_mu;

static void prof_mark(int i, cudaStream_t st) {
    if (!g_prof.load()) return;
    std::lock_guard<std::mutex> lk(g_ev_mu);
    if (!g_ev_ready) {
        for (auto &e : g_ev) cudaEventCreate(&e);
        g_ev_ready = true;
    }
    cudaEventRecord(g_ev[i], st);
    if (i == 2) g_ev_have_finalize = false;
    if (i == 3) g_ev_have_finalize = true;
}

static int cuda_fail(cudaError_t e, const char *what) {
    snprintf(g_err, sizeof g_err, "%s: %s", what, cudaGetErrorString(e));
    return RAD_ECUDA;
}
#define CK(call)                                              \
    do {                                                      \
        cudaError_t e_ = (call);                              \
        if (e_ != cudaSuccess) return cuda_fail(e_, #call);   \
    } while (0)

static int sm_count() {
    static int n = 0;
    if (n == 0) {
        int dev = 0;
        if (cudaGetDevice(&dev) != cudaSuccess) return 0;
        if (cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) n = 0;
    }
    return n;
}

static size_t align_up(size_t v, size_t a) { return (v + a - 1) / a * a; }

// Scratch taken from the stream-ordered pool goes back in stream order on every exit path.
struct PoolScratch {
    void *p = nullptr;
    cudaStream_t st = nullptr;
    ~PoolScratch() { if (p) cudaFreeAsync(p, st); }
};

// The launch plan is a pure function of the shapes (and the SM count, 148 assumed when no
// device is visible so that rad_workspace_bytes works on a CPU-only box).
struct Plan {
    int kernel;               // 0: rad_main_kernel (one phasor per eval), 1: rad_sep_kernel (separable phasor)
    int cpt, tiles, p_slices, t_slices, mode;
    int64_t t_pad;
    size_t off_packed, off_n, off_lam, off_start, off_partial, total;
};

static std::atomic<int> g_kernel_choice{0};          // rad_set_kernel: 0 auto, 1 direct, 2 separable

// The separable kernel works on tiles of 16 omega x 16 n_x x (16 or 8) n_y points: use it when padding
// the grid to whole tiles wastes less work than the kernel saves (it needs about half the FP64
// instructions per eval of the direct kernel).
static int choose_kernel(int n_omega, int n_thx, int n_thy, int nc) {
    const int choice = g_kernel_choice.load();
    if (choice == 1) return 0;
    if (choice == 2) return 1;
    const int ty = nc == 6 ? 8 : 16;
    const double padded = (double)((n_omega + 15) / 16 * 16) * ((n_thx + 15) / 16 * 16) * ((n_thy + ty - 1) / ty * ty);
    // measured speed-up of the separable kernel on full tiles: 1.8x (4 accumulators per point), 1.4x (6)
    const double break_even = nc == 6 ? 0.75 : 0.6;
    return (double)n_omega * n_thx * n_thy >= break_even * padded ? 1 : 0;
}

static Plan make_plan(int count, int64_t n_max, int n_omega, int n_thx, int n_thy, int nc, int kernel) {
    Plan pl{};
    pl.kernel = kernel;
    int sms = sm_count();
    if (sms <= 0) sms = 148;
    pl.cpt = (int)((n_max + CH - 1) / CH);
    pl.p_slices = 1; pl.t_slices = 1; pl.mode = MODE_DIRECT;
    size_t per_thread_p, per_thread_t;                // partial doubles per thread and slice
    if (kernel == 0) {
        const int64_t T = (int64_t)((n_omega + W - 1) / W) * n_thx * n_thy;
        pl.tiles = (int)((T + TPB - 1) / TPB);
        pl.t_pad = (int64_t)pl.tiles * TPB;
        per_thread_p = W; per_thread_t = (size_t)nc * W;
        // two CTAs per SM: the fewest slices k (>= 2 waves of work) whose tiles*k CTAs fill whole
        // waves of 2 * sms to >= 98.5 %
        const int slots = 2 * sms;
        if (pl.tiles < 8 * sms) {
            const int64_t kmax = std::max<int64_t>(1, (int64_t)count * std::max(1, pl.cpt));
            int best_k = 1;
            double best = 0.0;
            for (int64_t k = 1; k <= std::min<int64_t>(kmax, 8 * sms); ++k) {
                const int64_t ctas = (int64_t)pl.tiles * k;
                double eff = (double)ctas / (double)((ctas + slots - 1) / slots * slots);
                if (ctas < 2 * slots && k < kmax) eff *= 0.5;        // too few CTAs to balance: keep looking
                if (eff > best + 1e-9) { best = eff; best_k = (int)k; }
                if (eff >= 0.985) break;
            }
            if (best_k > 1) {
                if (count >= best_k) { pl.mode = MODE_PSLICE; pl.p_slices = best_k; }
                else {
                    int ts = std::min((best_k + count - 1) / count, std::max(1, pl.cpt));
                    if (ts > 1) { pl.mode = MODE_TSPLIT; pl.t_slices = ts; pl.p_slices = count; }
                    else if (count > 1) { pl.mode = MODE_PSLICE; pl.p_slices = count; }
                }
            }
        }
    } else {
        const int wy = nc == 6 ? 2 : 4, ev = 4 * wy;
        pl.tiles = ((n_omega + 15) / 16) * ((n_thx + 15) / 16) * ((n_thy + 4 * wy - 1) / (4 * wy));
        pl.t_pad = (int64_t)pl.tiles * SEP_CONS;
        per_thread_p = ev; per_thread_t = (size_t)nc * ev;
        // one CTA per SM: the fewest slices k whose tiles*k CTAs fill whole waves to >= 98.5 %
        if (pl.tiles < 8 * sms) {
            const int64_t kmax = std::max<int64_t>(1, (int64_t)count * std::max(1, pl.cpt / 2));
            int best_k = 1;
            double best = 0.0;
            for (int64_t k = 1; k <= std::min<int64_t>(kmax, 4 * sms); ++k) {
                const int64_t ctas = (int64_t)pl.tiles * k;
                const double eff = (double)ctas / (double)((ctas + sms - 1) / sms * sms);
                if (eff > best + 1e-9) { best = eff; best_k = (int)k; }
                if (eff >= 0.985) break;
            }
            if (best_k > 1) {
                if (count >= best_k) { pl.mode = MODE_PSLICE; pl.p_slices = best_k; }
                else {
                    int ts = std::min((best_k + count - 1) / count, std::max(1, pl.cpt / 2));
                    if (ts > 1) { pl.mode = MODE_TSPLIT; pl.t_slices = ts; pl.p_slices = count; }
                    else if (count > 1) { pl.mode = MODE_PSLICE; pl.p_slices = count; }
                }
            }
        }
    }
    size_t off = 0;
    pl.off_packed = off; off += align_up((size_t)count * pl.cpt * CHUNK_BYTES, 256);
    pl.off_n = off;      off += align_up((size_t)count * sizeof(int64_t), 256);
    pl.off_lam = off;    off += align_up((size_t)count * sizeof(double), 256);
    pl.off_start = off;  off += align_up((size_t)count * sizeof(int64_t), 256);
    pl.off_partial = off;
    if (pl.mode == MODE_PSLICE) off += align_up((size_t)pl.p_slices * per_thread_p * pl.t_pad * 8, 256);
    if (pl.mode == MODE_TSPLIT) off += align_up((size_t)count * pl.t_slices * per_thread_t * pl.t_pad * 8, 256);
    pl.total = off;
    return pl;
}

static bool grid_ok(const rad_grid *g) {
    return g && g->n_omega > 0 && g->n_thx > 0 && g->n_thy > 0 && g->omega && g->thx && g->thy;
}
static bool aligned8(const void *p) { return (reinterpret_cast<uintptr_t>(p) & 7) == 0; }

template <int NC, int DEG>
static cudaError_t launch_main(const MainParams &mp, dim3 grid, cudaStream_t st) {
    static std::once_flag once;
    static cudaError_t attr_err = cudaSuccess;
    std::call_once(once, [] {
        attr_err = cudaFuncSetAttribute(rad_main_kernel<NC, DEG>,
                                        cudaFuncAttributeMaxDynamicSharedMemorySize, SMEM_BYTES);
    });
    if (attr_err != cudaSuccess) return attr_err;
    rad_main_kernel<NC, DEG><<<grid, TPB, SMEM_BYTES, st>>>(mp);
    ++g_launches;
    return cudaGetLastError();
}

template <int NC, int WY>
static cudaError_t launch_sep(const MainParams &mp, dim3 grid, cudaStream_t st) {
    static std::once_flag once;
    static cudaError_t attr_err = cudaSuccess;
    std::call_once(once, [] {
        attr_err = cudaFuncSetAttribute(rad_sep_kernel<NC, WY>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                        SepShape<NC, WY>::SMEM);
    });
    if (attr_err != cudaSuccess) return attr_err;
    rad_sep_kernel<NC, WY><<<grid, SepRegs<NC>::THREADS, SepShape<NC, WY>::SMEM, st>>>(mp);
    ++g_launches;
    return cudaGetLastError();
}

// Everything: pack, main, finalize.  All device pointers; n_host / lam_host are host arrays.
// off_host (optional): first sample of each trajectory inside the arrays (sections of one long trajectory);
// NULL: row p starts at p * stride.
static int run_batch(const rad_traj_batch *b, const int64_t *n_host, const int64_t *off_host, const rad_grid *g,
                     int model, const double *lam_host, int accumulate, double *out,
                     void *workspace, size_t workspace_bytes, cudaStream_t st) {
    if (!b || b->count < 1 || !n_host || !grid_ok(g) || !out) return RAD_EINVAL;
    if (model < RAD_CLASSICAL || model > RAD_SPIN_HALF) return RAD_EINVAL;
    if (model != RAD_CLASSICAL && !lam_host) return RAD_EINVAL;
    const double *arrs[11] = {b->t, b->dz, b->x, b->y, b->vx, b->vy, b->dvz, b->ax, b->ay, b->az, b->gamma};
    for (const double *p : arrs)
        if (!p || !aligned8(p)) return RAD_EINVAL;
    if (!aligned8(out) || !aligned8(g->omega) || !aligned8(g->thx) || !aligned8(g->thy)) return RAD_EINVAL;
    int64_t n_max = 0;
    for (int p = 0; p < b->count; ++p) {
        if (n_host[p] < 2 || n_host[p] > b->stride) return RAD_EINVAL;
        if (off_host && (off_host[p] < 0 || off_host[p] + n_host[p] > b->stride)) return RAD_EINVAL;
        n_max = std::max(n_max, n_host[p]);
        if (model != RAD_CLASSICAL && !(lam_host[p] >= 0.0)) return RAD_EDOMAIN;
    }
    const int nc = model == RAD_SPIN_HALF ? 6 : 4;
    const Plan pl = make_plan(b->count, n_max, g->n_omega, g->n_thx, g->n_thy, nc,
                              choose_kernel(g->n_omega, g->n_thx, g->n_thy, nc));
    if (workspace && (reinterpret_cast<uintptr_t>(workspace) & 255)) return RAD_EINVAL;
    if (workspace && workspace_bytes < pl.total) return RAD_ENOSPACE;
    PoolScratch pool;
    char *ws = static_cast<char *>(workspace);
    if (!ws) {
        // keep freed scratch cached in the device's stream-ordered pool: with the default release
        // threshold (0) every synchronisation hands it back to the driver and the next call pays a
        // fresh allocation (measured: 3x slower steps on cfg 2)
        static std::once_flag pool_once;
        std::call_once(pool_once, [] {
            int dev = 0;
            cudaMemPool_t pool;
            if (cudaGetDevice(&dev) == cudaSuccess && cudaDeviceGetDefaultMemPool(&pool, dev) == cudaSuccess) {
                uint64_t keep = UINT64_MAX;
                cudaMemPoolSetAttribute(pool, cudaMemPoolAttrReleaseThreshold, &keep);
            }
            cudaGetLastError();
        });
        void *pnew = nullptr;
        CK(cudaMallocAsync(&pnew, pl.total, st));
        ws = static_cast<char *>(pnew);
        pool.p = pnew; pool.st = st;
    }
    double *packed = reinterpret_cast<double *>(ws + pl.off_packed);
    int64_t *n_dev = nullptr;
    double *lam_dev = nullptr;
    int64_t *off_dev = nullptr;
    if (off_host) {
        off_dev = reinterpret_cast<int64_t *>(ws + pl.off_start);
        CK(cudaMemcpyAsync(off_dev, off_host, (size_t)b->count * sizeof(int64_t), cudaMemcpyHostToDevice, st));
    }
    if (b->count > 1) {
        n_dev = reinterpret_cast<int64_t *>(ws + pl.off_n);
        CK(cudaMemcpyAsync(n_dev, n_host, (size_t)b->count * sizeof(int64_t), cudaMemcpyHostToDevice, st));
        if (model != RAD_CLASSICAL) {
            lam_dev = reinterpret_cast<double *>(ws + pl.off_lam);
            CK(cudaMemcpyAsync(lam_dev, lam_host, (size_t)b->count * sizeof(double), cudaMemcpyHostToDevice, st));
        }
    }
    prof_mark(0, st);
    {   // a0/a1: pack
        dim3 grid((unsigned)(((int64_t)pl.cpt * CH + 255) / 256), (unsigned)b->count);
        rad_pack_kernel<<<grid, 256, 0, st>>>(*b, n_dev, n_host[0], off_dev, pl.cpt, packed);
        ++g_launches;
        CK(cudaGetLastError());
    }
    prof_mark(1, st);
    MainParams mp{};
    mp.packed = packed; mp.n_dev = n_dev; mp.lam_dev = lam_dev;
    mp.n_single = n_host[0];
    mp.lam_single = model == RAD_CLASSICAL ? 0.0 : lam_host[0];
    mp.count = b->count; mp.cpt = pl.cpt;
    mp.omega = g->omega; mp.thx = g->thx; mp.thy = g->thy;
    mp.n_omega = g->n_omega; mp.n_thx = g->n_thx; mp.n_thy = g->n_thy;
    mp.model = model; mp.mode = pl.mode; mp.p_slices = pl.p_slices; mp.t_slices = pl.t_slices;
    mp.accumulate = accumulate ? 1 : 0;
    mp.out = out; mp.partial = reinterpret_cast<double *>(ws + pl.off_partial);
    mp.t_pad = pl.t_pad;
    const int slices = pl.mode == MODE_TSPLIT ? b->count * pl.t_slices : pl.p_slices;
    dim3 grid((unsigned)pl.tiles, (unsigned)slices);
    cudaError_t e;
    if (pl.kernel == 1) e = nc == 6 ? launch_sep<6, 2>(mp, grid, st) : launch_sep<4, 4>(mp, grid, st);
    else e = nc == 6 ? launch_main<6, RAD_DEG>(mp, grid, st) : launch_main<4, RAD_DEG>(mp, grid, st);
    if (e != cudaSuccess) return cuda_fail(e, pl.kernel == 1 ? "rad_sep_kernel" : "rad_main_kernel");
    prof_mark(2, st);
    if (pl.mode != MODE_DIRECT) {
        if (pl.kernel == 1) {
            if (nc == 6) rad_sep_finalize_kernel<6, 2><<<dim3(pl.tiles, 8), SEP_CONS, 0, st>>>(mp);
            else rad_sep_finalize_kernel<4, 4><<<dim3(pl.tiles, 16), SEP_CONS, 0, st>>>(mp);
        } else {
            if (nc == 6) rad_finalize_kernel<6><<<dim3(pl.tiles, W), TPB, 0, st>>>(mp);
            else rad_finalize_kernel<4><<<dim3(pl.tiles, W), TPB, 0, st>>>(mp);
        }
        ++g_launches;
        CK(cudaGetLastError());
        prof_mark(3, st);
    }
    return RAD_OK;
}

static int run_single(const rad_traj *t, const rad_grid *g, int model, double lam, double *out,
                      void *ws, size_t ws_bytes, cudaStream_t st) {
    if (!t) return RAD_EINVAL;
    rad_traj_batch b{1, t->n, nullptr, t->t, t->dz, t->x, t->y, t->vx, t->vy, t->dvz,
                     t->ax, t->ay, t->az, t->gamma};
    const int64_t n = t->n;
    return run_batch(&b, &n, nullptr, g, model, &lam, 0, out, ws, ws_bytes, st);
}

}  // namespace rad

// =============================================================================== C ABI
using namespace rad;

extern "C" {

int rad_classical(const rad_traj *traj, const rad_grid *grid, double *out,
                  void *workspace, size_t workspace_bytes, void *cuda_stream) {
    return run_single(traj, grid, RAD_CLASSICAL, 0.0, out, workspace, workspace_bytes,
                      static_cast<cudaStream_t>(cuda_stream));
}

int rad_semiclassical(const rad_traj *traj, const rad_grid *grid, int spin, double hbarc_over_E,
                      double *out, void *workspace, size_t workspace_bytes, void *cuda_stream) {
    if (spin != 0 && spin != 1) return RAD_EINVAL;
    if (!(hbarc_over_E >= 0.0)) return RAD_EDOMAIN;
    return run_single(traj, grid, spin == 0 ? RAD_SPIN0 : RAD_SPIN_HALF, hbarc_over_E, out,
                      workspace, workspace_bytes, static_cast<cudaStream_t>(cuda_stream));
}

int rad_ensemble_sum(const rad_traj_batch *batch, const rad_grid *grid, rad_model model,
                     const double *hbarc_over_E, int accumulate, double *out,
                     void *workspace, size_t workspace_bytes, void *cuda_stream) {
    if (!batch) return RAD_EINVAL;
    return run_batch(batch, batch->n, nullptr, grid, (int)model, hbarc_over_E, accumulate, out,
                     workspace, workspace_bytes, static_cast<cudaStream_t>(cuda_stream));
}

int rad_sections_sum(const rad_traj *traj, int32_t n_sections, const int64_t *start, const rad_grid *grid,
                     rad_model model, const double *hbarc_over_E, int accumulate, double *out,
                     void *workspace, size_t workspace_bytes, void *cuda_stream) {
    if (!traj || !start || n_sections < 1) return RAD_EINVAL;
    std::vector<int64_t> n(n_sections), off(n_sections);
    for (int s = 0; s < n_sections; ++s) {            // section s = samples start[s] .. start[s+1], both included
        if (start[s] < 0 || start[s + 1] <= start[s] || start[s + 1] > traj->n - 1) return RAD_EINVAL;
        off[s] = start[s];
        n[s] = start[s + 1] - start[s] + 1;
    }
    rad_traj_batch b{n_sections, traj->n, n.data(), traj->t, traj->dz, traj->x, traj->y, traj->vx, traj->vy,
                     traj->dvz, traj->ax, traj->ay, traj->az, traj->gamma};
    return run_batch(&b, n.data(), off.data(), grid, (int)model, hbarc_over_E, accumulate, out,
                     workspace, workspace_bytes, static_cast<cudaStream_t>(cuda_stream));
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

// omegas per slab of rad_angular_spectrum: the slab cube stays below ~256 MB, whole 16-omega tiles
static int spectrum_slab(int n_omega, int n_thx, int n_thy) {
    const int64_t per_omega = (int64_t)n_thx * n_thy * 8;
    int64_t k = std::max<int64_t>(16, ((int64_t)256 << 20) / per_omega / 16 * 16);
    return (int)std::min<int64_t>(k, n_omega);
}

size_t rad_angular_spectrum_workspace_bytes(int32_t count, int64_t n_max, int32_t n_omega, int32_t n_thx,
                                            int32_t n_thy) {
    if (count < 1 || n_max < 2 || n_omega < 1 || n_thx < 1 || n_thy < 1) return 0;
    const int k = spectrum_slab(n_omega, n_thx, n_thy);
    const size_t inner = rad_workspace_bytes(count, n_max, k, n_thx, n_thy);
    return align_up(inner, 256) + align_up((size_t)k * n_thx * n_thy * 8, 256);
}

int rad_angular_spectrum(const rad_traj_batch *batch, const rad_grid *grid, rad_model model,
                         const double *hbarc_over_E, double d_solid_angle, double theta_cut, double *spectrum,
                         void *workspace, size_t workspace_bytes, void *cuda_stream) {
    if (!batch || !grid_ok(grid) || !spectrum || !workspace) return RAD_EINVAL;
    if (reinterpret_cast<uintptr_t>(workspace) & 255) return RAD_EINVAL;
    int64_t n_max = 0;
    if (!batch->n || batch->count < 1) return RAD_EINVAL;
    for (int p = 0; p < batch->count; ++p) n_max = std::max(n_max, batch->n[p]);
    if (n_max < 2) return RAD_EINVAL;
    const int k = spectrum_slab(grid->n_omega, grid->n_thx, grid->n_thy);
    const size_t inner = align_up(rad_workspace_bytes(batch->count, n_max, k, grid->n_thx, grid->n_thy), 256);
    const size_t cube_bytes = align_up((size_t)k * grid->n_thx * grid->n_thy * 8, 256);
    if (workspace_bytes < inner + cube_bytes) return RAD_ENOSPACE;
    double *cube = reinterpret_cast<double *>(static_cast<char *>(workspace) + inner);
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    for (int w0 = 0; w0 < grid->n_omega; w0 += k) {    // one slab of omegas at a time: cube of the slab, then its sum
        const int kw = std::min(k, grid->n_omega - w0);
        rad_grid slab{kw, grid->n_thx, grid->n_thy, grid->omega + w0, grid->thx, grid->thy};
        int rc = run_batch(batch, batch->n, nullptr, &slab, (int)model, hbarc_over_E, 0, cube, workspace, inner, st);
        if (rc != RAD_OK) return rc;
        rc = rad_angular_sum(cube, &slab, d_solid_angle, theta_cut, spectrum + w0, cuda_stream);
        if (rc != RAD_OK) return rc;
    }
    return RAD_OK;
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
    const unsigned blocks = (unsigned)((count + 127) / 128);
    if (well == RAD_WELL_HARMONIC_MS)
        rad_traj_ms_kernel<<<blocks, 128, 0, st>>>(kappa, gamma, dt, sigma, seed, count, n, stride, x0, y0, vx0, vy0, o);
    else if (well == RAD_WELL_COSINE)
        rad_traj_kernel<0><<<blocks, 128, 0, st>>>(kappa, length, gamma, dt, count, n, stride, x0, y0, vx0, vy0, o);
    else
        rad_traj_kernel<1><<<blocks, 128, 0, st>>>(kappa, length, gamma, dt, count, n, stride, x0, y0, vx0, vy0, o);
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
    for (int kernel = 0; kernel < 2; ++kernel)
        for (int nc = 4; nc <= 6; nc += 2)
            need = std::max(need, make_plan(count, n_max, n_omega, n_thx, n_thy, nc, kernel).total);
    return need;
}

// ---- host-buffer variants: H2D once, compute, D2H once
int rad_ensemble_sum_host(const rad_traj_batch *b, const rad_grid *g, rad_model model,
                          const double *hbarc_over_E, int accumulate, double *out, void *cuda_stream) {
    if (!b || b->count < 1 || !b->n || !grid_ok(g) || !out) return RAD_EINVAL;
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    const size_t row = (size_t)b->stride, tot = row * b->count;
    const size_t M = (size_t)g->n_omega * g->n_thx * g->n_thy;
    const size_t ng = (size_t)g->n_omega + g->n_thx + g->n_thy;
    const double *src[11] = {b->t, b->dz, b->x, b->y, b->vx, b->vy, b->dvz, b->ax, b->ay, b->az, b->gamma};
    for (const double *p : src)
        if (!p) return RAD_EINVAL;
    double *dev = nullptr;
    CK(cudaMallocAsync(reinterpret_cast<void **>(&dev), (11 * tot + ng + M) * sizeof(double), st));
    PoolScratch pool;
    pool.p = dev; pool.st = st;
    const double *d[11];
    for (int i = 0; i < 11; ++i) {
        d[i] = dev + i * tot;
        CK(cudaMemcpyAsync(dev + i * tot, src[i], tot * sizeof(double), cudaMemcpyHostToDevice, st));
    }
    double *gw = dev + 11 * tot, *gx = gw + g->n_omega, *gy = gx + g->n_thx, *dout = gy + g->n_thy;
    CK(cudaMemcpyAsync(gw, g->omega, g->n_omega * sizeof(double), cudaMemcpyHostToDevice, st));
    CK(cudaMemcpyAsync(gx, g->thx, g->n_thx * sizeof(double), cudaMemcpyHostToDevice, st));
    CK(cudaMemcpyAsync(gy, g->thy, g->n_thy * sizeof(double), cudaMemcpyHostToDevice, st));
    if (accumulate) CK(cudaMemcpyAsync(dout, out, M * sizeof(double), cudaMemcpyHostToDevice, st));
    rad_traj_batch db{b->count, b->stride, b->n, d[0], d[1], d[2], d[3], d[4], d[5], d[6], d[7], d[8], d[9], d[10]};
    rad_grid dg{g->n_omega, g->n_thx, g->n_thy, gw, gx, gy};
    int rc = run_batch(&db, b->n, nullptr, &dg, (int)model, hbarc_over_E, accumulate, dout, nullptr, 0, st);
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
                  double *out, void *cuda_stream) {
    if (!t) return RAD_EINVAL;
    if (model != RAD_CLASSICAL && !(hbarc_over_E >= 0.0)) return RAD_EDOMAIN;
    const int64_t n = t->n;
    rad_traj_batch b{1, t->n, &n, t->t, t->dz, t->x, t->y, t->vx, t->vy, t->dvz, t->ax, t->ay, t->az, t->gamma};
    return rad_ensemble_sum_host(&b, g, model, &hbarc_over_E, 0, out, cuda_stream);
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

int rad_plan_kernel(int32_t n_omega, int32_t n_thx, int32_t n_thy, rad_model model) {
    if (n_omega < 1 || n_thx < 1 || n_thy < 1 || model < RAD_CLASSICAL || model > RAD_SPIN_HALF) return RAD_EINVAL;
    return choose_kernel(n_omega, n_thx, n_thy, model == RAD_SPIN_HALF ? 6 : 4) + 1;
}

double rad_formation_length(double gamma, double omega, double hbarc_over_E) {
    const double u = omega * hbarc_over_E;            // hbar omega / E
    if (!(gamma >= 1.0) || !(omega > 0.0) || !(u >= 0.0) || !(u < 1.0)) return -1.0;
    return 2.0 * gamma * gamma * (1.0 - u) / omega;   // l_f = 2 gamma^2 (E - w) / (E w)
}

int rad_plan_describe(int32_t count, int64_t n_max, int32_t n_omega, int32_t n_thx, int32_t n_thy, rad_model model,
                      int32_t *plan) {
    if (!plan || count < 1 || n_max < 2 || n_omega < 1 || n_thx < 1 || n_thy < 1) return RAD_EINVAL;
    if (model < RAD_CLASSICAL || model > RAD_SPIN_HALF) return RAD_EINVAL;
    const int nc = model == RAD_SPIN_HALF ? 6 : 4;
    const Plan pl = make_plan(count, n_max, n_omega, n_thx, n_thy, nc, choose_kernel(n_omega, n_thx, n_thy, nc));
    plan[0] = pl.kernel + 1;
    plan[1] = pl.mode;
    plan[2] = pl.tiles;
    plan[3] = pl.mode == MODE_TSPLIT ? count * pl.t_slices : pl.p_slices;      // gridDim.y
    plan[4] = pl.t_slices;
    plan[5] = pl.cpt;
    return RAD_OK;
}

int rad_set_kernel(int choice) {
    if (choice < 0 || choice > 2) return RAD_EINVAL;
    g_kernel_choice.store(choice);
    return RAD_OK;
}

int rad_profile_enable(int on) {
    g_prof.store(on ? 1 : 0);
    return RAD_OK;
}

int rad_profile_last(float *ms) {
    if (!ms) return RAD_EINVAL;
    std::lock_guard<std::mutex> lk(g_ev_mu);
    if (!g_ev_ready) return RAD_EINVAL;
    CK(cudaEventSynchronize(g_ev[g_ev_have_finalize ? 3 : 2]));
    CK(cudaEventElapsedTime(&ms[0], g_ev[0], g_ev[1]));
    CK(cudaEventElapsedTime(&ms[1], g_ev[1], g_ev[2]));
    ms[2] = 0.f;
    if (g_ev_have_finalize) CK(cudaEventElapsedTime(&ms[2], g_ev[2], g_ev[3]));
    return RAD_OK;
}

const char *rad_strerror(int code) {
    switch (code) {
        case RAD_OK: return "ok";
        case RAD_EINVAL: return "invalid argument";
        case RAD_EDOMAIN: return "parameter outside the method's domain";
        case RAD_ECUDA: return g_err;
        case RAD_ENOSPACE: return "workspace too small (see rad_workspace_bytes)";
        default: return "unknown status";
    }
}

}  // extern "C"
