// rad_fused.cuh -- single-launch kernel for one short trajectory on a grid too small to fill the GPU
// (north_star item 4; the paper's saturation knee).
//
// BASELINE config 1 (4096 grid points x 4000 samples) is 1.6e7 evals: 22 us of FP64 work for the whole GPU.
// Three dependent launches (pack, main, ordered reduction) cost more than that.  Here ONE cooperative launch
// does rows a0-a6:
//   a0/a1  every CTA packs its own samples on the fly from the caller's SoA arrays into shared memory (one sample
//          per thread and round; same record layout and the same double-double chunk base as rad_pack_kernel, so
//          the arithmetic downstream is the direct kernel's, bit for bit per sample)
//   a2-a4  the direct kernel's per-sample body (accumulate_sample): one angle x 8 omegas per thread
//   a6     the time axis is cut into as many slices as CTAs fit on the GPU at once (4 per SM); each CTA stores its
//          partial complex amplitudes, the grid synchronises (cooperative groups), and ALL threads then add the
//          slices in ascending time order and apply the epilogue (a5) -- a fixed order, no floating-point
//          atomics, nothing left in the workspace between calls.
// The split is across CTAs rather than across the lanes of a warp (row a6 names a warp shuffle): lanes keep
// distinct angles so that the trajectory reads stay shared-memory broadcasts; the grid-wide pass plays the role
// of the shuffle tree and runs on all 148 SMs.
#pragma once

#include <cooperative_groups.h>

namespace rad {

struct FusedParams {
    rad_traj tr;              // caller's SoA arrays (device)
    double lam;               // hbar c / E
    const double *omega, *thx, *thy;
    int n_omega, n_thx, n_thy;
    int model, accumulate;
    int tiles, slices;        // gridDim.x, gridDim.y
    double *partial;          // [slices][NC * W][tiles * FUSED_TPB]
    double *out;
};

constexpr int FUSED_CHUNK_DBL = HDR + FUSED_SUB * REC;
constexpr int FUSED_SMEM = FUSED_CHUNK_DBL * 8 + W * FUSED_TPB * 16;

template <int NC, int DEG>
__global__ void __launch_bounds__(FUSED_TPB, 4)
rad_fused_kernel(const FusedParams P) {
    static_assert(FUSED_SUB == FUSED_TPB, "one sample per thread and packing round");
    extern __shared__ __align__(128) unsigned char smem_raw[];
    double *ck = reinterpret_cast<double *>(smem_raw);                              // header + FUSED_SUB records
    double2 *wt_sm = reinterpret_cast<double2 *>(smem_raw + FUSED_CHUNK_DBL * 8);   // [W][FUSED_TPB]
    const int tid = threadIdx.x;
    const rad_traj &b = P.tr;
    const int64_t n = b.n;

    // ---- this thread's grid coordinates (as in rad_main_kernel: flattened (omega group, angle), angle fastest)
    const int A = P.n_thx * P.n_thy;
    const int n_wg = (P.n_omega + W - 1) / W;
    const int64_t T = (int64_t)n_wg * A;
    const int64_t t_pad = (int64_t)P.tiles * FUSED_TPB;
    const int64_t gid = (int64_t)blockIdx.x * FUSED_TPB + tid;
    const int64_t gc = min(gid, T - 1);
    const int wg = (int)(gc / A), a = (int)(gc % A);
    const double nx = P.thx[a % P.n_thx], ny = P.thy[a / P.n_thx];
    const dd h = half_theta2_dd(nx, ny);
    double wh[W];
#pragma unroll
    for (int j = 0; j < W; ++j) {
        const dd wt = omega_star_turns(P.omega[min(wg * W + j, P.n_omega - 1)], P.lam);
        wt_sm[j * FUSED_TPB + tid] = make_double2(wt.hi, wt.lo);
        wh[j] = wt.hi;
    }
    double acc[W][NC];
#pragma unroll
    for (int j = 0; j < W; ++j)
#pragma unroll
        for (int c = 0; c < NC; ++c) acc[j][c] = 0.0;

    // ---- this CTA's time slice, in rounds of FUSED_SUB samples
    const int slice = blockIdx.y;
    const int64_t k_begin = (int64_t)slice * n / P.slices, k_end = (int64_t)(slice + 1) * n / P.slices;
    for (int64_t c0 = k_begin; c0 < k_end; c0 += FUSED_SUB) {
        const int nvalid = (int)min((int64_t)FUSED_SUB, k_end - c0);
        const int64_t kb = c0 + min(FUSED_SUB / 2, nvalid - 1);            // base sample of the round
        {   // a0/a1: pack (the arithmetic of rad_pack_kernel)
            double ab;
            const dd P0b = phase_offset_dd(b.gamma[kb], b.t[kb], b.dz[kb], ab);
            if (tid == 0) {
                ck[0] = P0b.hi; ck[1] = P0b.lo;
                ck[2] = b.t[kb]; ck[3] = b.x[kb]; ck[4] = b.y[kb];
                ck[5] = b.gamma[0]; ck[6] = 0.0; ck[7] = 0.0;
            }
            double *rec = ck + HDR + tid * REC;
            const int64_t k = c0 + tid;
            if (tid >= nvalid) {                                           // zero-weight padding, q = 1
                rec[0] = 1.0;
#pragma unroll
                for (int j = 1; j < REC; ++j) rec[j] = 0.0;
            } else {
                const double tk = b.t[k];
                const double w = 0.5 * (b.t[min(k + 1, n - 1)] - b.t[max(k - 1, (int64_t)0)]);
                double ak;
                const dd P0k = phase_offset_dd(b.gamma[k], tk, b.dz[k], ak);
                const dd dP = dd_add(P0k, dd_neg(P0b));
                rec[0] = ak - b.dvz[k];
                rec[1] = b.vx[k];
                rec[2] = b.vy[k];
                rec[3] = w * b.ax[k];
                rec[4] = w * b.ay[k];
                rec[5] = w * b.az[k];
                rec[6] = dP.hi + dP.lo;
                rec[7] = tk - b.t[kb];
                rec[8] = b.x[k] - b.x[kb];
                rec[9] = b.y[k] - b.y[kb];
            }
        }
        __syncthreads();
        double p0[W];
        chunk_base_phase(ck, h, nx, ny, wt_sm + tid, FUSED_TPB, p0);
        const double *rec = ck + HDR;
#pragma unroll 1
        for (int k = 0; k < FUSED_SUB; ++k, rec += REC) accumulate_sample<NC, DEG>(rec, nx, ny, h.hi, wh, p0, acc);
        __syncthreads();                                                   // the round's records may be overwritten
    }

    // ---- a6: partial amplitudes -> grid-wide ordered reduction -> epilogue
    {
        double *dst = P.partial + (int64_t)slice * NC * W * t_pad + gid;
#pragma unroll
        for (int c = 0; c < NC; ++c)
#pragma unroll
            for (int j = 0; j < W; ++j) dst[(int64_t)(c * W + j) * t_pad] = acc[j][c];
    }
    cooperative_groups::this_grid().sync();
    const int64_t n_threads = (int64_t)gridDim.x * gridDim.y * FUSED_TPB;
    const int64_t me = ((int64_t)blockIdx.y * gridDim.x + blockIdx.x) * FUSED_TPB + tid;
    const double gamma0 = b.gamma[0];
    for (int64_t o = me; o < t_pad * W; o += n_threads) {                  // one (thread slot, omega of its tile) each
        const int64_t g = o % t_pad;
        const int j = (int)(o / t_pad);
        if (g >= T) continue;
        const int wg2 = (int)(g / A), a2 = (int)(g % A);
        const int iw = wg2 * W + j;
        if (iw >= P.n_omega) continue;
        double s[NC];
#pragma unroll
        for (int c = 0; c < NC; ++c) s[c] = 0.0;
        for (int sl = 0; sl < P.slices; ++sl) {                            // time slices ascending
            const double *src = P.partial + (int64_t)sl * NC * W * t_pad + g;
#pragma unroll
            for (int c = 0; c < NC; ++c) s[c] += src[(int64_t)(c * W + j) * t_pad];
        }
        const double v = spectrum_value<NC>(s, P.thx[a2 % P.n_thx], P.thy[a2 / P.n_thx], P.model,
                                            P.omega[iw] * P.lam, gamma0);
        double *dstp = P.out + (int64_t)iw * A + a2;
        *dstp = P.accumulate ? *dstp + v : v;
    }
}

}  // namespace rad
