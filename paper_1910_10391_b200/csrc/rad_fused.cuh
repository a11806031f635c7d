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
//          partial complex amplitudes, the grid synchronises (cooperative groups), and all warps then add the
//          slices in ascending time order -- one accumulator per lane, gathered by warp shuffle for the epilogue
//          (a5): a fixed order, no floating-point atomics, nothing left in the workspace between calls.
// The time axis is split across CTAs rather than across the lanes of a warp (row a6): lanes keep distinct angles so
// that the trajectory reads stay shared-memory broadcasts; the grid-wide pass runs on all 148 SMs.
// Measured on B200 (config 1, 8 tiles x 74 slices = 592 CTAs; phases switched off one at a time): launch +
// per-CTA prologue 14 -> 10 us (omega*/2pi once per CTA instead of once per thread, the base sample's P0 from its
// owner), sample loop 27 us (21.7 us would be 100 % of the FP64 pipe), grid sync 1.5 us, reduction + epilogue
// 16.5 -> 8 us (loads batched eight slices at a time and spread over the accumulators): 46 us by CUDA events.
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
    // GEN instantiation: the angles are the L-shaped rest of a two-part plan (the separable kernel took
    // [0, l_x0) x [0, l_y0) of the n_thx x n_thy plane) and the cube has its own strides
    int l_x0, l_y0, out_nx;
    int64_t out_plane;
};

// (i_x, i_y) of the a-th angle of a fused launch
template <bool GEN>
__device__ __forceinline__ void fused_angle_of(const FusedParams &P, int a, int &ix, int &iy) {
    if (!GEN) { ix = a % P.n_thx; iy = a / P.n_thx; return; }
    const int rx = P.n_thx - P.l_x0, n1 = rx * P.n_thy;
    if (a < n1) { ix = P.l_x0 + a % rx; iy = a / rx; }
    else { const int j = a - n1; ix = j % P.l_x0; iy = P.l_y0 + j / P.l_x0; }
}

constexpr int FUSED_CHUNK_DBL = HDR + FUSED_SUB * REC;
constexpr int FUSED_SMEM = FUSED_CHUNK_DBL * 8 + W * FUSED_TPB * 16;      // records + up to 64 omega groups' omega*/2pi

template <int NC, int DEG, bool GEN>
__global__ void __launch_bounds__(FUSED_TPB, 4)
rad_fused_kernel(const FusedParams P) {
    static_assert(FUSED_SUB == FUSED_TPB, "one sample per thread and packing round");
    extern __shared__ __align__(128) unsigned char smem_raw[];
    double *ck = reinterpret_cast<double *>(smem_raw);                              // header + FUSED_SUB records
    double2 *wt_sm = reinterpret_cast<double2 *>(smem_raw + FUSED_CHUNK_DBL * 8);   // [omega groups of the CTA][W]
    const int tid = threadIdx.x;
    const rad_traj &b = P.tr;
    const int64_t n = b.n;

    // ---- this thread's grid coordinates (as in rad_main_kernel: flattened (omega group, angle), angle fastest)
    const int A = GEN ? angle_count(P.n_thx, P.n_thy, P.l_x0, P.l_y0) : P.n_thx * P.n_thy;
    const int n_wg = (P.n_omega + W - 1) / W;
    const int64_t T = (int64_t)n_wg * A;
    const int64_t t_pad = (int64_t)P.tiles * FUSED_TPB;
    const int64_t gid = (int64_t)blockIdx.x * FUSED_TPB + tid;
    const int64_t gc = min(gid, T - 1);
    const int wg = (int)(gc / A), a = (int)(gc % A);
    int ix0, iy0;
    fused_angle_of<GEN>(P, a, ix0, iy0);
    const double nx = P.thx[ix0], ny = P.thy[iy0];
    const dd h = half_theta2_dd(nx, ny);
    // omega* / 2 pi (double-double: two FP64 divisions each) once per omega the CTA touches, not once per thread:
    // the prologue is paid by every time slice, i.e. dozens of times per tile
    const int wg_lo = (int)(min((int64_t)blockIdx.x * FUSED_TPB, T - 1) / A);
    const int wg_hi = (int)(min((int64_t)blockIdx.x * FUSED_TPB + FUSED_TPB - 1, T - 1) / A);
    for (int i = tid; i < (wg_hi - wg_lo + 1) * W; i += FUSED_TPB) {
        // (classical: omega* = omega, no divisions -- half a microsecond of a 47 us kernel.  Only here: the same
        // branch inside omega_star_turns costs the separable kernel's producers 2-14 %)
        const double om = P.omega[min(wg_lo * W + i, P.n_omega - 1)];
        const dd wt = P.lam == 0.0 ? dd_mul_d(dd{INV_2PI_HI, INV_2PI_LO}, om) : omega_star_turns(om, P.lam);
        wt_sm[i] = make_double2(wt.hi, wt.lo);
    }
    __syncthreads();
    const double2 *wt_mine = wt_sm + (wg - wg_lo) * W;
    double wh[W];
#pragma unroll
    for (int j = 0; j < W; ++j) wh[j] = wt_mine[j].x;
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
        {   // a0/a1: pack (the arithmetic of rad_pack_kernel; the base sample's P0 comes from the thread that owns it)
            double *rec = ck + HDR + tid * REC;
            const int64_t k = c0 + tid;
            dd P0k = {0.0, 0.0};
            double ak = 0.0;
            if (tid < nvalid) {
                P0k = phase_offset_dd(b.gamma[k], b.t[k], b.dz[k], ak);
                if (k == kb) {
                    ck[0] = P0k.hi; ck[1] = P0k.lo;
                    ck[2] = b.t[kb]; ck[3] = b.x[kb]; ck[4] = b.y[kb];
                    ck[5] = b.gamma[0]; ck[6] = 0.0; ck[7] = 0.0;
                }
            }
            __syncthreads();
            if (tid < nvalid) {                                            // (records beyond nvalid are never read)
                const dd P0b = {ck[0], ck[1]};
                const double tk = b.t[k];
                const double w = 0.5 * (b.t[min(k + 1, n - 1)] - b.t[max(k - 1, (int64_t)0)]);
                const dd dP = dd_add(P0k, dd_neg(P0b));
                rec[0] = ak - b.dvz[k];
                rec[1] = b.vx[k];
                rec[2] = b.vy[k];
                rec[3] = w * b.ax[k];
                rec[4] = w * b.ay[k];
                rec[5] = w * b.az[k];
                rec[6] = dP.hi + dP.lo;
                rec[7] = tk - ck[2];
                rec[8] = b.x[k] - ck[3];
                rec[9] = b.y[k] - ck[4];
            }
        }
        __syncthreads();
        double p0[W];
        chunk_base_phase(ck, h, nx, ny, wt_mine, 1, p0);
        const double *rec = ck + HDR;
#ifndef FUSED_SKIP_MAIN
#pragma unroll 1
        for (int k = 0; k < nvalid; ++k, rec += REC) accumulate_sample<NC, DEG>(rec, nx, ny, h.hi, wh, p0, acc);
#endif
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
#ifdef FUSED_SKIP_SYNC
    return;
#endif
    cooperative_groups::this_grid().sync();
#ifdef FUSED_SKIP_REDUCE
    return;
#endif
    // One work item per (thread slot g, omega j of its tile, accumulator c), c fastest: NC adjacent lanes of a warp
    // each add ONE accumulator's slices in ascending time order (loads issued eight slices at a time: the sum
    // is latency-bound, not bandwidth-bound), then hand their sums to the lane with c = 0 by warp shuffle, which
    // applies the epilogue.  Lane groups never straddle a warp: 32 is a multiple of neither 4 nor 6 in general, so
    // items are laid out per warp as (32 / NC) whole outputs.
    constexpr int OPW = 32 / NC;                                           // outputs per warp
    const int lane = tid & 31;
    const int64_t n_warps = (int64_t)gridDim.x * gridDim.y * (FUSED_TPB / 32);
    const int64_t warp = ((int64_t)blockIdx.y * gridDim.x + blockIdx.x) * (FUSED_TPB / 32) + (tid >> 5);
    const double gamma0 = b.gamma[0];
    const int64_t n_out = t_pad * W;
    for (int64_t o0 = warp * OPW; o0 < n_out; o0 += n_warps * OPW) {
        const int64_t o = o0 + lane / NC;
        const int c = lane % NC;
        const bool live = lane < OPW * NC && o < n_out;
        const int64_t g = live ? o % t_pad : 0;
        const int j = live ? (int)(o / t_pad) : 0;
        double sum = 0.0;
        if (live) {
            const double *src = P.partial + (int64_t)(c * W + j) * t_pad + g;
            const int64_t stride = (int64_t)NC * W * t_pad;
            int sl = 0;
            for (; sl + 8 <= P.slices; sl += 8) {                          // time slices ascending
                double v[8];
#pragma unroll
                for (int q = 0; q < 8; ++q) v[q] = src[(sl + q) * stride];
#pragma unroll
                for (int q = 0; q < 8; ++q) sum += v[q];
            }
            for (; sl < P.slices; ++sl) sum += src[sl * stride];
        }
        double s[NC];
#pragma unroll
        for (int q = 0; q < NC; ++q) s[q] = __shfl_sync(0xffffffffu, sum, (lane / NC) * NC + q);
        const int wg2 = (int)(g / A), a2 = (int)(g % A);
        const int iw = wg2 * W + j;
        if (live && c == 0 && g < T && iw < P.n_omega) {
            int ix, iy;
            fused_angle_of<GEN>(P, a2, ix, iy);
            const double v = spectrum_value<NC>(s, P.thx[ix], P.thy[iy], P.model, P.omega[iw] * P.lam, gamma0);
            double *dstp = GEN ? P.out + iw * P.out_plane + (int64_t)iy * P.out_nx + ix : P.out + (int64_t)iw * A + a2;
            *dstp = P.accumulate ? *dstp + v : v;
        }
    }
}

}  // namespace rad
