// rad_plan.h -- host-side launch planning of the radiation-integral library (included by rad.cu only).
//
// A call is evaluated by one or two PARTS (a sub-grid and the kernel that takes it), each with its own
// split of the (trajectory, time) axis over CTAs:
//   * one part, direct kernel            grids that fill the separable kernel's tiles badly
//   * one part, separable kernel         grids that fill them well (BASELINE configs 2-5)
//   * two parts                          separable kernel on the largest block of whole angle tiles, direct
//                                        kernel on the L-shaped rest of the angle plane (PAPER.md:149's typical
//                                        50 x 50 angles = 48 x 48 + 196)
//   * fused single-launch kernel         one short trajectory on a grid too small to fill the GPU (config 1)
// Everything here is a pure function of the shapes, the kernel option and the SM count.
#pragma once

#include <algorithm>
#include <cstddef>
#include <cstdint>

namespace rad {

enum Mode : int { MODE_DIRECT = 0, MODE_PSLICE = 1, MODE_TSPLIT = 2 };
enum KernelId : int { K_DIRECT = 0, K_SEP = 1, K_FUSED = 2 };

constexpr int PLAN_TPB = 128;     // threads per CTA of the direct kernel (= TPB in rad.cu)
constexpr int PLAN_W = 8;         // omegas per thread of the direct kernel (= W)
constexpr int PLAN_CH = 128;      // samples per packed chunk (= CH)
constexpr int PLAN_SEP_CONS = 256;
constexpr int FUSED_TPB = 64;     // threads per CTA of the fused kernel
constexpr int FUSED_SUB = 64;     // samples it packs per round (one per thread)

static inline size_t align_up(size_t v, size_t a) { return (v + a - 1) / a * a; }

struct Plan {                 // the (trajectory, time) split of one part
    int tiles, p_slices, t_slices, mode;
    int64_t t_pad;            // tiles * threads that own points
    size_t partial_bytes;     // scratch for partial amplitudes / spectra (0 in MODE_DIRECT)
    int slices() const { return mode == MODE_TSPLIT ? p_slices * t_slices : p_slices; }     // gridDim.y
};

struct Part {
    int kernel;               // K_DIRECT or K_SEP
    int n_thx, n_thy;         // angle extents of this part's view (separable: the interior; direct: the whole plane)
    int l_x0, l_y0;           // direct kernel on the rest outside [0, l_x0) x [0, l_y0); -1: the whole plane
    int angles;               // angles the part evaluates
    Plan plan;
    size_t off_partial;
    int cl;                   // separable kernel: 2 = launched as cluster pairs of CTAs on neighbouring y tiles that
                              // share the T table through distributed shared memory (needs an even y tile count);
                              // 3 = pairs on neighbouring omega tiles that share the F table (4 accumulators per
                              // point, even omega tile count, cube output); 1 = single CTAs
    int f_tiles, f_slices;    // > 0: this (direct) part runs through the fused single-launch kernel instead of
                              // main + ordered reduction: the L-shaped rest of a two-part plan of one short trajectory
};

struct CallPlan {
    int nparts;
    Part part[2];
    bool fused;               // the fused single-launch kernel takes the whole call (part[0] describes its grid)
    int fused_tiles, fused_slices;
    int cpt;                  // chunks per trajectory in the packed buffer
    size_t off_packed, off_n, off_lam, off_start, off_ang, total;
    int launches() const {
        if (fused) return 1;
        int l = 1;            // pack
        for (int i = 0; i < nparts; ++i) l += part[i].f_tiles > 0 ? 1 : 1 + (part[i].plan.mode != MODE_DIRECT);
        return l;
    }
};

// fewest slices k (at most kmax) for which tiles * k CTAs fill whole waves of `slots` resident CTAs to >= 98.5 %
static inline int best_slices(int tiles, int slots, int64_t kmax, int cap, bool want_two_waves) {
    int best_k = 1;
    double best = 0.0;
    for (int64_t k = 1; k <= std::min<int64_t>(kmax, cap); ++k) {
        const int64_t ctas = (int64_t)tiles * k;
        double eff = (double)ctas / (double)((ctas + slots - 1) / slots * slots);
        if (want_two_waves && ctas < 2 * slots && k < kmax) eff *= 0.5;      // too few CTAs to balance: keep looking
        if (eff > best + 1e-9) { best = eff; best_k = (int)k; }
        if (eff >= 0.985) break;
    }
    return best_k;
}

static inline Plan split_plan(int kernel, int count, int cpt, int n_omega, int angles_or_nx, int ny, int nc, int sms) {
    Plan pl{};
    pl.p_slices = 1; pl.t_slices = 1; pl.mode = MODE_DIRECT;
    size_t per_thread_p, per_thread_t;                // partial doubles per thread and slice
    int slots, chunk_units;
    if (kernel == K_DIRECT) {
        const int64_t T = (int64_t)((n_omega + PLAN_W - 1) / PLAN_W) * angles_or_nx;       // angles_or_nx = angles
        pl.tiles = (int)((T + PLAN_TPB - 1) / PLAN_TPB);
        pl.t_pad = (int64_t)pl.tiles * PLAN_TPB;
        per_thread_p = PLAN_W; per_thread_t = (size_t)nc * PLAN_W;
        slots = 2 * sms;                              // two CTAs per SM
        chunk_units = std::max(1, cpt);
    } else {
        const int wy = nc == 6 ? 2 : 4, ev = 4 * wy;
        pl.tiles = ((n_omega + 15) / 16) * ((angles_or_nx + 15) / 16) * ((ny + 4 * wy - 1) / (4 * wy));
        pl.t_pad = (int64_t)pl.tiles * PLAN_SEP_CONS;
        per_thread_p = ev; per_thread_t = (size_t)nc * ev;
        slots = sms;                                  // one CTA per SM
        chunk_units = std::max(1, cpt / 2);           // at least two chunks per time slice
    }
    if (pl.tiles < 8 * sms) {
        const int64_t kmax = std::max<int64_t>(1, (int64_t)count * chunk_units);
        const int best_k = best_slices(pl.tiles, slots, kmax, kernel == K_DIRECT ? 8 * sms : 4 * sms, kernel == K_DIRECT);
        if (best_k > 1) {
            if (count >= best_k) { pl.mode = MODE_PSLICE; pl.p_slices = best_k; }
            else {
                const int ts = std::min((best_k + count - 1) / count, chunk_units);
                if (ts > 1) { pl.mode = MODE_TSPLIT; pl.t_slices = ts; pl.p_slices = count; }
                else if (count > 1) { pl.mode = MODE_PSLICE; pl.p_slices = count; }
            }
        }
    }
    if (pl.mode == MODE_PSLICE) pl.partial_bytes = align_up((size_t)pl.p_slices * per_thread_p * pl.t_pad * 8, 256);
    if (pl.mode == MODE_TSPLIT) pl.partial_bytes = align_up((size_t)count * pl.t_slices * per_thread_t * pl.t_pad * 8, 256);
    return pl;
}

// Relative cost of one point in the direct kernel, in units of one PADDED point of the separable kernel: the
// measured break-even fills of round 1 (60 % with 4 accumulators per point, 75 % with 6; the separable kernel
// is 1.8x / 1.4x faster on full tiles and loses a little to the ordered reduction of its bigger partials).
static inline double direct_cost(int nc) { return nc == 6 ? 1.0 / 0.75 : 1.0 / 0.6; }

static inline int round_up(int v, int m) { return (v + m - 1) / m * m; }

// Which parts evaluate a grid.  `kernel` is the rad_kernel option (0 auto, 1 direct, 2 separable).
static inline void choose_parts(int n_omega, int n_thx, int n_thy, int nc, int kernel, double evals, bool allow_two,
                                Part *part, int &nparts) {
    const int ty = nc == 6 ? 8 : 16;
    auto whole = [&](int k) {
        part[0] = Part{k, n_thx, n_thy, -1, -1, n_thx * n_thy, Plan{}, 0, 1, 0, 0};
        nparts = 1;
    };
    if (kernel == 1) return whole(K_DIRECT);
    if (kernel == 2) return whole(K_SEP);
    const double r = direct_cost(nc);
    const double w16 = round_up(n_omega, 16), w8 = round_up(n_omega, PLAN_W);
    const double cost_direct = r * w8 * n_thx * n_thy;
    const double cost_sep = w16 * round_up(n_thx, 16) * round_up(n_thy, ty);
    double best = std::min(cost_direct, cost_sep);
    int bx = -1, by = -1;
    // two parts: interior of whole tiles along an axis whose remainder is cheaper in the direct kernel than as padding.
    // Worth it only where the work dwarfs the extra launches (>= 2e8 evals ~ 0.2 ms).
    if (allow_two && evals >= 2e8) {
        const int xs[2] = {n_thx / 16 * 16, n_thx}, ys[2] = {n_thy / ty * ty, n_thy};
        for (int a = 0; a < 2; ++a)
            for (int b = 0; b < 2; ++b) {
                const int x0 = xs[a], y0 = ys[b];
                if (x0 <= 0 || y0 <= 0 || (x0 == n_thx && y0 == n_thy)) continue;
                const double rest = (double)n_thx * n_thy - (double)x0 * y0;
                // the rest is a small grid: its time-split plan fills the GPU less well than a big one
                const double c = w16 * round_up(x0, 16) * round_up(y0, ty) + 1.15 * r * w8 * rest;
                if (c < 0.97 * best) { best = c; bx = x0; by = y0; }
            }
    }
    if (bx > 0) {
        part[0] = Part{K_SEP, bx, by, -1, -1, bx * by, Plan{}, 0, 1, 0, 0};
        part[1] = Part{K_DIRECT, n_thx, n_thy, bx, by, n_thx * n_thy - bx * by, Plan{}, 0, 1, 0, 0};
        nparts = 2;
        return;
    }
    whole(cost_sep <= cost_direct ? K_SEP : K_DIRECT);
}

// The fused single-launch kernel: one trajectory, direct-kernel arithmetic, every CTA resident at once
// (cooperative launch).  Tiles of FUSED_TPB threads x PLAN_W omegas; the time axis is cut into as many slices as
// fill `resident` CTAs (at least 32 samples each).
static inline bool fused_applies(int count, int64_t n_max, int n_omega, int n_thx, int n_thy, int resident,
                                 int &tiles, int &slices) {
    if (count != 1 || resident <= 0) return false;
    const int64_t T = (int64_t)((n_omega + PLAN_W - 1) / PLAN_W) * n_thx * n_thy;
    const int64_t t64 = (T + FUSED_TPB - 1) / FUSED_TPB;
    if (t64 > resident) return false;
    tiles = (int)t64;
    // at least 32 samples per slice: below that the per-CTA prologue (omega* as double-doubles, base phases)
    // is no longer small against the samples it serves
    const int64_t max_by_samples = std::max<int64_t>(1, n_max / 32);
    slices = (int)std::max<int64_t>(1, std::min<int64_t>(resident / tiles, max_by_samples));
    return true;
}

static inline CallPlan plan_call(int count, int64_t n_max, int n_omega, int n_thx, int n_thy, int nc, int kernel,
                                 bool angular, int sms, int fused_resident) {
    CallPlan cp{};
    if (sms <= 0) sms = 148;
    cp.cpt = (int)((n_max + PLAN_CH - 1) / PLAN_CH);
    const double evals = (double)n_omega * n_thx * n_thy * (double)n_max * count;
    cp.fused = false;
    if (!angular && (kernel == 3 || kernel == 0)) {
        int ft, fs;
        // auto: only small problems (< 2e8 evals ~ 0.3 ms, where launch overhead matters) with short trajectories
        // -- the fused kernel packs on the fly and has no TMA prefetch, which costs a few per cent on long ones
        if (fused_applies(count, n_max, n_omega, n_thx, n_thy, fused_resident, ft, fs)
            && (kernel == 3 || (n_max <= 32768 && evals < 2e8))) {
            Part tmp[2]; int np = 1;
            if (kernel == 0) choose_parts(n_omega, n_thx, n_thy, nc, 0, evals, false, tmp, np);
            if (kernel == 3 || tmp[0].kernel == K_DIRECT) {
                cp.fused = true; cp.fused_tiles = ft; cp.fused_slices = fs;
            }
        }
    }
    choose_parts(n_omega, n_thx, n_thy, nc, kernel == 3 ? 1 : kernel, evals, !angular, cp.part, cp.nparts);
    size_t off = 0;
    cp.off_packed = off; off += align_up((size_t)count * cp.cpt * (8 + PLAN_CH * 10) * 8, 256);
    cp.off_n = off;      off += align_up((size_t)count * sizeof(int64_t), 256);
    cp.off_lam = off;    off += align_up((size_t)count * sizeof(double), 256);
    cp.off_start = off;  off += align_up((size_t)count * sizeof(int64_t), 256);
    for (int i = 0; i < cp.nparts; ++i) {
        Part &pt = cp.part[i];
        pt.plan = pt.kernel == K_DIRECT ? split_plan(K_DIRECT, count, cp.cpt, n_omega, pt.angles, 0, nc, sms)
                                        : split_plan(K_SEP, count, cp.cpt, n_omega, pt.n_thx, pt.n_thy, nc, sms);
        pt.f_tiles = pt.f_slices = 0;
        if (pt.kernel == K_DIRECT && pt.l_x0 >= 0 && count == 1 && n_max <= 32768) {
            // the rest of a two-part plan is a small problem of its own: (n_omega / 8) x angles threads.  The fused
            // kernel evaluates it in one launch with sample-granular time slices (the direct kernel's slices are
            // whole 128-sample chunks: 24 chunks over 480 CTAs on the paper's grid) and no second pass
            const int64_t T = (int64_t)((n_omega + PLAN_W - 1) / PLAN_W) * pt.angles;
            const int64_t t64 = (T + FUSED_TPB - 1) / FUSED_TPB;
            if (fused_resident > 0 && t64 <= fused_resident) {
                pt.f_tiles = (int)t64;
                pt.f_slices = (int)std::max<int64_t>(1, std::min<int64_t>(fused_resident / t64, std::max<int64_t>(1, n_max / 32)));
                pt.plan.mode = MODE_TSPLIT; pt.plan.p_slices = 1; pt.plan.t_slices = pt.f_slices; pt.plan.tiles = pt.f_tiles;
                pt.plan.partial_bytes = align_up((size_t)pt.f_slices * nc * PLAN_W * pt.f_tiles * FUSED_TPB * 8, 256);
            }
        }
        pt.off_partial = off;
        off += pt.plan.partial_bytes;
        pt.cl = 1;
#ifndef RAD_SEP_NO_CLUSTER
        if (pt.kernel == K_SEP) {
            const int ty = nc == 6 ? 8 : 16;
            if (((pt.n_thy + ty - 1) / ty) % 2 == 0) pt.cl = 2;
            else if (nc == 4 && !angular && ((n_omega + 15) / 16) % 2 == 0) pt.cl = 3;
        }
#endif
    }
    if (cp.fused) {           // partial amplitudes of the fused kernel: [slices][nc * W][tiles * FUSED_TPB]
        cp.part[0].off_partial = cp.off_packed;       // it needs no packed buffer: reuse the space from the start
        const size_t need = align_up((size_t)cp.fused_slices * nc * PLAN_W * cp.fused_tiles * FUSED_TPB * 8, 256);
        off = std::max(off, need);
    }
    cp.off_ang = off;
    if (angular) {            // per-(tile, omega slot) sums of the fused angular spectrum
        const Part &pt = cp.part[0];
        const int groups = std::min((n_omega + PLAN_W - 1) / PLAN_W, (PLAN_TPB + pt.angles - 1) / pt.angles + 1);
        off += align_up(pt.kernel == K_SEP ? (size_t)pt.plan.tiles * 16 * 8
                                           : (size_t)pt.plan.tiles * groups * PLAN_W * 8, 256);
    }
    cp.total = off;
    return cp;
}

}  // namespace rad
