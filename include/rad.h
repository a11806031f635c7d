/*
 * rad.h -- C ABI of the B200 (sm_100a) FP64 radiation-integral evaluator.
 *
 * The operation (arXiv 1910.10391, cited by line of PAPER.md):
 *
 *   d2I/(dw dOmega) = e^2/4pi^2 | int f(t,n) e^{i w (t - n.x(t))} dt |^2        eq. (1)
 *
 * in the paper's small-angle, leading-order expanded form -- f_x, f_y, f_z of
 * eqs. (3)-(5), g of eq. (6), phase of eq. (7)
 * -- evaluated for EVERY point of a tensor grid (w, n_x, n_y) over
 * one sampled trajectory ("the integral over the same trajectory N_x x N_y x N_w
 * times"; result "saved in a cube"), classically or
 * with the semi-classical substitution w -> w* = w/(1 - hbar w/E):
 *
 *   spin-0   (substitution model) out = (w/w*) classical(w*)                     eq. (9),
 *   spin-1/2 (BCK model)          out = [ (E*^2+E^2)/2E^2 |I|^2
 *                                       + w^2/(2 E^2 gamma^2) |J|^2 ] / 4pi^2    eqs. (10)-(12)
 *
 * and summed over trajectories / crystal sections.
 * The time integral is the composite trapezoid rule on the given samples
 * (reading Q1); the acceleration is zero outside [t_0, t_{n-1}] (Q2).
 *
 * Units: c = 1; t, x, y, dz in one length unit (metres in all shipped workloads);
 * v dimensionless; accelerations per length; omega in rad per length.  Output in
 * units of e^2 (multiply by alpha = 1/137.036 for hbar = c = 1), 1/4pi^2 included.
 *
 * Conventions common to all calls
 *   - Every `const double*` inside rad_traj / rad_traj_batch / rad_grid and every
 *     `out` is DEVICE memory owned by the caller, 8-byte aligned, read-only for the
 *     inputs.  The *_host entry points at the end take HOST memory instead.
 *   - `workspace` is caller-owned DEVICE scratch of at least rad_workspace_bytes()
 *     bytes, 256-byte aligned.  If NULL, scratch is taken from the device's
 *     stream-ordered pool (cudaMallocAsync / cudaFreeAsync on `cuda_stream`) and
 *     released in stream order; the first such call raises that pool's release threshold
 *     (cudaMemPoolAttrReleaseThreshold) so that freed scratch stays cached in the pool instead
 *     of going back to the driver at every synchronisation.  The library keeps no pointer past
 *     the enqueued work and allocates nothing persistent of its own.
 *   - `cuda_stream` is a cudaStream_t (NULL = legacy default stream).  All work is
 *     enqueued on it; no call synchronises the host (the *_host calls do, once, at
 *     the end).  With a caller workspace the single-trajectory calls enqueue kernels only
 *     (no allocation, no host copy), so they can be captured in a CUDA graph and replayed.
 *   - Cube order: out[(i_w * n_thy + i_y) * n_thx + i_x]  (theta_x fastest).
 *   - Return value: RAD_OK (0) or a negative rad_status; nothing throws or aborts.
 *     Not checked (garbage in, NaN/inf out): non-monotone t, q <= 0, non-finite
 *     samples.  A grid point with u = omega * hbarc_over_E >= 1 (photon energy above
 *     the particle energy, no final state) yields NaN at that point (the omega array
 *     lives on the device; no host-side check, no sync).
 *   - `opt` (last argument but one of every compute call) carries per-call options; NULL = defaults.
 *     There is no process-wide switch: two threads may call with different options.
 *   - Results are deterministic run to run (fixed reduction order, no FP atomics).
 *   - There is no CPU fallback: without a CUDA device every compute call returns
 *     RAD_ECUDA.
 */
#ifndef RAD_H
#define RAD_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum {
    RAD_OK = 0,
    RAD_EINVAL = -1,      /* null pointer, n < 2, empty grid, bad spin/model, misaligned pointer */
    RAD_EDOMAIN = -2,     /* host-visible parameter outside the method's domain (hbarc_over_E < 0) */
    RAD_ECUDA = -3,       /* CUDA runtime error; rad_strerror gives the CUDA text of the last one */
    RAD_ENOSPACE = -4,    /* workspace given but smaller than rad_workspace_bytes() */
    RAD_ETOOBIG = -5      /* rad_eval_static: the call needs more scratch than rad_static_scratch_bytes() */
} rad_status;

typedef enum { RAD_CLASSICAL = 0, RAD_SPIN0 = 1, RAD_SPIN_HALF = 2 } rad_model;

/* Which main kernel evaluates the integrals.
 *   RAD_KERNEL_AUTO       chosen from the shapes (what every shipped workload uses):
 *                         - the separable-phasor kernel (e^{i w psi} = T(w, n_x) Y(w, n_y) on a tensor grid, exact
 *                           because theta^2 = n_x^2 + n_y^2, eq. (7)) on the part of the grid that
 *                           fills its 16 x 16 x 16 (spin-1/2: 16 x 16 x 8) point tiles; angle rows / columns left
 *                           over (e.g. the paper's typical 50 x 50 angles: 48 x 48 + an L-shaped
 *                           rest) go to the direct kernel in a second launch when that is cheaper than padding;
 *                         - the direct kernel (one phasor per eval) where the grid fills those tiles badly;
 *                         - the fused single-launch kernel for one short trajectory on a grid too small to fill
 *                           the GPU (a cooperative launch: pack, time split over all SMs, grid-wide ordered
 *                           reduction and epilogue in one kernel).
 *   RAD_KERNEL_DIRECT     always the direct kernel (separate pack / main / reduction launches)
 *   RAD_KERNEL_SEPARABLE  always the separable kernel, padding the grid to whole tiles
 *   RAD_KERNEL_FUSED      the fused single-launch kernel; RAD_EINVAL where it does not apply (count > 1,
 *                         more tiles than fit on the GPU at once)
 * All of them meet the same tolerance and are parity-tested separately. */
typedef enum { RAD_KERNEL_AUTO = 0, RAD_KERNEL_DIRECT = 1, RAD_KERNEL_SEPARABLE = 2, RAD_KERNEL_FUSED = 3 } rad_kernel;

/* Per-kernel timing of ONE call (bench.py's roofline needs the main kernel's own duration): an opaque set of
 * CUDA events created on the current device.  Pass it in rad_options.profile; the call records the events on
 * its stream around its pack / main / reduction launches; rad_profile_read waits for the last one and returns
 * ms[0..2] = pack, main (all main-kernel launches of the call), reduction durations (0 where not run).
 * One profile object must not be used by two calls at the same time. */
typedef struct rad_profile rad_profile;
rad_profile *rad_profile_create(void);                 /* NULL on failure (no device) */
void rad_profile_destroy(rad_profile *profile);
int rad_profile_read(rad_profile *profile, float *ms);

typedef struct {
    int32_t kernel;          /* rad_kernel; 0 = auto */
    int32_t reserved;        /* must be 0 */
    rad_profile *profile;    /* NULL: no timing */
} rad_options;

/* One trajectory (or one crystal section), structure of arrays, n >= 2 samples.
 * t: time; dz = z - beta0 t; x, y; vx, vy; dvz = v_z - beta0 (beta0 = 1 - 1/2gamma^2,
 * PAPER.md:28); ax, ay, az: accelerations; gamma: Lorentz factor per sample (Q6:
 * 1/2gamma_k^2 is used sample-wise, the J coefficient of eq. 10 uses gamma[0]). */
typedef struct {
    int64_t n;
    const double *t, *dz, *x, *y, *vx, *vy, *dvz, *ax, *ay, *az, *gamma;
} rad_traj;

/* `count` trajectories; row p of each array starts at element p*stride and holds
 * n[p] <= stride samples.  `n` is a HOST array (it sizes the launch). */
typedef struct {
    int32_t count;
    int64_t stride;
    const int64_t *n;
    const double *t, *dz, *x, *y, *vx, *vy, *dvz, *ax, *ay, *az, *gamma;
} rad_traj_batch;

/* Tensor grid: omega[n_omega] >= 0 (rad/length), thx[n_thx] = n_x, thy[n_thy] = n_y
 * (direction cosines, small; theta^2 = n_x^2 + n_y^2). */
typedef struct {
    int32_t n_omega, n_thx, n_thy;
    const double *omega, *thx, *thy;
} rad_grid;

/* Classical spectrum, eq. (1) with eqs. (3)-(7).  out: n_omega*n_thy*n_thx doubles. */
int rad_classical(const rad_traj *traj, const rad_grid *grid, double *out,
                  void *workspace, size_t workspace_bytes, const rad_options *opt, void *cuda_stream);

/* Semi-classical spectrum.  spin = 0: substitution model, eq. (9); spin = 1: spin-1/2,
 * BCK eq. (10).  hbarc_over_E = hbar c / E in the length unit, so that
 * u = hbar w / E = omega * hbarc_over_E and w* = omega / (1 - u). */
int rad_semiclassical(const rad_traj *traj, const rad_grid *grid, int spin,
                      double hbarc_over_E, double *out,
                      void *workspace, size_t workspace_bytes, const rad_options *opt, void *cuda_stream);

/* out[m] (+)= sum over p (ascending) of the spectrum of trajectory p.
 * hbarc_over_E: HOST array, one per trajectory (NULL allowed iff model is classical).
 * batch->n and hbarc_over_E are read on the host (they size the launch) and, for count > 1, copied to the device
 * through `cuda_stream` (cudaMemcpyAsync from the caller's memory): pageable memory is staged by the runtime before
 * the call returns -- which may make the call wait for earlier work of the stream -- and pinned memory must stay
 * valid and unchanged until the stream has passed the copy.  Up to 2^31 - 1 trajectories (more than 65 535 are
 * packed in several passes of one launch).
 * accumulate: 0 overwrites out, 1 adds to it (resume a partial ensemble). */
int rad_ensemble_sum(const rad_traj_batch *batch, const rad_grid *grid, rad_model model,
                     const double *hbarc_over_E, int accumulate, double *out,
                     void *workspace, size_t workspace_bytes, const rad_options *opt, void *cuda_stream);

/* dI/dw[i_w] = d_solid_angle * sum over the angles of the spectrum of an ensemble, optionally only where
 * n_x^2 + n_y^2 <= theta_cut^2 (theta_cut <= 0: no mask) -- the paper's "final sum over the spatial integrals"
 * -- WITHOUT the cube (3000^2 angles x 100 omegas "approach the limit" of GPU
 * memory at one double per integral).  When the grid fills the GPU (one CTA per tile, no time / trajectory
 * split) the sum over a tile's angles is formed in the main kernel's epilogue in a fixed order, one partial per
 * (tile, omega) is written and a small second pass adds the partials in tile order: no cube is written at all.
 * Smaller grids (fewer than 8 tiles per SM: their cube is < 40 MB) are evaluated into a cube inside the
 * workspace and summed by rad_angular_sum.
 * spectrum: n_omega doubles (device), overwritten.  workspace: DEVICE, 256-byte aligned, REQUIRED here, at
 * least rad_angular_spectrum_workspace_bytes() bytes.  batch->n and hbarc_over_E are HOST arrays as in
 * rad_ensemble_sum (count = 1 for a single trajectory).  Same values as cube + rad_angular_sum up to the
 * rounding of a different summation order. */
int rad_angular_spectrum(const rad_traj_batch *batch, const rad_grid *grid, rad_model model,
                         const double *hbarc_over_E, double d_solid_angle, double theta_cut, double *spectrum,
                         void *workspace, size_t workspace_bytes, const rad_options *opt, void *cuda_stream);
size_t rad_angular_spectrum_workspace_bytes(int32_t count, int64_t n_max, int32_t n_omega, int32_t n_thx,
                                            int32_t n_thy);

/* Photon NUMBER spectrum from an intensity spectrum (eqs. 8-9: the substitution model is
 * stated for dN/d(hbar w); dI = hbar w dN):  number[i] = spectrum[i] / (hbar_c * omega[i]), i.e. with
 * spectrum = dI/dw (per rad/length, as rad_angular_spectrum returns it) and hbar_c in energy x length this is
 * dN/dw = (dI/dw) / (hbar w); divide by hbar_c once more for dN/d(hbar w).  omega[i] = 0 gives +inf (or NaN for
 * 0/0), as the formula does.  All arrays DEVICE, n entries; number may alias spectrum. */
int rad_number_spectrum(const double *spectrum, const double *omega, int32_t n, double hbar_c, double *number,
                        void *cuda_stream);

/* One long trajectory cut into sections with their own energy -- the paper's treatment of energy
 * loss: "the total spectrum is then the sum of the spectra from each section".
 * out[m] (+)= sum over s (ascending) of the spectrum of samples start[s] .. start[s+1], BOTH included:
 * neighbouring sections share their boundary sample, so their trapezoid weights tile the time axis.
 * start: HOST array of n_sections + 1 strictly ascending sample indices in [0, traj->n - 1];
 * hbarc_over_E: HOST array, one per section (NULL allowed iff classical).
 * Boundary-sample rule: sample start[s] (s > 0) belongs to sections s - 1 and s and is read from the ONE array
 * entry both times -- gamma[start[s]] enters 1/(2 gamma_k^2) of both sections' end weights, and the J
 * coefficient of eq. (10) of section s uses gamma[start[s]] (its first sample).  A caller who fixes E per
 * section "to the value at entering the section" therefore stores the NEW section's gamma at the
 * boundary sample; the energies differ by the loss over one section, which is the approximation the paper
 * makes anyway.  Sections with exactly their own arrays are what rad_ensemble_sum takes.
 * Choosing the sections (each longer than the formation length) is the caller's business; this
 * call does not check it -- rad_sections_check does, on host-visible numbers.
 * start and hbarc_over_E are read before the call returns (copied to the device through the stream; pageable
 * memory is staged by the runtime, pinned memory must stay valid until the stream has passed the copy). */
int rad_sections_sum(const rad_traj *traj, int32_t n_sections, const int64_t *start, const rad_grid *grid,
                     rad_model model, const double *hbarc_over_E, int accumulate, double *out,
                     void *workspace, size_t workspace_bytes, const rad_options *opt, void *cuda_stream);

/* Formation length l_f = 2 gamma^2 (E - w)/(E w), in the length unit of omega (c = hbar = 1:
 * omega in rad/length, u = omega * hbarc_over_E = hbar w / E).  A section handed to rad_sections_sum must be
 * longer than this.  Host arithmetic only; returns -1 on arguments outside the domain (u >= 1, omega <= 0).
 * Note: for the paper's own example (50 GeV positron, 5 GeV photon) the formula gives 680 nm, while the
 * paper prints 71 nm -- the text is at odds with itself there; the formula is what this returns. */
double rad_formation_length(double gamma, double omega, double hbarc_over_E);

/* The check PAPER.md:73-75 asks of a sectioning ("section length longer than the formation length"), on HOST
 * arrays: section s spans t_start[s] .. t_start[s+1] (the times of the boundary samples, n_sections + 1
 * entries, ascending; c = 1 so a time is a length), has Lorentz factor gamma0[s] and hbarc_over_E[s] (NULL:
 * classical, u = 0).  The formation length is longest at the lowest frequency, so omega_min = the smallest
 * POSITIVE omega of the grid decides.  Writes to `short_sections` (capacity `cap`, may be NULL if cap = 0) the
 * indices of the sections with t_start[s+1] - t_start[s] <= l_f(gamma0[s], omega_min, hbarc_over_E[s]), in
 * ascending order, and returns how many there are (possibly more than cap); RAD_EINVAL / RAD_EDOMAIN
 * (negative) on bad arguments.  Host arithmetic only. */
int rad_sections_check(int32_t n_sections, const double *t_start, const double *gamma0,
                       const double *hbarc_over_E, double omega_min, int32_t *short_sections, int32_t cap);

/* dI/dw[i_w] = sum_{i_x,i_y} cube * d_omega_solid, optionally only where
 * n_x^2 + n_y^2 <= theta_cut^2 (theta_cut <= 0: no mask) -- the paper's "final sum over
 * the spatial integrals", done on the device.  `cube` is the output of
 * one of the calls above; spectrum: n_omega doubles (device). */
int rad_angular_sum(const double *cube, const rad_grid *grid, double d_solid_angle,
                    double theta_cut, double *spectrum, void *cuda_stream);

/* Trajectories of `count` particles in a static synthetic well, generated on the device in the SoA
 * layout the calls above read -- the paper's outlook "many particle trajectories evaluated in parallel
 * on the GPU", for the wells of BASELINE.json configs 2-5 (the paper's own solver
 * needs potential tables that are not available).  Fixed-step velocity Verlet:
 *   a_k = A(r_k), v_h = v_k + dt/2 a_k, r_{k+1} = r_k + dt v_h, v_{k+1} = v_h + dt/2 A(r_{k+1})
 *   RAD_WELL_COSINE:     A_x = -kappa sin(2 pi x / length), A_y = 0
 *   RAD_WELL_AXIAL_EXP:  A = -kappa (r/|r|) exp(-|r| / length), A(0) = 0
 * RAD_WELL_HARMONIC_MS (planar harmonic well with multiple-scattering kicks, the recipe of configs 2 and 4;
 * kappa = w_p^2, length unused but > 0): exact rotation of (x, u = vx / w_p) by w_p dt, then Gaussian kicks
 *   x_{k+1} = c x_k + s u_k,  u_{k+1} = c u_k - s x_k + (sigma/w_p) xi1_{k+1},  vy_{k+1} = vy_k + sigma xi2_{k+1},
 *   ax_k = -w_p^2 x_k + sigma xi1_k/dt, ay_k = sigma xi2_k/dt (xi_0 = 0), y = cumulative trapezoid of vy;
 *   xi1, xi2 of (particle p, step k) = Box-Muller of the uniforms (r + 1/2) 2^-32 from the first two words of
 *   Philox4x32-10 with counter (k low, k high, p, 0) and key (seed low, seed high): reproducible anywhere.
 * sigma and seed are ignored by the two deterministic wells.
 * and t_k = k dt, dvz = -(vx^2 + vy^2)/2, dz = cumulative trapezoid of dvz (dz_0 = 0),
 * az = -(vx ax + vy ay) (leading-order relations), gamma_k = gamma.
 * x0, y0, vx0, vy0: DEVICE arrays of `count` initial values.  out: DEVICE arrays [count][stride], the
 * first n entries of each row are written (pass them to rad_ensemble_sum as a rad_traj_batch with
 * the same stride).  One thread per particle: meant for many particles. */
typedef enum { RAD_WELL_COSINE = 0, RAD_WELL_AXIAL_EXP = 1, RAD_WELL_HARMONIC_MS = 2 } rad_well;
typedef struct {
    double *t, *dz, *x, *y, *vx, *vy, *dvz, *ax, *ay, *az, *gamma;
} rad_traj_buffers;
int rad_generate_trajectories(rad_well well, double kappa, double length, double gamma, double dt,
                              double sigma, uint64_t seed, int32_t count, int64_t n, int64_t stride,
                              const double *x0, const double *y0, const double *vx0, const double *vy0,
                              const rad_traj_buffers *out, void *cuda_stream);

/* out[i] (+)= cubes[0*m + i] + cubes[1*m + i] + ... + cubes[(count-1)*m + i], added in that
 * order (fixed order: deterministic).  Combines the partial cubes of ensemble shards -- other
 * GPUs' (after an all-gather) or successive batches' -- into the ensemble sum of PAPER.md:75,
 * 149.  cubes: count*m doubles, out: m doubles, both DEVICE; out must not overlap cubes. */
int rad_sum_cubes(const double *cubes, int32_t count, int64_t m, int accumulate, double *out,
                  void *cuda_stream);

/* Scratch needed by any call above for `count` trajectories of at most n_max samples on a
 * grid of the given shape (count = 1 for the single-trajectory calls).  0 on bad input. */
size_t rad_workspace_bytes(int32_t count, int64_t n_max,
                           int32_t n_omega, int32_t n_thx, int32_t n_thy);

/* HOST-buffer variants (the paper's flow: trajectory copied to the GPU once, cube copied
 * back once).  Every pointer inside traj/batch/grid and `out` is HOST memory
 * (pinned memory makes the copies asynchronous).  Device buffers come from the
 * stream-ordered pool; the call returns after the result is in `out` (it synchronises the stream once).
 * Arrays that follow one another in host memory in the order t, dz, x, y, vx, vy, dvz, ax, ay, az, gamma, omega, thx,
 * thy (any run of them in one allocation) are copied in one transfer instead of one each.
 * model: rad_model; hbarc_over_E ignored for RAD_CLASSICAL. */
int rad_eval_host(const rad_traj *traj, const rad_grid *grid, rad_model model,
                  double hbarc_over_E, double *out, const rad_options *opt, void *cuda_stream);
int rad_ensemble_sum_host(const rad_traj_batch *batch, const rad_grid *grid, rad_model model,
                          const double *hbarc_over_E, int accumulate, double *out,
                          const rad_options *opt, void *cuda_stream);

/* The entry point that ALLOCATES NOTHING: the cube of one trajectory (classical, spin-0 or spin-1/2; the same
 * operation and the same kernels as rad_classical / rad_semiclassical) for callers that must not reach cudaMalloc or
 * a memory pool -- code under CUDA graph capture, tight serving loops, harnesses that forbid allocation.  Its scratch
 * (packed trajectory records, partial amplitudes of a time split) lives in ONE file-scope device array of
 * rad_static_scratch_bytes() = 16 MiB that every GPU loading the library holds until the process exits.
 *   - All pointers DEVICE memory as in rad_classical; the caller passes inputs and `out` (n_omega*n_thy*n_thx doubles).
 *   - Limit: calls whose launch plan needs more than rad_static_scratch_bytes() return RAD_ETOOBIG and enqueue
 *     nothing (rad_workspace_bytes(1, n, n_omega, n_thx, n_thy) is an upper bound of the need; e.g. BASELINE
 *     config 1 fits, config 2's 16-way time split does not -- use rad_classical with a workspace there).
 *   - Calls no cudaMalloc / cudaMallocAsync / cudaFree and no allocating library routine; it enqueues kernels on
 *     `cuda_stream` and does not synchronise.  (The first call on a device asks the runtime for the array's device
 *     address, cudaGetSymbolAddress, once.)
 *   - Every call on a device shares the one array, which keeps the previous call's contents: the kernels overwrite
 *     every byte they later read, so nothing needs clearing, but two calls that OVERLAP on the GPU (different
 *     streams, or a captured graph replayed concurrently with itself) race on it -- keep them in one stream order.
 * hbarc_over_E is ignored for RAD_CLASSICAL. */
int rad_eval_static(const rad_traj *traj, const rad_grid *grid, rad_model model, double hbarc_over_E, double *out,
                    const rad_options *opt, void *cuda_stream);
size_t rad_static_scratch_bytes(void);

/* FP64 FMA peak of the current device, measured: runs a register-resident DFMA chain
 * kernel for about `millis` ms and returns FLOP/s (2 per FMA lane); <= 0 on error. */
double rad_measure_fp64_peak(double millis, void *cuda_stream);

/* Number of kernels the library has launched in this process (bench bookkeeping; a relaxed atomic counter,
 * the only process-wide state besides per-device attribute caches). */
int64_t rad_launch_count(void);

/* Which kernel a call on a grid of this shape uses for `count` trajectories of at most n_max samples under
 * the option `kernel` (a rad_kernel): 1 direct, 2 separable, 3 fused -- for the largest part of the grid when the
 * call is split in two launches.  A pure function of the arguments and the SM count (148 assumed when no device
 * is visible); RAD_EINVAL on bad input. */
int rad_plan_kernel(int32_t count, int64_t n_max, int32_t n_omega, int32_t n_thx, int32_t n_thy,
                    rad_model model, int32_t kernel);

/* The launch plan of such a call, for inspection and tests: plan[0] kernel of the first (largest) part (1 direct,
 * 2 separable, 3 fused), plan[1] its mode (0 one CTA per tile, 1 trajectory axis sliced, 2 time axis sliced),
 * plan[2] tiles = gridDim.x, plan[3] slices = gridDim.y, plan[4] time slices per trajectory, plan[5] chunks of
 * 128 samples per trajectory, plan[6] number of parts (2: separable interior + direct kernel on the L-shaped
 * rest of the angle plane), plan[7] angle columns and plan[8] angle rows of the separable interior (0 if none),
 * plan[9] kernel launches of the whole call, plan[10] CTAs per thread-block cluster of the first part (2: the
 * separable kernel runs as cluster pairs on neighbouring angle tiles that share one phasor table through
 * distributed shared memory -- whenever the part has an even number of theta_y tiles; 3: pairs on neighbouring
 * omega tiles that share the integrand table, for an odd theta_y tile count with 4 accumulators per point; else 1).
 * plan: HOST array of at least 11 entries. */
int rad_plan_describe(int32_t count, int64_t n_max, int32_t n_omega, int32_t n_thx, int32_t n_thy,
                      rad_model model, int32_t kernel, int32_t *plan);

/* Static text for a rad_status; for RAD_ECUDA the text of the last CUDA error seen. */
const char *rad_strerror(int code);

#ifdef __cplusplus
}
#endif
#endif /* RAD_H */
