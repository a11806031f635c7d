// rad_sep.cuh -- separable-phasor kernel for tensor angle grids.
//
// Eq. (7) on a tensor grid separates exactly, because theta^2 = n_x^2 + n_y^2:
//     omega* psi = omega* [ (t/2gamma^2 - dz) + (n_x^2 t/2 - n_x x) ]  +  omega* [ n_y^2 t/2 - n_y y ]
//     e^{i omega* psi} = T(omega, n_x, k) * Y(omega, n_y, k)
// so a CTA that owns a tile of 16 omega x 16 n_x x (4 WY) n_y points needs, per sample, only
// 256 + 64 WY phasors (one sincos each, exact chunk-relative phase as in rad_main_kernel) instead
// of 1024 WY, plus the 64 WY omega-independent integrands f_x, f_y (h) of eqs. (3), (4), (12).
// Per eval what remains is one complex multiply and the complex accumulation (8 or 10 FP64
// instructions instead of 24 or 26).
//
// CTA = 256 consumer + 128 (4 accumulators per point) or 256 (6) producer threads, warp-specialised, one CTA per SM,
// launched as thread-block CLUSTER PAIRS wherever the tile counts allow: the two CTAs of a pair own neighbouring
// theta_y tiles (same T table) or neighbouring omega tiles (same F table), compute half of the shared table each and
// store the peer's copy through distributed shared memory (st.async, counted on the peer's mbarrier); see the kernel.
//   warps 8-..  PRODUCERS (phase A): wait for trajectory chunks (TMA ring), build the T, Y, F (H)
//               tables of SEP_S samples per sub-block into a ring of SEP_NB table buffers in
//               shared memory (16-byte entries: (re, im) of T and Y, (w f_x, w f_y) of F).
//   warps 0-7   CONSUMERS (phase B): thread tile 2 omega x 2 n_x x WY n_y (WY = 4 with 4
//               accumulators per point, WY = 2 with 6); per sample 20 table entries are read
//               and 16 (8) points updated.  Lane bits (high to low) = (l_x, l_y, l_w) = (2, 2, 1),
//               warp = (w_w, w_x) = (2, 1) bits; the table layouts put the entries one load touches
//               across a warp into one contiguous piece of shared memory.  Shared-memory cost is
//               counted in 128-byte wavefronts of REQUESTS: only lanes 2k, 2k+1 reading the same
//               address are merged (measured), so l_w is the lowest lane bit -- the
//               F table (8 entries per thread, independent of omega) then costs half.
// full[] / empty[] mbarriers hand table buffers over; setmaxnreg moves registers from the
// producers to the consumers, whose accumulators need them (SepRegs).
#pragma once

namespace rad {

constexpr int SEP_CONS = 256;  // consumer threads
#ifndef RAD_SEP_PROD4
#define RAD_SEP_PROD4 128
#endif
#ifndef RAD_SEP_PROD6
#define RAD_SEP_PROD6 256
#endif
#ifndef RAD_SEP_S
#define RAD_SEP_S 8
#endif
#ifndef RAD_SEP_NB
#define RAD_SEP_NB 2
#endif
#ifndef RAD_SEP_DEG
#define RAD_SEP_DEG 5          // polynomial set of the table phasors (sincos_coeffs.h): 5 = 1e-13 (as the direct kernel), 6 = 2e-16
#endif
#ifndef RAD_SEP_REGS_CONS4          // registers per consumer thread after setmaxnreg, 4 / 6 accumulators per point
#define RAD_SEP_REGS_CONS4 192
#endif
#ifndef RAD_SEP_REGS_CONS6
#define RAD_SEP_REGS_CONS6 168
#endif
#ifndef RAD_SEP_PU4
#define RAD_SEP_PU4 1
#endif
#ifndef RAD_SEP_PU6
#define RAD_SEP_PU6 4
#endif
#ifndef RAD_SEP_HS4                 // sample groups of the producers: NPROD / HS threads own the table entries, group h
#define RAD_SEP_HS4 1               // of them fills samples [h S / HS, (h + 1) S / HS) of every sub-block
#endif
#ifndef RAD_SEP_HS6
#define RAD_SEP_HS6 2
#endif
constexpr int SEP_S = RAD_SEP_S;       // samples per table sub-block
constexpr int SEP_NB = RAD_SEP_NB;     // table buffers in flight
constexpr int SEP_STAGES = 3;  // trajectory-chunk ring depth
// Producer threads per CTA (RAD_SEP_PROD4 / RAD_SEP_PROD6) and the register split.
// setmaxnreg moves registers between the roles inside the pool the CTA got at launch
// (THREADS * REGS_LAUNCH): 256 * CONS + NPROD * PROD <= that pool, both multiples of 8.
// Measured (round 2, ncu source page split by role): with 6 accumulators per point the tables serve only 8 points
// per consumer thread and the kernel is PRODUCER-bound: the consumers wait for tables 14-21 % of their time while a
// lone producer warp per sub-partition issues only 13-15 % of the cycles -- it is latency-bound (fixed-latency
// dependency 31 %, shared-memory scoreboard 18 %), not short of issue slots.  Steps, each measured on config 3:
//   * full unroll of the producers' sample loop + registers moved to them (176 / 152)              +5.8 %
//   * cluster pairs sharing the T table (-25 % producer work; see rad_sep_kernel)                   +5.9 %
//   * EIGHT producer warps as two sample groups (RAD_SEP_HS6 = 2: threads [0, 128) fill samples 0-3 of a
//     sub-block, threads [128, 256) samples 4-7, same entries), 168 / 88 registers, 4-sample unroll   +7.0 %
//     (two warps per sub-partition overlap each other's latencies; 160 / 96: -0.7 %, 152 / 104: -7 %: the
//     consumers' 48 accumulators + 20 table entries in flight need their 168)
// With 4 accumulators per point (classical, spin-0) the consumers wait only 4 % and need 192 registers: eight
// producer warps (184 / 72, 176 / 80) lose 4-10 % there, so that variant keeps four.
// What did not help: one T and one Y-or-F entry per thread for eight producer warps (round 1), finer or deeper
// table rings (4-sample sub-blocks x 4), the magic-number range reduction instead of FRND.F64 (+-0).
template <int NC> struct SepRegs {
    static constexpr int NPROD = NC == 6 ? RAD_SEP_PROD6 : RAD_SEP_PROD4;     // producer threads
    static constexpr int THREADS = SEP_CONS + NPROD;
    static constexpr int REGS_LAUNCH = 65536 / THREADS / 8 * 8;               // __launch_bounds__(THREADS, 1)
    static constexpr int CONS = NC == 6 ? RAD_SEP_REGS_CONS6 : RAD_SEP_REGS_CONS4;
    static constexpr int PROD = ((THREADS * REGS_LAUNCH - SEP_CONS * CONS) / NPROD) / 8 * 8;
    // samples the producers work on at once: their phasor chains are ~15 dependent FP64 steps long, and one
    // producer warp per sub-partition has only its own instruction-level parallelism to hide that latency
    static constexpr int PROD_UNROLL = NC == 6 ? RAD_SEP_PU6 : RAD_SEP_PU4;
    static constexpr int HS = NC == 6 ? RAD_SEP_HS6 : RAD_SEP_HS4;            // sample groups
    static constexpr int NE = NPROD / HS;                                     // threads that own table entries
    static_assert(NPROD % HS == 0 && NE % 32 == 0 && SEP_S % HS == 0, "sample groups are whole warps");
    static_assert(CONS % 8 == 0 && PROD >= 24 && SEP_CONS * CONS + NPROD * PROD <= THREADS * REGS_LAUNCH,
                  "setmaxnreg.inc would wait forever for registers the CTA does not own");
};

template <int NC, int WY>
struct SepShape {
    static constexpr int YN = 64 * WY;            // entries of the Y and F tables per sample
    static constexpr int EV = 4 * WY;             // grid points per consumer thread
    static constexpr int BYTES_T = SEP_NB * SEP_S * 256 * 16;    // T table ring: (re, im) per entry
    static constexpr int BYTES_Y = SEP_NB * SEP_S * YN * 16;     // Y ring (re, im); F ring (w f_x, w f_y)
    static constexpr int OFF_T = SEP_STAGES * CHUNK_BYTES;
    static constexpr int OFF_Y = OFF_T + BYTES_T;
    static constexpr int OFF_F = OFF_Y + BYTES_Y;
    static constexpr int OFF_H = OFF_F + BYTES_Y;                // H ring: w h, 8 bytes per entry (spin-1/2 only)
    static constexpr int OFF_BAR = OFF_H + (NC == 6 ? BYTES_Y / 2 : 0);
    static constexpr int SMEM = OFF_BAR + (SEP_STAGES + 2 * SEP_NB) * 8;
};

// Grid coordinates of a thread's EV points.  blockIdx.x enumerates (omega tile, y tile, x tile),
// x fastest.  Point e = (i * 2 + j) * WY + m  <->  omega index iw0 + i, x index ix0 + j, y index iy0 + m.
template <int WY>
struct SepCoord {
    int bw, bx, by;                  // first omega / x / y index of the CTA tile
    int iw0, ix0, iy0;               // first omega / x / y index of this thread's points
    int lw, lx, ly, ww, wx;
    // cl = 2: the CTAs of a cluster pair (blocks 2k, 2k + 1) own neighbouring y tiles of one (omega, x) tile,
    // so that they share the T table (rad_sep_kernel); the y tile count is even then.  cl = 3: neighbouring omega
    // tiles of one angle tile (shared F table); the omega tile count is even then.
    __device__ __forceinline__ SepCoord(int block, int tid, int n_thx, int n_thy, int cl) {
        const int ntx = (n_thx + 15) / 16, nty = (n_thy + 4 * WY - 1) / (4 * WY);
        if (cl == 2) {
            const int rest = block >> 1, half = nty >> 1;
            bx = (rest % ntx) * 16;
            by = (((rest / ntx) % half) * 2 + (block & 1)) * 4 * WY;
            bw = (rest / (ntx * half)) * 16;
        } else if (cl == 3) {                         // pairs on neighbouring OMEGA tiles of one angle tile (shared F table)
            const int rest = block >> 1;
            bx = (rest % ntx) * 16;
            by = ((rest / ntx) % nty) * 4 * WY;
            bw = ((rest / (ntx * nty)) * 2 + (block & 1)) * 16;
        } else {
            bx = (block % ntx) * 16;
            by = ((block / ntx) % nty) * 4 * WY;
            bw = (block / (ntx * nty)) * 16;
        }
        const int lane = tid & 31, warp = tid >> 5;
        lw = lane & 1; ly = (lane >> 1) & 3; lx = (lane >> 3) & 3;
        ww = warp >> 1; wx = warp & 1;
        iw0 = bw + 4 * ww + 2 * lw;
        ix0 = bx + 8 * wx + 2 * lx;
        iy0 = by + WY * ly;
    }
};

// omega* / 2 pi as a double-double, shared by both kernels' prologues
__device__ __forceinline__ dd omega_star_turns(double om, double lam) {
    dd u = two_prod(om, lam);
    dd d = two_sum(1.0, -u.hi);
    d = fast_two_sum(d.hi, d.lo - u.lo);          // 1 - u
    dd wst = d_div_dd(om, d);                     // omega / (1 - u)
    return dd_mul(wst, dd{INV_2PI_HI, INV_2PI_LO});
}

__device__ __forceinline__ dd half_square_dd(double a) {      // a^2 / 2
    dd s = two_prod(a, a);
    return {0.5 * s.hi, 0.5 * s.lo};
}

// true (cos, sin) of 2 pi p
__device__ __forceinline__ double2 phasor_full(double p) {
    double c, s;
    phasor_turns<RAD_SEP_DEG>(p, c, s);
    return make_double2(c, s * 1.4142135623730951);
}

// spectrum value from true complex amplitudes acc = (Re Ax, Im Ax, Re Ay, Im Ay[, Re J, Im J])
template <int NC>
__device__ __forceinline__ double spectrum_value_true(const double *acc, double nx, double ny,
                                                      int model, double u, double gamma0) {
    const double INV_4PI2 = 0.025330295910584442860969;
    const double azr = -(nx * acc[0] + ny * acc[2]);
    const double azi = -(nx * acc[1] + ny * acc[3]);
    const double S = acc[0] * acc[0] + acc[1] * acc[1] + acc[2] * acc[2] + acc[3] * acc[3]
                   + azr * azr + azi * azi;
    if (!(u < 1.0)) return __longlong_as_double(0x7ff8000000000000LL);
    if (model == RAD_CLASSICAL) return S * INV_4PI2;
    const double e = 1.0 - u;
    if (model == RAD_SPIN0) return e * S * INV_4PI2;
    double J2 = 0.0;
    if (NC == 6) J2 = acc[4] * acc[4] + acc[5] * acc[5];
    return (0.5 * (1.0 + e * e) * S + u * u / (2.0 * gamma0 * gamma0) * J2) * INV_4PI2;
}

// ------------------------------------------------------------------------------ small PTX helpers
__device__ __forceinline__ void mbar_arrive(uint64_t *bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
template <int REGS> __device__ __forceinline__ void reg_alloc() {
    asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;" ::"n"(REGS));
}
template <int REGS> __device__ __forceinline__ void reg_dealloc() {
    asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" ::"n"(REGS));
}
// ---- cluster pair (CL = 2): distributed shared memory and cluster-scope barriers
__device__ __forceinline__ uint32_t cluster_ctarank() {
    uint32_t r;
    asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(r));
    return r;
}
__device__ __forceinline__ uint32_t map_to_cta(uint32_t smem_addr, uint32_t rank) {   // same offset in CTA `rank`
    uint32_t r;
    asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(r) : "r"(smem_addr), "r"(rank));
    return r;
}
// asynchronous 16-byte store into the peer CTA's shared memory; its completion is counted in bytes on the peer's
// mbarrier `bar` (both shared::cluster addresses) -- no fence on either side: the data has landed when the
// barrier's transaction count says so
__device__ __forceinline__ void st_async_v2(uint32_t addr, double2 v, uint32_t bar) {
    asm volatile("st.async.weak.shared::cluster.mbarrier::complete_tx::bytes.v2.f64 [%0], {%1, %2}, [%3];"
                 ::"r"(addr), "d"(v.x), "d"(v.y), "r"(bar) : "memory");
}
// arrive on a barrier of the peer CTA (consumer release of a table buffer: nothing to publish, program order
// keeps the arrive behind the loads whose values the warp has already used)
__device__ __forceinline__ void mbar_arrive_remote(uint32_t addr) {
    asm volatile("mbarrier.arrive.shared::cluster.b64 _, [%0];" ::"r"(addr) : "memory");
}
__device__ __forceinline__ void cluster_sync_all() {
    asm volatile("barrier.cluster.arrive.release.aligned;" ::: "memory");
    asm volatile("barrier.cluster.wait.acquire.aligned;" ::: "memory");
}
template <int NPROD> __device__ __forceinline__ void producer_bar_sync() {   // named barrier 1: the producer threads
    asm volatile("bar.sync 1, %0;" ::"n"(NPROD) : "memory");
}

// The sequence of (trajectory, chunk, sub-block) steps of one CTA.  Producers and consumers each run
// their own copy: both sides derive the same sequence from the launch parameters, so the only thing
// they exchange is table buffers.
struct SepCursor {
    static constexpr int SPC = CH / SEP_S;   // sub-blocks per chunk
    int p, p_end, ts;
    int c, c1;                 // chunk index, end of this trajectory's chunk range
    int sb, nsb;               // sub-block inside the chunk, end of this slice's sub-blocks inside the chunk
    int s_end;                 // end of the slice's sub-block range (index inside the trajectory)
    __device__ __forceinline__ SepCursor(const MainParams &P, int slice) {
        ts = 0;
        if (P.mode == MODE_TSPLIT) { p = slice / P.t_slices; p_end = p + 1; ts = slice % P.t_slices; }
        else { p = (int)((int64_t)slice * P.count / P.p_slices);
               p_end = (int)((int64_t)(slice + 1) * P.count / P.p_slices); }
        sb = 0; nsb = 0; c = 0; c1 = 0; s_end = 0;
        seek(P);
    }
    static __device__ __forceinline__ int64_t n_of(const MainParams &P, int q) {
        return P.n_dev ? P.n_dev[q] : P.n_single;
    }
    // Sub-blocks [s0, s1) of trajectory q that belong to this slice.  A time slice is a range of SUB-BLOCKS (8
    // samples), not of chunks: 24 chunks over 7 slices would give some CTAs 4 chunks and others 3 (the paper's
    // typical grid with N = 3000); 375 sub-blocks over 7 slices differ by one in 54.
    __device__ __forceinline__ void sb_range(const MainParams &P, int q, int &s0, int &s1) const {
        const int nsbt = (int)((n_of(P, q) + SEP_S - 1) / SEP_S);
        if (P.mode == MODE_TSPLIT) { s0 = (int)((int64_t)ts * nsbt / P.t_slices);
                                     s1 = (int)((int64_t)(ts + 1) * nsbt / P.t_slices); }
        else { s0 = 0; s1 = nsbt; }
    }
    __device__ __forceinline__ void set_nsb() { nsb = min(SPC, s_end - c * SPC); }
    __device__ __forceinline__ void seek(const MainParams &P) {   // first trajectory from p on with sub-blocks to do
        while (p < p_end) {
            int s0, s1;
            sb_range(P, p, s0, s1);
            if (s0 < s1) { c = s0 / SPC; c1 = (s1 + SPC - 1) / SPC; sb = s0 % SPC; s_end = s1; set_nsb(); break; }
            ++p;
        }
    }
    __device__ __forceinline__ bool valid() const { return p < p_end; }
    // advance by one sub-block; returns 0 (same chunk), 1 (chunk finished), 2 (trajectory finished)
    __device__ __forceinline__ int step(const MainParams &P) {
        if (++sb < nsb) return 0;
        sb = 0;
        if (++c < c1) { set_nsb(); return 1; }
        ++p;
        seek(P);
        return 2;
    }
};

// ------------------------------------------------------------------------------ main (a0-a7)
// CL = 2: launched as clusters of two CTAs that own neighbouring y tiles of one (omega, x) tile.  Their T tables are
// identical, so each CTA's producers compute HALF of the T entries and store them into both CTAs' table rings: the
// local half with an ordinary store, the peer's with st.async, whose bytes the peer's full[] barrier counts
// (expect_tx posted with the arrival of the peer's first producer warp).  empty[] counts the consumer warps of both
// CTAs, so a producer overwrites a buffer only when both CTAs have read it.  Y, F, H stay private.  Both CTAs step through the same (trajectory, chunk,
// CL = 3 (4 accumulators per point only): the pair owns neighbouring OMEGA tiles of one angle tile instead -- for
// grids with an odd number of y tiles, such as config 4's single 16 x 16 angle tile -- and what it shares is the
// omega-independent integrand table F, by the same mechanism.
// sub-block) sequence, so the protocol is symmetric; a cluster barrier at the start (barriers initialised before the
// peer arrives on them) and at the end (no CTA leaves while the peer may still store into it) frames it.
template <int NC, int WY, int CL>
__global__ void __launch_bounds__(SepRegs<NC>::THREADS, 1)
rad_sep_kernel(const MainParams P) {
    static_assert(CL == 1 || CL == 2 || (CL == 3 && NC == 4), "single CTA, pair sharing T, pair sharing F");
    constexpr bool PAIR = CL >= 2;
    using SH = SepShape<NC, WY>;
    constexpr int YN = SH::YN, EV = SH::EV, S = SEP_S, NB = SEP_NB;
    extern __shared__ __align__(128) unsigned char smem_raw[];
    double *ring = reinterpret_cast<double *>(smem_raw);
    double2 *Tt = reinterpret_cast<double2 *>(smem_raw + SH::OFF_T);      // [NB][S][256]  T = (re, im)
    double2 *Yt = reinterpret_cast<double2 *>(smem_raw + SH::OFF_Y);      // [NB][S][YN]   Y = (re, im)
    double2 *Ft = reinterpret_cast<double2 *>(smem_raw + SH::OFF_F);      // [NB][S][YN]   (w f_x, w f_y)
    double *Hh = reinterpret_cast<double *>(smem_raw + SH::OFF_H);        // [NB][S][YN]   w h (spin-1/2)
    uint64_t *bars = reinterpret_cast<uint64_t *>(smem_raw + SH::OFF_BAR);   // trajectory stages
    uint64_t *full = bars + SEP_STAGES, *empty = full + NB;
    const int tid = threadIdx.x;
    const int slice = blockIdx.y;

    if (tid == 0) {
        for (int s = 0; s < SEP_STAGES; ++s) mbar_init(&bars[s], 1);
        for (int b = 0; b < NB; ++b) { mbar_init(&full[b], SepRegs<NC>::NPROD / 32); mbar_init(&empty[b], (PAIR ? 2 : 1) * SEP_CONS / 32); }
        mbar_fence_init();
    }
    __syncthreads();
    uint32_t peer = 0, my_rank = 0;
    if (PAIR) {
        cluster_sync_all();                           // the peer's barriers are initialised
        my_rank = cluster_ctarank();
        peer = my_rank ^ 1u;
    }

    if (tid >= SEP_CONS) {
        // ====================================================================== PRODUCERS (phase A)
        reg_dealloc<SepRegs<NC>::PROD>();
        const int pt = tid - SEP_CONS;
        const int tile_bx = blockIdx.x;
        const SepCoord<WY> co(tile_bx, 0, P.n_thx, P.n_thy, CL);         // tile bases only
        // Entries per thread and sample.  T: 256 / NPROD.  Y and F: YN / NPROD each, or -- when there are more
        // producer threads than Y entries -- one Y entry for threads [0, YN) and one F entry for the rest
        // (whole warps take one role: YN is a multiple of 32).
        constexpr int NPROD = SepRegs<NC>::NPROD, NE = SepRegs<NC>::NE, HS = SepRegs<NC>::HS;
        const int pe = pt % NE, hs = pt / NE;            // entry slot, sample group
        constexpr bool SPLIT = YN < NE;
        static_assert(256 % NE == 0 && (SPLIT ? 2 * YN == NE : YN % NE == 0), "producer entry assignment");
        constexpr int TS = CL == 2 ? 2 : 1, FS = CL == 3 ? 2 : 1;           // CTAs that share the T / the F entries
        static_assert((256 / NE) % TS == 0 && (SPLIT ? FS == 1 : (YN / NE) % FS == 0),
                      "the shared entries of a thread are dealt out to the CTAs of the pair");
        constexpr int RT = 256 / NE / TS, RY = SPLIT ? 1 : YN / NE, RF = RY / FS;   // shared: entry slots r * 2 + rank
        const bool doY = !SPLIT || pe < YN, doF = !SPLIT || pe >= YN;
        const int ptF = SPLIT ? (pe >= YN ? pe - YN : 0) : pe, ptY = SPLIT ? (pe < YN ? pe : 0) : pe;
        double omT[RT], nxT[RT], omY[RY], nyY[RY], nxF[RF], nyF[RF], hF[RF];
        uint32_t peer_T = 0, peer_full = 0;           // the peer's T (F) ring and full[] barriers (shared::cluster addresses)
        if (PAIR) { peer_T = map_to_cta(smem_u32(CL == 2 ? Tt : Ft), peer); peer_full = map_to_cta(smem_u32(full), peer); }
#pragma unroll
        for (int r = 0; r < RT; ++r) {
            const int b = pe + (r * TS + (CL == 2 ? (int)my_rank : 0)) * NE;
            const int iw = co.bw + 4 * (b >> 6) + 2 * (b & 1) + ((b >> 4) & 1);
            const int ix = co.bx + 8 * ((b >> 5) & 1) + 2 * ((b >> 1) & 3) + ((b >> 3) & 1);
            omT[r] = P.omega[min(iw, P.n_omega - 1)];
            nxT[r] = P.thx[min(ix, P.n_thx - 1)];
        }
#pragma unroll
        for (int r = 0; r < RY; ++r) {
            {
                const int b = ptY + r * NE;
                const int q = b >> 3, m = q % WY, i = (q / WY) & 1, ww = (q / WY) >> 1;
                const int iw = co.bw + 4 * ww + 2 * (b & 1) + i;
                const int iy = co.by + WY * ((b >> 1) & 3) + m;
                omY[r] = P.omega[min(iw, P.n_omega - 1)];
                nyY[r] = P.thy[min(iy, P.n_thy - 1)];
            }
        }
#pragma unroll
        for (int r = 0; r < RF; ++r) {
            {
                const int b = ptF + (r * FS + (CL == 3 ? (int)my_rank : 0)) * NE;
                const int q = b >> 4, m = q % WY, j = (q / WY) & 1, wx = (q / WY) >> 1;
                const int ix = co.bx + 8 * wx + 2 * ((b >> 2) & 3) + j;
                const int iy = co.by + WY * (b & 3) + m;
                nxF[r] = P.thx[min(ix, P.n_thx - 1)];
                nyF[r] = P.thy[min(iy, P.n_thy - 1)];
                hF[r] = 0.5 * (nxF[r] * nxF[r] + nyF[r] * nyF[r]);
            }
        }

        // TMA producer cursor (thread pt == 0 only): its own copy of the step sequence, chunk by chunk
        SepCursor tc(P, slice);
        uint32_t issued = 0;
        auto produce = [&]() {
            if (!tc.valid()) return;
            const int s = issued % SEP_STAGES;
            mbar_expect_tx(&bars[s], CHUNK_BYTES);
            tma_load_1d(ring + (size_t)s * CHUNK_DBL,
                        P.packed + ((int64_t)tc.p * P.cpt + tc.c) * CHUNK_DBL, CHUNK_BYTES, &bars[s]);
            ++issued;
            tc.sb = tc.nsb - 1;                          // jump to the end of the chunk
            tc.step(P);
        };
        if (pt == 0)
            for (int s = 0; s < SEP_STAGES; ++s) produce();

        SepCursor cur(P, slice);
        uint32_t it = 0, g = 0;                          // chunks consumed, sub-blocks produced
        while (cur.valid()) {
            // ---- new chunk: wait for it, exact base phases of this thread's entries (a3)
            const int st = it % SEP_STAGES;
            mbar_wait(&bars[st], (it / SEP_STAGES) & 1);
            const double *ck = ring + (size_t)st * CHUNK_DBL;
            const double lam = P.lam_dev ? P.lam_dev[cur.p] : P.lam_single;
            double p0T[RT], whT[RT], hxT[RT], p0Y[RY], whY[RY], hyY[RY];
            {
                const double2 h01 = *reinterpret_cast<const double2 *>(ck);        // P0_b hi, lo
                const double2 h23 = *reinterpret_cast<const double2 *>(ck + 2);    // t_b, x_b
                const double yb = ck[4];
#pragma unroll
                for (int r = 0; r < RT; ++r) {
                    const dd wt = omega_star_turns(omT[r], lam);
                    const dd hx = half_square_dd(nxT[r]);
                    dd psi = {h01.x, h01.y};
                    psi = dd_add(psi, dd_mul_d(hx, h23.x));
                    psi = dd_add(psi, dd_neg(two_prod(nxT[r], h23.y)));
                    p0T[r] = dd_frac(dd_mul(wt, psi));
                    whT[r] = wt.hi; hxT[r] = hx.hi;
                }
#pragma unroll
                for (int r = 0; r < RY; ++r) {
                    if (!doY) continue;
                    const dd wt = omega_star_turns(omY[r], lam);
                    const dd hy = half_square_dd(nyY[r]);
                    dd psi = dd_mul_d(hy, h23.x);
                    psi = dd_add(psi, dd_neg(two_prod(nyY[r], yb)));
                    p0Y[r] = dd_frac(dd_mul(wt, psi));
                    whY[r] = wt.hi; hyY[r] = hy.hi;
                }
            }
            int adv = 0;
            do {                                         // sub-blocks of this chunk
                const int buf = g % NB;
                mbar_wait(&empty[buf], ((g / NB) & 1) ^ 1);
                const double *rec = ck + HDR + (cur.sb * S + hs * (S / HS)) * REC;
#pragma unroll SepRegs<NC>::PROD_UNROLL
                for (int s0 = 0; s0 < S / HS; ++s0, rec += REC) {
                    const int row = buf * S + hs * (S / HS) + s0;
                    const double2 r67 = *reinterpret_cast<const double2 *>(rec + 6);   // dP0, dt
                    const double2 r89 = *reinterpret_cast<const double2 *>(rec + 8);   // dx, dy
#pragma unroll
                    for (int r = 0; r < RT; ++r) {
                        const double dT = fma(-nxT[r], r89.x, fma(hxT[r], r67.y, r67.x));
                        const double2 ph = phasor_full(fma(whT[r], dT, p0T[r]));
                        const int e = row * 256 + pe + (r * TS + (CL == 2 ? (int)my_rank : 0)) * NE;
                        Tt[e] = ph;
                        if (CL == 2) st_async_v2(peer_T + (uint32_t)e * 16u, ph, peer_full + (uint32_t)buf * 8u);
                    }
#pragma unroll
                    for (int r = 0; r < RY; ++r) {
                        if (!doY) continue;
                        const double dY = fma(-nyY[r], r89.y, hyY[r] * r67.y);
                        const double2 ph = phasor_full(fma(whY[r], dY, p0Y[r]));
                        Yt[row * YN + ptY + r * NE] = ph;
                    }
                    if (!doF) continue;
                    const double2 r01 = *reinterpret_cast<const double2 *>(rec);       // D0, vx
                    const double2 r23 = *reinterpret_cast<const double2 *>(rec + 2);   // vy, w ax
                    const double2 r45 = *reinterpret_cast<const double2 *>(rec + 4);   // w ay, w az
#pragma unroll
                    for (int r = 0; r < RF; ++r) {       // a2: eqs. (3), (4), (6), (12), times the weight
                        const double D = r01.x - hF[r];
                        const double ux = nxF[r] - r01.y, uy = nyF[r] - r23.x;
                        const double bx = fma(nyF[r], uy, D);
                        const double by = fma(nxF[r], ux, D);
                        const double q = fma(nxF[r], ux, bx);
                        const double gq = inv_square(q);
                        const double s1 = fma(nyF[r], r45.x, r45.y);
                        const double s2 = fma(nxF[r], r23.y, r45.y);
                        const int e = row * YN + ptF + (r * FS + (CL == 3 ? (int)my_rank : 0)) * NE;
                        const double2 fv = make_double2(fma(s1, ux, -(bx * r23.y)) * gq, fma(s2, uy, -(by * r45.x)) * gq);
                        Ft[e] = fv;
                        if (CL == 3) st_async_v2(peer_T + (uint32_t)e * 16u, fv, peer_full + (uint32_t)buf * 8u);
                        if (NC == 6) Hh[e] = fma(nxF[r], r23.y, s1) * gq;
                    }
                }
                __syncwarp();
                if ((pt & 31) == 0) {
                    // the peer's half of the shared table arrives asynchronously: S samples x 128 entries x 16 bytes
                    if (PAIR && pt == 0) mbar_expect_tx(&full[buf], S * ((CL == 2 ? 256 : YN) / 2) * 16);
                    else mbar_arrive(&full[buf]);
                }
                ++g;
                adv = cur.step(P);
            } while (adv == 0);
            // ---- chunk finished by every producer: its ring stage can be refilled
            ++it;
            producer_bar_sync<NPROD>();
            if (pt == 0) produce();
        }
        if (PAIR) cluster_sync_all();                 // (matches the consumers' barrier at the end of the kernel)
        return;
    }

    // ========================================================================== CONSUMERS (phase B)
    reg_alloc<SepRegs<NC>::CONS>();
    const SepCoord<WY> co(blockIdx.x, tid, P.n_thx, P.n_thy, CL);
    uint32_t peer_empty = 0;
    if (PAIR) peer_empty = map_to_cta(smem_u32(empty), peer);
    const int64_t gid = (int64_t)blockIdx.x * SEP_CONS + tid;
    // read offsets (entries) of this thread inside one sample's tables
    const int rT = (co.ww * 2 + co.wx) * 32 + co.lx * 2 + co.lw;          // + (i*2 + j) * 8
    const int rY = co.ww * 2 * WY * 8 + co.ly * 2 + co.lw;                // + (i*WY + m) * 8
    const int rF = co.wx * 2 * WY * 16 + co.lx * 4 + co.ly;               // + (j*WY + m) * 16

    // ---- output slots of this thread: zero them, later every trajectory adds its spectrum
    auto out_slot = [&](int e) -> double * {          // nullptr: point outside the grid
        const int m = e % WY, j = (e / WY) & 1, i = e / (2 * WY);
        const int iw = co.iw0 + i, ix = co.ix0 + j, iy = co.iy0 + m;
        if (P.mode == MODE_PSLICE) return P.partial + ((int64_t)slice * EV + e) * P.t_pad + gid;
        if (iw >= P.n_omega || ix >= P.n_thx || iy >= P.n_thy) return nullptr;
        return P.out + iw * P.out_plane + (int64_t)iy * P.out_nx + ix;
    };
    const bool ang = P.mode == MODE_DIRECT && P.ang;
    double sw[2] = {0.0, 0.0};                        // angular spectrum: this thread's angles summed, per omega (N1)
    if (P.mode != MODE_TSPLIT && !(P.mode == MODE_DIRECT && P.accumulate) && !ang) {
#pragma unroll 1
        for (int e = 0; e < EV; ++e) {
            double *o = out_slot(e);
            if (o) *o = 0.0;
        }
    }

    double acc[EV][NC];
#pragma unroll
    for (int e = 0; e < EV; ++e)
#pragma unroll
        for (int c = 0; c < NC; ++c) acc[e][c] = 0.0;

    // The consumers only need to know how many sub-blocks each trajectory of their slice has.
    SepCursor cur(P, slice);
    if (P.mode == MODE_TSPLIT && !cur.valid()) {      // empty time slice: its partial amplitudes are zero
        double *dst = P.partial + (int64_t)slice * NC * EV * P.t_pad + gid;
        for (int k = 0; k < NC * EV; ++k) dst[(int64_t)k * P.t_pad] = 0.0;
    }
    int p_now = cur.p;
    const int p_end = cur.p_end;
    auto sub_blocks_of = [&](int p) -> int {          // sub-blocks of trajectory p inside this slice
        int s0, s1;
        cur.sb_range(P, p, s0, s1);
        return s1 - s0;
    };
    int todo = p_now < p_end ? sub_blocks_of(p_now) : 0;
    uint32_t g = 0;
    while (p_now < p_end) {
        const int buf = g % NB;
        mbar_wait(&full[buf], (g / NB) & 1);
#ifndef RAD_SEP_CU
#define RAD_SEP_CU 8
#endif
        constexpr int CU = RAD_SEP_CU;
#pragma unroll CU
        for (int s = 0; s < S; ++s) {                 // a4: complex multiply + accumulate
            const int row = buf * S + s;
            const double2 *tp = Tt + row * 256 + rT, *yp = Yt + row * YN + rY, *fp = Ft + row * YN + rF;
            const double *hp = Hh + row * YN + rF;
            double2 tv[2][2];
#pragma unroll
            for (int i = 0; i < 2; ++i)
#pragma unroll
                for (int j = 0; j < 2; ++j) tv[i][j] = tp[(i * 2 + j) * 8];
            // Groups g = (m, j): the two points (i = 0, 1) that share the integrand entry F[j][m].  The complex
            // products q = T Y of group g + 1 are formed while group g is accumulated, so that every operand
            // of the accumulation is old and the DFMAs can run in f-major order: runs that share one
            // multiplicand in the same operand slot (register-file bandwidth: DESIGN.md 5.4 (iii)).
            constexpr int G = 2 * WY;
            double qr[2], qi[2];
            auto products = [&](int g, double (&pr)[2], double (&pi)[2]) {
                const int m = g >> 1, j = g & 1;
#pragma unroll
                for (int i = 0; i < 2; ++i) {
                    const double2 y = yp[(i * WY + m) * 8];
                    pr[i] = tv[i][j].x * y.x;
                    pi[i] = tv[i][j].x * y.y;
                    pr[i] = fma(-tv[i][j].y, y.y, pr[i]);
                    pi[i] = fma(tv[i][j].y, y.x, pi[i]);
                }
            };
            // (The 64 accumulators of the 4-per-point variant leave ptxas so few registers that it renames
            // accumulators and moves them back: 106-194 IMAD.MOV per 1007 FP64 instructions of the loop, depending on
            // unrelated code around it; staged or not changes the throughput by +-1 %.)
#ifndef RAD_SEP_STAGED4
#define RAD_SEP_STAGED4 true
#endif
            constexpr bool STAGED = NC == 6 || RAD_SEP_STAGED4;
            if (STAGED) products(0, qr, qi);
#pragma unroll
            for (int g = 0; g < G; ++g) {
                const int m = g >> 1, j = g & 1;
                double nr[2], ni[2];
                if (!STAGED) products(g, qr, qi);
                else if (g + 1 < G) products(g + 1, nr, ni);
                const double2 f = fp[(j * WY + m) * 16];
                double *a0 = acc[(0 * 2 + j) * WY + m], *a1 = acc[(1 * 2 + j) * WY + m];
                a0[0] = fma(f.x, qr[0], a0[0]);
                a0[1] = fma(f.x, qi[0], a0[1]);
                a1[0] = fma(f.x, qr[1], a1[0]);
                a1[1] = fma(f.x, qi[1], a1[1]);
                a1[3] = fma(f.y, qi[1], a1[3]);
                a1[2] = fma(f.y, qr[1], a1[2]);
                a0[3] = fma(f.y, qi[0], a0[3]);
                a0[2] = fma(f.y, qr[0], a0[2]);
                if (NC == 6) {
                    const double hv = hp[(j * WY + m) * 16];
                    a0[4] = fma(hv, qr[0], a0[4]);
                    a0[5] = fma(hv, qi[0], a0[5]);
                    a1[4] = fma(hv, qr[1], a1[4]);
                    a1[5] = fma(hv, qi[1], a1[5]);
                }
                if (STAGED && g + 1 < G) {
#pragma unroll
                    for (int i = 0; i < 2; ++i) { qr[i] = nr[i]; qi[i] = ni[i]; }
                }
            }
        }
        __syncwarp();
        if ((tid & 31) == 0) {
            mbar_arrive(&empty[buf]);
            if (PAIR) mbar_arrive_remote(peer_empty + (uint32_t)buf * 8u);
        }
        ++g;
        if (--todo == 0) {
            // ================================================================ end of trajectory p_now (a5, a7)
            if (P.mode == MODE_TSPLIT) {
                double *dst = P.partial + (int64_t)slice * NC * EV * P.t_pad + gid;
#pragma unroll
                for (int e = 0; e < EV; ++e)
#pragma unroll
                    for (int c = 0; c < NC; ++c) dst[(int64_t)(c * EV + e) * P.t_pad] = acc[e][c];
            } else {
                const double lam = P.lam_dev ? P.lam_dev[p_now] : P.lam_single;
                const double gamma0 = P.packed[(int64_t)p_now * P.cpt * CHUNK_DBL + 5];
#pragma unroll
                for (int e = 0; e < EV; ++e) {
                    const int m = e % WY, j = (e / WY) & 1, i = e / (2 * WY);
                    const double om = P.omega[min(co.iw0 + i, P.n_omega - 1)];
                    const double nx = P.thx[min(co.ix0 + j, P.n_thx - 1)];
                    const double ny = P.thy[min(co.iy0 + m, P.n_thy - 1)];
                    const double v = spectrum_value_true<NC>(acc[e], nx, ny, P.model, om * lam, gamma0);
                    if (ang) {
                        const bool inside = co.iw0 + i < P.n_omega && co.ix0 + j < P.n_thx && co.iy0 + m < P.n_thy
                                            && (P.cut2 <= 0.0 || fma(nx, nx, ny * ny) <= P.cut2);
                        if (inside) sw[i] += v;
                    } else {
                        double *o = out_slot(e);
                        if (o) *o += v;
                    }
                }
            }
#pragma unroll
            for (int e = 0; e < EV; ++e)
#pragma unroll
                for (int c = 0; c < NC; ++c) acc[e][c] = 0.0;
            do {                                      // next trajectory of the slice that has work
                ++p_now;
                todo = p_now < p_end ? sub_blocks_of(p_now) : 0;
            } while (p_now < p_end && todo == 0);
        }
    }
    if (ang) {
        // ---- sum over the tile's angles per omega, fixed order: 16 omega slots (slot = i_w - bw = 4 ww + 2 lw + i),
        // each fed by the 32 consumer threads (2 warps x 16 lanes) that own that omega.  The trajectory ring is
        // free by now: every chunk was consumed before the last table block was handed over.
        asm volatile("bar.sync 2, 256;" ::: "memory");
        double *red = ring;                           // [256][2]
        red[tid * 2] = sw[0]; red[tid * 2 + 1] = sw[1];
        asm volatile("bar.sync 2, 256;" ::: "memory");
        if (tid < 16) {
            const int ww = tid >> 2, lw = (tid >> 1) & 1, i = tid & 1;
            double sum = 0.0;
            for (int wx = 0; wx < 2; ++wx)
                for (int l = 0; l < 16; ++l) sum += red[(((ww * 2 + wx) * 32) + l * 2 + lw) * 2 + i];
            P.ang_partial[(int64_t)blockIdx.x * 16 + tid] = sum;
        }
    }
    if (PAIR) cluster_sync_all();                     // the peer may still store table entries / arrive here until it is done
}

// angular spectrum, second pass for the separable kernel: spec[i_w] (+)= d_solid * sum over the angle tiles of
// omega tile i_w / 16 (contiguous block indices), ascending; one CTA per omega, fixed two-level order.
__global__ void __launch_bounds__(256)
rad_ang_final_sep_kernel(const double *partial, int angle_tiles, int n_omega, double d_solid, int accumulate,
                         double *spec) {
    __shared__ double red[256];
    const int iw = blockIdx.x, wt = iw / 16, slot = iw % 16;
    const int per = (angle_tiles + 255) / 256;
    double s = 0.0;
    for (int t = threadIdx.x * per; t < min(angle_tiles, (threadIdx.x + 1) * per); ++t)
        s += partial[((int64_t)wt * angle_tiles + t) * 16 + slot];
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
template <int NC, int WY>
__global__ void __launch_bounds__(SEP_CONS)
rad_sep_finalize_kernel(const MainParams P) {
    constexpr int EV = 4 * WY;
    const SepCoord<WY> co(blockIdx.x, threadIdx.x, P.n_thx, P.n_thy, P.cl);
    const int64_t gid = (int64_t)blockIdx.x * SEP_CONS + threadIdx.x;
    {                                                 // gridDim.y = EV: one of the thread's points per CTA row
        const int e = blockIdx.y;
        const int m = e % WY, j = (e / WY) & 1, i = e / (2 * WY);
        const int iw = co.iw0 + i, ix = co.ix0 + j, iy = co.iy0 + m;
        if (iw >= P.n_omega || ix >= P.n_thx || iy >= P.n_thy) return;
        double total = 0.0;
        if (P.mode == MODE_PSLICE) {
            for (int s = 0; s < P.p_slices; ++s)                       // slices ascending
                total += P.partial[((int64_t)s * EV + e) * P.t_pad + gid];
        } else {
            const double om = P.omega[iw], nx = P.thx[ix], ny = P.thy[iy];
            for (int p = 0; p < P.count; ++p) {                        // trajectories ascending
                double acc[NC];
#pragma unroll
                for (int c = 0; c < NC; ++c) acc[c] = 0.0;
                for (int s = 0; s < P.t_slices; ++s) {                 // time slices ascending
                    const double *src = P.partial + (int64_t)(p * P.t_slices + s) * NC * EV * P.t_pad + gid;
#pragma unroll
                    for (int c = 0; c < NC; ++c) acc[c] += src[(int64_t)(c * EV + e) * P.t_pad];
                }
                const double lam = P.lam_dev ? P.lam_dev[p] : P.lam_single;
                const double gamma0 = P.packed[(int64_t)p * P.cpt * CHUNK_DBL + 5];
                total += spectrum_value_true<NC>(acc, nx, ny, P.model, om * lam, gamma0);
            }
        }
        double *o = P.out + iw * P.out_plane + (int64_t)iy * P.out_nx + ix;
        *o = P.accumulate ? *o + total : total;
    }
}

}  // namespace rad
