// Lennard-Jones pair force, energy and virial over the neighbor list
// (PAPER.md:95, 103, 105, 284, 314-320), optionally with the velocity-Verlet
// half-steps and the r_buff/2 check fused in.
//
//   V_lj = 4 eps [(sigma/r)^12 - (sigma/r)^6],  f = -(1/r) dV/dr * d,  r < r_cut,ab
// with per-type-pair tables held as lj1 = 4 eps sigma^12, lj2 = 4 eps sigma^6:
//   -(1/r) dV/dr = r^-8 (12 lj1 r^-6 - 6 lj2),   V = r^-6 (lj1 r^-6 - lj2) - eshift.
// The pair functor idea of PAPER.md:284 (V(r) and -(1/r) dV/dr) is kept as the
// inlined pair_term() below.
//
// Design (round 2; the ncu numbers that led here are in profiles/r1c_* and r2_*).
// ONE BLOCK OWNS ONE TILE of cells (tile.cuh):
//   * the tile and its one-cell halo are staged once in shared memory, shifted to the
//     periodic image the tile sees: no minimum-image arithmetic per pair, and every
//     neighbor gather is ONE 16-byte shared-memory load.  The particle data is kept in
//     cell order, so a row of x-adjacent halo cells is one contiguous range of the
//     position array ("piece", two where the row wraps around the box): the block
//     reads cell_start at the ends of its (ty+2)(tz+2) halo rows, prefix-sums the
//     lengths (that IS the slot numbering the list build used) and copies each piece
//     with one cp.async.bulk (TMA bulk copy, completion on an mbarrier) straight into the staging area.  No per-tile
//     table is read (round 1 read a 4-byte source index per staged slot per step).
//     Only tiles whose halo touches a face of the box fix the periodic image, in place;
//   * list entries are 16-bit BYTE OFFSETS into the staging area (slot * 16 when the
//     staging area has at most 4096 slots), so an entry becomes the address of its
//     gather with one instruction;
//   * TPP threads share one particle; each takes EPL consecutive entries per iteration.
//     The rows arrive through a ring of cp.async copies per thread; a row ends at its
//     first padding entry (slot 0 = a dummy particle far away), so no row length is read.
//     The EPL gathers are issued back to back; a pair outside r_cut gets r^-2 := 0 by a
//     select, not by a branch;
//   * an inner step of hb_run_nve needs F only (nobody can read its U_i, W_i): the
//     THERMO = false variant has 3 accumulators and no force store at all;
//   * F (and U, W) are combined across the TPP lanes with warp shuffles and parked in
//     shared memory; after a block barrier thread t finishes the velocity-Verlet step
//     of particle t of the pass (second half kick of this step, first half kick and
//     drift of the next, wrap, image flags, r_buff/2 check) with v, x and x_build that
//     were prefetched into shared memory by cp.async while the pairs were evaluated,
//     and writes the new position into the OTHER position buffer, since the blocks
//     around still read the old one.  One kernel per time step.
#include "tile.cuh"
#include "integrate_dev.cuh"

__device__ __forceinline__ float rcp_approx(float x)
{
    float y;
    asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}

// cp.async (LDGSTS): global -> shared without a register or a scoreboard slot in between.
// List rows go through L1 (.ca): a row is read 16 or 8 bytes at a time, its 128-byte lines are fetched once.
template <int BYTES>
__device__ __forceinline__ void cp_async(void *smem_dst, const void *gsrc)
{
    const unsigned d = (unsigned)__cvta_generic_to_shared(smem_dst);
    asm volatile("cp.async.ca.shared.global [%0], [%1], %2;" ::"r"(d), "l"(gsrc), "n"(BYTES) : "memory");
}
// Particle data is read once per block: past L1 (.cg, 16 bytes).
__device__ __forceinline__ void cp_async_cg16(void *smem_dst, const void *gsrc)
{
    const unsigned d = (unsigned)__cvta_generic_to_shared(smem_dst);
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(d), "l"(gsrc) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N>
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }

// Depth of the per-thread ring of list copies (cp.async): how many iterations ahead a thread asks for its list entries.
// Measured on B200 (us per time step, N = 64,000 / 10^6 / Kob-Andersen 2^20): depth 4: 27.4 / 237.7 / 400; 2: 27.1 / 229.2 /
// 380; 1: 27.3 / 227.1 / 368.  The kernel is bound by the shared-memory pipe, and every copy of a warp costs 16 wavefronts
// (its 32 lanes read 16 different rows): the copies issued past the end of a row are pure cost, and a shallower ring
// leaves more shared memory for resident blocks.
constexpr int LIST_PF = 2;

struct Acc {
    float fx, fy, fz, u, wxx, wxy, wxz, wyy, wyz, wzz;
};

// One listed pair.  pj is already the nearest image.  The force sums are the same operations in both variants
// (fma(f/r, d, F)), so the trajectory does not depend on whether the energy and virial terms are compiled in.
// FN selects the functor (V(r) and -(1/r) dV/dr):
//   FN_LJ     Lennard-Jones, truncated or energy-shifted
//   FN_XPLOR  Lennard-Jones with XPLOR smoothing: V = V_lj S(r),
//             -(1/r) dV/dr = [-(1/r) dV_lj/dr] S - V_lj S'/r with
//             S = (rc^2 - r^2)^2 (rc^2 + 2 r^2 - 3 ron^2) / (rc^2 - ron^2)^3,  S'/r = 12 (rc^2 - r^2)(ron^2 - r^2) / (rc^2 - ron^2)^3
//             between r_on and r_cut, S = 1 below r_on
//   FN_GEN    Gaussian, Yukawa or Morse (reading f1; `pot` is uniform over the launch) with any of the three cutoff
//             treatments: eshift = V(r_cut) or 0, smoothing where invD != 0.
enum { FN_LJ = 0, FN_XPLOR = 1, FN_GEN = 2 };

template <bool THERMO, int FN>
__device__ __forceinline__ void pair_term(const float4 &pi, const float4 &pj, const float lj1x12, const float lj2x6,
                                          const PairParam &pp, const PairParamX &px, const int pot, Acc &a)
{
    const float dx = pi.x - pj.x, dy = pi.y - pj.y, dz = pi.z - pj.z;
    const float r2 = __fmaf_rn(dz, dz, __fmaf_rn(dy, dy, dx * dx));
    const bool in = r2 < pp.rcut2;                     // strict <
    float fdivr, v = 0.f;
    if (FN == FN_GEN) {
        const float r2s = in ? r2 : pp.rcut2;          // the dummy slot is 1e18 away: keep every intermediate finite
        float f;
        if (pot == HB_POT_GAUSS) {
            v = pp.lj1 * expf(-r2s * pp.lj2);
            f = v * (2.0f * pp.lj2);
        } else if (pot == HB_POT_YUKAWA) {
            const float r = sqrtf(r2s), ri = 1.0f / r;
            v = pp.lj1 * expf(-pp.lj2 * r) * ri;
            f = v * (pp.lj2 + ri) * ri;
        } else {
            const float r = sqrtf(r2s);
            const float e1 = expf(-pp.lj2 * (r - px.p2));
            v = pp.lj1 * (e1 * e1 - 2.0f * e1);
            f = 2.0f * pp.lj2 * pp.lj1 * (e1 * e1 - e1) / r;
        }
        if (px.invD != 0.0f && r2s > px.ron2) {
            const float d = pp.rcut2 - r2s;
            const float S = d * d * __fmaf_rn(2.0f, r2s, __fmaf_rn(-3.0f, px.ron2, pp.rcut2)) * px.invD;
            const float dS = 12.0f * d * (px.ron2 - r2s) * px.invD;
            f = __fmaf_rn(f, S, -v * dS);
            v *= S;
        }
        fdivr = in ? f : 0.0f;
        v = in ? v - pp.eshift : 0.0f;
    } else {
        const float r2inv = in ? rcp_approx(r2) : 0.0f;    // 0 switches the whole pair off: no branch (a branch per pair
        const float r4inv = r2inv * r2inv;                 // would serialise the EPL pairs of an iteration)
        const float r6inv = r4inv * r2inv;
        fdivr = (r4inv * r4inv) * __fmaf_rn(lj1x12, r6inv, -lj2x6);
        if (THERMO || FN == FN_XPLOR) v = r6inv * __fmaf_rn(pp.lj1, r6inv, -pp.lj2);
        if (FN == FN_XPLOR) {
            const float r2c = fminf(r2, pp.rcut2);         // the dummy slot is 1e18 away: keep (rc^2 - r^2)^2 finite
            const float d = pp.rcut2 - r2c;
            const bool sw = r2c > px.ron2;
            const float S = sw ? d * d * __fmaf_rn(2.0f, r2c, __fmaf_rn(-3.0f, px.ron2, pp.rcut2)) * px.invD : 1.0f;
            const float dS = sw ? 12.0f * d * (px.ron2 - r2c) * px.invD : 0.0f;
            fdivr = __fmaf_rn(fdivr, S, -v * dS);
            v *= S;
        }
        if (THERMO) v -= in ? pp.eshift : 0.0f;
    }
    a.fx = __fmaf_rn(fdivr, dx, a.fx);
    a.fy = __fmaf_rn(fdivr, dy, a.fy);
    a.fz = __fmaf_rn(fdivr, dz, a.fz);
    if (THERMO) {
        a.u += v;
        const float px_ = fdivr * dx, py_ = fdivr * dy, pz_ = fdivr * dz;
        a.wxx = __fmaf_rn(dx, px_, a.wxx); a.wxy = __fmaf_rn(dx, py_, a.wxy); a.wxz = __fmaf_rn(dx, pz_, a.wxz);
        a.wyy = __fmaf_rn(dy, py_, a.wyy); a.wyz = __fmaf_rn(dy, pz_, a.wyz); a.wzz = __fmaf_rn(dz, pz_, a.wzz);
    }
}

template <int EPL> struct Entries;
template <> struct Entries<4> { uint2 v; };
template <> struct Entries<8> { uint4 v; };

// byte offsets of the EPL gathers of one iteration
template <int EPL, bool SCALED>
__device__ __forceinline__ void unpack_entries(const Entries<EPL> &e, unsigned (&off)[EPL])
{
    const unsigned w[4] = {e.v.x, e.v.y, EPL == 8 ? ((const unsigned *)&e.v)[2] : 0u, EPL == 8 ? ((const unsigned *)&e.v)[3] : 0u};
#pragma unroll
    for (int k = 0; k < EPL / 2; k++) {
        if (SCALED) { off[2 * k] = w[k] & 0xffffu; off[2 * k + 1] = w[k] >> 16; }
        else { off[2 * k] = (w[k] & 0xffffu) << 4; off[2 * k + 1] = (w[k] >> 16) << 4; }
    }
}

struct ForceArgs {
    TileGeom g;
    const int *cell_start;
    const float4 *pos;
    const uint16_t *nlist;
    int pitch, N, ntypes, pot;
    const PairParam *params;
    const PairParamX *paramsx;
    float4 *force, *virial;
    int *flags;
    int do_nve;
    NveArgs nv;
};

// What the block knows about its tile (shared memory).
struct ForceTile {
    TileDesc d;                          // own rows, counts, centre
    int piece_src[2 * TILE_PROWS_MAX];   // storage index of the first particle of piece p
    int piece_slot[2 * TILE_PROWS_MAX + 1];   // its first slot; [npieces] = nslots
    int npieces, fix;
    alignas(8) uint64_t mbar;            // completion of the staging copies
};

// Fast geometry (tile + halo narrower than L/2): halo rows as contiguous pieces of the cell-ordered position array.
__device__ __forceinline__ bool force_tile_tables(const TileGeom &g, const int *__restrict__ cell_start, ForceTile &s)
{
    TileCtx t;
    tile_decode_xyz(g, blockIdx.x, blockIdx.y, blockIdx.z, t);
    const int tid = threadIdx.x, lane = tid & 31;
    const int hrows = t.hy * t.hz;
    const int m = g.m;
    // one thread per halo row: lengths of its (at most two) pieces
    for (int r = tid; r < hrows; r += blockDim.x) {
        const int jy = r % t.hy, jz = r / t.hy;
        int cy = t.y0 - 1 + jy, cz = t.z0 - 1 + jz;
        cy += cy < 0 ? m : (cy >= m ? -m : 0);
        cz += cz < 0 ? m : (cz >= m ? -m : 0);
        const int rowbase = m * (cy + m * cz);
        const int X0 = t.x0 - 1, X1 = t.x0 + t.ex;          // tile frame, inclusive
        int a0, a1, b0 = 0, b1 = -1;                         // piece A = cells a0..a1, piece B = cells b0..b1 (box frame)
        if (X0 < 0) { a0 = a1 = m - 1; b0 = 0; b1 = X1; }
        else if (X1 >= m) { a0 = X0; a1 = m - 1; b0 = b1 = 0; }
        else { a0 = X0; a1 = X1; }
        const int sa = __ldg(&cell_start[rowbase + a0]), ea = __ldg(&cell_start[rowbase + a1 + 1]);
        int sb = 0, eb = 0;
        if (b1 >= b0) { sb = __ldg(&cell_start[rowbase + b0]); eb = __ldg(&cell_start[rowbase + b1 + 1]); }
        s.piece_src[2 * r] = sa; s.piece_src[2 * r + 1] = sb;
        s.piece_slot[2 * r] = ea - sa; s.piece_slot[2 * r + 1] = eb - sb;
        // own rows: interior rows of the halo box
        const int ly = jy - 1, lz = jz - 1;
        if (ly >= 0 && ly < t.ey && lz >= 0 && lz < t.ez) {
            const int orow = ly + t.ey * lz;
            const int os = __ldg(&cell_start[rowbase + t.x0]), oe = __ldg(&cell_start[rowbase + t.x0 + t.ex - 1 + 1]);
            s.d.own_start[orow] = os;
            s.d.own_off[orow + 1] = oe - os;
            // slot of the first own particle, relative to the row's first slot: the cell left of x0 comes first
            s.d.own_slot[orow] = X0 < 0 ? (ea - sa) : (os - sa);
        }
    }
    __syncthreads();
    const int np = 2 * hrows;
    if (tid < 32) {   // exclusive scan of up to 2 * TILE_PROWS_MAX lengths: 6 per lane
        constexpr int PER = (2 * TILE_PROWS_MAX + 31) / 32;
        const int base = lane * PER;
        int v[PER], tsum = 0;
#pragma unroll
        for (int q = 0; q < PER; q++) { v[q] = base + q < np ? s.piece_slot[base + q] : 0; tsum += v[q]; }
        int incl = tsum;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) { const int y = __shfl_up_sync(0xffffffffu, incl, o); if (lane >= o) incl += y; }
        int run = 1 + incl - tsum;   // slot 0 is the dummy
#pragma unroll
        for (int q = 0; q < PER; q++) { if (base + q < np) s.piece_slot[base + q] = run; run += v[q]; }
        if (lane == 31) s.piece_slot[np] = run;
    }
    __syncthreads();
    if (tid < t.ey * t.ez) {
        const int ly = tid % t.ey, lz = tid / t.ey;
        s.d.own_slot[tid] += s.piece_slot[2 * ((lz + 1) * t.hy + (ly + 1))];
    }
    if (tid == 0) {
        int run = 0;
        const int nrows = t.ey * t.ez;
        s.d.own_off[0] = 0;
        for (int r = 0; r < nrows; r++) { const int n = s.d.own_off[r + 1]; s.d.own_off[r + 1] = run + n; run += n; }
        const float wcell = g.L / (float)m, hL = 0.5f * g.L;
        s.d.nslots = s.piece_slot[np];
        s.d.nown = run;
        s.d.nrows = nrows;
        s.d.cx = __fmaf_rn((float)t.x0 + 0.5f * (float)t.ex, wcell, -hL);
        s.d.cy = __fmaf_rn((float)t.y0 + 0.5f * (float)t.ey, wcell, -hL);
        s.d.cz = __fmaf_rn((float)t.z0 + 0.5f * (float)t.ez, wcell, -hL);
        s.npieces = np;
        // a staged particle can sit on the other side of the box only if the halo reaches the first or last cell of
        // an axis (a wrapped halo cell, or a particle that drifted through the face after the build)
        s.fix = (t.x0 <= 1 || t.x0 + t.ex >= m - 1 || t.y0 <= 1 || t.y0 + t.ey >= m - 1 || t.z0 <= 1 || t.z0 + t.ez >= m - 1) ? 1 : 0;
    }
    __syncthreads();
    return s.d.nslots <= g.cap;
}

template <int TPP, int EPL, bool ONE_TYPE, bool THERMO, bool SCALED, int FN>
__global__ void __launch_bounds__(TILE_THREADS, 4)   // <= 64 registers: 8 blocks of 128 threads per SM
lj_tile_kernel(const ForceArgs A)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    __shared__ ForceTile s;
    const TileGeom &g = A.g;
    const int nthreads = blockDim.x;
    const int PPB = nthreads / TPP;              // particles per block per pass
    constexpr int G = TPP * EPL;                 // entries per particle per iteration
    constexpr int PF = LIST_PF;                  // depth of the ring of list copies
    using EntryVec = decltype(Entries<EPL>::v);

    // dynamic shared memory: staging area | pair table | ring | own data of a pass (v, x, x_build; one buffer: a
    // thread group reads its particle's data into registers before it starts the copies of the next pass)
    unsigned char *sp = smem_raw;
    float4 *stage = reinterpret_cast<float4 *>(sp);                      sp += (size_t)g.cap * 16;
    PairParam *s_params = reinterpret_cast<PairParam *>(sp);             sp += ONE_TYPE ? 0 : ((A.ntypes * A.ntypes * sizeof(PairParam) + 15) & ~(size_t)15);
    PairParamX *s_paramsx = reinterpret_cast<PairParamX *>(sp);          sp += (ONE_TYPE || FN == FN_LJ) ? 0 : ((A.ntypes * A.ntypes * sizeof(PairParamX) + 15) & ~(size_t)15);
    EntryVec *ring = reinterpret_cast<EntryVec *>(sp) + threadIdx.x;     sp += (size_t)PF * sizeof(EntryVec) * nthreads;
    float4 *own = reinterpret_cast<float4 *>(sp);                        sp += (size_t)3 * PPB * 16;       // [v | x | x_build][PPB]
    TileShared &sgen = *reinterpret_cast<TileShared *>(sp);              // the general (small-box) geometry only
    const int ring_stride = nthreads;
    const NveArgs &nv = A.nv;
    const bool nve = A.do_nve != 0, drift = nve && nv.kick_drift;
    const bool block0 = (blockIdx.x | blockIdx.y | blockIdx.z) == 0;

    if (threadIdx.x == 0 && g.fast) mbar_init(&s.mbar, 1);
    if (!ONE_TYPE)
        for (int k = threadIdx.x; k < A.ntypes * A.ntypes; k += nthreads) {
            s_params[k] = A.params[k];
            if (FN != FN_LJ) s_paramsx[k] = A.paramsx[k];
        }
    if (drift && block0 && threadIdx.x == 0) A.flags[nv.need_clear] = 0;

    // ---- the tile: tables, staging ----
    bool fits;
    if (g.fast) {
        fits = force_tile_tables(g, A.cell_start, s);
        if (fits && threadIdx.x < 32) {
            // warp 0 hands the pieces to the TMA unit: one bulk copy per contiguous run of positions
            const int lane = threadIdx.x;
            if (lane == 0) {
                stage[0] = make_float4(1e18f, 1e18f, 1e18f, 0.f);
                mbar_expect_tx(&s.mbar, (unsigned)(s.d.nslots - 1) * 16u);
            }
            __syncwarp();
            for (int p = lane; p < s.npieces; p += 32) {
                const int s0 = s.piece_slot[p], len = s.piece_slot[p + 1] - s0;
                if (len > 0) bulk_g2s(stage + s0, A.pos + s.piece_src[p], (unsigned)len * 16u, &s.mbar);
            }
        }
    } else {
        TileCtx t;
        tile_decode_xyz(g, blockIdx.x, blockIdx.y, blockIdx.z, t);
        fits = tile_tables(g, A.cell_start, t, sgen, A.flags);
        if (threadIdx.x < sizeof(TileDesc) / 4) reinterpret_cast<int *>(&s.d)[threadIdx.x] = reinterpret_cast<const int *>(&sgen.d)[threadIdx.x];
        __syncthreads();
        if (fits) tile_stage_positions(g, t, sgen, A.pos, stage, nullptr);
    }
    const int nown = fits ? s.d.nown : 0;

    const int sub = threadIdx.x % TPP;
    const int ql = threadIdx.x / TPP;            // particle of the pass this thread group works for
    int gi_n = 0, slot_n = 0;
    bool active_n = false;
    // start of a pass: the particle of this thread group, the first PF copies of its row, and (lanes 0 and 1 of the
    // group) what the integration of the particle will need
    auto prep = [&](int q0) {
        const int q = q0 + ql;
        active_n = q < nown;
        gi_n = 0; slot_n = 0;
        if (active_n) tile_own(s.d, q, gi_n, slot_n);
        const uint16_t *row = A.nlist + (int64_t)gi_n * A.pitch + sub * EPL;
        if (nve && active_n) {
            float4 *o = own + ql;
            if (sub == 0) { cp_async_cg16(o, nv.vel + gi_n); if (nv.kick_drift) cp_async_cg16(o + PPB, A.pos + gi_n); }
            if (sub == 1 && nv.kick_drift) cp_async_cg16(o + 2 * PPB, nv.pos_build + gi_n);
        }
#pragma unroll
        for (int u = 0; u < PF; u++) {
            if (active_n) cp_async<EPL * 2>(ring + u * ring_stride, row + u * G);
            cp_async_commit();
        }
    };

    prep(0);                                     // list and integration data in flight behind the staging copies
    if (g.fast && fits) {
        mbar_wait(&s.mbar, 0);
        if (s.fix) {
            // the halo reaches a face of the box: move every staged particle to the image nearest to the tile centre.
            // Each thread fixes what it will not read before the barrier below.
            const float L = g.L, hL = 0.5f * g.L, cx = s.d.cx, cy = s.d.cy, cz = s.d.cz;
            for (int sl = 1 + threadIdx.x; sl < s.d.nslots; sl += nthreads) {
                float4 p = stage[sl];
                p.x = tile_image(p.x, cx, L, hL); p.y = tile_image(p.y, cy, L, hL); p.z = tile_image(p.z, cz, L, hL);
                stage[sl] = p;
            }
            __syncthreads();
        }
    } else {
        __syncthreads();
    }

    const PairParam pp1 = A.params[0];
    PairParamX px1 = {0.f, 0.f, 0.f, 0.f};
    if (FN != FN_LJ) px1 = A.paramsx[0];
    const float c12 = 12.0f * pp1.lj1, c6 = 6.0f * pp1.lj2;
    const float hdt = 0.5f * nv.dt, hL = 0.5f * g.L, L = g.L;
    const unsigned char *stage_b = reinterpret_cast<const unsigned char *>(stage);
    bool exceed = false;
    double ksum = 0.0;
    const float xi = (nve && nv.ens == 1) ? (float)nv.tstate[TS_XI] : 0.f;   // read by every block before the last one updates it

    for (int q0 = 0; q0 < nown; q0 += PPB) {     // block-uniform trip count: the shuffles need whole warps
        const bool active = active_n;
        const int gi = gi_n;
        const float4 pi = stage[slot_n];         // slot 0 (the dummy) for idle thread groups
        const uint16_t *row = A.nlist + (int64_t)gi * A.pitch + sub * EPL;
        const PairParam *prow = ONE_TYPE ? nullptr : s_params + __float_as_int(pi.w) * A.ntypes;
        const PairParamX *prowx = (ONE_TYPE || FN == FN_LJ) ? nullptr : s_paramsx + __float_as_int(pi.w) * A.ntypes;
        Acc a = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f};

        if (active) {
            int c = 0;
            cp_async_wait<PF - 1>();
            Entries<EPL> ent;
            ent.v = ring[0];
            for (int k = 0; k < A.pitch; k += G) {
                if ((ent.v.x & 0xffffu) == 0u) break;                    // padding: the row is over for this thread
                cp_async<EPL * 2>(ring + c * ring_stride, row + k + PF * G);   // refill PF iterations ahead (reads past the
                cp_async_commit();                                       // row's end are harmless: the array has slack)
                c = (c + 1 == PF) ? 0 : c + 1;
                unsigned off[EPL];
                unpack_entries<EPL, SCALED>(ent, off);
                float4 pj[EPL];
#pragma unroll
                for (int e = 0; e < EPL; e++) pj[e] = *reinterpret_cast<const float4 *>(stage_b + off[e]);
                cp_async_wait<PF - 1>();                                 // the next group of entries, read before the
                ent.v = ring[c * ring_stride];                           // arithmetic so that its latency hides behind it
#pragma unroll
                for (int e = 0; e < EPL; e++) {
                    if (ONE_TYPE) {
                        pair_term<THERMO, FN>(pi, pj[e], c12, c6, pp1, px1, A.pot, a);
                    } else {
                        const int tj = __float_as_int(pj[e].w);
                        const PairParam pp = prow[tj];
                        PairParamX px = {0.f, 0.f, 0.f, 0.f};
                        if (FN != FN_LJ) px = prowx[tj];
                        pair_term<THERMO, FN>(pi, pj[e], 12.0f * pp.lj1, 6.0f * pp.lj2, pp, px, A.pot, a);
                    }
                }
            }
        }
        cp_async_wait<0>();                          // the own data of this pass has landed; nothing of this pass may land
        __syncwarp();                                //   after the next pass's copies start; lane 1's copy visible to lane 0
        const float4 *o = own + ql;
        float4 v = make_float4(0.f, 0.f, 0.f, 0.f), p = v, pb = v;
        if (nve && active && sub == 0) { v = o[0]; if (nv.kick_drift) { p = o[PPB]; pb = o[2 * PPB]; } }
        if (q0 + PPB < nown) prep(q0 + PPB);             // the next pass's copies fly during the reduction and the integration

#pragma unroll
        for (int o2 = TPP >> 1; o2 > 0; o2 >>= 1) {
            a.fx += __shfl_xor_sync(0xffffffffu, a.fx, o2);
            a.fy += __shfl_xor_sync(0xffffffffu, a.fy, o2);
            a.fz += __shfl_xor_sync(0xffffffffu, a.fz, o2);
            if (THERMO) {
                a.u += __shfl_xor_sync(0xffffffffu, a.u, o2);
                a.wxx += __shfl_xor_sync(0xffffffffu, a.wxx, o2);
                a.wxy += __shfl_xor_sync(0xffffffffu, a.wxy, o2);
                a.wxz += __shfl_xor_sync(0xffffffffu, a.wxz, o2);
                a.wyy += __shfl_xor_sync(0xffffffffu, a.wyy, o2);
                a.wyz += __shfl_xor_sync(0xffffffffu, a.wyz, o2);
                a.wzz += __shfl_xor_sync(0xffffffffu, a.wzz, o2);
            }
        }
        if (!active) continue;
        // U_i = 1/2 sum V, W_i = 1/2 sum d f (reading c6.i)
        if (THERMO && sub == TPP - 1) {
            A.virial[2 * (int64_t)gi] = make_float4(0.5f * a.wxx, 0.5f * a.wxy, 0.5f * a.wxz, 0.5f * a.wyy);
            A.virial[2 * (int64_t)gi + 1] = make_float4(0.5f * a.wyz, 0.5f * a.wzz, 0.f, 0.f);
        }
        if (sub != 0) continue;
        if (THERMO) A.force[gi] = make_float4(a.fx, a.fy, a.fz, 0.5f * a.u);
        if (!nve) continue;
        // reading c7 (and n1, n2), operation by operation as nve_kernel does it
        if (nv.kick_prev) thermo_kick_prev(nv, xi, hdt, a.fx, a.fy, a.fz, v, nv.ens == 2 ? nv.tag[gi] : 0u);
        if (nv.kick_drift) {
            thermo_kick_first(nv, xi, hdt, a.fx, a.fy, a.fz, v);
            if (nv.ens == 1) ksum += 0.5 * (double)v.w * ((double)v.x * v.x + (double)v.y * v.y + (double)v.z * v.z);
            // p is the stored position: the staged one may be another periodic image of it
            p.x = __fmaf_rn(nv.dt, v.x, p.x);
            p.y = __fmaf_rn(nv.dt, v.y, p.y);
            p.z = __fmaf_rn(nv.dt, v.z, p.z);
            if (p.x >= hL) { p.x -= L; nv.image[gi] += 1; } else if (p.x < -hL) { p.x += L; nv.image[gi] -= 1; }
            if (p.y >= hL) { p.y -= L; nv.image[A.N + gi] += 1; } else if (p.y < -hL) { p.y += L; nv.image[A.N + gi] -= 1; }
            if (p.z >= hL) { p.z -= L; nv.image[2 * (int64_t)A.N + gi] += 1; }
            else if (p.z < -hL) { p.z += L; nv.image[2 * (int64_t)A.N + gi] -= 1; }
            nv.pos_out[gi] = p;
            float dx = p.x - pb.x, dy = p.y - pb.y, dz = p.z - pb.z;
            if (dx >= hL) dx -= L; else if (dx < -hL) dx += L;
            if (dy >= hL) dy -= L; else if (dy < -hL) dy += L;
            if (dz >= hL) dz -= L; else if (dz < -hL) dz += L;
            exceed = exceed || (dx * dx + dy * dy + dz * dz) > nv.half_buff2;
        }
        nv.vel[gi] = v;
    }

    if (drift) {
        if (exceed) A.flags[nv.need_set] = 1;
        step_epilogue(nv, A.flags, ksum, gridDim.x * gridDim.y * gridDim.z);
    }
}

static int force_ppb(const hb_system *h) { return force_block_of(h) / force_tpp(h); }

size_t force_smem_bytes(const hb_system *h)
{
    // staged positions, pair table, ring of PF (2) async list copies (16 B at most) per thread, own data (2 buffers x 3 arrays)
    // and forces of a pass
    return (size_t)h->geom.cap * 16 + (h->ntypes > 1 ? ((sizeof(PairParam) * h->ntypes * h->ntypes + 15) & ~(size_t)15) : 0) +
           (h->ntypes > 1 ? ((sizeof(PairParamX) * h->ntypes * h->ntypes + 15) & ~(size_t)15) : 0) +
           (size_t)LIST_PF * 16 * force_block_of(h) + (size_t)3 * 16 * force_ppb(h) + (h->geom.fast ? 0 : sizeof(TileShared));
}

template <int TPP, int EPL, bool THERMO, bool SCALED, int FN>
static cudaError_t launch_force_tts(hb_system *h, const NveArgs *nve)
{
    const size_t smem = force_smem_bytes(h);
    const dim3 grid((unsigned)h->geom.ntx, (unsigned)h->geom.nty, (unsigned)h->geom.ntz);
    ForceArgs A{};
    A.g = h->geom;
    A.cell_start = h->cell_start;
    A.pos = h->pos();
    A.nlist = h->nlist;
    A.pitch = h->row_pitch;
    A.N = (int)h->N;
    A.ntypes = h->ntypes;
    A.pot = h->pot;
    A.params = h->params;
    A.paramsx = h->paramsx;
    A.force = h->force;
    A.virial = h->virial;
    A.flags = h->flags;
    A.do_nve = nve ? 1 : 0;
    if (nve) A.nv = *nve;
    cudaError_t e;
#define LJ_LAUNCH(ONE)                                                                                                      \
    e = cudaFuncSetAttribute(lj_tile_kernel<TPP, EPL, ONE, THERMO, SCALED, FN>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_attr(h));        \
    if (e != cudaSuccess) return e;                                                                                         \
    lj_tile_kernel<TPP, EPL, ONE, THERMO, SCALED, FN><<<grid, force_block_of(h), smem, h->stream>>>(A);
    if (h->ntypes == 1) { LJ_LAUNCH(true) } else { LJ_LAUNCH(false) }
#undef LJ_LAUNCH
    h->stats.kernel_launches++;
    return cudaGetLastError();
}

template <int TPP, int EPL, int FN>
static cudaError_t launch_force_t(hb_system *h, const NveArgs *nve)
{
    // energies and virials of a step can only be read after hb_run_nve returns: with thermo_every = 0 the inner
    // steps of a chunk (both half kicks fused in) compute forces only
    const bool thermo = !(nve && nve->forces_only);
    const bool scaled = h->geom.eshift == 4;
    if (thermo) return scaled ? launch_force_tts<TPP, EPL, true, true, FN>(h, nve) : launch_force_tts<TPP, EPL, true, false, FN>(h, nve);
    return scaled ? launch_force_tts<TPP, EPL, false, true, FN>(h, nve) : launch_force_tts<TPP, EPL, false, false, FN>(h, nve);
}

cudaError_t launch_force(hb_system *h, const NveArgs *nve)
{
    // the smoothed and the generic functors come in the default thread layout only (tpp 2, epl 8); the tunables apply
    // to plain / shifted LJ
    if (h->pot != HB_POT_LJ) return launch_force_t<2, 8, FN_GEN>(h, nve);
    if (h->shift_mode == HB_XPLOR) return launch_force_t<2, 8, FN_XPLOR>(h, nve);
    const int epl = h->tun.epl == 8 ? 8 : 4;
    switch (h->tun.tpp) {
        case 2: return epl == 8 ? launch_force_t<2, 8, FN_LJ>(h, nve) : launch_force_t<2, 4, FN_LJ>(h, nve);
        case 8: return launch_force_t<8, 4, FN_LJ>(h, nve);   // 8 x 8 entries would read past the 32-entry row padding
        default: return epl == 8 ? launch_force_t<4, 8, FN_LJ>(h, nve) : launch_force_t<4, 4, FN_LJ>(h, nve);
    }
}

// accessor: (Fx, Fy, Fz, U) and the six virial components BY TAG
__global__ void unpack_forces_kernel(const float4 *__restrict__ force, const float4 *__restrict__ virial,
                                     const uint32_t *__restrict__ tag, int N, float *__restrict__ f4, float *__restrict__ vir6)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= N) return;
    const int64_t t = tag[i];
    if (f4) reinterpret_cast<float4 *>(f4)[t] = force[i];
    if (vir6) {
        const float4 a = virial[2 * (int64_t)i], b = virial[2 * (int64_t)i + 1];
        float *o = vir6 + 6 * t;
        o[0] = a.x; o[1] = a.y; o[2] = a.z; o[3] = a.w; o[4] = b.x; o[5] = b.y;
    }
}

cudaError_t launch_unpack_forces(hb_system *h, float *f4, float *vir6)
{
    unpack_forces_kernel<<<(unsigned)cdiv(h->N, 256), 256, 0, h->stream>>>(h->force, h->virial, h->tag, (int)h->N, f4, vir6);
    return cudaGetLastError();
}
