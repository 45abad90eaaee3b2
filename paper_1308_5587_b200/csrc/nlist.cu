// Neighbor list (Algorithm 3), re-designed for sm_100a.
//
// The paper runs one thread per particle and names the resulting scattered,
// unsynchronised row writes "a big bottleneck" that "GF100 does not have enough
// shared memory to regularize".  Here ONE BLOCK OWNS ONE TILE of
// cells (tile.cuh): the tile plus its one-cell halo is staged once in shared
// memory (one warp per halo cell), already moved to the periodic image the tile sees.
//
// PAIR ROWS.  ncu on the round-1 step kernel showed the shared-memory pipe as its limit: every listed pair costs one
// random 16-byte gather (profiles/r2a_kernels.md).  So two consecutive particles (a, a + 1) of an own (y, z) row of
// the tile share ONE list row, the UNION of their neighbor sets (they are about one sigma apart, the union is about
// 1.3 times one set): one gather in the step kernel then serves two pair evaluations.  Each 16-bit entry carries, beside
// the slot, two bits that say whose neighbor it is (bit 0: of a, bit 1: of a + 1), so the row still states N(a) and
// N(a + 1) exactly (hb_get_nlist reads them back); the two particles of a pair are never entries of their own row
// (the step kernel evaluates that one interaction directly; nlistn carries a flag if they are within r_max).
//
//   1. candidates: for every own row of the tile the block writes ONE list of candidate slots, column by column in x
//      (a column = the 3 x 3 cells around the row at one x), so that the 27 cells around any run of own cells are ONE
//      contiguous range of it (Alg. 3 l.11; no celladj table: PAPER.md:187 stored it to save registers);
//   2. a warp takes four consecutive particles of a row (two pairs): lane l tests candidates l, l + 32, ... of the
//      range that belongs to the cells of those four against all four (one candidate load serves four tests, Alg. 3
//      l.16-17) and records the hits as bits of four registers;
//   3. per pair the union mask is compacted with one warp prefix sum of popcounts (both pairs in one scan) and the
//      lanes write their entries straight into the row-major, 128-byte aligned list; the row ends with at least 32
//      entries of 0 (the step kernel reads no row length).
// List entries are slots of the tile's staging layout, not particle indices: the step kernel stages the same tile
// the same way and gathers from shared memory (hb_get_nlist translates back to tags).
// The kernel also finishes the reorder of the particle data: it copies the tile's own particles from the scratch set
// (cell order) back into the live arrays.
#include "cells_dev.cuh"
#include "tile.cuh"

constexpr int NL_PPI = 4;        // particles tested per candidate load = two pairs
constexpr int NL_CHUNK = 1024;   // candidates per pass over a group = 32 groups of 32 = one bit mask per particle

size_t nlist_smem_bytes(const hb_system *h)
{
    return (size_t)h->geom.cap * 16 + (size_t)h->geom.ccap * 2;   // staged positions | candidate lists
}

struct CopyBack {   // scratch set -> live arrays; pos == nullptr: skip
    float4 *pos, *vel;
    const float4 *vel2;
    int *image;
    const int *image2;
    uint32_t *tag, *rtag;
    const uint32_t *tag2;
    int N;
};

struct ListArgs {
    TileGeom g;
    const int *cell_start;
    const float4 *pos_build;
    float rmax2;
    const float *rmax2_pair;   // TYPED: [ntypes * ntypes] squared list cutoffs (r_cut,ab + r_buff)^2
    int ntypes;
    int pitch;
    uint16_t *nlist;
    int *nlistn, *flags;
    CopyBack cb;
};

struct ListShared {
    TileShared t;
    int colabs[TILE_HMAX + 1];       // start of column (own row, jx) in the candidate array, index row * hx + jx; [nrows * hx] = total
    int colmid[TILE_HMAX];           // where the centre cell of that column (the own row's cell at jx) starts
    int grp_off[TILE_ROWS_MAX + 1];  // groups of NL_PPI particles per own row, prefix
};

// Algorithm 3 for one tile, by one block
template <bool TYPED>
__device__ __forceinline__ void nlist_tile_body(const ListArgs &la, const int tile, unsigned char *smem_raw)
{
    const TileGeom &g = la.g;
    const int *__restrict__ cell_start = la.cell_start;
    const float4 *__restrict__ pos_build = la.pos_build;
    const float rmax2 = la.rmax2;
    const int pitch = la.pitch;
    uint16_t *__restrict__ nlist = la.nlist;
    int *__restrict__ nlistn = la.nlistn;
    int *__restrict__ flags = la.flags;
    const CopyBack &cb = la.cb;
    __shared__ ListShared s;
    __shared__ float s_rm2[TYPED ? 64 : 1];     // TYPED needs ntypes <= 8 (the host falls back to the single cutoff otherwise)
    float4 *stage = reinterpret_cast<float4 *>(smem_raw);
    uint16_t *clist = reinterpret_cast<uint16_t *>(smem_raw + (size_t)g.cap * 16);
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, nwarps = blockDim.x >> 5;
    constexpr unsigned FULL = 0xffffffffu;

    if (tile == 0 && threadIdx.x == 0) flags[FL_BUILDS] += 1;
    if (TYPED)
        for (int k = threadIdx.x; k < la.ntypes * la.ntypes; k += blockDim.x) s_rm2[k] = la.rmax2_pair[k];
    TileCtx t;
    tile_decode(g, tile, t);
    const bool fits = tile_tables(g, cell_start, t, s.t, flags);

    // the reorder's last leg: own particles, scratch set -> live arrays (always, so the state stays whole)
    if (cb.pos) {
        for (int q = threadIdx.x; q < t.nown; q += blockDim.x) {
            int gi, slot;
            tile_own(s.t.d, q, gi, slot);
            cb.pos[gi] = pos_build[gi];
            cb.vel[gi] = cb.vel2[gi];
            cb.image[gi] = cb.image2[gi];
            cb.image[cb.N + gi] = cb.image2[cb.N + gi];
            cb.image[2 * (int64_t)cb.N + gi] = cb.image2[2 * (int64_t)cb.N + gi];
            const uint32_t tg = cb.tag2[gi];
            cb.tag[gi] = tg;
            cb.rtag[tg] = gi;
        }
    }
    if (!fits) return;
    tile_stage_positions_by_cell(g, t, s.t, pos_build, stage, nullptr);

    // ---- 1. candidate columns: lengths, prefix, fill ----
    const int ncol = t.nrows * t.hx;
    for (int c = threadIdx.x; c < ncol; c += blockDim.x) {
        const int orow = c / t.hx, jx = c - orow * t.hx;
        const int ly = orow % t.ey, lz = orow / t.ey;
        int n = 0;
#pragma unroll
        for (int k = 0; k < 9; k++) {
            const int h = jx + t.hx * ((ly + k % 3) + t.hy * (lz + k / 3));   // (ly + 1 + dy, lz + 1 + dz), dy, dz = -1, 0, 1
            n += s.t.hslot[h + 1] - s.t.hslot[h];
        }
        s.colabs[c] = n;
    }
    if (threadIdx.x == 0) {
        int run = 0;
        s.grp_off[0] = 0;
        for (int r = 0; r < t.nrows; r++) { run += (s.t.d.own_off[r + 1] - s.t.d.own_off[r] + NL_PPI - 1) / NL_PPI; s.grp_off[r + 1] = run; }
    }
    __syncthreads();
    if (threadIdx.x < 32) {   // exclusive scan of up to TILE_HMAX column lengths: 8 per lane
        const int base = lane * 8;
        int v[8], tsum = 0;
#pragma unroll
        for (int q = 0; q < 8; q++) { v[q] = base + q < ncol ? s.colabs[base + q] : 0; tsum += v[q]; }
        int incl = tsum;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) { const int y = __shfl_up_sync(FULL, incl, o); if (lane >= o) incl += y; }
        int run = incl - tsum;
#pragma unroll
        for (int q = 0; q < 8; q++) { if (base + q < ncol) s.colabs[base + q] = run; run += v[q]; }
        if (lane == 31) s.colabs[ncol] = run;
    }
    __syncthreads();
    const int ctotal = s.colabs[ncol];
    if (ctotal > g.ccap) {    // the candidate lists need more room than the staging capacity was sized for: same repair
        if (threadIdx.x == 0) atomicMax(&flags[FL_STAGE_OVER], max(t.nslots + 1, (int)((int64_t)ctotal * g.cap / g.ccap) + 1));
        return;
    }
    for (int c = warp; c < ncol; c += nwarps) {
        const int orow = c / t.hx, jx = c - orow * t.hx;
        const int ly = orow % t.ey, lz = orow / t.ey;
        int at = s.colabs[c];
#pragma unroll
        for (int k = 0; k < 9; k++) {
            const int h = jx + t.hx * ((ly + k % 3) + t.hy * (lz + k / 3));
            const int s0 = s.t.hslot[h], n = s.t.hslot[h + 1] - s0;
            if (k == 4 && lane == 0) s.colmid[c] = at;
            for (int v = lane; v < n; v += 32) clist[at + v] = (uint16_t)(s0 + v);
            at += n;
        }
    }
    __syncthreads();

    // ---- 2., 3. groups of four particles (two pairs) ----
    int wmax_len = 0, wmax_need = 0;
    const int ngrp = s.grp_off[t.nrows];
    for (int grp = warp; grp < ngrp; grp += nwarps) {
        int orow = 0;
        while (orow + 1 < t.nrows && s.grp_off[orow + 1] <= grp) orow++;
        const int q0 = NL_PPI * (grp - s.grp_off[orow]);
        const int nvalid = min(NL_PPI, s.t.d.own_off[orow + 1] - s.t.d.own_off[orow] - q0);
        const int slot_f = s.t.d.own_slot[orow] + q0;
        const int gi_f = s.t.d.own_start[orow] + q0;
        const int ly = orow % t.ey, lz = orow / t.ey;
        const int hrow = ((lz + 1) * t.hy + (ly + 1)) * t.hx;     // halo cell (jx = 0) of the own row
        // own cell lx of a slot of this row: how many own cells start at or before it, minus one
        const int cell_first = lane < t.ex ? s.t.hslot[hrow + 1 + lane] : 0x7fffffff;
        float px[NL_PPI], py[NL_PPI], pz[NL_PPI];
        int self[NL_PPI], cnt[NL_PPI];
        const float *rmrow[NL_PPI];
        int lxa = 0, lxb = 0;
#pragma unroll
        for (int p = 0; p < NL_PPI; p++) {
            px[p] = py[p] = pz[p] = -1e18f;
            self[p] = -1;
            cnt[p] = 0;
            rmrow[p] = s_rm2;
            if (p < nvalid) {     // warp-uniform
                const int sp = slot_f + p;
                const float4 q = stage[sp];                      // same address in all lanes: one broadcast
                px[p] = q.x; py[p] = q.y; pz[p] = q.z;
                if (TYPED) rmrow[p] = s_rm2 + __float_as_int(q.w) * la.ntypes;
                const int lx = __popc(__ballot_sync(FULL, cell_first <= sp)) - 1;
                if (p == 0) lxa = lx;
                lxb = lx;
                self[p] = s.colmid[orow * t.hx + lx + 1] + (sp - s.t.hslot[hrow + 1 + lx]);
            }
        }
        const int c0 = s.colabs[orow * t.hx + lxa], c1 = s.colabs[orow * t.hx + lxb + 3];
        uint16_t *const rowA = nlist + (int64_t)gi_f * pitch, *const rowB = nlist + (int64_t)(gi_f + 2) * pitch;
        const int capA = nvalid >= 2 ? 2 * pitch : pitch, capB = nvalid >= 4 ? 2 * pitch : pitch;
        int totA = 0, totB = 0;
        bool abA = false, abB = false;

        for (int k0 = c0; k0 < c1; k0 += NL_CHUNK) {
            const int Tc = min(NL_CHUNK, c1 - k0);
            const int ngroups = (Tc + 31) >> 5;
            unsigned hits[NL_PPI] = {0u, 0u, 0u, 0u};
            // lane l tests candidates l, l+32, ...; bit gq of hits[p] records candidate 32 gq + l (Alg. 3 l.16-17)
#pragma unroll 2
            for (int gq = 0; gq < ngroups; gq++) {
                const int ci = k0 + (gq << 5) + lane;
                const float4 e = stage[ci < c1 ? clist[ci] : 0];      // slot 0 = the far-away dummy: never a hit
                const unsigned bit = 1u << gq;
#pragma unroll
                for (int p = 0; p < NL_PPI; p++) {
                    const float dx = e.x - px[p], dy = e.y - py[p], dz = e.z - pz[p];
                    const float d2 = __fmaf_rn(dz, dz, __fmaf_rn(dy, dy, __fmul_rn(dx, dx)));
                    const float rm = TYPED ? rmrow[p][__float_as_int(e.w)] : rmax2;
                    if (d2 < rm) hits[p] |= bit;   // strict <
                }
            }
            // the particles of a pair are not entries of their own row; whether they are within r_max of each other
            // (the test is symmetric bit for bit: dx and -dx square to the same number) goes into nlistn
#pragma unroll
            for (int p = 0; p < NL_PPI; p++) {
                const int rel = self[p] - k0;
                if (self[p] >= 0 && rel >= 0 && rel < Tc) {      // warp-uniform
                    const unsigned b = 1u << (rel >> 5);
                    const bool mine = (rel & 31) == lane;
                    if (p & 1) {   // second particle of its pair: is it a neighbor of the first?
                        const bool ab = __any_sync(FULL, mine && (hits[p - 1] & b));
                        if (p == 1) abA = abA || ab; else abB = abB || ab;
                    }
                    if (mine) { hits[p & ~1] &= ~b; hits[p | 1] &= ~b; }
                }
            }
#pragma unroll
            for (int p = 0; p < NL_PPI; p++) cnt[p] += __reduce_add_sync(FULL, __popc(hits[p]));
            // compact: one warp scan of the per-lane union counts of both pairs gives every lane its positions (l.18-19)
            unsigned UA = hits[0] | hits[1], UB = hits[2] | hits[3];
            const int x = __popc(UA) | (__popc(UB) << 16);
            int inc = x;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                const int y = __shfl_up_sync(FULL, inc, o);
                if (lane >= o) inc += y;
            }
            const int tot = __shfl_sync(FULL, inc, 31);
            int atA = totA + ((inc - x) & 0xffff), atB = totB + ((inc - x) >> 16);
            while (UA) {
                const int gq = __ffs(UA) - 1;
                UA &= UA - 1;
                const unsigned e = ((unsigned)clist[k0 + (gq << 5) + lane] << 2) | ((hits[0] >> gq) & 1u) | (((hits[1] >> gq) & 1u) << 1);
                if (atA < capA) rowA[atA] = (uint16_t)e;
                atA++;
            }
            while (UB) {
                const int gq = __ffs(UB) - 1;
                UB &= UB - 1;
                const unsigned e = ((unsigned)clist[k0 + (gq << 5) + lane] << 2) | ((hits[2] >> gq) & 1u) | (((hits[3] >> gq) & 1u) << 1);
                if (atB < capB) rowB[atB] = (uint16_t)e;
                atB++;
            }
            totA += tot & 0xffff;
            totB += tot >> 16;
        }

#pragma unroll
        for (int pr = 0; pr < 2; pr++) {
            if (2 * pr >= nvalid) break;      // warp-uniform
            const bool two = 2 * pr + 1 < nvalid;
            uint16_t *row = pr ? rowB : rowA;
            const int cap = pr ? capB : capA, tot = pr ? totB : totA;
            const int ab = (pr ? abB : abA) ? 1 : 0;
            const int ca = cnt[2 * pr] + ab, cbn = cnt[2 * pr + 1] + ab;
            const int nw = min(tot, cap);
            // at least 32 entries of 0 end the row: the step kernel stops at the first one it meets
            // (pad_end is even and the row is 128-byte aligned: one 16-bit store if nw is odd, then 32-bit words)
            const int pad_end = min(cap, (nw & ~(ROW_PAD - 1)) + 2 * ROW_PAD);
            const int e0 = (nw + 1) & ~1;
            if (lane == 0 && e0 != nw && nw < pad_end) row[nw] = 0;
            if (e0 + 2 * lane < pad_end) reinterpret_cast<uint32_t *>(row)[(e0 >> 1) + lane] = 0u;
            if (lane == 0) {                                     // l.22
                const int gi0 = gi_f + 2 * pr;
                nlistn[gi0] = ca | (ab << 30);                   // bit 30: the two particles of the pair are neighbors
                if (two) nlistn[gi0 + 1] = cbn;
            }
            wmax_len = max(wmax_len, two ? max(ca, cbn) : ca);
            // a pair's row is the two rows of its particles: the union must fit in 2 pitch, and (so that row_pitch
            // >= the longest neighbor set stays true) each set in one pitch
            wmax_need = max(wmax_need, two ? max(max(ca, cbn), (tot + 1) >> 1) : tot);
        }
    }
    // longest neighbor set and longest row needed by this build (may exceed the pitch: overflow)
    if (lane == 0) {
        if (wmax_len > __ldcg(&flags[FL_MAX_NBRS])) atomicMax(&flags[FL_MAX_NBRS], wmax_len);
        if (wmax_need > pitch) atomicMax(&flags[FL_OVERFLOWED], wmax_need);
    }
}

template <bool TYPED>
__global__ void __launch_bounds__(TILE_THREADS) nlist_tile_kernel(ListArgs la, const int *__restrict__ pred)
{
    if (pred && *pred == 0) return;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    nlist_tile_body<TYPED>(la, blockIdx.x, smem_raw);
}

// The whole rebuild in ONE cooperative launch: Algorithm 2 (count, scan, scatter), the reorder into cell
// order (gather) and Algorithm 3, with grid-wide barriers between the phases.  Inside hb_run_nve's graphs
// every step carries the rebuild's kernels as early-exit launches; one launch instead of five takes
// about 4 us off every step (N = 64,000, measured), and the phases lose their launch gaps.
template <bool TYPED, bool WITH_LIST>
__global__ void __launch_bounds__(TILE_THREADS, 4) rebuild_coop_kernel(CellArgs ca, GatherArgs ga, int do_sort, ListArgs la,
                                                                    const int *__restrict__ pred)
{
    if (pred && *pred == 0) return;   // every block takes the same way: no barrier is left waiting
    extern __shared__ __align__(16) unsigned char smem_raw[];
    __shared__ int scan_smem[SCAN_THREADS / 32];
    // Grid-wide barrier: the launch is cooperative, so all blocks are resident; every block adds one to a
    // counter and waits until the counter reaches (barriers passed so far + 1) x gridDim.x.  (cooperative_groups'
    // grid.sync() took about 5 us per barrier here, this one about 1 us.)  The counter of build b is
    // flags[FL_BAR0 + (b & 1)], b = flags[FL_BAR_GEN]: every block reads b before its first barrier, block 0
    // advances it after its last one and clears the other counter for the next build.
    int *const flags = la.flags;
    const int gen = *(volatile int *)&flags[FL_BAR_GEN];
    unsigned *const bar = reinterpret_cast<unsigned *>(flags + FL_BAR0 + (gen & 1));
    if (blockIdx.x == 0 && threadIdx.x == 0) flags[FL_BAR0 + ((gen + 1) & 1)] = 0;
    unsigned passed = 0;
    auto grid_barrier = [&]() {
        passed += gridDim.x;
        __syncthreads();
        if (threadIdx.x == 0) {
            __threadfence();
            atomicAdd(bar, 1u);
            while (*(volatile unsigned *)bar < passed) { }
            __threadfence();
        }
        __syncthreads();
    };
    const int64_t gtid = (int64_t)blockIdx.x * blockDim.x + threadIdx.x, gsize = (int64_t)gridDim.x * blockDim.x;

    for (int64_t i = gtid; i < ca.N; i += gsize) cell_count_one(ca, (int)i);
    grid_barrier();
    const int nscan = (int)((ca.ncells + SCAN_TILE - 1) / SCAN_TILE);
    for (int st = blockIdx.x; st < nscan; st += gridDim.x) {
        const int total = block_scan_tile(ca.cell_count, ca.ncells, ca.cell_local, 0, true, ca.cell_count, st);
        if (threadIdx.x == 0) ca.sums[st] = total;
    }
    grid_barrier();
    if (blockIdx.x == 0) scan_sums_in_place(ca.sums, nscan, scan_smem);
    grid_barrier();
    const int64_t nsc = ca.N > ca.ncells + 1 ? (int64_t)ca.N : ca.ncells + 1;
    for (int64_t i = gtid; i < nsc; i += gsize) cell_scatter_one(ca, i);
    grid_barrier();
    const int lane = threadIdx.x & 31;
    for (int64_t c = gtid >> 5; c < ca.ncells; c += gsize >> 5) cell_gather_one(ca.cell_start, ca.perm, ga, do_sort, c, lane);
    if (WITH_LIST) {
        if (blockIdx.x == 0 && threadIdx.x == 0) flags[FL_TILE_CTR] = 0;
        grid_barrier();
    }
    if (blockIdx.x == 0 && threadIdx.x == 0) flags[FL_BAR_GEN] = gen + 1;   // every block is past its first barrier
    if (WITH_LIST) {
        // tiles are handed out on demand, like the hardware hands out blocks to the stand-alone list kernel
        __shared__ int next_tile;
        for (;;) {
            if (threadIdx.x == 0) next_tile = atomicAdd(&flags[FL_TILE_CTR], 1);
            __syncthreads();
            const int tile = next_tile;
            if (tile >= la.g.ntiles) break;
            nlist_tile_body<TYPED>(la, tile, smem_raw);
            __syncthreads();              // the next tile reuses the staging area (and next_tile)
        }
    }
}

static ListArgs make_list_args(hb_system *h, bool copyback)
{
    ListArgs la{};
    la.g = h->geom;
    la.cell_start = h->cell_start;
    la.pos_build = h->pos_build;
    la.rmax2 = h->r_max * h->r_max;
    la.rmax2_pair = h->rmax2_pair;
    la.ntypes = h->ntypes;
    la.pitch = h->row_pitch;
    la.nlist = h->nlist;
    la.nlistn = h->nlistn;
    la.flags = h->flags;
    if (copyback) la.cb = CopyBack{h->pos(), h->vel, h->vel2, h->image, h->image2, h->tag, h->rtag, h->tag2, (int)h->N};
    return la;
}

// per-type-pair list cutoffs (tunable nlist_pair_rcut) need the table in shared memory
static bool list_typed(const hb_system *h) { return h->tun.nlist_pair_rcut != 0 && h->ntypes > 1 && h->ntypes <= 8; }

cudaError_t launch_nlist(hb_system *h, const int *pred, bool copyback)
{
    const size_t smem = nlist_smem_bytes(h);
    const unsigned grid = (unsigned)h->geom.ntiles;
    const ListArgs la = make_list_args(h, copyback);
    cudaError_t e;
#define NL_LAUNCH(TYPED)                                                                                                \
    e = cudaFuncSetAttribute(nlist_tile_kernel<TYPED>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);         \
    if (e != cudaSuccess) return e;                                                                                     \
    nlist_tile_kernel<TYPED><<<grid, h->tun.nlist_block, smem, h->stream>>>(la, pred);
    if (list_typed(h)) { NL_LAUNCH(true) } else { NL_LAUNCH(false) }
#undef NL_LAUNCH
    h->stats.kernel_launches++;
    return cudaGetLastError();
}

// count + scan + scatter + gather (+ list) in one cooperative launch (see rebuild_coop_kernel)
template <bool TYPED, bool WITH_LIST>
static cudaError_t launch_rebuild_coop_t(hb_system *h, const int *pred)
{
    const size_t smem = WITH_LIST ? nlist_smem_bytes(h) : 0;
    cudaError_t e = cudaFuncSetAttribute(rebuild_coop_kernel<TYPED, WITH_LIST>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    int per_sm = 0;
    e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, rebuild_coop_kernel<TYPED, WITH_LIST>, TILE_THREADS, smem);
    if (e != cudaSuccess) return e;
    if (per_sm < 1) return cudaErrorCooperativeLaunchTooLarge;
    // every phase strides over the grid; no more blocks than there is work for or than fit on the device at once
    const int64_t want = std::max<int64_t>(WITH_LIST ? h->geom.ntiles : 1, cdiv(h->N, TILE_THREADS));
    // the cells-only kernel is barrier-bound: few blocks make the grid-wide barriers cheap (coop_blocks per SM)
    if (!WITH_LIST) per_sm = std::min(per_sm, std::max(1, h->tun.coop_blocks));
    const unsigned grid = (unsigned)std::max<int64_t>(1, std::min<int64_t>(want, (int64_t)per_sm * h->sm_count));
    CellArgs ca = make_cell_args(h);
    GatherArgs ga = make_gather_args(h);
    int do_sort = h->tun.cell_sort;
    ListArgs la = make_list_args(h, true);
    void *args[] = {&ca, &ga, &do_sort, &la, (void *)&pred};
    e = cudaLaunchCooperativeKernel((const void *)rebuild_coop_kernel<TYPED, WITH_LIST>, dim3(grid), dim3(TILE_THREADS), args, smem,
                                    h->stream);
    h->stats.kernel_launches++;
    return e != cudaSuccess ? e : cudaGetLastError();
}

cudaError_t launch_rebuild_coop(hb_system *h, const int *pred, bool with_list)
{
    if (!with_list) return launch_rebuild_coop_t<false, false>(h, pred);
    return list_typed(h) ? launch_rebuild_coop_t<true, true>(h, pred) : launch_rebuild_coop_t<false, true>(h, pred);
}

// ---- accessors: the list BY TAG as CSR ----
__global__ void nlist_counts_by_tag_kernel(const int *__restrict__ nlistn, const uint32_t *__restrict__ tag, int N,
                                           int *__restrict__ counts)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < N) counts[tag[i]] = nlistn[i] & 0x3fffffff;
}

// One block per tile: slot -> storage index through the same tables, then the pair rows -> tags.  A warp reads the row
// of a pair 32 entries at a time; an entry goes to the first / second particle's output row if its bit 0 / 1 is set.
__global__ void __launch_bounds__(TILE_THREADS)
nlist_fill_by_tag_kernel(TileGeom g, const int *__restrict__ cell_start, const uint16_t *__restrict__ nlist,
                         const int *__restrict__ nlistn, int pitch, const uint32_t *__restrict__ tag,
                         const int64_t *__restrict__ row_start, uint32_t *__restrict__ out, int *__restrict__ flags)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    __shared__ TileShared s;
    int *gidx = reinterpret_cast<int *>(smem_raw);
    TileCtx t;
    tile_decode(g, blockIdx.x, t);
    if (!tile_tables(g, cell_start, t, s, flags)) return;
    for (int sl = 1 + threadIdx.x; sl < t.nslots; sl += TILE_THREADS) {
        const int h = tile_cell_of_slot(t, s, sl);
        gidx[sl] = s.hg[h] + (sl - s.hslot[h]);
    }
    __syncthreads();
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const unsigned lt = (1u << lane) - 1u;
    const int npairs = s.d.pair_off[s.d.nrows];
    for (int P = warp; P < npairs; P += TILE_THREADS / 32) {
        int gi0, slot0, np;
        tile_pair(s.d, P, gi0, slot0, np);
        const uint32_t ta = tag[gi0], tb = np == 2 ? tag[gi0 + 1] : 0u;
        int64_t oa = row_start[ta], ob = np == 2 ? row_start[tb] : 0;
        if (np == 2 && (nlistn[gi0] >> 30) & 1) {   // the two particles of the pair are neighbors of each other
            if (lane == 0) { out[oa] = tb; out[ob] = ta; }
            oa++; ob++;
        }
        const uint16_t *row = nlist + (int64_t)gi0 * pitch;
        const int cap = np == 2 ? 2 * pitch : pitch;
        for (int k0 = 0; k0 < cap; k0 += 32) {
            const unsigned e = k0 + lane < cap ? row[k0 + lane] : 0u;
            const unsigned ma = __ballot_sync(0xffffffffu, e & 1u), mb = __ballot_sync(0xffffffffu, e & 2u);
            const uint32_t tj = e ? tag[gidx[e >> 2]] : 0u;
            if (e & 1u) out[oa + __popc(ma & lt)] = tj;
            if (e & 2u) out[ob + __popc(mb & lt)] = tj;
            oa += __popc(ma); ob += __popc(mb);
            if (__any_sync(0xffffffffu, e == 0u)) break;      // padding: the row is over
        }
    }
}

// rows[k] = sum of counts[0 .. k), k = 0 .. N (int64): a single block walks the array in chunks of 2048 with a carry
// (an accessor, not the hot path: N / 2048 sequential block scans, 0.5 ms at N = 10^6)
__global__ void __launch_bounds__(SCAN_THREADS) nlist_rows_by_tag_kernel(const int *__restrict__ counts, int N, int64_t *__restrict__ rows)
{
    __shared__ int warp_tot[SCAN_THREADS / 32];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    int64_t carry = 0;
    for (int64_t base = 0; base < N; base += SCAN_TILE) {
        const int64_t k0 = base + (int64_t)threadIdx.x * SCAN_ITEMS;
        int x[SCAN_ITEMS], tsum = 0;
#pragma unroll
        for (int q = 0; q < SCAN_ITEMS; q++) { x[q] = k0 + q < N ? counts[k0 + q] : 0; tsum += x[q]; }
        int incl = tsum;
        for (int o = 1; o < 32; o <<= 1) { const int y = __shfl_up_sync(0xffffffffu, incl, o); if (lane >= o) incl += y; }
        if (lane == 31) warp_tot[warp] = incl;
        __syncthreads();
        int woff = 0, total = 0;
        for (int w = 0; w < SCAN_THREADS / 32; w++) { if (w < warp) woff += warp_tot[w]; total += warp_tot[w]; }
        int64_t run = carry + woff + incl - tsum;
#pragma unroll
        for (int q = 0; q < SCAN_ITEMS; q++) { if (k0 + q < N) rows[k0 + q] = run; run += x[q]; }
        carry += total;
        __syncthreads();
    }
    if (threadIdx.x == 0) rows[N] = carry;
}

cudaError_t launch_nlist_rows_by_tag(hb_system *h, const int *counts, int64_t *rows)
{
    nlist_rows_by_tag_kernel<<<1, SCAN_THREADS, 0, h->stream>>>(counts, (int)h->N, rows);
    return cudaGetLastError();
}

cudaError_t launch_nlist_counts_by_tag(hb_system *h, int *counts)
{
    nlist_counts_by_tag_kernel<<<(unsigned)cdiv(h->N, 256), 256, 0, h->stream>>>(h->nlistn, h->tag, (int)h->N, counts);
    return cudaGetLastError();
}

cudaError_t launch_nlist_fill_by_tag(hb_system *h, const int64_t *row_start, uint32_t *out)
{
    const size_t smem = (size_t)h->geom.cap * 4;
    cudaError_t e = cudaFuncSetAttribute(nlist_fill_by_tag_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    nlist_fill_by_tag_kernel<<<(unsigned)h->geom.ntiles, TILE_THREADS, smem, h->stream>>>(
        h->geom, h->cell_start, h->nlist, h->nlistn, h->row_pitch, h->tag, row_start, out, h->flags);
    return cudaGetLastError();
}
