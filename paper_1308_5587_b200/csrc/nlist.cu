// Neighbor list (Algorithm 3), re-designed for sm_100a.
//
// The paper runs one thread per particle and names the resulting scattered,
// unsynchronised row writes "a big bottleneck" that "GF100 does not have enough
// shared memory to regularize".  Here ONE BLOCK OWNS ONE TILE of
// cells (tile.cuh): the tile plus its one-cell halo is staged once in shared
// memory (one warp per halo cell), already moved to the periodic image the tile sees,
// and then ONE WARP OWNS ONE CELL of the tile (several warps split a cell's particles
// when the tile has fewer cells than the block has warps):
//   1. lanes 0..8 look up the nine x-rows of three adjacent cells (on the fly, no
//      celladj table: PAPER.md:187 stored it to save registers) -- in the staged
//      layout each row is one contiguous run of slots -- and the warp flattens the
//      nine runs into one list of candidate slots (16-bit), padded with the
//      far-away dummy slot 0 to whole groups of 32;
//   2. for every particle i of the cell (PPI at a time, so each candidate load
//      serves PPI distance tests) lane l tests candidates l, l+32, ... and records
//      the hits as bits of a register; one warp prefix sum of the per-lane __popc
//      counts gives every lane its positions in the row and the lanes write their
//      hits' SLOT NUMBERS (16 bit) straight into the row-major, 128-byte aligned
//      list; the row ends with at least 32 entries of slot 0 (the force kernel reads no row length).
// List entries are slots of the tile's staging layout, not particle indices: the
// force kernel stages the same tile the same way and gathers from shared memory
// (hb_get_nlist translates back to tags).  Half the bytes of a 32-bit index list.
// The kernel also finishes the reorder of the particle data: it copies the tile's
// own particles from the scratch set (cell order) back into the live arrays.
#include "cells_dev.cuh"
#include "tile.cuh"

constexpr int NL_CLIST = 1024;   // candidate slots per warp per chunk = 32 groups of 32 = one bit mask
constexpr int NL_WARPS = TILE_THREADS / 32;

size_t nlist_smem_bytes(const hb_system *h)
{
    return (size_t)h->geom.cap * 16 + (size_t)NL_WARPS * NL_CLIST * 2;   // sized for the largest block (8 warps)
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
    const float *rmax2_pair;   // TYPED: [ntypes * ntypes] squared list cutoffs (r_cut,ab + r_buff)^2 (tunable nlist_pair_rcut)
    int ntypes;
    int pitch;
    uint16_t *nlist;
    int *nlistn, *flags;
    CopyBack cb;
};

// Algorithm 3 for one tile, by one block of TILE_THREADS threads
template <int PPI, bool TYPED>
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
    const int eshift = g.eshift;
    __shared__ TileShared s;
    __shared__ float s_rm2[TYPED ? 64 : 1];     // per-type-pair list cutoffs (reading t1): ntypes <= 8, else the single cutoff
    float4 *stage = reinterpret_cast<float4 *>(smem_raw);
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    uint16_t *clist = reinterpret_cast<uint16_t *>(smem_raw + (size_t)g.cap * 16) + warp * NL_CLIST;

    if (tile == 0 && threadIdx.x == 0) flags[FL_BUILDS] += 1;
    if (TYPED)
        for (int k = threadIdx.x; k < la.ntypes * la.ntypes; k += blockDim.x) s_rm2[k] = la.rmax2_pair[k];
    TileCtx t;
    tile_decode(g, tile, t);
    const bool fits = tile_tables(g, cell_start, t, s, flags);

    // the reorder's last leg: own particles, scratch set -> live arrays (always, so the state stays whole)
    if (cb.pos) {
        for (int q = threadIdx.x; q < t.nown; q += blockDim.x) {
            int gi, slot;
            tile_own(s.d, q, gi, slot);
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
    __shared__ alignas(8) uint64_t stage_bar;
    if (g.fast) {
        tile_stage_positions_bulk(g, t, s, pos_build, stage, &stage_bar);
    } else {
        tile_stage_positions_by_cell(g, t, s, pos_build, stage, nullptr);
        __syncthreads();
    }

    int wmax = 0;
    const int ncell_own = t.ex * t.ey * t.ez;
    // a tile with fewer cells than the block has warps gives every cell several warps: they share the cell's
    // candidates and split its particles
    const int nwarps = blockDim.x >> 5;
    const int wpc = max(1, nwarps / max(1, ncell_own));
    for (int item = warp; item < ncell_own * wpc; item += nwarps) {
        const int oc = item / wpc, part = item % wpc;
        const int lx = oc % t.ex, ly = (oc / t.ex) % t.ey, lz = oc / (t.ex * t.ey);
        const int hc = ((lz + 1) * t.hy + (ly + 1)) * t.hx + (lx + 1);
        const int cslot0 = s.hslot[hc];
        const int n_c = s.hslot[hc + 1] - cslot0;
        if (n_c == 0) continue;
        const int cg0 = s.hg[hc];

        // ---- 1. nine runs of candidates (Alg. 3 l.11: the 27 adjacent cells) ----
        int rs = 0, rl = 0;
        if (lane < 9) {
            const int dy = lane % 3 - 1, dz = lane / 3 - 1;
            const int hrow = ((lz + 1 + dz) * t.hy + (ly + 1 + dy)) * t.hx + lx;
            rs = s.hslot[hrow];
            rl = s.hslot[hrow + 3] - rs;
        }
        int incl = rl;
#pragma unroll
        for (int o = 1; o < 16; o <<= 1) {
            const int y = __shfl_up_sync(0xffffffffu, incl, o);
            if (lane >= o) incl += y;
        }
        const int roff = incl - rl;
        const int T = __shfl_sync(0xffffffffu, incl, 8);
        // candidate number of the own cell's first member (run 4 = the own row)
        const int self0 = __shfl_sync(0xffffffffu, roff, 4) + (cslot0 - __shfl_sync(0xffffffffu, rs, 4));

        for (int k0 = 0; k0 < T; k0 += NL_CLIST) {
            const int Tc = min(NL_CLIST, T - k0);
            const int ngroups = (Tc + 31) >> 5;
            __syncwarp();
#pragma unroll
            for (int r = 0; r < 9; r++) {
                const int rs_r = __shfl_sync(0xffffffffu, rs, r), rl_r = __shfl_sync(0xffffffffu, rl, r);
                const int ro_r = __shfl_sync(0xffffffffu, roff, r);
                const int lo = max(ro_r, k0), hi = min(ro_r + rl_r, k0 + Tc);
                for (int v = lo + lane; v < hi; v += 32) clist[v - k0] = (uint16_t)(rs_r + (v - ro_r));
            }
            for (int v = Tc + lane; v < (ngroups << 5); v += 32) clist[v] = 0;   // dummy: never a hit
            __syncwarp();

            // ---- 2. every particle of the cell against every candidate ----
            for (int i0 = part * PPI; i0 < n_c; i0 += wpc * PPI) {
                float px[PPI], py[PPI], pz[PPI];
                int gidx[PPI], cnt0[PPI];
                unsigned hits[PPI];
                const float *rmrow[PPI];
#pragma unroll
                for (int p = 0; p < PPI; p++) {
                    gidx[p] = -1;
                    px[p] = py[p] = pz[p] = -1e18f;
                    cnt0[p] = 0;
                    hits[p] = 0u;
                    rmrow[p] = s_rm2;
                    if (i0 + p < n_c) {
                        const float4 q = stage[cslot0 + i0 + p];  // same address in all lanes: one broadcast
                        px[p] = q.x; py[p] = q.y; pz[p] = q.z;
                        if (TYPED) rmrow[p] = s_rm2 + __float_as_int(q.w) * la.ntypes;
                        gidx[p] = cg0 + i0 + p;
                        if (k0 > 0) cnt0[p] = __ldcg(&nlistn[gidx[p]]);
                    }
                }
                // lane l tests candidates l, l+32, ...; bit gq of hits[p] records candidate 32 gq + l (Alg. 3 l.16-17)
                const uint16_t *const clist_lane = clist + lane;
#pragma unroll 2
                for (int gq = 0; gq < ngroups; gq++) {
                    const float4 e = stage[clist_lane[gq << 5]];
                    const unsigned bit = 1u << gq;
#pragma unroll
                    for (int p = 0; p < PPI; p++) {
                        const float dx = e.x - px[p], dy = e.y - py[p], dz = e.z - pz[p];
                        const float d2 = __fmaf_rn(dz, dz, __fmaf_rn(dy, dy, __fmul_rn(dx, dx)));
                        const float rm = TYPED ? rmrow[p][__float_as_int(e.w)] : rmax2;
                        if (d2 < rm) hits[p] |= bit;   // strict <
                    }
                }
                // i != j: particle i0+p is candidate self0 + i0 + p; drop that one bit
#pragma unroll
                for (int p = 0; p < PPI; p++) {
                    const int ks = self0 + i0 + p - k0;
                    if (ks >= 0 && ks < Tc && (ks & 31) == lane) hits[p] &= ~(1u << (ks >> 5));
                }
                // compact: warp scans of the per-lane hit counts give every lane its positions (l.18-19); the counts of
                // two particles share one scan (16 bits each: a chunk has at most 1024 candidates)
                int at[PPI], total[PPI];
#pragma unroll
                for (int p = 0; p < PPI; p += 2) {
                    const int x = __popc(hits[p]) | (p + 1 < PPI ? __popc(hits[p + 1]) << 16 : 0);
                    int inc = x;
#pragma unroll
                    for (int o = 1; o < 32; o <<= 1) {
                        const int y = __shfl_up_sync(0xffffffffu, inc, o);
                        if (lane >= o) inc += y;
                    }
                    const int tot = __shfl_sync(0xffffffffu, inc, 31), exc = inc - x;   // no borrow: inclusive >= own, field by field
                    at[p] = cnt0[p] + (exc & 0xffff);
                    total[p] = cnt0[p] + (tot & 0xffff);
                    if (p + 1 < PPI) { at[p + 1] = cnt0[p + 1] + (exc >> 16); total[p + 1] = cnt0[p + 1] + (tot >> 16); }
                }
#pragma unroll
                for (int p = 0; p < PPI; p++) {
                    if (gidx[p] < 0) continue;   // warp-uniform
                    uint16_t *row = nlist + (int64_t)gidx[p] * pitch;
                    unsigned hm = hits[p];
                    uint16_t *w = row + at[p];
                    const uint16_t *cl = clist + lane;
                    if (total[p] <= pitch) {       // warp-uniform, the rule: no bound to test per entry
                        while (hm) {
                            const int gq = __ffs(hm) - 1;
                            hm &= hm - 1;
                            *w++ = (uint16_t)(cl[gq << 5] << eshift);
                        }
                    } else {                       // the row overflows: keep what fits, the host grows the rows
                        int a = at[p];
                        while (hm) {
                            const int gq = __ffs(hm) - 1;
                            hm &= hm - 1;
                            if (a < pitch) row[a] = (uint16_t)(cl[gq << 5] << eshift);
                            a++;
                        }
                    }
                    const int nw = min(total[p], pitch);
                    // at least 32 dummy entries end the row: the force kernel stops at the first one it meets
                    // (pad_end is even and the row is 128-byte aligned: one 16-bit store if nw is odd, then 32-bit words)
                    const int pad_end = min(pitch, (nw & ~(ROW_PAD - 1)) + 2 * ROW_PAD);
                    const int e0 = (nw + 1) & ~1;
                    if (lane == 0 && e0 != nw && nw < pad_end) row[nw] = 0;
                    if (e0 + 2 * lane < pad_end) reinterpret_cast<uint32_t *>(row)[(e0 >> 1) + lane] = 0u;
                    if (lane == 0) nlistn[gidx[p]] = nw;                      // l.22
                    wmax = max(wmax, total[p]);
                }
            }
        }
    }
    // longest row needed by this build (may exceed the pitch: overflow)
    if (lane == 0 && wmax > __ldcg(&flags[FL_MAX_NBRS])) {
        atomicMax(&flags[FL_MAX_NBRS], wmax);
        if (wmax > pitch) atomicMax(&flags[FL_OVERFLOWED], wmax);
    }
}

template <int PPI, bool TYPED>
__global__ void __launch_bounds__(TILE_THREADS) nlist_tile_kernel(ListArgs la, const int *__restrict__ pred)
{
    if (pred && *pred == 0) return;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    nlist_tile_body<PPI, TYPED>(la, blockIdx.x, smem_raw);
}

// The whole rebuild in ONE cooperative launch: Algorithm 2 (count, scan, scatter), the reorder into cell
// order (gather) and Algorithm 3, with grid-wide barriers between the phases.  Inside hb_run_nve's graphs
// every step carries the rebuild's kernels as early-exit launches; one launch instead of five takes
// about 4 us off every step (N = 64,000, measured), and the phases lose their launch gaps.
template <int PPI, bool WITH_LIST, bool TYPED>
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
            nlist_tile_body<PPI, TYPED>(la, tile, smem_raw);
            __syncthreads();              // the next tile reuses the staging area (and next_tile)
        }
    }
}

// per-type-pair list cutoffs (tunable nlist_pair_rcut): the table must fit the kernel's shared array
static bool list_typed(const hb_system *h) { return h->tun.nlist_pair_rcut != 0 && h->ntypes > 1 && h->ntypes <= 8; }

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

cudaError_t launch_nlist(hb_system *h, const int *pred, bool copyback)
{
    const size_t smem = nlist_smem_bytes(h);
    const unsigned grid = (unsigned)h->geom.ntiles;
    const ListArgs la = make_list_args(h, copyback);
    cudaError_t e;
#define NL_LAUNCH(PPI, TYPED)                                                                                           \
    e = cudaFuncSetAttribute(nlist_tile_kernel<PPI, TYPED>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_attr(h));    \
    if (e != cudaSuccess) return e;                                                                                     \
    nlist_tile_kernel<PPI, TYPED><<<grid, h->tun.nlist_block, smem, h->stream>>>(la, pred);
    if (list_typed(h)) { NL_LAUNCH(4, true) }      // the typed build comes with four particles per candidate load only
    else switch (h->tun.nlist_ppi) {
        case 1: NL_LAUNCH(1, false) break;
        case 2: NL_LAUNCH(2, false) break;
        default: NL_LAUNCH(4, false) break;
    }
#undef NL_LAUNCH
    h->stats.kernel_launches++;
    return cudaGetLastError();
}

// count + scan + scatter + gather (+ list) in one cooperative launch (see rebuild_coop_kernel)
template <int PPI, bool WITH_LIST, bool TYPED>
static cudaError_t launch_rebuild_coop_t(hb_system *h, const int *pred)
{
    const size_t smem = WITH_LIST ? nlist_smem_bytes(h) : 0;
    cudaError_t e = cudaFuncSetAttribute(rebuild_coop_kernel<PPI, WITH_LIST, TYPED>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_attr(h));
    if (e != cudaSuccess) return e;
    int per_sm = 0;
    e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, rebuild_coop_kernel<PPI, WITH_LIST, TYPED>, TILE_THREADS, smem);
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
    e = cudaLaunchCooperativeKernel((const void *)rebuild_coop_kernel<PPI, WITH_LIST, TYPED>, dim3(grid), dim3(TILE_THREADS), args, smem,
                                    h->stream);
    h->stats.kernel_launches++;
    return e != cudaSuccess ? e : cudaGetLastError();
}

cudaError_t launch_rebuild_coop(hb_system *h, const int *pred, bool with_list)
{
    if (!with_list) return launch_rebuild_coop_t<4, false, false>(h, pred);
    if (list_typed(h)) return launch_rebuild_coop_t<4, true, true>(h, pred);
    switch (h->tun.nlist_ppi) {
        case 1: return launch_rebuild_coop_t<1, true, false>(h, pred);
        case 2: return launch_rebuild_coop_t<2, true, false>(h, pred);
        default: return launch_rebuild_coop_t<4, true, false>(h, pred);
    }
}

// ---- accessors: the list BY TAG as CSR ----
__global__ void nlist_counts_by_tag_kernel(const int *__restrict__ nlistn, const uint32_t *__restrict__ tag, int N,
                                           int *__restrict__ counts)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < N) counts[tag[i]] = nlistn[i];
}

// One block per tile: slot -> storage index through the same tables, then rows -> tags.
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
    for (int q = warp; q < t.nown; q += TILE_THREADS / 32) {
        int gi, slot;
        tile_own(s.d, q, gi, slot);
        const int n = nlistn[gi];
        const int64_t o = row_start[tag[gi]];
        const uint16_t *row = nlist + (int64_t)gi * pitch;
        for (int k = lane; k < n; k += 32) out[o + k] = tag[gidx[row[k] >> g.eshift]];
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
    cudaError_t e = cudaFuncSetAttribute(nlist_fill_by_tag_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_attr(h));
    if (e != cudaSuccess) return e;
    nlist_fill_by_tag_kernel<<<(unsigned)h->geom.ntiles, TILE_THREADS, smem, h->stream>>>(
        h->geom, h->cell_start, h->nlist, h->nlistn, h->row_pitch, h->tag, row_start, out, h->flags);
    return cudaGetLastError();
}
