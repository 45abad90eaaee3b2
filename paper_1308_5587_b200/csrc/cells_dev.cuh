// Device-side pieces of the cell list build (Algorithm 2) and of the reorder into
// cell order, shared by the one-kernel-per-phase launchers in cells.cu and by the cooperative
// rebuild kernel in nlist.cu (all phases and the list build in ONE launch, grid-wide barriers between).
#pragma once
#include "hb_internal.cuh"

// Reading c1.iv: the canonical cell coordinate, binary32, each operation
// rounded separately (intrinsics are never contracted into an FMA).
__device__ __forceinline__ int cell_coord(float x, float b, float s, int m, bool &bad)
{
    const float u = __fmul_rn(__fsub_rn(x, b), s);
    bad = bad || !(u >= -1.0f && u <= (float)m + 1.0f);  // also catches NaN
    int c = (int)floorf(u);
    if (c >= m) c -= m;
    if (c < 0) c += m;
    return min(max(c, 0), m - 1);
}

struct CellArgs {
    const float4 *pos;
    int N;
    float b, s;
    int m;
    int64_t ncells;
    int *cell_count, *cell_local, *cell_start, *cell_id, *cell_rank, *perm, *sums, *flags;
};

// Algorithm 2 l.5-10 for particle i
__device__ __forceinline__ void cell_count_one(const CellArgs &a, int i)
{
    const float4 *pos = a.pos;
    const float b = a.b, s = a.s;
    const int m = a.m;
    int *cell_count = a.cell_count, *cell_id = a.cell_id, *cell_rank = a.cell_rank, *flags = a.flags;
    if (i == 0) flags[FL_MAX_NBRS] = 0;  // a new build starts: the list kernel takes the max again
    const float4 p = pos[i];
    bool bad = false;
    const int cx = cell_coord(p.x, b, s, m, bad);
    const int cy = cell_coord(p.y, b, s, m, bad);
    const int cz = cell_coord(p.z, b, s, m, bad);
    if (bad) flags[FL_BAD] = 1;
    const int c = cx + m * (cy + m * cz);
    cell_id[i] = c;
    cell_rank[i] = atomicAdd(&cell_count[c], 1);
}


// ---- scans ----
constexpr int SCAN_THREADS = 256;
constexpr int SCAN_ITEMS = 8;
constexpr int SCAN_TILE = SCAN_THREADS * SCAN_ITEMS;   // 2048: cell c belongs to scan tile c >> 11
constexpr int SCAN_SHIFT = 11;

__device__ __forceinline__ int block_reduce_sum(int v, int *smem)
{
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    if ((threadIdx.x & 31) == 0) smem[threadIdx.x >> 5] = v;
    __syncthreads();
    int t = 0;
    for (int w = 0; w < SCAN_THREADS / 32; w++) t += smem[w];
    __syncthreads();
    return t;
}

// exclusive scan of this block's SCAN_TILE elements; returns the block total
__device__ __forceinline__ int block_scan_tile(const int *__restrict__ in, int64_t n, int *__restrict__ out, int add, bool zero_in,
                                               int *in_mut, int64_t tile)
{
    __shared__ int warp_off[SCAN_THREADS / 32];
    const int64_t base = tile * SCAN_TILE + (int64_t)threadIdx.x * SCAN_ITEMS;
    int x[SCAN_ITEMS];
    int tsum = 0;
#pragma unroll
    for (int q = 0; q < SCAN_ITEMS; q++) {
        x[q] = (base + q < n) ? in[base + q] : 0;
        tsum += x[q];
    }
    int incl = tsum;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    for (int o = 1; o < 32; o <<= 1) {
        const int y = __shfl_up_sync(0xffffffffu, incl, o);
        if (lane >= o) incl += y;
    }
    if (lane == 31) warp_off[warp] = incl;
    __syncthreads();
    int woff = 0, total = 0;
    for (int w = 0; w < SCAN_THREADS / 32; w++) {
        if (w < warp) woff += warp_off[w];
        total += warp_off[w];
    }
    int run = add + woff + incl - tsum;
#pragma unroll
    for (int q = 0; q < SCAN_ITEMS; q++) {
        if (base + q < n) {
            out[base + q] = run;
            if (zero_in) in_mut[base + q] = 0;
        }
        run += x[q];
    }
    __syncthreads();
    return total;
}

// exclusive scan of nb block totals, in place, by ONE block of SCAN_THREADS threads: a contiguous chunk per thread
__device__ __forceinline__ void scan_sums_in_place(int *__restrict__ sums, int nb, int *smem)
{
    const int per = (nb + SCAN_THREADS - 1) / SCAN_THREADS;
    const int lo = min(nb, (int)threadIdx.x * per), hi = min(nb, lo + per);
    int tsum = 0;
    for (int k = lo; k < hi; k++) tsum += __ldcg(&sums[k]);
    int incl = tsum;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    for (int o = 1; o < 32; o <<= 1) {
        const int y = __shfl_up_sync(0xffffffffu, incl, o);
        if (lane >= o) incl += y;
    }
    if (lane == 31) smem[warp] = incl;
    __syncthreads();
    int woff = 0;
    for (int w = 0; w < warp; w++) woff += smem[w];
    int run = woff + incl - tsum;
    for (int k = lo; k < hi; k++) {
        const int v = __ldcg(&sums[k]);
        sums[k] = run;
        run += v;
    }
}


// perm[cell_start[c] + rank] = i, and the final cell_start for every later reader
__device__ __forceinline__ void cell_scatter_one(const CellArgs &a, int64_t i)
{
    const int N = a.N;
    const int64_t ncells = a.ncells;
    const int *cell_id = a.cell_id, *cell_rank = a.cell_rank, *cell_local = a.cell_local, *boff = a.sums;
    int *perm = a.perm, *cell_start = a.cell_start;
    if (i < N) {
        const int c = cell_id[i];
        perm[cell_local[c] + boff[c >> SCAN_SHIFT] + cell_rank[i]] = (int)i;
    }
    if (i < ncells) cell_start[i] = cell_local[i] + boff[i >> SCAN_SHIFT];
    else if (i == ncells) cell_start[i] = N;
}


struct GatherArgs {
    const float4 *pos, *vel;
    const int *image;
    const uint32_t *tag;
    float4 *pos_o, *vel_o;
    int *image_o;
    uint32_t *tag_o;
    int N;
};

__device__ __forceinline__ void gather_one(const GatherArgs &a, int dst, int src)
{
    a.pos_o[dst] = a.pos[src];
    a.vel_o[dst] = a.vel[src];
    a.image_o[dst] = a.image[src];
    a.image_o[a.N + dst] = a.image[a.N + src];
    a.image_o[2 * (int64_t)a.N + dst] = a.image[2 * (int64_t)a.N + src];
    a.tag_o[dst] = a.tag[src];
}

// One warp per cell: order the members by old index, then move their data.
__device__ __forceinline__ void cell_gather_one(const int *__restrict__ cell_start, const int *__restrict__ perm,
                                                const GatherArgs &a, int do_sort, int64_t c, int lane)
{
    const int start = cell_start[c];
    const int n = cell_start[c + 1] - start;
    if (n == 0) return;
    if (do_sort && n <= 32) {
        const int key = lane < n ? perm[start + lane] : 0x7fffffff;
        int rank = 0;
        for (int k = 0; k < n; k++) rank += (__shfl_sync(0xffffffffu, key, k) < key);
        if (lane < n) gather_one(a, start + rank, key);
    } else if (do_sort && n <= 256) {
        int key[8], rank[8];
#pragma unroll
        for (int q = 0; q < 8; q++) {
            const int k = q * 32 + lane;
            rank[q] = k < n ? 0 : -1;
            key[q] = k < n ? perm[start + k] : 0x7fffffff;
        }
        for (int k = 0; k < n; k++) {
            const int other = perm[start + k];
#pragma unroll
            for (int q = 0; q < 8; q++)
                if (rank[q] >= 0) rank[q] += (other < key[q]);
        }
#pragma unroll
        for (int q = 0; q < 8; q++)
            if (rank[q] >= 0) gather_one(a, start + rank[q], key[q]);
    } else {
        // more than 256 members (or cell_sort = 0): keep the atomic order (valid, not reproducible)
        for (int k = lane; k < n; k += 32) gather_one(a, start + k, perm[start + k]);
    }
}

static inline CellArgs make_cell_args(const hb_system *h)
{
    CellArgs a{};
    a.pos = h->pos();
    a.N = (int)h->N;
    a.b = -0.5f * h->L;
    a.s = (float)h->m / h->L;
    a.m = h->m;
    a.ncells = h->ncells;
    a.cell_count = h->cell_count; a.cell_local = h->cell_local; a.cell_start = h->cell_start;
    a.cell_id = h->cell_id; a.cell_rank = h->cell_rank; a.perm = h->perm; a.sums = h->scan_sums; a.flags = h->flags;
    return a;
}

// live arrays -> scratch set (positions into pos_build)
static inline GatherArgs make_gather_args(const hb_system *h)
{
    return GatherArgs{h->pos(), h->vel, h->image, h->tag, h->pos_build, h->vel2, h->image2, h->tag2, (int)h->N};
}
