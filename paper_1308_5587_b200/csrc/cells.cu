// Cell list (Algorithm 2) as a CSR structure, plus the reorder of
// the particle data into cell order that the tile kernels rely on:
//   cell_count[c]  <- atomicAdd, one per particle (the paper's celln / atomicInc, line 10)
//   cell_start     <- exclusive scan of cell_count
//   perm           <- old index i written at cell_start[c] + n   (the paper's celldata, line 11)
//   gather         <- members of each cell ordered by old index (reproducible run to run), then
//                     (R, v, image, tag) moved so that particle k of the new storage order lies
//                     in the cell whose CSR range holds k.  The paper's celldata stores (R, i)
//                     copies per cell; here the particle arrays THEMSELVES are the cell data, and
//                     the members of x-adjacent cells are one contiguous run.
// CSR instead of the paper's fixed-capacity celldata[n, cx, cy, cz]: no per-cell capacity, no
// overflow path.  Four launches: count, scan (one kernel: block-local scans, the last block to
// finish scans the block sums), scatter (+ final cell_start), gather.
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

__global__ void __launch_bounds__(256) cell_count_kernel(const float4 *__restrict__ pos, int N, float b, float s, int m,
                                                         int *__restrict__ cell_count, int *__restrict__ cell_id,
                                                         int *__restrict__ cell_rank, int *__restrict__ flags,
                                                         const int *__restrict__ pred)
{
    if (pred && *pred == 0) return;
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= N) return;
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
                                               int *in_mut)
{
    __shared__ int warp_off[SCAN_THREADS / 32];
    const int64_t base = (int64_t)blockIdx.x * SCAN_TILE + (int64_t)threadIdx.x * SCAN_ITEMS;
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

// One launch: every block scans its tile of cell_count into cell_local and clears cell_count for the
// next build; the last block to finish turns the block totals into block offsets (in place).
__global__ void __launch_bounds__(SCAN_THREADS) cell_scan_kernel(int *__restrict__ cell_count, int64_t ncells,
                                                                 int *__restrict__ cell_local, int *__restrict__ sums,
                                                                 int *__restrict__ flags, const int *__restrict__ pred)
{
    if (pred && *pred == 0) return;
    __shared__ int is_last;
    __shared__ int smem[SCAN_THREADS / 32];
    const int total = block_scan_tile(cell_count, ncells, cell_local, 0, true, cell_count);
    if (threadIdx.x == 0) {
        sums[blockIdx.x] = total;
        __threadfence();
        const int ticket = atomicAdd(&flags[FL_SCAN_CTR], 1);
        is_last = ticket == (int)gridDim.x - 1;
    }
    __syncthreads();
    if (!is_last) return;
    __threadfence();
    // exclusive scan of gridDim.x totals by one block: a contiguous chunk per thread
    const int nb = gridDim.x;
    const int per = (nb + SCAN_THREADS - 1) / SCAN_THREADS;
    const int lo = min(nb, (int)threadIdx.x * per), hi = min(nb, lo + per);
    int tsum = 0;
    for (int k = lo; k < hi; k++) tsum += __ldcg(&sums[k]);
    // block-wide exclusive prefix of tsum
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
    if (threadIdx.x == 0) flags[FL_SCAN_CTR] = 0;
}

// perm[cell_start[c] + rank] = i, and the final cell_start for every later reader
__global__ void __launch_bounds__(256) cell_scatter_kernel(int N, int64_t ncells, const int *__restrict__ cell_id,
                                                           const int *__restrict__ cell_rank,
                                                           const int *__restrict__ cell_local, const int *__restrict__ boff,
                                                           int *__restrict__ perm, int *__restrict__ cell_start,
                                                           const int *__restrict__ pred)
{
    if (pred && *pred == 0) return;
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
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
__global__ void __launch_bounds__(128) cell_gather_kernel(const int *__restrict__ cell_start, int64_t ncells,
                                                          const int *__restrict__ perm, GatherArgs a, int do_sort,
                                                          const int *__restrict__ pred)
{
    if (pred && *pred == 0) return;
    const int64_t c = (int64_t)blockIdx.x * 4 + (threadIdx.x >> 5);
    if (c >= ncells) return;
    const int lane = threadIdx.x & 31;
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

// scratch set -> live arrays (used when no list kernel follows; the list kernel does this per tile)
__global__ void __launch_bounds__(256) cell_copyback_kernel(GatherArgs a, uint32_t *__restrict__ rtag, const int *__restrict__ pred)
{
    if (pred && *pred == 0) return;
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= a.N) return;
    gather_one(a, i, i);
    rtag[a.tag[i]] = i;
}

cudaError_t launch_cell_count(hb_system *h, const int *pred)
{
    const float b = -0.5f * h->L;
    const float s = (float)h->m / h->L;
    cell_count_kernel<<<(unsigned)cdiv(h->N, 256), 256, 0, h->stream>>>(h->pos(), (int)h->N, b, s, h->m, h->cell_count,
                                                                        h->cell_id, h->cell_rank, h->flags, pred);
    h->stats.kernel_launches++;
    return cudaGetLastError();
}

cudaError_t launch_cell_scan(hb_system *h, const int *pred)
{
    const unsigned nb = (unsigned)cdiv(h->ncells, SCAN_TILE);
    cell_scan_kernel<<<nb, SCAN_THREADS, 0, h->stream>>>(h->cell_count, h->ncells, h->cell_local, h->scan_sums, h->flags, pred);
    h->stats.kernel_launches++;
    return cudaGetLastError();
}

cudaError_t launch_cell_scatter(hb_system *h, const int *pred)
{
    const int64_t n = std::max<int64_t>(h->N, h->ncells + 1);
    cell_scatter_kernel<<<(unsigned)cdiv(n, 256), 256, 0, h->stream>>>((int)h->N, h->ncells, h->cell_id, h->cell_rank,
                                                                       h->cell_local, h->scan_sums, h->perm, h->cell_start, pred);
    h->stats.kernel_launches++;
    return cudaGetLastError();
}

cudaError_t launch_cell_gather(hb_system *h, const int *pred)
{
    GatherArgs a{h->pos(), h->vel, h->image, h->tag, h->pos_build, h->vel2, h->image2, h->tag2, (int)h->N};
    cell_gather_kernel<<<(unsigned)cdiv(h->ncells, 4), 128, 0, h->stream>>>(h->cell_start, h->ncells, h->perm, a,
                                                                            h->tun.cell_sort, pred);
    h->stats.kernel_launches++;
    return cudaGetLastError();
}

cudaError_t launch_cell_copyback(hb_system *h, const int *pred)
{
    GatherArgs a{h->pos_build, h->vel2, h->image2, h->tag2, h->pos(), h->vel, h->image, h->tag, (int)h->N};
    cell_copyback_kernel<<<(unsigned)cdiv(h->N, 256), 256, 0, h->stream>>>(a, h->rtag, pred);
    h->stats.kernel_launches++;
    return cudaGetLastError();
}

// ---- generic exclusive scan of n ints in two kernels (used by the radix sort): block sums, then block-local scans ----
__global__ void __launch_bounds__(SCAN_THREADS) scan_sums_kernel(const int *__restrict__ in, int64_t n, int *__restrict__ sums)
{
    __shared__ int smem[SCAN_THREADS / 32];
    const int64_t base = (int64_t)blockIdx.x * SCAN_TILE;
    int v = 0;
#pragma unroll
    for (int q = 0; q < SCAN_ITEMS; q++) {
        const int64_t k = base + q * SCAN_THREADS + threadIdx.x;
        if (k < n) v += in[k];
    }
    const int t = block_reduce_sum(v, smem);
    if (threadIdx.x == 0) sums[blockIdx.x] = t;
}

__global__ void __launch_bounds__(SCAN_THREADS) scan_apply_kernel(const int *__restrict__ in, int64_t n, const int *__restrict__ sums,
                                                                  int *__restrict__ out)
{
    __shared__ int smem[SCAN_THREADS / 32];
    // offset of this block = sum of the earlier blocks' sums
    int v = 0;
    for (int k = threadIdx.x; k < (int)blockIdx.x; k += SCAN_THREADS) v += sums[k];
    const int block_off = block_reduce_sum(v, smem);
    const int total = block_scan_tile(in, n, out, block_off, false, nullptr);
    if (blockIdx.x == gridDim.x - 1 && threadIdx.x == 0) out[n] = block_off + total;
}

cudaError_t launch_scan_exclusive(hb_system *h, const int *in, int *out, int64_t n, int *tmp)
{
    const unsigned nb = (unsigned)cdiv(n, SCAN_TILE);
    scan_sums_kernel<<<nb, SCAN_THREADS, 0, h->stream>>>(in, n, tmp);
    scan_apply_kernel<<<nb, SCAN_THREADS, 0, h->stream>>>(in, n, tmp, out);
    h->stats.kernel_launches += 2;
    return cudaGetLastError();
}
