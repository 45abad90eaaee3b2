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
#include "cells_dev.cuh"

__global__ void __launch_bounds__(256) cell_count_kernel(CellArgs a, const int *__restrict__ pred)
{
    if (pred && *pred == 0) return;
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < a.N) cell_count_one(a, i);
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
    const int total = block_scan_tile(cell_count, ncells, cell_local, 0, true, cell_count, blockIdx.x);
    if (threadIdx.x == 0) {
        sums[blockIdx.x] = total;
        __threadfence();
        const int ticket = atomicAdd(&flags[FL_SCAN_CTR], 1);
        is_last = ticket == (int)gridDim.x - 1;
    }
    __syncthreads();
    if (!is_last) return;
    __threadfence();
    scan_sums_in_place(sums, gridDim.x, smem);
    if (threadIdx.x == 0) flags[FL_SCAN_CTR] = 0;
}

__global__ void __launch_bounds__(256) cell_scatter_kernel(CellArgs a, const int *__restrict__ pred)
{
    if (pred && *pred == 0) return;
    cell_scatter_one(a, (int64_t)blockIdx.x * blockDim.x + threadIdx.x);
}

__global__ void __launch_bounds__(128) cell_gather_kernel(const int *__restrict__ cell_start, int64_t ncells,
                                                          const int *__restrict__ perm, GatherArgs a, int do_sort,
                                                          const int *__restrict__ pred)
{
    if (pred && *pred == 0) return;
    const int64_t c = (int64_t)blockIdx.x * 4 + (threadIdx.x >> 5);
    if (c < ncells) cell_gather_one(cell_start, perm, a, do_sort, c, threadIdx.x & 31);
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
    cell_count_kernel<<<(unsigned)cdiv(h->N, 256), 256, 0, h->stream>>>(make_cell_args(h), pred);
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
    cell_scatter_kernel<<<(unsigned)cdiv(n, 256), 256, 0, h->stream>>>(make_cell_args(h), pred);
    h->stats.kernel_launches++;
    return cudaGetLastError();
}

cudaError_t launch_cell_gather(hb_system *h, const int *pred)
{
    const GatherArgs a = make_gather_args(h);
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
    const int total = block_scan_tile(in, n, out, block_off, false, nullptr, blockIdx.x);
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
