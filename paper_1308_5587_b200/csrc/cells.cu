// Cell list (Algorithm 2) as a CSR structure:
//   cell_count[c]  <- atomicAdd, one per particle (the paper's celln / atomicInc, line 10)
//   cell_start     <- exclusive scan of cell_count
//   cell_xyzi      <- (R, i) written at cell_start[c] + n     (the paper's celldata, line 11)
// CSR instead of the paper's fixed-capacity celldata[n, cx, cy, cz]: no per-cell
// capacity, no overflow path, and the members of x-adjacent cells are contiguous.
// An optional pass orders the members of each cell by particle index so that
// the neighbor list (and with it every fp32 sum) is reproducible run to run.
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

__global__ void __launch_bounds__(256) cell_bin_kernel(const float4 *__restrict__ pos, int N, float b, float s, int m,
                                                       int *__restrict__ cell_count, int *__restrict__ cell_rank,
                                                       int *__restrict__ flags, const int *__restrict__ pred)
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
    cell_rank[i] = atomicAdd(&cell_count[c], 1);
}

__global__ void __launch_bounds__(256) cell_scatter_kernel(const float4 *__restrict__ pos, int N, float b, float s, int m,
                                                           const int *__restrict__ cell_start,
                                                           const int *__restrict__ cell_rank,
                                                           float4 *__restrict__ cell_xyzi, float4 *__restrict__ pos_build,
                                                           const int *__restrict__ pred)
{
    if (pred && *pred == 0) return;
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= N) return;
    const float4 p = pos[i];
    bool bad = false;
    const int cx = cell_coord(p.x, b, s, m, bad);
    const int cy = cell_coord(p.y, b, s, m, bad);
    const int cz = cell_coord(p.z, b, s, m, bad);
    const int c = cx + m * (cy + m * cz);
    cell_xyzi[cell_start[c] + cell_rank[i]] = make_float4(p.x, p.y, p.z, __int_as_float(i));
    pos_build[i] = p;  // remembered for the r_buff/2 rule (reading c3)
}

// One warp per cell: order the members by particle index.
__global__ void __launch_bounds__(128) cell_sort_kernel(const int *__restrict__ cell_start, int64_t ncells,
                                                        float4 *__restrict__ cell_xyzi, const int *__restrict__ pred)
{
    if (pred && *pred == 0) return;
    const int64_t c = (int64_t)blockIdx.x * 4 + (threadIdx.x >> 5);
    if (c >= ncells) return;
    const int lane = threadIdx.x & 31;
    const int start = cell_start[c];
    const int n = cell_start[c + 1] - start;
    if (n <= 1) return;
    if (n <= 32) {
        float4 e = make_float4(0, 0, 0, 0);
        int key = 0x7fffffff;
        if (lane < n) {
            e = cell_xyzi[start + lane];
            key = __float_as_int(e.w);
        }
        int rank = 0;
        for (int k = 0; k < n; k++) rank += (__shfl_sync(0xffffffffu, key, k) < key);
        __syncwarp();
        if (lane < n) cell_xyzi[start + rank] = e;
    } else if (n <= 256) {
        float4 e[8];
        int rank[8];
#pragma unroll
        for (int q = 0; q < 8; q++) {
            rank[q] = -1;
            const int k = q * 32 + lane;
            if (k < n) {
                e[q] = cell_xyzi[start + k];
                rank[q] = 0;
            }
        }
        for (int k = 0; k < n; k++) {
            const int other = __float_as_int(cell_xyzi[start + k].w);
#pragma unroll
            for (int q = 0; q < 8; q++)
                if (rank[q] >= 0) rank[q] += (other < __float_as_int(e[q].w));
        }
        __syncwarp();
#pragma unroll
        for (int q = 0; q < 8; q++)
            if (rank[q] >= 0) cell_xyzi[start + rank[q]] = e[q];
    }
    // cells with more than 256 members keep the atomic order (valid, not reproducible)
}

// ---- exclusive scan of n ints in two kernels: block sums, then block-local scans ----
constexpr int SCAN_THREADS = 256;
constexpr int SCAN_ITEMS = 8;
constexpr int SCAN_TILE = SCAN_THREADS * SCAN_ITEMS;

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

__global__ void __launch_bounds__(SCAN_THREADS) scan_sums_kernel(const int *__restrict__ in, int64_t n, int *__restrict__ sums,
                                                                 const int *__restrict__ pred)
{
    if (pred && *pred == 0) return;
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
                                                                  int *__restrict__ out, const int *__restrict__ pred)
{
    if (pred && *pred == 0) return;
    __shared__ int smem[SCAN_THREADS / 32];
    __shared__ int warp_off[SCAN_THREADS / 32];
    // offset of this block = sum of the earlier blocks' sums
    int v = 0;
    for (int k = threadIdx.x; k < (int)blockIdx.x; k += SCAN_THREADS) v += sums[k];
    const int block_off = block_reduce_sum(v, smem);
    // each thread owns SCAN_ITEMS consecutive elements
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
    int woff = 0;
    for (int w = 0; w < warp; w++) woff += warp_off[w];
    int run = block_off + woff + incl - tsum;
#pragma unroll
    for (int q = 0; q < SCAN_ITEMS; q++) {
        if (base + q < n) out[base + q] = run;
        run += x[q];
        if (base + q == n - 1) out[n] = run;  // total
    }
}

__global__ void clear_ints_kernel(int *__restrict__ p, int64_t n, const int *__restrict__ pred)
{
    if (pred && *pred == 0) return;
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) p[i] = 0;
}

cudaError_t launch_cell_clear(hb_system *h, const int *pred)
{
    clear_ints_kernel<<<(unsigned)cdiv(h->ncells, 256), 256, 0, h->stream>>>(h->cell_count, h->ncells, pred);
    h->stats.kernel_launches++;
    return cudaGetLastError();
}

cudaError_t launch_cell_bin(hb_system *h, const int *pred)
{
    const float b = -0.5f * h->L;
    const float s = (float)h->m / h->L;
    cell_bin_kernel<<<(unsigned)cdiv(h->N, 256), 256, 0, h->stream>>>(h->pos, (int)h->N, b, s, h->m, h->cell_count,
                                                                      h->cell_rank, h->flags, pred);
    h->stats.kernel_launches++;
    return cudaGetLastError();
}

cudaError_t launch_scan_exclusive(hb_system *h, const int *in, int *out, int64_t n, int *tmp, const int *pred)
{
    const unsigned nb = (unsigned)cdiv(n, SCAN_TILE);
    scan_sums_kernel<<<nb, SCAN_THREADS, 0, h->stream>>>(in, n, tmp, pred);
    scan_apply_kernel<<<nb, SCAN_THREADS, 0, h->stream>>>(in, n, tmp, out, pred);
    h->stats.kernel_launches += 2;
    return cudaGetLastError();
}

cudaError_t launch_cell_scatter(hb_system *h, const int *pred)
{
    const float b = -0.5f * h->L;
    const float s = (float)h->m / h->L;
    cell_scatter_kernel<<<(unsigned)cdiv(h->N, 256), 256, 0, h->stream>>>(h->pos, (int)h->N, b, s, h->m, h->cell_start,
                                                                          h->cell_rank, h->cell_xyzi, h->pos_build, pred);
    h->stats.kernel_launches++;
    return cudaGetLastError();
}

cudaError_t launch_cell_sort(hb_system *h, const int *pred)
{
    cell_sort_kernel<<<(unsigned)cdiv(h->ncells, 4), 128, 0, h->stream>>>(h->cell_start, h->ncells, h->cell_xyzi, pred);
    h->stats.kernel_launches++;
    return cudaGetLastError();
}

// accessor: tags of the cell members in CSR order
__global__ void cell_tags_kernel(const float4 *__restrict__ cell_xyzi, const uint32_t *__restrict__ tag, int N,
                                 uint32_t *__restrict__ out)
{
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k < N) out[k] = tag[__float_as_int(cell_xyzi[k].w)];
}

cudaError_t launch_cell_tags(hb_system *h, uint32_t *out)
{
    cell_tags_kernel<<<(unsigned)cdiv(h->N, 256), 256, 0, h->stream>>>(h->cell_xyzi, h->tag, (int)h->N, out);
    return cudaGetLastError();
}
