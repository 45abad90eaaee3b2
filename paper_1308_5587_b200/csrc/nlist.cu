// Neighbor list (Algorithm 3), re-designed for sm_100a.
//
// The paper runs one thread per particle and names the resulting scattered,
// unsynchronised row writes "a big bottleneck" that "GF100 does not have enough
// shared memory to regularize".  Here ONE WARP OWNS ONE CELL:
//   1. lanes 0..26 look up the 27 adjacent cells (on the fly, no celladj table:
//      PAPER.md:187 stored it to save registers; a warp has lanes to spare) and
//      the periodic shift of each, and a warp scan turns their occupancies into
//      offsets;
//   2. the warp stages the candidates (R_j + shift, j) of all 27 cells, compacted,
//      in shared memory -- coalesced float4 reads of the CSR cell list;
//   3. for every particle i of the cell (PPI at a time, so each shared-memory
//      candidate load serves PPI distance tests) lane l tests candidates l, l+32,
//      ... and records the hits as bits of a register; one warp prefix sum of the
//      per-lane __popc counts then gives every lane its slots, the row is
//      assembled in shared memory and flushed with coalesced stores into a
//      row-major, 128-byte aligned, padded list.  (Round-1 ncu: a __ballot_sync
//      per 32 tests cost 27 instructions per test group; the bit mask costs 8.)
// The periodic shift is applied once to the staged copy, so no minimum-image
// arithmetic is left in the inner loop, and x_j + shift is exact or within one
// ulp of x (hard part 3).
#include "hb_internal.cuh"

constexpr int NL_WARPS = 4;

__host__ __device__ inline size_t nlist_warp_smem(int cap, int ppi, int pitch)
{
    return (size_t)cap * 16 + (size_t)ppi * pitch * 4 + 32 * 4 /*offs*/ + 32 * 4 /*astart*/ + 96 * 4 /*shift*/;
}

size_t nlist_smem_bytes(const hb_system *h)
{
    return NL_WARPS * nlist_warp_smem(h->tun.nlist_cap, h->tun.nlist_ppi, h->row_pitch);
}

template <int PPI>
__global__ void __launch_bounds__(NL_WARPS * 32)
nlist_kernel(const int *__restrict__ cell_start, const float4 *__restrict__ cell_xyzi, int m, int64_t ncells, float L,
             float rmax2, int cap, int pitch, int *__restrict__ nlist, int *__restrict__ nlistn, int *__restrict__ flags,
             const int *__restrict__ pred)
{
    if (pred && *pred == 0) return;
    if (blockIdx.x == 0 && threadIdx.x == 0) flags[FL_BUILDS] += 1;

    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    unsigned char *wbase = smem_raw + (size_t)warp * nlist_warp_smem(cap, PPI, pitch);
    float4 *cand = reinterpret_cast<float4 *>(wbase);
    int *rows = reinterpret_cast<int *>(wbase + (size_t)cap * 16);
    int *offs = rows + PPI * pitch;
    int *astart = offs + 32;
    float *shift = reinterpret_cast<float *>(astart + 32);

    const int64_t c = (int64_t)blockIdx.x * NL_WARPS + warp;
    if (c >= ncells) return;
    const int cstart = cell_start[c];
    const int n_c = cell_start[c + 1] - cstart;
    if (n_c == 0) return;

    // ---- 1. the 27 adjacent cells, their occupancies and periodic shifts ----
    const int cx = (int)(c % m), cy = (int)((c / m) % m), cz = (int)(c / ((int64_t)m * m));
    int a_start = 0, a_cnt = 0;
    float sx = 0.f, sy = 0.f, sz = 0.f;
    if (lane < 27) {
        int nx = cx + lane % 3 - 1, ny = cy + (lane / 3) % 3 - 1, nz = cz + lane / 9 - 1;
        if (nx < 0) { nx += m; sx = -L; } else if (nx >= m) { nx -= m; sx = L; }
        if (ny < 0) { ny += m; sy = -L; } else if (ny >= m) { ny -= m; sy = L; }
        if (nz < 0) { nz += m; sz = -L; } else if (nz >= m) { nz -= m; sz = L; }
        const int64_t nc = nx + (int64_t)m * (ny + (int64_t)m * nz);
        a_start = cell_start[nc];
        a_cnt = cell_start[nc + 1] - a_start;
    }
    int incl = a_cnt;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const int y = __shfl_up_sync(0xffffffffu, incl, o);
        if (lane >= o) incl += y;
    }
    const int T = __shfl_sync(0xffffffffu, incl, 31);
    const int self0 = __shfl_sync(0xffffffffu, incl - a_cnt, 13);  // candidate number of the own cell's first member
    offs[lane] = incl - a_cnt;  // lanes 27..31 hold T
    astart[lane] = a_start;
    shift[3 * lane + 0] = sx;
    shift[3 * lane + 1] = sy;
    shift[3 * lane + 2] = sz;
    __syncwarp();

    int wmax = 0;

    for (int k0 = 0; k0 < T; k0 += cap) {
        const int Tc = min(cap, T - k0);
        const int ngroups = (Tc + 31) >> 5;
        // ---- 2. stage the candidates, compacted, shifted to their periodic image; pad to whole groups ----
        for (int k = lane; k < (ngroups << 5); k += 32) {
            float4 e = make_float4(3e30f, 3e30f, 3e30f, __int_as_float(-2));
            if (k < Tc) {
                const int kk = k0 + k;
                int a = 0;
#pragma unroll
                for (int s = 16; s > 0; s >>= 1)
                    if (offs[a + s] <= kk) a += s;
                e = cell_xyzi[astart[a] + (kk - offs[a])];
                e.x += shift[3 * a + 0];
                e.y += shift[3 * a + 1];
                e.z += shift[3 * a + 2];
            }
            cand[k] = e;
        }
        __syncwarp();

        // ---- 3. every particle of the cell against every candidate ----
        for (int i0 = 0; i0 < n_c; i0 += PPI) {
            float px[PPI], py[PPI], pz[PPI];
            int pidx[PPI], cnt0[PPI];
            unsigned hits[PPI];
#pragma unroll
            for (int p = 0; p < PPI; p++) {
                pidx[p] = -1;
                px[p] = py[p] = pz[p] = 1e30f;
                cnt0[p] = 0;
                hits[p] = 0u;
                if (i0 + p < n_c) {
                    const float4 q = cell_xyzi[cstart + i0 + p];  // same address in all lanes: one broadcast
                    px[p] = q.x; py[p] = q.y; pz[p] = q.z;
                    pidx[p] = __float_as_int(q.w);
                    if (k0 > 0) cnt0[p] = __ldcg(&nlistn[pidx[p]]);
                }
            }
            // lane l tests candidates l, l+32, ...; bit g of hits[p] records candidate 32 g + l (Alg. 3 l.16-17)
#pragma unroll 2
            for (int g = 0; g < ngroups; g++) {
                const float4 e = cand[(g << 5) + lane];
                const unsigned bit = 1u << g;
#pragma unroll
                for (int p = 0; p < PPI; p++) {
                    const float dx = e.x - px[p], dy = e.y - py[p], dz = e.z - pz[p];
                    const float d2 = __fmaf_rn(dz, dz, __fmaf_rn(dy, dy, __fmul_rn(dx, dx)));
                    if (d2 < rmax2) hits[p] |= bit;   // strict <
                }
            }
            // i != j: particle i0+p is candidate self0 + i0 + p; drop that one bit
#pragma unroll
            for (int p = 0; p < PPI; p++) {
                const int ks = self0 + i0 + p - k0;
                if (ks >= 0 && ks < Tc && (ks & 31) == lane) hits[p] &= ~(1u << (ks >> 5));
            }
            // compact: warp scan of the per-lane hit counts gives every lane its slots (l.18-19)
#pragma unroll
            for (int p = 0; p < PPI; p++) {
                if (pidx[p] < 0) continue;   // warp-uniform
                const int cn = __popc(hits[p]);
                int inc = cn;
#pragma unroll
                for (int o = 1; o < 32; o <<= 1) {
                    const int y = __shfl_up_sync(0xffffffffu, inc, o);
                    if (lane >= o) inc += y;
                }
                const int total = cnt0[p] + __shfl_sync(0xffffffffu, inc, 31);
                int slot = cnt0[p] + inc - cn;
                unsigned hm = hits[p];
                while (hm) {
                    const int g = __ffs(hm) - 1;
                    hm &= hm - 1;
                    if (slot < pitch) rows[p * pitch + slot] = __float_as_int(cand[(g << 5) + lane].w);
                    slot++;
                }
                __syncwarp();
                const int nw = min(total, pitch);
                int *row = nlist + (int64_t)pidx[p] * pitch;
                for (int k = cnt0[p] + lane; k < nw; k += 32) row[k] = rows[p * pitch + k];   // coalesced 128 B stores
                if (lane == 0) nlistn[pidx[p]] = nw;                                            // l.22
                wmax = max(wmax, total);
            }
            __syncwarp();
        }
    }
    // longest row needed by this build (may exceed the pitch: overflow)
    if (lane == 0 && wmax > __ldcg(&flags[FL_MAX_NBRS])) {
        atomicMax(&flags[FL_MAX_NBRS], wmax);
        if (wmax > pitch) atomicMax(&flags[FL_OVERFLOWED], wmax);
    }
}

cudaError_t launch_nlist(hb_system *h, const int *pred)
{
    const size_t smem = nlist_smem_bytes(h);
    const unsigned grid = (unsigned)cdiv(h->ncells, NL_WARPS);
    const float rmax2 = h->r_max * h->r_max;
    cudaError_t e;
#define NL_LAUNCH(PPI)                                                                                              \
    e = cudaFuncSetAttribute(nlist_kernel<PPI>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);            \
    if (e != cudaSuccess) return e;                                                                                 \
    nlist_kernel<PPI><<<grid, NL_WARPS * 32, smem, h->stream>>>(h->cell_start, h->cell_xyzi, h->m, h->ncells, h->L, \
                                                                rmax2, h->tun.nlist_cap, h->row_pitch, h->nlist,    \
                                                                h->nlistn, h->flags, pred);
    switch (h->tun.nlist_ppi) {
        case 1: NL_LAUNCH(1) break;
        case 2: NL_LAUNCH(2) break;
        default: NL_LAUNCH(4) break;
    }
#undef NL_LAUNCH
    h->stats.kernel_launches++;
    return cudaGetLastError();
}

// ---- accessors: the list BY TAG as CSR ----
__global__ void nlist_counts_by_tag_kernel(const int *__restrict__ nlistn, const uint32_t *__restrict__ tag, int N,
                                           int *__restrict__ counts)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < N) counts[tag[i]] = nlistn[i];
}

__global__ void nlist_fill_by_tag_kernel(const int *__restrict__ nlist, const int *__restrict__ nlistn, int pitch,
                                         const uint32_t *__restrict__ tag, int N, const int64_t *__restrict__ row_start,
                                         uint32_t *__restrict__ out)
{
    const int i = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
    if (i >= N) return;
    const int lane = threadIdx.x & 31;
    const int n = nlistn[i];
    const int64_t o = row_start[tag[i]];
    for (int k = lane; k < n; k += 32) out[o + k] = tag[nlist[(int64_t)i * pitch + k]];
}

cudaError_t launch_nlist_counts_by_tag(hb_system *h, int *counts)
{
    nlist_counts_by_tag_kernel<<<(unsigned)cdiv(h->N, 256), 256, 0, h->stream>>>(h->nlistn, h->tag, (int)h->N, counts);
    return cudaGetLastError();
}

cudaError_t launch_nlist_fill_by_tag(hb_system *h, const int64_t *row_start, uint32_t *out)
{
    nlist_fill_by_tag_kernel<<<(unsigned)cdiv(h->N, 8), 256, 0, h->stream>>>(h->nlist, h->nlistn, h->row_pitch, h->tag,
                                                                             (int)h->N, row_start, out);
    return cudaGetLastError();
}
