// Space-filling-curve particle sort (the paper's "SFCPACK sort"),
// on the GPU -- the paper still ran it on the host and called it "a serial
// bottleneck".  Reading c8: Hilbert curve (Skilling's transpose algorithm) on a
// 2^8 grid per axis, ties in tag order (the key pass walks the particles by tag,
// the radix sort is stable), so the result does not depend on the storage order.
//   keys   : one thread per particle
//   sort   : hand-written LSD radix sort of (key, index), 8 bits per pass; a warp
//            owns a tile of 32 x RS_ITEMS keys; __match_any_sync gives each key its
//            stable rank among equal digits
//   gather : every per-particle array permuted into the scratch set (positions into pos_build,
//            which the next list build overwrites anyway)
#include "hb_internal.cuh"

constexpr int SFC_BITS = 8;

__device__ __forceinline__ uint32_t hilbert_key(uint32_t x0, uint32_t x1, uint32_t x2)
{
    uint32_t X[3] = {x0, x1, x2};
    const uint32_t M = 1u << (SFC_BITS - 1);
    for (uint32_t Q = M; Q > 1; Q >>= 1) {
        const uint32_t P = Q - 1;
#pragma unroll
        for (int i = 0; i < 3; i++) {
            if (X[i] & Q) X[0] ^= P;
            else { const uint32_t t = (X[0] ^ X[i]) & P; X[0] ^= t; X[i] ^= t; }
        }
    }
    X[1] ^= X[0];
    X[2] ^= X[1];
    uint32_t t = 0;
    for (uint32_t Q = M; Q > 1; Q >>= 1)
        if (X[2] & Q) t ^= Q - 1;
    X[0] ^= t; X[1] ^= t; X[2] ^= t;
    uint32_t key = 0;
#pragma unroll
    for (int b = SFC_BITS - 1; b >= 0; b--) {
        key = (key << 1) | ((X[0] >> b) & 1u);
        key = (key << 1) | ((X[1] >> b) & 1u);
        key = (key << 1) | ((X[2] >> b) & 1u);
    }
    return key;
}

__device__ __forceinline__ uint32_t grid_coord(float x, float b, float s)
{
    const int G = 1 << SFC_BITS;
    int g = (int)floorf(__fmul_rn(__fsub_rn(x, b), s));
    if (g >= G) g -= G;
    if (g < 0) g += G;
    return (uint32_t)min(max(g, 0), G - 1);
}

__global__ void sfc_keys_kernel(const float4 *__restrict__ pos, const uint32_t *__restrict__ rtag, int N, float b, float s,
                                uint32_t *__restrict__ keys, uint32_t *__restrict__ perm)
{
    const int t = blockIdx.x * blockDim.x + threadIdx.x;   // tag
    if (t >= N) return;
    const uint32_t i = rtag[t];
    const float4 p = pos[i];
    keys[t] = hilbert_key(grid_coord(p.x, b, s), grid_coord(p.y, b, s), grid_coord(p.z, b, s));
    perm[t] = i;
}

cudaError_t launch_sfc_keys(hb_system *h)
{
    const float b = -0.5f * h->L;
    const float s = (float)(1 << SFC_BITS) / h->L;
    sfc_keys_kernel<<<(unsigned)cdiv(h->N, 256), 256, 0, h->stream>>>(h->pos(), h->rtag, (int)h->N, b, s, h->keys, h->sperm);
    h->stats.kernel_launches++;
    return cudaGetLastError();
}

// ---- LSD radix sort, 8 bits per pass ----
constexpr int RS_ITEMS = 16;               // keys per lane
constexpr int RS_TILE = 32 * RS_ITEMS;     // keys per warp
constexpr int RS_WARPS = 4;

// counts[d * ntiles + tile] = number of keys of the tile whose digit is d
__global__ void __launch_bounds__(RS_WARPS * 32)
radix_hist_kernel(const uint32_t *__restrict__ keys, int N, int shift, int ntiles, int *__restrict__ counts)
{
    __shared__ int hist[RS_WARPS][256];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int tile = blockIdx.x * RS_WARPS + warp;
    for (int d = lane; d < 256; d += 32) hist[warp][d] = 0;
    __syncwarp();
    if (tile < ntiles) {
        const int base = tile * RS_TILE;
        for (int q = 0; q < RS_ITEMS; q++) {
            const int k = base + q * 32 + lane;
            if (k < N) atomicAdd(&hist[warp][(keys[k] >> shift) & 255u], 1);
        }
        __syncwarp();
        for (int d = lane; d < 256; d += 32) counts[(int64_t)d * ntiles + tile] = hist[warp][d];
    }
}

// offsets = exclusive scan of counts (digit-major), so offsets[d * ntiles + tile] is
// where the tile's first key with digit d goes.  Inside the tile keys are taken
// in index order, 32 at a time: equal digits keep their order (stable).
__global__ void __launch_bounds__(RS_WARPS * 32)
radix_scatter_kernel(const uint32_t *__restrict__ keys, const uint32_t *__restrict__ vals, int N, int shift, int ntiles,
                     const int *__restrict__ offsets, uint32_t *__restrict__ keys_out, uint32_t *__restrict__ vals_out)
{
    __shared__ int next[RS_WARPS][256];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int tile = blockIdx.x * RS_WARPS + warp;
    if (tile >= ntiles) return;
    for (int d = lane; d < 256; d += 32) next[warp][d] = offsets[(int64_t)d * ntiles + tile];
    __syncwarp();
    const int base = tile * RS_TILE;
    const unsigned lt_mask = (1u << lane) - 1u;
    for (int q = 0; q < RS_ITEMS; q++) {
        const int k = base + q * 32 + lane;
        const bool valid = k < N;
        const unsigned act = __ballot_sync(0xffffffffu, valid);
        if (valid) {
            const uint32_t key = keys[k];
            const uint32_t d = (key >> shift) & 255u;
            const unsigned peers = __match_any_sync(act, d);
            const int rank = __popc(peers & lt_mask);
            const int dst = next[warp][d] + rank;
            keys_out[dst] = key;
            vals_out[dst] = vals[k];
            __syncwarp(act);
            if (rank == 0) next[warp][d] += __popc(peers);
        }
        __syncwarp();
    }
}

cudaError_t launch_radix_sort(hb_system *h, int key_bits)
{
    const int N = (int)h->N;
    const int ntiles = (int)cdiv(N, RS_TILE);
    const unsigned grid = (unsigned)cdiv(ntiles, RS_WARPS);
    uint32_t *kin = h->keys, *kout = h->keys2, *vin = h->sperm, *vout = h->sperm2;
    for (int shift = 0; shift < key_bits; shift += 8) {
        radix_hist_kernel<<<grid, RS_WARPS * 32, 0, h->stream>>>(kin, N, shift, ntiles, h->radix_counts);
        h->stats.kernel_launches++;
        // in-place exclusive scan over the 256 x ntiles counts (out[n] lands in the spare slot)
        cudaError_t e = launch_scan_exclusive(h, h->radix_counts, h->radix_counts + h->radix_counts_len,
                                              (int64_t)256 * ntiles, h->scan_tmp);
        if (e != cudaSuccess) return e;
        radix_scatter_kernel<<<grid, RS_WARPS * 32, 0, h->stream>>>(kin, vin, N, shift, ntiles,
                                                                    h->radix_counts + h->radix_counts_len, kout, vout);
        h->stats.kernel_launches++;
        uint32_t *t = kin; kin = kout; kout = t;
        t = vin; vin = vout; vout = t;
    }
    // an odd number of passes leaves the result in the second buffers
    if (kin != h->keys) {
        uint32_t *t = h->keys; h->keys = h->keys2; h->keys2 = t;
        t = h->sperm; h->sperm = h->sperm2; h->sperm2 = t;
    }
    return cudaGetLastError();
}

// new slot k takes the particle that was at perm[k]
__global__ void gather_state_kernel(const uint32_t *__restrict__ perm, int N, const float4 *__restrict__ pos,
                                    const float4 *__restrict__ vel, const float4 *__restrict__ force,
                                    const float4 *__restrict__ virial, const int *__restrict__ image,
                                    const uint32_t *__restrict__ tag, float4 *__restrict__ pos2, float4 *__restrict__ vel2,
                                    float4 *__restrict__ force2, float4 *__restrict__ virial2, int *__restrict__ image2,
                                    uint32_t *__restrict__ tag2, uint32_t *__restrict__ rtag)
{
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= N) return;
    const int64_t o = perm[k];
    pos2[k] = pos[o];
    vel2[k] = vel[o];
    force2[k] = force[o];
    virial2[2 * (int64_t)k] = virial[2 * o];
    virial2[2 * (int64_t)k + 1] = virial[2 * o + 1];
    image2[k] = image[o];
    image2[N + k] = image[N + o];
    image2[2 * (int64_t)N + k] = image[2 * (int64_t)N + o];
    const uint32_t t = tag[o];
    tag2[k] = t;
    rtag[t] = k;
}

cudaError_t launch_gather_state(hb_system *h)
{
    gather_state_kernel<<<(unsigned)cdiv(h->N, 256), 256, 0, h->stream>>>(h->sperm, (int)h->N, h->pos(), h->vel, h->force, h->virial,
                                                                          h->image, h->tag, h->pos_build, h->vel2, h->force2,
                                                                          h->virial2, h->image2, h->tag2, h->rtag);
    h->stats.kernel_launches++;
    return cudaGetLastError();
}

// tag -> storage slot, recomputed from the tag array (after a restore)
__global__ void rtag_kernel(const uint32_t *__restrict__ tag, int N, uint32_t *__restrict__ rtag)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < N) rtag[tag[i]] = i;
}

cudaError_t launch_rtag(hb_system *h)
{
    rtag_kernel<<<(unsigned)cdiv(h->N, 256), 256, 0, h->stream>>>(h->tag, (int)h->N, h->rtag);
    return cudaGetLastError();
}
