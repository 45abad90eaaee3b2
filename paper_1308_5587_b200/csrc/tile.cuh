// Tile staging shared by the list build (nlist.cu), the force kernel (force.cu)
// and the list accessor: the SAME function lays the halo of a tile out in shared
// memory in all three, so a shared-memory slot number written into the list by
// the build means the same particle to the force kernel.
//
// The paper's first GPU list kernel staged neighbor cells in shared memory with one
// block per cell and was dropped because cell occupancies vary too much for 16 KB
// (PAPER.md:177); its successor reads neighbors through the cache and names the
// scattered traffic the bottleneck.  With 227 KB per SM the
// capacity objection is gone: a block owns a brick of cells, stages the brick
// plus a one-cell halo ONCE with coalesced reads (the particle data is kept in
// cell order, so x-adjacent cells are one contiguous run), applies the periodic
// shift while staging (no minimum-image arithmetic is left in any inner loop),
// and every later gather is a shared-memory access.
//
// Layout: halo cell h = jx + hx (jy + hy jz), jx in [0, ex + 2) etc.; slots are
// handed out in h order, slot 0 is a dummy particle far away from everything, so
// list rows can be padded with 0 and need no bounds test in the force loop.
#pragma once
#include "hb_internal.cuh"

// TMA bulk copy global -> shared (UBLKCP), completion counted in bytes on an mbarrier: one instruction moves a whole
// piece of the halo (a contiguous run of positions), no per-particle instruction at all.
__device__ __forceinline__ void mbar_inval(uint64_t *bar)
{
    asm volatile("mbarrier.inval.shared::cta.b64 [%0];" ::"r"((unsigned)__cvta_generic_to_shared(bar)) : "memory");
}
__device__ __forceinline__ void mbar_init(uint64_t *bar, unsigned count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"((unsigned)__cvta_generic_to_shared(bar)), "r"(count) : "memory");
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t *bar, unsigned bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"((unsigned)__cvta_generic_to_shared(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void bulk_g2s(void *smem_dst, const void *gsrc, unsigned bytes, uint64_t *bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
                     (unsigned)__cvta_generic_to_shared(smem_dst)),
                 "l"(gsrc), "r"(bytes), "r"((unsigned)__cvta_generic_to_shared(bar))
                 : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t *bar, unsigned parity)
{
    const unsigned a = (unsigned)__cvta_generic_to_shared(bar);
    unsigned ok;
    do {
        asm volatile("{\n .reg .pred p;\n mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n selp.u32 %0, 1, 0, p;\n}"
                     : "=r"(ok) : "r"(a), "r"(parity) : "memory");
    } while (!ok);
}


struct TileCtx {
    int x0, y0, z0;   // first own cell
    int ex, ey, ez;   // own extent in cells (clipped tile)
    int hx, hy, hz;   // halo box = extent + 2
    int nh;           // halo cells
    int nslots;       // 1 + staged particles
    int nown;         // own particles
    int nrows;        // own (y, z) rows = ey * ez
};

// What a kernel needs to know about its tile.  It depends on cell_start only; every block derives it
// from cell_start at its start (tile_tables / force_tile_tables) and keeps it in shared memory.
struct TileDesc {
    int nslots;       // 1 + staged particles (1 = nothing staged: the build found the tile too big)
    int nown;         // own particles
    int nrows;        // own (y, z) rows
    float cx, cy, cz; // centre of the tile
    int own_start[TILE_ROWS_MAX];    // storage index of the first own particle of row r
    int own_off[TILE_ROWS_MAX + 1];  // tile-local number of the first own particle of row r
    int own_slot[TILE_ROWS_MAX];     // its slot
    int pad;
};
static_assert(sizeof(TileDesc) == 416, "force.cu copies it word by word; keep it a multiple of 4 bytes");

struct TileShared {
    int hslot[TILE_HMAX + 1];   // first slot of halo cell h
    int hg[TILE_HMAX];          // storage index of the first particle of halo cell h
    TileDesc d;
};

__device__ __forceinline__ void tile_decode(const TileGeom &g, int tile, TileCtx &t)
{
    const int tix = tile % g.ntx, tiy = (tile / g.ntx) % g.nty, tiz = tile / (g.ntx * g.nty);
    t.x0 = tix * g.tx; t.y0 = tiy * g.ty; t.z0 = tiz * g.tz;
    t.ex = min(g.tx, g.m - t.x0); t.ey = min(g.ty, g.m - t.y0); t.ez = min(g.tz, g.m - t.z0);
    t.hx = t.ex + 2; t.hy = t.ey + 2; t.hz = t.ez + 2;
    t.nh = t.hx * t.hy * t.hz;
    t.nrows = t.ey * t.ez;
}

// the same from the three tile coordinates (a 3-D grid launch: no integer division)
__device__ __forceinline__ void tile_decode_xyz(const TileGeom &g, int tix, int tiy, int tiz, TileCtx &t)
{
    t.x0 = tix * g.tx; t.y0 = tiy * g.ty; t.z0 = tiz * g.tz;
    t.ex = min(g.tx, g.m - t.x0); t.ey = min(g.ty, g.m - t.y0); t.ez = min(g.tz, g.m - t.z0);
    t.hx = t.ex + 2; t.hy = t.ey + 2; t.hz = t.ez + 2;
    t.nh = t.hx * t.hy * t.hz;
    t.nrows = t.ey * t.ez;
}

// wrap a halo cell coordinate into the box; shift = what to add to a coordinate of that cell's particles
__device__ __forceinline__ int tile_wrap(int c, int m, float L, float &shift)
{
    shift = 0.f;
    if (c < 0) { c += m; shift = -L; }
    else if (c >= m) { c -= m; shift = L; }
    return c;
}

// Halo table, slot prefix, own-row table.  Returns false (for the whole block) when the tile
// needs more slots than g.cap; FL_STAGE_OVER then carries the number needed.
__device__ __forceinline__ bool tile_tables(const TileGeom &g, const int *__restrict__ cell_start, TileCtx &t, TileShared &s,
                                            int *__restrict__ flags)
{
    const int tid = threadIdx.x, lane = tid & 31;
    for (int h = tid; h < t.nh; h += blockDim.x) {
        const int jx = h % t.hx, jy = (h / t.hx) % t.hy, jz = h / (t.hx * t.hy);
        float dummy;
        const int cx = tile_wrap(t.x0 - 1 + jx, g.m, g.L, dummy);
        const int cy = tile_wrap(t.y0 - 1 + jy, g.m, g.L, dummy);
        const int cz = tile_wrap(t.z0 - 1 + jz, g.m, g.L, dummy);
        const int c = cx + g.m * (cy + g.m * cz);
        const int s0 = cell_start[c];
        s.hg[h] = s0;
        s.hslot[h] = cell_start[c + 1] - s0;
    }
    __syncthreads();
    if (tid < 32) {  // exclusive scan of up to 256 counts: 8 per lane
        const int base = lane * 8;
        int v[8], tsum = 0;
#pragma unroll
        for (int q = 0; q < 8; q++) {
            v[q] = (base + q < t.nh) ? s.hslot[base + q] : 0;
            tsum += v[q];
        }
        int incl = tsum;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const int y = __shfl_up_sync(0xffffffffu, incl, o);
            if (lane >= o) incl += y;
        }
        int run = 1 + incl - tsum;  // slot 0 is the dummy
#pragma unroll
        for (int q = 0; q < 8; q++) {
            if (base + q < t.nh) s.hslot[base + q] = run;
            run += v[q];
        }
        if (lane == 31) s.hslot[t.nh] = run;
    }
    __syncthreads();
    t.nslots = s.hslot[t.nh];
    if (tid < t.nrows) {
        const int ly = tid % t.ey, lz = tid / t.ey;
        const int hrow = ((lz + 1) * t.hy + (ly + 1)) * t.hx;
        const int first = hrow + 1, last = hrow + t.ex;
        s.d.own_start[tid] = s.hg[first];
        s.d.own_slot[tid] = s.hslot[first];
        s.d.own_off[tid + 1] = s.hslot[last + 1] - s.hslot[first];   // own cells of a row are consecutive halo cells
    }
    __syncthreads();
    if (tid == 0) {
        int run = 0;
        s.d.own_off[0] = 0;
        for (int r = 0; r < t.nrows; r++) { const int n = s.d.own_off[r + 1]; s.d.own_off[r + 1] = run + n; run += n; }
        const float wcell = g.L / (float)g.m, hL = 0.5f * g.L;
        s.d.nslots = t.nslots;
        s.d.nown = run;
        s.d.nrows = t.nrows;
        s.d.cx = __fmaf_rn((float)t.x0 + 0.5f * (float)t.ex, wcell, -hL);
        s.d.cy = __fmaf_rn((float)t.y0 + 0.5f * (float)t.ey, wcell, -hL);
        s.d.cz = __fmaf_rn((float)t.z0 + 0.5f * (float)t.ez, wcell, -hL);
        s.d.pad = 0;
    }
    __syncthreads();
    t.nown = s.d.nown;
    if (t.nslots > g.cap) {
        if (tid == 0) atomicMax(&flags[FL_STAGE_OVER], t.nslots);
        return false;
    }
    return true;
}

// halo cell of slot sl: the largest h with hslot[h] <= sl
__device__ __forceinline__ int tile_cell_of_slot(const TileCtx &t, const TileShared &s, int sl)
{
    int h = 0;
#pragma unroll
    for (int st = TILE_HMAX / 2; st > 0; st >>= 1)
        if (h + st < t.nh && s.hslot[h + st] <= sl) h += st;
    return h;
}

// image of coordinate x nearest to the centre cc of the (possibly out-of-box) halo cell it belongs to
__device__ __forceinline__ float tile_image(float x, float cc, float L, float hL)
{
    const float d = x - cc;
    if (d > hL) x -= L;
    else if (d < -hL) x += L;
    return x;
}

// Positions of all halo cells into stage[1 .. nslots), each moved to the periodic image that lies in
// the halo cell as this tile sees it (a cell left of the box for the tile at x0 = 0, and so on);
// stage[0] = dummy.  The image is chosen from the POSITION, relative to the centre of the halo cell
// in the tile's frame, not from the cell index alone: between two builds a particle near a face of
// the box may have been wrapped to the other side, and must still be seen next to its neighbors.
// At build time (particles inside their cells) this adds exactly -L, 0 or +L per axis.
__device__ __forceinline__ void tile_stage_positions(const TileGeom &g, const TileCtx &t, const TileShared &s,
                                                     const float4 *__restrict__ pos, float4 *__restrict__ stage,
                                                     int *__restrict__ src_out /* nullable: [cap] storage index per slot */)
{
    constexpr int U = 4;
    const int nt = blockDim.x;
    const float wcell = g.L / (float)g.m, hL = 0.5f * g.L;
    const bool fast = g.fast != 0;
    if (threadIdx.x == 0) stage[0] = make_float4(1e18f, 1e18f, 1e18f, 0.f);
    for (int s0 = 1 + threadIdx.x; s0 < t.nslots; s0 += U * nt) {
        int src[U];
        float cx[U], cy[U], cz[U];
#pragma unroll
        for (int u = 0; u < U; u++) {
            const int sl = s0 + u * nt;
            src[u] = -1;
            if (sl < t.nslots) {
                const int h = tile_cell_of_slot(t, s, sl);
                src[u] = s.hg[h] + (sl - s.hslot[h]);
                if (fast) {   // the whole halo box is narrower than L/2: the image nearest to the tile centre is the one
                    cx[u] = s.d.cx; cy[u] = s.d.cy; cz[u] = s.d.cz;
                } else {
                    const int jx = h % t.hx, jy = (h / t.hx) % t.hy, jz = h / (t.hx * t.hy);
                    cx[u] = __fmaf_rn((float)(t.x0 - 1 + jx) + 0.5f, wcell, -hL);
                    cy[u] = __fmaf_rn((float)(t.y0 - 1 + jy) + 0.5f, wcell, -hL);
                    cz[u] = __fmaf_rn((float)(t.z0 - 1 + jz) + 0.5f, wcell, -hL);
                }
                if (src_out) src_out[sl] = src[u];
            }
        }
        float4 p[U];
#pragma unroll
        for (int u = 0; u < U; u++)
            if (src[u] >= 0) p[u] = pos[src[u]];
#pragma unroll
        for (int u = 0; u < U; u++)
            if (src[u] >= 0)
                stage[s0 + u * nt] = make_float4(tile_image(p[u].x, cx[u], g.L, hL), tile_image(p[u].y, cy[u], g.L, hL),
                                                 tile_image(p[u].z, cz[u], g.L, hL), p[u].w);
    }
}

// The same result, one warp per halo cell (three cells in flight per warp): no search for the cell of a slot.
// Fewer instructions, longer latency; the list build, whose blocks live long, uses this one.
__device__ __forceinline__ void tile_stage_positions_by_cell(const TileGeom &g, const TileCtx &t, const TileShared &s,
                                                             const float4 *__restrict__ pos, float4 *__restrict__ stage,
                                                             int *__restrict__ src_out)
{
    constexpr int U = 3;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, nwarps = blockDim.x >> 5;
    const float wcell = g.L / (float)g.m, hL = 0.5f * g.L;
    const bool fast = g.fast != 0;
    if (threadIdx.x == 0) stage[0] = make_float4(1e18f, 1e18f, 1e18f, 0.f);
    for (int h0 = warp; h0 < t.nh; h0 += U * nwarps) {
        int s0[U], cnt[U], g0[U], kmax = 0;
        float cx[U], cy[U], cz[U];
#pragma unroll
        for (int u = 0; u < U; u++) {
            const int h = h0 + u * nwarps;
            s0[u] = 0; cnt[u] = 0; g0[u] = 0;
            cx[u] = s.d.cx; cy[u] = s.d.cy; cz[u] = s.d.cz;
            if (h < t.nh) {
                s0[u] = s.hslot[h];
                cnt[u] = s.hslot[h + 1] - s0[u];
                g0[u] = s.hg[h];
                if (!fast) {
                    const int jx = h % t.hx, jy = (h / t.hx) % t.hy, jz = h / (t.hx * t.hy);
                    cx[u] = __fmaf_rn((float)(t.x0 - 1 + jx) + 0.5f, wcell, -hL);
                    cy[u] = __fmaf_rn((float)(t.y0 - 1 + jy) + 0.5f, wcell, -hL);
                    cz[u] = __fmaf_rn((float)(t.z0 - 1 + jz) + 0.5f, wcell, -hL);
                }
            }
            kmax = max(kmax, cnt[u]);
        }
        for (int k = lane; k < kmax; k += 32) {
            float4 p[U];
#pragma unroll
            for (int u = 0; u < U; u++)
                if (k < cnt[u]) p[u] = pos[g0[u] + k];
#pragma unroll
            for (int u = 0; u < U; u++)
                if (k < cnt[u]) {
                    stage[s0[u] + k] = make_float4(tile_image(p[u].x, cx[u], g.L, hL), tile_image(p[u].y, cy[u], g.L, hL),
                                                   tile_image(p[u].z, cz[u], g.L, hL), p[u].w);
                    if (src_out) src_out[s0[u] + k] = g0[u] + k;
                }
        }
    }
}

// The same result for the FAST geometry with the TMA unit: consecutive halo cells of a row that are consecutive in the
// cell-ordered position array (all of them, unless the row wraps around the box) go as ONE bulk copy, issued by the
// thread that owns the halo row; then the tiles whose halo touches a face of the box fix the periodic image in place.
// `bar` is a shared-memory mbarrier used for this one staging (initialised and invalidated here).
__device__ __forceinline__ void tile_stage_positions_bulk(const TileGeom &g, const TileCtx &t, const TileShared &s,
                                                          const float4 *__restrict__ pos, float4 *__restrict__ stage, uint64_t *bar)
{
    if (threadIdx.x == 0) {
        mbar_init(bar, 1);
        stage[0] = make_float4(1e18f, 1e18f, 1e18f, 0.f);
        mbar_expect_tx(bar, (unsigned)(t.nslots - 1) * 16u);
    }
    __syncthreads();
    const int hrows = t.hy * t.hz;
    for (int r = threadIdx.x; r < hrows; r += blockDim.x) {
        const int h0 = r * t.hx;
        int first = h0;                                   // first cell of the running piece
        for (int h = h0; h < h0 + t.hx; h++) {
            const bool last = h + 1 == h0 + t.hx;
            const int cnt_h = s.hslot[h + 1] - s.hslot[h];
            if (last || s.hg[h + 1] != s.hg[h] + cnt_h) {     // the piece ends with cell h
                const int len = s.hslot[h + 1] - s.hslot[first];
                if (len > 0) bulk_g2s(stage + s.hslot[first], pos + s.hg[first], (unsigned)len * 16u, bar);
                first = h + 1;
            }
        }
    }
    mbar_wait(bar, 0);
    const bool fix = t.x0 <= 1 || t.x0 + t.ex >= g.m - 1 || t.y0 <= 1 || t.y0 + t.ey >= g.m - 1 || t.z0 <= 1 || t.z0 + t.ez >= g.m - 1;
    if (fix) {
        const float L = g.L, hL = 0.5f * g.L, cx = s.d.cx, cy = s.d.cy, cz = s.d.cz;
        for (int sl = 1 + threadIdx.x; sl < t.nslots; sl += blockDim.x) {
            float4 p = stage[sl];
            p.x = tile_image(p.x, cx, L, hL); p.y = tile_image(p.y, cy, L, hL); p.z = tile_image(p.z, cz, L, hL);
            stage[sl] = p;
        }
    }
    __syncthreads();
    if (threadIdx.x == 0) mbar_inval(bar);
}

// tile-local own particle q -> own row r (rows are few: linear scan)
__device__ __forceinline__ int tile_row_of(const TileDesc &d, int q)
{
    int r = 0;
    while (r + 1 < d.nrows && d.own_off[r + 1] <= q) r++;
    return r;
}

// storage index and slot of own particle q
__device__ __forceinline__ void tile_own(const TileDesc &d, int q, int &gi, int &slot)
{
    const int r = tile_row_of(d, q);
    const int off = q - d.own_off[r];
    gi = d.own_start[r] + off;
    slot = d.own_slot[r] + off;
}
