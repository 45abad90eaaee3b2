// Lennard-Jones pair force, energy and virial over the neighbor list
// (PAPER.md:95, 103, 105, 284, 314-320), optionally with the velocity-Verlet
// half-steps and the r_buff/2 check fused in.
//
//   V_lj = 4 eps [(sigma/r)^12 - (sigma/r)^6],  f = -(1/r) dV/dr * d,  r < r_cut,ab
// with per-type-pair tables held as lj1 = 4 eps sigma^12, lj2 = 4 eps sigma^6:
//   -(1/r) dV/dr = r^-2 r^-6 (12 lj1 r^-6 - 6 lj2),   V = r^-6 (lj1 r^-6 - lj2) - eshift.
// The pair functor idea of PAPER.md:284 (V(r) and -(1/r) dV/dr) is kept as the
// inlined pair_term() below.
//
// Design.  Round-1 ncu of the first version (one 16-byte global gather per pair):
// 46 % of the stall samples on the gathers, every warp gather touching ~32 cache
// lines, the L1 wavefront queue the limiter.  Now ONE BLOCK OWNS ONE TILE of cells
// (tile.cuh):
//   * the tile and its halo are staged once in shared memory with coalesced
//     loads, shifted to the periodic image the tile sees: no minimum-image
//     arithmetic per pair, and every neighbor gather is a 16-byte shared-memory
//     load (list entries are 16-bit slots of this staging layout);
//   * the list build leaves a descriptor and a slot table per tile behind, so the
//     staging here is: descriptor -> storage index of every slot -> position;
//   * TPP threads share one particle (2 by default); each takes EPL (8) consecutive
//     16-bit entries per iteration.  The rows arrive through a ring of four
//     cp.async copies per thread, not through registers (see cp_async below); a row
//     ends at its first padding entry, so no row length is read.  The EPL gathers
//     are issued back to back and the pairs evaluated without a branch: a pair
//     outside r_cut gets r^-2 := 0, the padding is the far-away dummy slot;
//   * F, U, W are combined across the TPP lanes with warp shuffles;
//   * when asked, the same thread finishes the velocity-Verlet step of its
//     particle with the force it just computed (second half kick of this step,
//     first half kick and drift of the next, wrap, image flags, r_buff/2 check),
//     writing the new position into the OTHER position buffer, since the blocks
//     around still read the old one.  One kernel per time step.
#include "tile.cuh"

__device__ __forceinline__ float rcp_approx(float x)
{
    float y;
    asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}

// cp.async (LDGSTS): global -> shared without a register or a scoreboard slot in between.  ncu of the
// register-prefetch version showed 40 % of the warp time in long-scoreboard stalls at the first use of
// a list entry however far ahead it was loaded: scoreboard slots count, so a consumer waits for every
// later load on its slot too.  Async-copy groups are tracked separately.
template <int BYTES>
__device__ __forceinline__ void cp_async(void *smem_dst, const void *gsrc)
{
    const unsigned d = (unsigned)__cvta_generic_to_shared(smem_dst);
    asm volatile("cp.async.ca.shared.global [%0], [%1], %2;" ::"r"(d), "l"(gsrc), "n"(BYTES) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N>
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }

struct Acc {
    float fx, fy, fz, u, wxx, wxy, wxz, wyy, wyz, wzz;
};

template <bool THERMO>
__device__ __forceinline__ void pair_term(const float4 &pi, const float4 &pj, const PairParam &pp, Acc &a)
{
    const float dx = pi.x - pj.x, dy = pi.y - pj.y, dz = pi.z - pj.z;   // pj is already the nearest image
    const float r2 = __fmaf_rn(dz, dz, __fmaf_rn(dy, dy, dx * dx));
    const bool in = r2 < pp.rcut2;                     // strict <
    const float r2inv = in ? rcp_approx(r2) : 0.0f;    // 0 switches the whole pair off
    const float r6inv = r2inv * r2inv * r2inv;
    const float fdivr = r2inv * r6inv * __fmaf_rn(12.0f * pp.lj1, r6inv, -6.0f * pp.lj2);
    // explicit roundings: the force sums must not depend on whether the energy and virial terms are compiled in
    const float px = __fmul_rn(fdivr, dx), py = __fmul_rn(fdivr, dy), pz = __fmul_rn(fdivr, dz);
    a.fx = __fadd_rn(a.fx, px); a.fy = __fadd_rn(a.fy, py); a.fz = __fadd_rn(a.fz, pz);
    if (!THERMO) return;   // an inner step of hb_run_nve with thermo_every = 0: nobody can read U_i, W_i of this step
    const float e = __fmaf_rn(r6inv, __fmaf_rn(pp.lj1, r6inv, -pp.lj2), in ? -pp.eshift : 0.0f);
    a.u += e;
    a.wxx = __fmaf_rn(dx, px, a.wxx); a.wxy = __fmaf_rn(dx, py, a.wxy); a.wxz = __fmaf_rn(dx, pz, a.wxz);
    a.wyy = __fmaf_rn(dy, py, a.wyy); a.wyz = __fmaf_rn(dy, pz, a.wyz); a.wzz = __fmaf_rn(dz, pz, a.wzz);
}

template <int EPL> struct Entries;
template <> struct Entries<4> { uint2 v; };
template <> struct Entries<8> { uint4 v; };

template <int EPL>
__device__ __forceinline__ Entries<EPL> load_entries(const uint16_t *p)
{
    Entries<EPL> e;
    if constexpr (EPL == 4) e.v = __ldg(reinterpret_cast<const uint2 *>(p));
    else e.v = __ldg(reinterpret_cast<const uint4 *>(p));
    return e;
}

template <int EPL>
__device__ __forceinline__ void unpack_entries(const Entries<EPL> &e, int (&sl)[EPL])
{
    sl[0] = e.v.x & 0xffffu; sl[1] = e.v.x >> 16; sl[2] = e.v.y & 0xffffu; sl[3] = e.v.y >> 16;
    if constexpr (EPL == 8) { sl[4] = e.v.z & 0xffffu; sl[5] = e.v.z >> 16; sl[6] = e.v.w & 0xffffu; sl[7] = e.v.w >> 16; }
}

template <int TPP, int EPL, bool ONE_TYPE, bool THERMO>
__global__ void __launch_bounds__(TILE_THREADS, 4)   // <= 64 registers: 8 blocks of 128 threads per SM
lj_tile_kernel(TileGeom g, const int *__restrict__ cell_start, const float4 *__restrict__ pos,
               const uint16_t *__restrict__ nlist, const int *__restrict__ nlistn, int pitch, int N, int ntypes,
               const PairParam *__restrict__ params, float4 *__restrict__ force, float4 *__restrict__ virial,
               int *__restrict__ flags, int do_nve, NveArgs nv, const int *__restrict__ stage_src,
               const TileDesc *__restrict__ desc)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    __shared__ TileShared s;
    float4 *stage = reinterpret_cast<float4 *>(smem_raw);
    PairParam *s_params = reinterpret_cast<PairParam *>(smem_raw + (size_t)g.cap * 16);
    constexpr int G = TPP * EPL;                 // entries per particle per iteration

    if (!ONE_TYPE)
        for (int k = threadIdx.x; k < ntypes * ntypes; k += blockDim.x) s_params[k] = params[k];
    if (do_nve && nv.kick_drift && blockIdx.x == 0 && threadIdx.x == 0) flags[nv.need_clear] = 0;

    const int sub = threadIdx.x % TPP;
    const int PPB = blockDim.x / TPP;            // particles per block per pass
    // List rows reach the threads through a ring of PF async copies per thread: entry group k of the
    // row is copied PF iterations before it is used.  A row ends at its first padding entry (slot 0;
    // the build pads every row with at least 32 of them), so the row length is never loaded.
    constexpr int PF = 4;
    using EntryVec = decltype(Entries<EPL>::v);
    EntryVec *ring = reinterpret_cast<EntryVec *>(smem_raw + (size_t)g.cap * 16 +
                                                  (ONE_TYPE ? 0 : ((ntypes * ntypes * sizeof(PairParam) + 15) & ~(size_t)15))) +
                     threadIdx.x;
    const int ring_stride = blockDim.x;
    int gi_n = 0, slot_n = 0;
    bool active_n = false;
    // particle of pass q0 for this thread group; start the copies of its first PF entry groups
    auto prep = [&](int q0, int nown) {
        const int q = q0 + threadIdx.x / TPP;
        active_n = q < nown;
        gi_n = 0; slot_n = 0;
        if (active_n) tile_own(s.d, q, gi_n, slot_n);
        const uint16_t *row = nlist + (int64_t)gi_n * pitch + sub * EPL;
#pragma unroll
        for (int u = 0; u < PF; u++) {
            if (active_n) cp_async<EPL * 2>(ring + u * ring_stride, row + u * G);
            cp_async_commit();
        }
    };

    bool fits;
    if (g.fast) {
        // the list build left this tile's descriptor and the storage index of every slot behind
        if (threadIdx.x < sizeof(TileDesc) / 4)
            reinterpret_cast<int *>(&s.d)[threadIdx.x] = __ldg(reinterpret_cast<const int *>(desc + blockIdx.x) + threadIdx.x);
        __syncthreads();
        fits = s.d.nslots <= g.cap;
        prep(0, fits ? s.d.nown : 0);            // list copies in flight while the tile is staged
        if (fits) tile_stage_from_table(s.d, stage_src + (int64_t)blockIdx.x * g.cap, pos, stage, g.L);
    } else {
        TileCtx t;
        tile_decode(g, blockIdx.x, t);
        fits = tile_tables(g, cell_start, t, s, flags);
        prep(0, fits ? s.d.nown : 0);
        if (fits) tile_stage_positions(g, t, s, pos, stage, nullptr);
    }
    __syncthreads();

    const PairParam pp1 = params[0];
    const float hdt = 0.5f * nv.dt, hL = 0.5f * g.L, L = g.L;
    bool exceed = false;

    const int nown = fits ? s.d.nown : 0;
    for (int q0 = 0; q0 < nown; q0 += PPB) {     // block-uniform trip count: the shuffles need whole warps
        const bool active = active_n;
        const int gi = gi_n;
        const float4 pi = stage[slot_n];         // slot 0 (the dummy) for idle thread groups
        const uint16_t *row = nlist + (int64_t)gi * pitch + sub * EPL;
        const PairParam *prow = ONE_TYPE ? nullptr : s_params + __float_as_int(pi.w) * ntypes;
        Acc a = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f};

        if (active) {
            int c = 0;
            cp_async_wait<PF - 1>();
            Entries<EPL> ent;
            ent.v = ring[0];
            for (int k = 0; k < pitch; k += G) {
                if ((ent.v.x & 0xffffu) == 0u) break;                    // padding: the row is over for this thread
                cp_async<EPL * 2>(ring + c * ring_stride, row + k + PF * G);   // refill PF iterations ahead (reads past the
                cp_async_commit();                                       // row's end are harmless: the array has slack)
                c = (c + 1 == PF) ? 0 : c + 1;
                int sl[EPL];
                unpack_entries<EPL>(ent, sl);
                float4 pj[EPL];
#pragma unroll
                for (int e = 0; e < EPL; e++) pj[e] = stage[sl[e]];
                cp_async_wait<PF - 1>();                                 // the next group of entries, read before the
                ent.v = ring[c * ring_stride];                           // arithmetic so that its latency hides behind it
#pragma unroll
                for (int e = 0; e < EPL; e++) {
                    if (ONE_TYPE) pair_term<THERMO>(pi, pj[e], pp1, a);
                    else pair_term<THERMO>(pi, pj[e], prow[__float_as_int(pj[e].w)], a);
                }
            }
        }
        cp_async_wait<0>();                          // nothing of this pass may land after the next pass's copies start
        if (q0 + PPB < nown) prep(q0 + PPB, nown);   // they fly during the reduction and the integration below
        // what the integration will need, all three loads in flight at once and behind the reduction (ncu: placed
        // where they are used they were three L2 round trips in a row at the very end of the block; issued before
        // the pair loop they cost registers the loop needs)
        float4 v_in = make_float4(0.f, 0.f, 0.f, 0.f), p_in = v_in, pb_in = v_in;
        if (do_nve && active && sub == 0) {
            v_in = nv.vel[gi];
            if (nv.kick_drift) { p_in = pos[gi]; pb_in = nv.pos_build[gi]; }
        }

#pragma unroll
        for (int o = TPP >> 1; o > 0; o >>= 1) {
            a.fx += __shfl_xor_sync(0xffffffffu, a.fx, o);
            a.fy += __shfl_xor_sync(0xffffffffu, a.fy, o);
            a.fz += __shfl_xor_sync(0xffffffffu, a.fz, o);
            if (THERMO) {
                a.u += __shfl_xor_sync(0xffffffffu, a.u, o);
                a.wxx += __shfl_xor_sync(0xffffffffu, a.wxx, o);
                a.wxy += __shfl_xor_sync(0xffffffffu, a.wxy, o);
                a.wxz += __shfl_xor_sync(0xffffffffu, a.wxz, o);
                a.wyy += __shfl_xor_sync(0xffffffffu, a.wyy, o);
                a.wyz += __shfl_xor_sync(0xffffffffu, a.wyz, o);
                a.wzz += __shfl_xor_sync(0xffffffffu, a.wzz, o);
            }
        }
        if (!active) continue;
        // U_i = 1/2 sum V, W_i = 1/2 sum d f (reading c6.i)
        if (sub == 0) {
            force[gi] = make_float4(a.fx, a.fy, a.fz, 0.5f * a.u);
            if (do_nve) {
                // reading c7, operation by operation as nve_kernel does it
                float4 v = v_in;
                if (nv.kick_prev) {
                    v.x = __fmaf_rn(hdt, a.fx, v.x);
                    v.y = __fmaf_rn(hdt, a.fy, v.y);
                    v.z = __fmaf_rn(hdt, a.fz, v.z);
                }
                if (nv.kick_drift) {
                    v.x = __fmaf_rn(hdt, a.fx, v.x);
                    v.y = __fmaf_rn(hdt, a.fy, v.y);
                    v.z = __fmaf_rn(hdt, a.fz, v.z);
                    float4 p = p_in;      // the stored position: pi may be another periodic image of it
                    p.x = __fmaf_rn(nv.dt, v.x, p.x);
                    p.y = __fmaf_rn(nv.dt, v.y, p.y);
                    p.z = __fmaf_rn(nv.dt, v.z, p.z);
                    if (p.x >= hL) { p.x -= L; nv.image[gi] += 1; } else if (p.x < -hL) { p.x += L; nv.image[gi] -= 1; }
                    if (p.y >= hL) { p.y -= L; nv.image[N + gi] += 1; } else if (p.y < -hL) { p.y += L; nv.image[N + gi] -= 1; }
                    if (p.z >= hL) { p.z -= L; nv.image[2 * (int64_t)N + gi] += 1; }
                    else if (p.z < -hL) { p.z += L; nv.image[2 * (int64_t)N + gi] -= 1; }
                    nv.pos_out[gi] = p;
                    const float4 pb = pb_in;
                    float dx = p.x - pb.x, dy = p.y - pb.y, dz = p.z - pb.z;
                    if (dx >= hL) dx -= L; else if (dx < -hL) dx += L;
                    if (dy >= hL) dy -= L; else if (dy < -hL) dy += L;
                    if (dz >= hL) dz -= L; else if (dz < -hL) dz += L;
                    exceed = exceed || (dx * dx + dy * dy + dz * dz) > nv.half_buff2;
                }
                nv.vel[gi] = v;
            }
        } else if (THERMO && TPP >= 4 && sub == 1) {
            virial[2 * (int64_t)gi] = make_float4(0.5f * a.wxx, 0.5f * a.wxy, 0.5f * a.wxz, 0.5f * a.wyy);
        } else if (THERMO && TPP >= 4 && sub == 2) {
            virial[2 * (int64_t)gi + 1] = make_float4(0.5f * a.wyz, 0.5f * a.wzz, 0.f, 0.f);
        }
        if (THERMO && TPP < 4 && sub == TPP - 1) {
            virial[2 * (int64_t)gi] = make_float4(0.5f * a.wxx, 0.5f * a.wxy, 0.5f * a.wxz, 0.5f * a.wyy);
            virial[2 * (int64_t)gi + 1] = make_float4(0.5f * a.wyz, 0.5f * a.wzz, 0.f, 0.f);
        }
    }

    if (do_nve && nv.kick_drift) {
        if (exceed) flags[nv.need_set] = 1;
        if (nv.use_cond) {
            __syncthreads();
            if (threadIdx.x == 0) {
                __threadfence();
                const int ticket = atomicAdd(&flags[FL_DONE_CTR], 1);
                if (ticket == (int)gridDim.x - 1) {
                    __threadfence();
                    const int need = *((volatile int *)&flags[nv.need_set]);
                    cudaGraphSetConditional(nv.cond, need ? 1u : 0u);
                    flags[FL_DONE_CTR] = 0;
                }
            }
        }
    }
}

size_t force_smem_bytes(const hb_system *h)
{
    // staged positions, pair table, ring of 4 async list copies (16 B at most) per thread
    return (size_t)h->geom.cap * 16 + (h->ntypes > 1 ? ((sizeof(PairParam) * h->ntypes * h->ntypes + 15) & ~(size_t)15) : 0) +
           (size_t)4 * 16 * force_block_of(h);
}

template <int TPP, int EPL, bool THERMO>
static cudaError_t launch_force_tt(hb_system *h, const NveArgs *nve)
{
    const size_t smem = force_smem_bytes(h);
    const unsigned grid = (unsigned)h->geom.ntiles;
    NveArgs nv{};
    if (nve) nv = *nve;
    cudaError_t e;
#define LJ_LAUNCH(ONE)                                                                                                      \
    e = cudaFuncSetAttribute(lj_tile_kernel<TPP, EPL, ONE, THERMO>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);        \
    if (e != cudaSuccess) return e;                                                                                         \
    lj_tile_kernel<TPP, EPL, ONE, THERMO><<<grid, force_block_of(h), smem, h->stream>>>(h->geom, h->cell_start, h->pos(), h->nlist,      \
                                                                           h->nlistn, h->row_pitch, (int)h->N, h->ntypes,  \
                                                                           h->params, h->force, h->virial, h->flags,       \
                                                                           nve ? 1 : 0, nv, h->stage_src,                  \
                                                                           (const TileDesc *)h->tile_desc);
    if (h->ntypes == 1) { LJ_LAUNCH(true) } else { LJ_LAUNCH(false) }
#undef LJ_LAUNCH
    h->stats.kernel_launches++;
    return cudaGetLastError();
}

template <int TPP, int EPL>
static cudaError_t launch_force_t(hb_system *h, const NveArgs *nve)
{
    // energies and virials of a step can only be read after hb_run_nve returns: with thermo_every = 0 the inner
    // steps of a chunk (both half kicks fused in) compute forces only
    if (nve && nve->forces_only) return launch_force_tt<TPP, EPL, false>(h, nve);
    return launch_force_tt<TPP, EPL, true>(h, nve);
}

cudaError_t launch_force(hb_system *h, const NveArgs *nve)
{
    const int epl = h->tun.epl == 8 ? 8 : 4;
    switch (h->tun.tpp) {
        case 2: return epl == 8 ? launch_force_t<2, 8>(h, nve) : launch_force_t<2, 4>(h, nve);
        case 8: return launch_force_t<8, 4>(h, nve);   // 8 x 8 entries would read past the 32-entry row padding
        default: return epl == 8 ? launch_force_t<4, 8>(h, nve) : launch_force_t<4, 4>(h, nve);
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
