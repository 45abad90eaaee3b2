// Lennard-Jones pair force, energy and virial over the neighbor list
// (PAPER.md:95, 103, 105, 284, 314-320).
//
//   V_lj = 4 eps [(sigma/r)^12 - (sigma/r)^6],  f = -(1/r) dV/dr * d,  r < r_cut,ab
// with per-type-pair tables held as lj1 = 4 eps sigma^12, lj2 = 4 eps sigma^6:
//   -(1/r) dV/dr = r^-2 r^-6 (12 lj1 r^-6 - 6 lj2),   V = r^-6 (lj1 r^-6 - lj2) - eshift.
// The pair functor idea of PAPER.md:284 (V(r) and -(1/r) dV/dr) is kept as the
// inlined lj_pair() below.
//
// Design (round-1 ncu: the first version was issue-bound at 83 warp instructions
// per row segment, with no loads in flight across its divergent cutoff branch):
//   * TPP threads share one particle.  Each reads FOUR consecutive list entries
//     as one 16-byte load (rows are 128-byte aligned), then issues the four
//     16-byte position gathers back to back, then evaluates the four pairs
//     without a branch: a pair outside r_cut (or past the end of the row) gets
//     r^-2 := 0, which zeroes its force, energy and virial terms.
//   * Minimum-image arithmetic only where it can matter: a warp whose particles
//     all lie farther than r_max + r_buff from every face of the box cannot have
//     a listed neighbor across the boundary and runs the loop without it.
//   * A block walks `passes` consecutive tiles of particles, so the positions it
//     gathers stay in its SM's L1 (particles are Hilbert-ordered).
//   * F, U, W are combined across the TPP lanes with warp shuffles; lane 0 of the
//     group stores the force, lanes 1 and 2 the two virial vectors.
#include "hb_internal.cuh"

__device__ __forceinline__ float rcp_approx(float x)
{
    float y;
    asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}

struct Acc {
    float fx, fy, fz, u, wxx, wxy, wxz, wyy, wyz, wzz;
};

template <bool MI>
__device__ __forceinline__ void pair_term(const float4 &pi, const float4 &pj, bool valid, const PairParam &pp, float L,
                                          float invL, Acc &a)
{
    float dx = pi.x - pj.x, dy = pi.y - pj.y, dz = pi.z - pj.z;
    if (MI) {  // nearest image (Alg. 3 l.16); |d| < L because both particles are inside the box
        dx = __fmaf_rn(-L, rintf(dx * invL), dx);
        dy = __fmaf_rn(-L, rintf(dy * invL), dy);
        dz = __fmaf_rn(-L, rintf(dz * invL), dz);
    }
    const float r2 = __fmaf_rn(dz, dz, __fmaf_rn(dy, dy, dx * dx));
    const bool in = valid && (r2 < pp.rcut2);          // strict <
    const float r2inv = in ? rcp_approx(r2) : 0.0f;    // 0 switches the whole pair off
    const float r6inv = r2inv * r2inv * r2inv;
    const float fdivr = r2inv * r6inv * __fmaf_rn(12.0f * pp.lj1, r6inv, -6.0f * pp.lj2);
    const float e = __fmaf_rn(r6inv, __fmaf_rn(pp.lj1, r6inv, -pp.lj2), in ? -pp.eshift : 0.0f);
    const float px = fdivr * dx, py = fdivr * dy, pz = fdivr * dz;
    a.fx += px; a.fy += py; a.fz += pz;
    a.u += e;
    a.wxx = __fmaf_rn(dx, px, a.wxx); a.wxy = __fmaf_rn(dx, py, a.wxy); a.wxz = __fmaf_rn(dx, pz, a.wxz);
    a.wyy = __fmaf_rn(dy, py, a.wyy); a.wyz = __fmaf_rn(dy, pz, a.wyz); a.wzz = __fmaf_rn(dz, pz, a.wzz);
}

// One row: entries sub*4 .. sub*4+3, then + 4*TPP, ...
template <int TPP, bool ONE_TYPE, bool MI>
__device__ __forceinline__ void accumulate_row(const float4 *__restrict__ pos, const int *__restrict__ row, int n, int self,
                                               int sub, const float4 &pi, const PairParam *__restrict__ prow,
                                               const PairParam &pp1, float L, float invL, Acc &a)
{
    for (int k = sub * 4; k < n; k += 4 * TPP) {
        const int4 jj = __ldg(reinterpret_cast<const int4 *>(row + k));
        const int rem = n - k;
        const int j0 = jj.x;                       // k < n always
        const int j1 = rem > 1 ? jj.y : self;      // past the end: any in-bounds index, switched off below
        const int j2 = rem > 2 ? jj.z : self;
        const int j3 = rem > 3 ? jj.w : self;
        const float4 p0 = __ldg(&pos[j0]);
        const float4 p1 = __ldg(&pos[j1]);
        const float4 p2 = __ldg(&pos[j2]);
        const float4 p3 = __ldg(&pos[j3]);
        if (ONE_TYPE) {
            pair_term<MI>(pi, p0, true, pp1, L, invL, a);
            pair_term<MI>(pi, p1, rem > 1, pp1, L, invL, a);
            pair_term<MI>(pi, p2, rem > 2, pp1, L, invL, a);
            pair_term<MI>(pi, p3, rem > 3, pp1, L, invL, a);
        } else {
            pair_term<MI>(pi, p0, true, prow[__float_as_int(p0.w)], L, invL, a);
            pair_term<MI>(pi, p1, rem > 1, prow[__float_as_int(p1.w)], L, invL, a);
            pair_term<MI>(pi, p2, rem > 2, prow[__float_as_int(p2.w)], L, invL, a);
            pair_term<MI>(pi, p3, rem > 3, prow[__float_as_int(p3.w)], L, invL, a);
        }
    }
}

template <int TPP, bool ONE_TYPE>
__global__ void __launch_bounds__(256)
lj_force_kernel(const float4 *__restrict__ pos, const int *__restrict__ nlist, const int *__restrict__ nlistn, int pitch,
                int N, float L, float inner, int passes, int ntypes, const PairParam *__restrict__ params,
                float4 *__restrict__ force, float4 *__restrict__ virial, int *__restrict__ flags)
{
    extern __shared__ PairParam s_params[];
    if (!ONE_TYPE) {
        for (int k = threadIdx.x; k < ntypes * ntypes; k += blockDim.x) s_params[k] = params[k];
        __syncthreads();
    }
    if (blockIdx.x == 0 && threadIdx.x == 0) flags[FL_NEED_BUILD] = 0;  // this step's rebuild decision has been consumed
    const float invL = 1.0f / L;
    const int ppb = blockDim.x / TPP;            // particles per block per pass
    const int sub = threadIdx.x % TPP;
    PairParam pp1 = params[0];

    for (int pass = 0; pass < passes; pass++) {
        const int ig = (blockIdx.x * passes + pass) * ppb + threadIdx.x / TPP;
        const bool active = ig < N;              // inactive threads stay for the shuffles
        const int i = active ? ig : N - 1;
        const float4 pi = pos[i];
        const int n = active ? nlistn[i] : 0;
        const int *row = nlist + (int64_t)i * pitch;
        const PairParam *prow = ONE_TYPE ? nullptr : s_params + __float_as_int(pi.w) * ntypes;
        Acc a = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f};

        const bool interior = fmaxf(fmaxf(fabsf(pi.x), fabsf(pi.y)), fabsf(pi.z)) < inner;
        if (__all_sync(0xffffffffu, interior)) accumulate_row<TPP, ONE_TYPE, false>(pos, row, n, i, sub, pi, prow, pp1, L, invL, a);
        else accumulate_row<TPP, ONE_TYPE, true>(pos, row, n, i, sub, pi, prow, pp1, L, invL, a);

#pragma unroll
        for (int o = TPP >> 1; o > 0; o >>= 1) {
            a.fx += __shfl_xor_sync(0xffffffffu, a.fx, o);
            a.fy += __shfl_xor_sync(0xffffffffu, a.fy, o);
            a.fz += __shfl_xor_sync(0xffffffffu, a.fz, o);
            a.u += __shfl_xor_sync(0xffffffffu, a.u, o);
            a.wxx += __shfl_xor_sync(0xffffffffu, a.wxx, o);
            a.wxy += __shfl_xor_sync(0xffffffffu, a.wxy, o);
            a.wxz += __shfl_xor_sync(0xffffffffu, a.wxz, o);
            a.wyy += __shfl_xor_sync(0xffffffffu, a.wyy, o);
            a.wyz += __shfl_xor_sync(0xffffffffu, a.wyz, o);
            a.wzz += __shfl_xor_sync(0xffffffffu, a.wzz, o);
        }
        if (!active) continue;
        // U_i = 1/2 sum V, W_i = 1/2 sum d f (reading c6.i)
        if (TPP >= 4) {
            if (sub == 0) force[i] = make_float4(a.fx, a.fy, a.fz, 0.5f * a.u);
            else if (sub == 1) virial[2 * (int64_t)i] = make_float4(0.5f * a.wxx, 0.5f * a.wxy, 0.5f * a.wxz, 0.5f * a.wyy);
            else if (sub == 2) virial[2 * (int64_t)i + 1] = make_float4(0.5f * a.wyz, 0.5f * a.wzz, 0.f, 0.f);
        } else if (sub == 0) {
            force[i] = make_float4(a.fx, a.fy, a.fz, 0.5f * a.u);
            virial[2 * (int64_t)i] = make_float4(0.5f * a.wxx, 0.5f * a.wxy, 0.5f * a.wxz, 0.5f * a.wyy);
            virial[2 * (int64_t)i + 1] = make_float4(0.5f * a.wyz, 0.5f * a.wzz, 0.f, 0.f);
        }
    }
}

template <int TPP>
static cudaError_t launch_force_tpp(hb_system *h)
{
    const int block = h->tun.force_block;
    const int ppb = block / TPP;
    // passes: consecutive tiles per block, chosen so that the grid still fills the GPU about twice over
    int passes = h->tun.force_passes;
    if (passes <= 0) {
        const int64_t tiles = cdiv(h->N, ppb);
        passes = (int)std::max<int64_t>(1, std::min<int64_t>(16, tiles / ((int64_t)h->sm_count * 16)));
    }
    const unsigned grid = (unsigned)cdiv(h->N, (int64_t)ppb * passes);
    // listed pairs are closer than r_max + r_buff now; beyond that distance from every face no pair crosses the boundary
    const float inner = 0.5f * h->L - (h->r_max + h->r_buff);
    if (h->ntypes == 1) {
        lj_force_kernel<TPP, true><<<grid, block, 0, h->stream>>>(h->pos, h->nlist, h->nlistn, h->row_pitch, (int)h->N, h->L,
                                                                 inner, passes, 1, h->params, h->force, h->virial, h->flags);
    } else {
        const size_t smem = sizeof(PairParam) * h->ntypes * h->ntypes;
        lj_force_kernel<TPP, false><<<grid, block, smem, h->stream>>>(h->pos, h->nlist, h->nlistn, h->row_pitch, (int)h->N,
                                                                     h->L, inner, passes, h->ntypes, h->params, h->force,
                                                                     h->virial, h->flags);
    }
    h->stats.kernel_launches++;
    return cudaGetLastError();
}

cudaError_t launch_force(hb_system *h)
{
    switch (h->tun.tpp) {
        case 1: return launch_force_tpp<1>(h);
        case 2: return launch_force_tpp<2>(h);
        case 4: return launch_force_tpp<4>(h);
        default: return launch_force_tpp<8>(h);
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
