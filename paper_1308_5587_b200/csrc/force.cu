// Lennard-Jones pair force, energy and virial over the neighbor list
// (PAPER.md:95, 103, 105, 284, 314-320).
//
//   V_lj = 4 eps [(sigma/r)^12 - (sigma/r)^6],  f = -(1/r) dV/dr * d,  r < r_cut,ab
// with per-type-pair tables held as lj1 = 4 eps sigma^12, lj2 = 4 eps sigma^6:
//   -(1/r) dV/dr = r^-2 r^-6 (12 lj1 r^-6 - 6 lj2),   V = r^-6 (lj1 r^-6 - lj2) - eshift.
// The pair functor idea of PAPER.md:284 (V(r) and -(1/r) dV/dr) is kept as the
// inlined lj_pair() below.
//
// TPP threads share one particle: they stride over its row (consecutive lanes
// read consecutive 4-byte indices), gather pos[j] as one 16-byte load each, and
// combine F, U and W with warp shuffles.  Lane 0 of the group writes the force,
// lanes 1 and 2 the two virial vectors, so the epilogue is three 16 B stores.
#include "hb_internal.cuh"

__device__ __forceinline__ float min_image(float d, float L, float hL)
{
    // both particles are inside the box, so |d| < L: one conditional shift suffices
    if (d >= hL) d -= L;
    else if (d < -hL) d += L;
    return d;
}

__device__ __forceinline__ void lj_pair(float r2, const PairParam &pp, float &fdivr, float &e)
{
    const float r2inv = __frcp_rn(r2);
    const float r6inv = r2inv * r2inv * r2inv;
    fdivr = r2inv * r6inv * (12.0f * pp.lj1 * r6inv - 6.0f * pp.lj2);
    e = r6inv * (pp.lj1 * r6inv - pp.lj2) - pp.eshift;
}

template <int TPP, bool ONE_TYPE>
__global__ void __launch_bounds__(256)
lj_force_kernel(const float4 *__restrict__ pos, const int *__restrict__ nlist, const int *__restrict__ nlistn, int pitch,
                int N, float L, int ntypes, const PairParam *__restrict__ params, float4 *__restrict__ force,
                float4 *__restrict__ virial, int *__restrict__ flags)
{
    extern __shared__ PairParam s_params[];
    if (!ONE_TYPE) {
        for (int k = threadIdx.x; k < ntypes * ntypes; k += blockDim.x) s_params[k] = params[k];
        __syncthreads();
    }
    const int gid = blockIdx.x * blockDim.x + threadIdx.x;
    if (gid == 0) flags[FL_NEED_BUILD] = 0;  // the rebuild decision of this step has been consumed
    const int ig = gid / TPP;
    const int sub = gid % TPP;
    const bool active = ig < N;        // inactive threads stay for the shuffles below
    const int i = active ? ig : N - 1;

    const float hL = 0.5f * L;
    const float4 pi = pos[i];
    const int n = active ? nlistn[i] : 0;
    const int *row = nlist + (int64_t)i * pitch;
    PairParam pp;
    const PairParam *prow = nullptr;
    if (ONE_TYPE) pp = params[0];
    else prow = s_params + __float_as_int(pi.w) * ntypes;

    float fx = 0.f, fy = 0.f, fz = 0.f, u = 0.f;
    float wxx = 0.f, wxy = 0.f, wxz = 0.f, wyy = 0.f, wyz = 0.f, wzz = 0.f;

#pragma unroll 4
    for (int k = sub; k < n; k += TPP) {
        const int j = row[k];
        const float4 pj = __ldg(&pos[j]);
        const float dx = min_image(pi.x - pj.x, L, hL);
        const float dy = min_image(pi.y - pj.y, L, hL);
        const float dz = min_image(pi.z - pj.z, L, hL);
        const float r2 = dx * dx + dy * dy + dz * dz;
        if (!ONE_TYPE) pp = prow[__float_as_int(pj.w)];
        if (r2 < pp.rcut2) {
            float fdivr, e;
            lj_pair(r2, pp, fdivr, e);
            const float px = fdivr * dx, py = fdivr * dy, pz = fdivr * dz;
            fx += px; fy += py; fz += pz;
            u += e;
            wxx += dx * px; wxy += dx * py; wxz += dx * pz;
            wyy += dy * py; wyz += dy * pz; wzz += dz * pz;
        }
    }
#pragma unroll
    for (int o = TPP >> 1; o > 0; o >>= 1) {
        fx += __shfl_xor_sync(0xffffffffu, fx, o);
        fy += __shfl_xor_sync(0xffffffffu, fy, o);
        fz += __shfl_xor_sync(0xffffffffu, fz, o);
        u += __shfl_xor_sync(0xffffffffu, u, o);
        wxx += __shfl_xor_sync(0xffffffffu, wxx, o);
        wxy += __shfl_xor_sync(0xffffffffu, wxy, o);
        wxz += __shfl_xor_sync(0xffffffffu, wxz, o);
        wyy += __shfl_xor_sync(0xffffffffu, wyy, o);
        wyz += __shfl_xor_sync(0xffffffffu, wyz, o);
        wzz += __shfl_xor_sync(0xffffffffu, wzz, o);
    }
    if (!active) return;
    // U_i = 1/2 sum V, W_i = 1/2 sum d f (reading c6.i)
    if (TPP >= 4) {
        if (sub == 0) force[i] = make_float4(fx, fy, fz, 0.5f * u);
        else if (sub == 1) virial[2 * (int64_t)i] = make_float4(0.5f * wxx, 0.5f * wxy, 0.5f * wxz, 0.5f * wyy);
        else if (sub == 2) virial[2 * (int64_t)i + 1] = make_float4(0.5f * wyz, 0.5f * wzz, 0.f, 0.f);
    } else if (sub == 0) {
        force[i] = make_float4(fx, fy, fz, 0.5f * u);
        virial[2 * (int64_t)i] = make_float4(0.5f * wxx, 0.5f * wxy, 0.5f * wxz, 0.5f * wyy);
        virial[2 * (int64_t)i + 1] = make_float4(0.5f * wyz, 0.5f * wzz, 0.f, 0.f);
    }
}

template <int TPP>
static cudaError_t launch_force_tpp(hb_system *h)
{
    const int block = h->tun.force_block;
    const int64_t threads = h->N * TPP;
    const unsigned grid = (unsigned)cdiv(threads, block);
    if (h->ntypes == 1) {
        lj_force_kernel<TPP, true><<<grid, block, 0, h->stream>>>(h->pos, h->nlist, h->nlistn, h->row_pitch, (int)h->N, h->L,
                                                                 1, h->params, h->force, h->virial, h->flags);
    } else {
        const size_t smem = sizeof(PairParam) * h->ntypes * h->ntypes;
        lj_force_kernel<TPP, false><<<grid, block, smem, h->stream>>>(h->pos, h->nlist, h->nlistn, h->row_pitch, (int)h->N,
                                                                     h->L, h->ntypes, h->params, h->force, h->virial,
                                                                     h->flags);
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
        case 16: return launch_force_tpp<16>(h);
        case 32: return launch_force_tpp<32>(h);
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
