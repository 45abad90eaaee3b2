// The per-particle velocity updates of the three integration methods and the end-of-drift bookkeeping, shared by
// the stand-alone integrator kernel (nve.cu) and the fused step kernel (force.cu).
//   NVE          v += (dt/2) F / m                                               (reading c7)
//   Nose-Hoover  first half  v' = (v + (dt/2) F / m) / (1 + (dt/2) xi)
//                second half v  = v' + (dt/2) (F / m - xi v')                     (reading n1)
//                after every drift the LAST block to finish advances xi and eta from sum m v'^2
//   Langevin     NVE, and after the second half kick v = v (1 - gamma dt / m) + sqrt(6 gamma T dt) / m u,
//                u = counter-based uniform in (-1, 1) of (seed, time step, 3 tag + component)   (reading n2)
// The mass is v.w (1 unless hb_set_mass was called); F / m is formed as F * (1 / m) with 1 / m = __frcp_rn(m), which
// leaves every operation of the m = 1 path bit for bit what it was (F * 1 = F).
#pragma once
#include "hb_internal.cuh"

__device__ __forceinline__ unsigned long long hb_mix64(unsigned long long z)
{
    z ^= z >> 30; z *= 0xBF58476D1CE4E5B9ULL;
    z ^= z >> 27; z *= 0x94D049BB133111EBULL;
    z ^= z >> 31;
    return z;
}

// splitmix64 finaliser of (seed, stream, index), as workloads.py states it; 23 bits -> (2k + 1 - 2^23) / 2^23, exact in binary32
__device__ __forceinline__ float hb_uniform_pm1(unsigned long long seed_stream, unsigned long long index)
{
    const unsigned long long G = 0x9E3779B97F4A7C15ULL;
    const unsigned long long x = hb_mix64(seed_stream + (index + 1ULL) * G);
    const int k = (int)(x >> 41);
    return (float)(2 * k + 1 - 8388608) * 1.1920928955078125e-07f;
}

__device__ __forceinline__ unsigned long long hb_seed_stream(unsigned long long seed, unsigned long long stream)
{
    const unsigned long long G = 0x9E3779B97F4A7C15ULL;
    return hb_mix64(hb_mix64(seed + G) + stream * G);
}

// second half kick of a step (v is v'), with what the method adds to it
__device__ __forceinline__ void thermo_kick_prev(const NveArgs &nv, float xi, float hdt, float fx, float fy, float fz, float4 &v, unsigned tag)
{
    const float im = __frcp_rn(v.w);
    fx *= im; fy *= im; fz *= im;
    if (nv.ens == 1) {
        v.x = __fmaf_rn(hdt, __fmaf_rn(-xi, v.x, fx), v.x);
        v.y = __fmaf_rn(hdt, __fmaf_rn(-xi, v.y, fy), v.y);
        v.z = __fmaf_rn(hdt, __fmaf_rn(-xi, v.z, fz), v.z);
        return;
    }
    v.x = __fmaf_rn(hdt, fx, v.x);
    v.y = __fmaf_rn(hdt, fy, v.y);
    v.z = __fmaf_rn(hdt, fz, v.z);
    if (nv.ens == 2) {
        const float c = 1.0f - (nv.par * nv.dt) * im, sg = sqrtf(6.0f * nv.par * nv.T * nv.dt) * im;
        const unsigned long long step = (unsigned long long)(*reinterpret_cast<const long long *>(nv.tstate + TS_LBASE)) + (unsigned long long)nv.kick_step;
        const unsigned long long ss = hb_seed_stream(nv.seed, step);
        v.x = __fmaf_rn(sg, hb_uniform_pm1(ss, 3ULL * tag + 0ULL), v.x * c);
        v.y = __fmaf_rn(sg, hb_uniform_pm1(ss, 3ULL * tag + 1ULL), v.y * c);
        v.z = __fmaf_rn(sg, hb_uniform_pm1(ss, 3ULL * tag + 2ULL), v.z * c);
    }
}

// first half kick of a step
__device__ __forceinline__ void thermo_kick_first(const NveArgs &nv, float xi, float hdt, float fx, float fy, float fz, float4 &v)
{
    const float im = __frcp_rn(v.w);
    v.x = __fmaf_rn(hdt, fx * im, v.x);
    v.y = __fmaf_rn(hdt, fy * im, v.y);
    v.z = __fmaf_rn(hdt, fz * im, v.z);
    if (nv.ens == 1) {
        const float den = __fmaf_rn(hdt, xi, 1.0f);
        v.x = __fdiv_rn(v.x, den); v.y = __fdiv_rn(v.y, den); v.z = __fdiv_rn(v.z, den);
    }
}

// After a drift: Nose-Hoover's kinetic-energy sum, and the work of the last block to finish: advance the thermostat
// (every block read xi when it started, so nobody sees the new value before the next kernel) and hand the rebuild
// decision to a conditional graph node if there is one.  ksum: this thread's m v'^2 / 2.
__device__ __forceinline__ void step_epilogue(const NveArgs &nv, int *__restrict__ flags, double ksum, unsigned nblocks)
{
    if (nv.ens == 1) {
        for (int o = 16; o > 0; o >>= 1) ksum += __shfl_xor_sync(0xffffffffu, ksum, o);
        if ((threadIdx.x & 31) == 0 && ksum != 0.0) atomicAdd(nv.tstate + TS_KSUM, ksum);
    }
    if (nv.ens != 1 && !nv.use_cond) return;
    __syncthreads();
    if (threadIdx.x == 0) {
        __threadfence();
        const int ticket = atomicAdd(&flags[FL_DONE_CTR], 1);
        if (ticket == (int)nblocks - 1) {
            __threadfence();
            if (nv.ens == 1) {
                volatile double *ts = nv.tstate;
                const double K = ts[TS_KSUM], xi = ts[TS_XI];
                const double xin = xi + (double)nv.dt / ((double)nv.par * (double)nv.par) * ((2.0 * K / nv.gdof) / (double)nv.T - 1.0);
                ts[TS_ETA] = ts[TS_ETA] + 0.5 * (double)nv.dt * (xi + xin);
                ts[TS_XI] = xin;
                ts[TS_KSUM] = 0.0;
            }
            if (nv.use_cond) {
                const int need = *((volatile int *)&flags[nv.need_set]);
                cudaGraphSetConditional(nv.cond, need ? 1u : 0u);
            }
            flags[FL_DONE_CTR] = 0;
        }
    }
}
