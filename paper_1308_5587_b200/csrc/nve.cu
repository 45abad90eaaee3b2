// Velocity-Verlet NVE half-steps, the buffer-exceedance check
// that decides when the neighbor list is rebuilt (reading c3), the
// thermodynamic reduction and the state pack/unpack kernels.
#include "hb_internal.cuh"
#include "integrate_dev.cuh"

// The stand-alone integrator kernel (hb_step_nve, the first drift of a run, fuse_nve = 0):
//   kick_prev  : v += (dt/2) F   -- second half of the previous step (reading c7)
//   kick_drift : v += (dt/2) F;  x += dt v;  wrap into [-L/2, L/2) with image +-1;
//                set the drift's FL_NEED flag if |minimage(x - x_build)| > r_buff / 2
// Inside hb_run_nve the same arithmetic, operation by operation, runs at the end of the
// force kernel (force.cu).  With use_cond the last block to finish hands the rebuild
// decision to the CUDA graph's conditional node, so the host never sees it.
__global__ void __launch_bounds__(256)
nve_kernel(float4 *pos, const float4 *__restrict__ force, int N, float L, int *__restrict__ flags, NveArgs nv)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    const float hdt = 0.5f * nv.dt, hL = 0.5f * L, dt = nv.dt;
    bool exceed = false;
    double ksum = 0.0;
    const float xi = nv.ens == 1 ? (float)nv.tstate[TS_XI] : 0.f;     // read by every block before the last one updates it
    if (nv.kick_drift && i == 0) flags[nv.need_clear] = 0;
    if (i < N) {
        float4 v = nv.vel[i];
        const float4 f = force[i];
        if (nv.kick_prev) thermo_kick_prev(nv, xi, hdt, f.x, f.y, f.z, v, nv.ens == 2 ? nv.tag[i] : 0u);
        if (nv.kick_drift) {
            thermo_kick_first(nv, xi, hdt, f.x, f.y, f.z, v);
            if (nv.ens == 1) ksum = 0.5 * (double)v.w * ((double)v.x * v.x + (double)v.y * v.y + (double)v.z * v.z);
            float4 p = pos[i];
            p.x = __fmaf_rn(dt, v.x, p.x);
            p.y = __fmaf_rn(dt, v.y, p.y);
            p.z = __fmaf_rn(dt, v.z, p.z);
            if (p.x >= hL) { p.x -= L; nv.image[i] += 1; } else if (p.x < -hL) { p.x += L; nv.image[i] -= 1; }
            if (p.y >= hL) { p.y -= L; nv.image[N + i] += 1; } else if (p.y < -hL) { p.y += L; nv.image[N + i] -= 1; }
            if (p.z >= hL) { p.z -= L; nv.image[2 * (int64_t)N + i] += 1; }
            else if (p.z < -hL) { p.z += L; nv.image[2 * (int64_t)N + i] -= 1; }
            nv.pos_out[i] = p;
            const float4 pb = nv.pos_build[i];
            float dx = p.x - pb.x, dy = p.y - pb.y, dz = p.z - pb.z;
            if (dx >= hL) dx -= L; else if (dx < -hL) dx += L;
            if (dy >= hL) dy -= L; else if (dy < -hL) dy += L;
            if (dz >= hL) dz -= L; else if (dz < -hL) dz += L;
            exceed = (dx * dx + dy * dy + dz * dz) > nv.half_buff2;
        }
        nv.vel[i] = v;
    }
    if (nv.kick_drift) {
        if (__any_sync(0xffffffffu, exceed) && (threadIdx.x & 31) == 0) flags[nv.need_set] = 1;
        step_epilogue(nv, flags, ksum, gridDim.x);
    }
}

cudaError_t launch_nve(hb_system *h, const NveArgs &a)
{
    const unsigned grid = (unsigned)cdiv(h->N, 256);
    nve_kernel<<<grid, 256, 0, h->stream>>>(h->pos(), h->force, (int)h->N, h->L, h->flags, a);
    h->stats.kernel_launches++;
    return cudaGetLastError();
}

// Reading c3 on demand (hb_needs_rebuild): has any particle moved more than r_buff/2 since the build?
__global__ void __launch_bounds__(256)
disp_check_kernel(const float4 *__restrict__ pos, const float4 *__restrict__ pos_build, int N, float L, float half_buff2,
                  int *__restrict__ flags)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    const float hL = 0.5f * L;
    bool exceed = false;
    if (i < N) {
        const float4 p = pos[i], pb = pos_build[i];
        float dx = p.x - pb.x, dy = p.y - pb.y, dz = p.z - pb.z;
        if (dx >= hL) dx -= L; else if (dx < -hL) dx += L;
        if (dy >= hL) dy -= L; else if (dy < -hL) dy += L;
        if (dz >= hL) dz -= L; else if (dz < -hL) dz += L;
        exceed = (dx * dx + dy * dy + dz * dz) > half_buff2;
    }
    if (__any_sync(0xffffffffu, exceed) && (threadIdx.x & 31) == 0) flags[FL_CHECK] = 1;
}

cudaError_t launch_disp_check(hb_system *h)
{
    const float hb = 0.5f * h->r_buff;
    disp_check_kernel<<<(unsigned)cdiv(h->N, 256), 256, 0, h->stream>>>(h->pos(), h->pos_build, (int)h->N, h->L, hb * hb, h->flags);
    return cudaGetLastError();
}

// ---- thermodynamic sums, accumulated in binary64, deterministic two-stage reduction ----
constexpr int TH_VALS = 11;  // K, U, W[6], px, py, pz
constexpr int TH_THREADS = 256;

__global__ void __launch_bounds__(TH_THREADS)
thermo_partial_kernel(const float4 *__restrict__ vel, const float4 *__restrict__ force, const float4 *__restrict__ virial,
                      int N, double *__restrict__ part)
{
    double a[TH_VALS];
#pragma unroll
    for (int q = 0; q < TH_VALS; q++) a[q] = 0.0;
    for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < N; i += gridDim.x * blockDim.x) {
        const float4 v = vel[i];
        const float4 f = force[i];
        const float4 w0 = virial[2 * (int64_t)i], w1 = virial[2 * (int64_t)i + 1];
        const double m = (double)v.w;
        a[0] += 0.5 * m * ((double)v.x * v.x + (double)v.y * v.y + (double)v.z * v.z);
        a[1] += f.w;
        a[2] += w0.x; a[3] += w0.y; a[4] += w0.z; a[5] += w0.w; a[6] += w1.x; a[7] += w1.y;
        a[8] += m * v.x; a[9] += m * v.y; a[10] += m * v.z;
    }
    __shared__ double sm[TH_THREADS / 32][TH_VALS];
#pragma unroll
    for (int q = 0; q < TH_VALS; q++) {
        double x = a[q];
        for (int o = 16; o > 0; o >>= 1) x += __shfl_xor_sync(0xffffffffu, x, o);
        if ((threadIdx.x & 31) == 0) sm[threadIdx.x >> 5][q] = x;
    }
    __syncthreads();
    if (threadIdx.x < TH_VALS) {
        double x = 0.0;
        for (int w = 0; w < TH_THREADS / 32; w++) x += sm[w][threadIdx.x];
        part[(int64_t)blockIdx.x * TH_VALS + threadIdx.x] = x;
    }
}

__global__ void thermo_final_kernel(const double *__restrict__ part, int nblocks, double *__restrict__ out)
{
    if (threadIdx.x < TH_VALS) {
        double x = 0.0;
        for (int b = 0; b < nblocks; b++) x += part[(int64_t)b * TH_VALS + threadIdx.x];
        out[threadIdx.x] = x;
    }
}

cudaError_t launch_thermo(hb_system *h)
{
    thermo_partial_kernel<<<h->thermo_blocks, TH_THREADS, 0, h->stream>>>(h->vel, h->force, h->virial, (int)h->N, h->thermo_part);
    thermo_final_kernel<<<1, 32, 0, h->stream>>>(h->thermo_part, h->thermo_blocks,
                                                h->thermo_part + (int64_t)h->thermo_blocks * TH_VALS);
    h->stats.kernel_launches += 2;
    return cudaGetLastError();
}

// ---- state upload / download ----
__global__ void pack_state_kernel(const float *__restrict__ pos_xyz, const int32_t *__restrict__ type,
                                  const float *__restrict__ vel_xyz, const int32_t *__restrict__ image_in, int N,
                                  int ntypes, float4 *__restrict__ pos, float4 *__restrict__ vel, int *__restrict__ image,
                                  uint32_t *__restrict__ tag, uint32_t *__restrict__ rtag, int *__restrict__ flags)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= N) return;
    int t = type ? type[i] : 0;
    if (t < 0 || t >= ntypes) { flags[FL_BADTYPE] = 1; t = 0; }   // the force kernel indexes its pair table with it
    pos[i] = make_float4(pos_xyz[3 * (int64_t)i], pos_xyz[3 * (int64_t)i + 1], pos_xyz[3 * (int64_t)i + 2],
                         __int_as_float(t));
    vel[i] = make_float4(vel_xyz[3 * (int64_t)i], vel_xyz[3 * (int64_t)i + 1], vel_xyz[3 * (int64_t)i + 2], 1.0f);   // .w = mass
    for (int a = 0; a < 3; a++) image[(int64_t)a * N + i] = image_in ? image_in[3 * (int64_t)i + a] : 0;
    tag[i] = i;
    rtag[i] = i;
}

__global__ void unpack_state_kernel(const float4 *__restrict__ pos, const float4 *__restrict__ vel,
                                    const int *__restrict__ image, const uint32_t *__restrict__ tag, int N,
                                    float *__restrict__ pos_xyz, int32_t *__restrict__ type, float *__restrict__ vel_xyz,
                                    int32_t *__restrict__ image_out)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= N) return;
    const int64_t t = tag[i];
    const float4 p = pos[i], v = vel[i];
    if (pos_xyz) { pos_xyz[3 * t] = p.x; pos_xyz[3 * t + 1] = p.y; pos_xyz[3 * t + 2] = p.z; }
    if (type) type[t] = __float_as_int(p.w);
    if (vel_xyz) { vel_xyz[3 * t] = v.x; vel_xyz[3 * t + 1] = v.y; vel_xyz[3 * t + 2] = v.z; }
    if (image_out)
        for (int a = 0; a < 3; a++) image_out[3 * t + a] = image[(int64_t)a * N + i];
}

cudaError_t launch_pack_state(hb_system *h, const float *pos_xyz, const int32_t *type, const float *vel_xyz, const int32_t *image)
{
    pack_state_kernel<<<(unsigned)cdiv(h->N, 256), 256, 0, h->stream>>>(pos_xyz, type, vel_xyz, image, (int)h->N, h->ntypes, h->pos(),
                                                                        h->vel, h->image, h->tag, h->rtag, h->flags);
    return cudaGetLastError();
}

cudaError_t launch_unpack_state(hb_system *h, float *pos_xyz, int32_t *type, float *vel_xyz, int32_t *image)
{
    unpack_state_kernel<<<(unsigned)cdiv(h->N, 256), 256, 0, h->stream>>>(h->pos(), h->vel, h->image, h->tag, (int)h->N, pos_xyz,
                                                                          type, vel_xyz, image);
    return cudaGetLastError();
}

// per-particle mass lives in vel.w; the accessors go by tag
__global__ void mass_kernel(float4 *__restrict__ vel, const uint32_t *__restrict__ tag, int N, const float *__restrict__ mass_in,
                            float *__restrict__ mass_out, int *__restrict__ flags)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= N) return;
    const uint32_t t = tag[i];
    if (mass_in) {
        const float m = mass_in[t];
        if (!(m > 0.f) || !(m < 3.0e38f)) flags[FL_BADTYPE] = 1;
        else vel[i].w = m;
    }
    if (mass_out) mass_out[t] = vel[i].w;
}

cudaError_t launch_mass(hb_system *h, const float *mass_in, float *mass_out)
{
    mass_kernel<<<(unsigned)cdiv(h->N, 256), 256, 0, h->stream>>>(h->vel, h->tag, (int)h->N, mass_in, mass_out, h->flags);
    return cudaGetLastError();
}

// The state a chunk of hb_run_nve can be rolled back to (positions, velocities, image flags, tags, thermostat state):
// ONE kernel instead of five device-to-device copies (a chunk of 20 steps is 600 us; five copy launches were 15 of them).
__global__ void __launch_bounds__(256)
state_copy_kernel(const float4 *__restrict__ pos, const float4 *__restrict__ vel, const int *__restrict__ image,
                  const uint32_t *__restrict__ tag, const double *__restrict__ ts, int N, float4 *__restrict__ pos_o,
                  float4 *__restrict__ vel_o, int *__restrict__ image_o, uint32_t *__restrict__ tag_o, double *__restrict__ ts_o)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < TS_COUNT) ts_o[i] = ts[i];
    if (i >= N) return;
    pos_o[i] = pos[i];
    vel_o[i] = vel[i];
    image_o[i] = image[i];
    image_o[N + i] = image[N + i];
    image_o[2 * (int64_t)N + i] = image[2 * (int64_t)N + i];
    tag_o[i] = tag[i];
}

cudaError_t launch_state_copy(hb_system *h, bool restore)
{
    const unsigned grid = (unsigned)cdiv(h->N, 256);
    if (!restore)
        state_copy_kernel<<<grid, 256, 0, h->stream>>>(h->pos(), h->vel, h->image, h->tag, h->tstate, (int)h->N, h->bk_pos, h->bk_vel,
                                                       h->bk_image, h->bk_tag, h->bk_tstate);
    else
        state_copy_kernel<<<grid, 256, 0, h->stream>>>(h->bk_pos, h->bk_vel, h->bk_image, h->bk_tag, h->bk_tstate, (int)h->N, h->pos(),
                                                       h->vel, h->image, h->tag, h->tstate);
    return cudaGetLastError();
}
