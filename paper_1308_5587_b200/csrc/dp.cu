// The binary64 variant of the path (HOOMD's double-precision build removes
// the momentum drift of the single-precision one and lowers the energy drift, Table 2).  Tunable "precision" = 64:
//   * positions, velocities, forces, virials and image flags are kept in binary64 arrays indexed BY TAG (they never
//     move when the list build or hb_sort re-orders the binary32 arrays);
//   * Algorithm 2 and Algorithm 3 run unchanged on the binary32 mirror of the positions (updated after every drift): a
//     rounding of 4e-6 sigma is far inside r_buff / 2, so the list still holds every pair inside r_cut;
//   * the pair sums walk the same list (slots of a tile's staging layout -> tags), take the positions in binary64 from
//     global memory, apply the minimum image per pair, evaluate the functor in binary64 and reduce over a warp with
//     shuffles (one warp per particle, fixed order: deterministic);
//   * velocity Verlet in binary64, one step per host iteration (the rebuild flag is read by the host: this variant is
//     about what the arithmetic conserves, not about time steps per second).
// Everything here is a plain kernel; the roofline work is in force.cu / nlist.cu.
#include "tile.cuh"

struct DpPair {   // per type pair, binary64
    double eps, sigma, p2, rcut2, ron2, invD, eshift;
};

__device__ __forceinline__ void dp_pair(const int pot, const DpPair &q, const double r2, double &V, double &fdivr)
{
    // V(r) and -(1/r) dV/dr of reading f1's potentials; cutoff treatments of PAPER.md:105, 314, 355-367
    double v, f;
    if (pot == HB_POT_GAUSS) {
        v = q.eps * exp(-0.5 * r2 / (q.sigma * q.sigma));
        f = v / (q.sigma * q.sigma);
    } else if (pot == HB_POT_YUKAWA) {
        const double r = sqrt(r2);
        v = q.eps * exp(-q.sigma * r) / r;
        f = v * (q.sigma + 1.0 / r) / r;
    } else if (pot == HB_POT_MORSE) {
        const double r = sqrt(r2);
        const double e1 = exp(-q.sigma * (r - q.p2));
        v = q.eps * (e1 * e1 - 2.0 * e1);
        f = 2.0 * q.sigma * q.eps * (e1 * e1 - e1) / r;
    } else {
        const double s2 = q.sigma * q.sigma / r2;
        const double s6 = s2 * s2 * s2;
        v = 4.0 * q.eps * (s6 * s6 - s6);
        f = (48.0 * q.eps * s6 * s6 - 24.0 * q.eps * s6) / r2;
    }
    if (q.invD != 0.0 && r2 >= q.ron2) {      // XPLOR: V S, F S - V S'/r
        const double d = q.rcut2 - r2;
        const double S = d * d * (q.rcut2 + 2.0 * r2 - 3.0 * q.ron2) * q.invD;
        const double dS = 12.0 * d * (q.ron2 - r2) * q.invD;
        f = f * S - v * dS;
        v = v * S;
    }
    V = v - q.eshift;
    fdivr = f;
}

struct DpArgs {
    TileGeom g;
    const int *cell_start;
    const uint16_t *nlist;
    const int *nlistn;
    int pitch, N, ntypes, pot;
    const float4 *pos32;          // storage order: .w = type
    const uint32_t *tag;
    const double4 *x;             // by tag
    const DpPair *pairs;
    double L;
    double4 *f;                   // by tag: Fx, Fy, Fz, U_i
    double *vir;                  // by tag [N][6]
    int *flags;
};

// One block per tile (the list's entries are slots of the tile's staging layout), one warp per own particle.
__global__ void __launch_bounds__(TILE_THREADS) dp_force_kernel(const DpArgs A)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    __shared__ TileShared s;
    int *gidx = reinterpret_cast<int *>(smem_raw);      // slot -> storage index
    TileCtx t;
    tile_decode(A.g, blockIdx.x, t);
    if (!tile_tables(A.g, A.cell_start, t, s, A.flags)) return;
    for (int sl = 1 + threadIdx.x; sl < t.nslots; sl += TILE_THREADS) {
        const int h = tile_cell_of_slot(t, s, sl);
        gidx[sl] = s.hg[h] + (sl - s.hslot[h]);
    }
    __syncthreads();
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const double L = A.L;
    for (int q = warp; q < t.nown; q += TILE_THREADS / 32) {
        int gi, slot;
        tile_own(s.d, q, gi, slot);
        const uint32_t ti = A.tag[gi];
        const double4 xi = A.x[ti];
        const int typ_i = __float_as_int(A.pos32[gi].w);
        const int n = A.nlistn[gi];
        const uint16_t *row = A.nlist + (int64_t)gi * A.pitch;
        double a[10] = {0, 0, 0, 0, 0, 0, 0, 0, 0, 0};
        for (int k = lane; k < n; k += 32) {
            const int gj = gidx[row[k] >> A.g.eshift];
            const double4 xj = A.x[A.tag[gj]];
            const DpPair &pq = A.pairs[typ_i * A.ntypes + __float_as_int(A.pos32[gj].w)];
            double dx = xi.x - xj.x, dy = xi.y - xj.y, dz = xi.z - xj.z;
            dx -= L * rint(dx / L); dy -= L * rint(dy / L); dz -= L * rint(dz / L);     // minimum image (Alg. 3 l.16)
            const double r2 = dx * dx + dy * dy + dz * dz;
            if (r2 < pq.rcut2) {                                                       // strict <
                double V, fd;
                dp_pair(A.pot, pq, r2, V, fd);
                const double fx = fd * dx, fy = fd * dy, fz = fd * dz;
                a[0] += fx; a[1] += fy; a[2] += fz; a[3] += 0.5 * V;
                a[4] += 0.5 * dx * fx; a[5] += 0.5 * dx * fy; a[6] += 0.5 * dx * fz;
                a[7] += 0.5 * dy * fy; a[8] += 0.5 * dy * fz; a[9] += 0.5 * dz * fz;
            }
        }
#pragma unroll
        for (int c = 0; c < 10; c++)
            for (int o = 16; o > 0; o >>= 1) a[c] += __shfl_xor_sync(0xffffffffu, a[c], o);
        if (lane == 0) {
            A.f[ti] = make_double4(a[0], a[1], a[2], a[3]);
            double *w = A.vir + 6 * (int64_t)ti;
            for (int c = 0; c < 6; c++) w[c] = a[4 + c];
        }
    }
}

// velocity Verlet in binary64, by tag; what = 1: first half kick + drift + wrap + binary32 mirror; 2: second half kick
struct DpNve {
    double4 *x, *v;
    const double4 *f;
    int *img;            // [3][N] by tag
    float4 *pos32, *vel32;
    const uint32_t *rtag;
    int N;
    double dt, L;
};

__global__ void __launch_bounds__(256) dp_nve_kernel(DpNve a, int what)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= a.N) return;
    double4 v = a.v[i];
    const double4 f = a.f[i];
    const double hdt = 0.5 * a.dt, hL = 0.5 * a.L;
    v.x = v.x + hdt * f.x / v.w;      // reading c7 with the mass of PAPER.md:105 (v.w)
    v.y = v.y + hdt * f.y / v.w;
    v.z = v.z + hdt * f.z / v.w;
    a.v[i] = v;
    const uint32_t r = a.rtag[i];
    a.vel32[r] = make_float4((float)v.x, (float)v.y, (float)v.z, (float)v.w);
    if (what != 1) return;
    double4 x = a.x[i];
    x.x += a.dt * v.x; x.y += a.dt * v.y; x.z += a.dt * v.z;
    if (x.x >= hL) { x.x -= a.L; a.img[i] += 1; } else if (x.x < -hL) { x.x += a.L; a.img[i] -= 1; }
    if (x.y >= hL) { x.y -= a.L; a.img[a.N + i] += 1; } else if (x.y < -hL) { x.y += a.L; a.img[a.N + i] -= 1; }
    if (x.z >= hL) { x.z -= a.L; a.img[2 * (int64_t)a.N + i] += 1; } else if (x.z < -hL) { x.z += a.L; a.img[2 * (int64_t)a.N + i] -= 1; }
    a.x[i] = x;
    // the binary32 mirror the cell list and the neighbor list are built from (a coordinate that rounds up to L/2 is
    // still binned correctly: reading c1.iii)
    const float w = a.pos32[r].w;
    a.pos32[r] = make_float4((float)x.x, (float)x.y, (float)x.z, w);
}

// binary32 state (storage order) -> binary64 arrays by tag; or binary64 input (by tag = input order) -> both
__global__ void __launch_bounds__(256) dp_init_kernel(const float4 *pos32, const float4 *vel32, const int *image, const uint32_t *tag,
                                                      int N, double4 *x, double4 *v, int *img)
{
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= N) return;
    const uint32_t t = tag[k];
    const float4 p = pos32[k], u = vel32[k];
    x[t] = make_double4(p.x, p.y, p.z, 0.0);
    v[t] = make_double4(u.x, u.y, u.z, u.w);
    for (int a = 0; a < 3; a++) img[(int64_t)a * N + t] = image[(int64_t)a * N + k];
}

__global__ void __launch_bounds__(256) dp_set_kernel(const double *pos, const double *vel, const int32_t *image, int N, double L,
                                                     double4 *x, double4 *v, int *img, float *pos_f, float *vel_f, int *flags)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= N) return;
    const double hL = 0.5 * L;
    const double px = pos[3 * (int64_t)i], py = pos[3 * (int64_t)i + 1], pz = pos[3 * (int64_t)i + 2];
    if (!(px >= -hL && px < hL && py >= -hL && py < hL && pz >= -hL && pz < hL)) flags[FL_BAD] = 1;
    x[i] = make_double4(px, py, pz, 0.0);
    v[i] = make_double4(vel[3 * (int64_t)i], vel[3 * (int64_t)i + 1], vel[3 * (int64_t)i + 2], 1.0);
    for (int a = 0; a < 3; a++) {
        img[(int64_t)a * N + i] = image ? image[3 * (int64_t)i + a] : 0;
        pos_f[3 * (int64_t)i + a] = (float)pos[3 * (int64_t)i + a];
        vel_f[3 * (int64_t)i + a] = (float)vel[3 * (int64_t)i + a];
    }
}

__global__ void __launch_bounds__(256) dp_get_kernel(const double4 *x, const double4 *v, const int *img, const double4 *f,
                                                     const double *vir, int N, double *pos, double *vel, int32_t *image,
                                                     double *f4, double *vir6, float *f4_f, float *vir6_f)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= N) return;
    if (pos) { const double4 p = x[i]; pos[3 * (int64_t)i] = p.x; pos[3 * (int64_t)i + 1] = p.y; pos[3 * (int64_t)i + 2] = p.z; }
    if (vel) { const double4 u = v[i]; vel[3 * (int64_t)i] = u.x; vel[3 * (int64_t)i + 1] = u.y; vel[3 * (int64_t)i + 2] = u.z; }
    if (image) for (int a = 0; a < 3; a++) image[3 * (int64_t)i + a] = img[(int64_t)a * N + i];
    if (f4 || f4_f) {
        const double4 q = f[i];
        if (f4) { f4[4 * (int64_t)i] = q.x; f4[4 * (int64_t)i + 1] = q.y; f4[4 * (int64_t)i + 2] = q.z; f4[4 * (int64_t)i + 3] = q.w; }
        if (f4_f) { f4_f[4 * (int64_t)i] = (float)q.x; f4_f[4 * (int64_t)i + 1] = (float)q.y; f4_f[4 * (int64_t)i + 2] = (float)q.z; f4_f[4 * (int64_t)i + 3] = (float)q.w; }
    }
    for (int c = 0; c < 6; c++) {
        if (vir6) vir6[6 * (int64_t)i + c] = vir[6 * (int64_t)i + c];
        if (vir6_f) vir6_f[6 * (int64_t)i + c] = (float)vir[6 * (int64_t)i + c];
    }
}

// K = 1/2 sum m v^2, U, W[6], p = sum m v in binary64; one block, fixed order (deterministic); an accessor, not the hot path
__global__ void __launch_bounds__(1024) dp_thermo_kernel(const double4 *v, const double4 *f, const double *vir, int N, double *out)
{
    __shared__ double sm[32][11];
    double a[11] = {0, 0, 0, 0, 0, 0, 0, 0, 0, 0, 0};
    for (int i = threadIdx.x; i < N; i += blockDim.x) {
        const double4 u = v[i];
        a[0] += 0.5 * u.w * (u.x * u.x + u.y * u.y + u.z * u.z);
        a[1] += f[i].w;
        for (int c = 0; c < 6; c++) a[2 + c] += vir[6 * (int64_t)i + c];
        a[8] += u.w * u.x; a[9] += u.w * u.y; a[10] += u.w * u.z;
    }
    for (int c = 0; c < 11; c++) {
        double x = a[c];
        for (int o = 16; o > 0; o >>= 1) x += __shfl_xor_sync(0xffffffffu, x, o);
        if ((threadIdx.x & 31) == 0) sm[threadIdx.x >> 5][c] = x;
    }
    __syncthreads();
    if (threadIdx.x < 11) {
        double x = 0.0;
        for (int w = 0; w < (int)(blockDim.x >> 5); w++) x += sm[w][threadIdx.x];
        out[threadIdx.x] = x;
    }
}

__global__ void dp_mass_kernel(double4 *v, const float4 *vel32, const uint32_t *rtag, int N)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < N) v[i].w = (double)vel32[rtag[i]].w;
}

// ---- host side ----
int dp_ensure(hb_system *h)
{
    if (h->dp.x) return HB_OK;
    const size_t N = (size_t)h->N;
    auto al = [&](void **p, size_t bytes) -> int {
        *p = nullptr;
        if (h->has_alloc) { *p = h->alloc.alloc(bytes, (void *)h->stream, h->alloc.user); return *p ? HB_OK : HB_ENOMEM; }
        if (cudaMalloc(p, bytes) != cudaSuccess) { cudaGetLastError(); return HB_ENOMEM; }
        return HB_OK;
    };
    int rc = HB_OK;
    if ((rc = al((void **)&h->dp.x, N * 32)) || (rc = al((void **)&h->dp.v, N * 32)) || (rc = al((void **)&h->dp.f, N * 32)) ||
        (rc = al((void **)&h->dp.vir, N * 48)) || (rc = al((void **)&h->dp.img, N * 12)) ||
        (rc = al((void **)&h->dp.pairs, sizeof(DpPair) * 64 * 64)) || (rc = al((void **)&h->dp.out, 16 * 8))) {
        h->err = "binary64 arrays: allocation failed";
        return rc;
    }
    return HB_OK;
}

void dp_release(hb_system *h)
{
    void *ptrs[] = {h->dp.x, h->dp.v, h->dp.f, h->dp.vir, h->dp.img, h->dp.pairs, h->dp.out};
    for (void *p : ptrs) {
        if (!p) continue;
        if (h->has_alloc) h->alloc.free(p, (void *)h->stream, h->alloc.user);
        else cudaFree(p);
    }
    h->dp = hb_system::Dp{};
}

int dp_upload_pairs(hb_system *h)
{
    const int nt2 = h->ntypes * h->ntypes;
    std::vector<DpPair> t((size_t)nt2);
    for (int p = 0; p < nt2; p++) {
        const double e = h->eps[p], s = h->sigma[p], rc = h->rcut[p], ron = h->ron[p], p2 = h->p2[p];
        DpPair q{};
        q.eps = e; q.sigma = s; q.p2 = p2; q.rcut2 = rc * rc; q.ron2 = ron * ron;
        const double d = rc * rc - ron * ron;
        q.invD = (h->shift_mode == HB_XPLOR && ron < rc) ? 1.0 / (d * d * d) : 0.0;
        q.eshift = 0.0;
        if (h->shift_mode == HB_SHIFT_ENERGY) {
            switch (h->pot) {
                case HB_POT_GAUSS: q.eshift = e * std::exp(-0.5 * (rc / s) * (rc / s)); break;
                case HB_POT_YUKAWA: q.eshift = e * std::exp(-s * rc) / rc; break;
                case HB_POT_MORSE: { const double e1 = std::exp(-s * (rc - p2)); q.eshift = e * (e1 * e1 - 2.0 * e1); break; }
                default: { const double s6 = std::pow(s / rc, 6.0); q.eshift = 4.0 * e * (s6 * s6 - s6); }
            }
        }
        t[(size_t)p] = q;
    }
    HB_CK(cudaMemcpyAsync(h->dp.pairs, t.data(), sizeof(DpPair) * nt2, cudaMemcpyHostToDevice, h->stream));
    HB_CK(cudaStreamSynchronize(h->stream));
    return HB_OK;
}

// binary32 state -> binary64 arrays (hb_set_state in this mode, or the mode switched on with a state in place)
int dp_from_f32(hb_system *h)
{
    HB_TRY(dp_ensure(h));
    dp_init_kernel<<<(unsigned)cdiv(h->N, 256), 256, 0, h->stream>>>(h->pos(), h->vel, h->image, h->tag, (int)h->N,
                                                                     (double4 *)h->dp.x, (double4 *)h->dp.v, h->dp.img);
    HB_CK(cudaGetLastError());
    h->dp.forces_valid = false;
    h->dp.have = true;
    return HB_OK;
}

int dp_sync_mass(hb_system *h)
{
    if (!h->dp.have) return HB_OK;
    dp_mass_kernel<<<(unsigned)cdiv(h->N, 256), 256, 0, h->stream>>>((double4 *)h->dp.v, h->vel, h->rtag, (int)h->N);
    HB_CK(cudaGetLastError());
    return HB_OK;
}

int dp_force(hb_system *h)
{
    HB_TRY(dp_upload_pairs(h));
    DpArgs A{};
    A.g = h->geom;
    A.cell_start = h->cell_start;
    A.nlist = h->nlist;
    A.nlistn = h->nlistn;
    A.pitch = h->row_pitch;
    A.N = (int)h->N;
    A.ntypes = h->ntypes;
    A.pot = h->pot;
    A.pos32 = h->pos();
    A.tag = h->tag;
    A.x = (const double4 *)h->dp.x;
    A.pairs = (const DpPair *)h->dp.pairs;
    A.L = (double)h->L;
    A.f = (double4 *)h->dp.f;
    A.vir = h->dp.vir;
    A.flags = h->flags;
    const size_t smem = (size_t)h->geom.cap * 4;
    HB_CK(cudaFuncSetAttribute(dp_force_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_attr(h)));
    dp_force_kernel<<<(unsigned)h->geom.ntiles, TILE_THREADS, smem, h->stream>>>(A);
    HB_CK(cudaGetLastError());
    h->stats.kernel_launches++;
    h->dp.forces_valid = true;
    return HB_OK;
}

int dp_nve(hb_system *h, double dt, int what)
{
    DpNve a{(double4 *)h->dp.x, (double4 *)h->dp.v, (const double4 *)h->dp.f, h->dp.img, h->pos(), h->vel, h->rtag, (int)h->N, dt, (double)h->L};
    dp_nve_kernel<<<(unsigned)cdiv(h->N, 256), 256, 0, h->stream>>>(a, what);
    HB_CK(cudaGetLastError());
    h->stats.kernel_launches++;
    return HB_OK;
}

int dp_set_state(hb_system *h, const double *pos, const double *vel, const int32_t *image, float *pos_f, float *vel_f)
{
    HB_TRY(dp_ensure(h));
    dp_set_kernel<<<(unsigned)cdiv(h->N, 256), 256, 0, h->stream>>>(pos, vel, image, (int)h->N, (double)h->L, (double4 *)h->dp.x,
                                                                    (double4 *)h->dp.v, h->dp.img, pos_f, vel_f, h->flags);
    HB_CK(cudaGetLastError());
    h->dp.forces_valid = false;
    h->dp.have = true;
    return HB_OK;
}

int dp_get(hb_system *h, double *pos, double *vel, int32_t *image, double *f4, double *vir6, float *f4_f, float *vir6_f)
{
    dp_get_kernel<<<(unsigned)cdiv(h->N, 256), 256, 0, h->stream>>>((const double4 *)h->dp.x, (const double4 *)h->dp.v, h->dp.img,
                                                                    (const double4 *)h->dp.f, h->dp.vir, (int)h->N, pos, vel, image,
                                                                    f4, vir6, f4_f, vir6_f);
    HB_CK(cudaGetLastError());
    return HB_OK;
}

int dp_thermo(hb_system *h, double *out11)
{
    dp_thermo_kernel<<<1, 1024, 0, h->stream>>>((const double4 *)h->dp.v, (const double4 *)h->dp.f, h->dp.vir, (int)h->N, h->dp.out);
    HB_CK(cudaGetLastError());
    HB_CK(cudaMemcpyAsync(h->h_thermo, h->dp.out, 11 * sizeof(double), cudaMemcpyDeviceToHost, h->stream));
    HB_CK(cudaStreamSynchronize(h->stream));
    for (int c = 0; c < 11; c++) out11[c] = h->h_thermo[c];
    return HB_OK;
}
