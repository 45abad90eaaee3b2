// libhb: the C ABI of include/hb.h.  Host-side orchestration only -- every step
// of the hot path is a kernel in cells.cu / nlist.cu / force.cu / nve.cu / sort.cu.
#include <cmath>
#include <cstdio>
#include <cstring>
#include <new>

#include <nvtx3/nvToolsExt.h>

#include "hb_internal.cuh"

namespace {

// NVTX range per stage (tracing): shows up in nsys / ncu timelines, costs nothing without a tool.
struct Range {
    explicit Range(const char *name) { nvtxRangePushA(name); }
    ~Range() { nvtxRangePop(); }
};

int coop_mode(const hb_system *h) { return h->tun.coop_rebuild >= 0 ? h->tun.coop_rebuild : (h->N < 200000 ? 2 : 1); }
int rebuild_kernels(const hb_system *h) { return coop_mode(h) == 2 ? 1 : coop_mode(h) == 1 ? 2 : 5; }  // see enqueue_rebuild

int dev_alloc(hb_system *h, void **p, size_t bytes)
{
    *p = nullptr;
    if (bytes == 0) bytes = 256;
    if (h->has_alloc) {
        *p = h->alloc.alloc(bytes, (void *)h->stream, h->alloc.user);
        if (!*p) { h->err = "allocator returned NULL for " + std::to_string(bytes) + " bytes"; return HB_ENOMEM; }
        return HB_OK;
    }
    cudaError_t e = cudaMalloc(p, bytes);
    if (e != cudaSuccess) {
        cudaGetLastError();
        h->err = std::string("cudaMalloc(") + std::to_string(bytes) + "): " + cudaGetErrorString(e);
        return HB_ENOMEM;
    }
    return HB_OK;
}

void dev_free(hb_system *h, void *p)
{
    if (!p) return;
    if (h->has_alloc) h->alloc.free(p, (void *)h->stream, h->alloc.user);
    else cudaFree(p);
}

template <typename T>
int dev_alloc_t(hb_system *h, T **p, size_t count) { return dev_alloc(h, (void **)p, count * sizeof(T)); }

template <typename T>
void dev_free_t(hb_system *h, T *&p) { dev_free(h, (void *)p); p = nullptr; }

int round_up(int x, int q) { return (x + q - 1) / q * q; }

void destroy_graphs(hb_system *h)
{
    for (auto &kv : h->graphs) {
        if (kv.second.e) cudaGraphExecDestroy(kv.second.e);
        if (kv.second.g) cudaGraphDestroy(kv.second.g);
    }
    h->graphs.clear();
}

// Unshifted V(r) of the chosen potential in binary64 (for the energy shift V(r_cut)); reading f1.
double pair_energy(int pot, double r, double e, double s, double p2)
{
    switch (pot) {
        case HB_POT_GAUSS: return e * std::exp(-0.5 * (r / s) * (r / s));
        case HB_POT_YUKAWA: return e * std::exp(-s * r) / r;
        case HB_POT_MORSE: { const double e1 = std::exp(-s * (r - p2)); return e * (e1 * e1 - 2.0 * e1); }
        default: { const double sr6 = std::pow(s / r, 6.0); return 4.0 * e * (sr6 * sr6 - sr6); }
    }
}

// Per-type-pair device table from eps, sigma, r_cut (binary64 -> rounded once).
int upload_params(hb_system *h)
{
    const int nt2 = h->ntypes * h->ntypes;
    h->h_params.resize(nt2);
    h->h_paramsx.resize(nt2);
    double rc_max = 0.0;
    for (int p = 0; p < nt2; p++) {
        const double e = h->eps[p], s = h->sigma[p], rc = h->rcut[p], p2 = h->p2[p];
        PairParam pp;
        if (h->pot == HB_POT_LJ) {
            const double s6 = std::pow(s, 6.0);
            pp.lj1 = (float)(4.0 * e * s6 * s6);
            pp.lj2 = (float)(4.0 * e * s6);
        } else if (h->pot == HB_POT_GAUSS) {
            pp.lj1 = (float)e;
            pp.lj2 = (float)(0.5 / (s * s));
        } else {
            pp.lj1 = (float)e;      // Yukawa: eps, kappa; Morse: D0, a
            pp.lj2 = (float)s;
        }
        pp.rcut2 = (float)(rc * rc);
        pp.eshift = h->shift_mode == HB_SHIFT_ENERGY ? (float)pair_energy(h->pot, rc, e, s, p2) : 0.0f;
        h->h_params[p] = pp;
        const double ron = h->ron[p], d = rc * rc - ron * ron;
        // the smoothing is on where invD != 0: in HB_XPLOR mode and only where r_on < r_cut (reading x1)
        const bool smooth = h->shift_mode == HB_XPLOR && ron < rc;
        h->h_paramsx[p] = PairParamX{(float)(ron * ron), smooth ? (float)(1.0 / (d * d * d)) : 0.0f, (float)p2, 0.0f};
        if (rc > rc_max) rc_max = rc;
    }
    h->r_cut_max = (float)rc_max;
    HB_CK(cudaMemcpyAsync(h->params, h->h_params.data(), sizeof(PairParam) * nt2, cudaMemcpyHostToDevice, h->stream));
    HB_CK(cudaMemcpyAsync(h->paramsx, h->h_paramsx.data(), sizeof(PairParamX) * nt2, cudaMemcpyHostToDevice, h->stream));
    HB_CK(cudaStreamSynchronize(h->stream));  // h_params is pageable
    return HB_OK;
}

int stage_cap_max(const hb_system *h)
{
    // what is left of the opt-in shared memory after the static tables (TileShared and the scan scratch, < 4 KB) and
    // the larger of the two kernels' extras beside the staging area itself (both functions count cap * 16 bytes)
    const size_t extra = std::max(nlist_smem_bytes(h), force_smem_bytes(h)) - (size_t)h->geom.cap * 16;
    const int64_t left = (int64_t)h->smem_max - 8192 - (int64_t)extra;      // smem_attr(): the dynamic shared memory a launch may ask for
    return (int)std::max<int64_t>(64, std::min<int64_t>(65535, left / 16));
}

// Tile dimensions and staging capacity (tile.cuh).  Tunables override the choice.
int choose_tiles(hb_system *h, int min_cap)
{
    const int m = h->m;
    int tx = h->tun.tile_x, ty = h->tun.tile_y, tz = h->tun.tile_z;
    auto ntiles_of = [&](int ax, int ay, int az) {
        return (int64_t)cdiv(m, std::min(ax, m)) * cdiv(m, std::min(ay, m)) * cdiv(m, std::min(az, m));
    };
    if (tx <= 0 || ty <= 0 || tz <= 0) {
        // The largest brick (least halo per own particle) that still leaves every SM several tiles and holds at
        // most ~256 own particles (measured on B200: 2x2x1 at N = 64,000, 4x2x2 at 10^6, 4x4x4 for the WCA fluid
        // with its 2.5 particles per cell).
        const int cand[7][3] = {{4, 4, 4}, {4, 4, 2}, {4, 2, 2}, {2, 2, 2}, {2, 2, 1}, {2, 1, 1}, {1, 1, 1}};
        const double per_cell = (double)h->N / (double)h->ncells;
        int pick = 6;
        for (int k = 0; k < 7; k++) {
            const int ax = std::min(cand[k][0], m), ay = std::min(cand[k][1], m), az = std::min(cand[k][2], m);
            if (ntiles_of(ax, ay, az) >= (int64_t)6 * h->sm_count && per_cell * ax * ay * az <= 256.0) { pick = k; break; }
        }
        tx = cand[pick][0]; ty = cand[pick][1]; tz = cand[pick][2];
    }
    tx = std::min(tx, m); ty = std::min(ty, m); tz = std::min(tz, m);
    if ((tx + 2) * (ty + 2) * (tz + 2) > TILE_HMAX || ty * tz > TILE_ROWS_MAX) {
        h->err = "tile too large: (tx+2)(ty+2)(tz+2) must be <= 256 and ty*tz <= 32";
        return HB_EINVAL;
    }
    TileGeom g{};
    g.m = m; g.tx = tx; g.ty = ty; g.tz = tz;
    g.ntx = (int)cdiv(m, tx); g.nty = (int)cdiv(m, ty); g.ntz = (int)cdiv(m, tz);
    const int64_t nt = (int64_t)g.ntx * g.nty * g.ntz;
    if (nt > 0x7fffffff) { h->err = "too many tiles"; return HB_EINVAL; }
    g.ntiles = (int)nt;
    g.L = h->L;
    int cap = h->tun.stage_cap;
    if (cap <= 0) {
        const double per_cell = (double)h->N / (double)h->ncells;
        const double est = per_cell * (tx + 2) * (ty + 2) * (tz + 2);
        cap = (int)(1.3 * est) + 48;
    }
    cap = std::max(cap, min_cap);
    cap = round_up(std::max(cap, 64), 32);
    if (cap > stage_cap_max(h)) {
        if (min_cap > stage_cap_max(h) && tx * ty * tz > 1) {
            // shrink to one cell per tile (27 staged cells) and scale the requirement with the halo volume
            const int nh = (tx + 2) * (ty + 2) * (tz + 2);
            h->tun.tile_x = h->tun.tile_y = h->tun.tile_z = 1;
            return choose_tiles(h, (int)((int64_t)min_cap * 27 / nh));
        }
        if (min_cap > stage_cap_max(h)) {
            h->err = "a tile of cells with its halo holds " + std::to_string(min_cap) +
                     " particles: more than fit in shared memory; use smaller tiles (tile_x/y/z = 1)";
            return HB_ENOMEM;
        }
        cap = stage_cap_max(h);
    }
    g.cap = cap;
    h->own_est = (double)h->N / (double)h->ncells * tx * ty * tz;
    // fast geometry: tile + halo + what a particle can drift between builds is narrower than L/2 on every axis,
    // so the periodic image nearest to the tile centre is the right one for every staged particle
    {
        const double w = (double)h->L / m;
        const int tmax = std::max(tx, std::max(ty, tz));
        g.fast = ((0.5 * tmax + 1.0) * w + 2.0 * (double)h->r_buff + 0.05 * w < 0.5 * (double)h->L) ? 1 : 0;
    }
    g.eshift = g.cap <= 4096 ? 4 : 0;
    if (memcmp(&g, &h->geom, sizeof g) != 0) {
        destroy_graphs(h);
        h->nlist_valid = false;
    }
    h->geom = g;
    return HB_OK;
}

// r_max, m, cell arrays, tiles.  Reading c1.ii: m = floor(L / r_max) in binary64
// from the binary32 values of L and r_max.
int configure_geometry(hb_system *h)
{
    const float r_max = h->r_cut_max + h->r_buff;  // binary32 sum
    const int m = (int)std::floor((double)h->L / (double)r_max);
    if (!(r_max > 0.f) || m < 3 || (double)h->L < 2.0 * (double)r_max) {
        char buf[200];
        snprintf(buf, sizeof buf, "box too small: L = %g, r_max = %g gives m = %d cells per axis (need >= 3)", h->L, r_max, m);
        h->err = buf;
        return HB_EBOX;
    }
    if (r_max != h->r_max || m != h->m) {
        destroy_graphs(h);
        h->cells_valid = h->nlist_valid = false;
    }
    h->r_max = r_max;
    h->m = m;
    h->geometry_dirty = false;
    h->ncells = (int64_t)m * m * m;
    if (h->ncells > h->ncells_alloc) {
        dev_free_t(h, h->cell_count);
        dev_free_t(h, h->cell_local);
        dev_free_t(h, h->cell_start);
        dev_free_t(h, h->scan_sums);
        HB_TRY(dev_alloc_t(h, &h->cell_count, (size_t)h->ncells));
        HB_TRY(dev_alloc_t(h, &h->cell_local, (size_t)h->ncells));
        HB_TRY(dev_alloc_t(h, &h->cell_start, (size_t)h->ncells + 1));
        h->scan_sums_len = cdiv(h->ncells, 2048) + 16;
        HB_TRY(dev_alloc_t(h, &h->scan_sums, (size_t)h->scan_sums_len));
        HB_CK(cudaMemsetAsync(h->cell_count, 0, sizeof(int) * (size_t)h->ncells, h->stream));  // kept zero between builds
        h->ncells_alloc = h->ncells;
        destroy_graphs(h);
    }
    HB_TRY(choose_tiles(h, 0));
    h->stats.cells_per_axis = m;
    {   // per-type-pair list cutoffs (tunable nlist_pair_rcut): (r_cut,ab + r_buff)^2, each operation in binary32
        std::vector<float> t2((size_t)h->ntypes * h->ntypes);
        for (size_t p = 0; p < t2.size(); p++) { const float r = (float)h->rcut[p] + h->r_buff; t2[p] = r * r; }
        HB_CK(cudaMemcpyAsync(h->rmax2_pair, t2.data(), t2.size() * sizeof(float), cudaMemcpyHostToDevice, h->stream));
        HB_CK(cudaStreamSynchronize(h->stream));
    }
    return HB_OK;
}

int ensure_rows(hb_system *h, int pitch)
{
    pitch = round_up(pitch < 64 ? 64 : pitch, 64);   // 16-bit entries: 64 = 128 B
    const int64_t need = h->N * (int64_t)pitch + 1024;   // slack: the force kernel's list prefetch runs past a row's end
    if (need > h->nlist_alloc) {
        dev_free_t(h, h->nlist);
        HB_TRY(dev_alloc_t(h, &h->nlist, (size_t)need));
        h->nlist_alloc = need;
        destroy_graphs(h);
    }
    if (pitch != h->row_pitch) destroy_graphs(h);
    h->row_pitch = pitch;
    h->stats.row_pitch = pitch;
    h->nlist_valid = false;
    return HB_OK;
}

int initial_pitch(const hb_system *h)
{
    if (h->tun.row_pitch > 0) return h->tun.row_pitch;
    const double kPi = 3.14159265358979323846;
    const double n_est = 4.0 / 3.0 * kPi * std::pow((double)h->r_max, 3.0) * (double)h->N / std::pow((double)h->L, 3.0);
    return (int)(1.5 * n_est) + 24;
}

int read_flags(hb_system *h)
{
    HB_CK(cudaMemcpyAsync(h->h_flags, h->flags, sizeof(int) * FL_COUNT, cudaMemcpyDeviceToHost, h->stream));
    HB_CK(cudaStreamSynchronize(h->stream));
    return HB_OK;
}

int set_flag(hb_system *h, int which, int value)
{
    HB_CK(cudaMemsetAsync(h->flags + which, 0, sizeof(int), h->stream));
    if (value != 0) {
        h->h_flags[which] = value;
        HB_CK(cudaMemcpyAsync(h->flags + which, h->h_flags + which, sizeof(int), cudaMemcpyHostToDevice, h->stream));
        HB_CK(cudaStreamSynchronize(h->stream));
    }
    return HB_OK;
}

int clear_need_flags(hb_system *h)
{
    HB_CK(cudaMemsetAsync(h->flags + FL_NEED0, 0, 2 * sizeof(int), h->stream));
    return HB_OK;
}

// Algorithm 2 and the reorder into cell order: count (atomic slot per particle), scan, scatter, gather.
int enqueue_cells(hb_system *h, const int *pred)
{
    HB_CK(launch_cell_count(h, pred));
    HB_CK(launch_cell_scan(h, pred));
    HB_CK(launch_cell_scatter(h, pred));
    HB_CK(launch_cell_gather(h, pred));
    return HB_OK;
}

// Algorithm 2 + Algorithm 3, no host interaction (pred: device flag for early exit, or NULL).
int enqueue_rebuild(hb_system *h, const int *pred)
{
    if (coop_mode(h) == 2) {
        HB_CK(launch_rebuild_coop(h, pred, true));
        return HB_OK;
    }
    if (coop_mode(h) == 1) HB_CK(launch_rebuild_coop(h, pred, false));
    else HB_TRY(enqueue_cells(h, pred));
    HB_CK(launch_nlist(h, pred, true));
    return HB_OK;
}

// Build with the host in the loop: detects row and staging overflow, grows, rebuilds.
int build_nlist_sync(hb_system *h)
{
    if (!h->have_state) { h->err = "no state: call hb_set_state first"; return HB_ESTATE; }
    if (h->geometry_dirty || h->m == 0) HB_TRY(configure_geometry(h));   // hb_set_rcut_pair after a build: new r_max, m, table
    if (h->row_pitch == 0) HB_TRY(ensure_rows(h, initial_pitch(h)));
    for (int attempt = 0; attempt < 16; attempt++) {
        HB_TRY(enqueue_rebuild(h, nullptr));
        HB_TRY(read_flags(h));
        h->forces_valid = false;   // the storage order changed under the force array
        h->moved = false;
        if (h->h_flags[FL_BAD]) {
            h->err = "a particle is non-finite or outside the box";
            set_flag(h, FL_BAD, 0);
            h->cells_valid = h->nlist_valid = false;
            return HB_ENAN;
        }
        h->stats.rebuilds = h->h_flags[FL_BUILDS];
        if (h->h_flags[FL_STAGE_OVER]) {
            const int needed = h->h_flags[FL_STAGE_OVER];
            h->stats.overflow_retries++;
            HB_TRY(set_flag(h, FL_STAGE_OVER, 0));
            HB_TRY(set_flag(h, FL_OVERFLOWED, 0));
            HB_TRY(choose_tiles(h, (int)(needed * (1.0 + 0.01 * h->tun.grow_pct)) + 32));
            continue;
        }
        h->stats.max_nbrs = h->h_flags[FL_MAX_NBRS];
        if (h->h_flags[FL_MAX_NBRS] <= h->row_pitch) {
            HB_TRY(set_flag(h, FL_OVERFLOWED, 0));
            HB_TRY(clear_need_flags(h));
            h->cells_valid = h->nlist_valid = true;
            return HB_OK;
        }
        h->stats.overflow_retries++;
        HB_TRY(ensure_rows(h, (int)(h->h_flags[FL_MAX_NBRS] * (1.0 + 0.01 * h->tun.grow_pct)) + 8));
    }
    h->err = "neighbor-list rows keep overflowing";
    return HB_ENOMEM;
}

int ensure_forces(hb_system *h)
{
    if (!h->nlist_valid) HB_TRY(build_nlist_sync(h));
    if (!h->forces_valid) {
        HB_CK(launch_force(h, nullptr));
        h->forces_valid = true;
    }
    return HB_OK;
}

int ensure_sort_buffers(hb_system *h)
{
    if (h->keys) return HB_OK;
    const size_t N = (size_t)h->N;
    HB_TRY(dev_alloc_t(h, &h->keys, N));
    HB_TRY(dev_alloc_t(h, &h->keys2, N));
    HB_TRY(dev_alloc_t(h, &h->sperm, N));
    HB_TRY(dev_alloc_t(h, &h->sperm2, N));
    HB_TRY(dev_alloc_t(h, &h->force2, N));
    HB_TRY(dev_alloc_t(h, &h->virial2, 2 * N));
    const int64_t ntiles = cdiv(h->N, 512);
    h->radix_counts_len = 256 * ntiles;
    HB_TRY(dev_alloc_t(h, &h->radix_counts, (size_t)(2 * h->radix_counts_len + 8)));
    const int64_t need_tmp = cdiv(h->radix_counts_len, 2048) + 16;
    if (need_tmp > h->scan_tmp_len) {
        dev_free_t(h, h->scan_tmp);
        HB_TRY(dev_alloc_t(h, &h->scan_tmp, (size_t)need_tmp));
        h->scan_tmp_len = need_tmp;
    }
    return HB_OK;
}

int sort_internal(hb_system *h)
{
    if (!h->have_state) { h->err = "no state"; return HB_ESTATE; }
    HB_TRY(ensure_sort_buffers(h));
    HB_CK(launch_sfc_keys(h));
    HB_CK(launch_radix_sort(h, 24));
    HB_CK(launch_gather_state(h));
    // copy back rather than swap pointers: captured graphs keep pointing at the live set
    const size_t N = (size_t)h->N;
    HB_CK(cudaMemcpyAsync(h->pos(), h->pos_build, N * sizeof(float4), cudaMemcpyDeviceToDevice, h->stream));
    HB_CK(cudaMemcpyAsync(h->vel, h->vel2, N * sizeof(float4), cudaMemcpyDeviceToDevice, h->stream));
    HB_CK(cudaMemcpyAsync(h->force, h->force2, N * sizeof(float4), cudaMemcpyDeviceToDevice, h->stream));
    HB_CK(cudaMemcpyAsync(h->virial, h->virial2, 2 * N * sizeof(float4), cudaMemcpyDeviceToDevice, h->stream));
    HB_CK(cudaMemcpyAsync(h->image, h->image2, 3 * N * sizeof(int), cudaMemcpyDeviceToDevice, h->stream));
    HB_CK(cudaMemcpyAsync(h->tag, h->tag2, N * sizeof(uint32_t), cudaMemcpyDeviceToDevice, h->stream));
    h->cells_valid = h->nlist_valid = false;
    h->moved = true;
    h->bk_valid = false;
    h->stats.sorts++;
    h->since_sort = 0;
    return HB_OK;
}

NveArgs make_nve(hb_system *h, float dt, bool kick_prev, bool kick_drift, float4 *pos_out, cudaGraphConditionalHandle cond,
                 bool use_cond)
{
    NveArgs a{};
    a.vel = h->vel;
    a.image = h->image;
    a.pos_build = h->pos_build;
    a.pos_out = pos_out;
    a.dt = dt;
    const float hb = 0.5f * h->r_buff;
    a.half_buff2 = hb * hb;
    a.kick_prev = kick_prev ? 1 : 0;
    a.kick_drift = kick_drift ? 1 : 0;
    a.forces_only = (kick_prev && kick_drift && h->tun.thermo_every == 0) ? 1 : 0;
    a.need_set = FL_NEED0 + (h->parity & 1);
    a.need_clear = FL_NEED0 + ((h->parity + 1) & 1);
    a.cond = cond;
    a.use_cond = use_cond ? 1 : 0;
    a.ens = h->ens.mode;
    a.T = (float)h->ens.T;
    a.par = (float)h->ens.par;
    a.gdof = 3.0 * (double)h->N - 3.0;
    a.seed = h->ens.seed;
    a.kick_step = h->parity - h->parity0 - 1;   // the step whose drift was the last one launched
    a.tstate = h->tstate;
    a.tag = h->tag;
    return a;
}

// The launches of an n-step chunk without conditional nodes (graph_mode 1 inside a capture, graph_mode 3 straight
// into the stream): every rebuild kernel takes the drift's flag as its predicate.  Advances h->cur / h->parity.
int enqueue_chunk_pred(hb_system *h, int n, float dt)
{
    const bool fuse = h->tun.fuse_nve != 0;
    for (int s = 0; s < n; s++) {
        const int need_flag = FL_NEED0 + (h->parity & 1);
        if (s == 0) {
            HB_CK(launch_nve(h, make_nve(h, dt, false, true, h->pos(), 0, false)));
        } else if (fuse) {
            const NveArgs a = make_nve(h, dt, true, true, h->posbuf[h->cur ^ 1], 0, false);
            HB_CK(launch_force(h, &a));
            h->cur ^= 1;
        } else {
            HB_CK(launch_force(h, nullptr));
            HB_CK(launch_nve(h, make_nve(h, dt, true, true, h->pos(), 0, false)));
        }
        h->parity++;
        HB_TRY(enqueue_rebuild(h, h->flags + need_flag));
    }
    if (fuse) {
        const NveArgs a = make_nve(h, dt, true, false, h->pos(), 0, false);
        HB_CK(launch_force(h, &a));
    } else {
        HB_CK(launch_force(h, nullptr));
        HB_CK(launch_nve(h, make_nve(h, dt, true, false, h->pos(), 0, false)));
    }
    return HB_OK;
}

// ---- hb_run_nve: n steps as one CUDA graph ----
// fuse_nve = 1:  nve(drift) [rebuild?]  { lj+nve(kick, kick, drift) [rebuild?] } x (n-1)  lj+nve(kick)
// fuse_nve = 0:  nve(drift) [rebuild?]  { lj  nve(kick, kick, drift) [rebuild?] } x (n-1)  lj  nve(kick)
int build_graph(hb_system *h, int n, float dt, hb_system::GraphEntry *out)
{
    const int mode = h->tun.graph_mode;
    const bool fuse = h->tun.fuse_nve != 0;
    cudaStream_t cs = nullptr, cs2 = nullptr;
    HB_CK(cudaStreamCreateWithFlags(&cs, cudaStreamNonBlocking));
    HB_CK(cudaStreamCreateWithFlags(&cs2, cudaStreamNonBlocking));
    cudaGraph_t g = nullptr;
    HB_CK(cudaGraphCreate(&g, 0));
    cudaStream_t saved = h->stream;
    const int64_t saved_launches = h->stats.kernel_launches;
    const int saved_cur = h->cur, saved_parity = h->parity, saved_parity0 = h->parity0;
    h->cur = 0;       // every chunk starts from posbuf[0] and drift parity 0 (run_chunk sees to it): one graph per n
    h->parity = 0;
    h->parity0 = 0;   // make_nve bakes kick_step = parity - parity0 - 1 into the captured kernel parameters: a value left
                      // by hb_step_nve (step_sync) would shift the Langevin generator's step number by the call history
    int rc = HB_OK;
    auto fail = [&](const char *what, cudaError_t e) {
        h->err = std::string(what) + ": " + cudaGetErrorString(e);
        rc = HB_ECUDA;
    };
    cudaError_t e = cudaStreamBeginCaptureToGraph(cs, g, nullptr, nullptr, 0, cudaStreamCaptureModeRelaxed);
    if (e != cudaSuccess) { fail("cudaStreamBeginCaptureToGraph", e); }
    if (rc == HB_OK) {
        h->stream = cs;
        for (int s = 0; s < n && rc == HB_OK; s++) {
            cudaGraphConditionalHandle cond = 0;
            if (mode == 2) {
                e = cudaGraphConditionalHandleCreate(&cond, g, 0, cudaGraphCondAssignDefault);
                if (e != cudaSuccess) { fail("cudaGraphConditionalHandleCreate", e); break; }
            }
            // the drift of step s (after the force of the state it starts from, except for s = 0: forces are valid)
            const int need_flag = FL_NEED0 + (h->parity & 1);
            if (s == 0) {
                e = launch_nve(h, make_nve(h, dt, false, true, h->pos(), cond, mode == 2));
            } else if (fuse) {
                float4 *other = h->posbuf[h->cur ^ 1];
                const NveArgs a = make_nve(h, dt, true, true, other, cond, mode == 2);
                e = launch_force(h, &a);
                h->cur ^= 1;
            } else {
                e = launch_force(h, nullptr);
                if (e == cudaSuccess) e = launch_nve(h, make_nve(h, dt, true, true, h->pos(), cond, mode == 2));
            }
            if (e != cudaSuccess) { fail("step kernel (capture)", e); break; }
            h->parity++;
            if (mode == 2) {
                cudaStreamCaptureStatus st;
                const cudaGraphNode_t *deps = nullptr;
                size_t ndeps = 0;
                cudaGraph_t cg = nullptr;
                e = cudaStreamGetCaptureInfo_v2(cs, &st, nullptr, &cg, &deps, &ndeps);
                if (e != cudaSuccess) { fail("cudaStreamGetCaptureInfo_v2", e); break; }
                cudaGraphNodeParams np = {cudaGraphNodeTypeConditional};
                np.type = cudaGraphNodeTypeConditional;
                np.conditional.handle = cond;
                np.conditional.type = cudaGraphCondTypeIf;
                np.conditional.size = 1;
                cudaGraphNode_t node = nullptr;
                e = cudaGraphAddNode(&node, g, deps, ndeps, &np);
                if (e != cudaSuccess) { fail("cudaGraphAddNode(conditional)", e); break; }
                cudaGraph_t body = np.conditional.phGraph_out[0];
                e = cudaStreamBeginCaptureToGraph(cs2, body, nullptr, nullptr, 0, cudaStreamCaptureModeRelaxed);
                if (e != cudaSuccess) { fail("cudaStreamBeginCaptureToGraph(body)", e); break; }
                h->stream = cs2;
                rc = enqueue_rebuild(h, nullptr);
                h->stream = cs;
                cudaGraph_t tmp = nullptr;
                e = cudaStreamEndCapture(cs2, &tmp);
                if (rc != HB_OK) break;
                if (e != cudaSuccess) { fail("cudaStreamEndCapture(body)", e); break; }
                e = cudaStreamUpdateCaptureDependencies(cs, &node, 1, cudaStreamSetCaptureDependencies);
                if (e != cudaSuccess) { fail("cudaStreamUpdateCaptureDependencies", e); break; }
            } else {
                rc = enqueue_rebuild(h, h->flags + need_flag);
                if (rc != HB_OK) break;
            }
        }
        if (rc == HB_OK) {
            // forces of the last state and the second half kick of the last step
            if (fuse) {
                const NveArgs a = make_nve(h, dt, true, false, h->pos(), 0, false);
                e = launch_force(h, &a);
            } else {
                e = launch_force(h, nullptr);
                if (e == cudaSuccess) e = launch_nve(h, make_nve(h, dt, true, false, h->pos(), 0, false));
            }
            if (e != cudaSuccess) fail("final kernel (capture)", e);
        }
        cudaGraph_t tmp = nullptr;
        e = cudaStreamEndCapture(cs, &tmp);
        if (rc == HB_OK && e != cudaSuccess) fail("cudaStreamEndCapture", e);
    }
    h->stream = saved;
    h->stats.kernel_launches = saved_launches;
    h->cur = saved_cur;
    h->parity = saved_parity;
    h->parity0 = saved_parity0;
    cudaGraphExec_t ex = nullptr;
    if (rc == HB_OK) {
        e = cudaGraphInstantiate(&ex, g, 0);
        if (e != cudaSuccess) fail("cudaGraphInstantiate", e);
    }
    cudaStreamDestroy(cs);
    cudaStreamDestroy(cs2);
    if (rc != HB_OK) {
        cudaGetLastError();
        if (g) cudaGraphDestroy(g);
        return rc;
    }
    out->g = g;
    out->e = ex;
    h->stats.graph_builds++;
    out->nkernels_fixed = (fuse ? n + 1 : 2 * n + 1) + (mode == 1 ? n * rebuild_kernels(h) : 0);
    return HB_OK;
}

int backup_state(hb_system *h)
{
    const size_t N = (size_t)h->N;
    if (!h->bk_pos) {
        HB_TRY(dev_alloc_t(h, &h->bk_pos, N));
        HB_TRY(dev_alloc_t(h, &h->bk_vel, N));
        HB_TRY(dev_alloc_t(h, &h->bk_image, 3 * N));
        HB_TRY(dev_alloc_t(h, &h->bk_tag, N));
    }
    HB_CK(launch_state_copy(h, false));
    h->bk_cur = h->cur;
    h->bk_parity = h->parity;
    h->bk_valid = true;
    return HB_OK;
}

int restore_state(hb_system *h)
{
    h->cur = h->bk_cur;
    h->parity = h->bk_parity;
    HB_CK(launch_state_copy(h, true));
    HB_CK(launch_rtag(h));
    HB_TRY(clear_need_flags(h));
    // forces and virials are not saved: the rebuild that follows a restore changes the order, they are recomputed
    h->nlist_valid = h->cells_valid = h->forces_valid = false;
    h->moved = true;
    return HB_OK;
}

// One step with the host reading the rebuild flag (hb_step_nve and graph_mode 0).
int step_sync(hb_system *h, float dt)
{
    HB_TRY(ensure_forces(h));
    h->parity0 = h->parity;
    if (h->ens.mode == 2) {
        *reinterpret_cast<long long *>(h->h_tstate + TS_LBASE) = (long long)h->lang_steps;
        HB_CK(cudaMemcpyAsync(h->tstate + TS_LBASE, h->h_tstate + TS_LBASE, sizeof(double), cudaMemcpyHostToDevice, h->stream));
    }
    const NveArgs a = make_nve(h, dt, false, true, h->pos(), 0, false);
    HB_CK(launch_nve(h, a));
    h->parity++;
    h->moved = true;
    HB_TRY(read_flags(h));
    if (h->h_flags[a.need_set]) HB_TRY(build_nlist_sync(h));
    HB_CK(launch_force(h, nullptr));
    h->forces_valid = true;
    HB_CK(launch_nve(h, make_nve(h, dt, true, false, h->pos(), 0, false)));
    h->stats.steps++;
    if (h->ens.mode == 2) h->lang_steps++;
    return HB_OK;
}

// Every chunk starts from posbuf[0] and drift parity 0, so that ONE graph per chunk length serves every call.
int normalize_for_chunk(hb_system *h)
{
    if (h->cur != 0) {
        HB_CK(cudaMemcpyAsync(h->posbuf[0], h->posbuf[1], (size_t)h->N * sizeof(float4), cudaMemcpyDeviceToDevice, h->stream));
        h->cur = 0;
    }
    h->parity = 0;
    h->parity0 = 0;
    if (h->ens.mode == 2) {       // the generator's stream = number of the time step: tell the device where the chunk starts
        *reinterpret_cast<long long *>(h->h_tstate + TS_LBASE) = (long long)h->lang_steps;
        HB_CK(cudaMemcpyAsync(h->tstate + TS_LBASE, h->h_tstate + TS_LBASE, sizeof(double), cudaMemcpyHostToDevice, h->stream));
    }
    return clear_need_flags(h);   // no decision is pending between chunks: every drift's rebuild ran inside its chunk
}

int chunk_kernels(const hb_system *h, int n) { return (h->tun.fuse_nve ? n + 1 : 2 * n + 1) + n * rebuild_kernels(h); }

// The chunk lengths hb_run_nve uses are graph_steps and the powers of two below it; all their graphs are built at
// the first call, so that no later call captures or instantiates anything (hb_stats: graph_builds).
int ensure_graphs(hb_system *h, float dt)
{
    if (dt != h->graph_dt || !(h->ens == h->graph_ens)) { destroy_graphs(h); h->graph_dt = dt; h->graph_ens = h->ens; }
    if (!h->graphs.empty() || h->tun.graph_mode == 0 || h->tun.graph_mode == 3) return HB_OK;
    Range r("hb:build_graphs");
    std::vector<int> sizes{h->tun.graph_steps};
    for (int n = 1; n < h->tun.graph_steps; n <<= 1) sizes.push_back(n);
    for (int n : sizes) {
        hb_system::GraphEntry ge;
        HB_TRY(build_graph(h, n, dt, &ge));
        h->graphs.emplace((int64_t)n, ge);
    }
    return HB_OK;
}

int run_chunk(hb_system *h, float dt, int n)
{
    if (h->tun.graph_mode == 0) {
        for (int s = 0; s < n; s++) HB_TRY(step_sync(h, dt));
        return HB_OK;
    }
    Range r("hb:chunk");
    for (int attempt = 0; attempt < 8; attempt++) {
        HB_TRY(ensure_forces(h));
        HB_TRY(ensure_graphs(h, dt));
        HB_TRY(normalize_for_chunk(h));
        const bool plain = h->tun.graph_mode == 3;   // the launches of mode 1, issued one by one (for profilers)
        auto it = h->graphs.find((int64_t)n);
        if (!plain && it == h->graphs.end()) {       // a length outside the prebuilt set (never from hb_run_nve)
            hb_system::GraphEntry ge;
            HB_TRY(build_graph(h, n, dt, &ge));
            it = h->graphs.emplace((int64_t)n, ge).first;
        }
        HB_TRY(backup_state(h));
        const int builds_before = h->h_flags[FL_BUILDS];
        if (plain) {
            const int64_t l0 = h->stats.kernel_launches;
            HB_TRY(enqueue_chunk_pred(h, n, dt));
            h->cur = 0; h->parity = 0;              // advanced again below, as after a graph launch
            h->stats.kernel_launches = l0;
        } else {
            HB_CK(cudaGraphLaunch(it->second.e, h->stream));
            h->stats.graph_launches++;
        }
        HB_TRY(read_flags(h));
        const int nb = h->h_flags[FL_BUILDS] - builds_before;
        h->stats.kernel_launches += chunk_kernels(h, n) - (h->tun.graph_mode == 2 ? (n - nb) * rebuild_kernels(h) : 0);
        h->stats.rebuilds = h->h_flags[FL_BUILDS];
        if (h->tun.fuse_nve) h->cur ^= (n - 1) & 1;
        h->parity += n;
        h->moved = true;
        h->forces_valid = true;   // the graph's last kernel evaluated the forces in the final order
        const int rows_needed = h->h_flags[FL_OVERFLOWED], slots_needed = h->h_flags[FL_STAGE_OVER];
        if (!rows_needed && !slots_needed) {
            if (h->h_flags[FL_BAD]) {
                h->err = "a particle is non-finite or outside the box";
                set_flag(h, FL_BAD, 0);
                h->nlist_valid = h->cells_valid = h->forces_valid = false;
                return HB_ENAN;
            }
            if (nb > 0) h->stats.max_nbrs = h->h_flags[FL_MAX_NBRS];
            h->stats.steps += n;
            if (h->ens.mode == 2) h->lang_steps += n;
            return HB_OK;
        }
        // Some build inside the chunk overflowed its rows or its staging area: go back, grow, redo.
        // This comes BEFORE the bad-particle test: the steps after the overflowing build ran with truncated rows
        // or skipped tiles, so whatever they flagged (a particle thrown out of the box) is a consequence and is
        // undone with them.
        h->stats.overflow_retries++;
        HB_TRY(restore_state(h));
        HB_TRY(set_flag(h, FL_OVERFLOWED, 0));
        HB_TRY(set_flag(h, FL_STAGE_OVER, 0));
        HB_TRY(set_flag(h, FL_BAD, 0));
        if (slots_needed) HB_TRY(choose_tiles(h, (int)(slots_needed * (1.0 + 0.01 * h->tun.grow_pct)) + 32));
        if (rows_needed) HB_TRY(ensure_rows(h, (int)(rows_needed * (1.0 + 0.01 * h->tun.grow_pct)) + 8));
        HB_TRY(build_nlist_sync(h));
    }
    h->err = "neighbor-list rows keep overflowing inside hb_run_nve";
    return HB_ENOMEM;
}

// The binary64 variant (tunable precision = 64, dp.cu): one velocity-Verlet step per host iteration.
int dp_run(hb_system *h, double dt, int64_t nsteps, int64_t sort_period)
{
    if (h->ens.mode != 0) { h->err = "the binary64 variant integrates NVE only"; return HB_EINVAL; }
    if (!h->dp.have) HB_TRY(dp_from_f32(h));
    for (int64_t s = 0; s < nsteps; s++) {
        if (sort_period > 0 && (h->since_sort < 0 || h->since_sort >= sort_period)) {
            if (!h->nlist_valid) HB_TRY(build_nlist_sync(h));
            HB_TRY(sort_internal(h));
            h->since_sort = 0;
        }
        if (!h->nlist_valid) { HB_TRY(build_nlist_sync(h)); h->dp.forces_valid = false; }
        if (!h->dp.forces_valid) HB_TRY(dp_force(h));
        HB_TRY(dp_nve(h, dt, 1));
        h->moved = true;
        h->forces_valid = false;          // the binary32 force arrays are not kept up in this mode
        HB_TRY(set_flag(h, FL_CHECK, 0));
        HB_CK(launch_disp_check(h));      // reading c3 on the binary32 mirror
        HB_TRY(read_flags(h));
        if (h->h_flags[FL_CHECK]) HB_TRY(build_nlist_sync(h));
        HB_TRY(dp_force(h));
        HB_TRY(dp_nve(h, dt, 2));
        h->stats.steps++;
        if (h->since_sort >= 0) h->since_sort++;
    }
    return HB_OK;
}

// accessor staging area, owned by the handle (grows, never shrinks)
int ensure_stage(hb_system *h, size_t bytes)
{
    if (bytes <= h->acc_cap) return HB_OK;
    dev_free(h, h->acc_stage);
    h->acc_stage = nullptr;
    h->acc_cap = 0;
    HB_TRY(dev_alloc(h, &h->acc_stage, bytes));
    h->acc_cap = bytes;
    return HB_OK;
}

}  // namespace

#define HB_NEED(h)            \
    if (!(h)) return HB_EINVAL; \
    (h)->err.clear();

extern "C" {

const char *hb_version(void) { return "libhb 0.1 (sm_100a)"; }

const char *hb_last_error(hb_system *h) { return h ? h->err.c_str() : "null handle"; }

int hb_create(hb_system **out, int64_t N, double L, int ntypes, const double *eps, const double *sigma, void *cuda_stream,
              const hb_allocator *alloc)
{
    if (!out) return HB_EINVAL;
    *out = nullptr;
    if (N <= 0 || N >= (int64_t)1 << 31 || !(L > 0.0) || ntypes <= 0 || ntypes > 64 || !eps || !sigma) return HB_EINVAL;
    for (int a = 0; a < ntypes; a++)
        for (int b = 0; b < ntypes; b++)
            if (eps[a * ntypes + b] != eps[b * ntypes + a] || sigma[a * ntypes + b] != sigma[b * ntypes + a] ||
                !(sigma[a * ntypes + b] > 0.0))
                return HB_EINVAL;
    hb_system *h = new (std::nothrow) hb_system();
    if (!h) return HB_ENOMEM;
    h->N = N;
    h->L = (float)L;
    h->ntypes = ntypes;
    h->eps.assign(eps, eps + ntypes * ntypes);
    h->sigma.assign(sigma, sigma + ntypes * ntypes);
    h->rcut.resize(ntypes * ntypes);
    for (int p = 0; p < ntypes * ntypes; p++) h->rcut[p] = (double)(float)(2.5 * sigma[p]);
    h->ron.resize(ntypes * ntypes);
    for (int p = 0; p < ntypes * ntypes; p++) h->ron[p] = (double)(float)(1.5 * sigma[p]);
    h->p2.assign((size_t)ntypes * ntypes, 0.0);
    h->stream = (cudaStream_t)cuda_stream;
    if (alloc && alloc->alloc && alloc->free) { h->alloc = *alloc; h->has_alloc = true; }
    *out = h;  // from here on the caller can read hb_last_error and must hb_destroy

    const size_t n = (size_t)N;
    HB_TRY(dev_alloc_t(h, &h->posbuf[0], n));
    HB_TRY(dev_alloc_t(h, &h->posbuf[1], n));
    HB_TRY(dev_alloc_t(h, &h->vel, n));
    HB_TRY(dev_alloc_t(h, &h->force, n));
    HB_TRY(dev_alloc_t(h, &h->virial, 2 * n));
    HB_TRY(dev_alloc_t(h, &h->image, 3 * n));
    HB_TRY(dev_alloc_t(h, &h->tag, n));
    HB_TRY(dev_alloc_t(h, &h->rtag, n));
    HB_TRY(dev_alloc_t(h, &h->pos_build, n));
    HB_TRY(dev_alloc_t(h, &h->vel2, n));
    HB_TRY(dev_alloc_t(h, &h->image2, 3 * n));
    HB_TRY(dev_alloc_t(h, &h->tag2, n));
    HB_TRY(dev_alloc_t(h, &h->cell_id, n));
    HB_TRY(dev_alloc_t(h, &h->cell_rank, n));
    HB_TRY(dev_alloc_t(h, &h->perm, n));
    HB_TRY(dev_alloc_t(h, &h->nlistn, n));
    HB_TRY(dev_alloc_t(h, &h->params, (size_t)ntypes * ntypes));
    HB_TRY(dev_alloc_t(h, &h->paramsx, (size_t)ntypes * ntypes));
    HB_TRY(dev_alloc_t(h, &h->rmax2_pair, (size_t)ntypes * ntypes));
    HB_TRY(dev_alloc_t(h, &h->flags, (size_t)FL_COUNT));
    HB_CK(cudaMallocHost((void **)&h->h_flags, sizeof(int) * FL_COUNT));
    HB_CK(cudaMallocHost((void **)&h->h_thermo, sizeof(double) * 16));
    HB_CK(cudaMallocHost((void **)&h->h_total, sizeof(int) * 2));
    HB_CK(cudaMallocHost((void **)&h->h_tstate, sizeof(double) * TS_COUNT));
    memset(h->h_tstate, 0, sizeof(double) * TS_COUNT);
    HB_TRY(dev_alloc_t(h, &h->tstate, (size_t)TS_COUNT));
    HB_TRY(dev_alloc_t(h, &h->bk_tstate, (size_t)TS_COUNT));
    HB_CK(cudaMemsetAsync(h->tstate, 0, sizeof(double) * TS_COUNT, h->stream));
    HB_TRY(dev_alloc_t(h, &h->acc_counts, n + 1));
    HB_TRY(dev_alloc_t(h, &h->acc_rows, n + 2));
    memset(h->h_flags, 0, sizeof(int) * FL_COUNT);
    HB_CK(cudaMemsetAsync(h->flags, 0, sizeof(int) * FL_COUNT, h->stream));
    HB_CK(cudaMemsetAsync(h->posbuf[1], 0, sizeof(float4) * n, h->stream));   // never read before it is written, but never garbage
    HB_CK(cudaMemsetAsync(h->force, 0, sizeof(float4) * n, h->stream));
    HB_CK(cudaMemsetAsync(h->virial, 0, sizeof(float4) * 2 * n, h->stream));
    int dev = 0, sms = 148, smem = 227 * 1024;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    cudaDeviceGetAttribute(&smem, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev);
    h->sm_count = sms;
    h->smem_max = smem;
    h->thermo_blocks = (int)std::min<int64_t>(cdiv(N, 256), (int64_t)sms * 4);
    HB_TRY(dev_alloc_t(h, &h->thermo_part, (size_t)(h->thermo_blocks + 2) * 11));
    HB_TRY(upload_params(h));
    return HB_OK;
}

int hb_destroy(hb_system *h)
{
    if (!h) return HB_EINVAL;
    cudaStreamSynchronize(h->stream);
    destroy_graphs(h);
    dp_release(h);
    dev_free(h, h->acc_stage);
    dev_free(h, h->acc_counts);
    dev_free(h, h->acc_rows);
    if (h->h_total) cudaFreeHost(h->h_total);
    if (h->h_tstate) cudaFreeHost(h->h_tstate);
    dev_free(h, h->tstate);
    dev_free(h, h->bk_tstate);
    void *ptrs[] = {h->posbuf[0], h->posbuf[1], h->vel, h->force, h->virial, h->image, h->tag, h->rtag, h->pos_build, h->vel2,
                    h->force2, h->virial2, h->image2, h->tag2, h->bk_pos, h->bk_vel, h->bk_force, h->bk_virial, h->bk_image,
                    h->bk_tag, h->params, h->paramsx, h->rmax2_pair, h->cell_count, h->cell_local, h->cell_start, h->cell_id, h->cell_rank, h->perm,
                    h->scan_sums, h->scan_tmp, h->nlist, h->nlistn, h->keys, h->keys2, h->sperm, h->sperm2, h->radix_counts,
                    h->flags, h->thermo_part};
    for (void *p : ptrs) dev_free(h, p);
    if (h->h_flags) cudaFreeHost(h->h_flags);
    if (h->h_thermo) cudaFreeHost(h->h_thermo);
    cudaGetLastError();
    delete h;
    return HB_OK;
}

int hb_set_state(hb_system *h, const float *pos_xyz, const int32_t *type, const float *vel_xyz, const int32_t *image,
                 int on_device)
{
    HB_NEED(h);
    if (!pos_xyz || !vel_xyz) { h->err = "pos_xyz and vel_xyz are required"; return HB_EINVAL; }
    const size_t N = (size_t)h->N;
    const float *dpos = pos_xyz, *dvel = vel_xyz;
    const int32_t *dtype = type, *dimg = image;
    if (!on_device) {
        const size_t bytes = N * (3 * 4 + 4 + 3 * 4 + 3 * 4);
        HB_TRY(ensure_stage(h, bytes));
        char *base = (char *)h->acc_stage;
        float *spos = (float *)base;
        float *svel = (float *)(base + N * 12);
        int32_t *stype = (int32_t *)(base + N * 24);
        int32_t *simg = (int32_t *)(base + N * 28);
        HB_CK(cudaMemcpyAsync(spos, pos_xyz, N * 12, cudaMemcpyHostToDevice, h->stream));
        HB_CK(cudaMemcpyAsync(svel, vel_xyz, N * 12, cudaMemcpyHostToDevice, h->stream));
        if (type) HB_CK(cudaMemcpyAsync(stype, type, N * 4, cudaMemcpyHostToDevice, h->stream));
        if (image) HB_CK(cudaMemcpyAsync(simg, image, N * 12, cudaMemcpyHostToDevice, h->stream));
        dpos = spos; dvel = svel; dtype = type ? stype : nullptr; dimg = image ? simg : nullptr;
    }
    HB_CK(launch_pack_state(h, dpos, dtype, dvel, dimg));
    HB_TRY(read_flags(h));    // synchronises: the caller's host buffers may be pageable; and the type check below
    h->have_state = true;
    h->cells_valid = h->nlist_valid = h->forces_valid = h->bk_valid = false;
    h->moved = true;
    h->since_sort = -1;
    h->lang_steps = 0;
    HB_CK(cudaMemsetAsync(h->tstate, 0, sizeof(double) * TS_COUNT, h->stream));
    if (h->h_flags[FL_BADTYPE]) {
        HB_TRY(set_flag(h, FL_BADTYPE, 0));
        h->have_state = false;
        h->err = "a particle type is outside 0 .. ntypes-1";
        return HB_EINVAL;
    }
    h->dp.have = h->dp.forces_valid = false;
    if (h->tun.precision == 64) HB_TRY(dp_from_f32(h));
    return HB_OK;
}

int hb_set_state_f64(hb_system *h, const double *pos_xyz, const int32_t *type, const double *vel_xyz, const int32_t *image, int on_device)
{
    HB_NEED(h);
    if (!pos_xyz || !vel_xyz) { h->err = "pos_xyz and vel_xyz are required"; return HB_EINVAL; }
    const size_t N = (size_t)h->N;
    // staging: [pos f64 | vel f64 | type | image | pos f32 | vel f32]
    HB_TRY(ensure_stage(h, N * (24 + 24 + 4 + 12 + 12 + 12)));
    char *base = (char *)h->acc_stage;
    double *dpos = (double *)base, *dvel = (double *)(base + N * 24);
    int32_t *dtype = (int32_t *)(base + N * 48), *dimg = (int32_t *)(base + N * 52);
    float *fpos = (float *)(base + N * 64), *fvel = (float *)(base + N * 76);
    const cudaMemcpyKind kind = on_device ? cudaMemcpyDeviceToDevice : cudaMemcpyHostToDevice;
    HB_CK(cudaMemcpyAsync(dpos, pos_xyz, N * 24, kind, h->stream));
    HB_CK(cudaMemcpyAsync(dvel, vel_xyz, N * 24, kind, h->stream));
    if (type) HB_CK(cudaMemcpyAsync(dtype, type, N * 4, kind, h->stream));
    if (image) HB_CK(cudaMemcpyAsync(dimg, image, N * 12, kind, h->stream));
    HB_TRY(dp_set_state(h, dpos, dvel, image ? dimg : nullptr, fpos, fvel));
    HB_CK(launch_pack_state(h, fpos, type ? dtype : nullptr, fvel, image ? dimg : nullptr));
    HB_TRY(read_flags(h));
    h->have_state = true;
    h->cells_valid = h->nlist_valid = h->forces_valid = h->bk_valid = false;
    h->moved = true;
    h->since_sort = -1;
    h->lang_steps = 0;
    HB_CK(cudaMemsetAsync(h->tstate, 0, sizeof(double) * TS_COUNT, h->stream));
    if (h->h_flags[FL_BADTYPE] || h->h_flags[FL_BAD]) {
        const bool badtype = h->h_flags[FL_BADTYPE] != 0;
        HB_TRY(set_flag(h, FL_BADTYPE, 0));
        HB_TRY(set_flag(h, FL_BAD, 0));
        h->have_state = false;
        h->dp.have = false;
        h->err = badtype ? "a particle type is outside 0 .. ntypes-1" : "a position is outside [-L/2, L/2) or not finite";
        return badtype ? HB_EINVAL : HB_ENAN;
    }
    return HB_OK;
}

int hb_get_state_f64(hb_system *h, double *pos_xyz, double *vel_xyz, int32_t *image, int on_device)
{
    HB_NEED(h);
    if (!h->have_state) { h->err = "no state"; return HB_ESTATE; }
    if (!h->dp.have || h->tun.precision != 64) HB_TRY(dp_from_f32(h));     // binary32 mode: the binary32 state, widened
    const size_t N = (size_t)h->N;
    if (on_device) return dp_get(h, pos_xyz, vel_xyz, image, nullptr, nullptr, nullptr, nullptr);
    HB_TRY(ensure_stage(h, N * 60));
    char *base = (char *)h->acc_stage;
    double *dpos = (double *)base, *dvel = (double *)(base + N * 24);
    int32_t *dimg = (int32_t *)(base + N * 48);
    HB_TRY(dp_get(h, pos_xyz ? dpos : nullptr, vel_xyz ? dvel : nullptr, image ? dimg : nullptr, nullptr, nullptr, nullptr, nullptr));
    if (pos_xyz) HB_CK(cudaMemcpyAsync(pos_xyz, dpos, N * 24, cudaMemcpyDeviceToHost, h->stream));
    if (vel_xyz) HB_CK(cudaMemcpyAsync(vel_xyz, dvel, N * 24, cudaMemcpyDeviceToHost, h->stream));
    if (image) HB_CK(cudaMemcpyAsync(image, dimg, N * 12, cudaMemcpyDeviceToHost, h->stream));
    HB_CK(cudaStreamSynchronize(h->stream));
    return HB_OK;
}

int hb_get_forces_f64(hb_system *h, double *f_xyz_u, double *virial6, int on_device)
{
    HB_NEED(h);
    if (h->tun.precision != 64) { h->err = "hb_get_forces_f64 needs the binary64 variant (tunable precision = 64)"; return HB_ESTATE; }
    if (!h->dp.forces_valid) { h->err = "forces are stale: call hb_compute_lj first"; return HB_ESTATE; }
    const size_t N = (size_t)h->N;
    if (on_device) return dp_get(h, nullptr, nullptr, nullptr, f_xyz_u, virial6, nullptr, nullptr);
    HB_TRY(ensure_stage(h, N * 80));
    double *sf = (double *)h->acc_stage, *sv = (double *)((char *)h->acc_stage + N * 32);
    HB_TRY(dp_get(h, nullptr, nullptr, nullptr, f_xyz_u ? sf : nullptr, virial6 ? sv : nullptr, nullptr, nullptr));
    if (f_xyz_u) HB_CK(cudaMemcpyAsync(f_xyz_u, sf, N * 32, cudaMemcpyDeviceToHost, h->stream));
    if (virial6) HB_CK(cudaMemcpyAsync(virial6, sv, N * 48, cudaMemcpyDeviceToHost, h->stream));
    HB_CK(cudaStreamSynchronize(h->stream));
    return HB_OK;
}

int hb_get_state(hb_system *h, float *pos_xyz, int32_t *type, float *vel_xyz, int32_t *image, uint32_t *order, int on_device)
{
    HB_NEED(h);
    if (!h->have_state) { h->err = "no state"; return HB_ESTATE; }
    const size_t N = (size_t)h->N;
    const bool dp = h->tun.precision == 64 && h->dp.have;     // the image flags of this mode live with the binary64 arrays
    if (on_device) {
        HB_CK(launch_unpack_state(h, pos_xyz, type, vel_xyz, dp ? nullptr : image));
        if (dp && image) HB_TRY(dp_get(h, nullptr, nullptr, image, nullptr, nullptr, nullptr, nullptr));
        if (order) HB_CK(cudaMemcpyAsync(order, h->tag, N * 4, cudaMemcpyDeviceToDevice, h->stream));
        return HB_OK;
    }
    HB_TRY(ensure_stage(h, N * 40));
    char *base = (char *)h->acc_stage;
    float *spos = (float *)base;
    float *svel = (float *)(base + N * 12);
    int32_t *stype = (int32_t *)(base + N * 24);
    int32_t *simg = (int32_t *)(base + N * 28);
    HB_CK(launch_unpack_state(h, pos_xyz ? spos : nullptr, type ? stype : nullptr, vel_xyz ? svel : nullptr,
                              (image && !dp) ? simg : nullptr));
    if (dp && image) HB_TRY(dp_get(h, nullptr, nullptr, simg, nullptr, nullptr, nullptr, nullptr));
    if (pos_xyz) HB_CK(cudaMemcpyAsync(pos_xyz, spos, N * 12, cudaMemcpyDeviceToHost, h->stream));
    if (vel_xyz) HB_CK(cudaMemcpyAsync(vel_xyz, svel, N * 12, cudaMemcpyDeviceToHost, h->stream));
    if (type) HB_CK(cudaMemcpyAsync(type, stype, N * 4, cudaMemcpyDeviceToHost, h->stream));
    if (image) HB_CK(cudaMemcpyAsync(image, simg, N * 12, cudaMemcpyDeviceToHost, h->stream));
    if (order) HB_CK(cudaMemcpyAsync(order, h->tag, N * 4, cudaMemcpyDeviceToHost, h->stream));
    HB_CK(cudaStreamSynchronize(h->stream));
    return HB_OK;
}

int hb_set_rcut_pair(hb_system *h, const double *rcut)
{
    HB_NEED(h);
    if (!rcut) { h->err = "rcut is NULL"; return HB_EINVAL; }
    const int nt = h->ntypes;
    for (int a = 0; a < nt; a++)
        for (int b = 0; b < nt; b++)
            if (rcut[a * nt + b] != rcut[b * nt + a] || !(rcut[a * nt + b] > 0.0)) { h->err = "r_cut table must be symmetric and positive"; return HB_EINVAL; }
    for (int p = 0; p < nt * nt; p++) h->rcut[p] = (double)(float)rcut[p];
    h->rcut_user = true;
    h->geometry_dirty = true;     // r_cut,max and with it r_max, m and the per-pair list cutoffs may have changed
    h->nlist_valid = h->cells_valid = h->forces_valid = false;
    destroy_graphs(h);
    return upload_params(h);
}

int hb_set_ron_pair(hb_system *h, const double *ron)
{
    HB_NEED(h);
    if (!ron) { h->err = "ron is NULL"; return HB_EINVAL; }
    const int nt = h->ntypes;
    for (int a = 0; a < nt; a++)
        for (int b = 0; b < nt; b++)
            if (ron[a * nt + b] != ron[b * nt + a] || !(ron[a * nt + b] > 0.0)) { h->err = "r_on table must be symmetric and positive"; return HB_EINVAL; }
    for (int p = 0; p < nt * nt; p++) h->ron[p] = (double)(float)ron[p];
    h->forces_valid = false;
    return upload_params(h);
}

int hb_set_pair_potential(hb_system *h, int pot, const double *p2)
{
    HB_NEED(h);
    if (pot < HB_POT_LJ || pot > HB_POT_MORSE) { h->err = "unknown pair potential"; return HB_EINVAL; }
    const int nt = h->ntypes;
    if (p2)
        for (int a = 0; a < nt; a++)
            for (int b = 0; b < nt; b++)
                if (p2[a * nt + b] != p2[b * nt + a]) { h->err = "p2 table must be symmetric"; return HB_EINVAL; }
    for (int p = 0; p < nt * nt; p++) h->p2[p] = p2 ? (double)(float)p2[p] : 0.0;
    h->pot = pot;
    h->forces_valid = false;
    destroy_graphs(h);          // the captured step kernels are instantiated for one pair functor
    if (h->m > 0) HB_TRY(choose_tiles(h, 0));   // the functor decides the block size and with it the shared-memory budget
    return upload_params(h);
}

int hb_set_mass(hb_system *h, const float *mass, int on_device)
{
    HB_NEED(h);
    if (!mass) { h->err = "mass is NULL"; return HB_EINVAL; }
    if (!h->have_state) { h->err = "no state: call hb_set_state first (it resets the masses to 1)"; return HB_ESTATE; }
    const size_t N = (size_t)h->N;
    const float *d = mass;
    if (!on_device) {
        HB_TRY(ensure_stage(h, N * 4));
        HB_CK(cudaMemcpyAsync(h->acc_stage, mass, N * 4, cudaMemcpyHostToDevice, h->stream));
        d = (const float *)h->acc_stage;
    }
    HB_CK(launch_mass(h, d, nullptr));
    HB_TRY(read_flags(h));
    if (h->h_flags[FL_BADTYPE]) {
        HB_TRY(set_flag(h, FL_BADTYPE, 0));
        h->err = "masses must be positive and finite (some were not; the others have been set)";
        return HB_EINVAL;
    }
    h->bk_valid = false;
    return dp_sync_mass(h);
}

int hb_get_mass(hb_system *h, float *mass, int on_device)
{
    HB_NEED(h);
    if (!mass) { h->err = "mass is NULL"; return HB_EINVAL; }
    if (!h->have_state) { h->err = "no state"; return HB_ESTATE; }
    const size_t N = (size_t)h->N;
    if (on_device) { HB_CK(launch_mass(h, nullptr, mass)); return HB_OK; }
    HB_TRY(ensure_stage(h, N * 4));
    HB_CK(launch_mass(h, nullptr, (float *)h->acc_stage));
    HB_CK(cudaMemcpyAsync(mass, h->acc_stage, N * 4, cudaMemcpyDeviceToHost, h->stream));
    HB_CK(cudaStreamSynchronize(h->stream));
    return HB_OK;
}

int hb_build_cells(hb_system *h)
{
    HB_NEED(h);
    Range nvtx_range("hb_build_cells");
    if (!h->have_state) { h->err = "no state: call hb_set_state first"; return HB_ESTATE; }
    HB_TRY(configure_geometry(h));
    if (h->cells_valid && !h->moved) return HB_OK;   // the cell list of these very positions is in place
    HB_TRY(enqueue_cells(h, nullptr));
    HB_CK(launch_cell_copyback(h, nullptr));
    HB_TRY(read_flags(h));
    h->nlist_valid = h->forces_valid = false;        // the storage order changed
    if (h->h_flags[FL_BAD]) {
        h->err = "a particle is non-finite or outside the box";
        set_flag(h, FL_BAD, 0);
        h->cells_valid = false;
        return HB_ENAN;
    }
    h->cells_valid = true;
    h->moved = false;
    return HB_OK;
}

int hb_build_nlist(hb_system *h, double r_cut, double r_buff)
{
    HB_NEED(h);
    Range nvtx_range("hb_build_nlist");
    if (!h->have_state) { h->err = "no state: call hb_set_state first"; return HB_ESTATE; }
    if (!(r_buff >= 0.0)) { h->err = "r_buff must be >= 0"; return HB_EINVAL; }
    if (r_cut > 0.0 && !h->rcut_user) {
        for (auto &rc : h->rcut) rc = (double)(float)r_cut;
        HB_TRY(upload_params(h));
        h->forces_valid = false;
    }
    if ((float)r_buff != h->r_buff) destroy_graphs(h);
    h->r_buff = (float)r_buff;
    HB_TRY(configure_geometry(h));
    return build_nlist_sync(h);
}

int hb_needs_rebuild(hb_system *h, int *need)
{
    HB_NEED(h);
    if (!need) return HB_EINVAL;
    if (!h->nlist_valid) { *need = 1; return HB_OK; }
    HB_TRY(set_flag(h, FL_CHECK, 0));
    HB_CK(launch_disp_check(h));
    HB_TRY(read_flags(h));
    *need = h->h_flags[FL_CHECK] ? 1 : 0;
    return HB_OK;
}

int hb_compute_lj(hb_system *h, int shift_mode)
{
    HB_NEED(h);
    Range nvtx_range("hb_compute_lj");
    if (shift_mode != HB_SHIFT_NONE && shift_mode != HB_SHIFT_ENERGY && shift_mode != HB_XPLOR) { h->err = "unknown shift mode"; return HB_EINVAL; }
    if (!h->nlist_valid) { h->err = "no neighbor list: call hb_build_nlist first"; return HB_ESTATE; }
    if (shift_mode != h->shift_mode) {
        h->shift_mode = shift_mode;
        destroy_graphs(h);     // the captured step kernels are instantiated for one pair functor
        HB_TRY(upload_params(h));
    }
    if (h->tun.precision == 64) {
        if (!h->dp.have) HB_TRY(dp_from_f32(h));
        return dp_force(h);
    }
    HB_CK(launch_force(h, nullptr));
    h->forces_valid = true;
    return HB_OK;
}

int hb_step_nve(hb_system *h, double dt)
{
    HB_NEED(h);
    Range nvtx_range("hb_step_nve");
    if (!h->have_state) { h->err = "no state"; return HB_ESTATE; }
    if (h->m == 0) HB_TRY(configure_geometry(h));
    if (h->tun.precision == 64) return dp_run(h, (double)(float)dt, 1, 0);
    return step_sync(h, (float)dt);
}

static int run_md(hb_system *h, double dt, int64_t nsteps, int64_t sort_period, const Ensemble &ens)
{
    if (!h->have_state) { h->err = "no state"; return HB_ESTATE; }
    if (nsteps < 0 || sort_period < 0) return HB_EINVAL;
    if (h->m == 0) HB_TRY(configure_geometry(h));
    h->ens = ens;
    if (h->tun.precision == 64) {
        const int rcd = dp_run(h, (double)(float)dt, nsteps, sort_period);
        h->ens = Ensemble{};
        return rcd;
    }
    int64_t done = 0;
    int rc = HB_OK;
    while (done < nsteps && rc == HB_OK) {
        // sort before the first step ever run, then every sort_period steps (counted across calls)
        if (sort_period > 0 && (h->since_sort < 0 || h->since_sort >= sort_period)) {
            if ((rc = ensure_forces(h)) != HB_OK) break;
            if ((rc = sort_internal(h)) != HB_OK) break;
            h->since_sort = 0;
        }
        int64_t n = std::min<int64_t>(h->tun.graph_steps, nsteps - done);
        if (sort_period > 0) n = std::min<int64_t>(n, sort_period - h->since_sort);
        if (n < h->tun.graph_steps && !h->graphs.count(n) && h->graphs.size() >= 24 && h->tun.graph_mode != 0 && h->tun.graph_mode != 3) {
            // a remainder runs as ONE chunk with a graph of exactly its length, captured the first time that length is
            // met and kept; once two dozen lengths are cached, the largest power of two that fits (those exist)
            int64_t p2 = 1;
            while (2 * p2 <= n) p2 *= 2;
            n = p2;
        }
        rc = run_chunk(h, (float)dt, (int)n);
        done += n;
        if (h->since_sort >= 0) h->since_sort += n;
    }
    h->ens = Ensemble{};      // hb_step_nve and the accessors integrate NVE
    return rc;
}

int hb_run_nve(hb_system *h, double dt, int64_t nsteps, int64_t sort_period)
{
    HB_NEED(h);
    Range nvtx_range("hb_run_nve");
    return run_md(h, dt, nsteps, sort_period, Ensemble{});
}

int hb_run_nvt(hb_system *h, double dt, int64_t nsteps, int64_t sort_period, double T, double tau)
{
    HB_NEED(h);
    Range nvtx_range("hb_run_nvt");
    if (!(T > 0.0) || !(tau > 0.0)) { h->err = "hb_run_nvt: T and tau must be positive"; return HB_EINVAL; }
    Ensemble e;
    e.mode = 1; e.T = (double)(float)T; e.par = (double)(float)tau;
    return run_md(h, dt, nsteps, sort_period, e);
}

int hb_run_langevin(hb_system *h, double dt, int64_t nsteps, int64_t sort_period, double T, double gamma, uint64_t seed)
{
    HB_NEED(h);
    Range nvtx_range("hb_run_langevin");
    if (!(T >= 0.0) || !(gamma >= 0.0)) { h->err = "hb_run_langevin: T and gamma must not be negative"; return HB_EINVAL; }
    Ensemble e;
    e.mode = 2; e.T = (double)(float)T; e.par = (double)(float)gamma; e.seed = seed;
    return run_md(h, dt, nsteps, sort_period, e);
}

int hb_get_thermostat(hb_system *h, double *xi, double *eta, int64_t *langevin_steps)
{
    HB_NEED(h);
    HB_CK(cudaMemcpyAsync(h->h_tstate, h->tstate, sizeof(double) * TS_COUNT, cudaMemcpyDeviceToHost, h->stream));
    HB_CK(cudaStreamSynchronize(h->stream));
    if (xi) *xi = h->h_tstate[TS_XI];
    if (eta) *eta = h->h_tstate[TS_ETA];
    if (langevin_steps) *langevin_steps = h->lang_steps;
    return HB_OK;
}

int hb_set_thermostat(hb_system *h, double xi, double eta, int64_t langevin_steps)
{
    HB_NEED(h);
    if (langevin_steps < 0) return HB_EINVAL;
    memset(h->h_tstate, 0, sizeof(double) * TS_COUNT);
    h->h_tstate[TS_XI] = xi;
    h->h_tstate[TS_ETA] = eta;
    HB_CK(cudaMemcpyAsync(h->tstate, h->h_tstate, sizeof(double) * TS_COUNT, cudaMemcpyHostToDevice, h->stream));
    HB_CK(cudaStreamSynchronize(h->stream));
    h->lang_steps = langevin_steps;
    return HB_OK;
}

int hb_sort(hb_system *h)
{
    HB_NEED(h);
    Range nvtx_range("hb_sort");
    return sort_internal(h);
}

int hb_thermo(hb_system *h, hb_thermo_t *out)
{
    HB_NEED(h);
    Range nvtx_range("hb_thermo");
    if (!out) return HB_EINVAL;
    if (!h->have_state) { h->err = "no state"; return HB_ESTATE; }
    if (h->tun.precision == 64) {
        if (h->m == 0) HB_TRY(configure_geometry(h));
        if (!h->dp.have) HB_TRY(dp_from_f32(h));
        if (!h->nlist_valid) { HB_TRY(build_nlist_sync(h)); h->dp.forces_valid = false; }
        if (!h->dp.forces_valid) HB_TRY(dp_force(h));
        double t[11];
        HB_TRY(dp_thermo(h, t));
        out->K = t[0];
        out->U = t[1];
        for (int a = 0; a < 6; a++) out->W[a] = t[2 + a];
        out->px = t[8]; out->py = t[9]; out->pz = t[10];
        const double V = (double)h->L * (double)h->L * (double)h->L;
        out->P = (2.0 * out->K + out->W[0] + out->W[3] + out->W[5]) / (3.0 * V);
        return HB_OK;
    }
    if (!h->forces_valid) {       // U, W and P come from the per-particle arrays of the last force evaluation
        if (h->m == 0) HB_TRY(configure_geometry(h));
        HB_TRY(ensure_forces(h));
    }
    HB_CK(launch_thermo(h));
    HB_CK(cudaMemcpyAsync(h->h_thermo, h->thermo_part + (int64_t)h->thermo_blocks * 11, sizeof(double) * 11,
                          cudaMemcpyDeviceToHost, h->stream));
    HB_CK(cudaStreamSynchronize(h->stream));
    const double *t = h->h_thermo;
    out->K = t[0];
    out->U = t[1];
    for (int a = 0; a < 6; a++) out->W[a] = t[2 + a];
    out->px = t[8]; out->py = t[9]; out->pz = t[10];
    const double V = (double)h->L * (double)h->L * (double)h->L;
    out->P = (2.0 * out->K + out->W[0] + out->W[3] + out->W[5]) / (3.0 * V);
    return HB_OK;
}

int hb_get_cells(hb_system *h, int32_t *m_out, int32_t *cell_start, uint32_t *cell_tags, int on_device)
{
    HB_NEED(h);
    if (!h->cells_valid) { h->err = "no cell list: call hb_build_cells first"; return HB_ESTATE; }
    if (m_out) {
        int32_t mm[3] = {h->m, h->m, h->m};
        if (on_device) HB_CK(cudaMemcpyAsync(m_out, mm, sizeof mm, cudaMemcpyHostToDevice, h->stream));
        else memcpy(m_out, mm, sizeof mm);
    }
    const cudaMemcpyKind kind = on_device ? cudaMemcpyDeviceToDevice : cudaMemcpyDeviceToHost;
    if (cell_start) HB_CK(cudaMemcpyAsync(cell_start, h->cell_start, sizeof(int) * (size_t)(h->ncells + 1), kind, h->stream));
    // the particle data is kept in cell order: the members of cell c are the storage slots of its CSR range
    if (cell_tags) HB_CK(cudaMemcpyAsync(cell_tags, h->tag, (size_t)h->N * 4, kind, h->stream));
    HB_CK(cudaStreamSynchronize(h->stream));
    return HB_OK;
}

int hb_get_nlist(hb_system *h, int64_t *row_start, uint32_t *nbr_tags, int on_device)
{
    HB_NEED(h);
    if (!h->nlist_valid) { h->err = "no neighbor list: call hb_build_nlist first"; return HB_ESTATE; }
    if (!row_start) { h->err = "row_start is NULL"; return HB_EINVAL; }
    const size_t N = (size_t)h->N;
    // row lengths by tag -> exclusive scan on the device (scratch owned by the handle: no allocation per call)
    HB_CK(launch_nlist_counts_by_tag(h, h->acc_counts));
    HB_CK(launch_nlist_rows_by_tag(h, h->acc_counts, h->acc_rows));
    if (on_device) {
        HB_CK(cudaMemcpyAsync(row_start, h->acc_rows, (N + 1) * 8, cudaMemcpyDeviceToDevice, h->stream));
        if (nbr_tags) HB_CK(launch_nlist_fill_by_tag(h, h->acc_rows, nbr_tags));
        return HB_OK;
    }
    HB_CK(cudaMemcpyAsync(row_start, h->acc_rows, (N + 1) * 8, cudaMemcpyDeviceToHost, h->stream));
    HB_CK(cudaStreamSynchronize(h->stream));
    if (nbr_tags) {
        const size_t total = (size_t)row_start[N];
        HB_TRY(ensure_stage(h, (total + 1) * 4));
        HB_CK(launch_nlist_fill_by_tag(h, h->acc_rows, (uint32_t *)h->acc_stage));
        HB_CK(cudaMemcpyAsync(nbr_tags, h->acc_stage, total * 4, cudaMemcpyDeviceToHost, h->stream));
        HB_CK(cudaStreamSynchronize(h->stream));
    }
    return HB_OK;
}

int hb_get_forces(hb_system *h, float *f_xyz_u, float *virial6, int on_device)
{
    HB_NEED(h);
    const size_t N = (size_t)h->N;
    if (h->tun.precision == 64) {      // the binary64 sums, rounded
        if (!h->dp.forces_valid) { h->err = "forces are stale: call hb_compute_lj first"; return HB_ESTATE; }
        if (on_device) return dp_get(h, nullptr, nullptr, nullptr, nullptr, nullptr, f_xyz_u, virial6);
        HB_TRY(ensure_stage(h, N * 40));
        float *sf = (float *)h->acc_stage, *sv = (float *)((char *)h->acc_stage + N * 16);
        HB_TRY(dp_get(h, nullptr, nullptr, nullptr, nullptr, nullptr, f_xyz_u ? sf : nullptr, virial6 ? sv : nullptr));
        if (f_xyz_u) HB_CK(cudaMemcpyAsync(f_xyz_u, sf, N * 16, cudaMemcpyDeviceToHost, h->stream));
        if (virial6) HB_CK(cudaMemcpyAsync(virial6, sv, N * 24, cudaMemcpyDeviceToHost, h->stream));
        HB_CK(cudaStreamSynchronize(h->stream));
        return HB_OK;
    }
    if (!h->forces_valid) { h->err = "forces are stale: call hb_compute_lj first"; return HB_ESTATE; }
    if (on_device) {
        HB_CK(launch_unpack_forces(h, f_xyz_u, virial6));
        return HB_OK;
    }
    HB_TRY(ensure_stage(h, N * 40));
    float *sf = (float *)h->acc_stage;
    float *sv = (float *)((char *)h->acc_stage + N * 16);
    HB_CK(launch_unpack_forces(h, f_xyz_u ? sf : nullptr, virial6 ? sv : nullptr));
    if (f_xyz_u) HB_CK(cudaMemcpyAsync(f_xyz_u, sf, N * 16, cudaMemcpyDeviceToHost, h->stream));
    if (virial6) HB_CK(cudaMemcpyAsync(virial6, sv, N * 24, cudaMemcpyDeviceToHost, h->stream));
    HB_CK(cudaStreamSynchronize(h->stream));
    return HB_OK;
}

int hb_stats(hb_system *h, hb_stats_t *out)
{
    HB_NEED(h);
    if (!out) return HB_EINVAL;
    HB_TRY(read_flags(h));
    h->stats.rebuilds = h->h_flags[FL_BUILDS];
    *out = h->stats;
    return HB_OK;
}

int hb_time_stage(hb_system *h, const char *stage, int reps, int64_t flush_l2_bytes, double *mean_ms)
{
    HB_NEED(h);
    if (!stage || reps <= 0 || reps > 100000 || !mean_ms || flush_l2_bytes < 0) return HB_EINVAL;
    if (!h->nlist_valid) { h->err = "no neighbor list: call hb_build_nlist first"; return HB_ESTATE; }
    int which = -1;
    const char *names[] = {"lj_force", "nlist", "cells", "rebuild", "nve", "lj_nve", "cells_coop"};
    for (int k = 0; k < 7; k++) if (!strcmp(stage, names[k])) which = k;
    if (which < 0) { h->err = std::string("unknown stage ") + stage; return HB_EINVAL; }
    void *scratch = nullptr;
    if (flush_l2_bytes > 0) HB_TRY(dev_alloc(h, &scratch, (size_t)flush_l2_bytes));
    const int nev = flush_l2_bytes > 0 ? reps : 1;
    std::vector<cudaEvent_t> ev0(nev), ev1(nev);
    for (int k = 0; k < nev; k++) { cudaEventCreate(&ev0[k]); cudaEventCreate(&ev1[k]); }
    int rc = HB_OK;
    auto launch = [&]() -> int {
        switch (which) {
            case 0: HB_CK(launch_force(h, nullptr)); break;
            case 1: HB_CK(launch_nlist(h, nullptr, false)); break;
            case 2: HB_TRY(enqueue_cells(h, nullptr)); break;
            case 3: HB_TRY(enqueue_rebuild(h, nullptr)); break;
            case 4: HB_CK(launch_nve(h, make_nve(h, 0.0f, true, true, h->pos(), 0, false))); break;
            case 6: HB_CK(launch_rebuild_coop(h, nullptr, false)); break;
            default: {
                const NveArgs a = make_nve(h, 0.0f, true, true, h->posbuf[h->cur ^ 1], 0, false);
                HB_CK(launch_force(h, &a));
                break;
            }
        }
        return HB_OK;
    };
    cudaGraph_t tg = nullptr;
    cudaGraphExec_t tge = nullptr;
    if (flush_l2_bytes) {
        for (int r = 0; r < reps && rc == HB_OK; r++) {
            cudaMemsetAsync(scratch, r & 0xff, (size_t)flush_l2_bytes, h->stream);
            cudaEventRecord(ev0[r], h->stream);
            rc = launch();
            cudaEventRecord(ev1[r], h->stream);
        }
    } else {
        // The reps launches go into ONE graph, so that the device runs them back to back: launched one by
        // one from the host, a kernel shorter than the host's launch cost would be timed at the host's pace.
        cudaStream_t cs = nullptr, saved = h->stream;
        const int64_t saved_launches = h->stats.kernel_launches;
        if (cudaStreamCreateWithFlags(&cs, cudaStreamNonBlocking) != cudaSuccess ||
            cudaStreamBeginCapture(cs, cudaStreamCaptureModeRelaxed) != cudaSuccess) {
            h->err = "hb_time_stage: cannot start a capture";
            rc = HB_ECUDA;
        } else {
            h->stream = cs;
            for (int r = 0; r < reps && rc == HB_OK; r++) rc = launch();
            h->stream = saved;
            cudaError_t ce = cudaStreamEndCapture(cs, &tg);
            if (rc == HB_OK && ce == cudaSuccess) ce = cudaGraphInstantiate(&tge, tg, 0);
            if (rc == HB_OK && ce != cudaSuccess) { h->err = std::string("hb_time_stage: ") + cudaGetErrorString(ce); rc = HB_ECUDA; }
        }
        h->stats.kernel_launches = saved_launches + (rc == HB_OK ? 2 * (h->stats.kernel_launches - saved_launches) : 0);
        if (cs) cudaStreamDestroy(cs);
        if (rc == HB_OK) {
            cudaGraphLaunch(tge, h->stream);   // warm-up
            cudaEventRecord(ev0[0], h->stream);
            cudaGraphLaunch(tge, h->stream);
            cudaEventRecord(ev1[0], h->stream);
        }
    }
    cudaError_t e = cudaStreamSynchronize(h->stream);
    double total = 0.0;
    if (rc == HB_OK && e == cudaSuccess) {
        for (int k = 0; k < nev; k++) { float ms = 0.f; cudaEventElapsedTime(&ms, ev0[k], ev1[k]); total += ms; }
        *mean_ms = total / reps;
    } else if (rc == HB_OK) {
        h->err = std::string("hb_time_stage: ") + cudaGetErrorString(e);
        rc = HB_ECUDA;
    }
    for (int k = 0; k < nev; k++) { cudaEventDestroy(ev0[k]); cudaEventDestroy(ev1[k]); }
    if (tge) cudaGraphExecDestroy(tge);
    if (tg) cudaGraphDestroy(tg);
    dev_free(h, scratch);
    if (rc == HB_OK) rc = clear_need_flags(h);
    if (rc == HB_OK && (which == 2 || which == 3 || which == 6 || (which == 5 && h->tun.thermo_every == 0))) {
        // the timed cell builds re-ordered the scratch set (and, for "rebuild", the particles): make the list whole again
        h->nlist_valid = false;
        rc = ensure_forces(h);
    }
    return rc;
}

int hb_measure_peak(hb_system *h, const char *which, double *value)
{
    HB_NEED(h);
    if (!which || !value) return HB_EINVAL;
    Range nvtx_range("hb_measure_peak");
    return measure_peak(h, which, value);
}

static int *tunable_slot(hb_system *h, const char *name)
{
    if (!name) return nullptr;
    if (!strcmp(name, "tpp")) return &h->tun.tpp;
    if (!strcmp(name, "epl")) return &h->tun.epl;
    if (!strcmp(name, "force_block")) return &h->tun.force_block;
    if (!strcmp(name, "nlist_ppi")) return &h->tun.nlist_ppi;
    if (!strcmp(name, "nlist_block")) return &h->tun.nlist_block;
    if (!strcmp(name, "nlist_pair_rcut")) return &h->tun.nlist_pair_rcut;
    if (!strcmp(name, "precision")) return &h->tun.precision;
    if (!strcmp(name, "tile_x")) return &h->tun.tile_x;
    if (!strcmp(name, "tile_y")) return &h->tun.tile_y;
    if (!strcmp(name, "tile_z")) return &h->tun.tile_z;
    if (!strcmp(name, "stage_cap")) return &h->tun.stage_cap;
    if (!strcmp(name, "row_pitch")) return &h->tun.row_pitch;
    if (!strcmp(name, "cell_sort")) return &h->tun.cell_sort;
    if (!strcmp(name, "fuse_nve")) return &h->tun.fuse_nve;
    if (!strcmp(name, "thermo_every")) return &h->tun.thermo_every;
    if (!strcmp(name, "grow_pct")) return &h->tun.grow_pct;
    if (!strcmp(name, "coop_rebuild")) return &h->tun.coop_rebuild;
    if (!strcmp(name, "coop_blocks")) return &h->tun.coop_blocks;
    if (!strcmp(name, "graph_mode")) return &h->tun.graph_mode;
    if (!strcmp(name, "graph_steps")) return &h->tun.graph_steps;
    return nullptr;
}

int hb_set_tunable(hb_system *h, const char *name, int value)
{
    HB_NEED(h);
    int *slot = tunable_slot(h, name);
    if (!slot) { h->err = std::string("unknown tunable ") + (name ? name : "(null)"); return HB_EINVAL; }
    bool ok = true;
    if (slot == &h->tun.tpp) ok = value == 2 || value == 4 || value == 8;
    else if (slot == &h->tun.epl) ok = value == 4 || value == 8;
    else if (slot == &h->tun.force_block) ok = value == 0 || value == 128 || value == 256;
    else if (slot == &h->tun.nlist_block) ok = value == 128 || value == 256;
    else if (slot == &h->tun.nlist_ppi) ok = value == 1 || value == 2 || value == 4;
    else if (slot == &h->tun.tile_x || slot == &h->tun.tile_y || slot == &h->tun.tile_z) ok = value >= 0 && value <= 16;
    else if (slot == &h->tun.stage_cap) ok = value >= 0 && value <= 65535;
    else if (slot == &h->tun.row_pitch) ok = value >= 0 && value <= 4096;
    else if (slot == &h->tun.cell_sort || slot == &h->tun.fuse_nve || slot == &h->tun.thermo_every || slot == &h->tun.nlist_pair_rcut) ok = value == 0 || value == 1;
    else if (slot == &h->tun.coop_rebuild) ok = value >= -1 && value <= 2;
    else if (slot == &h->tun.coop_blocks) ok = value >= 1 && value <= 8;
    else if (slot == &h->tun.grow_pct) ok = value >= 0 && value <= 400;
    else if (slot == &h->tun.graph_mode) ok = value >= 0 && value <= 3;
    else if (slot == &h->tun.graph_steps) ok = value >= 1 && value <= 2000;
    else if (slot == &h->tun.precision) ok = value == 32 || value == 64;
    if (!ok) { h->err = std::string("value out of range for tunable ") + name; return HB_EINVAL; }
    *slot = value;
    destroy_graphs(h);
    if (slot == &h->tun.row_pitch && value > 0) HB_TRY(ensure_rows(h, value));
    if (slot == &h->tun.nlist_pair_rcut) h->nlist_valid = false;
    if (slot == &h->tun.precision) {
        h->dp.have = h->dp.forces_valid = false;
        h->forces_valid = false;
        if (value == 64 && h->have_state) HB_TRY(dp_from_f32(h));
    }
    if (slot == &h->tun.tile_x || slot == &h->tun.tile_y || slot == &h->tun.tile_z || slot == &h->tun.stage_cap) {
        h->nlist_valid = false;
        if (h->m > 0) HB_TRY(choose_tiles(h, 0));
    }
    return HB_OK;
}

int hb_get_tunable(hb_system *h, const char *name, int *value)
{
    HB_NEED(h);
    int *slot = tunable_slot(h, name);
    if (!slot || !value) return HB_EINVAL;
    *value = *slot;
    return HB_OK;
}

}  // extern "C"
