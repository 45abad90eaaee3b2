// Internal declarations of libhb (sm_100a).  Not part of the ABI.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <string>
#include <vector>
#include <map>
#include <algorithm>
#include <string.h>

#include "../../include/hb.h"

// Device-side flag words (one int array, mirrored in pinned host memory).
enum {
    FL_NEED0 = 0,       // rebuild decision of the drifts with even / odd drift number: the drift kernel of
    FL_NEED1 = 1,       //   drift d sets FL_NEED0 + (d & 1) and clears the other one for drift d + 1
    FL_MAX_NBRS = 2,    // atomicMax of row lengths NEEDED by the last build (may exceed row_pitch => overflow)
    FL_BAD = 3,         // non-finite / out-of-box particle seen while binning
    FL_BUILDS = 4,      // number of list builds done on the device
    FL_DONE_CTR = 5,    // "last block done" counter of the drift kernels
    FL_OVERFLOWED = 6,  // sticky: some build since the last host check overflowed its rows (value = rows needed)
    FL_STAGE_OVER = 7,  // sticky: some tile needed more shared-memory slots than stage_cap (value = slots needed)
    FL_SCAN_CTR = 8,    // "last block done" counter of the cell scan
    FL_CHECK = 9,       // result of the on-demand displacement check (hb_needs_rebuild)
    FL_BAR0 = 10,       // arrival counters of the cooperative rebuild kernel's grid barrier; build b uses
    FL_BAR1 = 11,       //   FL_BAR0 + (b & 1) and clears the other one
    FL_BAR_GEN = 12,    // b: launches of the cooperative kernel that got past their barriers
    FL_TILE_CTR = 13,   // next tile of the cooperative kernel's list phase
    FL_BADTYPE = 14,    // hb_set_state saw a type outside 0 .. ntypes-1
    FL_COUNT = 16
};

struct PairParam {  // one per type pair, 16 B
    float lj1;      // LJ: 4 eps sigma^12 | Gauss: eps            | Yukawa: eps   | Morse: D0
    float lj2;      // LJ: 4 eps sigma^6  | Gauss: 1/(2 sigma^2)  | Yukawa: kappa | Morse: a
    float rcut2;    // r_cut^2
    float eshift;   // V(r_cut) if energy shift, else 0
};

struct PairParamX {  // XPLOR smoothing and the third parameter, one per type pair, 16 B
    float ron2;     // r_on^2
    float invD;     // 1 / (r_cut^2 - r_on^2)^3, 0 where r_on >= r_cut (no switching interval)
    float p2;       // Morse: r0
    float pad;
};

// A tile is a brick of tx x ty x tz cells (clipped at the upper faces of the box).  One
// thread block owns one tile: it stages the positions of the tile's cells and of the
// one-cell halo around them in shared memory, already shifted to the periodic image
// the tile sees, and both the list build and the force evaluation work on that copy.
struct TileGeom {
    int m;              // cells per axis
    int tx, ty, tz;     // tile dimensions in cells
    int ntx, nty, ntz;  // tiles per axis
    int ntiles;
    int cap;            // shared-memory slots (slot 0 is the far-away dummy)
    int fast;           // 1: tile + halo narrower than L/2 on every axis (image by tile centre, halo rows staged as contiguous pieces)
    int eshift;         // list entries are slot << eshift: 4 (the byte offset of the staged position) when cap <= 4096, else 0
    float L;
};

constexpr int TILE_THREADS = 256;
constexpr int TILE_HMAX = 256;        // halo cells per tile, at most
constexpr int TILE_ROWS_MAX = 32;     // own (y, z) rows per tile, at most
constexpr int TILE_PROWS_MAX = 86;    // halo (y, z) rows per tile, at most: TILE_HMAX / 3
constexpr int ROW_PAD = 32;           // list rows are padded with dummy entries to a multiple of this

struct Tunables {
    int tpp = 2;           // threads per particle in the force kernel
    int epl = 8;           // list entries per thread per iteration (4 or 8)
    int force_block = 0;   // threads per block of the force kernel (128 or 256; 0 = one pass over the tile's particles if possible)
    int nlist_ppi = 4;     // particles tested per candidate load
    int nlist_block = 256; // threads per block of the stand-alone list kernel (128 or 256)
    int nlist_pair_rcut = 0;   // 1: the list keeps pair (i, j) iff d < r_cut(type i, type j) + r_buff (reading t1); 0: one r_max (reading c2.iii)
    int tile_x = 0, tile_y = 0, tile_z = 0;   // 0 = chosen from m and the SM count
    int stage_cap = 0;     // 0 = estimated from the density
    int row_pitch = 0;
    int grow_pct = 25;     // head room given when rows or the staging area are grown after an overflow
    int cell_sort = 1;
    int coop_blocks = 4;   // blocks per SM of the cooperative cell kernel (at most)
    int thermo_every = 0;  // 0: U_i and W_i only in the last step of every chunk of hb_run_nve (nothing can read those of an
                           //    inner step); 1: in every step (the paper's kernel computes them always)
    int fuse_nve = 1;      // hb_run_nve: integrate inside the force kernel
    int coop_rebuild = -1; // -1: 2 below 200,000 particles, else 1 (measured on B200); 1: Algorithm 2 + reorder as ONE cooperative kernel, then the list kernel; 2: the list too; 0: five launches
    int graph_mode = 1;    // measured on B200: five early-exit kernels per step cost less than one conditional node
    int graph_steps = 100;
    int precision = 32;    // 64: the binary64 variant of the force sums and the integration (dp.cu)
};

enum { TS_XI = 0, TS_ETA = 1, TS_KSUM = 2, TS_LBASE = 3, TS_COUNT = 8 };

struct Ensemble {
    int mode = 0;               // 0 NVE, 1 Nose-Hoover, 2 Langevin
    double T = 0, par = 0;
    unsigned long long seed = 0;
    bool operator==(const Ensemble &o) const { return mode == o.mode && T == o.T && par == o.par && seed == o.seed; }
};

struct hb_system {
    int64_t N = 0;
    int ntypes = 1;
    float L = 0, r_cut_max = 0, r_buff = 0, r_max = 0;
    bool geometry_dirty = false;  // a cutoff changed since configure_geometry last ran: r_max, m, the tiles and the typed-list
                                  // table are out of date; build_nlist_sync reconfigures before it builds
    int shift_mode = HB_SHIFT_ENERGY;
    int pot = HB_POT_LJ;     // pair potential (hb_set_pair_potential)
    bool rcut_user = false;  // hb_set_rcut_pair was called
    std::vector<double> eps, sigma, rcut, ron, p2;
    std::vector<PairParam> h_params;
    std::vector<PairParamX> h_paramsx;
    cudaStream_t stream = nullptr;
    hb_allocator alloc{};
    bool has_alloc = false;
    Tunables tun;
    std::string err;

    // particle data (storage order), SoA of 16 B vectors
    float4 *posbuf[2] = {nullptr, nullptr};  // x, y, z, type bits; posbuf[cur] is current (the fused step ping-pongs)
    int cur = 0;
    float4 *vel = nullptr;      // vx, vy, vz, mass (1 unless hb_set_mass)
    float4 *force = nullptr;    // Fx, Fy, Fz, U_i
    float4 *virial = nullptr;   // [2N]: (xx, xy, xz, yy), (yz, zz, 0, 0)
    int *image = nullptr;       // [3][N]
    uint32_t *tag = nullptr;    // storage slot -> tag
    uint32_t *rtag = nullptr;   // tag -> storage slot
    float4 *pos_build = nullptr;  // positions at the last list build, in the storage order that build made
    // scratch set: target of the reorder at every build and of hb_sort's gather
    float4 *vel2 = nullptr, *force2 = nullptr, *virial2 = nullptr;
    int *image2 = nullptr;
    uint32_t *tag2 = nullptr;
    // backup for hb_run_nve's chunk redo
    float4 *bk_pos = nullptr, *bk_vel = nullptr, *bk_force = nullptr, *bk_virial = nullptr;
    int *bk_image = nullptr;
    uint32_t *bk_tag = nullptr;
    int bk_cur = 0, bk_parity = 0;
    PairParam *params = nullptr;
    PairParamX *paramsx = nullptr;
    float *rmax2_pair = nullptr;   // [ntypes^2] (r_cut,ab + r_buff)^2 for the typed list build

    float4 *pos() const { return posbuf[cur]; }

    // cell list (CSR); after a build particle k of the storage order lies in the cell whose range holds k
    int m = 0;
    int64_t ncells = 0, ncells_alloc = 0;
    int *cell_count = nullptr;   // [ncells] zero between builds
    int *cell_local = nullptr;   // [ncells] exclusive scan inside a scan tile
    int *cell_start = nullptr;   // [ncells + 1]
    int *cell_id = nullptr;      // [N] cell of particle i (old order)
    int *cell_rank = nullptr;    // [N] slot inside the cell handed out by the atomic
    int *perm = nullptr;         // [N] new slot -> old slot
    int *scan_sums = nullptr;    // block sums / block offsets of the cell scan
    int64_t scan_sums_len = 0;

    // neighbor list: row i = nlist[i * row_pitch .. + nlistn[i]), entries are shared-memory slots of i's tile
    TileGeom geom{};
    double own_est = 0;          // expected own particles per tile
    int row_pitch = 0;
    uint16_t *nlist = nullptr;
    int *nlistn = nullptr;
    int64_t nlist_alloc = 0;

    // sort scratch
    uint32_t *keys = nullptr, *keys2 = nullptr, *sperm = nullptr, *sperm2 = nullptr;
    int *radix_counts = nullptr;
    int64_t radix_counts_len = 0;
    int *scan_tmp = nullptr;
    int64_t scan_tmp_len = 0;

    // flags + reductions
    int *flags = nullptr;        // device [FL_COUNT]
    int *h_flags = nullptr;      // pinned host mirror
    double *thermo_part = nullptr;  // [blocks][12]
    double *h_thermo = nullptr;     // pinned [12]
    int thermo_blocks = 0;
    int sm_count = 148;
    int smem_max = 227 * 1024;

    // host-side state machine
    bool have_state = false, cells_valid = false, nlist_valid = false, forces_valid = false, bk_valid = false;
    bool moved = true;           // positions changed since the last cell build
    int parity = 0;              // number of drifts done so far, mod 2
    int parity0 = 0;             // its value at the start of the running chunk (0 for graph chunks)
    Ensemble ens, graph_ens;     // the integration method of the running call, and the one the cached graphs were captured for
    double *tstate = nullptr, *bk_tstate = nullptr;   // device [TS_COUNT]: thermostat state (NveArgs::tstate), and its chunk backup
    double *h_tstate = nullptr;  // pinned [TS_COUNT]
    int64_t lang_steps = 0;      // Langevin steps taken since hb_set_state (the stream of the generator)
    hb_stats_t stats{};
    int64_t since_sort = -1;     // steps since the last hb_sort inside hb_run_nve (-1 = never sorted)

    // graph cache: key = nsteps -> exec (every chunk starts from posbuf[0] and drift parity 0, see run_chunk)
    struct GraphEntry { cudaGraph_t g = nullptr; cudaGraphExec_t e = nullptr; int nkernels_fixed = 0; };
    std::map<int64_t, GraphEntry> graphs;
    float graph_dt = 0;

    // binary64 variant (tunable precision = 64): arrays BY TAG
    struct Dp {
        void *x = nullptr, *v = nullptr, *f = nullptr, *pairs = nullptr;   // double4 [N]: (x, y, z, -), (vx, vy, vz, m), (Fx, Fy, Fz, U_i); pair table
        double *vir = nullptr, *out = nullptr;                             // [N][6]; reduction result
        int *img = nullptr;                                                // [3][N]
        bool have = false, forces_valid = false;
    } dp;

    // accessor scratch (host <-> device staging of hb_set_state / hb_get_state / hb_get_forces / hb_get_nlist)
    void *acc_stage = nullptr;
    size_t acc_cap = 0;
    int *acc_counts = nullptr;       // [N] list row lengths by tag
    int64_t *acc_rows = nullptr;     // [N + 1] CSR row starts by tag
    int *h_total = nullptr;          // pinned [2]
};

#define HB_CK(call)                                                                          \
    do {                                                                                     \
        cudaError_t e_ = (call);                                                             \
        if (e_ != cudaSuccess) {                                                             \
            h->err = std::string(#call) + ": " + cudaGetErrorString(e_);                     \
            return HB_ECUDA;                                                                 \
        }                                                                                    \
    } while (0)

#define HB_TRY(expr)              \
    do {                          \
        int rc_ = (expr);         \
        if (rc_ != HB_OK) return rc_; \
    } while (0)

static inline int64_t cdiv(int64_t a, int64_t b) { return (a + b - 1) / b; }

// cudaFuncAttributeMaxDynamicSharedMemorySize is state of the FUNCTION, shared by every handle and host thread of the
// process: it is always set to the same value (all the opt-in shared memory but 8 KB for the kernels' static tables,
// which is also what stage_cap_max budgets with), so that concurrent handles cannot lower it under each other.
static inline int smem_attr(const hb_system *h) { return h->smem_max - 8192; }

// threads per particle of the step kernel actually launched (the smoothed functor exists in the default layout only)
static inline int force_tpp(const hb_system *h) { return (h->shift_mode == HB_XPLOR || h->pot != HB_POT_LJ) ? 2 : h->tun.tpp; }

static inline int force_block_of(const hb_system *h)
{
    if (h->tun.force_block > 0) return h->tun.force_block;
    return h->own_est * force_tpp(h) > 160.0 ? 256 : 128;
}

// What the drift part of a step kernel needs (nve_kernel and the fused force kernel).
struct NveArgs {
    float4 *vel;
    int *image;
    const float4 *pos_build;
    float4 *pos_out;       // where the drifted positions go (== pos_in for the stand-alone kernel)
    float dt, half_buff2;
    int kick_prev, kick_drift;
    int forces_only;       // fused step whose U_i, W_i nobody can read: skip them
    int need_set, need_clear;   // flag indices
    cudaGraphConditionalHandle cond;
    int use_cond;
    // thermostats (readings n1, n2).  ens: 0 NVE, 1 Nose-Hoover, 2 Langevin
    int ens;
    float T, par;               // set temperature; tau (Nose-Hoover) or gamma (Langevin)
    double gdof;                // 3N - 3
    unsigned long long seed;    // Langevin
    int kick_step;              // number, inside the chunk, of the time step whose second half kick this launch makes
    double *tstate;             // device: [0] xi, [1] eta, [2] sum of v'^2 / 2 of the running drift, [3] (as int64) Langevin steps done before the chunk
    const uint32_t *tag;        // Langevin: the generator is indexed by the particle's identity
};


// ---- kernel launchers (each enqueues on h->stream and returns cudaGetLastError) ----
// cells.cu: Algorithm 2 + reorder of the particle data into cell order
cudaError_t launch_cell_count(hb_system *h, const int *pred);
cudaError_t launch_cell_scan(hb_system *h, const int *pred);
cudaError_t launch_cell_scatter(hb_system *h, const int *pred);
cudaError_t launch_cell_gather(hb_system *h, const int *pred);
cudaError_t launch_cell_copyback(hb_system *h, const int *pred);   // when no list kernel follows
cudaError_t launch_scan_exclusive(hb_system *h, const int *in, int *out, int64_t n, int *tmp);
// nlist.cu
cudaError_t launch_nlist(hb_system *h, const int *pred, bool copyback);
cudaError_t launch_rebuild_coop(hb_system *h, const int *pred, bool with_list);   // cells + reorder (+ list) in one cooperative launch
size_t nlist_smem_bytes(const hb_system *h);
// force.cu
cudaError_t launch_force(hb_system *h, const NveArgs *nve /* nullable: forces only */);
size_t force_smem_bytes(const hb_system *h);
// nve.cu
cudaError_t launch_nve(hb_system *h, const NveArgs &a);
cudaError_t launch_disp_check(hb_system *h);
cudaError_t launch_thermo(hb_system *h);
cudaError_t launch_state_copy(hb_system *h, bool restore);   // chunk backup of hb_run_nve (restore: the way back)
// sort.cu
cudaError_t launch_sfc_keys(hb_system *h);
cudaError_t launch_radix_sort(hb_system *h, int key_bits);  // keys/sperm -> sorted in keys/sperm
cudaError_t launch_gather_state(hb_system *h);              // by sperm into the scratch set (positions into pos_build)
cudaError_t launch_rtag(hb_system *h);
// dp.cu: the binary64 variant
int dp_ensure(hb_system *h);
void dp_release(hb_system *h);
int dp_from_f32(hb_system *h);
int dp_sync_mass(hb_system *h);
int dp_force(hb_system *h);
int dp_nve(hb_system *h, double dt, int what /* 1: half kick + drift, 2: half kick */);
int dp_set_state(hb_system *h, const double *pos, const double *vel, const int32_t *image, float *pos_f, float *vel_f);
int dp_get(hb_system *h, double *pos, double *vel, int32_t *image, double *f4, double *vir6, float *f4_f, float *vir6_f);
int dp_thermo(hb_system *h, double *out11);
// peaks.cu
int measure_peak(hb_system *h, const char *which, double *value);
// accessors
cudaError_t launch_pack_state(hb_system *h, const float *pos_xyz, const int32_t *type, const float *vel_xyz, const int32_t *image);
cudaError_t launch_unpack_state(hb_system *h, float *pos_xyz, int32_t *type, float *vel_xyz, int32_t *image);
cudaError_t launch_unpack_forces(hb_system *h, float *f4, float *vir6);
cudaError_t launch_mass(hb_system *h, const float *mass_in, float *mass_out);   // by tag: set (mass_in) or get (mass_out)
cudaError_t launch_nlist_counts_by_tag(hb_system *h, int *counts);
cudaError_t launch_nlist_fill_by_tag(hb_system *h, const int64_t *row_start, uint32_t *out);
cudaError_t launch_nlist_rows_by_tag(hb_system *h, const int *counts, int64_t *rows);   // exclusive scan, rows[N] = total
