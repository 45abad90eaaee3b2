// Internal declarations of libhb (sm_100a).  Not part of the ABI.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <string>
#include <vector>
#include <map>
#include <algorithm>

#include "../../include/hb.h"

// Device-side flag words (one int array, mirrored in pinned host memory).
enum {
    FL_NEED_BUILD = 0,  // set by the drift kernel when a particle exceeded r_buff/2; cleared by the force kernel
    FL_MAX_NBRS = 1,    // atomicMax of row lengths NEEDED by the last build (may exceed row_pitch => overflow)
    FL_BAD = 2,         // non-finite / out-of-box particle seen while binning
    FL_BUILDS = 3,      // number of list builds done on the device
    FL_DONE_CTR = 4,    // "last block done" counter of the drift kernel
    FL_OVERFLOWED = 5,  // sticky: some build since the last host check overflowed its rows
    FL_COUNT = 8
};

struct PairParam {  // one per type pair, 16 B
    float lj1;      // 4 eps sigma^12
    float lj2;      // 4 eps sigma^6
    float rcut2;    // r_cut^2
    float eshift;   // V_lj(r_cut) if energy shift, else 0
};

struct Tunables {
    int tpp = 8;
    int force_block = 128;
    int force_passes = 0;  // 0 = auto
    int nlist_ppi = 4;
    int nlist_cap = 512;
    int row_pitch = 0;
    int cell_sort = 1;
    int graph_mode = 2;
    int graph_steps = 50;
};

struct hb_system {
    int64_t N = 0;
    int ntypes = 1;
    float L = 0, r_cut_max = 0, r_buff = 0, r_max = 0;
    int shift_mode = HB_SHIFT_ENERGY;
    bool rcut_user = false;  // hb_set_rcut_pair was called
    std::vector<double> eps, sigma, rcut;
    std::vector<PairParam> h_params;
    cudaStream_t stream = nullptr;
    hb_allocator alloc{};
    bool has_alloc = false;
    Tunables tun;
    std::string err;

    // particle data (storage order), SoA of 16 B vectors
    float4 *pos = nullptr;      // x, y, z, type bits
    float4 *vel = nullptr;      // vx, vy, vz, unused
    float4 *force = nullptr;    // Fx, Fy, Fz, U_i
    float4 *virial = nullptr;   // [2N]: (xx, xy, xz, yy), (yz, zz, 0, 0)
    int *image = nullptr;       // [3][N]
    uint32_t *tag = nullptr;    // storage slot -> tag
    uint32_t *rtag = nullptr;   // tag -> storage slot
    float4 *pos_build = nullptr;
    // second set for hb_sort's gather and hb_run_nve's chunk backup
    float4 *pos2 = nullptr, *vel2 = nullptr, *force2 = nullptr, *virial2 = nullptr;
    int *image2 = nullptr;
    uint32_t *tag2 = nullptr;
    float4 *bk_pos = nullptr, *bk_vel = nullptr, *bk_force = nullptr, *bk_virial = nullptr, *bk_pos_build = nullptr;
    int *bk_image = nullptr;
    PairParam *params = nullptr;

    // cell list (CSR)
    int m = 0;
    int64_t ncells = 0, ncells_alloc = 0;
    int *cell_count = nullptr;   // [ncells]
    int *cell_start = nullptr;   // [ncells + 1]
    int *cell_rank = nullptr;    // [N] slot inside the cell handed out by the atomic
    float4 *cell_xyzi = nullptr; // [N] (x, y, z, index bits) in CSR order -- the paper's celldata
    int *scan_tmp = nullptr;     // block sums
    int64_t scan_tmp_len = 0;

    // neighbor list: row i = nlist[i * row_pitch .. + nlistn[i])
    int row_pitch = 0;
    int *nlist = nullptr;
    int *nlistn = nullptr;
    int64_t nlist_alloc = 0;

    // sort scratch
    uint32_t *keys = nullptr, *keys2 = nullptr, *perm = nullptr, *perm2 = nullptr;
    int *radix_counts = nullptr;
    int64_t radix_counts_len = 0;

    // flags + reductions
    int *flags = nullptr;        // device [FL_COUNT]
    int *h_flags = nullptr;      // pinned host mirror
    double *thermo_part = nullptr;  // [blocks][12]
    double *h_thermo = nullptr;     // pinned [12]
    int thermo_blocks = 0;
    int sm_count = 148;

    // host-side state machine
    bool have_state = false, cells_valid = false, nlist_valid = false, forces_valid = false, bk_valid = false;
    hb_stats_t stats{};
    int64_t builds_seen = 0;
    int64_t since_sort = -1;     // steps since the last hb_sort inside hb_run_nve (-1 = never sorted)

    // graph cache: key = (nsteps, mode, flags) -> exec
    struct GraphEntry { cudaGraph_t g = nullptr; cudaGraphExec_t e = nullptr; int nkernels_fixed = 0; };
    std::map<int64_t, GraphEntry> graphs;
    float graph_dt = 0;
    int graph_sig = 0;
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

// ---- kernel launchers (each enqueues on h->stream and returns cudaGetLastError) ----
// cells.cu
cudaError_t launch_cell_clear(hb_system *h, const int *pred);
cudaError_t launch_cell_bin(hb_system *h, const int *pred);
cudaError_t launch_scan_exclusive(hb_system *h, const int *in, int *out, int64_t n, int *tmp, const int *pred);
cudaError_t launch_cell_scatter(hb_system *h, const int *pred);
cudaError_t launch_cell_sort(hb_system *h, const int *pred);
// nlist.cu
cudaError_t launch_nlist(hb_system *h, const int *pred);
size_t nlist_smem_bytes(const hb_system *h);
// force.cu
cudaError_t launch_force(hb_system *h);
// nve.cu
//   mode bit 0: do the second half kick of the previous step first; bit 1: do the first half kick + drift
cudaError_t launch_nve(hb_system *h, float dt, bool kick_prev, bool kick_drift, cudaGraphConditionalHandle cond, bool use_cond);
cudaError_t launch_thermo(hb_system *h);
// sort.cu
cudaError_t launch_sfc_keys(hb_system *h);
cudaError_t launch_radix_sort(hb_system *h, int key_bits);  // keys/perm -> sorted in keys/perm
cudaError_t launch_gather_state(hb_system *h);              // by perm into the second set
cudaError_t launch_rtag(hb_system *h);
// accessors
cudaError_t launch_pack_state(hb_system *h, const float *pos_xyz, const int32_t *type, const float *vel_xyz, const int32_t *image);
cudaError_t launch_unpack_state(hb_system *h, float *pos_xyz, int32_t *type, float *vel_xyz, int32_t *image);
cudaError_t launch_unpack_forces(hb_system *h, float *f4, float *vir6);
cudaError_t launch_cell_tags(hb_system *h, uint32_t *out);
cudaError_t launch_nlist_counts_by_tag(hb_system *h, int *counts);
cudaError_t launch_nlist_fill_by_tag(hb_system *h, const int64_t *row_start, uint32_t *out);
