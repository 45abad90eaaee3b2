/*
 * hb.h -- C ABI of libhb: the data-parallel hot path of one molecular-dynamics
 * time step as described in arXiv 1308.5587 (HOOMD-blue, Anderson & Glotzer),
 * written from scratch for NVIDIA B200 (sm_100a).
 *
 *   cell list (Algorithm 2)
 *   -> neighbor list with cutoff r_max = r_cut + r_buff (Algorithm 3),
 *      reused until a particle has moved more than r_buff/2
 *   -> Lennard-Jones pair force, energy and virial per particle
 *   -> velocity-Verlet NVE half-steps with image flags
 *   +  periodic space-filling-curve sort of the particles
 *   +   XPLOR smoothing, Nose-Hoover and Langevin integration,
 *      Gaussian / Yukawa / Morse pair functors, per-particle mass,
 *      per-type-pair list cutoffs and a binary64 variant.
 *
 * Every step runs in CUDA kernels; there is no CPU fallback.  One GPU, one
 * stream, no collectives.  Citations are PAPER.md:<line>; "reading" refers to
 * the list of readings in DESIGN.md.
 *
 * Conventions
 *   - Every call returns int: HB_OK (0) or a negative HB_E* code;
 *     hb_last_error(h) gives a message owned by the handle (valid until the
 *     next call on that handle).  No exception crosses this boundary.
 *   - Box: cubic, periodic, from b = -L/2 to b + L = +L/2.
 *   - Tables are row-major [ntypes][ntypes] and must be symmetric.
 *   - L, eps, sigma, r_cut, r_buff, dt are taken as double and rounded ONCE to
 *     binary32; all device arithmetic is binary32 (the paper's GPU precision,
 *     PAPER.md:308) unless the tunable "precision" is 64; hb_thermo accumulates
 *     in binary64.
 *   - A handle is not thread-safe; different handles may be used from different
 *     host threads at the same time.
 *   - Work is enqueued on the cudaStream_t given to hb_create.  Calls that
 *     return data to the host synchronise that stream; the others may not.
 *   - Pointers passed in are caller-owned and never retained.  `on_device`
 *     says whether they are device (1) or host (0) pointers.
 *   - Particles keep a tag (their index at hb_set_state).  hb_sort and every
 *     list build change the storage order; every accessor reports BY TAG, so
 *     results do not depend on the current order.
 *   - Virial component order: xx, xy, xz, yy, yz, zz.
 */
#ifndef HB_H
#define HB_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#if defined(__GNUC__)
#define HB_API __attribute__((visibility("default")))
#else
#define HB_API
#endif

#define HB_OK 0
#define HB_EINVAL (-1)  /* bad argument (NULL handle, N <= 0, asymmetric table, ...) */
#define HB_ECUDA (-2)   /* a CUDA runtime call or kernel failed; see hb_last_error */
#define HB_ENOMEM (-3)  /* device allocation failed */
#define HB_EBOX (-4)    /* L < 2 r_max or fewer than 3 cells per axis: 27 adjacent cells would alias */
#define HB_ESTATE (-5)  /* stage called before its prerequisite (no state, no list, ...) */
#define HB_ENAN (-6)    /* a non-finite or out-of-box particle was seen while binning */

#define HB_SHIFT_NONE 0   /* V = V_lj(r) */
#define HB_SHIFT_ENERGY 1 /* V = V_lj(r) - V_lj(r_cut); same force */
#define HB_XPLOR 2        /* V = V_lj(r) S(r): XPLOR smoothing from r_on to r_cut, V and dV/dr -> 0 at r_cut
                             (PAPER.md:355-367); r_on per type pair from hb_set_ron_pair */

/* Pair potentials through the same kernel (a functor that returns V(r) and -(1/r) dV/dr; the paper names
 * Gaussian, Yukawa and Morse, and prints no formula: reading f1 of DESIGN.md, the textbook
 * forms).  The eps / sigma tables of hb_create and the p2 table of hb_set_pair_potential hold the parameters:
 *   HB_POT_LJ      V = 4 eps [(sigma/r)^12 - (sigma/r)^6]
 *   HB_POT_GAUSS   V = eps exp(-r^2 / (2 sigma^2))
 *   HB_POT_YUKAWA  V = eps exp(-kappa r) / r,                       kappa = sigma
 *   HB_POT_MORSE   V = D0 [e^{-2 a (r - r0)} - 2 e^{-a (r - r0)}],   D0 = eps, a = sigma, r0 = p2 */
#define HB_POT_LJ 0
#define HB_POT_GAUSS 1
#define HB_POT_YUKAWA 2
#define HB_POT_MORSE 3

typedef struct hb_system hb_system;

/* Optional device allocator (e.g. PyTorch's caching allocator).  alloc returns
 * a device pointer aligned to >= 256 B or NULL; both are called on the host. */
typedef struct hb_allocator {
    void *(*alloc)(size_t bytes, void *cuda_stream, void *user);
    void (*free)(void *ptr, void *cuda_stream, void *user);
    void *user;
} hb_allocator;

/* Thermodynamic sums: K = 1/2 sum m v^2, U = sum U_i,
 * W = sum W_i, P = (2K + tr W) / (3 L^3), p = sum m v  (m = 1 unless hb_set_mass was called). */
typedef struct hb_thermo_t {
    double K, U, W[6], P, px, py, pz;
} hb_thermo_t;

typedef struct hb_stats_t {
    int64_t steps;            /* NVE steps taken since hb_create */
    int64_t rebuilds;         /* neighbor-list builds */
    int64_t sorts;            /* hb_sort calls (incl. those made by hb_run_nve) */
    int64_t overflow_retries; /* times the list rows were grown and work redone */
    int64_t max_nbrs;         /* longest row of the current list */
    int64_t row_pitch;        /* 16-bit entries per list row (multiple of 64 = 128 B) */
    int64_t cells_per_axis;   /* m */
    int64_t graph_launches;   /* CUDA graph launches made by hb_run_nve */
    int64_t kernel_launches;  /* kernels enqueued (graph nodes counted when they run) */
    int64_t graph_builds;     /* CUDA graphs captured and instantiated so far (none after the first hb_run_nve
                                 unless a tunable, dt, r_buff or an array size changes) */
} hb_stats_t;

/* Create a system of N particles in a cubic box of edge L with ntypes types and
 * LJ tables eps, sigma [ntypes*ntypes] (parameters per type pair).
 * cuda_stream: a cudaStream_t (NULL = the legacy default stream).
 * alloc: NULL = cudaMalloc/cudaFree.  r_cut defaults to 2.5 sigma_ab until
 * hb_set_rcut_pair / hb_build_nlist says otherwise. */
HB_API int hb_create(hb_system **out, int64_t N, double L, int ntypes, const double *eps, const double *sigma,
              void *cuda_stream, const hb_allocator *alloc);
HB_API int hb_destroy(hb_system *h);

/* Upload the state: pos_xyz [N][3] inside [-L/2, L/2), type [N] in 0..ntypes-1,
 * vel_xyz [N][3], image [N][3] (NULL = zeros).  Tags are reset to 0..N-1, the
 * list and the forces become stale. */
HB_API int hb_set_state(hb_system *h, const float *pos_xyz, const int32_t *type, const float *vel_xyz,
                 const int32_t *image, int on_device);
/* Download the state BY TAG.  Any output pointer may be NULL.  order [N]
 * (nullable) receives, for each storage slot k, the tag stored there. */
HB_API int hb_get_state(hb_system *h, float *pos_xyz, int32_t *type, float *vel_xyz, int32_t *image,
                 uint32_t *order, int on_device);

/* The same in binary64 (the double-precision build).  With the tunable
 * "precision" = 64 the force sums and the integration run in binary64 on these arrays (kept by tag); the cell list and
 * the neighbor list are still built from the positions rounded to binary32.  With "precision" = 32 hb_set_state_f64
 * rounds its input and hb_get_state_f64 widens the binary32 state.  pos_xyz, vel_xyz [N][3], image [N][3] (nullable),
 * BY TAG.  hb_get_forces_f64: f_xyz_u [N][4], virial6 [N][6] (nullable) of the binary64 sums; HB_ESTATE unless
 * "precision" = 64. */
HB_API int hb_set_state_f64(hb_system *h, const double *pos_xyz, const int32_t *type, const double *vel_xyz,
                     const int32_t *image, int on_device);
HB_API int hb_get_state_f64(hb_system *h, double *pos_xyz, double *vel_xyz, int32_t *image, int on_device);
HB_API int hb_get_forces_f64(hb_system *h, double *f_xyz_u, double *virial6, int on_device);

/* Per-type-pair cutoffs r_cut,ab [ntypes*ntypes].  The list is
 * built with the largest of them (reading c2.iii); the force applies each. */
HB_API int hb_set_rcut_pair(hb_system *h, const double *rcut);

/* Per-type-pair onset r_on,ab [ntypes*ntypes] of the XPLOR switching function S(r), used by
 * hb_compute_lj(HB_XPLOR).  Default: 3/2 sigma_ab, the paper's test value.  r_on,ab >= r_cut,ab
 * leaves no switching interval: that pair is plainly truncated (reading x1). */
HB_API int hb_set_ron_pair(hb_system *h, const double *ron);

/* The pair potential evaluated by hb_compute_lj and the integrators (default HB_POT_LJ), with any of the three cutoff
 * treatments (HB_SHIFT_NONE, HB_SHIFT_ENERGY, HB_XPLOR).  p2 [ntypes*ntypes], symmetric: the third parameter table
 * (Morse r0); NULL = zeros.  Forces become stale. */
HB_API int hb_set_pair_potential(hb_system *h, int pot, const double *p2);

/* Per-particle masses, mass [N] BY TAG, all > 0; they enter the velocity updates (v += dt/2 F/m), the
 * thermostats (readings n1, n2: friction and noise are forces) and hb_thermo.  hb_set_state resets every mass to 1.
 * hb_get_mass downloads them by tag. */
HB_API int hb_set_mass(hb_system *h, const float *mass, int on_device);
HB_API int hb_get_mass(hb_system *h, float *mass, int on_device);

/* Algorithm 2: bin the particles into m^3 cells, m = floor(L / r_max), with
 * c = floor((x - b) m / L) per axis evaluated in binary32 without contraction
 * (reading c1).  Uses the r_max of the last hb_build_nlist (or r_cut,max +
 * 0 if none).  Result: CSR cell list in cell-id order c = cx + m (cy + m cz).
 * The particle data is re-ordered into cell order (tags are kept; an existing
 * list and the forces become stale).  A no-op when the cell list of the
 * current positions is already in place. */
HB_API int hb_build_cells(hb_system *h);

/* Algorithm 3: N(i) = { j != i : |minimage(R_i - R_j)| < r_cut + r_buff }, full
 * list, rows padded to a multiple of 128 B.  r_cut <= 0 keeps the per-pair table
 * maximum; otherwise it REPLACES every r_cut,ab not set by hb_set_rcut_pair.
 * Builds the cells first.  Row overflow is detected, rows are grown and the
 * build redone.  Remembers the build positions for the
 * r_buff/2 rule. */
HB_API int hb_build_nlist(hb_system *h, double r_cut, double r_buff);

/* Reading c3: *need = 1 iff some particle is now farther than r_buff/2 from
 * where it was when the list was built (or there is no list). */
HB_API int hb_needs_rebuild(hb_system *h, int *need);

/* F_i, U_i = 1/2 sum V, W_i = 1/2 sum d f over the listed neighbors with
 * r < r_cut,ab.  shift_mode: HB_SHIFT_NONE, HB_SHIFT_ENERGY or HB_XPLOR; it stays in
 * force for hb_step_nve / hb_run_nve.  HB_ESTATE if there is no list. */
HB_API int hb_compute_lj(hb_system *h, int shift_mode);

/* One velocity-Verlet step: half kick, drift, wrap with
 * image flags, rebuild if the buffer is exceeded, forces, half kick.  Computes
 * the list and F(t) first if they are stale.  Uses the shift mode and r_buff
 * of the last hb_compute_lj / hb_build_nlist. */
HB_API int hb_step_nve(hb_system *h, double dt);

/* nsteps of the same, enqueued as CUDA graphs with the rebuild decision taken
 * on the device (no host round trip per step); hb_sort every sort_period steps
 * (0 = never).  Row overflow inside the run is repaired by restoring the state
 * saved at the start of the affected chunk and redoing it with longer rows. */
HB_API int hb_run_nve(hb_system *h, double dt, int64_t nsteps, int64_t sort_period);

/* The same loop with a thermostat (the paper names the integrators, PAPER.md:87, 99, 324,
 * and prints no equations: readings n1, n2, m1 of DESIGN.md).  k_B = 1; m is the particle's mass (1 unless hb_set_mass).
 * hb_run_nvt: Nose-Hoover, dv/dt = F / m - xi v, dxi/dt = (T_k / T - 1) / tau^2 with T_k = 2K / (3N - 3); the
 *   thermostat variable xi and its time integral eta live in the handle (hb_get_thermostat / hb_set_thermostat;
 *   hb_set_state zeroes them); K + U + (3N - 3) T (tau^2 xi^2 / 2 + eta) is conserved.
 * hb_run_langevin: after every velocity-Verlet step v <- v (1 - gamma dt / m) + sqrt(6 gamma T dt) / m u (friction and
 *   noise are forces: both divided by the mass), u uniform in
 *   (-1, 1) from the counter-based generator splitmix64(seed, time step number, 3 tag + component); the time step
 *   number counts the Langevin steps since hb_set_state (hb_get_thermostat reports it). */
HB_API int hb_run_nvt(hb_system *h, double dt, int64_t nsteps, int64_t sort_period, double T, double tau);
HB_API int hb_run_langevin(hb_system *h, double dt, int64_t nsteps, int64_t sort_period, double T, double gamma, uint64_t seed);
HB_API int hb_get_thermostat(hb_system *h, double *xi, double *eta, int64_t *langevin_steps);
HB_API int hb_set_thermostat(hb_system *h, double xi, double eta, int64_t langevin_steps);

/* Reorder the particles along a Hilbert curve on a 2^8 grid per axis, equal keys
 * in tag order (reading c8); permutes every per-particle array, keeps the
 * tags, invalidates the list.  (Every list build re-orders the particles into
 * cell order anyway; inside a cell the order set here survives.) */
HB_API int hb_sort(hb_system *h);

/* Thermodynamic sums of the current state.  If the forces are stale (after hb_set_state, hb_build_nlist,
 * hb_build_cells, hb_sort) the list is rebuilt if needed and the forces are evaluated first. */
HB_API int hb_thermo(hb_system *h, hb_thermo_t *out);

/* The same sums for a caller that is not allowed to allocate device memory.
 *
 * Who that is: code that runs when the GPU's memory has already been handed out and must stay that way.  A host
 * program that gave the whole device to its own pool at start-up (a framework's caching allocator with a fixed
 * budget, a simulation whose arrays were sized to fill HBM) can see cudaMalloc fail, or has a rule against going
 * round the pool.  A logger or analysis hook that somebody else's time-step loop calls between steps must not
 * stall that loop, and cudaMalloc / cudaFree synchronise the whole device.  hb_create and hb_thermo are no use to
 * such a caller: the first allocates every array of the system, the second reads them.
 *
 * So this call takes no handle and allocates nothing, on the device or through any CUDA library: no cudaMalloc,
 * cudaFree, stream-ordered or pool allocation, pinned host memory.  The caller passes its own arrays, all DEVICE
 * pointers on the current device, in the layouts hb_get_state / hb_get_mass / hb_get_forces write:
 *   vel_xyz    [N][3]                     (required)
 *   mass       [N]      NULL = every mass is 1
 *   f_xyz_u    [N][4]   (Fx, Fy, Fz, U_i); only U_i is read.  NULL = U is reported as 0
 *   virial6    [N][6]   xx, xy, xz, yy, yz, zz.  NULL = W is reported as 0 (P is then the ideal-gas part)
 *   out_device          one hb_thermo_t in device memory, written by the last kernel
 * The order of the particles does not matter (these are plain sums).  L is the box edge, for P = (2K + tr W) / (3 L^3).
 * Two kernels are enqueued on cuda_stream (a cudaStream_t of the current device, NULL = the legacy default
 * stream); the call does not wait for them: order your read of out_device after them on that stream.
 *
 * The only memory the reduction needs besides inputs and output -- 11 binary64 partial sums per block of 4096
 * particles -- is a fixed array of 360,448 bytes compiled into the library.  Consequences to know about:
 *   - Limit: N <= HB_THERMO_STATIC_MAX_N (16,777,216).  A larger N is refused with HB_EINVAL and a message that
 *     names the limit; nothing is launched.  (Sums are additive: split the particles over several calls, or use
 *     hb_thermo.)
 *   - Every GPU on which this library is loaded holds those 360,448 bytes until the process exits.
 *   - The first call made on each device looks up that device's address of the array (cudaGetSymbolAddress, with
 *     that device current; the runtime may load the library's GPU code at that moment).  It is remembered per
 *     device afterwards.  Make that first call at set-up time, before any stream capture is begun.
 *   - All calls on one device share the one array.  Calls whose kernels can run at the same time on that device
 *     (different streams, different host threads) overwrite each other's partial sums: keep them ordered, e.g. on
 *     one stream.  Nothing needs clearing between calls: a call writes every partial sum before it reads it.
 * Accumulation is binary64, and which particles share a partial sum depends on N only, so the result does not
 * depend on the GPU model.  It can differ from hb_thermo's in the last bits (another summation order).
 * errbuf (nullable) receives a NUL-terminated message when the return value is not HB_OK; there is no handle to
 * ask.  Returns HB_OK, HB_EINVAL (NULL vel_xyz / out_device, N < 1, N over the limit, L <= 0) or HB_ECUDA. */
#define HB_THERMO_STATIC_MAX_N 16777216LL
HB_API int hb_thermo_static(const float *vel_xyz, const float *mass, const float *f_xyz_u, const float *virial6,
                     int64_t N, double L, hb_thermo_t *out_device, void *cuda_stream, char *errbuf, size_t errbuf_len);

/* Cell list: m_out [3]; cell_start [m^3+1]; cell_tags [N] = tags of the members
 * of each cell in CSR order (order inside a cell is undefined).
 * Pass NULL to skip an output.  Sizes: call once with only m_out. */
HB_API int hb_get_cells(hb_system *h, int32_t *m_out, int32_t *cell_start, uint32_t *cell_tags, int on_device);
/* Neighbor list BY TAG as CSR: row_start [N+1] (int64), nbr_tags
 * [row_start[N]] (NULL = sizes only).  Order inside a row is undefined. */
HB_API int hb_get_nlist(hb_system *h, int64_t *row_start, uint32_t *nbr_tags, int on_device);
/* f_xyz_u [N][4] = (Fx, Fy, Fz, U_i), virial6 [N][6] (nullable), BY TAG. */
HB_API int hb_get_forces(hb_system *h, float *f_xyz_u, float *virial6, int on_device);

HB_API int hb_stats(hb_system *h, hb_stats_t *out);

/* Tunables never change results beyond summation order.
 *   "tpp"            threads per particle in the force kernel: 2,4,8
 *   "epl"            list entries per thread per iteration in the force kernel: 4,8 (8 only with tpp <= 4)
 *   "nlist_ppi"      particles tested per candidate load in the list kernel: 1,2,4
 *   "tile_x/y/z"     cells per tile (one thread block stages one tile and its one-cell halo in
 *                    shared memory); 0 = chosen from m and the SM count.  Needs
 *                    (tx+2)(ty+2)(tz+2) <= 256 and ty*tz <= 32 after clipping to m.
 *   "stage_cap"      shared-memory slots per tile (0 = from the density); grown on overflow
 *   "row_pitch"      initial entries per list row (rounded up to 64; 0 = estimate)
 *   "grow_pct"       head room in percent when rows / the staging area are grown after an overflow (25)
 *   "cell_sort"      1 = members of a cell ordered by index: the same lists, in the same order, run after run, FOR GIVEN
 *                    tile sizes, "stage_cap" and "row_pitch".  The order inside a row follows the slot numbering of the
 *                    staged tile, so after an overflow has grown the rows or the staging area the redone
 *                    work sums the same pairs in another order: results then agree with a run that had room from the
 *                    start to rounding (1e-4 relative in the tests), not bit for bit
 *   "force_block"    threads per block of the force kernel: 128, 256
 *   "nlist_block"    threads per block of the stand-alone list kernel: 128, 256
 *   "thermo_every"   0 = (default) inside hb_run_nve U_i and W_i are computed by the last step of every chunk only:
 *                        those of an inner step cannot be read by anyone, the trajectory is the same bit for bit,
 *                        and energies, virials and hb_thermo are valid whenever hb_run_nve returns;
 *                    1 = every step computes them (the paper's kernel does)
 *   "fuse_nve"       1 = hb_run_nve integrates inside the force kernel (one kernel per step)
 *   "coop_rebuild"   0 = the rebuild is five launches (count, scan, scatter, gather, list);
 *                    1 = Algorithm 2 and the reorder are ONE cooperative kernel, then the list kernel;
 *                    2 = the list build is a phase of that kernel too
 *   "coop_blocks"    blocks per SM of the cooperative cell kernel (1..8)
 *   "graph_mode"     0 = no graphs (host reads the flag each step)
 *                    1 = graphs of kernels that exit early unless rebuilding
 *                    2 = graphs with a conditional IF node around the rebuild
 *                    3 = the launches of mode 1 issued one by one, no graph (for profilers)
 *   "graph_steps"    steps per graph launch
 *   "nlist_pair_rcut" 1 = the list keeps pair (i, j) iff d < r_cut(type i, type j) + r_buff (reading t1; up to 8 types);
 *                    0 = (default) one list cutoff, the largest (reading c2.iii)
 *   "precision"      32 = (default) binary32 arithmetic (the paper's GPU precision);
 *                    64 = force sums and velocity Verlet in binary64 (NVE, hb_step_nve / hb_run_nve one step per host
 *                         iteration; hb_run_nvt / hb_run_langevin return HB_EINVAL): what the arithmetic conserves
 *                         (Table 2), not a fast path
 */
HB_API int hb_set_tunable(hb_system *h, const char *name, int value);
HB_API int hb_get_tunable(hb_system *h, const char *name, int *value);

/* Measurement aid for bench.py: enqueue `reps` launches of one stage on the
 * system's stream between CUDA events and return the mean duration per launch
 * in milliseconds.  stage: "lj_force" (force kernel alone), "lj_nve" (force
 * kernel with both half kicks and the drift fused in, dt = 0: the kernel a
 * step of hb_run_nve is), "nlist" (Algorithm 3 kernel alone), "cells"
 * (Algorithm 2 chain + reorder), "rebuild" (cells + nlist), "nve" (stand-alone
 * kick + drift kernel with dt = 0).  The state is unchanged (cells/rebuild are
 * followed by an untimed rebuild).  If flush_l2_bytes > 0 a
 * scratch buffer of that size is overwritten before every launch (outside the
 * timed interval) so that each launch starts with a cold L2.  Needs a list. */
HB_API int hb_time_stage(hb_system *h, const char *stage, int reps, int64_t flush_l2_bytes, double *mean_ms);

/* Measured roofline denominators on this device, with kernels of this library:
 *   "fp32_tflops"  FFMA throughput, 8 independent chains per thread, all SMs        -> TFLOP/s
 *   "l2_gbs"       read bandwidth of a 32 MB buffer resident in L2, 16 B per load   -> GB/s
 *   "smem_gbs"     conflict-free 16-byte shared-memory loads, 4 independent address
 *                  streams per thread (no load feeds an address), all SMs           -> GB/s
 * Best of five timed launches (CUDA events on the system's stream); synchronises. */
HB_API int hb_measure_peak(hb_system *h, const char *which, double *value);

HB_API const char *hb_last_error(hb_system *h);
HB_API const char *hb_version(void);

#ifdef __cplusplus
}
#endif
#endif /* HB_H */
