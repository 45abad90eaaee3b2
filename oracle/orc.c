/*
 * orc.c -- the ORACLE: a plain, slow, fp64 CPU statement of what the hot path
 * of arXiv 1308.5587 (HOOMD-blue) computes for one Lennard-Jones NVE time step.
 *
 * THIS IS TEST INFRASTRUCTURE, NOT PRODUCT CODE.  Only tests/, the smoke check
 * in __graft_entry__.py and bench.py's cpu_baseline / --impl reference legs may
 * build, load or call it.  It shares no code, header, table or helper with the
 * CUDA library (paper_1308_5587_b200/csrc) and neither includes the other.
 *
 * Style: every function is the paper's definition written out, in the paper's
 * order and notation, in double precision.  No blocking, fusion, tiling or
 * reordering; the only parallelism is an optional `omp parallel for` over the
 * particle index i, which leaves each particle's arithmetic untouched.
 *
 * Parity status: every function below is pinned by tests/test_oracle_*.py
 * (closed forms, O(N^2) brute force, invariants); nothing is "parity unpinned".
 *
 * Citations are PAPER.md:<line> (the extracted paper) and the readings of
 * SURVEY.md section 8(c) / DESIGN.md "Readings".
 *
 * Conventions
 *   box      cubic, periodic, from b = -L/2 to b + L = +L/2
 *   pos      double [N][3];  type int32 [N];  tables [ntypes*ntypes] row-major
 *   cell id  c = cx + m*(cy + m*cz)
 *   virial   six components in the order xx, xy, xz, yy, yz, zz
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#define ORC_OK 0
#define ORC_EBOX -1   /* L < 2 r_max or fewer than 3 cells per axis */
#define ORC_ECAP -2   /* caller's buffer too small */
#define ORC_ENOMEM -3

/* ------------------------------------------------------------------ c1 ---- */
/* Cells per axis.  [reading c1.ii] m = floor(L / r_max), so that the cell
 * width L/m >= r_max and the 27 adjacent cells of Alg. 3 l.11 suffice. */
int orc_cell_dim(double L, double r_max)
{
    return (int)floor(L / r_max);
}

/* Algorithm 2 lines 5-9: shift to the box origin, scale by
 * s = m/L, floor.  [reading c1.i] "r + b" is read as x - b with b = -L/2.
 * [reading c1.iii] a result outside 0..m-1 is wrapped periodically.
 * [reading c1.iv] CANONICAL value: the same expression in IEEE binary32,
 * each operation rounded separately (no fused multiply-add), because
 * "bit-exact membership" needs one pinned formula.  Compile with
 * -ffp-contract=off. */
void orc_cell_index_f32(const float *pos, int64_t N, float L, int m, int32_t *cell)
{
    const float b = -0.5f * L;
    const float s = (float)m / L;
    for (int64_t i = 0; i < N; i++) {
        int c[3];
        for (int a = 0; a < 3; a++) {
            volatile float r = pos[3 * i + a] - b;   /* line 6 */
            volatile float u = r * s;                /* lines 7-9 */
            int ca = (int)floorf(u);
            if (ca >= m) ca -= m;
            if (ca < 0) ca += m;
            c[a] = ca;
        }
        cell[i] = c[0] + m * (c[1] + m * c[2]);
    }
}

/* The same index from the geometry in double.  margin[i] = distance of the
 * scaled coordinate to the nearest integer (min over axes): where it is tiny
 * the fp32 and fp64 answers may legitimately differ. */
void orc_cell_index_f64(const double *pos, int64_t N, double L, int m, int32_t *cell, double *margin)
{
    const double b = -0.5 * L;
    const double s = (double)m / L;
    for (int64_t i = 0; i < N; i++) {
        int c[3];
        double mg = 1.0;
        for (int a = 0; a < 3; a++) {
            double u = (pos[3 * i + a] - b) * s;
            double fl = floor(u);
            double d = fmin(u - fl, fl + 1.0 - u);
            if (d < mg) mg = d;
            int ca = (int)fl;
            if (ca >= m) ca -= m;
            if (ca < 0) ca += m;
            c[a] = ca;
        }
        cell[i] = c[0] + m * (c[1] + m * c[2]);
        if (margin) margin[i] = mg;
    }
}

/* Algorithm 2 lines 10-11: celln counts, then each particle
 * takes the next free slot of its cell.  Run serially in index order, so the
 * (undefined) entry order is ascending i.  Stored as CSR: members of cell c are
 * cell_members[cell_start[c] .. cell_start[c+1]). */
void orc_build_cells(const int32_t *cell, int64_t N, int m, int64_t *cell_start, int32_t *cell_members)
{
    const int64_t nc = (int64_t)m * m * m;
    int64_t *celln = (int64_t *)calloc((size_t)nc + 1, sizeof(int64_t));
    for (int64_t i = 0; i < N; i++) celln[cell[i]]++;
    cell_start[0] = 0;
    for (int64_t c = 0; c < nc; c++) cell_start[c + 1] = cell_start[c] + celln[c];
    memset(celln, 0, (size_t)nc * sizeof(int64_t));
    for (int64_t i = 0; i < N; i++) {
        int64_t n = celln[cell[i]]++;                 /* line 10: n <= atomicInc */
        cell_members[cell_start[cell[i]] + n] = (int32_t)i; /* line 11 */
    }
    free(celln);
}

/* ------------------------------------------------------------------ c2 ---- */
/* minimage (Alg. 3 l.16): nearest periodic image of a separation component. */
static inline double minimage(double d, double L)
{
    return d - L * rint(d / L);
}

static inline double dist2(const double *pos, int64_t i, int64_t j, double L, double d[3])
{
    d[0] = minimage(pos[3 * i + 0] - pos[3 * j + 0], L);
    d[1] = minimage(pos[3 * i + 1] - pos[3 * j + 1], L);
    d[2] = minimage(pos[3 * i + 2] - pos[3 * j + 2], L);
    return d[0] * d[0] + d[1] * d[1] + d[2] * d[2];
}

/* The DEFINITION of the neighbor set: N(i) = { j != i : |minimage(Ri-Rj)| < r_max }
 * (Alg. 3 l.17, strict <), by testing every pair.  Full list, ascending j.
 * Call with nbr == NULL to get the counts only. */
int orc_nlist_brute(const double *pos, int64_t N, double L, double r_max,
                    int32_t *count, const int64_t *row_start, int32_t *nbr)
{
    if (L < 2.0 * r_max) return ORC_EBOX;
    const double r_max2 = r_max * r_max;
#pragma omp parallel for schedule(dynamic, 64)
    for (int64_t i = 0; i < N; i++) {
        int32_t n = 0;
        double d[3];
        for (int64_t j = 0; j < N; j++) {
            if (j == i) continue;
            if (dist2(pos, i, j, L, d) < r_max2) {
                if (nbr) nbr[row_start[i] + n] = (int32_t)j;
                n++;
            }
        }
        count[i] = n;
    }
    return ORC_OK;
}

/* The same set for a SAMPLE of particles (full-size spot checks): rows for
 * sample[0..S) only, each tested against all N. */
int orc_nlist_brute_sample(const double *pos, int64_t N, double L, double r_max,
                           const int64_t *sample, int64_t S,
                           int32_t *count, const int64_t *row_start, int32_t *nbr)
{
    if (L < 2.0 * r_max) return ORC_EBOX;
    const double r_max2 = r_max * r_max;
#pragma omp parallel for schedule(dynamic, 4)
    for (int64_t k = 0; k < S; k++) {
        const int64_t i = sample[k];
        int32_t n = 0;
        double d[3];
        for (int64_t j = 0; j < N; j++) {
            if (j == i) continue;
            if (dist2(pos, i, j, L, d) < r_max2) {
                if (nbr) nbr[row_start[k] + n] = (int32_t)j;
                n++;
            }
        }
        count[k] = n;
    }
    return ORC_OK;
}

/* Algorithm 3, step by step, one particle at a time.
 * [reading c2.i] line 15 is read as (R_j, j) <= celldata[o, d].
 * [reading c2.ii] nlistn is written after the loop over a.
 * `cell` is the cell of every particle as used to build cell_start/members
 * (lines 5-9 recompute exactly that).  celladj (line 12) is computed on the fly:
 * the 27 cells (cx+ax, cy+ay, cz+az), a in {-1,0,1}^3, wrapped periodically.
 * Call with nbr == NULL to get the counts only. */
int orc_nlist_cells(const double *pos, int64_t N, double L, double r_max, int m,
                    const int32_t *cell, const int64_t *cell_start, const int32_t *cell_members,
                    int32_t *count, const int64_t *row_start, int32_t *nbr)
{
    if (m < 3 || L < 2.0 * r_max || L / m < r_max) return ORC_EBOX;
    const double r_max2 = r_max * r_max;
#pragma omp parallel for schedule(dynamic, 64)
    for (int64_t i = 0; i < N; i++) {
        const int cx = cell[i] % m, cy = (cell[i] / m) % m, cz = cell[i] / (m * m);
        int32_t n_neigh = 0;                                   /* line 10 */
        for (int a = 0; a < 27; a++) {                         /* line 11 */
            const int dx = (cx + (a % 3) - 1 + m) % m;         /* line 12 */
            const int dy = (cy + ((a / 3) % 3) - 1 + m) % m;
            const int dz = (cz + (a / 9) - 1 + m) % m;
            const int64_t dcell = dx + (int64_t)m * (dy + (int64_t)m * dz);
            const int64_t n_d = cell_start[dcell + 1] - cell_start[dcell]; /* line 13 */
            for (int64_t o = 0; o < n_d; o++) {                /* line 14 */
                const int64_t j = cell_members[cell_start[dcell] + o]; /* line 15 */
                double r[3];
                const double r2 = dist2(pos, i, j, L, r);      /* line 16 */
                if (r2 < r_max2 && i != j) {                   /* line 17 */
                    if (nbr) nbr[row_start[i] + n_neigh] = (int32_t)j; /* line 18 */
                    n_neigh++;                                 /* line 19 */
                }
            }
        }
        count[i] = n_neigh;                                    /* line 22 */
    }
    return ORC_OK;
}

/* NEXT-3: per-type-pair cutoff in the LIST.  The paper gives every pair of types its own r_cut and
 * builds the list with r_cut + r_buff; the base path uses the single largest cutoff for the list
 * [reading c2.iii].  [reading t1] With per-pair list cutoffs the definition becomes
 *   N(i) = { j != i : |minimage(Ri - Rj)| < r_list(type_i, type_j) },  r_list,ab = r_cut,ab + r_buff  (strict <),
 * rlist[ntypes*ntypes] symmetric.  Definition by testing every pair, ascending j. */
int orc_nlist_brute_typed(const double *pos, const int32_t *type, int64_t N, double L, int ntypes, const double *rlist,
                          int32_t *count, const int64_t *row_start, int32_t *nbr)
{
    for (int p = 0; p < ntypes * ntypes; p++) if (L < 2.0 * rlist[p]) return ORC_EBOX;
#pragma omp parallel for schedule(dynamic, 64)
    for (int64_t i = 0; i < N; i++) {
        int32_t n = 0;
        double d[3];
        for (int64_t j = 0; j < N; j++) {
            if (j == i) continue;
            const double rl = rlist[type[i] * ntypes + type[j]];
            if (dist2(pos, i, j, L, d) < rl * rl) {
                if (nbr) nbr[row_start[i] + n] = (int32_t)j;
                n++;
            }
        }
        count[i] = n;
    }
    return ORC_OK;
}

/* The method's way: Algorithm 3 over the cells of the LARGEST list cutoff (r_max = max rlist: the 27 cells hold every
 * candidate), line 17 tested against the pair's own r_list. */
int orc_nlist_cells_typed(const double *pos, const int32_t *type, int64_t N, double L, int ntypes, const double *rlist, int m,
                          const int32_t *cell, const int64_t *cell_start, const int32_t *cell_members,
                          int32_t *count, const int64_t *row_start, int32_t *nbr)
{
    double r_max = 0.0;
    for (int p = 0; p < ntypes * ntypes; p++) if (rlist[p] > r_max) r_max = rlist[p];
    if (m < 3 || L < 2.0 * r_max || L / m < r_max) return ORC_EBOX;
#pragma omp parallel for schedule(dynamic, 64)
    for (int64_t i = 0; i < N; i++) {
        const int cx = cell[i] % m, cy = (cell[i] / m) % m, cz = cell[i] / (m * m);
        int32_t n_neigh = 0;
        for (int a = 0; a < 27; a++) {
            const int dx = (cx + (a % 3) - 1 + m) % m;
            const int dy = (cy + ((a / 3) % 3) - 1 + m) % m;
            const int dz = (cz + (a / 9) - 1 + m) % m;
            const int64_t dcell = dx + (int64_t)m * (dy + (int64_t)m * dz);
            const int64_t n_d = cell_start[dcell + 1] - cell_start[dcell];
            for (int64_t o = 0; o < n_d; o++) {
                const int64_t j = cell_members[cell_start[dcell] + o];
                double r[3];
                const double r2 = dist2(pos, i, j, L, r);
                const double rl = rlist[type[i] * ntypes + type[j]];
                if (r2 < rl * rl && i != j) {
                    if (nbr) nbr[row_start[i] + n_neigh] = (int32_t)j;
                    n_neigh++;
                }
            }
        }
        count[i] = n_neigh;
    }
    return ORC_OK;
}

/* ------------------------------------------------------------------ c3 ---- */
/* [reading c3] Rebuild rule: the list built at R^build stays valid while no
 * particle has moved more than r_buff/2 (PAPER.md:167 only says r_buff exists).
 * Returns max_i |minimage(R_i - R_i^build)|^2; rebuild iff it is > (r_buff/2)^2. */
double orc_max_disp2(const double *pos, const double *pos_build, int64_t N, double L)
{
    double mx = 0.0;
    for (int64_t i = 0; i < N; i++) {
        double s = 0.0;
        for (int a = 0; a < 3; a++) {
            double d = minimage(pos[3 * i + a] - pos_build[3 * i + a], L);
            s += d * d;
        }
        if (s > mx) mx = s;
    }
    return mx;
}

/* ------------------------------------------------------------- c4, c5 ---- */
/* V_lj(r) = 4 eps [ (sigma/r)^12 - alpha (sigma/r)^6 ], alpha = 1
 * -(1/r) dV/dr = (1/r^2) (48 eps (sigma/r)^12 - 24 eps (sigma/r)^6)
 * active iff r < r_cut; shift: V = V_lj(r) - V_lj(r_cut).
 * `shift` in the sums below is the mode: 0 plain, 1 energy shift, 2 XPLOR smoothing with r_on per type pair
 * (`ron`, nullable unless mode 2). */
static inline double vlj(double r, double eps, double sigma)
{
    const double sr = sigma / r;
    const double sr6 = sr * sr * sr * sr * sr * sr;
    return 4.0 * eps * (sr6 * sr6 - sr6);
}

void orc_lj_pair(double r, double eps, double sigma, double r_cut, int shift,
                 double *V, double *minus_dVdr_over_r)
{
    if (!(r < r_cut)) { *V = 0.0; *minus_dVdr_over_r = 0.0; return; }
    const double sr = sigma / r;
    const double sr6 = sr * sr * sr * sr * sr * sr;
    *minus_dVdr_over_r = (48.0 * eps * sr6 * sr6 - 24.0 * eps * sr6) / (r * r);
    *V = vlj(r, eps, sigma) - (shift ? vlj(r_cut, eps, sigma) : 0.0);
}

/* XPLOR smoothing (section 8.2.2):  V(r) = V_lj(r) S(r) with
 *   S(r) = 1                                                        r <  r_on
 *        = (rc^2 - r^2)^2 (rc^2 + 2 r^2 - 3 ron^2) / (rc^2 - ron^2)^3   r_on <= r <= r_cut
 *        = 0                                                        r >  r_cut
 * so that V and its first derivative go to 0 at r_cut.  The force follows by the
 * product rule:  -dV/dr = (-dV_lj/dr) S - V_lj S',
 *   S'(r) = 12 r (rc^2 - r^2)(ron^2 - r^2) / (rc^2 - ron^2)^3   (derivative of the line above),
 * returned, like orc_lj_pair, as -(1/r) dV/dr.  No energy shift is applied (S does that job).
 * [reading x1] r_on >= r_cut leaves no switching interval: S = 1 inside r_cut, i.e. the
 * plain truncated potential (the paper gives no rule for this case). */
void orc_lj_pair_xplor(double r, double eps, double sigma, double r_cut, double r_on,
                       double *V, double *minus_dVdr_over_r)
{
    double Vlj, flj;
    orc_lj_pair(r, eps, sigma, r_cut, 0, &Vlj, &flj);
    if (!(r < r_cut)) { *V = 0.0; *minus_dVdr_over_r = 0.0; return; }
    double S = 1.0, dS_over_r = 0.0;
    if (r >= r_on && r_on < r_cut) {
        const double rc2 = r_cut * r_cut, ron2 = r_on * r_on, r2 = r * r;
        const double D = (rc2 - ron2) * (rc2 - ron2) * (rc2 - ron2);
        S = (rc2 - r2) * (rc2 - r2) * (rc2 + 2.0 * r2 - 3.0 * ron2) / D;
        dS_over_r = 12.0 * (rc2 - r2) * (ron2 - r2) / D;          /* S'(r) / r */
    }
    *V = Vlj * S;
    *minus_dVdr_over_r = flj * S - Vlj * dS_over_r;
}

/* NEXT-3: other pair potentials through the same sums.  The paper names them (Gaussian; Yukawa and
 * Morse) and describes the mechanism -- a functor that returns V(r) and -(1/r) dV/dr --
 * but prints no formula; [reading f1] the textbook forms, with the per-type-pair tables `eps`, `sigma` and `p2`
 * reused as the potential's parameters:
 *   pot 0  Lennard-Jones   V = 4 eps [(sigma/r)^12 - (sigma/r)^6]
 *   pot 1  Gaussian        V = eps exp(-r^2 / (2 sigma^2))           -dV/dr = V r / sigma^2
 *   pot 2  Yukawa          V = eps exp(-kappa r) / r, kappa = sigma   -dV/dr = V (kappa + 1/r)
 *   pot 3  Morse           V = D0 [e^{-2 a (r - r0)} - 2 e^{-a (r - r0)}], D0 = eps, a = sigma, r0 = p2
 *                          -dV/dr = 2 a D0 [e^{-2 a (r - r0)} - e^{-a (r - r0)}]
 * Unshifted value and -(1/r) dV/dr at r (no cutoff applied here). */
void orc_pair_bare(int pot, double r, double eps, double sigma, double p2, double *V, double *minus_dVdr_over_r)
{
    if (pot == 1) {
        *V = eps * exp(-0.5 * (r / sigma) * (r / sigma));
        *minus_dVdr_over_r = *V / (sigma * sigma);
    } else if (pot == 2) {
        *V = eps * exp(-sigma * r) / r;
        *minus_dVdr_over_r = *V * (sigma + 1.0 / r) / r;
    } else if (pot == 3) {
        const double e1 = exp(-sigma * (r - p2));
        *V = eps * (e1 * e1 - 2.0 * e1);
        *minus_dVdr_over_r = 2.0 * sigma * eps * (e1 * e1 - e1) / r;
    } else {
        const double sr = sigma / r;
        const double sr6 = sr * sr * sr * sr * sr * sr;
        *V = 4.0 * eps * (sr6 * sr6 - sr6);
        *minus_dVdr_over_r = (48.0 * eps * sr6 * sr6 - 24.0 * eps * sr6) / (r * r);
    }
}

/* Any potential with the three cutoff treatments the paper describes for "every pair force":
 * mode 0 truncated, 1 energy-shifted V - V(r_cut), 2 XPLOR-smoothed V S(r). */
void orc_pair_generic(int pot, double r, double eps, double sigma, double p2, double r_cut, double r_on, int mode,
                      double *V, double *minus_dVdr_over_r)
{
    if (!(r < r_cut)) { *V = 0.0; *minus_dVdr_over_r = 0.0; return; }
    double v, f;
    orc_pair_bare(pot, r, eps, sigma, p2, &v, &f);
    if (mode == 1) {
        double vc, fc;
        orc_pair_bare(pot, r_cut, eps, sigma, p2, &vc, &fc);
        v -= vc;
    } else if (mode == 2 && r >= r_on && r_on < r_cut) {
        const double rc2 = r_cut * r_cut, ron2 = r_on * r_on, r2 = r * r;
        const double D = (rc2 - ron2) * (rc2 - ron2) * (rc2 - ron2);
        const double S = (rc2 - r2) * (rc2 - r2) * (rc2 + 2.0 * r2 - 3.0 * ron2) / D;
        const double dS_over_r = 12.0 * (rc2 - r2) * (ron2 - r2) / D;
        f = f * S - v * dS_over_r;
        v = v * S;
    }
    *V = v;
    *minus_dVdr_over_r = f;
}

/* The third per-type-pair table (Morse r0) of the force sums below; [ntypes*ntypes], copied.  NULL: zeros. */
static double g_p2[64 * 64];
void orc_set_p2(const double *p2, int n)
{
    for (int k = 0; k < 64 * 64; k++) g_p2[k] = (p2 && k < n) ? p2[k] : 0.0;
}

/* one entry point for the force sums.  `shift` carries the cutoff treatment in its two low bits (0 = plain,
 * 1 = energy shift, 2 = XPLOR) and the potential above them (shift >> 2: 0 LJ, 1 Gaussian, 2 Yukawa, 3 Morse). */
static inline void pair_by_mode(double r, double eps, double sigma, double p2, double r_cut, double r_on, int shift,
                                double *V, double *fdivr)
{
    const int mode = shift & 3, pot = shift >> 2;
    if (pot != 0) { orc_pair_generic(pot, r, eps, sigma, p2, r_cut, r_on, mode, V, fdivr); return; }
    if (mode == 2) orc_lj_pair_xplor(r, eps, sigma, r_cut, r_on, V, fdivr);
    else orc_lj_pair(r, eps, sigma, r_cut, mode, V, fdivr);
}

/* ------------------------------------------------------------------ c6 ---- */
/* One pair's contribution to particle i:  F_i += f, U_i += V/2,
 * W_i^{ab} += (1/2) d^a f^b  with d = minimage(R_i - R_j), f = [-(1/r)dV/dr] d. */
static inline void add_pair(const double d[3], double r2, double eps, double sigma, double p2, double r_cut, double r_on,
                            int shift, double *F, double *U, double *W,
                            double band, double *allow)
{
    const double r = sqrt(r2);
    double V, fdivr;
    pair_by_mode(r, eps, sigma, p2, r_cut, r_on, shift, &V, &fdivr);
    const double f[3] = { fdivr * d[0], fdivr * d[1], fdivr * d[2] };
    F[0] += f[0]; F[1] += f[1]; F[2] += f[2];
    *U += 0.5 * V;
    W[0] += 0.5 * d[0] * f[0]; W[1] += 0.5 * d[0] * f[1]; W[2] += 0.5 * d[0] * f[2];
    W[3] += 0.5 * d[1] * f[1]; W[4] += 0.5 * d[1] * f[2]; W[5] += 0.5 * d[2] * f[2];
    /* [reading c6.ii] cutoff-flip allowance: the truncated force jumps at
     * r_cut, so an fp32 implementation may legitimately decide
     * r < r_cut differently for a pair within `band` of the cutoff.  allow[0..2]
     * accumulate what such a pair could change: |f|, |V|/2, |d||f|/2, taken
     * at the cutoff from inside. */
    if (allow && fabs(r - r_cut) <= band) {
        const double rc = nextafter(r_cut, 0.0);
        double Vc, fc;
        pair_by_mode(rc, eps, sigma, p2, r_cut, r_on, shift, &Vc, &fc);
        allow[0] += fabs(fc) * rc;
        allow[1] += 0.5 * fabs(Vc);
        allow[2] += 0.5 * fabs(fc) * rc * rc;
    }
}

/* DEFINITION: sums over all j != i (O(N^2)).  F[N][3], U[N], W[N][6]. */
int orc_compute_lj_brute(const double *pos, const int32_t *type, int64_t N, double L, int ntypes,
                         const double *eps, const double *sigma, const double *rcut, const double *ron, int shift,
                         double *F, double *U, double *W)
{
#pragma omp parallel for schedule(dynamic, 64)
    for (int64_t i = 0; i < N; i++) {
        double Fi[3] = {0, 0, 0}, Ui = 0, Wi[6] = {0, 0, 0, 0, 0, 0};
        for (int64_t j = 0; j < N; j++) {
            if (j == i) continue;
            double d[3];
            const double r2 = dist2(pos, i, j, L, d);
            const int p = type[i] * ntypes + type[j];
            if (r2 < rcut[p] * rcut[p]) add_pair(d, r2, eps[p], sigma[p], g_p2[p], rcut[p], ron ? ron[p] : rcut[p], shift, Fi, &Ui, Wi, 0.0, NULL);
        }
        memcpy(F + 3 * i, Fi, sizeof Fi); U[i] = Ui; memcpy(W + 6 * i, Wi, sizeof Wi);
    }
    return ORC_OK;
}

/* Sampled definition for full-size spot checks: rows sample[0..S) only. */
int orc_compute_lj_brute_sample(const double *pos, const int32_t *type, int64_t N, double L, int ntypes,
                                const double *eps, const double *sigma, const double *rcut, const double *ron, int shift,
                                const int64_t *sample, int64_t S, double band,
                                double *F, double *U, double *W, double *allow)
{
#pragma omp parallel for schedule(dynamic, 4)
    for (int64_t k = 0; k < S; k++) {
        const int64_t i = sample[k];
        double Fi[3] = {0, 0, 0}, Ui = 0, Wi[6] = {0, 0, 0, 0, 0, 0}, al[3] = {0, 0, 0};
        for (int64_t j = 0; j < N; j++) {
            if (j == i) continue;
            double d[3];
            const double r2 = dist2(pos, i, j, L, d);
            const int p = type[i] * ntypes + type[j];
            const double rc = rcut[p] + band;
            if (r2 < rc * rc) add_pair(d, r2, eps[p], sigma[p], g_p2[p], rcut[p], ron ? ron[p] : rcut[p], shift, Fi, &Ui, Wi, band, al);
        }
        memcpy(F + 3 * k, Fi, sizeof Fi); U[k] = Ui; memcpy(W + 6 * k, Wi, sizeof Wi);
        if (allow) memcpy(allow + 3 * k, al, sizeof al);
    }
    return ORC_OK;
}

/* The method's way: the same sums restricted to the listed
 * neighbors, each tested against its type pair's r_cut.  allow[N][3] (nullable)
 * receives the cutoff-flip allowances for pairs within `band` of r_cut. */
int orc_compute_lj_nlist(const double *pos, const int32_t *type, int64_t N, double L, int ntypes,
                         const double *eps, const double *sigma, const double *rcut, const double *ron, int shift,
                         const int32_t *count, const int64_t *row_start, const int32_t *nbr,
                         double band, double *F, double *U, double *W, double *allow)
{
#pragma omp parallel for schedule(dynamic, 64)
    for (int64_t i = 0; i < N; i++) {
        double Fi[3] = {0, 0, 0}, Ui = 0, Wi[6] = {0, 0, 0, 0, 0, 0}, al[3] = {0, 0, 0};
        for (int32_t k = 0; k < count[i]; k++) {
            const int64_t j = nbr[row_start[i] + k];
            double d[3];
            const double r2 = dist2(pos, i, j, L, d);
            const int p = type[i] * ntypes + type[j];
            /* add_pair() itself applies r < r_cut; pairs just outside are
             * visited only so that their allowance is recorded. */
            const double rc = rcut[p] + band;
            if (r2 < rc * rc) add_pair(d, r2, eps[p], sigma[p], g_p2[p], rcut[p], ron ? ron[p] : rcut[p], shift, Fi, &Ui, Wi, band, al);
        }
        memcpy(F + 3 * i, Fi, sizeof Fi); U[i] = Ui; memcpy(W + 6 * i, Wi, sizeof Wi);
        if (allow) memcpy(allow + 3 * i, al, sizeof al);
    }
    return ORC_OK;
}

/* NEXT-3: per-particle mass ("HOOMD version 0.8.1 allows a mass ... to be specified for each
 * particle"; the base path has m = 1, reading c7).  The table is test-infrastructure state: orc_set_mass(m, N)
 * before a call, orc_set_mass(NULL, 0) for m = 1, in which case every expression below is the m = 1 one. */
static const double *g_mass = NULL;
void orc_set_mass(const double *mass, int64_t N) { (void)N; g_mass = mass; }

/* ------------------------------------------------------------------ c7 ---- */
/* Velocity Verlet, first half ([reading c7] m = 1):
 *   v' = v + (dt/2) F(t);  x(t+dt) = x + dt v';
 * then wrap each axis into [-L/2, L/2), image -/+ 1 per crossing. */
void orc_nve_step1(double *pos, double *vel, const double *F, int32_t *image, int64_t N, double L, double dt)
{
    for (int64_t k = 0; k < 3 * N; k++) {
        if (g_mass) vel[k] = vel[k] + 0.5 * dt * F[k] / g_mass[k / 3];
        else vel[k] = vel[k] + 0.5 * dt * F[k];
        double x = pos[k] + dt * vel[k];
        if (x >= 0.5 * L) { x -= L; image[k] += 1; }
        else if (x < -0.5 * L) { x += L; image[k] -= 1; }
        pos[k] = x;
    }
}

/* second half: v(t+dt) = v' + (dt/2) F(t+dt). */
void orc_nve_step2(double *vel, const double *F, int64_t N, double dt)
{
    if (g_mass) { for (int64_t k = 0; k < 3 * N; k++) vel[k] = vel[k] + 0.5 * dt * F[k] / g_mass[k / 3]; return; }
    for (int64_t k = 0; k < 3 * N; k++) vel[k] = vel[k] + 0.5 * dt * F[k];
}

/* ------------------------------------------------------------------ c9 ---- */
/* out[12] = K, U, W[6], P, px, py, pz with K = (1/2) sum v^2 (m = 1),
 * P = (2K + tr W) / (3 L^3)  (PAPER.md:330 lists K, E, P as logged). */
void orc_thermo(const double *vel, const double *U, const double *W, int64_t N, double L, double *out)
{
    memset(out, 0, 12 * sizeof(double));
    for (int64_t i = 0; i < N; i++) {
        const double mi = g_mass ? g_mass[i] : 1.0;
        for (int a = 0; a < 3; a++) {
            out[0] += 0.5 * mi * vel[3 * i + a] * vel[3 * i + a];
            out[9 + a] += mi * vel[3 * i + a];
        }
        out[1] += U[i];
        for (int a = 0; a < 6; a++) out[2 + a] += W[6 * i + a];
    }
    out[8] = (2.0 * out[0] + out[2] + out[5] + out[7]) / (3.0 * L * L * L);
}

/* ------------------------------------------------------------------ c8 ---- */
/* Hilbert index of a point on the 2^B grid, B bits per axis (Skilling,
 * "Programming the Hilbert curve", AIP Conf. Proc. 707 (2004): AxestoTranspose,
 * then the transposed bits are interleaved, X[0] most significant).
 * [reading c8] The paper names only "SFCPACK sort"; the
 * curve, B = 8 and the tie-break are this build's readings. */
uint32_t orc_hilbert_key(uint32_t ix, uint32_t iy, uint32_t iz, int B)
{
    uint32_t X[3] = { ix, iy, iz };
    const uint32_t M = 1u << (B - 1);
    uint32_t P, Q, t;
    for (Q = M; Q > 1; Q >>= 1) {              /* inverse undo */
        P = Q - 1;
        for (int i = 0; i < 3; i++) {
            if (X[i] & Q) X[0] ^= P;           /* invert */
            else { t = (X[0] ^ X[i]) & P; X[0] ^= t; X[i] ^= t; } /* exchange */
        }
    }
    for (int i = 1; i < 3; i++) X[i] ^= X[i - 1];   /* Gray encode */
    t = 0;
    for (Q = M; Q > 1; Q >>= 1) if (X[2] & Q) t ^= Q - 1;
    for (int i = 0; i < 3; i++) X[i] ^= t;
    uint32_t key = 0;
    for (int b = B - 1; b >= 0; b--)
        for (int i = 0; i < 3; i++) key = (key << 1) | ((X[i] >> b) & 1u);
    return key;
}

/* key_i from the position: grid coordinate floor((x - b) 2^B / L) per axis,
 * evaluated -- like the cell index, and for the same reason -- in binary32
 * without contraction, wrapped into 0 .. 2^B-1. */
void orc_sfc_keys(const float *pos, int64_t N, float L, int B, uint32_t *key)
{
    const float b = -0.5f * L;
    const int G = 1 << B;
    const float s = (float)G / L;
    for (int64_t i = 0; i < N; i++) {
        uint32_t g[3];
        for (int a = 0; a < 3; a++) {
            volatile float r = pos[3 * i + a] - b;
            volatile float u = r * s;
            int ga = (int)floorf(u);
            if (ga >= G) ga -= G;
            if (ga < 0) ga += G;
            g[a] = (uint32_t)ga;
        }
        key[i] = orc_hilbert_key(g[0], g[1], g[2], B);
    }
}

/* New order: stable sort by (key, current index).  perm[k] = old index of the
 * particle that moves to position k.  Insertion into counting buckets keeps it
 * obviously stable. */
int orc_sort_perm(const uint32_t *key, int64_t N, int B, int64_t *perm)
{
    const int64_t nk = (int64_t)1 << (3 * B);
    int64_t *start = (int64_t *)calloc((size_t)nk + 1, sizeof(int64_t));
    if (!start) return ORC_ENOMEM;
    for (int64_t i = 0; i < N; i++) start[key[i] + 1]++;
    for (int64_t k = 0; k < nk; k++) start[k + 1] += start[k];
    for (int64_t i = 0; i < N; i++) perm[start[key[i]]++] = i;
    free(start);
    return ORC_OK;
}

/* ------------------------------------------------------ the whole loop ---- */
/* nsteps of NVE with the list rebuilt on buffer exceedance; used for the
 * trajectory parity case, the conservation pins and the timed CPU baseline.
 * State arrays are updated in place.  F, U, W hold F(t), U_i, W_i on entry if
 * have_forces != 0 (else they are computed first) and on return.
 * log_KU (nullable) [nsteps+1][2] receives K and U at every step incl. step 0.
 * stats[0] = number of list builds, stats[1] = max list length seen.
 * Uses its own fp64 binning (any self-consistent binning with cell width >=
 * r_max yields the exact set -- pinned against orc_nlist_brute). */
int orc_run_nve(double *pos, double *vel, int32_t *image, const int32_t *type, int64_t N, double L,
                int ntypes, const double *eps, const double *sigma, const double *rcut, const double *ron, int shift,
                double r_buff, double dt, int64_t nsteps, int have_forces,
                double *F, double *U, double *W, double *log_KU, int64_t *stats)
{
    double r_cut_max = 0.0;
    for (int p = 0; p < ntypes * ntypes; p++) if (rcut[p] > r_cut_max) r_cut_max = rcut[p];
    const double r_max = r_cut_max + r_buff;
    const int m = orc_cell_dim(L, r_max);
    if (m < 3) return ORC_EBOX;
    const int64_t nc = (int64_t)m * m * m;
    int32_t *cell = (int32_t *)malloc((size_t)N * sizeof(int32_t));
    int64_t *cell_start = (int64_t *)malloc((size_t)(nc + 1) * sizeof(int64_t));
    int32_t *members = (int32_t *)malloc((size_t)N * sizeof(int32_t));
    int32_t *count = (int32_t *)malloc((size_t)N * sizeof(int32_t));
    int64_t *row_start = (int64_t *)malloc((size_t)(N + 1) * sizeof(int64_t));
    double *pos_build = (double *)malloc((size_t)3 * N * sizeof(double));
    int32_t *nbr = NULL;
    int64_t cap = 0, builds = 0, maxlen = 0;
    int rc = ORC_OK, need_build = 1;
    if (!cell || !cell_start || !members || !count || !row_start || !pos_build) { rc = ORC_ENOMEM; goto done; }

    for (int64_t step = 0; step <= nsteps; step++) {
        if (step > 0) {
            orc_nve_step1(pos, vel, F, image, N, L, dt);
            const double half = 0.5 * r_buff;
            if (!need_build && orc_max_disp2(pos, pos_build, N, L) > half * half) need_build = 1;
        }
        if (step > 0 || !have_forces) {
            if (need_build) {
                orc_cell_index_f64(pos, N, L, m, cell, NULL);
                orc_build_cells(cell, N, m, cell_start, members);
                rc = orc_nlist_cells(pos, N, L, r_max, m, cell, cell_start, members, count, NULL, NULL);
                if (rc) goto done;
                row_start[0] = 0;
                for (int64_t i = 0; i < N; i++) {
                    row_start[i + 1] = row_start[i] + count[i];
                    if (count[i] > maxlen) maxlen = count[i];
                }
                if (row_start[N] > cap) {
                    free(nbr);
                    cap = row_start[N] + row_start[N] / 8 + 16;
                    nbr = (int32_t *)malloc((size_t)cap * sizeof(int32_t));
                    if (!nbr) { rc = ORC_ENOMEM; goto done; }
                }
                orc_nlist_cells(pos, N, L, r_max, m, cell, cell_start, members, count, row_start, nbr);
                memcpy(pos_build, pos, (size_t)3 * N * sizeof(double));
                need_build = 0;
                builds++;
            }
            orc_compute_lj_nlist(pos, type, N, L, ntypes, eps, sigma, rcut, ron, shift,
                                 count, row_start, nbr, 0.0, F, U, W, NULL);
        }
        if (step > 0) orc_nve_step2(vel, F, N, dt);
        if (log_KU) {
            double K = 0.0, Ut = 0.0;
            for (int64_t k = 0; k < 3 * N; k++) K += 0.5 * (g_mass ? g_mass[k / 3] : 1.0) * vel[k] * vel[k];
            for (int64_t i = 0; i < N; i++) Ut += U[i];
            log_KU[2 * step] = K; log_KU[2 * step + 1] = Ut;
        }
    }
    if (stats) { stats[0] = builds; stats[1] = maxlen; }
done:
    free(cell); free(cell_start); free(members); free(count); free(row_start); free(pos_build); free(nbr);
    return rc;
}

/* ------------------------------------------------ NEXT-2: thermostats ---- */
/* The paper names a Nose-Hoover NVT integrator with a time constant ("The time constants for
 * NVT and NPT are all set to 1.0") and a Langevin / Brownian-dynamics integrator that needs parallel random
 * numbers, and prints no equation for either.  Readings (DESIGN.md n1, n2):
 *
 * [n1] Nose-Hoover: dv/dt = F/m - xi v,  dxi/dt = (T_k / T - 1) / tau^2,  deta/dt = xi,
 *      T_k = 2 K / g with g = 3 N - 3 degrees of freedom (the total momentum is conserved), m = 1, k_B = 1.
 *      One step, a time-reversible splitting around the force evaluation:
 *        v' = (v + (dt/2) F(t)) / (1 + (dt/2) xi);   x(t+dt) = x + dt v'  (wrap, image flags as in c7)
 *        xi' = xi + (dt / tau^2) (T_k(v') / T - 1);   eta' = eta + (dt/2)(xi + xi')
 *        F(t+dt);   v(t+dt) = v' + (dt/2) (F(t+dt) - xi' v')
 *      Conserved: H' = K + U + g T (tau^2 xi^2 / 2 + eta).
 *
 * [n2] Langevin: dv/dt = F/m - gamma v + R(t), <R_a(t) R_b(t')> = 2 gamma T delta_ab delta(t - t').
 *      One step: the velocity-Verlet step of c7, then the thermostat acts on the new velocity for a whole step,
 *        v <- v (1 - gamma dt) + sqrt(6 gamma T dt) u,   u uniform in (-1, 1) per component (variance 1/3),
 *      so that for free particles <v^2> = T / (1 - gamma dt / 2) per component.
 *      u comes from a counter-based generator: splitmix64 finaliser of (seed, stream = time step number,
 *      index = 3 tag + component), the generator of workloads.py; 23 bits k give u = (2k + 1 - 2^23) / 2^23,
 *      exact in binary32, so a binary32 implementation draws the same numbers. */
static inline uint64_t orc_mix64(uint64_t z)
{
    z ^= z >> 30; z *= 0xBF58476D1CE4E5B9ULL;
    z ^= z >> 27; z *= 0x94D049BB133111EBULL;
    z ^= z >> 31;
    return z;
}

uint64_t orc_counter_u64(uint64_t seed, uint64_t stream, uint64_t index)
{
    const uint64_t G = 0x9E3779B97F4A7C15ULL;
    uint64_t s = orc_mix64(seed + G);
    s = orc_mix64(s + stream * G);
    return orc_mix64(s + (index + 1) * G);
}

double orc_uniform_pm1(uint64_t seed, uint64_t stream, uint64_t index)
{
    const uint64_t k = orc_counter_u64(seed, stream, index) >> 41;          /* 23 bits */
    return ((double)(2 * (int64_t)k + 1) - 8388608.0) / 8388608.0;
}

/* nsteps of thermostatted dynamics with the list rebuilt on buffer exceedance (same loop as orc_run_nve).
 * mode 1: Nose-Hoover, par = tau, state[0..1] = (xi, eta) in and out.
 * mode 2: Langevin, par = gamma, state[0] = number of the first time step (stream of the generator), advanced.
 * log (nullable) [nsteps+1][4]: K, U, xi, eta at every step incl. step 0.  The generator identifies a particle by
 * its index i (the oracle never reorders particles). */
int orc_run_thermostat(int mode, double *pos, double *vel, int32_t *image, const int32_t *type, int64_t N, double L,
                       int ntypes, const double *eps, const double *sigma, const double *rcut, const double *ron, int shift,
                       double r_buff, double dt, int64_t nsteps, double T, double par, uint64_t seed, double *state,
                       int have_forces, double *F, double *U, double *W, double *log, int64_t *stats)
{
    double r_cut_max = 0.0;
    for (int p = 0; p < ntypes * ntypes; p++) if (rcut[p] > r_cut_max) r_cut_max = rcut[p];
    const double r_max = r_cut_max + r_buff;
    const int m = orc_cell_dim(L, r_max);
    if (m < 3) return ORC_EBOX;
    if (mode != 1 && mode != 2) return ORC_ECAP;
    const int64_t nc = (int64_t)m * m * m;
    int32_t *cell = (int32_t *)malloc((size_t)N * sizeof(int32_t));
    int64_t *cell_start = (int64_t *)malloc((size_t)(nc + 1) * sizeof(int64_t));
    int32_t *members = (int32_t *)malloc((size_t)N * sizeof(int32_t));
    int32_t *count = (int32_t *)malloc((size_t)N * sizeof(int32_t));
    int64_t *row_start = (int64_t *)malloc((size_t)(N + 1) * sizeof(int64_t));
    double *pos_build = (double *)malloc((size_t)3 * N * sizeof(double));
    int32_t *nbr = NULL;
    int64_t cap = 0, builds = 0, maxlen = 0;
    int rc = ORC_OK, need_build = 1;
    const double g = 3.0 * (double)N - 3.0;
    double xi = mode == 1 ? state[0] : 0.0, eta = mode == 1 ? state[1] : 0.0;
    uint64_t tstep = mode == 2 ? (uint64_t)state[0] : 0;
    if (!cell || !cell_start || !members || !count || !row_start || !pos_build) { rc = ORC_ENOMEM; goto done; }

    for (int64_t step = 0; step <= nsteps; step++) {
        if (step > 0) {
            if (mode == 1) {
                /* [n1] first half: friction implicit, drift, wrap */
                for (int64_t k = 0; k < 3 * N; k++) {
                    vel[k] = (vel[k] + 0.5 * dt * F[k] / (g_mass ? g_mass[k / 3] : 1.0)) / (1.0 + 0.5 * dt * xi);
                    double x = pos[k] + dt * vel[k];
                    if (x >= 0.5 * L) { x -= L; image[k] += 1; }
                    else if (x < -0.5 * L) { x += L; image[k] -= 1; }
                    pos[k] = x;
                }
                double K = 0.0;
                for (int64_t k = 0; k < 3 * N; k++) K += 0.5 * (g_mass ? g_mass[k / 3] : 1.0) * vel[k] * vel[k];
                const double xi_new = xi + dt / (par * par) * ((2.0 * K / g) / T - 1.0);
                eta += 0.5 * dt * (xi + xi_new);
                xi = xi_new;
            } else {
                orc_nve_step1(pos, vel, F, image, N, L, dt);
            }
            const double half = 0.5 * r_buff;
            if (!need_build && orc_max_disp2(pos, pos_build, N, L) > half * half) need_build = 1;
        }
        if (step > 0 || !have_forces) {
            if (need_build) {
                orc_cell_index_f64(pos, N, L, m, cell, NULL);
                orc_build_cells(cell, N, m, cell_start, members);
                rc = orc_nlist_cells(pos, N, L, r_max, m, cell, cell_start, members, count, NULL, NULL);
                if (rc) goto done;
                row_start[0] = 0;
                for (int64_t i = 0; i < N; i++) {
                    row_start[i + 1] = row_start[i] + count[i];
                    if (count[i] > maxlen) maxlen = count[i];
                }
                if (row_start[N] > cap) {
                    free(nbr);
                    cap = row_start[N] + row_start[N] / 8 + 16;
                    nbr = (int32_t *)malloc((size_t)cap * sizeof(int32_t));
                    if (!nbr) { rc = ORC_ENOMEM; goto done; }
                }
                orc_nlist_cells(pos, N, L, r_max, m, cell, cell_start, members, count, row_start, nbr);
                memcpy(pos_build, pos, (size_t)3 * N * sizeof(double));
                need_build = 0;
                builds++;
            }
            orc_compute_lj_nlist(pos, type, N, L, ntypes, eps, sigma, rcut, ron, shift,
                                 count, row_start, nbr, 0.0, F, U, W, NULL);
        }
        if (step > 0) {
            if (mode == 1) {
                for (int64_t k = 0; k < 3 * N; k++)                                                          /* [n1] second half */
                    vel[k] = vel[k] + 0.5 * dt * (F[k] / (g_mass ? g_mass[k / 3] : 1.0) - xi * vel[k]);
            } else {
                orc_nve_step2(vel, F, N, dt);
                const double c = 1.0 - par * dt, sgm = sqrt(6.0 * par * T * dt);                        /* [n2] */
                if (g_mass) {                                /* friction and noise are forces: both divided by m */
                    for (int64_t k = 0; k < 3 * N; k++)
                        vel[k] = vel[k] * (1.0 - par * dt / g_mass[k / 3]) + sgm / g_mass[k / 3] * orc_uniform_pm1(seed, tstep, (uint64_t)k);
                } else
                for (int64_t k = 0; k < 3 * N; k++) vel[k] = vel[k] * c + sgm * orc_uniform_pm1(seed, tstep, (uint64_t)k);
                tstep++;
            }
        }
        if (log) {
            double K = 0.0, Ut = 0.0;
            for (int64_t k = 0; k < 3 * N; k++) K += 0.5 * (g_mass ? g_mass[k / 3] : 1.0) * vel[k] * vel[k];
            for (int64_t i = 0; i < N; i++) Ut += U[i];
            log[4 * step] = K; log[4 * step + 1] = Ut; log[4 * step + 2] = xi; log[4 * step + 3] = eta;
        }
    }
    if (mode == 1) { state[0] = xi; state[1] = eta; } else state[0] = (double)tstep;
    if (stats) { stats[0] = builds; stats[1] = maxlen; }
done:
    free(cell); free(cell_start); free(members); free(count); free(row_start); free(pos_build); free(nbr);
    return rc;
}

int orc_num_threads(void)
{
#ifdef _OPENMP
    extern int omp_get_max_threads(void);
    return omp_get_max_threads();
#else
    return 1;
#endif
}
