/*
 * nb_oracle.c -- plain, slow, fp64 CPU oracle for the cluster-pair short-range
 * non-bonded step.  TEST INFRASTRUCTURE ONLY: nothing in the product path
 * (paper_2006_09167_b200/) may include, link or call this file.  It shares no
 * code, header, table or constant with the CUDA path.
 *
 * What it states (citations: P:L<n> = /root/reference/PAPER.md line n,
 * S:<sec> = SURVEY.md section, BJ = BASELINE.json):
 *
 *  - Forces/energies/virial: the DEFINITION the cluster-pair method reaches
 *    "up to rounding order": all-pairs minimum-image summation within the
 *    cut-off (BJ:north_star; S:8.3.1).  The paper names the interactions
 *    (Lennard-Jones P:L65, Ewald real-space correction P:L137, reaction-field
 *    P:L249) but prints no formula; the textbook forms of S:8.3.1 / DESIGN.md
 *    readings A1-A9 are written out in oracle_pair() below.
 *  - Lists: the cluster bounding-box predicate and the atom-pair
 *    distance prune predicate evaluated over ALL cluster pairs and
 *    shifts, in the fp32 operation order fixed by reading A12, on the slot
 *    layout exported by the library (layout is an input: reading A20).
 *
 * Pins (tests/test_oracle_*.py, run with -m "not gpu"): closed-form single
 * pairs T1/T2/T3, beta T4, image brute force T5, Newton T6, translation T7,
 * finite differences T8, virial identities T9, pair-count T14, exclusion
 * extremes T15; oracle_forces_split: parts sum to the whole, the local part equals the all-pairs sum of
 * the local atoms alone (tests/test_oracle_split.py).  No function here is "parity unpinned".
 *
 * Build: gcc -O2 -fopenmp -ffp-contract=off -shared -fPIC (oracle/build_oracle.py).
 * -ffp-contract=off matters: the list predicates below must round exactly where
 * written (reading A12).
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef struct {
    int32_t coulomb;     /* 0 = Ewald real space, 1 = reaction field, 2 = none (LJ only: charges ignored) */
    int32_t lj_shift;    /* 1 = potential-shift on LJ energy */
    int32_t coul_shift;  /* 1 = potential-shift on Ewald energy (RF: c_rf always applied, A6) */
    int32_t ntypes;
    double rc;           /* cut-off, nm */
    double beta;         /* Ewald splitting parameter, 1/nm */
    double eps_rf;       /* <= 0 means infinity */
    double epsfac;       /* 1/(4 pi eps0), kJ mol^-1 nm e^-2 (A2: 138.935458) */
    double rc_vdw;       /* twin cut-offs (PME load balancing scales only the electrostatics
                            cut-off): LJ interacts iff r < rc_vdw <= rc, its potential shift is taken at rc_vdw;
                            <= 0 means rc_vdw = rc (single cut-off, reading A19) */
} oracle_params;

#define TWO_OVER_SQRT_PI 1.1283791670955125738961589031215

int oracle_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/* A3: beta from erfc(beta*rc) = rtol, bisection in fp64. */
double oracle_beta_from_rtol(double rc, double rtol)
{
    double lo = 0.0, hi = 1.0;
    while (erfc(hi * rc) > rtol) hi *= 2.0;
    for (int it = 0; it < 200; it++) {
        double mid = 0.5 * (lo + hi);
        if (erfc(mid * rc) > rtol) lo = mid; else hi = mid;
    }
    return 0.5 * (lo + hi);
}

static void rf_constants(const oracle_params* p, double* krf, double* crf)
{
    double rc = p->rc;
    /* A6: eps_r = 1;  k_rf = (eps_rf - 1)/((2 eps_rf + 1) rc^3), -> 1/(2 rc^3) for eps_rf = inf */
    if (p->eps_rf <= 0.0 || isinf(p->eps_rf)) *krf = 1.0 / (2.0 * rc * rc * rc);
    else *krf = (p->eps_rf - 1.0) / ((2.0 * p->eps_rf + 1.0) * rc * rc * rc);
    *crf = 1.0 / rc + (*krf) * rc * rc;
}

/*
 * One pair at distance r < rc (S:8.3.1 table; LJ only below rc_vdw).  qq = q_i*q_j (without epsfac).
 * Outputs: energies V_lj, V_c (kJ/mol) and RADIAL forces F_lj, F_c = -dV/dr
 * (positive = repulsive).  excluded != 0 selects the exclusion-correction rows
 * (A4: no LJ; Ewald: -A erf(beta r)/r without shift (A5); RF: A (k_rf r^2 - c_rf)).
 */
void oracle_pair(const oracle_params* p, double r, double qq, double c6, double c12, int excluded,
                 double* V_lj, double* V_c, double* F_lj, double* F_c)
{
    double A = p->epsfac * qq;
    double rc = p->rc;
    double rcv = p->rc_vdw > 0.0 ? p->rc_vdw : rc;     /* LJ cut-off (twin cut-offs), strict like A7 */
    *V_lj = 0.0; *F_lj = 0.0;
    if (!excluded && r * r < rcv * rcv) {
        double r2 = r * r, r6 = r2 * r2 * r2, r12 = r6 * r6;
        *V_lj = c12 / r12 - c6 / r6;
        if (p->lj_shift) {
            double rc6 = rcv * rcv * rcv * rcv * rcv * rcv;
            *V_lj -= c12 / (rc6 * rc6) - c6 / rc6;
        }
        *F_lj = 12.0 * c12 / (r12 * r) - 6.0 * c6 / (r6 * r);
    }
    if (p->coulomb == 2) {
        *V_c = 0.0;
        *F_c = 0.0;
    } else if (p->coulomb == 0) {
        double b = p->beta;
        double g = TWO_OVER_SQRT_PI * b * exp(-b * b * r * r);
        if (!excluded) {
            *V_c = A * erfc(b * r) / r;
            if (p->coul_shift) *V_c -= A * erfc(b * rc) / rc;
            *F_c = A * (erfc(b * r) / (r * r) + g / r);
        } else {
            *V_c = -A * erf(b * r) / r;
            *F_c = -A * (erf(b * r) / (r * r) - g / r);
        }
    } else {
        double krf, crf;
        rf_constants(p, &krf, &crf);
        if (!excluded) {
            *V_c = A * (1.0 / r + krf * r * r - crf);
            *F_c = A * (1.0 / (r * r) - 2.0 * krf * r);
        } else {
            *V_c = A * (krf * r * r - crf);
            *F_c = -2.0 * A * krf * r;
        }
    }
}

static int is_excluded(const int32_t* excl_off, const int32_t* excl_idx, int i, int j)
{
    for (int k = excl_off[i]; k < excl_off[i + 1]; k++)
        if (excl_idx[k] == j) return 1;
    return 0;
}

typedef struct {
    double* f;        /* [n*3] */
    double E[2];      /* E_lj, E_coul */
    double vir[9];
    long long npairs[2]; /* within rc: non-excluded, excluded */
} accum;

/* Adds the contribution of the pair (i,j) with separation vector d = x_i - x_j (+image). */
static inline void add_pair(const oracle_params* p, const double* q, const int32_t* type, const float* lj,
                            const int32_t* excl_off, const int32_t* excl_idx, int i, int j, const double d[3],
                            accum* a)
{
    double r2 = d[0] * d[0] + d[1] * d[1] + d[2] * d[2];
    if (r2 >= p->rc * p->rc) return;            /* A7: interact iff r^2 < rc^2 (strict) */
    int ex = is_excluded(excl_off, excl_idx, i, j);
    double r = sqrt(r2);
    const float* t = lj + 2 * ((size_t)type[i] * p->ntypes + type[j]);
    double Vlj, Vc, Flj, Fc;
    oracle_pair(p, r, q[i] * q[j], (double)t[0], (double)t[1], ex, &Vlj, &Vc, &Flj, &Fc);
    double F = Flj + Fc;
    for (int k = 0; k < 3; k++) {
        double Fk = F * d[k] / r;
        a->f[3 * i + k] += Fk;
        a->f[3 * j + k] -= Fk;
        for (int l = 0; l < 3; l++) a->vir[3 * l + k] -= 0.5 * d[l] * Fk;   /* A8: Xi = -1/2 sum d (x) F */
    }
    a->E[0] += Vlj;
    a->E[1] += Vc;
    a->npairs[ex ? 1 : 0]++;
}

static void min_image(double d[3], const double* box)
{
    for (int k = 0; k < 3; k++) d[k] -= box[k] * nearbyint(d[k] / box[k]);
}

static void reduce_accum(int n, int nt, accum* part, double* f, double* E, double* vir, long long* npairs)
{
    memset(f, 0, sizeof(double) * 3 * (size_t)n);
    E[0] = E[1] = 0.0;
    for (int k = 0; k < 9; k++) vir[k] = 0.0;
    npairs[0] = npairs[1] = 0;
    for (int t = 0; t < nt; t++) {
        for (size_t k = 0; k < 3 * (size_t)n; k++) f[k] += part[t].f[k];
        E[0] += part[t].E[0]; E[1] += part[t].E[1];
        for (int k = 0; k < 9; k++) vir[k] += part[t].vir[k];
        npairs[0] += part[t].npairs[0]; npairs[1] += part[t].npairs[1];
        free(part[t].f);
    }
    free(part);
}

static accum* alloc_accum(int n, int nt)
{
    accum* part = (accum*)calloc((size_t)nt, sizeof(accum));
    for (int t = 0; t < nt; t++) part[t].f = (double*)calloc(3 * (size_t)n, sizeof(double));
    return part;
}

/*
 * THE DEFINITION (S:8.3.1, BJ:north_star): for i<j, minimum image, cut-off, exclusion,
 * pair formulas.  x is fp64 (callers promote the fp32 inputs exactly).
 */
int oracle_forces_allpairs(int n, const double* x, const double* q, const int32_t* type, const double* box,
                           const float* lj, const int32_t* excl_off, const int32_t* excl_idx,
                           const oracle_params* p, double* f, double* E, double* vir, long long* npairs)
{
    int nt = oracle_num_threads();
    accum* part = alloc_accum(n, nt);
#pragma omp parallel num_threads(nt)
    {
#ifdef _OPENMP
        accum* a = &part[omp_get_thread_num()];
#else
        accum* a = &part[0];
#endif
#pragma omp for schedule(dynamic, 16)
        for (int i = 0; i < n; i++) {
            for (int j = i + 1; j < n; j++) {
                double d[3] = { x[3 * i] - x[3 * j], x[3 * i + 1] - x[3 * j + 1], x[3 * i + 2] - x[3 * j + 2] };
                min_image(d, box);
                add_pair(p, q, type, lj, excl_off, excl_idx, i, j, d, a);
            }
        }
    }
    reduce_accum(n, nt, part, f, E, vir, npairs);
    return 0;
}

/*
 * Local / non-local split (with domain decomposition "non-bonded work [is split] into two kernels: one for
 * local-only interactions and one for interactions that involve non-local particles"; reading A25): atoms
 * [0, nlocal) are the domain's local (home) atoms, atoms [nlocal, n) its non-local (halo) atoms.  The same double
 * loop as oracle_forces_allpairs restricted to   which = 1: pairs with BOTH atoms local;
 * which = 2: pairs with AT LEAST ONE non-local atom;   which = 0: every pair.  (Which non-local/non-local pairs a
 * rank of a decomposed run owns is a domain-decomposition rule, out of scope: here every pair of the system belongs
 * to exactly one of the two parts, so part 1 + part 2 = the whole.)
 */
int oracle_forces_split(int n, int nlocal, int which, const double* x, const double* q, const int32_t* type,
                        const double* box, const float* lj, const int32_t* excl_off, const int32_t* excl_idx,
                        const oracle_params* p, double* f, double* E, double* vir, long long* npairs)
{
    accum* part = alloc_accum(n, 1);
    for (int i = 0; i < n; i++) {
        for (int j = i + 1; j < n; j++) {
            int both_local = i < nlocal && j < nlocal;
            if (which == 1 && !both_local) continue;
            if (which == 2 && both_local) continue;
            double d[3] = { x[3 * i] - x[3 * j], x[3 * i + 1] - x[3 * j + 1], x[3 * i + 2] - x[3 * j + 2] };
            min_image(d, box);
            add_pair(p, q, type, lj, excl_off, excl_idx, i, j, d, &part[0]);
        }
    }
    reduce_accum(n, 1, part, f, E, vir, npairs);
    return 0;
}

/*
 * Brute force over periodic images (pin T5): every image n in {-1,0,1}^3 of every
 * pair i<j with r < rc contributes; no minimum-image convention is used.
 */
int oracle_forces_images(int n, const double* x, const double* q, const int32_t* type, const double* box,
                         const float* lj, const int32_t* excl_off, const int32_t* excl_idx,
                         const oracle_params* p, double* f, double* E, double* vir, long long* npairs)
{
    accum* part = alloc_accum(n, 1);
    for (int i = 0; i < n; i++)
        for (int j = i + 1; j < n; j++)
            for (int nx = -1; nx <= 1; nx++)
                for (int ny = -1; ny <= 1; ny++)
                    for (int nz = -1; nz <= 1; nz++) {
                        double d[3] = { x[3 * i] - x[3 * j] + nx * box[0], x[3 * i + 1] - x[3 * j + 1] + ny * box[1],
                                        x[3 * i + 2] - x[3 * j + 2] + nz * box[2] };
                        add_pair(p, q, type, lj, excl_off, excl_idx, i, j, d, &part[0]);
                    }
    reduce_accum(n, 1, part, f, E, vir, npairs);
    return 0;
}

/*
 * Same sum as oracle_forces_allpairs with a plain linked-cell candidate loop (cell
 * side >= rc, no clusters) -- S:8.4 "oracle_cells": used where O(N^2) is a strawman
 * (configs 3-4) and as the timed CPU baseline.  Returns -1 if the box holds fewer
 * than 3 cells along some axis (then use all-pairs).
 */
int oracle_forces_cells(int n, const double* x, const double* q, const int32_t* type, const double* box,
                        const float* lj, const int32_t* excl_off, const int32_t* excl_idx,
                        const oracle_params* p, double* f, double* E, double* vir, long long* npairs)
{
    int nc[3];
    for (int k = 0; k < 3; k++) {
        nc[k] = (int)floor(box[k] / p->rc);
        if (nc[k] < 3) return -1;
    }
    size_t ncell = (size_t)nc[0] * nc[1] * nc[2];
    int* head = (int*)malloc(sizeof(int) * (ncell + 1));
    int* cell_of = (int*)malloc(sizeof(int) * (size_t)n);
    int* order = (int*)malloc(sizeof(int) * (size_t)n);
    memset(head, 0, sizeof(int) * (ncell + 1));
    for (int i = 0; i < n; i++) {
        int c[3];
        for (int k = 0; k < 3; k++) {
            double w = x[3 * i + k] - box[k] * floor(x[3 * i + k] / box[k]);
            c[k] = (int)(w / box[k] * nc[k]);
            if (c[k] >= nc[k]) c[k] = nc[k] - 1;
            if (c[k] < 0) c[k] = 0;
        }
        cell_of[i] = (c[0] * nc[1] + c[1]) * nc[2] + c[2];
        head[cell_of[i] + 1]++;
    }
    for (size_t c = 0; c < ncell; c++) head[c + 1] += head[c];
    int* fill = (int*)malloc(sizeof(int) * ncell);
    for (size_t c = 0; c < ncell; c++) fill[c] = head[c];
    for (int i = 0; i < n; i++) order[fill[cell_of[i]]++] = i;
    free(fill);

    int nt = oracle_num_threads();
    accum* part = alloc_accum(n, nt);
#pragma omp parallel num_threads(nt)
    {
#ifdef _OPENMP
        accum* a = &part[omp_get_thread_num()];
#else
        accum* a = &part[0];
#endif
#pragma omp for schedule(dynamic, 4)
        for (long c = 0; c < (long)ncell; c++) {
            int cz = (int)(c % nc[2]), cy = (int)((c / nc[2]) % nc[1]), cx = (int)(c / ((long)nc[2] * nc[1]));
            for (int ii = head[c]; ii < head[c + 1]; ii++) {
                int i = order[ii];
                for (int ox = -1; ox <= 1; ox++)
                    for (int oy = -1; oy <= 1; oy++)
                        for (int oz = -1; oz <= 1; oz++) {
                            int c2 = (((cx + ox + nc[0]) % nc[0]) * nc[1] + (cy + oy + nc[1]) % nc[1]) * nc[2]
                                     + (cz + oz + nc[2]) % nc[2];
                            for (int jj = head[c2]; jj < head[c2 + 1]; jj++) {
                                int j = order[jj];
                                if (j <= i) continue;   /* each unordered pair once, seen from its lower index */
                                double d[3] = { x[3 * i] - x[3 * j], x[3 * i + 1] - x[3 * j + 1],
                                                x[3 * i + 2] - x[3 * j + 2] };
                                min_image(d, box);
                                add_pair(p, q, type, lj, excl_off, excl_idx, i, j, d, a);
                            }
                        }
            }
        }
    }
    reduce_accum(n, nt, part, f, E, vir, npairs);
    free(head); free(cell_of); free(order);
    return 0;
}

/*
 * Virial through the shift-force identity the kernel uses (A8):
 *   Xi = -1/2 ( sum_i xw_i (x) f_i + sum_s (s L) (x) S_s ),
 * xw = coordinates wrapped into [0,L), s = the integer image vector of the pair as
 * seen from its first atom (d = xw_i + s L - xw_j), S_s = sum of first-atom forces of
 * all pairs evaluated under s.  Pin T9 checks this equals the pair-sum virial.
 */
int oracle_virial_shift_identity(int n, const double* x, const double* q, const int32_t* type,
                                 const double* box, const float* lj, const int32_t* excl_off,
                                 const int32_t* excl_idx, const oracle_params* p, double* vir)
{
    double* xw = (double*)malloc(sizeof(double) * 3 * (size_t)n);
    double* f = (double*)calloc(3 * (size_t)n, sizeof(double));
    double S[27][3];
    memset(S, 0, sizeof(S));
    for (int i = 0; i < n; i++)
        for (int k = 0; k < 3; k++) xw[3 * i + k] = x[3 * i + k] - box[k] * floor(x[3 * i + k] / box[k]);
    for (int i = 0; i < n; i++)
        for (int j = i + 1; j < n; j++) {
            double d[3]; int s[3];
            for (int k = 0; k < 3; k++) {
                double dk = xw[3 * i + k] - xw[3 * j + k];
                s[k] = -(int)nearbyint(dk / box[k]);
                d[k] = dk + s[k] * box[k];
            }
            double r2 = d[0] * d[0] + d[1] * d[1] + d[2] * d[2];
            if (r2 >= p->rc * p->rc) continue;
            int ex = is_excluded(excl_off, excl_idx, i, j);
            double r = sqrt(r2), Vlj, Vc, Flj, Fc;
            const float* t = lj + 2 * ((size_t)type[i] * p->ntypes + type[j]);
            oracle_pair(p, r, q[i] * q[j], (double)t[0], (double)t[1], ex, &Vlj, &Vc, &Flj, &Fc);
            int sid = (s[0] + 1) * 9 + (s[1] + 1) * 3 + (s[2] + 1);
            for (int k = 0; k < 3; k++) {
                double Fk = (Flj + Fc) * d[k] / r;
                f[3 * i + k] += Fk; f[3 * j + k] -= Fk;
                S[sid][k] += Fk;
            }
        }
    for (int k = 0; k < 9; k++) vir[k] = 0.0;
    for (int i = 0; i < n; i++)
        for (int l = 0; l < 3; l++)
            for (int k = 0; k < 3; k++) vir[3 * l + k] -= 0.5 * xw[3 * i + l] * f[3 * i + k];
    for (int sid = 0; sid < 27; sid++) {
        int s[3] = { sid / 9 - 1, (sid / 3) % 3 - 1, sid % 3 - 1 };
        for (int l = 0; l < 3; l++)
            for (int k = 0; k < 3; k++) vir[3 * l + k] -= 0.5 * s[l] * box[l] * S[sid][k];
    }
    free(xw); free(f);
    return 0;
}

/* ------------------------------------------------------------------------------------------
 * Lists (S:8.3.2).  Inputs are the library's exported slot table and wrapped fp32 xq, so the
 * layout (which atom sits in which cluster) is an input and is not re-derived here (A20).
 * Cluster c owns slots [c*C, (c+1)*C); atom_of_slot < 0 marks padding.
 * A shift s = (sx,sy,sz) displaces the FIRST cluster of the triple: d = x_a + s L - x_b.
 * Canonical half (A14): s >lex 0 in (sx,sy,sz) order with any (ci,cj), or s = 0 and cj >= ci.
 * ------------------------------------------------------------------------------------------ */

/* bb over the valid atoms of each cluster (exact in fp32).  nvalid[c] == 0 -> no bb. */
void oracle_cluster_bb(int nclusters, int C, const int32_t* atom_of_slot, const float* xq,
                       float* lo /*[nclusters*3]*/, float* hi, int32_t* nvalid)
{
    for (int c = 0; c < nclusters; c++) {
        nvalid[c] = 0;
        for (int k = 0; k < 3; k++) { lo[3 * c + k] = INFINITY; hi[3 * c + k] = -INFINITY; }
        for (int a = 0; a < C; a++) {
            int s = c * C + a;
            if (atom_of_slot[s] < 0) continue;
            nvalid[c]++;
            for (int k = 0; k < 3; k++) {
                float v = xq[4 * s + k];
                if (v < lo[3 * c + k]) lo[3 * c + k] = v;
                if (v > hi[3 * c + k]) hi[3 * c + k] = v;
            }
        }
    }
}

/* A12: D2_bb in the specified fp32 order. */
static float bb_dist2(const float* lo_i, const float* hi_i, const float* lo_j, const float* hi_j,
                      const int* s, const float* box)
{
    float g[3];
    for (int k = 0; k < 3; k++) {
        float a = fmaf((float)s[k], box[k], lo_i[k]) - hi_j[k];
        float b = lo_j[k] - fmaf((float)s[k], box[k], hi_i[k]);
        float m = a > b ? a : b;
        g[k] = m > 0.0f ? m : 0.0f;
    }
    return fmaf(g[2], g[2], fmaf(g[1], g[1], g[0] * g[0]));
}

/* A12: atom-pair d2 in the specified fp32 order. */
static float atom_dist2(const float* xa, const float* xb, const int* s, const float* box)
{
    float d[3];
    for (int k = 0; k < 3; k++) d[k] = fmaf((float)s[k], box[k], xa[k]) - xb[k];
    return fmaf(d[2], d[2], fmaf(d[1], d[1], d[0] * d[0]));
}

static int canonical(int ci, int cj, const int* s)
{
    if (s[0] != 0) return s[0] > 0;
    if (s[1] != 0) return s[1] > 0;
    if (s[2] != 0) return s[2] > 0;
    return cj >= ci;
}

static int inner_test(int C, const int32_t* atom_of_slot, const float* xq, const float* box, int ci, int cj,
                      const int* s, float rl2)
{
    int diag = (ci == cj && s[0] == 0 && s[1] == 0 && s[2] == 0);
    for (int a = 0; a < C; a++) {
        if (atom_of_slot[ci * C + a] < 0) continue;
        for (int b = 0; b < C; b++) {
            if (atom_of_slot[cj * C + b] < 0) continue;
            if (diag && b <= a) continue;
            if (atom_dist2(xq + 4 * (ci * C + a), xq + 4 * (cj * C + b), s, box) < rl2) return 1;
        }
    }
    return 0;
}

/* pairmask bit a*C+b = valid(a) & valid(b) & !excluded & !(diagonal & b<=a)   (S:8.3.2) */
static uint64_t pair_mask(int C, const int32_t* atom_of_slot, const int32_t* excl_off, const int32_t* excl_idx,
                          int ci, int cj, const int* s)
{
    int diag = (ci == cj && s[0] == 0 && s[1] == 0 && s[2] == 0);
    uint64_t m = 0;
    for (int a = 0; a < C; a++) {
        int ia = atom_of_slot[ci * C + a];
        if (ia < 0) continue;
        for (int b = 0; b < C; b++) {
            int jb = atom_of_slot[cj * C + b];
            if (jb < 0) continue;
            if (diag && b <= a) continue;
            if (ia == jb) continue;
            if (is_excluded(excl_off, excl_idx, ia, jb)) continue;
            m |= (uint64_t)1 << (a * C + b);
        }
    }
    return m;
}

/*
 * Enumerates canonical triples (ci,cj,s) with D2_bb < fl32(rlist_outer^2) whose FIRST OR SECOND
 * cluster lies in [c_begin, c_end) (use [0,nclusters) for the whole list; a sub-range gives the
 * "sampled outputs" check at full size).  For each: inner flag (some atom pair with
 * d2 < fl32(rlist_inner^2)) and pairmask.  Returns the number found; fills at most `cap`.
 * Output order: ci, then cj, then s lexicographic.
 */
long long oracle_lists(int nclusters, int C, const int32_t* atom_of_slot, const float* xq, const float* box,
                       float rlist_outer, float rlist_inner, const int32_t* excl_off, const int32_t* excl_idx,
                       int c_begin, int c_end, long long cap, int32_t* out_ci, int32_t* out_cj,
                       int8_t* out_s /*[cap*3]*/, uint8_t* out_inner, uint64_t* out_mask)
{
    float* lo = (float*)malloc(sizeof(float) * 3 * (size_t)nclusters);
    float* hi = (float*)malloc(sizeof(float) * 3 * (size_t)nclusters);
    int32_t* nv = (int32_t*)malloc(sizeof(int32_t) * (size_t)nclusters);
    oracle_cluster_bb(nclusters, C, atom_of_slot, xq, lo, hi, nv);
    float ro2 = rlist_outer * rlist_outer, ri2 = rlist_inner * rlist_inner;   /* fl32(r*r) */
    long long total = 0;
    long long* cnt = (long long*)calloc((size_t)nclusters + 1, sizeof(long long));
    for (int pass = 0; pass < 2; pass++) {
#pragma omp parallel for schedule(dynamic, 8)
        for (int ci = 0; ci < nclusters; ci++) {
            if (nv[ci] == 0) continue;
            long long k = pass ? cnt[ci] : 0;
            /* first OR second cluster in [c_begin, c_end): all cj for a ci inside the range, else the cj inside it */
            const int ci_in = (ci >= c_begin && ci < c_end);
            for (int cj = ci_in ? 0 : c_begin; cj < (ci_in ? nclusters : (c_end < nclusters ? c_end : nclusters)); cj++) {
                if (nv[cj] == 0) continue;
                for (int sx = -1; sx <= 1; sx++)
                    for (int sy = -1; sy <= 1; sy++)
                        for (int sz = -1; sz <= 1; sz++) {
                            int s[3] = { sx, sy, sz };
                            if (!canonical(ci, cj, s)) continue;
                            if (!(bb_dist2(lo + 3 * ci, hi + 3 * ci, lo + 3 * cj, hi + 3 * cj, s, box) < ro2)) continue;
                            if (pass && k < cap) {
                                out_ci[k] = ci; out_cj[k] = cj;
                                out_s[3 * k] = (int8_t)sx; out_s[3 * k + 1] = (int8_t)sy; out_s[3 * k + 2] = (int8_t)sz;
                                out_inner[k] = (uint8_t)inner_test(C, atom_of_slot, xq, box, ci, cj, s, ri2);
                                out_mask[k] = pair_mask(C, atom_of_slot, excl_off, excl_idx, ci, cj, s);
                            }
                            k++;
                        }
            }
            if (!pass) cnt[ci + 1] = k;
        }
        if (!pass) {
            for (int c = 0; c < nclusters; c++) cnt[c + 1] += cnt[c];
            total = cnt[nclusters];
        }
    }
    free(lo); free(hi); free(nv); free(cnt);
    return total;
}

/*
 * The inner list at SUB-cluster granularity on the j side (DESIGN.md section 5 "compact inner list", reading A22; the
 * paper's "splitting j-clusters" while pruning: the search's cluster pairs are "pruned into" narrower ones).
 * This is the list the force kernel streams, so it gets its own definition, for groups of G consecutive j atoms
 * (G = C/2: half j-clusters, the paper's 8x4 shape; G = 1: single j atoms):
 *
 *   for every canonical triple (ci,cj,s) of S_outer (bb predicate, as in oracle_lists):
 *     - if its pair mask is NOT trivial (some pair of real atoms is excluded, or the triple is the
 *       zero-shift diagonal ci == cj): the WHOLE cluster pair is kept iff inner_test() holds
 *       -> one entry {ci, cj, s, kind 1};
 *     - else, for each group h in 0 .. C/G - 1 of cj (atoms h*G .. h*G + G - 1): the group is kept iff
 *       some real atom of the group is within fl32(rlist_inner^2) of some real atom of ci (A12 order)
 *       -> one entry {ci, (C/G)*cj + h, s, kind 0}     (G = 1: the entry is the j atom's slot).
 *
 * Same enumeration, sub-range rule, return value and output order (ci, cj, s, then kind-0 groups
 * in h order) as oracle_lists.  Pins: tests/test_oracle_lists.py (numpy recomputation on a layout
 * the test makes up, union-of-groups == inner flag of oracle_lists, completeness by k-d tree).
 */
static long long group_lists(int nclusters, int C, int G, const int32_t* atom_of_slot, const float* xq, const float* box,
                             float rlist_outer, float rlist_inner, const int32_t* excl_off, const int32_t* excl_idx,
                             int c_begin, int c_end, long long cap, int32_t* out_ci, int32_t* out_entry,
                             int8_t* out_s /*[cap*3]*/, uint8_t* out_kind)
{
    float* lo = (float*)malloc(sizeof(float) * 3 * (size_t)nclusters);
    float* hi = (float*)malloc(sizeof(float) * 3 * (size_t)nclusters);
    int32_t* nv = (int32_t*)malloc(sizeof(int32_t) * (size_t)nclusters);
    oracle_cluster_bb(nclusters, C, atom_of_slot, xq, lo, hi, nv);
    float ro2 = rlist_outer * rlist_outer, ri2 = rlist_inner * rlist_inner;   /* fl32(r*r) */
    const int H = G, NG = C / G;   /* atoms per group, groups per j-cluster */
    long long total = 0;
    long long* cnt = (long long*)calloc((size_t)nclusters + 1, sizeof(long long));
    for (int pass = 0; pass < 2; pass++) {
#pragma omp parallel for schedule(dynamic, 8)
        for (int ci = 0; ci < nclusters; ci++) {
            if (nv[ci] == 0) continue;
            long long k = pass ? cnt[ci] : 0;
            /* first OR second cluster in [c_begin, c_end): all cj for a ci inside the range, else the cj inside it */
            const int ci_in = (ci >= c_begin && ci < c_end);
            for (int cj = ci_in ? 0 : c_begin; cj < (ci_in ? nclusters : (c_end < nclusters ? c_end : nclusters)); cj++) {
                if (nv[cj] == 0) continue;
                for (int sx = -1; sx <= 1; sx++)
                    for (int sy = -1; sy <= 1; sy++)
                        for (int sz = -1; sz <= 1; sz++) {
                            int s[3] = { sx, sy, sz };
                            if (!canonical(ci, cj, s)) continue;
                            if (!(bb_dist2(lo + 3 * ci, hi + 3 * ci, lo + 3 * cj, hi + 3 * cj, s, box) < ro2)) continue;
                            /* trivial mask: every pair of real atoms interacts */
                            uint64_t m = pair_mask(C, atom_of_slot, excl_off, excl_idx, ci, cj, s), full = 0;
                            for (int a = 0; a < C; a++)
                                for (int b = 0; b < C; b++)
                                    if (atom_of_slot[ci * C + a] >= 0 && atom_of_slot[cj * C + b] >= 0)
                                        full |= (uint64_t)1 << (a * C + b);
                            if (m != full) {
                                if (inner_test(C, atom_of_slot, xq, box, ci, cj, s, ri2)) {
                                    if (pass && k < cap) {
                                        out_ci[k] = ci; out_entry[k] = cj; out_kind[k] = 1;
                                        out_s[3 * k] = (int8_t)sx; out_s[3 * k + 1] = (int8_t)sy; out_s[3 * k + 2] = (int8_t)sz;
                                    }
                                    k++;
                                }
                                continue;
                            }
                            for (int h = 0; h < NG; h++) {
                                int keep = 0;
                                for (int a = 0; a < C && !keep; a++) {
                                    if (atom_of_slot[ci * C + a] < 0) continue;
                                    for (int b = h * H; b < (h + 1) * H; b++) {
                                        if (atom_of_slot[cj * C + b] < 0) continue;
                                        if (atom_dist2(xq + 4 * (ci * C + a), xq + 4 * (cj * C + b), s, box) < ri2) { keep = 1; break; }
                                    }
                                }
                                if (!keep) continue;
                                if (pass && k < cap) {
                                    out_ci[k] = ci; out_entry[k] = NG * cj + h; out_kind[k] = 0;
                                    out_s[3 * k] = (int8_t)sx; out_s[3 * k + 1] = (int8_t)sy; out_s[3 * k + 2] = (int8_t)sz;
                                }
                                k++;
                            }
                        }
            }
            if (!pass) cnt[ci + 1] = k;
        }
        if (!pass) {
            for (int c = 0; c < nclusters; c++) cnt[c + 1] += cnt[c];
            total = cnt[nclusters];
        }
    }
    free(lo); free(hi); free(nv); free(cnt);
    return total;
}

/* G = C/2: half j-clusters (entry = 2*cj + half). */
long long oracle_half_lists(int nclusters, int C, const int32_t* atom_of_slot, const float* xq, const float* box,
                            float rlist_outer, float rlist_inner, const int32_t* excl_off, const int32_t* excl_idx,
                            int c_begin, int c_end, long long cap, int32_t* out_ci, int32_t* out_entry,
                            int8_t* out_s /*[cap*3]*/, uint8_t* out_kind)
{
    return group_lists(nclusters, C, C / 2, atom_of_slot, xq, box, rlist_outer, rlist_inner, excl_off, excl_idx, c_begin, c_end, cap,
                       out_ci, out_entry, out_s, out_kind);
}

/* G = 1: single j atoms (entry = the j atom's slot index cj*C + b): a j atom of an unmasked cluster pair is listed for
 * the i-cluster iff it is within rlist_inner of one of its real atoms. */
long long oracle_atom_lists(int nclusters, int C, const int32_t* atom_of_slot, const float* xq, const float* box,
                            float rlist_outer, float rlist_inner, const int32_t* excl_off, const int32_t* excl_idx,
                            int c_begin, int c_end, long long cap, int32_t* out_ci, int32_t* out_entry,
                            int8_t* out_s /*[cap*3]*/, uint8_t* out_kind)
{
    return group_lists(nclusters, C, 1, atom_of_slot, xq, box, rlist_outer, rlist_inner, excl_off, excl_idx, c_begin, c_end, cap,
                       out_ci, out_entry, out_s, out_kind);
}
