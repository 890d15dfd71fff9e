/*
 * md_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * A plain, slow, fp64 CPU statement of what the neighbor-list MD hot path of
 * "JAX, M.D." (arXiv 1912.04232; /root/reference/PAPER.md) computes, written
 * from the paper's definitions.  It shares no code, header, table or helper
 * with the CUDA path (paper_1912_04232_b200/csrc) and neither includes the
 * other.  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * --impl reference legs may load it.
 *
 * What each function follows (PAPER.md line, section):
 *   orc_neighbor_list   L84 §3.2.3 "pairs (i,j) such that ||r_i - r_j|| < sigma";
 *                       dense N x N_nbrs rows L74 §3.2.1; static capacity L47 §3.1
 *   orc_cell_list       L84 "places them into cells where each cell has size sigma"
 *   orc_energy_force    L78 §3.2.2  U = 1/2 sum_{i!=j} u(r_i - r_j),  m r'' = -grad U;
 *                       L104 §3.3.2 Lennard-Jones, soft-sphere; force = -grad U;
 *                       L301 App. A  sigma_AB = (sigma_A + sigma_B)/2
 *   orc_needs_rebuild   L49 §3.1 "whenever a particle moves by more than the halo"
 *   orc_nve_run         L100 §3.3.1 NVE (init, update);  L72 shift function mu
 *   displacement        L72 §3.2.1 "displacement between a particle and the
 *                       nearest image of the second particle"
 *   (the "next" rows)
 *   kinds 2, 3, 4, 5    L104 Morse [75], Buckingham-type [71-73], per-species LJ tables (L298-L305),
 *                       BKS-type exp-6 + damped shifted-force Coulomb per species pair
 *   orc_fire_run        L100 "Fire Descent [68]", used at L322 (Bitzek et al.'s algorithm)
 *   orc_brownian_run    L100 "Brownian" (Euler-Maruyama; kT = 0: "Gradient Descent")
 *   orc_langevin_run    L100 "Langevin" (BAOAB splitting)
 *   orc_nose_hoover_run L100 "Nose-Hoover [67]" (chains of 1..8 thermostats, MTK splitting)
 *   orc_normals         the counter-based normal generator both sides implement
 *   orc_flock_*         App. B: boids energies eqs. 3-10, forward Euler eqs. 4-5;
 *                       obstacles eq. 11 (L411-L418), predators eqs. 12-13 (L420-L438)
 * Readings of everything the paper leaves open (strict <, half-skin, truncated
 * and shifted LJ, wrap convention, rounding of the inclusion predicate) are
 * SURVEY.md §8c A1-A18, restated in DESIGN.md §3.
 *
 * Parity pins (tests/test_oracle_pins.py): every function here is pinned to
 * something other than itself -- FCC shell counts and lattice sums, two-body
 * closed forms, finite differences, Newton's third law, translation
 * invariance, scipy's periodic cKDTree, NVE invariants, the harmonic
 * oscillator's exact discrete frequency; for the "next" rows: closed-form two-body
 * values and gradients of every potential, FIRE's schedule in closed form and its
 * reduction to velocity Verlet, generator moments, free diffusion, exact friction
 * decay and stationary variance, Nose-Hoover's conserved quantity at second order
 * (single thermostat and chains), its decoupled limit, time reversibility and the second
 * link's equation of motion, the Madelung constant of rock salt for the damped
 * shifted-force Coulomb term, the boids energies on a pair by hand with finite-difference
 * gradients and rotation / translation invariance, the obstacle and predator terms in
 * closed form for one boid / one clump.  The one unpinned thing is a chaotic
 * trajectory beyond ~100 steps ("parity unpinned" by design).
 *
 * Arithmetic: fp64 everywhere, except the canonical inclusion predicate
 * (predicate = 0), which is evaluated in singly-rounded fp32 because it decides
 * an integer (set membership) that the fp32 GPU path must reproduce to the
 * bit.  Build with -ffp-contract=off (no implicit FMA).
 *
 * Positions are double[n*3] (z ignored in 2-D); box is double[3]; diameters
 * double[n]; indices int32.  Rows of a neighbor list are ascending, padded
 * with n.  OpenMP only splits the outer loop over particles; there is no
 * blocking, fusion or reordering beyond the definitions.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define ORC_OK 0
#define ORC_EINVAL (-1)
#define ORC_ENOMEM (-2)

#define KIND_LJ 0
#define KIND_SOFT 1
#define KIND_MORSE 2
#define KIND_BUCK 3
#define KIND_LJ_SPECIES 4
#define KIND_BKS 5

int orc_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

void orc_set_num_threads(int t)
{
#ifdef _OPENMP
    if (t > 0) omp_set_num_threads(t);
#else
    (void)t;
#endif
}

/* ---------------------------------------------------------------- space -- */

/* fp64 nearest-image displacement a - b, one component. */
static double disp64(double a, double b, double L)
{
    double d = a - b;
    return d - L * round(d / L);
}

/* Canonical fp32 nearest-image displacement, one component:
 * every operation singly rounded; the inner subtraction of L is exact. */
static float disp32(float xi, float xj, float L)
{
    float h = L / 2.0f;
    float d = xi - xj;
    if (d > h) {
        float t = xi - L;
        d = t - xj;
    } else if (d < -h) {
        float t = xj - L;
        d = xi - t;
    }
    return d;
}

/* Shift function mu(r, dr) folded into [0, L). */
static double wrap64(double x, double L)
{
    x = x - L * floor(x / L);
    if (x >= L) x = 0.0;
    if (x < 0.0) x = 0.0;
    return x;
}

/* fp32 list radius R = fl(fl32(r_cut) + fl32(skin)). */
static float list_radius32(float r_cut, float skin)
{
    float R = r_cut + skin;
    return R;
}

/* inclusion predicate P(i,j): canonical fp32 (0) or fp64 (1) */
static int within(int predicate, int dim, const double *pi, const double *pj,
                  const double *box, float R32)
{
    if (predicate == 0) {
        float R2 = R32 * R32;
        float dx = disp32((float)pi[0], (float)pj[0], (float)box[0]);
        float dy = disp32((float)pi[1], (float)pj[1], (float)box[1]);
        float r2 = fmaf(dy, dy, dx * dx);
        if (dim == 3) {
            float dz = disp32((float)pi[2], (float)pj[2], (float)box[2]);
            r2 = fmaf(dz, dz, r2);
        }
        return r2 < R2;
    } else {
        double R = (double)R32;
        double r2 = 0.0;
        for (int k = 0; k < dim; ++k) {
            double d = disp64(pi[k], pj[k], box[k]);
            r2 += d * d;
        }
        return r2 < R * R;
    }
}

/* ----------------------------------------------------------- cell list -- */

/* Cells per side n_k = floor(L_k / R), evaluated in fp64. */
static void cells_per_side(int dim, const double *box, float R32, int32_t *nc)
{
    nc[0] = nc[1] = nc[2] = 1;
    for (int k = 0; k < dim; ++k) {
        int v = (int)floor(box[k] / (double)R32);
        nc[k] = v < 1 ? 1 : v;
    }
}

/* Canonical cell coordinate: fp32 product, truncation, clamp. */
static int cell_coord32(double x, double L, int nk)
{
    float inv = (float)nk / (float)L;
    float t = (float)x * inv;
    int c = (int)t;
    if (c > nk - 1) c = nk - 1;
    if (c < 0) c = 0;
    return c;
}

/* The oracle's own binning for its cell-binned search: plain fp64. */
static int cell_coord64(double x, double L, int nk)
{
    int c = (int)floor(x / L * (double)nk);
    if (c > nk - 1) c = nk - 1;
    if (c < 0) c = 0;
    return c;
}

/*
 * orc_cell_list: canonical cell index per particle, and the counting sort by
 * cell with ascending particle ids inside each cell.
 *   ncell[3]   out: cells per side (1 in unused dimensions)
 *   cell_of    out: int32[n] linear cell index (cz*ny + cy)*nx + cx
 *   cell_start out: int32[cells+1] (may be NULL)
 *   members    out: int32[n] particle ids grouped by cell (may be NULL)
 */
int orc_cell_list(int n, int dim, const double *pos, const double *box,
                  float r_cut, float skin, int32_t *ncell, int32_t *cell_of,
                  int32_t *cell_start, int32_t *members)
{
    if (n <= 0 || (dim != 2 && dim != 3)) return ORC_EINVAL;
    float R = list_radius32(r_cut, skin);
    int32_t nc[3];
    cells_per_side(dim, box, R, nc);
    ncell[0] = nc[0]; ncell[1] = nc[1]; ncell[2] = nc[2];
    int64_t cells = (int64_t)nc[0] * nc[1] * nc[2];
    for (int i = 0; i < n; ++i) {
        int c[3] = {0, 0, 0};
        for (int k = 0; k < dim; ++k)
            c[k] = cell_coord32(pos[3 * i + k], box[k], nc[k]);
        cell_of[i] = (c[2] * nc[1] + c[1]) * nc[0] + c[0];
    }
    if (cell_start && members) {
        for (int64_t c = 0; c <= cells; ++c) cell_start[c] = 0;
        for (int i = 0; i < n; ++i) cell_start[cell_of[i] + 1] += 1;
        for (int64_t c = 0; c < cells; ++c) cell_start[c + 1] += cell_start[c];
        int32_t *fill = (int32_t *)calloc((size_t)cells, sizeof(int32_t));
        if (!fill) return ORC_ENOMEM;
        for (int i = 0; i < n; ++i) {   /* ascending i => ascending inside a cell */
            int c = cell_of[i];
            members[cell_start[c] + fill[c]++] = i;
        }
        free(fill);
    }
    return ORC_OK;
}

/* ------------------------------------------------------- neighbor list -- */

static int cmp_i32(const void *a, const void *b)
{
    int32_t x = *(const int32_t *)a, y = *(const int32_t *)b;
    return (x > y) - (x < y);
}

/*
 * orc_neighbor_list: S_i = { j != i : P(i,j) } for every i,
 * as dense rows of `capacity` int32, ascending, padded with n (L74).
 *   predicate 0: canonical fp32 (bit-exact target of the GPU list)
 *             1: fp64 (the definition)
 *   method    0: O(N^2) brute force over all j
 *             1: the oracle's own cell-binned search (fp64 binning into cells of
 *                side >= R, 3^D stencil; any dimension with fewer than 3 cells
 *                scans all of its cells once)
 *   nbr_count  out: TRUE count per particle (may exceed capacity)
 *   status[0]  out: 1 if any count > capacity (rows then hold the first
 *                   `capacity` ascending entries); status[1]: max true count
 */
int orc_neighbor_list(int n, int dim, const double *pos, const double *box,
                      float r_cut, float skin, int capacity, int predicate,
                      int method, int32_t *nbr_idx, int32_t *nbr_count,
                      int32_t *status)
{
    if (n <= 0 || (dim != 2 && dim != 3) || capacity <= 0) return ORC_EINVAL;
    float R = list_radius32(r_cut, skin);
    int32_t nc[3];
    cells_per_side(dim, box, R, nc);
    int64_t cells = (int64_t)nc[0] * nc[1] * nc[2];
    int32_t *cstart = NULL, *cmem = NULL, *cof = NULL;
    if (method == 1) {
        cstart = (int32_t *)calloc((size_t)cells + 1, sizeof(int32_t));
        cmem = (int32_t *)malloc((size_t)n * sizeof(int32_t));
        cof = (int32_t *)malloc((size_t)n * sizeof(int32_t));
        if (!cstart || !cmem || !cof) { free(cstart); free(cmem); free(cof); return ORC_ENOMEM; }
        for (int i = 0; i < n; ++i) {
            int c[3] = {0, 0, 0};
            for (int k = 0; k < dim; ++k)
                c[k] = cell_coord64(pos[3 * i + k], box[k], nc[k]);
            cof[i] = (c[2] * nc[1] + c[1]) * nc[0] + c[0];
            cstart[cof[i] + 1] += 1;
        }
        for (int64_t c = 0; c < cells; ++c) cstart[c + 1] += cstart[c];
        int32_t *fill = (int32_t *)calloc((size_t)cells, sizeof(int32_t));
        if (!fill) { free(cstart); free(cmem); free(cof); return ORC_ENOMEM; }
        for (int i = 0; i < n; ++i) cmem[cstart[cof[i]] + fill[cof[i]]++] = i;
        free(fill);
    }
    int max_count = 0;
    int fail = 0;
#pragma omp parallel
    {
        int cap_tmp = 256;
        int32_t *tmp = (int32_t *)malloc((size_t)cap_tmp * sizeof(int32_t));
        int local_max = 0;
#pragma omp for schedule(dynamic, 64)
        for (int i = 0; i < n; ++i) {
            if (!tmp) { fail = 1; continue; }
            int cnt = 0;
            const double *pi = pos + 3 * (size_t)i;
            if (method == 0) {
                for (int j = 0; j < n; ++j) {
                    if (j == i) continue;
                    if (within(predicate, dim, pi, pos + 3 * (size_t)j, box, R)) {
                        if (cnt == cap_tmp) {
                            cap_tmp *= 2;
                            tmp = (int32_t *)realloc(tmp, (size_t)cap_tmp * sizeof(int32_t));
                            if (!tmp) { fail = 1; break; }
                        }
                        tmp[cnt++] = j;
                    }
                }
            } else {
                int ci[3] = {0, 0, 0}, lo[3] = {0, 0, 0}, hi[3] = {0, 0, 0};
                int c = cof[i];
                ci[0] = c % nc[0]; ci[1] = (c / nc[0]) % nc[1]; ci[2] = c / (nc[0] * nc[1]);
                for (int k = 0; k < 3; ++k) {
                    if (k >= dim) { lo[k] = hi[k] = 0; }
                    else if (nc[k] < 3) { lo[k] = -ci[k]; hi[k] = nc[k] - 1 - ci[k]; }
                    else { lo[k] = -1; hi[k] = 1; }
                }
                for (int oz = lo[2]; oz <= hi[2] && tmp; ++oz)
                for (int oy = lo[1]; oy <= hi[1] && tmp; ++oy)
                for (int ox = lo[0]; ox <= hi[0] && tmp; ++ox) {
                    int cx = (ci[0] + ox + nc[0]) % nc[0];
                    int cy = (ci[1] + oy + nc[1]) % nc[1];
                    int cz = (ci[2] + oz + nc[2]) % nc[2];
                    int cc = (cz * nc[1] + cy) * nc[0] + cx;
                    for (int s = cstart[cc]; s < cstart[cc + 1]; ++s) {
                        int j = cmem[s];
                        if (j == i) continue;
                        if (within(predicate, dim, pi, pos + 3 * (size_t)j, box, R)) {
                            if (cnt == cap_tmp) {
                                cap_tmp *= 2;
                                tmp = (int32_t *)realloc(tmp, (size_t)cap_tmp * sizeof(int32_t));
                                if (!tmp) { fail = 1; break; }
                            }
                            tmp[cnt++] = j;
                        }
                    }
                }
            }
            if (!tmp) continue;
            qsort(tmp, (size_t)cnt, sizeof(int32_t), cmp_i32);
            nbr_count[i] = cnt;
            if (cnt > local_max) local_max = cnt;
            int32_t *row = nbr_idx + (size_t)i * capacity;
            for (int k = 0; k < capacity; ++k) row[k] = k < cnt ? tmp[k] : n;
        }
        free(tmp);
#pragma omp critical
        { if (local_max > max_count) max_count = local_max; }
    }
    free(cstart); free(cmem); free(cof);
    if (fail) return ORC_ENOMEM;
    status[0] = max_count > capacity ? 1 : 0;
    status[1] = max_count;
    return ORC_OK;
}

/*
 * orc_predicate_band: ties the canonical fp32 predicate to the paper's
 * "within sigma".  Over all pairs (brute force, method 0)
 * or all stencil pairs (method 1) it counts the pairs on which the fp32 and
 * fp64 predicates differ, the largest |r64 - R|/R among those, and the smallest
 * |r64 - R| over all pairs examined.
 */
int orc_predicate_band(int n, int dim, const double *pos, const double *box,
                       float r_cut, float skin, int method,
                       int64_t *n_disagree, double *max_rel_band, double *closest)
{
    if (n <= 0 || (dim != 2 && dim != 3)) return ORC_EINVAL;
    float R = list_radius32(r_cut, skin);
    int cap = 256;
    int rc = ORC_OK;
    int32_t *idx = NULL, *cnt = NULL, status[2];
    /* candidate superset: fp64 list at radius R*(1+1e-3) from the chosen method */
    float Rw = R * 1.001f;
    idx = (int32_t *)malloc((size_t)n * cap * sizeof(int32_t));
    cnt = (int32_t *)malloc((size_t)n * sizeof(int32_t));
    if (!idx || !cnt) { free(idx); free(cnt); return ORC_ENOMEM; }
    rc = orc_neighbor_list(n, dim, pos, box, Rw, 0.0f, cap, 1, method, idx, cnt, status);
    if (rc != ORC_OK || status[0]) { free(idx); free(cnt); return rc ? rc : ORC_EINVAL; }
    int64_t nd = 0; double band = 0.0, close = 1e300;
    for (int i = 0; i < n; ++i) {
        for (int k = 0; k < cnt[i]; ++k) {
            int j = idx[(size_t)i * cap + k];
            const double *pi = pos + 3 * (size_t)i, *pj = pos + 3 * (size_t)j;
            int a = within(0, dim, pi, pj, box, R);
            int b = within(1, dim, pi, pj, box, R);
            double r2 = 0.0;
            for (int q = 0; q < dim; ++q) { double d = disp64(pi[q], pj[q], box[q]); r2 += d * d; }
            double gap = fabs(sqrt(r2) - (double)R);
            if (gap < close) close = gap;
            if (a != b) { nd++; if (gap / (double)R > band) band = gap / (double)R; }
        }
    }
    free(idx); free(cnt);
    *n_disagree = nd; *max_rel_band = band; *closest = close;
    return ORC_OK;
}

/* ------------------------------------------------------- pair functions -- */

/* Lennard-Jones u(r) (unshifted) and -u'(r)/r, from r^2 (PAPER.md:L104 [69]). */
static void lj_pair(double r2, double eps, double sigma, double *u, double *fr)
{
    double s2 = sigma * sigma / r2;
    double s6 = s2 * s2 * s2;
    double s12 = s6 * s6;
    *u = 4.0 * eps * (s12 - s6);
    *fr = 24.0 * eps * (2.0 * s12 - s6) / r2;
}

/* Morse u(r) = D (1 - exp(-alpha (r - r0)))^2 - D and -u'(r)/r (PAPER.md:L104 [75]; the paper
 * names the potential only: the standard form with well depth D at r0, reading A19). */

static void morse_pair(double r, double D, double r0, double alpha, double *u, double *fr)
{
    double x = exp(-alpha * (r - r0));
    *u = D * (1.0 - x) * (1.0 - x) - D;
    *fr = r > 0.0 ? -2.0 * D * alpha * x * (1.0 - x) / r : 0.0;
}

/* Buckingham-type u(r) = A exp(-B r) - C / r^6 and -u'(r)/r (PAPER.md:L104 [71-73]; the paper names
 * the family only: the exp-6 form without the Coulomb term of BKS, reading A24).
 * A = eps, B = orc_params.morse_alpha, C = sigma. */
static void buck_pair(double r, double A, double B, double Cc, double *u, double *fr)
{
    double x = A * exp(-B * r), r2 = r * r, r6 = r2 * r2 * r2;
    *u = x - Cc / r6;
    *fr = r > 0.0 ? (B * x - 6.0 * Cc / (r6 * r)) / r : 0.0;
}

/* Species x species Lennard-Jones (PAPER.md:L104 pair potentials with per-species parameters, the
 * sigma matrix of L298-L305 App. A): kind 4 reads eps_ab, sigma_ab and the truncation radius rc_ab
 * from tables set here; the species of particle i is (int)diam[i] (the pos.w channel). */
#define ORC_MAX_SPECIES 4
#define ORC_MAX_NH_CHAIN 8
/* The parameters of kinds 2-5 and the Nose-Hoover chain length travel with every call as one struct (the
 * Python wrapper owns it); nothing of them is process state.  Unset fields make the call that needs them
 * fail with ORC_EINVAL: morse_alpha = NaN, ns = 0, bks_ns = 0. */
typedef struct orc_params {
    double morse_alpha;                                   /* kind 2: alpha; kind 3: B */
    int32_t ns;                                           /* kind 4 */
    int32_t bks_ns;                                       /* kind 5 */
    int32_t nh_chain;                                     /* 1..ORC_MAX_NH_CHAIN */
    int32_t pad_;
    double sp_eps[ORC_MAX_SPECIES * ORC_MAX_SPECIES], sp_sig[ORC_MAX_SPECIES * ORC_MAX_SPECIES],
           sp_rc[ORC_MAX_SPECIES * ORC_MAX_SPECIES];
    double bks_A[ORC_MAX_SPECIES * ORC_MAX_SPECIES], bks_B[ORC_MAX_SPECIES * ORC_MAX_SPECIES],
           bks_C[ORC_MAX_SPECIES * ORC_MAX_SPECIES], bks_q[ORC_MAX_SPECIES], bks_a, bks_k;
} orc_params;

void orc_params_reset(orc_params *p)
{
    memset(p, 0, sizeof(*p));
    p->morse_alpha = NAN;
    p->nh_chain = 1;
    p->bks_k = 1.0;
}
int orc_params_size(void) { return (int)sizeof(orc_params); }

int orc_params_species_lj(orc_params *p, int ns, const double *eps, const double *sigma, const double *rc)
{
    if (!p || ns < 1 || ns > ORC_MAX_SPECIES) return ORC_EINVAL;
    p->ns = ns;
    for (int k = 0; k < ns * ns; ++k) { p->sp_eps[k] = eps[k]; p->sp_sig[k] = sigma[k]; p->sp_rc[k] = rc[k]; }
    return ORC_OK;
}

/* BKS-type potential ("Buckingham / BKS" [71-73]; named only, reading A27):
 * the exp-6 term with per-species-pair A_ab, B_ab, C_ab plus the Coulomb interaction of point charges
 * q_a.  A bare 1/r cannot live on a cutoff list, so the Coulomb term is the damped shifted-force form
 * (Fennell & Gezelter 2006), whose energy AND force vanish at r_c:
 *   u_C(r) = k q_a q_b [ erfc(a r)/r - erfc(a rc)/rc + (erfc(a rc)/rc^2 + 2a/sqrt(pi) exp(-a^2 rc^2)/rc)(r - rc) ]
 *   -u_C'(r) = k q_a q_b [ erfc(a r)/r^2 + 2a/sqrt(pi) exp(-a^2 r^2)/r - erfc(a rc)/rc^2 - 2a/sqrt(pi) exp(-a^2 rc^2)/rc ]
 * kind 5: species = (int)diam[i]; r_cut is the one truncation radius; shift applies to the exp-6 term. */
int orc_params_species_bks(orc_params *p, int ns, const double *A, const double *B, const double *Cc, const double *q,
                           double coulomb_alpha, double k_e)
{
    if (!p || ns < 1 || ns > ORC_MAX_SPECIES || !(coulomb_alpha >= 0.0)) return ORC_EINVAL;
    p->bks_ns = ns; p->bks_a = coulomb_alpha; p->bks_k = k_e;
    for (int k = 0; k < ns * ns; ++k) { p->bks_A[k] = A[k]; p->bks_B[k] = B[k]; p->bks_C[k] = Cc[k]; }
    for (int k = 0; k < ns; ++k) p->bks_q[k] = q[k];
    return ORC_OK;
}

static void dsf_pair(double r, double qq, double a, double rc, double *u, double *fr)
{
    const double tsp = 2.0 * a / sqrt(3.14159265358979323846);
    const double ec = erfc(a * rc) / rc, fc = ec / rc + tsp * exp(-a * a * rc * rc) / rc;
    *u = qq * (erfc(a * r) / r - ec + fc * (r - rc));
    *fr = qq * (erfc(a * r) / (r * r) + tsp * exp(-a * a * r * r) / r - fc) / r;
}

static double lj_u_cut(double eps, double sigma, double r_cut)
{
    double u, fr;
    lj_pair(r_cut * r_cut, eps, sigma, &u, &fr);
    return u;
}

/*
 * orc_energy_force: e_i = 1/2 sum_j u(r_ij), E = sum_i e_i,
 * F_i = -grad_{r_i} E in closed form, r_ij = ||d(r_i, r_j)||, fp64.
 *   kind 0 LJ:   u = 4 eps[(s/r)^12 - (s/r)^6] - shift*u(r_cut)  for r < r_cut
 *   kind 1 SOFT: u = eps/2 (1 - r/d_ij)^2 for r < d_ij, d_ij = (d_i + d_j)/2
 *                (PAPER.md:L301); r = 0 gives energy eps/2 and zero force
 *   kind 2 MORSE: u = eps (1 - exp(-alpha (r - sigma)))^2 - eps - shift*u(r_cut) for r < r_cut,
 *                alpha = par->morse_alpha (PAPER.md:L104 [75])
 *   kind 4 LJ_SPECIES: LJ with eps, sigma, r_cut taken per species pair from the tables of par (orc_params_species_lj),
 *                species = (int)diam[i]; eps, sigma, r_cut arguments unused
 *   kind 3 BUCKINGHAM: u = eps exp(-alpha r) - sigma / r^6 - shift*u(r_cut) for r < r_cut
 *                (A = eps, B = alpha, C = sigma; PAPER.md:L104 [71-73])
 *   kind 5 BKS:  exp-6 with A, B, C per species pair plus damped shifted-force Coulomb between the
 *                species' charges (orc_params_species_bks); eps, sigma unused; one r_cut
 *   nbr_idx == NULL: all pairs j != i (the definition);
 *   else: over the list rows (L80 smap.neighbors), entries >= n are padding.
 *   force double[n*3] (z = 0 in 2-D), e_i double[n], *E double.
 */
int orc_energy_force(int n, int dim, const double *pos, const double *diam,
                     const double *box, int kind, double eps, double sigma,
                     double r_cut, int shift, const int32_t *nbr_idx,
                     const int32_t *nbr_count, int capacity, double *force,
                     double *e_i, double *E, const orc_params *par)
{
    if (n <= 0 || (dim != 2 && dim != 3)) return ORC_EINVAL;
    if (kind != KIND_LJ && kind != KIND_SOFT && kind != KIND_MORSE && kind != KIND_BUCK &&
        kind != KIND_LJ_SPECIES && kind != KIND_BKS) return ORC_EINVAL;
    if ((kind == KIND_SOFT || kind == KIND_LJ_SPECIES || kind == KIND_BKS) && !diam) return ORC_EINVAL;
    if (kind != KIND_LJ && kind != KIND_SOFT && !par) return ORC_EINVAL;
    if (kind == KIND_LJ_SPECIES && par->ns < 1) return ORC_EINVAL;
    if (kind == KIND_BKS && par->bks_ns < 1) return ORC_EINVAL;
    if ((kind == KIND_MORSE || kind == KIND_BUCK) && !(par->morse_alpha == par->morse_alpha)) return ORC_EINVAL;   /* unset */
    const double g_morse_alpha = par ? par->morse_alpha : NAN;
    const int g_ns = par ? par->ns : 0, g_bks_ns = par ? par->bks_ns : 0;
    const double *g_sp_eps = par ? par->sp_eps : NULL, *g_sp_sig = par ? par->sp_sig : NULL, *g_sp_rc = par ? par->sp_rc : NULL;
    const double *g_bks_A = par ? par->bks_A : NULL, *g_bks_B = par ? par->bks_B : NULL, *g_bks_C = par ? par->bks_C : NULL;
    const double *g_bks_q = par ? par->bks_q : NULL, g_bks_a = par ? par->bks_a : 0.0, g_bks_k = par ? par->bks_k : 1.0;
    double u_c = (kind == KIND_LJ && shift) ? lj_u_cut(eps, sigma, r_cut) : 0.0;
    if (kind == KIND_MORSE && shift) {
        double fr_unused;
        morse_pair(r_cut, eps, sigma, g_morse_alpha, &u_c, &fr_unused);
    }
    if (kind == KIND_BUCK && shift) {
        double fr_unused;
        buck_pair(r_cut, eps, g_morse_alpha, sigma, &u_c, &fr_unused);
    }
#pragma omp parallel for schedule(dynamic, 64)
    for (int i = 0; i < n; ++i) {
        double f[3] = {0.0, 0.0, 0.0}, e = 0.0;
        int m = nbr_idx ? (nbr_count[i] < capacity ? nbr_count[i] : capacity) : n;
        for (int k = 0; k < m; ++k) {
            int j = nbr_idx ? nbr_idx[(size_t)i * capacity + k] : k;
            if (j == i || j >= n || j < 0) continue;
            double d[3] = {0.0, 0.0, 0.0}, r2 = 0.0;
            for (int q = 0; q < dim; ++q) {
                d[q] = disp64(pos[3 * (size_t)i + q], pos[3 * (size_t)j + q], box[q]);
                r2 += d[q] * d[q];
            }
            if (kind == KIND_LJ) {
                if (r2 < r_cut * r_cut) {
                    double u, fr;
                    lj_pair(r2, eps, sigma, &u, &fr);
                    e += 0.5 * (u - u_c);
                    for (int q = 0; q < dim; ++q) f[q] += fr * d[q];
                }
            } else if (kind == KIND_LJ_SPECIES) {
                int sa = (int)diam[i], sb = (int)diam[j];
                if (sa < 0 || sa >= g_ns || sb < 0 || sb >= g_ns) continue;
                int t = sa * g_ns + sb;
                if (r2 < g_sp_rc[t] * g_sp_rc[t]) {
                    double u, fr;
                    lj_pair(r2, g_sp_eps[t], g_sp_sig[t], &u, &fr);
                    e += 0.5 * (u - (shift ? lj_u_cut(g_sp_eps[t], g_sp_sig[t], g_sp_rc[t]) : 0.0));
                    for (int q = 0; q < dim; ++q) f[q] += fr * d[q];
                }
            } else if (kind == KIND_BKS) {
                int sa = (int)diam[i], sb = (int)diam[j];
                if (sa < 0 || sa >= g_bks_ns || sb < 0 || sb >= g_bks_ns) continue;
                int t = sa * g_bks_ns + sb;
                if (r2 < r_cut * r_cut && r2 > 0.0) {
                    double u, fr, uc, fc_unused, ue, fe;
                    const double r = sqrt(r2);
                    buck_pair(r, g_bks_A[t], g_bks_B[t], g_bks_C[t], &u, &fr);
                    buck_pair(r_cut, g_bks_A[t], g_bks_B[t], g_bks_C[t], &uc, &fc_unused);
                    dsf_pair(r, g_bks_k * g_bks_q[sa] * g_bks_q[sb], g_bks_a, r_cut, &ue, &fe);
                    e += 0.5 * (u - (shift ? uc : 0.0) + ue);
                    for (int q = 0; q < dim; ++q) f[q] += (fr + fe) * d[q];
                }
            } else if (kind == KIND_BUCK) {
                if (r2 < r_cut * r_cut) {
                    double u, fr;
                    buck_pair(sqrt(r2), eps, g_morse_alpha, sigma, &u, &fr);
                    e += 0.5 * (u - u_c);
                    for (int q = 0; q < dim; ++q) f[q] += fr * d[q];
                }
            } else if (kind == KIND_MORSE) {
                if (r2 < r_cut * r_cut) {
                    double u, fr;
                    morse_pair(sqrt(r2), eps, sigma, g_morse_alpha, &u, &fr);
                    e += 0.5 * (u - u_c);
                    for (int q = 0; q < dim; ++q) f[q] += fr * d[q];
                }
            } else {
                double dij = 0.5 * (diam[i] + diam[j]);
                double r = sqrt(r2);
                if (r < dij) {
                    double x = 1.0 - r / dij;
                    e += 0.5 * (0.5 * eps * x * x);
                    if (r > 0.0) {
                        double fr = eps / dij * x / r;
                        for (int q = 0; q < dim; ++q) f[q] += fr * d[q];
                    }
                }
            }
        }
        force[3 * (size_t)i + 0] = f[0];
        force[3 * (size_t)i + 1] = f[1];
        force[3 * (size_t)i + 2] = f[2];
        e_i[i] = e;
    }
    double tot = 0.0;
    for (int i = 0; i < n; ++i) tot += e_i[i];
    *E = tot;
    return ORC_OK;
}

/* ---------------------------------------------------------- rebuild test -- */

/*
 * orc_needs_rebuild: flag = max_i ||d(r_i, ref_i)||^2 >
 * (skin/2)^2, strict, nearest-image displacement, fp64.
 */
int orc_needs_rebuild(int n, int dim, const double *pos, const double *ref,
                      const double *box, double skin, int32_t *flag,
                      double *max_disp2)
{
    if (n <= 0 || (dim != 2 && dim != 3)) return ORC_EINVAL;
    double m = 0.0;
    for (int i = 0; i < n; ++i) {
        double r2 = 0.0;
        for (int q = 0; q < dim; ++q) {
            double d = disp64(pos[3 * (size_t)i + q], ref[3 * (size_t)i + q], box[q]);
            r2 += d * d;
        }
        if (r2 > m) m = r2;
    }
    *max_disp2 = m;
    *flag = m > (0.5 * skin) * (0.5 * skin) ? 1 : 0;
    return ORC_OK;
}

/* ------------------------------------------------------------------ NVE -- */

/*
 * orc_nve_run: nsteps of kick-drift-kick velocity
 * Verlet in fp64 (PAPER.md:L100, L78 m r'' = -grad U, L72 shift function):
 *     v <- v + (dt/2m) F;  r <- wrap(r + dt v);  F <- F(r);  v <- v + (dt/2m) F
 * `force` must hold F(pos) on entry.
 *   use_list 0: forces by brute force over all pairs (no list anywhere)
 *            1: forces over the oracle's own fp64 cell-binned list of radius
 *               r_cut + skin, rebuilt when orc_needs_rebuild fires after the
 *               drift (this is the loop bench.py times as the CPU baseline)
 *   energies  out (may be NULL): double[(nsteps+1)*2] = (KE, PE) at every step
 *             boundary, entry 0 being the state on entry
 *   stats     out int32[3]: rebuilds, overflow (0/1), max neighbor count seen
 */
int orc_nve_run(int n, int dim, double *pos, double *vel, double *force,
                const double *diam, const double *box, int kind, double eps,
                double sigma, double r_cut, int shift, double dt, double mass,
                int nsteps, int use_list, float skin, int capacity,
                double *energies, int32_t *stats, const orc_params *par)
{
    if (n <= 0 || (dim != 2 && dim != 3) || dt <= 0.0 || mass <= 0.0) return ORC_EINVAL;
    int rc = ORC_OK;
    double *e_i = (double *)malloc((size_t)n * sizeof(double));
    double *ref = NULL;
    int32_t *idx = NULL, *cnt = NULL;
    int32_t st[2] = {0, 0};
    int rebuilds = 0, overflow = 0, maxc = 0;
    double E = 0.0;
    if (!e_i) return ORC_ENOMEM;
    if (use_list) {
        ref = (double *)malloc((size_t)n * 3 * sizeof(double));
        idx = (int32_t *)malloc((size_t)n * capacity * sizeof(int32_t));
        cnt = (int32_t *)malloc((size_t)n * sizeof(int32_t));
        if (!ref || !idx || !cnt) { rc = ORC_ENOMEM; goto done; }
        rc = orc_neighbor_list(n, dim, pos, box, (float)r_cut, skin, capacity, 1, 1, idx, cnt, st);
        if (rc) goto done;
        memcpy(ref, pos, (size_t)n * 3 * sizeof(double));
        overflow |= st[0]; if (st[1] > maxc) maxc = st[1];
    }
    if (energies) {
        double ke = 0.0;
        rc = orc_energy_force(n, dim, pos, diam, box, kind, eps, sigma, r_cut, shift,
                              idx, cnt, capacity, force, e_i, &E, par);
        if (rc) goto done;
        for (int i = 0; i < n; ++i)
            for (int q = 0; q < dim; ++q) ke += vel[3 * (size_t)i + q] * vel[3 * (size_t)i + q];
        energies[0] = 0.5 * mass * ke; energies[1] = E;
    }
    double a = dt / (2.0 * mass);
    for (int s = 0; s < nsteps; ++s) {
        for (int i = 0; i < n; ++i)
            for (int q = 0; q < dim; ++q) {
                size_t t = 3 * (size_t)i + q;
                vel[t] = vel[t] + a * force[t];
                pos[t] = wrap64(pos[t] + dt * vel[t], box[q]);
            }
        if (use_list) {
            int32_t flag; double md2;
            orc_needs_rebuild(n, dim, pos, ref, box, (double)skin, &flag, &md2);
            if (flag) {
                rc = orc_neighbor_list(n, dim, pos, box, (float)r_cut, skin, capacity, 1, 1, idx, cnt, st);
                if (rc) goto done;
                memcpy(ref, pos, (size_t)n * 3 * sizeof(double));
                rebuilds++; overflow |= st[0]; if (st[1] > maxc) maxc = st[1];
            }
        }
        rc = orc_energy_force(n, dim, pos, diam, box, kind, eps, sigma, r_cut, shift,
                              idx, cnt, capacity, force, e_i, &E, par);
        if (rc) goto done;
        double ke = 0.0;
        for (int i = 0; i < n; ++i)
            for (int q = 0; q < dim; ++q) {
                size_t t = 3 * (size_t)i + q;
                vel[t] = vel[t] + a * force[t];
                ke += vel[t] * vel[t];
            }
        if (energies) { energies[2 * (s + 1)] = 0.5 * mass * ke; energies[2 * (s + 1) + 1] = E; }
    }
    if (stats) { stats[0] = rebuilds; stats[1] = overflow; stats[2] = maxc; }
done:
    free(e_i); free(ref); free(idx); free(cnt);
    return rc;
}

/* ------------------------------------------------------------------ FIRE -- */

/*
 * orc_fire_run: FIRE minimisation (PAPER.md:L100 names "FIRE Descent" among the simulation
 * environments and uses it to relax packings in section 4.2; the paper gives no formulas, so
 * this is the algorithm of its reference [Bitzek et al. 2006] around the same velocity-Verlet
 * step and force call, reading A20).  Unit mass.  Per step, with the current dt, alpha:
 *   1. v += dt/2 F;  r = wrap(r + dt v);  F = F(r);  v += dt/2 F          (velocity Verlet)
 *   2. P = sum F.v,  |F| = sqrt(sum F.F),  |v| = sqrt(sum v.v)
 *   3. P > 0:  v = (1 - alpha) v + alpha |v| F / |F|;  n_pos += 1;
 *              if n_pos > n_min: dt = min(dt f_inc, dt_max), alpha = alpha f_alpha
 *      else:   v = 0;  n_pos = 0;  dt = dt f_dec;  alpha = alpha_start
 * Forces by the all-pairs definition (orc_energy_force without a list).
 *   par   in  double[7] = {dt_start, dt_max, n_min, f_inc, f_dec, alpha_start, f_alpha}
 *   state in/out double[3] = {dt, alpha, n_pos}; pass dt <= 0 to start from dt_start, alpha_start, 0
 *   energies out (may be NULL) double[nsteps+1]: potential energy at every step boundary
 */
int orc_fire_run(int n, int dim, double *pos, double *vel, double *force, const double *diam,
                 const double *box, int kind, double eps, double sigma, double r_cut, int shift,
                 const double *fire, double *state, int nsteps, double *energies, const orc_params *par)
{
    if (n <= 0 || (dim != 2 && dim != 3) || !fire || !state) return ORC_EINVAL;
    double *e_i = (double *)malloc((size_t)n * sizeof(double));
    if (!e_i) return ORC_ENOMEM;
    double dt = state[0], alpha = state[1];
    int n_pos = (int)state[2];
    if (dt <= 0.0) { dt = fire[0]; alpha = fire[5]; n_pos = 0; }
    double E = 0.0;
    int rc = orc_energy_force(n, dim, pos, diam, box, kind, eps, sigma, r_cut, shift,
                              NULL, NULL, 0, force, e_i, &E, par);
    if (rc) { free(e_i); return rc; }
    if (energies) energies[0] = E;
    for (int s = 0; s < nsteps; ++s) {
        for (int i = 0; i < n; ++i)
            for (int q = 0; q < dim; ++q) {
                size_t t = 3 * (size_t)i + q;
                vel[t] = vel[t] + 0.5 * dt * force[t];
                pos[t] = wrap64(pos[t] + dt * vel[t], box[q]);
            }
        rc = orc_energy_force(n, dim, pos, diam, box, kind, eps, sigma, r_cut, shift,
                              NULL, NULL, 0, force, e_i, &E, par);
        if (rc) break;
        double P = 0.0, FF = 0.0, VV = 0.0;
        for (int i = 0; i < n; ++i)
            for (int q = 0; q < dim; ++q) {
                size_t t = 3 * (size_t)i + q;
                vel[t] = vel[t] + 0.5 * dt * force[t];
                P += force[t] * vel[t]; FF += force[t] * force[t]; VV += vel[t] * vel[t];
            }
        if (P > 0.0) {
            double c2 = FF > 0.0 ? alpha * sqrt(VV) / sqrt(FF) : 0.0;
            for (int i = 0; i < n; ++i)
                for (int q = 0; q < dim; ++q) {
                    size_t t = 3 * (size_t)i + q;
                    vel[t] = (1.0 - alpha) * vel[t] + c2 * force[t];
                }
            n_pos += 1;
            if (n_pos > (int)fire[2]) {
                dt = dt * fire[3] < fire[1] ? dt * fire[3] : fire[1];
                alpha = alpha * fire[6];
            }
        } else {
            for (size_t t = 0; t < 3 * (size_t)n; ++t) vel[t] = 0.0;
            n_pos = 0; dt = dt * fire[4]; alpha = fire[5];
        }
        if (energies) energies[s + 1] = E;
    }
    state[0] = dt; state[1] = alpha; state[2] = (double)n_pos;
    free(e_i);
    return rc;
}

/* -------------------------------------------------- Brownian / gradient descent -- */

/*
 * Counter-based standard normals (SURVEY 8f-f3 "needs a counter-based device RNG"; each side
 * implements the same generator): key = (seed, step, particle id, pair index c) -> splitmix64
 * finaliser -> two 24-bit uniforms u1 in (0,1], u2 in [0,1) -> Box-Muller pair
 *   g0 = sqrt(-2 ln u1) cos(2 pi u2),  g1 = sqrt(-2 ln u1) sin(2 pi u2).
 * Components x, y come from c = 0, component z from g0 of c = 1.
 */
static void orc_normal_pair(uint32_t seed, uint32_t step, uint32_t id, uint32_t c, double *g0, double *g1)
{
    uint64_t z = (uint64_t)seed * 0x9E3779B97F4A7C15ull + (uint64_t)step * 0xBF58476D1CE4E5B9ull
               + (uint64_t)id * 0x94D049BB133111EBull + (uint64_t)c;
    z ^= z >> 30; z *= 0xBF58476D1CE4E5B9ull;
    z ^= z >> 27; z *= 0x94D049BB133111EBull;
    z ^= z >> 31;
    double u1 = (double)((z >> 40) + 1ull) * (1.0 / 16777216.0);
    double u2 = (double)((z >> 8) & 0xFFFFFFull) * (1.0 / 16777216.0);
    double r = sqrt(-2.0 * log(u1)), a = 2.0 * 3.14159265358979323846 * u2;
    *g0 = r * cos(a); *g1 = r * sin(a);
}

void orc_normals(uint32_t seed, uint32_t step, int n, int dim, double *out /* n*3 */)
{
    for (int i = 0; i < n; ++i) {
        double g0, g1, g2, g3;
        orc_normal_pair(seed, step, (uint32_t)i, 0u, &g0, &g1);
        orc_normal_pair(seed, step, (uint32_t)i, 1u, &g2, &g3);
        out[3 * (size_t)i] = g0; out[3 * (size_t)i + 1] = g1; out[3 * (size_t)i + 2] = dim == 3 ? g2 : 0.0;
    }
}

/*
 * orc_brownian_run: overdamped (Brownian) dynamics at temperature kT, "Brownian
 * simulations at constant temperature"; kT = 0 is the paper's "Gradient Descent" (L100).  The paper
 * gives no formulas: Euler-Maruyama, reading A21.  Per step s (global index step0 + s):
 *   r_i = wrap(r_i + (dt/gamma) F_i(r) + sqrt(2 kT dt / gamma) xi_i),  xi_i = orc_normals(seed, step, i)
 * with F by the all-pairs definition.  force holds F of the final positions on exit.
 */
int orc_brownian_run(int n, int dim, double *pos, double *force, const double *diam, const double *box,
                     int kind, double eps, double sigma, double r_cut, int shift, double dt,
                     double gamma, double kT, uint32_t seed, uint32_t step0, int nsteps, double *energies,
                     const orc_params *par)
{
    if (n <= 0 || (dim != 2 && dim != 3) || dt <= 0.0 || gamma <= 0.0 || kT < 0.0) return ORC_EINVAL;
    double *e_i = (double *)malloc((size_t)n * sizeof(double));
    if (!e_i) return ORC_ENOMEM;
    double E = 0.0;
    int rc = orc_energy_force(n, dim, pos, diam, box, kind, eps, sigma, r_cut, shift, NULL, NULL, 0, force, e_i, &E, par);
    if (energies) energies[0] = E;
    const double mu = dt / gamma, amp = sqrt(2.0 * kT * dt / gamma);
    for (int s = 0; s < nsteps && !rc; ++s) {
        for (int i = 0; i < n; ++i) {
            double g[4];
            orc_normal_pair(seed, step0 + (uint32_t)s, (uint32_t)i, 0u, &g[0], &g[1]);
            orc_normal_pair(seed, step0 + (uint32_t)s, (uint32_t)i, 1u, &g[2], &g[3]);
            for (int q = 0; q < dim; ++q) {
                size_t t = 3 * (size_t)i + q;
                pos[t] = wrap64(pos[t] + mu * force[t] + amp * g[q], box[q]);
            }
        }
        rc = orc_energy_force(n, dim, pos, diam, box, kind, eps, sigma, r_cut, shift, NULL, NULL, 0, force, e_i, &E, par);
        if (energies) energies[s + 1] = E;
    }
    free(e_i);
    return rc;
}

/* ------------------------------------------------------------- Langevin -- */

/*
 * orc_langevin_run: Langevin dynamics at temperature kT ("Langevin ... simulations
 * at constant temperature"; no formulas in the paper: the BAOAB splitting, reading A22).
 * Per step s (global index step0 + s), a = dt/(2m):
 *   B: v += a F;  A: r += dt/2 v;  O: v = c1 v + c2 xi, c1 = exp(-gamma dt), c2 = sqrt(kT/m (1 - c1^2));
 *   A: r = wrap(r + dt/2 v);  F = F(r);  B: v += a F
 * xi = orc_normals(seed, step, i).  gamma = 0 (c1 = 1, c2 = 0) is velocity Verlet.  All-pairs forces;
 * force must hold F(pos) on entry.
 */
int orc_langevin_run(int n, int dim, double *pos, double *vel, double *force, const double *diam,
                     const double *box, int kind, double eps, double sigma, double r_cut, int shift,
                     double dt, double mass, double gamma, double kT, uint32_t seed, uint32_t step0,
                     int nsteps, const orc_params *par)
{
    if (n <= 0 || (dim != 2 && dim != 3) || dt <= 0.0 || mass <= 0.0 || gamma < 0.0 || kT < 0.0) return ORC_EINVAL;
    double *e_i = (double *)malloc((size_t)n * sizeof(double));
    if (!e_i) return ORC_ENOMEM;
    const double a = dt / (2.0 * mass), c1 = exp(-gamma * dt), c2 = sqrt(kT / mass * (1.0 - c1 * c1));
    double E = 0.0;
    int rc = ORC_OK;
    for (int s = 0; s < nsteps && !rc; ++s) {
        for (int i = 0; i < n; ++i) {
            double g[4];
            orc_normal_pair(seed, step0 + (uint32_t)s, (uint32_t)i, 0u, &g[0], &g[1]);
            orc_normal_pair(seed, step0 + (uint32_t)s, (uint32_t)i, 1u, &g[2], &g[3]);
            for (int q = 0; q < dim; ++q) {
                size_t t = 3 * (size_t)i + q;
                double v = vel[t] + a * force[t];
                double r = pos[t] + 0.5 * dt * v;
                v = c1 * v + c2 * g[q];
                pos[t] = wrap64(r + 0.5 * dt * v, box[q]);
                vel[t] = v;
            }
        }
        rc = orc_energy_force(n, dim, pos, diam, box, kind, eps, sigma, r_cut, shift, NULL, NULL, 0, force, e_i, &E, par);
        for (int i = 0; i < n; ++i)
            for (int q = 0; q < dim; ++q) {
                size_t t = 3 * (size_t)i + q;
                vel[t] = vel[t] + a * force[t];
            }
    }
    free(e_i);
    return rc;
}

/* ---------------------------------------------------------- Nose-Hoover -- */

/*
 * orc_nose_hoover_run: NVT by a Nose-Hoover thermostat ("Nose-Hoover [67]"; no
 * formulas in the paper: one thermostat variable, the explicit reversible splitting of Martyna,
 * Tuckerman, Tobias and Klein around the velocity-Verlet step, reading A23).
 * dof = dim n, Q = dof kT tau^2.  Thermostat half step T(dt):
 *   K2 = sum m v^2;  G = (K2 - dof kT)/Q;  vxi += dt/4 G;  s = exp(-dt/2 vxi);  v *= s;
 *   xi += dt/2 vxi;  K2 *= s^2;  G = (K2 - dof kT)/Q;  vxi += dt/4 G
 * Step: T(dt);  v += dt/(2m) F;  r = wrap(r + dt v);  F = F(r);  v += dt/(2m) F;  T(dt).
 * Conserved: H' = K + U + Q vxi^2 / 2 + dof kT xi.
 *   state in/out double[2] = {xi, vxi};  conserved out (may be NULL) double[nsteps+1] = H'
 */
/* Chain length M (Martyna, Klein and Tuckerman's chains [67]; 1 = the single thermostat above).
 * Masses Q_1 = dof kT tau^2, Q_j = kT tau^2 (j >= 2).  Thermostat half step T(dt), d = dt/2:
 *   G_1 = (K2 - dof kT)/Q_1,  G_j = (Q_{j-1} v_{j-1}^2 - kT)/Q_j
 *   v_M += d/2 G_M;  for j = M-1 .. 1:  a = exp(-d/4 v_{j+1}),  v_j = (v_j a + d/2 G_j) a
 *   s = exp(-d v_1);  v *= s;  K2 *= s^2;  xi_j += d v_j (all j)
 *   for j = 1 .. M-1:  a = exp(-d/4 v_{j+1}),  v_j = (v_j a + d/2 G_j) a  (G_j from the updated
 *   v_{j-1}, K2);  v_M += d/2 G_M
 * Conserved: H' = K + U + sum_j Q_j v_j^2 / 2 + dof kT xi_1 + kT sum_{j>=2} xi_j.
 * state = {xi_1..xi_M, v_1..v_M}. */
static double nh_G(int j, int M, double K2, double dofkT, double kT, const double *Q, const double *v)
{
    (void)M;
    return j == 0 ? (K2 - dofkT) / Q[0] : (Q[j - 1] * v[j - 1] * v[j - 1] - kT) / Q[j];
}

static void nh_half(int n, int dim, double *vel, double mass, double dofkT, double kT, const double *Q, int M,
                    double dt, double *xi, double *v)
{
    double K2 = 0.0;
    for (int i = 0; i < n; ++i)
        for (int q = 0; q < dim; ++q) K2 += mass * vel[3 * (size_t)i + q] * vel[3 * (size_t)i + q];
    v[M - 1] += 0.25 * dt * nh_G(M - 1, M, K2, dofkT, kT, Q, v);
    for (int j = M - 2; j >= 0; --j) {
        double a = exp(-0.125 * dt * v[j + 1]);
        v[j] = (v[j] * a + 0.25 * dt * nh_G(j, M, K2, dofkT, kT, Q, v)) * a;
    }
    double sc = exp(-0.5 * dt * v[0]);
    for (int i = 0; i < n; ++i)
        for (int q = 0; q < dim; ++q) vel[3 * (size_t)i + q] *= sc;
    for (int j = 0; j < M; ++j) xi[j] += 0.5 * dt * v[j];
    K2 *= sc * sc;
    for (int j = 0; j < M - 1; ++j) {
        double a = exp(-0.125 * dt * v[j + 1]);
        v[j] = (v[j] * a + 0.25 * dt * nh_G(j, M, K2, dofkT, kT, Q, v)) * a;
    }
    v[M - 1] += 0.25 * dt * nh_G(M - 1, M, K2, dofkT, kT, Q, v);
}

int orc_nose_hoover_run(int n, int dim, double *pos, double *vel, double *force, const double *diam,
                        const double *box, int kind, double eps, double sigma, double r_cut, int shift,
                        double dt, double mass, double kT, double tau, double *state, int nsteps,
                        double *conserved, const orc_params *par)
{
    if (n <= 0 || (dim != 2 && dim != 3) || dt <= 0.0 || mass <= 0.0 || kT <= 0.0 || tau <= 0.0 || !state || !par ||
        par->nh_chain < 1 || par->nh_chain > ORC_MAX_NH_CHAIN)
        return ORC_EINVAL;
    double *e_i = (double *)malloc((size_t)n * sizeof(double));
    if (!e_i) return ORC_ENOMEM;
    const double dofkT = (double)dim * n * kT, a = dt / (2.0 * mass);
    const int M = par->nh_chain;
    double Q[ORC_MAX_NH_CHAIN], xi[ORC_MAX_NH_CHAIN], vxi[ORC_MAX_NH_CHAIN], E = 0.0;
    for (int j = 0; j < M; ++j) { Q[j] = (j == 0 ? dofkT : kT) * tau * tau; xi[j] = state[j]; vxi[j] = state[M + j]; }
    int rc = orc_energy_force(n, dim, pos, diam, box, kind, eps, sigma, r_cut, shift, NULL, NULL, 0, force, e_i, &E, par);
    for (int s = 0; s <= nsteps && !rc; ++s) {
        if (conserved) {
            double K2 = 0.0;
            for (int i = 0; i < n; ++i)
                for (int q = 0; q < dim; ++q) K2 += mass * vel[3 * (size_t)i + q] * vel[3 * (size_t)i + q];
            double H = 0.5 * K2 + E + dofkT * xi[0];
            for (int j = 0; j < M; ++j) H += 0.5 * Q[j] * vxi[j] * vxi[j] + (j > 0 ? kT * xi[j] : 0.0);
            conserved[s] = H;
        }
        if (s == nsteps) break;
        nh_half(n, dim, vel, mass, dofkT, kT, Q, M, dt, xi, vxi);
        for (int i = 0; i < n; ++i)
            for (int q = 0; q < dim; ++q) {
                size_t t = 3 * (size_t)i + q;
                vel[t] += a * force[t];
                pos[t] = wrap64(pos[t] + dt * vel[t], box[q]);
            }
        rc = orc_energy_force(n, dim, pos, diam, box, kind, eps, sigma, r_cut, shift, NULL, NULL, 0, force, e_i, &E, par);
        for (int i = 0; i < n; ++i)
            for (int q = 0; q < dim; ++q) vel[3 * (size_t)i + q] += a * force[3 * (size_t)i + q];
        nh_half(n, dim, vel, mass, dofkT, kT, Q, M, dt, xi, vxi);
    }
    for (int j = 0; j < M; ++j) { state[j] = xi[j]; state[M + j] = vxi[j]; }
    free(e_i);
    return rc;
}

/* -------------------------------------------------------------- flocking -- */

/*
 * Boids as an energy model (App. B), 2-D, state (R_i, theta_i), N(theta) =
 * (cos theta, sin theta).  DESIGN.md reading A25 for what the text leaves open:
 *   rho(r; Rc)   = (1/alpha)(1 - r/Rc)^alpha for r < Rc, else 0                          (eq. 6)
 *   E_align      = 1/2 sum_{i != j} J_al rho(r_ij; R_al) (1 - N_i.N_j)^2                  (eq. 7)
 *                  with a stop-gradient on the displacement: it has NO gradient in R
 *   E_avoid      = 1/2 sum_{i != j} J_av rho(r_ij; R_av)                                  (eq. 8)
 *   E_cohesion   = sum_i 1/2 J_co (1 - Dhat_i.N_i)^2,  D_i = sum_{j in N_i} (R_j - R_i),
 *                  N_i = {j : r_ij < R_co}; 0 when N_i is empty or D_i = 0       (eqs. 9-10; the
 *                  normalised mean of eq. 9 equals the normalised sum; the set is held fixed)
 * par = {J_al, R_al, J_av, R_av, J_co, R_co, alpha}.  Outputs: energies[3] = (align, avoid, cohesion),
 * gR double[n*2] = grad_R E (align excluded by the stop-gradient), gth double[n] = grad_theta E.
 */
static double flock_rho(double r, double Rc, double alpha) { return r < Rc ? pow(1.0 - r / Rc, alpha) / alpha : 0.0; }
static double flock_drho(double r, double Rc, double alpha) { return r < Rc ? -pow(1.0 - r / Rc, alpha - 1.0) / Rc : 0.0; }

int orc_flock_energy_grad(int n, const double *pos /* n*3, z ignored */, const double *theta, const double *box,
                          const double *par, double *energies, double *gR, double *gth)
{
    if (n <= 0 || !par) return ORC_EINVAL;
    const double Jal = par[0], Ral = par[1], Jav = par[2], Rav = par[3], Jco = par[4], Rco = par[5], al = par[6];
    double *G = (double *)calloc((size_t)n * 2, sizeof(double));      /* g_i = d e_i / d D_i */
    int *cntN = (int *)calloc((size_t)n, sizeof(int));
    if (!G || !cntN) { free(G); free(cntN); return ORC_ENOMEM; }
    double Ea = 0.0, Ev = 0.0, Ec = 0.0;
    for (int i = 0; i < n; ++i) { gR[2 * i] = gR[2 * i + 1] = 0.0; gth[i] = 0.0; }
    for (int i = 0; i < n; ++i) {
        const double ci = cos(theta[i]), si = sin(theta[i]);
        double D[2] = {0.0, 0.0};
        int m = 0;
        for (int j = 0; j < n; ++j) {
            if (j == i) continue;
            double d[2];
            d[0] = disp64(pos[3 * (size_t)i], pos[3 * (size_t)j], box[0]);       /* R_i - R_j */
            d[1] = disp64(pos[3 * (size_t)i + 1], pos[3 * (size_t)j + 1], box[1]);
            const double r = sqrt(d[0] * d[0] + d[1] * d[1]);
            /* alignment: theta gradient only */
            const double cd = ci * cos(theta[j]) + si * sin(theta[j]);            /* N_i.N_j = cos(th_i - th_j) */
            const double sd = si * cos(theta[j]) - ci * sin(theta[j]);            /* sin(th_i - th_j) */
            const double ra = flock_rho(r, Ral, al);
            Ea += 0.5 * Jal * ra * (1.0 - cd) * (1.0 - cd);
            gth[i] += Jal * ra * 2.0 * (1.0 - cd) * sd;                           /* both ordered pairs: 1/2 * 2 */
            /* avoidance */
            Ev += 0.5 * Jav * flock_rho(r, Rav, al);
            if (r > 0.0) {
                const double dr = Jav * flock_drho(r, Rav, al);                   /* 1/2 * 2 ordered pairs */
                gR[2 * i] += dr * d[0] / r; gR[2 * i + 1] += dr * d[1] / r;
            }
            if (r < Rco) { D[0] -= d[0]; D[1] -= d[1]; ++m; }                     /* R_j - R_i */
        }
        cntN[i] = m;
        const double Dn = sqrt(D[0] * D[0] + D[1] * D[1]);
        if (m > 0 && Dn > 0.0) {
            const double hx = D[0] / Dn, hy = D[1] / Dn, c = hx * ci + hy * si;
            Ec += 0.5 * Jco * (1.0 - c) * (1.0 - c);
            /* d e / d D = -J (1 - c) (N - c Dhat) / |D| */
            G[2 * i] = -Jco * (1.0 - c) * (ci - c * hx) / Dn;
            G[2 * i + 1] = -Jco * (1.0 - c) * (si - c * hy) / Dn;
            /* d e / d theta = -J (1 - c) Dhat . dN/dtheta,  dN/dtheta = (-sin, cos) */
            gth[i] += -Jco * (1.0 - c) * (-hx * si + hy * ci);
        }
    }
    /* grad_{R_k} E_co = -|N_k| g_k + sum_{i : k in N_i} g_i  (the relation r < R_co is symmetric) */
    for (int k = 0; k < n; ++k) {
        gR[2 * k] += -cntN[k] * G[2 * k]; gR[2 * k + 1] += -cntN[k] * G[2 * k + 1];
        for (int i = 0; i < n; ++i) {
            if (i == k) continue;
            const double dx = disp64(pos[3 * (size_t)k], pos[3 * (size_t)i], box[0]);
            const double dy = disp64(pos[3 * (size_t)k + 1], pos[3 * (size_t)i + 1], box[1]);
            if (sqrt(dx * dx + dy * dy) < Rco) { gR[2 * k] += G[2 * i]; gR[2 * k + 1] += G[2 * i + 1]; }
        }
    }
    if (energies) { energies[0] = Ea; energies[1] = Ev; energies[2] = Ec; }
    free(G); free(cntN);
    return ORC_OK;
}

/*
 * Obstacles (App. B.3.1, eq. 11): disks o with centre C_o and radius D_o;
 *   e_io = J_ob rho(r_io; D_o) (1 + N_i . Rhat_io)^2,  R_io = C_o - R_i (nearest image), r_io = |R_io|
 * -- zero unless the boid is inside the disk, smallest when it heads straight away from the centre
 * (reading A26: the range of rho is the disk's own radius; R_io points from the boid to
 * the obstacle, the sign convention of eqs. 9-10; gradients in R and theta both act).
 *   d e / d theta = 2 J rho (1 + c) (-sin th u_x + cos th u_y),      u = R_io / r, c = N . u
 *   grad_{R_i} e  = -J [ rho'(r) (1 + c)^2 u + 2 rho (1 + c) (N - c u) / r ]
 * orc_flock_obstacle_energy_grad ADDS to gR / gth and returns the energy in *energy.
 */
int orc_flock_obstacle_energy_grad(int n, const double *pos, const double *theta, const double *box, int nobs,
                                   const double *centre /* nobs*2 */, const double *radius, double J,
                                   double alpha, double *energy, double *gR, double *gth)
{
    if (n <= 0 || nobs < 0) return ORC_EINVAL;
    double E = 0.0;
    for (int i = 0; i < n; ++i) {
        const double ci = cos(theta[i]), si = sin(theta[i]);
        for (int o = 0; o < nobs; ++o) {
            const double dx = disp64(centre[2 * o], pos[3 * (size_t)i], box[0]);          /* C_o - R_i */
            const double dy = disp64(centre[2 * o + 1], pos[3 * (size_t)i + 1], box[1]);
            const double r = sqrt(dx * dx + dy * dy);
            if (!(r < radius[o]) || !(r > 0.0)) continue;
            const double ux = dx / r, uy = dy / r, c = ci * ux + si * uy;
            const double rho = flock_rho(r, radius[o], alpha), drho = flock_drho(r, radius[o], alpha);
            E += J * rho * (1.0 + c) * (1.0 + c);
            if (gth) gth[i] += 2.0 * J * rho * (1.0 + c) * (-si * ux + ci * uy);
            if (gR) {
                gR[2 * i] += -J * (drho * (1.0 + c) * (1.0 + c) * ux + 2.0 * rho * (1.0 + c) * (ci - c * ux) / r);
                gR[2 * i + 1] += -J * (drho * (1.0 + c) * (1.0 + c) * uy + 2.0 * rho * (1.0 + c) * (si - c * uy) / r);
            }
        }
    }
    if (energy) *energy = E;
    return ORC_OK;
}

/* obstacles seen by orc_flock_run (none by default) */
#define ORC_MAX_OBSTACLES 16
static int g_nobs = 0;
static double g_obs_centre[2 * ORC_MAX_OBSTACLES], g_obs_radius[ORC_MAX_OBSTACLES], g_obs_J = 0.0;

int orc_flock_set_obstacles(int nobs, const double *centre, const double *radius, double J)
{
    if (nobs < 0 || nobs > ORC_MAX_OBSTACLES) return ORC_EINVAL;
    g_nobs = nobs; g_obs_J = J;
    for (int o = 0; o < nobs; ++o) {
        g_obs_centre[2 * o] = centre[2 * o]; g_obs_centre[2 * o + 1] = centre[2 * o + 1];
        g_obs_radius[o] = radius[o];
    }
    return ORC_OK;
}

/*
 * Predators (App. B.3.2, eqs. 12-13; reading A28): a second, small population with
 * the same kind of state (R_p, theta_p).  Two-player game: each side descends ITS OWN energy in its own
 * coordinates only.
 *   boids:     E_boid = eqs. 7-10 + obstacles + sum_{i,p} J_flee rho(r_ip; R_flee)(1 + N_i . Rhat_ip)^2
 *              -- "the same obstacle avoiding energy" with the predator as a moving disk of radius R_flee:
 *              orc_flock_obstacle_energy_grad with centre = predator positions serves it unchanged.
 *   predators: E_pred = sum_p [ 1/2 J_chase (1 - Dhat_p . N_p)^2 + obstacles ],
 *              D_p = sum_{i: |R_i - R_p| < R_chase} (R_i - R_p) -- "reuse the cohesion function": the
 *              predator heads for the centre of mass of the boids near it; 0 if there are none.
 *              d e/d theta_p = -J (1 - c)(-hx sin + hy cos);  grad_{R_p} e = +m J (1 - c)(N - c Dhat)/|D|
 *              (the set held fixed, m its size), c = Dhat . N.
 * orc_predator_energy_grad: the chase term alone; gR double[np*2], gth double[np] are OVERWRITTEN.
 */
int orc_predator_energy_grad(int n, const double *pos, const double *box, int np, const double *ppos /* np*2 */,
                             const double *pth, double J, double R, double *energy, double *gR, double *gth)
{
    if (n <= 0 || np < 0) return ORC_EINVAL;
    double E = 0.0;
    for (int p = 0; p < np; ++p) {
        double D[2] = {0.0, 0.0};
        int m = 0;
        for (int i = 0; i < n; ++i) {
            const double dx = disp64(pos[3 * (size_t)i], ppos[2 * p], box[0]);            /* R_i - R_p */
            const double dy = disp64(pos[3 * (size_t)i + 1], ppos[2 * p + 1], box[1]);
            if (sqrt(dx * dx + dy * dy) < R) { D[0] += dx; D[1] += dy; ++m; }
        }
        gR[2 * p] = gR[2 * p + 1] = 0.0; gth[p] = 0.0;
        const double Dn = sqrt(D[0] * D[0] + D[1] * D[1]);
        if (m > 0 && Dn > 0.0) {
            const double cp = cos(pth[p]), sn = sin(pth[p]);
            const double hx = D[0] / Dn, hy = D[1] / Dn, c = hx * cp + hy * sn;
            E += 0.5 * J * (1.0 - c) * (1.0 - c);
            gth[p] = -J * (1.0 - c) * (-hx * sn + hy * cp);
            gR[2 * p] = m * J * (1.0 - c) * (cp - c * hx) / Dn;
            gR[2 * p + 1] = m * J * (1.0 - c) * (sn - c * hy) / Dn;
        }
    }
    if (energy) *energy = E;
    return ORC_OK;
}

/*
 * orc_flock_run_predators: forward Euler for both populations, every gradient from the state at the
 * start of the step.  ppar = {J_flee, R_flee, J_chase, R_chase, speed_pred}; obstacles as set by
 * orc_flock_set_obstacles act on both.  ppos double[np*2], pth double[np] in/out.
 */
int orc_flock_run_predators(int n, double *pos, double *theta, const double *box, const double *par, double speed,
                            double dt, int nsteps, int np, double *ppos, double *pth, const double *ppar)
{
    if (np < 0 || np > ORC_MAX_OBSTACLES) return ORC_EINVAL;
    double *gR = (double *)malloc((size_t)n * 2 * sizeof(double)), *gth = (double *)malloc((size_t)n * sizeof(double));
    if (!gR || !gth) { free(gR); free(gth); return ORC_ENOMEM; }
    double qR[2 * ORC_MAX_OBSTACLES], qth[ORC_MAX_OBSTACLES], p3[3 * ORC_MAX_OBSTACLES], rfl[ORC_MAX_OBSTACLES];
    int rc = ORC_OK;
    for (int s = 0; s < nsteps && !rc; ++s) {
        rc = orc_flock_energy_grad(n, pos, theta, box, par, NULL, gR, gth);
        if (!rc && g_nobs > 0)
            rc = orc_flock_obstacle_energy_grad(n, pos, theta, box, g_nobs, g_obs_centre, g_obs_radius, g_obs_J,
                                                par[6], NULL, gR, gth);
        for (int p = 0; p < np; ++p) rfl[p] = ppar[1];
        if (!rc && np > 0)          /* boids flee: predators as moving disks */
            rc = orc_flock_obstacle_energy_grad(n, pos, theta, box, np, ppos, rfl, ppar[0], par[6], NULL, gR, gth);
        if (!rc && np > 0) {        /* predators chase, and avoid the obstacles */
            rc = orc_predator_energy_grad(n, pos, box, np, ppos, pth, ppar[2], ppar[3], NULL, qR, qth);
            for (int p = 0; p < np; ++p) { p3[3 * p] = ppos[2 * p]; p3[3 * p + 1] = ppos[2 * p + 1]; p3[3 * p + 2] = 0.0; }
            if (!rc && g_nobs > 0)
                rc = orc_flock_obstacle_energy_grad(np, p3, pth, box, g_nobs, g_obs_centre, g_obs_radius, g_obs_J,
                                                    par[6], NULL, qR, qth);
        }
        for (int i = 0; i < n && !rc; ++i) {
            const double c = cos(theta[i]), sn = sin(theta[i]);
            pos[3 * (size_t)i] = wrap64(pos[3 * (size_t)i] + dt * (speed * c - gR[2 * i]), box[0]);
            pos[3 * (size_t)i + 1] = wrap64(pos[3 * (size_t)i + 1] + dt * (speed * sn - gR[2 * i + 1]), box[1]);
            theta[i] -= dt * gth[i];
        }
        for (int p = 0; p < np && !rc; ++p) {
            const double c = cos(pth[p]), sn = sin(pth[p]);
            ppos[2 * p] = wrap64(ppos[2 * p] + dt * (ppar[4] * c - qR[2 * p]), box[0]);
            ppos[2 * p + 1] = wrap64(ppos[2 * p + 1] + dt * (ppar[4] * sn - qR[2 * p + 1]), box[1]);
            pth[p] -= dt * qth[p];
        }
    }
    free(gR); free(gth);
    return rc;
}

/*
 * orc_flock_run: forward Euler (eqs. 4-5): R_i' = mu(R_i, dt (v N(theta_i) - grad_{R_i} E)),
 * theta_i' = theta_i - dt grad_{theta_i} E, both from the state at the start of the step.
 */
int orc_flock_run(int n, double *pos, double *theta, const double *box, const double *par, double speed,
                  double dt, int nsteps)
{
    double *gR = (double *)malloc((size_t)n * 2 * sizeof(double)), *gth = (double *)malloc((size_t)n * sizeof(double));
    if (!gR || !gth) { free(gR); free(gth); return ORC_ENOMEM; }
    int rc = ORC_OK;
    for (int s = 0; s < nsteps && !rc; ++s) {
        rc = orc_flock_energy_grad(n, pos, theta, box, par, NULL, gR, gth);
        if (!rc && g_nobs > 0)
            rc = orc_flock_obstacle_energy_grad(n, pos, theta, box, g_nobs, g_obs_centre, g_obs_radius, g_obs_J,
                                                par[6], NULL, gR, gth);
        for (int i = 0; i < n && !rc; ++i) {
            const double c = cos(theta[i]), sn = sin(theta[i]);
            pos[3 * (size_t)i] = wrap64(pos[3 * (size_t)i] + dt * (speed * c - gR[2 * i]), box[0]);
            pos[3 * (size_t)i + 1] = wrap64(pos[3 * (size_t)i + 1] + dt * (speed * sn - gR[2 * i + 1]), box[1]);
            theta[i] -= dt * gth[i];
        }
    }
    free(gR); free(gth);
    return rc;
}
