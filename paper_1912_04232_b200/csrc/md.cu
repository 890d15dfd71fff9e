// md.cu -- host side of libmd_b200: the C ABI declared in include/md.h.
// Argument checking, workspace carving, kernel launches and the CUDA-graph step loop.
// Every step of the path runs in the kernels of md_kernels.cuh; there is no CPU fallback.
#include "md.h"
#include "md_kernels.cuh"
#include "md_force32.cuh"
#include "md_nbr2.cuh"
#include "md_fire.cuh"
#include "md_brownian.cuh"
#include "md_nh.cuh"
#include "md_flock.cuh"

#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <mutex>
#include <new>

using namespace mdk;

// Scratch of md_cell_list_static: part of the library image, so every GPU that loads the library holds these
// 832 KB until the process exits.  Layout in ints: cell_of[MAX_N] | rank[MAX_N] | perm_tmp[MAX_N] |
// cell_count[MAX_CELLS].  In HOST code this name is a host-side stand-in, not a device address: the address
// the kernels get comes from cudaGetSymbolAddress (static_scratch_address below), once per device.
static __device__ __align__(256) int g_cell_static_scratch[3 * MD_STATIC_MAX_N + MD_STATIC_MAX_CELLS];
static_assert(MD_STATIC_MAX_CELLS <= SCAN_ONE_BLOCK, "md_cell_list_static scans its cells with the one-block kernel");

namespace {

thread_local char g_err[512] = "";

int fail(int code, const char *fmt, ...) {
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_err, sizeof(g_err), fmt, ap);
    va_end(ap);
    return code;
}

#define CU(call)                                                                        \
    do {                                                                                \
        cudaError_t e_ = (call);                                                        \
        if (e_ != cudaSuccess)                                                          \
            return fail(MD_ECUDA, "%s: %s (%s:%d)", #call, cudaGetErrorString(e_),      \
                        __FILE__, __LINE__);                                            \
    } while (0)

#define LAUNCH_OK()                                                                     \
    do {                                                                                \
        cudaError_t e_ = cudaGetLastError();                                            \
        if (e_ != cudaSuccess)                                                          \
            return fail(MD_ECUDA, "kernel launch: %s (%s:%d)", cudaGetErrorString(e_),  \
                        __FILE__, __LINE__);                                            \
    } while (0)

constexpr size_t ALIGN = 256;
size_t up(size_t x) { return (x + ALIGN - 1) / ALIGN * ALIGN; }
bool aligned16(const void *p) { return (reinterpret_cast<uintptr_t>(p) & 15u) == 0; }
int blocks_for(long long threads, int block = 256) { return (int)((threads + block - 1) / block); }

enum { RULE_FIRE = 1, RULE_BROWNIAN, RULE_LANGEVIN, RULE_NH, RULE_FLOCK };

// Everything one step of an update rule other than NVE depends on (plain data, compared bytewise
// to decide whether the cached graphs still apply).
struct RuleArgs {
    int rule;
    void *pos, *vel, *force, *state;
    int *id, *nbr_idx, *nbr_count, *stats;
    md_potential pot;
    float dt, mass, gamma, kT, tau;
    unsigned seed, step0;
    md_fire_params fire;
    md_flock_params flock;
    int nobs;                       // md_flock_obstacles: disks (x, y, radius) and J
    float obs[3 * MD_MAX_OBSTACLES], J_obs;
    int npred;                      // md_flock_predators
    void *pred;
    md_predator_params ppar;
    int nh_chain;                   // Nose-Hoover chain length
    int fast32, builder, nb_parts, remap;
    float est_thr;
};

struct StepKey {
    const void *pos, *vel, *force, *id, *nbr_idx, *nbr_count, *stats;
    float dt, mass;
    md_potential pot;
    int tpp, fast32, builder, fused;
    float est_thr;
};

} // namespace

struct md_system {
    md_config cfg;
    int n;
    int device;          // CUDA device that owns the workspace
    Geom g;
    char *ws;
    size_t ws_bytes;
    // workspace slices
    int *words;          // [0] rebuild flag (even steps of a fused graph), [1..2] internal status,
                         // [3] rebuild flag (odd steps), [8..15] counters
    int *scan_tmp;       // block sums + ticket of the two-launch cell scan
    double *fire_tmp;    // md_fire_minimize: per-block partial sums, then {c1, c2} as floats
    double *pred_tmp;    // md_flock_predators: per-chunk partial sums (D_x, D_y, count)
    int *cell_count, *cell_start_i, *perm_i, *cell_of, *rank_tmp, *perm_tmp, *id_s;
    float4 *pos_s, *vel_s, *ref_pos, *pos_alt;   // pos_alt: second position buffer of the fused step
    // tuning
    int tpp;             // lanes per particle in the force kernel (1, 2, 4)
    int nb_warps;        // tiles per block in the neighbor-list builder
    size_t nb_smem;      // its dynamic shared memory per block
    int use_graph;
    int fused;           // fused step: the force kernel also opens the next step (graph mode, fast32)
    int remap;           // force kernel: block -> tile remap period (the SM count), 0 = off
    int nb_parts;        // builder: warps per tile (0 = by system size, 1, 2, 4)
    int flagged;         // the rebuild of the step loops as flagged launches instead of an IF node: -1 by size, 0, 1
    int fork;            // fused loop: the flagged rebuild + its own force launch on a branch beside the force kernel
    cudaEvent_t ev_fork, ev_join;
    int cell_coop;       // cell list as one cooperative launch with this many blocks at most (0: five kernels)
    int cell_coop_max;   // what the device allows
    int ns;              // md_set_species_lj: number of species and the tables (row-major)
    float sp_eps[16], sp_sig[16], sp_rc[16];
    int bks_ns;          // md_set_species_bks: A, B, C per species pair, charges, DSF damping, Coulomb constant
    float bks_A[16], bks_B[16], bks_C[16], bks_q[4], bks_alpha, bks_ke;
    int nobs;            // md_flock_obstacles
    float obs[3 * MD_MAX_OBSTACLES], J_obs;
    int r0, r1;          // md_set_range: the particles [r0, r1) this context builds rows and forces for
    int nh_chain;        // option "nh_chain": thermostats in the Nose-Hoover chain (1..8)
    int npred;           // md_flock_predators: count, DEVICE state (caller's), parameters
    void *pred;
    md_predator_params ppar;
    int builder;         // neighbor-list builder: 2 = bit-mask (md_nbr2.cuh), 1 = column append
    int fast32;          // LJ 3-D: fp32 fast path + fp64 re-evaluation (md_force32.cuh)
    float est_thr;       // its error-estimate threshold
    // graph cache of md_nve_step
    cudaStream_t cap_stream, body_stream;
    StepKey key;
    bool key_valid;
    cudaGraphExec_t exec1, execU;
    int unroll;
    // graph cache of the other update rules (FIRE, Brownian, Langevin, Nose-Hoover)
    RuleArgs rule_key;
    bool rule_key_valid;
    cudaGraphExec_t rule_exec1, rule_execU;
};

namespace {

// The library links its own (static) CUDA runtime: every ABI call makes the device that owns the
// workspace current on the calling thread for its duration and puts the caller's device back on return.
struct DeviceScope {
    int prev, rc;
    explicit DeviceScope(int device) : prev(-1), rc(MD_OK) {
        cudaError_t e = cudaGetDevice(&prev);
        if (e == cudaSuccess && prev != device) e = cudaSetDevice(device); else if (e == cudaSuccess) prev = -1;
        if (e != cudaSuccess) { prev = -1; rc = fail(MD_ECUDA, "selecting device %d: %s", device, cudaGetErrorString(e)); }
    }
    ~DeviceScope() { if (prev >= 0) cudaSetDevice(prev); }
    DeviceScope(const DeviceScope &) = delete;
    DeviceScope &operator=(const DeviceScope &) = delete;
};
static_assert(sizeof(md_potential) == 24 && sizeof(md_fire_params) == 28 && sizeof(md_flock_params) == 32 &&
              sizeof(md_predator_params) == 20, "graph keys are compared bytewise: these structs hold no padding");

// Device address of g_cell_static_scratch on `device`, resolved once per device with that device current
// (the caller holds a DeviceScope on it).
constexpr int STATIC_MAX_DEVICES = 64;
std::mutex g_static_mu;
int *g_static_addr[STATIC_MAX_DEVICES];
int static_scratch_address(int device, int **out) {
    if (device < 0 || device >= STATIC_MAX_DEVICES) return fail(MD_EINVAL, "device ordinal %d out of range", device);
    std::lock_guard<std::mutex> lock(g_static_mu);
    if (!g_static_addr[device]) {
        void *p = nullptr;
        CU(cudaGetSymbolAddress(&p, g_cell_static_scratch));
        if (!p) return fail(MD_ECUDA, "cudaGetSymbolAddress returned a null address on device %d", device);
        g_static_addr[device] = static_cast<int *>(p);
    }
    *out = g_static_addr[device];
    return MD_OK;
}

struct Layout {
    size_t words, scan_tmp, fire_tmp, pred_tmp, cell_count, cell_start_i, perm_i, cell_of, rank_tmp, perm_tmp, id_s, pos_s,
        vel_s, ref_pos, pos_alt, total;
};

Layout layout(int n, long long cells) {
    Layout l;
    size_t o = 0;
    auto take = [&](size_t bytes) { size_t at = o; o += up(bytes); return at; };
    l.words = take(64 * sizeof(int));
    l.scan_tmp = take((size_t)std::max<long long>((cells + SCAN_CHUNK - 1) / SCAN_CHUNK + 2, 4096) * sizeof(int));   // also the cooperative cell list's block sums
    l.fire_tmp = take(((size_t)(n + FIRE_BLOCK - 1) / FIRE_BLOCK * 3 + 2) * sizeof(double));
    l.pred_tmp = take((size_t)FLOCK_PRED_CHUNKS * MD_MAX_PREDATORS * 3 * sizeof(double));
    l.cell_count = take((size_t)(cells + 4) * sizeof(int));
    l.cell_start_i = take((size_t)(cells + 1) * sizeof(int));
    l.perm_i = take((size_t)n * sizeof(int));
    l.cell_of = take((size_t)n * sizeof(int));
    l.rank_tmp = take((size_t)n * sizeof(int));
    l.perm_tmp = take((size_t)n * sizeof(int));
    l.id_s = take((size_t)n * sizeof(int));
    l.pos_s = take((size_t)n * sizeof(float4));
    l.vel_s = take((size_t)n * sizeof(float4));
    l.ref_pos = take((size_t)n * sizeof(float4));
    l.pos_alt = take((size_t)n * sizeof(float4));
    l.total = o;
    return l;
}

// Validates cfg and fills the geometry.
int make_geom(const md_config *cfg, int n, Geom *g) {
    if (!cfg) return fail(MD_EINVAL, "cfg is NULL");
    if (n <= 0) return fail(MD_EINVAL, "n = %d must be positive", n);
    if (cfg->dim != 2 && cfg->dim != 3) return fail(MD_EINVAL, "dim = %d must be 2 or 3", cfg->dim);
    if (cfg->capacity <= 0 || cfg->capacity % 4) return fail(MD_EINVAL, "capacity = %d must be a positive multiple of 4", cfg->capacity);
    if (!(cfg->r_cut > 0.0f)) return fail(MD_EINVAL, "r_cut must be positive");
    if (!(cfg->skin >= 0.0f)) return fail(MD_EINVAL, "skin must be non-negative");
    memset(g, 0, sizeof(*g));
    g->dim = cfg->dim; g->n = n; g->ntot = n; g->capacity = cfg->capacity;
    const float R = cfg->r_cut + cfg->skin;              // fl32(r_cut + skin)
    g->R2 = R * R;
    const float hs = cfg->skin * 0.5f;
    g->half_skin2 = hs * hs;
    g->face = R + cfg->skin;
    long long cells = 1;
    for (int k = 0; k < 3; ++k) {
        g->nc[k] = 1; g->L[k] = 1.0f; g->h[k] = 0.5f; g->inv_cell[k] = 1.0f; g->inv_L[k] = 1.0f;
        if (k >= cfg->dim) continue;
        const float L = cfg->box[k];
        if (!(L > 0.0f) || !std::isfinite(L)) return fail(MD_EINVAL, "box[%d] must be positive", k);
        const int nk = (int)std::floor((double)L / (double)R);
        if (nk < 3) return fail(MD_EBOX, "box[%d] = %g holds %d cells of side >= %g; need >= 3", k, L, nk, R);
        if ((double)L / nk - (double)R < 1e-5 * (double)L)
            return fail(MD_EBOX, "box[%d] = %g: cell side %.9g exceeds R = %.9g by less than 1e-5 L", k, L, (double)L / nk, (double)R);
        g->nc[k] = nk; g->L[k] = L; g->h[k] = L / 2.0f;
        g->inv_cell[k] = (float)nk / L;
        g->inv_L[k] = 1.0f / L;
        cells *= nk;
    }
    if (cells > 0x7fffffffLL / 2) return fail(MD_EINVAL, "too many cells");
    g->cells = (int)cells;
    return MD_OK;
}

int make_pair(const md_system *sys, const md_potential *pot, Pair *pp) {
    if (!pot) return fail(MD_EINVAL, "potential is NULL");
    if (pot->kind != MD_KIND_LJ && pot->kind != MD_KIND_SOFT && pot->kind != MD_KIND_MORSE &&
        pot->kind != MD_KIND_BUCKINGHAM && pot->kind != MD_KIND_LJ_SPECIES && pot->kind != MD_KIND_BKS)
        return fail(MD_EINVAL, "unknown potential kind %d", pot->kind);
    if (pot->kind != MD_KIND_LJ_SPECIES && pot->kind != MD_KIND_BKS && !(pot->epsilon > 0.0f))
        return fail(MD_EINVAL, "epsilon must be positive");
    memset(pp, 0, sizeof(*pp));
    pp->kind = pot->kind;
    pp->deps = (double)pot->epsilon;
    if (pot->kind == MD_KIND_LJ) {
        if (!(pot->r_cut > 0.0f) || !(pot->sigma > 0.0f)) return fail(MD_EINVAL, "LJ needs sigma > 0 and r_cut > 0");
        if (pot->r_cut > sys->cfg.r_cut) return fail(MD_EINVAL, "potential r_cut %g exceeds the list r_cut %g", pot->r_cut, sys->cfg.r_cut);
        const double s = pot->sigma, rc = pot->r_cut;
        pp->dsig6x2 = 2.0 * std::pow(s, 6.0); pp->drc2 = rc * rc;
        const double s6 = std::pow(s / rc, 6.0);
        pp->du_cut4 = pot->shift ? (s6 * s6 - s6) : 0.0;
    } else if (pot->kind == MD_KIND_MORSE) {
        if (!(pot->r_cut > 0.0f) || !(pot->sigma > 0.0f) || !(pot->alpha > 0.0f))
            return fail(MD_EINVAL, "Morse needs sigma (r0) > 0, alpha > 0 and r_cut > 0");
        if (pot->r_cut > sys->cfg.r_cut) return fail(MD_EINVAL, "potential r_cut %g exceeds the list r_cut %g", pot->r_cut, sys->cfg.r_cut);
        const double rc = pot->r_cut, x = std::exp(-(double)pot->alpha * (rc - (double)pot->sigma));
        pp->dalpha = pot->alpha; pp->dr0 = pot->sigma; pp->drc2 = rc * rc; pp->dsig6x2 = 2.0;
        pp->du_cutm = pot->shift ? ((1.0 - x) * (1.0 - x) - 1.0) : 0.0;
    } else if (pot->kind == MD_KIND_LJ_SPECIES) {
        if (sys->ns < 1) return fail(MD_EINVAL, "MD_KIND_LJ_SPECIES needs md_set_species_lj first");
        pp->ns = sys->ns; pp->dsig6x2 = 2.0; pp->drc2 = 0.0;
        for (int t = 0; t < sys->ns * sys->ns; ++t) {
            const double e = sys->sp_eps[t], sg = sys->sp_sig[t], rc = sys->sp_rc[t];
            if (rc > sys->cfg.r_cut) return fail(MD_EINVAL, "species r_cut %g exceeds the list r_cut %g", rc, sys->cfg.r_cut);
            const double s6 = std::pow(sg, 6.0), q6 = std::pow(sg / rc, 6.0);
            pp->sp_sig6x2[t] = 2.0 * s6; pp->sp_fs[t] = 24.0 * e * s6; pp->sp_es[t] = 2.0 * e;
            pp->sp_rc2[t] = rc * rc; pp->sp_ucut4[t] = pot->shift ? (q6 * q6 - q6) : 0.0;
        }
    } else if (pot->kind == MD_KIND_BKS) {
        if (sys->bks_ns < 1) return fail(MD_EINVAL, "MD_KIND_BKS needs md_set_species_bks first");
        if (!(pot->r_cut > 0.0f) || pot->r_cut > sys->cfg.r_cut)
            return fail(MD_EINVAL, "potential r_cut %g must be positive and at most the list r_cut %g", pot->r_cut, sys->cfg.r_cut);
        const double rc = pot->r_cut, a = sys->bks_alpha;
        pp->ns = sys->bks_ns; pp->dsig6x2 = 2.0; pp->drc2 = rc * rc;
        for (int t = 0; t < sys->bks_ns * sys->bks_ns; ++t) {
            const double A = sys->bks_A[t], B = sys->bks_B[t], Cc = sys->bks_C[t];
            pp->sp_sig6x2[t] = A; pp->sp_fs[t] = B; pp->sp_es[t] = Cc;
            pp->sp_rc2[t] = (double)sys->bks_ke * (double)sys->bks_q[t / sys->bks_ns] * (double)sys->bks_q[t % sys->bks_ns];
            pp->sp_ucut4[t] = pot->shift ? (A * std::exp(-B * rc) - Cc / std::pow(rc, 6.0)) : 0.0;
        }
        pp->bks_a = a; pp->bks_tsp = 2.0 * a / std::sqrt(3.14159265358979323846);
        pp->bks_ec = std::erfc(a * rc) / rc;
        pp->bks_fc = pp->bks_ec / rc + pp->bks_tsp * std::exp(-a * a * rc * rc) / rc;
        pp->bks_rc = rc;
    } else if (pot->kind == MD_KIND_BUCKINGHAM) {
        if (!(pot->r_cut > 0.0f) || !(pot->sigma >= 0.0f) || !(pot->alpha > 0.0f))
            return fail(MD_EINVAL, "Buckingham needs alpha (B) > 0, sigma (C) >= 0 and r_cut > 0");
        if (pot->r_cut > sys->cfg.r_cut) return fail(MD_EINVAL, "potential r_cut %g exceeds the list r_cut %g", pot->r_cut, sys->cfg.r_cut);
        const double rc = pot->r_cut;
        pp->dA = pot->epsilon; pp->dalpha = pot->alpha; pp->dC = pot->sigma; pp->drc2 = rc * rc; pp->dsig6x2 = 2.0;
        pp->du_cutm = pot->shift ? (pp->dA * std::exp(-pp->dalpha * rc) - pp->dC / std::pow(rc, 6.0)) : 0.0;
    } else {
        pp->dsig6x2 = 2.0; pp->drc2 = 1e300;
    }
    return MD_OK;
}

// ------------------------------------------------------------------ launch helpers ------

int launch_cell_build(md_system *s, float4 *pos, float4 *vel, int *id, int *cell_start,
                      int *perm, int *status, const int *cond, cudaStream_t st, bool cooperative = false) {
    const Geom &g = s->g;
    const int nb = blocks_for(g.n);
    const bool resort = s->cfg.resort != 0;
    const int coop = cooperative ? s->cell_coop_max : s->cell_coop;
    if (coop > 0) {
        // one cooperative launch (grid-wide barriers between the phases); needs every block resident
        const int grid = std::min(nb, coop);
        Geom gg = g;
        float4 *velp = (resort && vel) ? vel : nullptr, *vel_s = (resort && vel) ? s->vel_s : nullptr;
        int *idp = id, *id_s = (resort && id) ? s->id_s : nullptr;
        int *cell_of = s->cell_of, *rank_tmp = s->rank_tmp, *cell_count = s->cell_count, *perm_tmp = s->perm_tmp;
        float4 *pos_s = s->pos_s;
        int *block_sum = s->scan_tmp;
        int rs = resort ? 1 : 0;
        void *args[] = {&gg, &pos, &velp, &idp, &cell_of, &rank_tmp, &cell_count, &cell_start, &perm_tmp, &perm,
                        &pos_s, &vel_s, &id_s, &block_sum, &status, &cond, &rs};
        CU(cudaLaunchCooperativeKernel((const void *)k_cell_all, dim3(grid), dim3(256), args, 0, st));
        return MD_OK;
    }
    k_cell_assign<<<nb, 256, 0, st>>>(g, pos, s->cell_of, s->rank_tmp, s->cell_count, cond);
    LAUNCH_OK();
    if (g.cells <= SCAN_ONE_BLOCK) {
        k_cell_scan<<<1, 1024, 0, st>>>(g.cells, s->cell_count, cell_start, status, cond);
        LAUNCH_OK();
    } else {
        const int nbs = (g.cells + SCAN_CHUNK - 1) / SCAN_CHUNK;
        k_cell_sum<<<nbs, 1024, 0, st>>>(g.cells, s->cell_count, s->scan_tmp, s->scan_tmp + nbs + 1, status, cond);
        LAUNCH_OK();
        k_cell_scan2<<<nbs, 1024, 0, st>>>(g.cells, s->cell_count, cell_start, s->scan_tmp, cond);
        LAUNCH_OK();
    }
    k_cell_scatter<<<nb, 256, 0, st>>>(g.n, s->cell_of, s->rank_tmp, cell_start, s->perm_tmp, cond);
    LAUNCH_OK();
    k_cell_order_gather<<<nb, 256, 0, st>>>(g.n, s->cell_of, cell_start, s->perm_tmp, id, pos,
                                            (resort && vel) ? vel : nullptr, perm, s->pos_s,
                                            (resort && vel) ? s->vel_s : nullptr,
                                            (resort && id) ? s->id_s : nullptr, cond);
    LAUNCH_OK();
    if (resort) {
        k_copy_back<<<nb, 256, 0, st>>>(g.n, s->pos_s, s->vel_s, s->id_s, pos, vel, id, cond);
        LAUNCH_OK();
    }
    return MD_OK;
}

int launch_nbr_build(md_system *s, const float4 *spos, const int *cell_start, const int *map,
                     int *nbr_idx, int *nbr_count, int *status, const int *cond, int incremental,
                     cudaStream_t st) {
    const Geom &g = s->g;
    const int ntiles = (g.n + TILE - 1) / TILE;
    if (s->builder == 2) {          // bit-mask builder (md_nbr2.cuh)
        // warps per tile: small systems wait for the latency of one tile, large ones for throughput
        int parts = s->nb_parts;
        // measured (nbr build, us): 864 particles 58 / 39 / 33 for 1 / 2 / 4 warps per tile, 32k 62 / 48 / 44,
        // 256k 151 / 200 / 182, 1M 414 / 662 / 618: sharing pays only while the GPU is not full
        if (parts == 0) parts = ntiles <= 2048 ? 4 : 1;
        const int tpb = NB2_WARPS / parts;
        const int tile0 = s->r0 / TILE, tile1 = (s->r1 + TILE - 1) / TILE;          // md_set_range
        const int nb = std::max(1, (tile1 - tile0 + tpb - 1) / tpb);
        const int threads = NB2_WARPS * 32;
        const size_t sm = NB2_WARPS * sizeof(Nb2Warp);
#define MD_NB2_LAUNCH(D, M, P) k_nbr_build2<D, M, P><<<nb, threads, sm, st>>>(g, spos, cell_start, map, nbr_idx, nbr_count, status, s->ref_pos, cond, incremental, tile0, tile1)
#define MD_NB2_PARTS(D, M) do { if (parts == 4) MD_NB2_LAUNCH(D, M, 4); else if (parts == 2) MD_NB2_LAUNCH(D, M, 2); else MD_NB2_LAUNCH(D, M, 1); } while (0)
        if (g.dim == 3) { if (map) MD_NB2_PARTS(3, true); else MD_NB2_PARTS(3, false); }
        else { if (map) MD_NB2_PARTS(2, true); else MD_NB2_PARTS(2, false); }
#undef MD_NB2_PARTS
#undef MD_NB2_LAUNCH
        LAUNCH_OK();
        return MD_OK;
    }
    if (s->r0 != 0 || s->r1 != g.n) return fail(MD_EINVAL, "md_set_range needs the bit-mask builder (builder = 2)");
    const int nb = (ntiles + s->nb_warps - 1) / s->nb_warps;
    const int threads = s->nb_warps * 32;
    if (g.dim == 3) {
        if (map) k_nbr_build<3, true><<<nb, threads, s->nb_smem, st>>>(g, spos, cell_start, map, nbr_idx, nbr_count, status, s->ref_pos, cond);
        else k_nbr_build<3, false><<<nb, threads, s->nb_smem, st>>>(g, spos, cell_start, map, nbr_idx, nbr_count, status, s->ref_pos, cond);
    } else {
        if (map) k_nbr_build<2, true><<<nb, threads, s->nb_smem, st>>>(g, spos, cell_start, map, nbr_idx, nbr_count, status, s->ref_pos, cond);
        else k_nbr_build<2, false><<<nb, threads, s->nb_smem, st>>>(g, spos, cell_start, map, nbr_idx, nbr_count, status, s->ref_pos, cond);
    }
    LAUNCH_OK();
    return MD_OK;
}

template <int KIND, int DIM, bool ENERGY>
int launch_force_t(md_system *s, const Pair &pp, const float4 *pos, const int *nbr_idx,
                   const int *nbr_count, float4 *force, float4 *vel, float a, double *etot,
                   Book book, cudaStream_t st) {
    Geom g = s->g;
    g.n = s->r1;                    // md_set_range: particles [r0, r1) of this context
    const int m = s->r1 - s->r0;
    if (s->tpp == 0) {          // streaming kernel: one lane per particle, one warp per list tile
        k_force_stream<KIND, DIM, ENERGY><<<blocks_for(m, FS_WARPS * 32), FS_WARPS * 32, 0, st>>>(
            g, pp, pos, nbr_idx, nbr_count, force, vel, a, etot, book, s->r0);
        LAUNCH_OK();
        return MD_OK;
    }
    const int nb = blocks_for((long long)m * s->tpp, 128);
#define MD_FORCE_CASE(T)                                                                       \
    case T:                                                                                    \
        k_force<KIND, DIM, T, ENERGY><<<nb, 128, 0, st>>>(g, pp, pos, nbr_idx, nbr_count,     \
                                                          force, vel, a, etot, book, s->r0);  \
        break;
    switch (s->tpp) {
        MD_FORCE_CASE(1) MD_FORCE_CASE(2) MD_FORCE_CASE(4)
    default: return fail(MD_EINVAL, "threads per particle %d", s->tpp);
    }
#undef MD_FORCE_CASE
    LAUNCH_OK();
    return MD_OK;
}

// ---- the rebuild inside a step loop
// Captured in a graph, the rebuild is either the body of an IF node that the drift raises, or launches that
// are part of every step and return at once while the step's device flag is 0.  Measured on B200 (a lattice at
// rest, 256,000 particles, no rebuild ever fires): a step costs 39.6 us without any rebuild machinery, 48.7 us
// with the IF node (9 us whether or not it fires), 42.3 us with one cooperative kernel that returns at once
// and 2.7-3.0 us more per further kernel.  So where the cooperative cell list keeps up with its five kernels
// (at 1M particles it is 24 us slower per rebuild, more than the launches save) the rebuild is TWO flagged
// launches, cooperative cell list and builder, and no IF node.
constexpr int FLAGGED_MAX_N = 600000;
bool rebuild_is_flagged(const md_system *s) {
    if (s->flagged == 0 || !(s->cell_coop_max > 0)) return false;
    return s->flagged > 0 || s->g.n <= FLAGGED_MAX_N;
}
// flag: device word; the launches do nothing while it is 0
int launch_rebuild_flagged(md_system *s, float4 *pos, float4 *vel, int *id, int *nbr_idx, int *nbr_count,
                           const int *flag, cudaStream_t st) {
    int *status = s->words + 1;
    const bool resort = s->cfg.resort != 0;
    int rc = launch_cell_build(s, pos, vel, id, s->cell_start_i, s->perm_i, status, flag, st, rebuild_is_flagged(s));
    if (rc) return rc;
    return launch_nbr_build(s, resort ? pos : s->pos_s, s->cell_start_i, resort ? nullptr : s->perm_i,
                            nbr_idx, nbr_count, status, flag, 1, st);
}

// The kinds md_force32.cuh serves (3-D only): fp32 pair math, error estimate, fp64 re-evaluation.
static bool fast32_kind(const md_system *s, const Pair &pp) {
    return s->fast32 && s->g.dim == 3 &&
           (pp.kind == MD_KIND_LJ || pp.kind == MD_KIND_MORSE || pp.kind == MD_KIND_BUCKINGHAM);
}

// want_energy: also e_i into force.w (and the fp64 total when etot != NULL); the step loop
// does not need it and skips those fp64 operations (force.w = 0 there).
int launch_force(md_system *s, const Pair &pp, const float4 *pos, const int *nbr_idx,
                 const int *nbr_count, float4 *force, float4 *vel, float a, double *etot,
                 bool want_energy, Book book, cudaStream_t st, NextStep nx = NextStep()) {
    if (fast32_kind(s, pp)) {
        Pair32 q;
        memset(&q, 0, sizeof(q));
        q.rc2 = (float)pp.drc2;
        q.sig6x2 = (float)pp.dsig6x2;
        q.ucut4 = (float)pp.du_cut4;
        q.fscale = (float)(12.0 * pp.deps * pp.dsig6x2);
        q.escale = (float)(2.0 * pp.deps);
        q.near_band = 1e-5f * q.rc2;
        q.est_thr = s->est_thr;
        if (pp.kind == MD_KIND_MORSE) {
            const double k = -pp.dalpha * 1.4426950408889634;
            q.k_hi = (float)k; q.k_lo = (float)(k - (double)q.k_hi); q.s_unit = 0.022f;
            q.m_r0 = (float)pp.dr0; q.m_2a = (float)(2.0 * pp.dalpha); q.m_a = (float)pp.dalpha;
            q.ucut4 = (float)pp.du_cutm; q.fscale = (float)pp.deps; q.escale = (float)(0.5 * pp.deps);
        } else if (pp.kind == MD_KIND_BUCKINGHAM) {
            const double k = -pp.dalpha * 1.4426950408889634;
            q.k_hi = (float)k; q.k_lo = (float)(k - (double)q.k_hi); q.s_unit = 0.0175f;
            q.b_A = (float)pp.dA; q.b_B = (float)pp.dalpha; q.b_C = (float)pp.dC;
            q.ucut4 = (float)pp.du_cutm; q.fscale = 1.0f; q.escale = 0.5f;
        }
        Geom gr = s->g;
        gr.n = s->r1;                                  // md_set_range: lanes beyond r1 are idle
        const int nb = blocks_for(s->r1 - s->r0, F32_WARPS * 32);
        int *nfix = s->words + 8;
        int P = 0, grid = nb;
        if (s->remap > 0 && nb > 4 * s->remap) { P = s->remap; grid = P * ((nb + P - 1) / P); }
#define MD_F32_CASE(K)                                                                                      \
    case K:                                                                                                 \
        if (want_energy) k_force32<K, true><<<grid, F32_WARPS * 32, 0, st>>>(gr, pp, q, pos, nbr_idx, nbr_count, force, vel, a, etot, book, nfix, nx, P, nb, s->r0); \
        else k_force32<K, false><<<grid, F32_WARPS * 32, 0, st>>>(gr, pp, q, pos, nbr_idx, nbr_count, force, vel, a, etot, book, nfix, nx, P, nb, s->r0); \
        break;
        switch (pp.kind) { MD_F32_CASE(0) MD_F32_CASE(2) MD_F32_CASE(3) }
#undef MD_F32_CASE
        LAUNCH_OK();
        return MD_OK;
    }
#define MD_FORCE_DISPATCH(K, D)                                                                 \
    (want_energy ? launch_force_t<K, D, true>(s, pp, pos, nbr_idx, nbr_count, force, vel, a,   \
                                              etot, book, st)                                  \
                 : launch_force_t<K, D, false>(s, pp, pos, nbr_idx, nbr_count, force, vel, a,  \
                                               etot, book, st))
    if (pp.kind == MD_KIND_LJ) return s->g.dim == 3 ? MD_FORCE_DISPATCH(0, 3) : MD_FORCE_DISPATCH(0, 2);
    if (pp.kind == MD_KIND_MORSE) return s->g.dim == 3 ? MD_FORCE_DISPATCH(2, 3) : MD_FORCE_DISPATCH(2, 2);
    if (pp.kind == MD_KIND_LJ_SPECIES) return s->g.dim == 3 ? MD_FORCE_DISPATCH(4, 3) : MD_FORCE_DISPATCH(4, 2);
    if (pp.kind == MD_KIND_BUCKINGHAM) return s->g.dim == 3 ? MD_FORCE_DISPATCH(3, 3) : MD_FORCE_DISPATCH(3, 2);
    if (pp.kind == MD_KIND_BKS) return s->g.dim == 3 ? MD_FORCE_DISPATCH(5, 3) : MD_FORCE_DISPATCH(5, 2);
    return s->g.dim == 3 ? MD_FORCE_DISPATCH(1, 3) : MD_FORCE_DISPATCH(1, 2);
#undef MD_FORCE_DISPATCH
}

__global__ void k_init_stats(int *stats, int *words) {
    stats[0] = 0; stats[1] = 0; stats[2] = -1; stats[3] = 0;
    words[0] = 0; words[3] = 0;          // rebuild flags
    words[5] = 0; words[6] = 0; words[7] = 0;      // and those of the forked fused loop
}

// the noise stream of a stochastic rule: {seed, step0} as device words ([20], [21])
__global__ void k_set_noise(int *words, unsigned seed, unsigned step0) {
    words[20] = (int)seed; words[21] = (int)step0;
}

__global__ void k_unpermute(int n, const int *__restrict__ id, const float4 *__restrict__ a,
                            const float4 *__restrict__ b, const float4 *__restrict__ c,
                            float4 *__restrict__ ao, float4 *__restrict__ bo, float4 *__restrict__ co) {
    int s = blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= n) return;
    int i = id[s];
    ao[i] = a[s]; bo[i] = b[s]; co[i] = c[s];
}

// ---- slab decomposition: exact coordinate translations between a rank's local frame and the box
__device__ __forceinline__ float slab_to_local(const md_slab_frame &f, float x) {
    if (f.kind == 0) return x >= f.g2l_thr ? (x - f.L) + f.Lx : x;
    if (f.kind == 2) return x < f.g2l_thr ? x : x - f.T;
    return x - f.T;
}
__device__ __forceinline__ float slab_to_global(const md_slab_frame &f, float x) {
    float g;
    if (f.kind == 0) g = x >= f.l2g_thr ? (x - f.Lx) + f.L : x;
    else if (f.kind == 2) g = x < f.l2g_thr ? x : x + f.T;
    else g = x + f.T;
    return g >= f.L ? 0.0f : g;
}
__global__ void k_slab_convert(md_slab_frame f, float4 *pos, int n, int mode) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    float x = pos[i].x;
    if (mode == 0) x = slab_to_global(f, x);
    else if (mode == 1) x = slab_to_local(f, x);
    else x = slab_to_local(f, slab_to_global(f, x));      // back on the global fp32 grid
    pos[i].x = x;
}
// The opening of a slab rank's step in one kernel: k_kick_drift, then x put back on the global fp32 grid, then
// the half-skin test on that x (differences of local coordinates are differences of global ones).  Does
// nothing while *stop != 0: the host enqueues steps ahead and a stale list has been met (Book::skip).  Halo
// copies (id < 0) are left alone: their positions arrive from their owners, whose own test covers them (a copy
// whose owner has stepped just outside the halo zone has a local x below 0 that must not be wrapped or tested).
template <int DIM>
__global__ void __launch_bounds__(256)
k_slab_kick_drift(Geom g, md_slab_frame f, float4 *__restrict__ pos, float4 *__restrict__ vel,
                  const float4 *__restrict__ force, const float4 *__restrict__ ref, const int *__restrict__ id,
                  float a, float dt, int *flag, const int *stop) {
    if (stop && ld_volatile(stop)) return;
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    bool moved = false;
    if (i < g.n && id[i] >= 0) {
        float4 p = pos[i], v = vel[i];
        const float4 fo = force[i];
        v.x = fmaf(a, fo.x, v.x);
        v.y = fmaf(a, fo.y, v.y);
        p.x = wrap(fmaf(dt, v.x, p.x), g.L[0], g.inv_L[0]);
        p.y = wrap(fmaf(dt, v.y, p.y), g.L[1], g.inv_L[1]);
        if (DIM == 3) {
            v.z = fmaf(a, fo.z, v.z);
            p.z = wrap(fmaf(dt, v.z, p.z), g.L[2], g.inv_L[2]);
        }
        p.x = slab_to_local(f, slab_to_global(f, p.x));
        pos[i] = p; vel[i] = v;
        moved = disp2_from_ref<DIM>(g, p, ref[i]) > g.half_skin2;
    }
    if (__any_sync(FULL, moved) && (threadIdx.x & 31) == 0) *flag = 1;
}

__global__ void k_slab_pack(md_slab_frame f, const float4 *__restrict__ pos, const int *__restrict__ slots, int k,
                            float4 *__restrict__ rows) {
    const int t = blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= k) return;
    float4 p = pos[slots[t]];
    p.x = slab_to_global(f, p.x);
    rows[t] = p;
}
__global__ void k_slab_unpack(md_slab_frame f, const float4 *__restrict__ rows, const int *__restrict__ slots, int k,
                              float4 *__restrict__ pos) {
    const int t = blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= k) return;
    float4 p = rows[t];
    p.x = slab_to_local(f, p.x);
    pos[slots[t]] = p;
}

// ---- slab decomposition: the rebuild (migration, border selection, assembly of the local system, exchange plan)
// Position in a compacted output: one atomic per warp, lanes in order behind it.
__device__ __forceinline__ int slab_take(bool mine, int *counter) {
    const unsigned m = __ballot_sync(FULL, mine);
    const int lane = threadIdx.x & 31;
    int base = 0;
    if (m && lane == __ffs(m) - 1) base = atomicAdd(counter, __popc(m));
    base = __shfl_sync(FULL, base, m ? __ffs(m) - 1 : 0);
    return base + __popc(m & ((1u << lane) - 1u));
}
// counts: {stayers, to previous, to next, errors}
__global__ void k_slab_split(md_slab_frame f, float lo, float hi, const float4 *__restrict__ pos,
                             const float4 *__restrict__ vel, const int *__restrict__ id, int n,
                             float4 *own_pos, float4 *own_vel, int *own_id, float4 *prev_rows, int *prev_ids,
                             float4 *next_rows, int *next_ids, int cap_rows, int *counts) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    const bool owned = i < n && id[i] >= 0;
    float4 p = make_float4(0.f, 0.f, 0.f, 0.f);
    int kind = -1;                                      // 0 stays, 1 to the previous rank, 2 to the next
    if (owned) {
        p = pos[i];
        p.x = slab_to_global(f, p.x);
        if (p.x >= lo && p.x < hi) kind = 0;
        else {
            // the nearer way round the periodic box
            const float up = p.x >= hi ? p.x - hi : (p.x + f.L) - hi;
            const float down = p.x < lo ? lo - p.x : (lo + f.L) - p.x;
            kind = up < down ? 2 : 1;
        }
    }
    const int a = slab_take(kind == 0, counts + 0);
    const int b = slab_take(kind == 1, counts + 1);
    const int c = slab_take(kind == 2, counts + 2);
    if (kind == 0) { own_pos[a] = p; own_vel[a] = vel[i]; own_id[a] = id[i]; }
    else if (kind > 0) {
        const int t = kind == 1 ? b : c;
        if (t >= cap_rows) { atomicAdd(counts + 3, 1); return; }
        float4 *rows = kind == 1 ? prev_rows : next_rows;
        rows[2 * t] = p; rows[2 * t + 1] = vel[i];
        (kind == 1 ? prev_ids : next_ids)[t] = id[i];
    }
}
// migrants join the owned set at [offset, offset + m); one outside [lo, hi) skipped a whole slab: an error
__global__ void k_slab_append(const float4 *__restrict__ rows, const int *__restrict__ ids, int m, float lo, float hi,
                              float4 *own_pos, float4 *own_vel, int *own_id, int offset, int *errors) {
    const int t = blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= m) return;
    const float4 p = rows[2 * t];
    if (!(p.x >= lo && p.x < hi)) atomicAdd(errors, 1);
    own_pos[offset + t] = p; own_vel[offset + t] = rows[2 * t + 1]; own_id[offset + t] = ids[t];
}
// owned particles within the halo width of a face: what the neighbours copy.  counts: {for previous, for next, errors}
__global__ void k_slab_border(float lo_edge, float hi_edge, const float4 *__restrict__ own_pos,
                              const int *__restrict__ own_id, int n_own, float4 *prev_rows, int *prev_ids,
                              float4 *next_rows, int *next_ids, int cap_rows, int *map_prev, int *map_next,
                              int *counts) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    float4 p = make_float4(0.f, 0.f, 0.f, 0.f);
    bool lo_side = false, hi_side = false;
    int gid = 0;
    if (i < n_own) {
        p = own_pos[i]; gid = own_id[i];
        lo_side = p.x < lo_edge; hi_side = p.x >= hi_edge;
    }
    const int a = slab_take(lo_side, counts + 0);
    const int b = slab_take(hi_side, counts + 1);
    if (lo_side) {
        if (a < cap_rows) { prev_rows[a] = p; prev_ids[a] = gid; map_prev[gid] = a; } else atomicAdd(counts + 2, 1);
    }
    if (hi_side) {
        if (b < cap_rows) { next_rows[b] = p; next_ids[b] = gid; map_next[gid] = b; } else atomicAdd(counts + 2, 1);
    }
}
// local system = owned, then the copies from the previous rank, then those from the next; x local
__global__ void k_slab_load(md_slab_frame f, const float4 *__restrict__ own_pos, const float4 *__restrict__ own_vel,
                            const int *__restrict__ own_id, int n_own, const float4 *__restrict__ hp_rows,
                            const int *__restrict__ hp_ids, int h_prev, const float4 *__restrict__ hn_rows,
                            const int *__restrict__ hn_ids, int h_next, float4 *pos, float4 *vel, int *id,
                            int *map_halo) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n_own + h_prev + h_next) return;
    float4 p, v = make_float4(0.f, 0.f, 0.f, 0.f);
    int g;
    if (i < n_own) { p = own_pos[i]; v = own_vel[i]; g = own_id[i]; }
    else {
        const int q = i - n_own;
        if (q < h_prev) { p = hp_rows[q]; g = hp_ids[q]; } else { p = hn_rows[q - h_prev]; g = hn_ids[q - h_prev]; }
        map_halo[g] = q;
        g = -1 - g;
    }
    p.x = slab_to_local(f, p.x);
    pos[i] = p; vel[i] = v; id[i] = g;
}
// after the lists are built: copies take no force (count 0); where every border particle and every copy sits now,
// in the order of the messages; the maps go back to -1
__global__ void k_slab_plan(const int *__restrict__ id, int n, int *nbr_count, int *map_prev, int *map_next,
                            int *map_halo, int *border_prev, int *border_next, int *halo_slots) {
    const int s = blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= n) return;
    const int g = id[s];
    if (g < 0) {
        nbr_count[s] = 0;
        const int q = map_halo[-1 - g];
        if (q >= 0) { halo_slots[q] = s; map_halo[-1 - g] = -1; }
    } else {
        const int a = map_prev[g], b = map_next[g];
        if (a >= 0) { border_prev[a] = s; map_prev[g] = -1; }
        if (b >= 0) { border_next[b] = s; map_next[g] = -1; }
    }
}

// both messages of a step in one launch: threads [0, k0) serve the first list, [k0, k0 + k1) the second
__global__ void k_slab_pack2(md_slab_frame f, const float4 *__restrict__ pos, const int *__restrict__ slots0, int k0,
                             float4 *__restrict__ rows0, const int *__restrict__ slots1, int k1,
                             float4 *__restrict__ rows1) {
    const int t = blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= k0 + k1) return;
    const bool first = t < k0;
    const int u = first ? t : t - k0;
    float4 p = pos[(first ? slots0 : slots1)[u]];
    p.x = slab_to_global(f, p.x);
    (first ? rows0 : rows1)[u] = p;
}
__global__ void k_slab_unpack2(md_slab_frame f, const float4 *__restrict__ rows0, const int *__restrict__ slots0, int k0,
                               const float4 *__restrict__ rows1, const int *__restrict__ slots1, int k1,
                               float4 *__restrict__ pos) {
    const int t = blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= k0 + k1) return;
    const bool first = t < k0;
    const int u = first ? t : t - k0;
    float4 p = (first ? rows0 : rows1)[u];
    p.x = slab_to_local(f, p.x);
    pos[(first ? slots0 : slots1)[u]] = p;
}

__global__ void k_iota(int n, int *id) {
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) id[i] = i;
}

// Adds an IF node (condition `cond`) after the current capture front of `st` whose body is the
// rebuild (cell list + re-sort + neighbor list) of the state held in `pos`; `st` continues after it.
int record_rebuild_if(md_system *s, cudaStream_t st, cudaGraphConditionalHandle cond, float4 *pos,
                      float4 *vel, int *id, int *nbr_idx, int *nbr_count) {
    int *status = s->words + 1;
    const bool resort = s->cfg.resort != 0;
    cudaStreamCaptureStatus cs;
    cudaGraph_t graph = nullptr;
    const cudaGraphNode_t *deps = nullptr;
    size_t ndeps = 0;
    CU(cudaStreamGetCaptureInfo(st, &cs, nullptr, &graph, &deps, &ndeps));
    if (cs != cudaStreamCaptureStatusActive || !graph) return fail(MD_ECUDA, "stream is not capturing");
    cudaGraphNodeParams np = {cudaGraphNodeTypeConditional};
    np.type = cudaGraphNodeTypeConditional;
    np.conditional.handle = cond;
    np.conditional.type = cudaGraphCondTypeIf;
    np.conditional.size = 1;
    cudaGraphNode_t node;
    CU(cudaGraphAddNode(&node, graph, deps, ndeps, &np));
    cudaGraph_t body = np.conditional.phGraph_out[0];
    if (!s->body_stream) CU(cudaStreamCreateWithFlags(&s->body_stream, cudaStreamNonBlocking));
    CU(cudaStreamBeginCaptureToGraph(s->body_stream, body, nullptr, nullptr, 0, cudaStreamCaptureModeThreadLocal));
    int rc = launch_cell_build(s, pos, vel, id, s->cell_start_i, s->perm_i, status, nullptr, s->body_stream);
    if (!rc) rc = launch_nbr_build(s, resort ? pos : s->pos_s, s->cell_start_i, resort ? nullptr : s->perm_i,
                                   nbr_idx, nbr_count, status, nullptr, 1, s->body_stream);
    cudaGraph_t ended = nullptr;
    cudaError_t e = cudaStreamEndCapture(s->body_stream, &ended);
    if (rc) return rc;
    if (e != cudaSuccess) return fail(MD_ECUDA, "capturing the rebuild body: %s", cudaGetErrorString(e));
    CU(cudaStreamUpdateCaptureDependencies(st, &node, 1, cudaStreamSetCaptureDependencies));
    return MD_OK;
}

// One velocity-Verlet step as launches on `st` (captured into a graph or run directly).
// in_graph: `st` is capturing; the rebuild kernels go into the body of an IF node whose condition
// the drift kernel raises, so a step without a rebuild launches two kernels.  Otherwise every
// rebuild kernel is launched and returns at once while the device flag is 0.
int record_step(md_system *s, const Pair &pp, float4 *pos, float4 *vel, float4 *force, int *id,
                int *nbr_idx, int *nbr_count, float dt, float mass, int *stats, cudaStream_t st,
                bool in_graph) {
    const Geom &g = s->g;
    const float a = dt / (2.0f * mass);
    int *flag = s->words + 0;
    int *status = s->words + 1;
    const int nb = blocks_for(g.n);
    int rc;
    if (!in_graph || rebuild_is_flagged(s)) {
        cudaGraphConditionalHandle none = 0;
        if (g.dim == 3) k_kick_drift<3, false><<<nb, 256, 0, st>>>(g, pos, vel, force, s->ref_pos, a, dt, flag, none);
        else k_kick_drift<2, false><<<nb, 256, 0, st>>>(g, pos, vel, force, s->ref_pos, a, dt, flag, none);
        LAUNCH_OK();
        rc = launch_rebuild_flagged(s, pos, vel, id, nbr_idx, nbr_count, flag, st);
        if (rc) return rc;
    } else {
        cudaStreamCaptureStatus cs;
        cudaGraph_t graph = nullptr;
        CU(cudaStreamGetCaptureInfo(st, &cs, nullptr, &graph, nullptr, nullptr));
        if (cs != cudaStreamCaptureStatusActive || !graph) return fail(MD_ECUDA, "stream is not capturing");
        cudaGraphConditionalHandle cond;
        CU(cudaGraphConditionalHandleCreate(&cond, graph, 0, cudaGraphCondAssignDefault));
        if (g.dim == 3) k_kick_drift<3, true><<<nb, 256, 0, st>>>(g, pos, vel, force, s->ref_pos, a, dt, flag, cond);
        else k_kick_drift<2, true><<<nb, 256, 0, st>>>(g, pos, vel, force, s->ref_pos, a, dt, flag, cond);
        LAUNCH_OK();
        rc = record_rebuild_if(s, st, cond, pos, vel, id, nbr_idx, nbr_count);
        if (rc) return rc;
    }
    Book book = {flag, status, stats};
    return launch_force(s, pp, pos, nbr_idx, nbr_count, force, vel, a, nullptr, false, book, st);
}

int run_fused_direct(md_system *s, const Pair &pp, float4 *pos, float4 *vel, float4 *force, int *id,
                     int *nbr_idx, int *nbr_count, float dt, float mass, int *stats, int nsteps,
                     cudaStream_t st);

// `reps` fused steps on the capturing stream `st` (3-D LJ fast path): one k_kick_drift opens the
// first step, every force kernel but the last also opens the next step and writes the drifted
// positions to the other buffer (pos <-> pos_alt); reps is 1 or odd, so the state ends in `pos`.
int record_fused(md_system *s, const Pair &pp, float4 *pos, float4 *vel, float4 *force, int *id,
                 int *nbr_idx, int *nbr_count, float dt, float mass, int *stats, int reps,
                 cudaStream_t st) {
    // the rebuild as launches that return at once on a zero flag: no IF nodes, the plain loop is the graph
    if (rebuild_is_flagged(s))
        return run_fused_direct(s, pp, pos, vel, force, id, nbr_idx, nbr_count, dt, mass, stats, reps, st);
    const Geom &g = s->g;
    const float a = dt / (2.0f * mass);
    int *flags[2] = {s->words + 0, s->words + 3};
    int *status = s->words + 1;
    cudaStreamCaptureStatus cs;
    cudaGraph_t graph = nullptr;
    CU(cudaStreamGetCaptureInfo(st, &cs, nullptr, &graph, nullptr, nullptr));
    if (cs != cudaStreamCaptureStatusActive || !graph) return fail(MD_ECUDA, "stream is not capturing");
    cudaGraphConditionalHandle cond;
    CU(cudaGraphConditionalHandleCreate(&cond, graph, 0, cudaGraphCondAssignDefault));
    k_kick_drift<3, true><<<blocks_for(g.n), 256, 0, st>>>(g, pos, vel, force, s->ref_pos, a, dt, flags[0], cond);
    LAUNCH_OK();
    float4 *cur = pos, *other = s->pos_alt;
    for (int r = 0; r < reps; ++r) {
        int rc = record_rebuild_if(s, st, cond, cur, vel, id, nbr_idx, nbr_count);
        if (rc) return rc;
        Book book = {flags[r & 1], status, stats};
        NextStep nx = NextStep();
        if (r + 1 < reps) {
            CU(cudaGraphConditionalHandleCreate(&cond, graph, 0, cudaGraphCondAssignDefault));
            nx.pos_out = other; nx.ref = s->ref_pos; nx.dt = dt; nx.flag = flags[(r + 1) & 1];
            nx.cond = cond; nx.has_cond = 1;
        }
        rc = launch_force(s, pp, cur, nbr_idx, nbr_count, force, vel, a, nullptr, false, book, st, nx);
        if (rc) return rc;
        if (r + 1 < reps) std::swap(cur, other);
    }
    if (cur != pos) return fail(MD_EINVAL, "fused graph of %d steps does not end in the caller's buffer", reps);
    return MD_OK;
}

// The fused loop with the rebuild on a branch of its own.  In a step without a rebuild the two flagged launches
// of launch_rebuild_flagged cost 5.7 us in series with the force kernel (a kernel node that does nothing still
// takes 2.7 us); here they run BESIDE it: after every step the stream forks; the side branch holds the flagged
// rebuild followed by a second launch of the force kernel that runs only if the step's flag is up (only_if),
// the main branch the force kernel that runs only if it is not (skip); then the branches join.  Exactly one of
// the two force launches does the step.  Measured on a lattice at rest (no rebuild fires): 42.7 us per step
// against 45.3 in series and 39.6 without any rebuild machinery.
// The flag of step r is read by launches on both branches for as long as step r lasts, so no launch of step r
// may clear it: three flag words rotate, step r reads F[r % 3], its force kernel raises F[(r + 1) % 3] for
// the next step and clears F[(r + 2) % 3], which step r - 1 has finished with and step r + 1 will raise.
int run_fused_forked(md_system *s, const Pair &pp, float4 *pos, float4 *vel, float4 *force, int *id,
                     int *nbr_idx, int *nbr_count, float dt, float mass, int *stats, int nsteps,
                     cudaStream_t st) {
    const Geom &g = s->g;
    const float a = dt / (2.0f * mass);
    int *F[3] = {s->words + 5, s->words + 6, s->words + 7};
    int *status = s->words + 1;
    if (!s->body_stream) CU(cudaStreamCreateWithFlags(&s->body_stream, cudaStreamNonBlocking));
    if (!s->ev_fork) CU(cudaEventCreateWithFlags(&s->ev_fork, cudaEventDisableTiming));
    if (!s->ev_join) CU(cudaEventCreateWithFlags(&s->ev_join, cudaEventDisableTiming));
    cudaStream_t side = s->body_stream;
    cudaGraphConditionalHandle none = 0;
    CU(cudaMemsetAsync(F[0], 0, 3 * sizeof(int), st));          // whatever the last loop left behind
    k_kick_drift<3, false><<<blocks_for(g.n), 256, 0, st>>>(g, pos, vel, force, s->ref_pos, a, dt, F[0], none);
    LAUNCH_OK();
    float4 *cur = pos, *other = s->pos_alt;
    for (int r = 0; r < nsteps; ++r) {
        int *flag = F[r % 3];
        NextStep nx = NextStep();
        if (r + 1 < nsteps) {
            nx.pos_out = other; nx.ref = s->ref_pos; nx.dt = dt; nx.flag = F[(r + 1) % 3];
            nx.cond = none; nx.has_cond = 0;
        }
        CU(cudaEventRecord(s->ev_fork, st));
        CU(cudaStreamWaitEvent(side, s->ev_fork, 0));
        // side branch: the rebuild and the force kernel behind it, both only if the flag is up
        int rc = launch_rebuild_flagged(s, cur, vel, id, nbr_idx, nbr_count, flag, side);
        if (rc) return rc;
        Book alt = {flag, status, stats, nullptr, nullptr, nullptr, flag, F[(r + 2) % 3]};
        rc = launch_force(s, pp, cur, nbr_idx, nbr_count, force, vel, a, nullptr, false, alt, side, nx);
        if (rc) return rc;
        CU(cudaEventRecord(s->ev_join, side));
        // main branch: the force kernel, only if the flag is not up
        Book mainb = {flag, status, stats, flag, nullptr, nullptr, nullptr, F[(r + 2) % 3]};
        rc = launch_force(s, pp, cur, nbr_idx, nbr_count, force, vel, a, nullptr, false, mainb, st, nx);
        if (rc) return rc;
        CU(cudaStreamWaitEvent(st, s->ev_join, 0));
        if (r + 1 < nsteps) std::swap(cur, other);
    }
    if (cur != pos) return fail(MD_EINVAL, "fused loop of %d steps does not end in the caller's buffer", nsteps);
    return MD_OK;
}

// The fused step loop as plain launches (option use_graph = 0; what a profiler can list kernel by
// kernel): the kernels and their order are those of record_fused, the rebuild kernels are launched
// every step and return at once while the step's device flag is 0.  nsteps must be odd (the
// position buffers swap nsteps - 1 times and the state must end in the caller's).
int run_fused_direct(md_system *s, const Pair &pp, float4 *pos, float4 *vel, float4 *force, int *id,
                     int *nbr_idx, int *nbr_count, float dt, float mass, int *stats, int nsteps,
                     cudaStream_t st) {
    const Geom &g = s->g;
    const float a = dt / (2.0f * mass);
    if (s->fork && rebuild_is_flagged(s))
        return run_fused_forked(s, pp, pos, vel, force, id, nbr_idx, nbr_count, dt, mass, stats, nsteps, st);
    int *flags[2] = {s->words + 0, s->words + 3};
    int *status = s->words + 1;
    cudaGraphConditionalHandle none = 0;
    k_kick_drift<3, false><<<blocks_for(g.n), 256, 0, st>>>(g, pos, vel, force, s->ref_pos, a, dt, flags[0], none);
    LAUNCH_OK();
    float4 *cur = pos, *other = s->pos_alt;
    for (int r = 0; r < nsteps; ++r) {
        int *flag = flags[r & 1];
        int rc = launch_rebuild_flagged(s, cur, vel, id, nbr_idx, nbr_count, flag, st);
        if (rc) return rc;
        Book book = {flag, status, stats};
        NextStep nx = NextStep();
        if (r + 1 < nsteps) {
            nx.pos_out = other; nx.ref = s->ref_pos; nx.dt = dt; nx.flag = flags[(r + 1) & 1];
            nx.cond = none; nx.has_cond = 0;
        }
        rc = launch_force(s, pp, cur, nbr_idx, nbr_count, force, vel, a, nullptr, false, book, st, nx);
        if (rc) return rc;
        if (r + 1 < nsteps) std::swap(cur, other);
    }
    if (cur != pos) return fail(MD_EINVAL, "fused loop of %d steps does not end in the caller's buffer", nsteps);
    return MD_OK;
}

void drop_graphs(md_system *s) {
    if (s->exec1) cudaGraphExecDestroy(s->exec1);
    if (s->execU) cudaGraphExecDestroy(s->execU);
    if (s->rule_exec1) cudaGraphExecDestroy(s->rule_exec1);
    if (s->rule_execU) cudaGraphExecDestroy(s->rule_execU);
    s->exec1 = s->execU = s->rule_exec1 = s->rule_execU = nullptr;
    s->key_valid = false;
    s->rule_key_valid = false;
}

int capture(md_system *s, const Pair &pp, const StepKey &k, int reps, cudaGraphExec_t *out) {
    if (!s->cap_stream) CU(cudaStreamCreateWithFlags(&s->cap_stream, cudaStreamNonBlocking));
    CU(cudaStreamBeginCapture(s->cap_stream, cudaStreamCaptureModeThreadLocal));
    int rc = MD_OK;
    if (fast32_kind(s, pp) && s->fused && (reps & 1))
        rc = record_fused(s, pp, (float4 *)k.pos, (float4 *)k.vel, (float4 *)k.force, (int *)k.id,
                          (int *)k.nbr_idx, (int *)k.nbr_count, k.dt, k.mass, (int *)k.stats, reps,
                          s->cap_stream);
    else
        for (int r = 0; r < reps && rc == MD_OK; ++r)
            rc = record_step(s, pp, (float4 *)k.pos, (float4 *)k.vel, (float4 *)k.force, (int *)k.id,
                             (int *)k.nbr_idx, (int *)k.nbr_count, k.dt, k.mass, (int *)k.stats,
                             s->cap_stream, true);
    cudaGraph_t graph = nullptr;
    cudaError_t e = cudaStreamEndCapture(s->cap_stream, &graph);
    if (rc) { if (graph) cudaGraphDestroy(graph); return rc; }
    if (e != cudaSuccess) return fail(MD_ECUDA, "cudaStreamEndCapture: %s", cudaGetErrorString(e));
    e = cudaGraphInstantiate(out, graph, 0);
    cudaGraphDestroy(graph);
    if (e != cudaSuccess) return fail(MD_ECUDA, "cudaGraphInstantiate: %s", cudaGetErrorString(e));
    return MD_OK;
}

// One step of an update rule other than NVE on `st`: the rule's opening kernels up to the drift (which
// raises the rebuild flag / graph condition), the rebuild (an IF node when capturing, kernels that
// return at once on a zero flag otherwise), the force, the rule's closing kernels.
int record_rule_step(md_system *s, const Pair &pp, const RuleArgs &A, cudaStream_t st, bool in_graph) {
    const Geom &g = s->g;
    int *flag = s->words + 0, *status = s->words + 1;
    const int nb = blocks_for(g.n);
    float4 *p4 = (float4 *)A.pos, *v4 = (float4 *)A.vel, *f4 = (float4 *)A.force;
    Raise rs = {flag, 0, 0};
    const bool use_if = in_graph && !rebuild_is_flagged(s);
    if (use_if) {
        cudaStreamCaptureStatus cs;
        cudaGraph_t graph = nullptr;
        CU(cudaStreamGetCaptureInfo(st, &cs, nullptr, &graph, nullptr, nullptr));
        if (cs != cudaStreamCaptureStatusActive || !graph) return fail(MD_ECUDA, "stream is not capturing");
        CU(cudaGraphConditionalHandleCreate(&rs.cond, graph, 0, cudaGraphCondAssignDefault));
        rs.has_cond = 1;
    }
    const float a = A.dt / (2.0f * A.mass);           // half-kick factor (Langevin, Nose-Hoover)
    float4 *force_vel = nullptr;                      // velocities the force kernel half-kicks
    float force_a = 0.0f;
    const int nbk = blocks_for(g.n, NH_BLOCK), nbf = blocks_for(g.n, FIRE_BLOCK);
    double *partial = s->fire_tmp;
    switch (A.rule) {
    case RULE_FIRE: {
        // the mixing of the previous step (coef, written by its k_fire_finalize) happens in this kernel
        const float *coef = reinterpret_cast<const float *>(s->fire_tmp + (size_t)nbf * 3);
        if (g.dim == 3) k_fire_kick_drift<3><<<nb, 256, 0, st>>>(g, p4, v4, f4, s->ref_pos, (const float *)A.state, coef, rs);
        else k_fire_kick_drift<2><<<nb, 256, 0, st>>>(g, p4, v4, f4, s->ref_pos, (const float *)A.state, coef, rs);
        break;
    }
    case RULE_BROWNIAN: {
        const float mu = A.dt / A.gamma, amp = std::sqrt(2.0f * A.kT * A.dt / A.gamma);
        if (g.dim == 3) k_brownian_drift<3><<<nb, 256, 0, st>>>(g, p4, f4, A.id, s->ref_pos, mu, amp, reinterpret_cast<const unsigned *>(s->words + 20), A.stats, rs);
        else k_brownian_drift<2><<<nb, 256, 0, st>>>(g, p4, f4, A.id, s->ref_pos, mu, amp, reinterpret_cast<const unsigned *>(s->words + 20), A.stats, rs);
        break;
    }
    case RULE_LANGEVIN: {
        const double c1d = std::exp(-(double)A.gamma * (double)A.dt);
        const float c1 = (float)c1d, c2 = (float)std::sqrt((double)A.kT / (double)A.mass * (1.0 - c1d * c1d));
        if (g.dim == 3) k_langevin_baoa<3><<<nb, 256, 0, st>>>(g, p4, v4, f4, A.id, s->ref_pos, a, A.dt, c1, c2, reinterpret_cast<const unsigned *>(s->words + 20), A.stats, rs);
        else k_langevin_baoa<2><<<nb, 256, 0, st>>>(g, p4, v4, f4, A.id, s->ref_pos, a, A.dt, c1, c2, reinterpret_cast<const unsigned *>(s->words + 20), A.stats, rs);
        force_vel = v4; force_a = a;
        break;
    }
    case RULE_NH: {
        const double dofkT = (double)g.dim * g.n * (double)A.kT, tau2 = (double)A.tau * (double)A.tau;
        // scale = {this half step's factor, the previous step's closing factor (still to be applied), 1}
        float *scale = reinterpret_cast<float *>(s->fire_tmp + nbk);
        k_nh_ke<<<nbk, NH_BLOCK, 0, st>>>(g.n, g.dim, v4, partial, scale + 1);
        k_nh_finalize<<<1, 256, 0, st>>>(nbk, partial, (double)A.mass, dofkT, (double)A.kT, tau2, A.nh_chain,
                                         (double)A.dt, (double *)A.state, scale);
        if (g.dim == 3) k_nh_kick_drift<3><<<nb, 256, 0, st>>>(g, p4, v4, f4, s->ref_pos, a, A.dt, scale, scale + 1, rs);
        else k_nh_kick_drift<2><<<nb, 256, 0, st>>>(g, p4, v4, f4, s->ref_pos, a, A.dt, scale, scale + 1, rs);
        force_vel = v4; force_a = a;
        break;
    }
    case RULE_FLOCK: {
        // forward Euler uses the gradients of the CURRENT state: two passes over the list, then the
        // update (which raises the rebuild), the rebuild for the next step, the bookkeeping
        FlockPar fq = {A.flock.J_align, A.flock.R_align, A.flock.J_avoid, A.flock.R_avoid,
                       A.flock.J_cohesion, A.flock.R_cohesion, A.flock.alpha, A.flock.speed};
        fq.nobs = A.nobs; fq.Job = A.J_obs;
        for (int o = 0; o < A.nobs; ++o) { fq.ox[o] = A.obs[3 * o]; fq.oy[o] = A.obs[3 * o + 1]; fq.oD[o] = A.obs[3 * o + 2]; }
        fq.npred = A.npred; fq.pred = (const float4 *)A.pred;
        fq.Jfl = A.ppar.J_flee; fq.Rfl = A.ppar.R_flee; fq.Jch = A.ppar.J_chase; fq.Rch = A.ppar.R_chase; fq.vpred = A.ppar.speed;
        const int nbp = blocks_for(g.n, 128);
        double2 *cs = reinterpret_cast<double2 *>(s->pos_s);       // free between rebuilds
        k_flock_trig<<<nb, 256, 0, st>>>(g.n, p4, cs);
        const int ai = (int)A.flock.alpha;
#define FLOCK_PASS1(AI) k_flock_pass1<AI><<<nbp, 128, 0, st>>>(g, fq, p4, cs, A.nbr_idx, A.nbr_count, s->vel_s, s->pos_alt)
        if ((float)ai != A.flock.alpha) FLOCK_PASS1(0);
        else if (ai == 1) FLOCK_PASS1(1);
        else if (ai == 2) FLOCK_PASS1(2);
        else if (ai == 3) FLOCK_PASS1(3);
        else if (ai == 4) FLOCK_PASS1(4);
        else FLOCK_PASS1(0);
#undef FLOCK_PASS1
        k_flock_pass2<<<nbp, 128, 0, st>>>(g, fq, p4, A.nbr_idx, A.nbr_count, s->vel_s, s->pos_alt);
        if (A.npred > 0) {
            const int nchunk = std::max(1, std::min(FLOCK_PRED_CHUNKS, g.n / 1024));
            double *part = s->pred_tmp;
            k_flock_pred_partial<<<dim3(nchunk, A.npred), 256, 0, st>>>(g, fq, p4, (const float4 *)A.pred, part);
#define FLOCK_PRED(AI) k_flock_predators<AI><<<A.npred, 32, 0, st>>>(g, fq, (float4 *)A.pred, part, nchunk, A.dt)
            if ((float)ai != A.flock.alpha) FLOCK_PRED(0);
            else if (ai == 1) FLOCK_PRED(1);
            else if (ai == 2) FLOCK_PRED(2);
            else if (ai == 3) FLOCK_PRED(3);
            else if (ai == 4) FLOCK_PRED(4);
            else FLOCK_PRED(0);
#undef FLOCK_PRED
        }
        k_flock_update<<<nb, 256, 0, st>>>(g, fq, p4, s->vel_s, s->ref_pos, A.dt, rs);
        break;
    }
    default: return fail(MD_EINVAL, "unknown update rule %d", A.rule);
    }
    LAUNCH_OK();
    float4 *sort_vel = (A.rule == RULE_BROWNIAN || A.rule == RULE_FLOCK) ? nullptr : v4;
    int rc;
    if (use_if) {
        rc = record_rebuild_if(s, st, rs.cond, p4, sort_vel, A.id, A.nbr_idx, A.nbr_count);
        if (rc) return rc;
    } else {
        rc = launch_rebuild_flagged(s, p4, sort_vel, A.id, A.nbr_idx, A.nbr_count, flag, st);
        if (rc) return rc;
    }
    Book book = {flag, status, A.stats};
    if (A.rule == RULE_FLOCK) {
        k_flock_book<<<1, 1, 0, st>>>(book);
        LAUNCH_OK();
        return MD_OK;
    }
    rc = launch_force(s, pp, p4, A.nbr_idx, A.nbr_count, f4, force_vel, force_a, nullptr, false, book, st);
    if (rc) return rc;
    if (A.rule == RULE_FIRE) {
        const FirePar fp = {A.fire.dt_start, A.fire.dt_max, A.fire.n_min, A.fire.f_inc, A.fire.f_dec,
                            A.fire.alpha_start, A.fire.f_alpha};
        float *coef = reinterpret_cast<float *>(s->fire_tmp + (size_t)nbf * 3);
        k_fire_kick_reduce<<<nbf, FIRE_BLOCK, 0, st>>>(g.n, g.dim, v4, f4, (const float *)A.state, partial);
        k_fire_finalize<<<1, 256, 0, st>>>(nbf, partial, fp, (float *)A.state, coef);
        LAUNCH_OK();      // the mixing v = c1 v + c2 F: in the next step's k_fire_kick_drift, or in run_rule when the call ends
    } else if (A.rule == RULE_NH) {
        const double dofkT = (double)g.dim * g.n * (double)A.kT, tau2 = (double)A.tau * (double)A.tau;
        float *scale = reinterpret_cast<float *>(s->fire_tmp + nbk);
        k_nh_ke<<<nbk, NH_BLOCK, 0, st>>>(g.n, g.dim, v4, partial, scale + 2);
        k_nh_finalize<<<1, 256, 0, st>>>(nbk, partial, (double)A.mass, dofkT, (double)A.kT, tau2, A.nh_chain,
                                         (double)A.dt, (double *)A.state, scale + 1);
        LAUNCH_OK();      // v *= scale[1]: in the next step's k_nh_ke / k_nh_kick_drift, or in run_rule when the call ends
    }
    return MD_OK;
}

int capture_rule(md_system *s, const Pair &pp, const RuleArgs &A, int reps, cudaGraphExec_t *out) {
    if (!s->cap_stream) CU(cudaStreamCreateWithFlags(&s->cap_stream, cudaStreamNonBlocking));
    CU(cudaStreamBeginCapture(s->cap_stream, cudaStreamCaptureModeThreadLocal));
    int rc = MD_OK;
    for (int r = 0; r < reps && rc == MD_OK; ++r) rc = record_rule_step(s, pp, A, s->cap_stream, true);
    cudaGraph_t graph = nullptr;
    cudaError_t e = cudaStreamEndCapture(s->cap_stream, &graph);
    if (rc) { if (graph) cudaGraphDestroy(graph); return rc; }
    if (e != cudaSuccess) return fail(MD_ECUDA, "cudaStreamEndCapture: %s", cudaGetErrorString(e));
    e = cudaGraphInstantiate(out, graph, 0);
    cudaGraphDestroy(graph);
    if (e != cudaSuccess) return fail(MD_ECUDA, "cudaGraphInstantiate: %s", cudaGetErrorString(e));
    return MD_OK;
}

// nsteps of an update rule: stats reset, then graphs of 8 steps and of 1 step (or direct launches).
// What a rule leaves for the next step's opening kernel is applied here when the call ends, so that the
// caller's velocities are final: FIRE's mixing, Nose-Hoover's closing scale factor.
int finish_rule(md_system *s, const RuleArgs &A, cudaStream_t st) {
    const int n = s->g.n, nb = blocks_for(n);
    if (A.rule == RULE_FIRE) {
        const float *coef = reinterpret_cast<const float *>(s->fire_tmp + (size_t)blocks_for(n, FIRE_BLOCK) * 3);
        k_fire_mix<<<nb, 256, 0, st>>>(n, (float4 *)A.vel, (const float4 *)A.force, coef);
        LAUNCH_OK();
    } else if (A.rule == RULE_NH) {
        const float *scale = reinterpret_cast<const float *>(s->fire_tmp + blocks_for(n, NH_BLOCK));
        k_nh_scale<<<nb, 256, 0, st>>>(n, (float4 *)A.vel, scale + 1);
        LAUNCH_OK();
    }
    return MD_OK;
}

int run_rule(md_system *s, const Pair &pp, RuleArgs &A, int nsteps, cudaStream_t st) {
    if (s->r0 != 0 || s->r1 != s->g.n) return fail(MD_EINVAL, "a range is set (md_set_range): drive the step with md_kick_drift / md_half_kick");
    A.fast32 = s->fast32; A.builder = s->builder; A.nb_parts = s->nb_parts; A.remap = s->remap; A.est_thr = s->est_thr;
    k_init_stats<<<1, 1, 0, st>>>(A.stats, s->words + 0);
    k_set_noise<<<1, 1, 0, st>>>(s->words, A.seed, A.step0);
    LAUNCH_OK();
    A.seed = 0; A.step0 = 0;          // not part of what a captured graph depends on
    if (A.rule == RULE_NH) {
        k_nh_begin<<<1, 1, 0, st>>>(reinterpret_cast<float *>(s->fire_tmp + blocks_for(s->g.n, NH_BLOCK)));
        LAUNCH_OK();
    }
    if (!s->use_graph) {
        for (int k = 0; k < nsteps; ++k) { int rc = record_rule_step(s, pp, A, st, false); if (rc) return rc; }
        return finish_rule(s, A, st);
    }
    if (!s->rule_key_valid || memcmp(&A, &s->rule_key, sizeof(A)) != 0) {
        if (s->rule_exec1) cudaGraphExecDestroy(s->rule_exec1);
        if (s->rule_execU) cudaGraphExecDestroy(s->rule_execU);
        s->rule_exec1 = s->rule_execU = nullptr;
        s->rule_key = A;
        s->rule_key_valid = true;
    }
    const int U = 8;
    int left = nsteps, rc;
    if (left >= U) {
        if (!s->rule_execU) { rc = capture_rule(s, pp, A, U, &s->rule_execU); if (rc) return rc; }
        for (; left >= U; left -= U) CU(cudaGraphLaunch(s->rule_execU, st));
    }
    if (left > 0) {
        if (!s->rule_exec1) { rc = capture_rule(s, pp, A, 1, &s->rule_exec1); if (rc) return rc; }
        for (; left > 0; --left) CU(cudaGraphLaunch(s->rule_exec1, st));
    }
    return finish_rule(s, A, st);
}

} // namespace

// ------------------------------------------------------------------------- C ABI --------

extern "C" {

const char *md_last_error(void) { return g_err; }

int md_workspace_bytes(const md_config *cfg, int n, size_t *bytes) {
    if (!bytes) return fail(MD_EINVAL, "bytes is NULL");
    Geom g;
    int rc = make_geom(cfg, n, &g);
    if (rc) return rc;
    *bytes = layout(n, g.cells).total;
    return MD_OK;
}

int md_create(const md_config *cfg, int n, void *workspace, size_t bytes, md_system **out) {
    if (!out) return fail(MD_EINVAL, "out is NULL");
    *out = nullptr;
    Geom g;
    int rc = make_geom(cfg, n, &g);
    if (rc) return rc;
    Layout l = layout(n, g.cells);
    if (!workspace || (reinterpret_cast<uintptr_t>(workspace) % ALIGN) || bytes < l.total)
        return fail(MD_EWORKSPACE, "workspace must be a 256-byte aligned device buffer of >= %zu bytes (got %zu)", l.total, bytes);
    cudaPointerAttributes attr;
    CU(cudaPointerGetAttributes(&attr, workspace));
    if (attr.type != cudaMemoryTypeDevice && attr.type != cudaMemoryTypeManaged)
        return fail(MD_EWORKSPACE, "workspace is not device memory");
    DeviceScope scope_(attr.device);
    if (scope_.rc) return scope_.rc;
    md_system *s = new (std::nothrow) md_system;
    if (!s) return fail(MD_EINVAL, "out of host memory");
    memset(s, 0, sizeof(*s));
    s->cfg = *cfg; s->n = n; s->g = g; s->device = attr.device;
    s->ws = (char *)workspace; s->ws_bytes = bytes;
    s->words = (int *)(s->ws + l.words);
    s->scan_tmp = (int *)(s->ws + l.scan_tmp);
    s->fire_tmp = (double *)(s->ws + l.fire_tmp);
    s->pred_tmp = (double *)(s->ws + l.pred_tmp);
    s->cell_count = (int *)(s->ws + l.cell_count);
    s->cell_start_i = (int *)(s->ws + l.cell_start_i);
    s->perm_i = (int *)(s->ws + l.perm_i);
    s->cell_of = (int *)(s->ws + l.cell_of);
    s->rank_tmp = (int *)(s->ws + l.rank_tmp);
    s->perm_tmp = (int *)(s->ws + l.perm_tmp);
    s->id_s = (int *)(s->ws + l.id_s);
    s->pos_s = (float4 *)(s->ws + l.pos_s);
    s->vel_s = (float4 *)(s->ws + l.vel_s);
    s->ref_pos = (float4 *)(s->ws + l.ref_pos);
    s->pos_alt = (float4 *)(s->ws + l.pos_alt);
    s->tpp = n >= 32768 ? 0 : 4;     // 0 = streaming kernel; small systems: 4 lanes per particle
    s->use_graph = 1;
    s->nh_chain = 1;
    s->r0 = 0; s->r1 = n;
    s->fast32 = 1;
    s->builder = 2;
    s->flagged = -1;
    s->fork = 1;
    {   // block -> tile remap period: a quarter of the SM count measured best (46.7 -> 44.9 us at N = 256k on 148 SMs)
        int sms = 0;
        cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, attr.device);
        s->remap = sms >= 4 ? sms / 4 : 0;
    }
    s->fused = 1;
    {   // the cell list as one cooperative launch: as many blocks as are resident at once
        int per_sm = 0, sms = 0, coop = 0;
        cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, attr.device);
        cudaDeviceGetAttribute(&coop, cudaDevAttrCooperativeLaunch, attr.device);
        if (coop && cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, k_cell_all, 256, 0) == cudaSuccess)
        {
                s->cell_coop_max = std::min(std::min(per_sm, 4) * sms, 4095);
                s->cell_coop = n <= 65536 ? s->cell_coop_max : 0;     // measured: pays below, costs above
            }
    }
    s->est_thr = 3.5f;
    s->unroll = 9;      // odd: a fused graph swaps position buffers steps-1 times and must end in the caller's
    {   // neighbor-list builder: one warp per tile, a capacity x 32 column block + a candidate
        // chunk of shared memory per warp; as many warps per block as fit (at most NB_WARPS)
        const size_t per_warp = nb_smem_per_warp(cfg->capacity);
        int dev_smem = 0;
        cudaDeviceGetAttribute(&dev_smem, cudaDevAttrMaxSharedMemoryPerBlockOptin, attr.device);
        int w = (int)std::min<size_t>(NB_WARPS, (size_t)dev_smem / per_warp);
        if (w < 1) { delete s; return fail(MD_EINVAL, "capacity %d needs %zu bytes of shared memory per tile; the device offers %d", cfg->capacity, per_warp, dev_smem); }
        s->nb_warps = w;
        s->nb_smem = per_warp * w;
        cudaError_t ea = cudaSuccess;
        if (g.dim == 3) {
            ea = cudaFuncSetAttribute(k_nbr_build<3, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)s->nb_smem);
            if (ea == cudaSuccess) ea = cudaFuncSetAttribute(k_nbr_build<3, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)s->nb_smem);
        } else {
            ea = cudaFuncSetAttribute(k_nbr_build<2, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)s->nb_smem);
            if (ea == cudaSuccess) ea = cudaFuncSetAttribute(k_nbr_build<2, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)s->nb_smem);
        }
        const int sm2 = (int)(NB2_WARPS * sizeof(Nb2Warp));
#define MD_NB2_ATTR(D, M, P) if (ea == cudaSuccess) ea = cudaFuncSetAttribute(k_nbr_build2<D, M, P>, cudaFuncAttributeMaxDynamicSharedMemorySize, sm2)
        MD_NB2_ATTR(3, true, 1); MD_NB2_ATTR(3, false, 1); MD_NB2_ATTR(2, true, 1); MD_NB2_ATTR(2, false, 1);
        MD_NB2_ATTR(3, true, 2); MD_NB2_ATTR(3, false, 2); MD_NB2_ATTR(2, true, 2); MD_NB2_ATTR(2, false, 2);
        MD_NB2_ATTR(3, true, 4); MD_NB2_ATTR(3, false, 4); MD_NB2_ATTR(2, true, 4); MD_NB2_ATTR(2, false, 4);
#undef MD_NB2_ATTR
        if (ea != cudaSuccess) { delete s; return fail(MD_ECUDA, "cudaFuncSetAttribute: %s", cudaGetErrorString(ea)); }
    }
    cudaError_t e = cudaMemset(workspace, 0, l.total);
    if (e == cudaSuccess) e = cudaDeviceSynchronize();
    if (e != cudaSuccess) { delete s; return fail(MD_ECUDA, "clearing the workspace: %s", cudaGetErrorString(e)); }
    *out = s;
    return MD_OK;
}

int md_destroy(md_system *sys) {
    if (!sys) return MD_OK;
    DeviceScope scope_(sys->device);
    drop_graphs(sys);
    if (sys->cap_stream) cudaStreamDestroy(sys->cap_stream);
    if (sys->body_stream) cudaStreamDestroy(sys->body_stream);
    if (sys->ev_fork) cudaEventDestroy(sys->ev_fork);
    if (sys->ev_join) cudaEventDestroy(sys->ev_join);
    delete sys;
    return MD_OK;
}

int md_num_cells(const md_system *sys, int *ncell) {
    if (!sys || !ncell) return fail(MD_EINVAL, "NULL argument");
    ncell[0] = sys->g.nc[0]; ncell[1] = sys->g.nc[1]; ncell[2] = sys->g.nc[2];
    return MD_OK;
}

int md_nbr_layout(const md_system *sys, long *tile, long *tile_stride, long *particle_stride,
                  long *slot_stride, long *length) {
    if (!sys || !tile || !tile_stride || !particle_stride || !slot_stride || !length)
        return fail(MD_EINVAL, "NULL argument");
    *tile = TILE;
    *tile_stride = (long)TILE * sys->g.capacity;
    *particle_stride = 1;
    *slot_stride = TILE;
    *length = (long)((sys->n + TILE - 1) / TILE) * TILE * sys->g.capacity;
    return MD_OK;
}

int md_set_species_lj(md_system *sys, int nspecies, const float *epsilon, const float *sigma,
                      const float *r_cut) {
    if (!sys || !epsilon || !sigma || !r_cut) return fail(MD_EINVAL, "NULL argument");
    if (nspecies < 1 || nspecies > 4) return fail(MD_EINVAL, "nspecies = %d must be in 1..4", nspecies);
    for (int t = 0; t < nspecies * nspecies; ++t)
        if (!(epsilon[t] >= 0.0f) || !(sigma[t] > 0.0f) || !(r_cut[t] > 0.0f) || r_cut[t] > sys->cfg.r_cut)
            return fail(MD_EINVAL, "species pair %d: epsilon >= 0, sigma > 0, 0 < r_cut <= list r_cut", t);
    sys->ns = nspecies;
    for (int t = 0; t < nspecies * nspecies; ++t) { sys->sp_eps[t] = epsilon[t]; sys->sp_sig[t] = sigma[t]; sys->sp_rc[t] = r_cut[t]; }
    drop_graphs(sys);
    return MD_OK;
}

int md_counters(md_system *sys, int32_t *out, int reset, void *stream) {
    if (!sys || !out) return fail(MD_EINVAL, "NULL argument");
    DeviceScope scope_(sys->device);
    if (scope_.rc) return scope_.rc;
    cudaStream_t st = (cudaStream_t)stream;
    CU(cudaMemcpyAsync(out, sys->words + 8, 8 * sizeof(int), cudaMemcpyDeviceToDevice, st));
    if (reset) CU(cudaMemsetAsync(sys->words + 8, 0, 8 * sizeof(int), st));
    return MD_OK;
}

int md_set_option(md_system *sys, const char *name, double value) {
    if (!sys || !name) return fail(MD_EINVAL, "NULL argument");
    if (!strcmp(name, "threads_per_particle")) {
        int t = (int)value;
        if (!(t == 0 || t == 1 || t == 2 || t == 4)) return fail(MD_EINVAL, "threads_per_particle must be 0 (streaming kernel), 1, 2 or 4");
        sys->tpp = t;
    } else if (!strcmp(name, "use_graph")) sys->use_graph = value != 0.0;
    else if (!strcmp(name, "fast32")) sys->fast32 = value != 0.0;
    else if (!strcmp(name, "fused")) sys->fused = value != 0.0;
    else if (!strcmp(name, "remap")) sys->remap = (int)value;
    else if (!strcmp(name, "cell_coop")) {
        if (value != 0.0 && !(sys->cell_coop_max > 0)) return fail(MD_EINVAL, "the device offers no cooperative launch");
        sys->cell_coop = value != 0.0 ? sys->cell_coop_max : 0;
    }
    else if (!strcmp(name, "builder_parts")) {
        if (value != 0.0 && value != 1.0 && value != 2.0 && value != 4.0) return fail(MD_EINVAL, "builder_parts must be 0, 1, 2 or 4");
        sys->nb_parts = (int)value;
    }
    else if (!strcmp(name, "rebuild_flagged")) {
        if (value != -1.0 && value != 0.0 && value != 1.0) return fail(MD_EINVAL, "rebuild_flagged must be -1 (by size), 0 or 1");
        if (value == 1.0 && !(sys->cell_coop_max > 0)) return fail(MD_EINVAL, "the device offers no cooperative launch");
        sys->flagged = (int)value;
    }
    else if (!strcmp(name, "step_fork")) sys->fork = value != 0.0;
    else if (!strcmp(name, "builder")) {
        if (value != 1.0 && value != 2.0) return fail(MD_EINVAL, "builder must be 1 or 2");
        sys->builder = (int)value;
    }
    else if (!strcmp(name, "nh_chain")) {
        if (!(value >= 1.0 && value <= (double)NH_MAX_CHAIN) || value != (double)(int)value)
            return fail(MD_EINVAL, "nh_chain must be an integer in 1..%d", NH_MAX_CHAIN);
        sys->nh_chain = (int)value;
    }
    else if (!strcmp(name, "est_thr")) {
        if (!(value > 0.0)) return fail(MD_EINVAL, "est_thr must be positive");
        sys->est_thr = (float)value;
    }
    else return fail(MD_EINVAL, "unknown option %s", name);
    drop_graphs(sys);
    return MD_OK;
}

int md_get_option(md_system *sys, const char *name, double *value) {
    if (!sys || !name || !value) return fail(MD_EINVAL, "NULL argument");
    DeviceScope scope_(sys->device);
    if (scope_.rc) return scope_.rc;
    if (!strcmp(name, "rebuild_flagged")) *value = rebuild_is_flagged(sys) ? 1.0 : 0.0;   // what the step loops do
    else if (!strcmp(name, "est_thr")) *value = sys->est_thr;
    else if (!strcmp(name, "fast32")) *value = sys->fast32;
    else if (!strcmp(name, "use_graph")) *value = sys->use_graph;
    else if (!strcmp(name, "step_fork")) *value = sys->fork;
    else if (!strcmp(name, "threads_per_particle")) *value = sys->tpp;
    else return fail(MD_EINVAL, "unknown option %s", name);
    return MD_OK;
}

int md_cell_list_build(md_system *sys, void *pos, void *vel, int32_t *id, int32_t *cell_start,
                       int32_t *perm, void *stream) {
    if (!sys || !pos || !cell_start || !perm) return fail(MD_EINVAL, "NULL argument");
    if (!aligned16(pos) || (vel && !aligned16(vel))) return fail(MD_EINVAL, "pos/vel must be 16-byte aligned");
    DeviceScope scope_(sys->device);
    if (scope_.rc) return scope_.rc;
    return launch_cell_build(sys, (float4 *)pos, (float4 *)vel, id, cell_start, perm, nullptr,
                             nullptr, (cudaStream_t)stream);
}

int md_cell_list_static(const md_config *cfg, int n, const void *pos, int32_t *cell_start, int32_t *perm,
                        void *pos_sorted, void *stream) {
    if (!cfg || !pos || !cell_start || !perm || !pos_sorted) return fail(MD_EINVAL, "NULL argument");
    // sizes first, before any CUDA call
    if (n > MD_STATIC_MAX_N)
        return fail(MD_EINVAL, "md_cell_list_static: n = %d exceeds MD_STATIC_MAX_N = %d (the static scratch holds no more; "
                               "use md_create + md_cell_list_build with a workspace of your own)", n, MD_STATIC_MAX_N);
    Geom g;
    int rc = make_geom(cfg, n, &g);                      // host arithmetic only
    if (rc) return rc;
    if (g.cells > MD_STATIC_MAX_CELLS)
        return fail(MD_EINVAL, "md_cell_list_static: %d cells exceed MD_STATIC_MAX_CELLS = %d (the static scratch holds no more; "
                               "use md_create + md_cell_list_build with a workspace of your own)", g.cells, MD_STATIC_MAX_CELLS);
    if (!aligned16(pos) || !aligned16(pos_sorted)) return fail(MD_EINVAL, "pos/pos_sorted must be 16-byte aligned");
    if (pos == pos_sorted) return fail(MD_EINVAL, "pos_sorted must not alias pos");
    cudaPointerAttributes attr;
    CU(cudaPointerGetAttributes(&attr, pos));
    if (attr.type != cudaMemoryTypeDevice && attr.type != cudaMemoryTypeManaged)
        return fail(MD_EINVAL, "pos is not device memory");
    DeviceScope scope_(attr.device);
    if (scope_.rc) return scope_.rc;
    int *scr = nullptr;
    rc = static_scratch_address(attr.device, &scr);
    if (rc) return rc;
    int *cell_of = scr, *rank_tmp = scr + MD_STATIC_MAX_N, *perm_tmp = scr + 2 * MD_STATIC_MAX_N;
    int *cell_count = scr + 3 * MD_STATIC_MAX_N;
    cudaStream_t st = (cudaStream_t)stream;
    // the array keeps what the last call (perhaps of another geometry, perhaps aborted) left: the histogram
    // must start at zero; cell_of, rank and perm_tmp are written for every i < n before they are read
    CU(cudaMemsetAsync(cell_count, 0, (size_t)g.cells * sizeof(int), st));
    const int nb = blocks_for(n);
    const float4 *p4 = (const float4 *)pos;
    k_cell_assign<<<nb, 256, 0, st>>>(g, p4, cell_of, rank_tmp, cell_count, nullptr);
    LAUNCH_OK();
    k_cell_scan<<<1, 1024, 0, st>>>(g.cells, cell_count, cell_start, nullptr, nullptr);
    LAUNCH_OK();
    k_cell_scatter<<<nb, 256, 0, st>>>(n, cell_of, rank_tmp, cell_start, perm_tmp, nullptr);
    LAUNCH_OK();
    k_cell_order_gather<<<nb, 256, 0, st>>>(n, cell_of, cell_start, perm_tmp, nullptr, p4, nullptr, perm,
                                            (float4 *)pos_sorted, nullptr, nullptr, nullptr);
    LAUNCH_OK();
    return MD_OK;
}

int md_neighbor_list_build(md_system *sys, const void *pos, const int32_t *cell_start,
                           const int32_t *perm, int32_t *nbr_idx, int32_t *nbr_count,
                           int32_t *status, void *stream) {
    if (!sys || !pos || !cell_start || !perm || !nbr_idx || !nbr_count || !status)
        return fail(MD_EINVAL, "NULL argument");
    if (!aligned16(pos) || !aligned16(nbr_idx)) return fail(MD_EINVAL, "pos/nbr_idx must be 16-byte aligned");
    DeviceScope scope_(sys->device);
    if (scope_.rc) return scope_.rc;
    cudaStream_t st = (cudaStream_t)stream;
    CU(cudaMemsetAsync(status, 0, 2 * sizeof(int), st));
    const float4 *spos = (const float4 *)pos;
    const int *map = nullptr;
    if (!sys->cfg.resort) {
        k_gather_pos<<<blocks_for(sys->n), 256, 0, st>>>(sys->n, perm, (const float4 *)pos, sys->pos_s);
        LAUNCH_OK();
        spos = sys->pos_s; map = perm;
    }
    return launch_nbr_build(sys, spos, cell_start, map, nbr_idx, nbr_count, status, nullptr, 0, st);
}

int md_needs_rebuild(md_system *sys, const void *pos, int32_t *flag, void *stream) {
    if (!sys || !pos || !flag) return fail(MD_EINVAL, "NULL argument");
    if (!aligned16(pos)) return fail(MD_EINVAL, "pos must be 16-byte aligned");
    DeviceScope scope_(sys->device);
    if (scope_.rc) return scope_.rc;
    cudaStream_t st = (cudaStream_t)stream;
    CU(cudaMemsetAsync(flag, 0, sizeof(int), st));
    const int nb = blocks_for(sys->n);
    if (sys->g.dim == 3) k_needs_rebuild<3><<<nb, 256, 0, st>>>(sys->g, (const float4 *)pos, sys->ref_pos, flag);
    else k_needs_rebuild<2><<<nb, 256, 0, st>>>(sys->g, (const float4 *)pos, sys->ref_pos, flag);
    LAUNCH_OK();
    return MD_OK;
}

int md_pair_energy_force(md_system *sys, const md_potential *pot, const void *pos,
                         const int32_t *nbr_idx, const int32_t *nbr_count, void *force,
                         double *energy_total, void *stream) {
    if (!sys || !pos || !nbr_idx || !nbr_count || !force) return fail(MD_EINVAL, "NULL argument");
    if (!aligned16(pos) || !aligned16(force)) return fail(MD_EINVAL, "pos/force must be 16-byte aligned");
    Pair pp;
    int rc = make_pair(sys, pot, &pp);
    if (rc) return rc;
    DeviceScope scope_(sys->device);
    if (scope_.rc) return scope_.rc;
    cudaStream_t st = (cudaStream_t)stream;
    if (energy_total) CU(cudaMemsetAsync(energy_total, 0, sizeof(double), st));
    Book book = {nullptr, nullptr, nullptr};
    return launch_force(sys, pp, (const float4 *)pos, nbr_idx, nbr_count, (float4 *)force, nullptr,
                        0.0f, energy_total, true, book, st);
}

int md_nve_step(md_system *sys, const md_potential *pot, void *pos, void *vel, void *force,
                int32_t *id, int32_t *nbr_idx, int32_t *nbr_count, float dt, float mass,
                int nsteps, int32_t *stats, void *stream) {
    if (!sys || !pos || !vel || !force || !nbr_idx || !nbr_count || !stats)
        return fail(MD_EINVAL, "NULL argument");
    if (!aligned16(pos) || !aligned16(vel) || !aligned16(force)) return fail(MD_EINVAL, "pos/vel/force must be 16-byte aligned");
    if (!(dt > 0.0f) || !(mass > 0.0f) || nsteps < 0) return fail(MD_EINVAL, "dt and mass must be positive, nsteps >= 0");
    if (sys->r0 != 0 || sys->r1 != sys->g.n) return fail(MD_EINVAL, "a range is set (md_set_range): drive the step with md_kick_drift / md_half_kick");
    Pair pp;
    int rc = make_pair(sys, pot, &pp);
    if (rc) return rc;
    DeviceScope scope_(sys->device);
    if (scope_.rc) return scope_.rc;
    cudaStream_t st = (cudaStream_t)stream;
    k_init_stats<<<1, 1, 0, st>>>(stats, sys->words + 0);
    LAUNCH_OK();
    if (!sys->use_graph) {
        int left = nsteps;
        if (fast32_kind(sys, pp) && sys->fused && left > 0) {
            // fused loop over an odd number of steps; an even count takes its first step unfused
            if (!(left & 1)) {
                rc = record_step(sys, pp, (float4 *)pos, (float4 *)vel, (float4 *)force, id, nbr_idx,
                                 nbr_count, dt, mass, stats, st, false);
                if (rc) return rc;
                --left;
            }
            return run_fused_direct(sys, pp, (float4 *)pos, (float4 *)vel, (float4 *)force, id, nbr_idx,
                                    nbr_count, dt, mass, stats, left, st);
        }
        for (int s = 0; s < left; ++s) {
            rc = record_step(sys, pp, (float4 *)pos, (float4 *)vel, (float4 *)force, id, nbr_idx,
                             nbr_count, dt, mass, stats, st, false);
            if (rc) return rc;
        }
        return MD_OK;
    }
    StepKey k;
    memset(&k, 0, sizeof(k));
    k.pos = pos; k.vel = vel; k.force = force; k.id = id; k.nbr_idx = nbr_idx;
    k.nbr_count = nbr_count; k.stats = stats; k.dt = dt; k.mass = mass; k.pot = *pot;
    k.tpp = sys->tpp; k.fast32 = sys->fast32; k.builder = sys->builder; k.fused = sys->fused; k.est_thr = sys->est_thr;
    if (!sys->key_valid || memcmp(&k, &sys->key, sizeof(k)) != 0) {
        drop_graphs(sys);
        sys->key = k;
        sys->key_valid = true;
    }
    int left = nsteps;
    const int U = sys->unroll;
    if (left >= U) {
        if (!sys->execU) { rc = capture(sys, pp, k, U, &sys->execU); if (rc) return rc; }
        for (; left >= U; left -= U) CU(cudaGraphLaunch(sys->execU, st));
    }
    if (left > 0) {
        if (!sys->exec1) { rc = capture(sys, pp, k, 1, &sys->exec1); if (rc) return rc; }
        for (; left > 0; --left) CU(cudaGraphLaunch(sys->exec1, st));
    }
    return MD_OK;
}

int md_brownian_step(md_system *sys, const md_potential *pot, void *pos, void *force, int32_t *id,
                     int32_t *nbr_idx, int32_t *nbr_count, float dt, float gamma, float kT,
                     uint32_t seed, uint32_t step0, int nsteps, int32_t *stats, void *stream) {
    if (!sys || !pos || !force || !nbr_idx || !nbr_count || !stats) return fail(MD_EINVAL, "NULL argument");
    if (!aligned16(pos) || !aligned16(force)) return fail(MD_EINVAL, "pos/force must be 16-byte aligned");
    if (!(dt > 0.0f) || !(gamma > 0.0f) || !(kT >= 0.0f) || nsteps < 0)
        return fail(MD_EINVAL, "dt and gamma must be positive, kT and nsteps non-negative");
    Pair pp;
    int rc = make_pair(sys, pot, &pp);
    if (rc) return rc;
    DeviceScope scope_(sys->device);
    if (scope_.rc) return scope_.rc;
    RuleArgs A;
    memset(&A, 0, sizeof(A));
    A.rule = RULE_BROWNIAN; A.pos = pos; A.force = force; A.id = id; A.nbr_idx = nbr_idx; A.nbr_count = nbr_count;
    A.stats = stats; A.pot = *pot; A.dt = dt; A.mass = 1.0f; A.gamma = gamma; A.kT = kT; A.seed = seed; A.step0 = step0;
    return run_rule(sys, pp, A, nsteps, (cudaStream_t)stream);
}

int md_langevin_step(md_system *sys, const md_potential *pot, void *pos, void *vel, void *force,
                     int32_t *id, int32_t *nbr_idx, int32_t *nbr_count, float dt, float mass,
                     float gamma, float kT, uint32_t seed, uint32_t step0, int nsteps, int32_t *stats,
                     void *stream) {
    if (!sys || !pos || !vel || !force || !nbr_idx || !nbr_count || !stats) return fail(MD_EINVAL, "NULL argument");
    if (!aligned16(pos) || !aligned16(vel) || !aligned16(force)) return fail(MD_EINVAL, "pos/vel/force must be 16-byte aligned");
    if (!(dt > 0.0f) || !(mass > 0.0f) || !(gamma >= 0.0f) || !(kT >= 0.0f) || nsteps < 0)
        return fail(MD_EINVAL, "dt and mass must be positive, gamma, kT and nsteps non-negative");
    Pair pp;
    int rc = make_pair(sys, pot, &pp);
    if (rc) return rc;
    DeviceScope scope_(sys->device);
    if (scope_.rc) return scope_.rc;
    RuleArgs A;
    memset(&A, 0, sizeof(A));
    A.rule = RULE_LANGEVIN; A.pos = pos; A.vel = vel; A.force = force; A.id = id; A.nbr_idx = nbr_idx;
    A.nbr_count = nbr_count; A.stats = stats; A.pot = *pot; A.dt = dt; A.mass = mass; A.gamma = gamma; A.kT = kT;
    A.seed = seed; A.step0 = step0;
    return run_rule(sys, pp, A, nsteps, (cudaStream_t)stream);
}

int md_nose_hoover_step(md_system *sys, const md_potential *pot, void *pos, void *vel, void *force,
                        int32_t *id, int32_t *nbr_idx, int32_t *nbr_count, float dt, float mass,
                        float kT, float tau, double *nh_state, int nsteps, int32_t *stats, void *stream) {
    if (!sys || !pos || !vel || !force || !nbr_idx || !nbr_count || !nh_state || !stats)
        return fail(MD_EINVAL, "NULL argument");
    if (!aligned16(pos) || !aligned16(vel) || !aligned16(force)) return fail(MD_EINVAL, "pos/vel/force must be 16-byte aligned");
    if (!(dt > 0.0f) || !(mass > 0.0f) || !(kT > 0.0f) || !(tau > 0.0f) || nsteps < 0)
        return fail(MD_EINVAL, "dt, mass, kT and tau must be positive, nsteps non-negative");
    Pair pp;
    int rc = make_pair(sys, pot, &pp);
    if (rc) return rc;
    DeviceScope scope_(sys->device);
    if (scope_.rc) return scope_.rc;
    RuleArgs A;
    memset(&A, 0, sizeof(A));
    A.rule = RULE_NH; A.pos = pos; A.vel = vel; A.force = force; A.state = nh_state; A.id = id; A.nbr_idx = nbr_idx;
    A.nbr_count = nbr_count; A.stats = stats; A.pot = *pot; A.dt = dt; A.mass = mass; A.kT = kT; A.tau = tau;
    A.nh_chain = sys->nh_chain;
    return run_rule(sys, pp, A, nsteps, (cudaStream_t)stream);
}

int md_set_range(md_system *sys, int begin, int end) {
    if (!sys) return fail(MD_EINVAL, "NULL argument");
    // a range is a range of the cell-sorted order: without the physical re-sort the builder's rows,
    // counts and reference positions of slots [begin, end) belong to particles anywhere in [0, n)
    if (!sys->cfg.resort && !(begin == 0 && end == sys->n))
        return fail(MD_EINVAL, "md_set_range needs a system created with resort = 1");
    if (begin < 0 || end > sys->n || begin >= end || begin % TILE != 0 || (end % TILE != 0 && end != sys->n))
        return fail(MD_EINVAL, "range [%d, %d) must be non-empty, inside [0, %d) and aligned to list tiles of %d", begin, end, sys->n, TILE);
    sys->r0 = begin; sys->r1 = end;
    drop_graphs(sys);
    return MD_OK;
}

int md_kick_drift(md_system *sys, void *pos, void *vel, const void *force, float dt, float mass,
                  int32_t *flag, void *stream) {
    if (!sys || !pos || !vel || !force || !flag) return fail(MD_EINVAL, "NULL argument");
    if (!aligned16(pos) || !aligned16(vel) || !aligned16(force)) return fail(MD_EINVAL, "pos/vel/force must be 16-byte aligned");
    if (!(dt > 0.0f) || !(mass > 0.0f)) return fail(MD_EINVAL, "dt and mass must be positive");
    DeviceScope scope_(sys->device);
    if (scope_.rc) return scope_.rc;
    cudaStream_t st = (cudaStream_t)stream;
    CU(cudaMemsetAsync(flag, 0, sizeof(int), st));
    Geom gr = sys->g;
    gr.n = sys->r1 - sys->r0;                          // an elementwise kernel: the range by pointer offset
    const size_t o = (size_t)sys->r0;
    const float a = dt / (2.0f * mass);
    cudaGraphConditionalHandle none = 0;
    if (gr.dim == 3) k_kick_drift<3, false><<<blocks_for(gr.n), 256, 0, st>>>(gr, (float4 *)pos + o, (float4 *)vel + o, (const float4 *)force + o, sys->ref_pos + o, a, dt, flag, none);
    else k_kick_drift<2, false><<<blocks_for(gr.n), 256, 0, st>>>(gr, (float4 *)pos + o, (float4 *)vel + o, (const float4 *)force + o, sys->ref_pos + o, a, dt, flag, none);
    LAUNCH_OK();
    return MD_OK;
}

int md_force_half_kick(md_system *sys, const md_potential *pot, const void *pos, const int32_t *nbr_idx,
                       const int32_t *nbr_count, void *force, void *vel, float dt, float mass, void *stream) {
    if (!sys || !pos || !nbr_idx || !nbr_count || !force || !vel) return fail(MD_EINVAL, "NULL argument");
    if (!aligned16(pos) || !aligned16(force) || !aligned16(vel)) return fail(MD_EINVAL, "pos/force/vel must be 16-byte aligned");
    if (!(dt > 0.0f) || !(mass > 0.0f)) return fail(MD_EINVAL, "dt and mass must be positive");
    Pair pp;
    int rc = make_pair(sys, pot, &pp);
    if (rc) return rc;
    DeviceScope scope_(sys->device);
    if (scope_.rc) return scope_.rc;
    Book book = {nullptr, nullptr, nullptr};
    return launch_force(sys, pp, (const float4 *)pos, nbr_idx, nbr_count, (float4 *)force, (float4 *)vel,
                        dt / (2.0f * mass), nullptr, false, book, (cudaStream_t)stream);
}

static int check_frame(const md_slab_frame *f) {
    if (!f) return fail(MD_EINVAL, "frame is NULL");
    if (f->kind < 0 || f->kind > 2 || !(f->T >= 0.0f) || !(f->Lx > 0.0f) || !(f->L > 0.0f))
        return fail(MD_EINVAL, "slab frame: kind in 0..2, T >= 0, Lx > 0, L > 0");
    return MD_OK;
}

int md_slab_kick_drift(md_system *sys, const md_slab_frame *frame, void *pos, void *vel, const void *force,
                       const int32_t *id, float dt, float mass, int32_t *flag, const int32_t *stop, void *stream) {
    if (int rc = check_frame(frame)) return rc;
    if (!sys || !pos || !vel || !force || !id || !flag) return fail(MD_EINVAL, "NULL argument");
    if (!aligned16(pos) || !aligned16(vel) || !aligned16(force)) return fail(MD_EINVAL, "pos/vel/force must be 16-byte aligned");
    if (!(dt > 0.0f) || !(mass > 0.0f)) return fail(MD_EINVAL, "dt and mass must be positive");
    if (sys->r0 != 0 || sys->r1 != sys->n) return fail(MD_EINVAL, "a slab rank steps its whole local system: md_set_range must cover it");
    DeviceScope scope_(sys->device);
    if (scope_.rc) return scope_.rc;
    cudaStream_t st = (cudaStream_t)stream;
    const Geom &g = sys->g;
    const float a = dt / (2.0f * mass);
    if (g.dim == 3) k_slab_kick_drift<3><<<blocks_for(g.n), 256, 0, st>>>(g, *frame, (float4 *)pos, (float4 *)vel, (const float4 *)force, sys->ref_pos, id, a, dt, flag, stop);
    else k_slab_kick_drift<2><<<blocks_for(g.n), 256, 0, st>>>(g, *frame, (float4 *)pos, (float4 *)vel, (const float4 *)force, sys->ref_pos, id, a, dt, flag, stop);
    LAUNCH_OK();
    return MD_OK;
}

int md_slab_force_half_kick(md_system *sys, const md_potential *pot, const void *pos, const int32_t *nbr_idx,
                            const int32_t *nbr_count, void *force, void *vel, float dt, float mass,
                            const int32_t *flag, int32_t *stop, int32_t *done, void *stream) {
    if (!sys || !pos || !nbr_idx || !nbr_count || !force || !vel) return fail(MD_EINVAL, "NULL argument");
    if (!aligned16(pos) || !aligned16(force) || !aligned16(vel)) return fail(MD_EINVAL, "pos/force/vel must be 16-byte aligned");
    if (!(dt > 0.0f) || !(mass > 0.0f)) return fail(MD_EINVAL, "dt and mass must be positive");
    Pair pp;
    int rc = make_pair(sys, pot, &pp);
    if (rc) return rc;
    DeviceScope scope_(sys->device);
    if (scope_.rc) return scope_.rc;
    Book book = {nullptr, nullptr, nullptr, flag, stop, done};
    return launch_force(sys, pp, (const float4 *)pos, nbr_idx, nbr_count, (float4 *)force, (float4 *)vel,
                        dt / (2.0f * mass), nullptr, false, book, (cudaStream_t)stream);
}

int md_slab_convert(const md_slab_frame *frame, void *pos, int n, int to_local, void *stream) {
    if (int rc = check_frame(frame)) return rc;
    if (!pos || n < 0 || !aligned16(pos)) return fail(MD_EINVAL, "pos must be a 16-byte aligned array, n >= 0");
    if (n == 0) return MD_OK;
    k_slab_convert<<<blocks_for(n), 256, 0, (cudaStream_t)stream>>>(*frame, (float4 *)pos, n, to_local ? 1 : 0);
    LAUNCH_OK();
    return MD_OK;
}

int md_slab_pack(const md_slab_frame *frame, const void *pos, const int32_t *slots, int k, void *rows_out,
                 void *stream) {
    if (int rc = check_frame(frame)) return rc;
    if (k < 0 || (k > 0 && (!pos || !slots || !rows_out))) return fail(MD_EINVAL, "NULL argument");
    if (k == 0) return MD_OK;
    k_slab_pack<<<blocks_for(k), 256, 0, (cudaStream_t)stream>>>(*frame, (const float4 *)pos, slots, k, (float4 *)rows_out);
    LAUNCH_OK();
    return MD_OK;
}

int md_slab_unpack(const md_slab_frame *frame, const void *rows, const int32_t *slots, int k, void *pos,
                   void *stream) {
    if (int rc = check_frame(frame)) return rc;
    if (k < 0 || (k > 0 && (!pos || !slots || !rows))) return fail(MD_EINVAL, "NULL argument");
    if (k == 0) return MD_OK;
    k_slab_unpack<<<blocks_for(k), 256, 0, (cudaStream_t)stream>>>(*frame, (const float4 *)rows, slots, k, (float4 *)pos);
    LAUNCH_OK();
    return MD_OK;
}

int md_slab_step_open(md_system *sys, const md_slab_frame *frame, void *pos, void *vel, const void *force,
                      const int32_t *id, float dt, float mass, int32_t *flag, const int32_t *stop,
                      const int32_t *border_prev, int k_prev, void *rows_prev, const int32_t *border_next,
                      int k_next, void *rows_next, void *stream) {
    if (k_prev < 0 || k_next < 0 || (k_prev > 0 && (!border_prev || !rows_prev)) || (k_next > 0 && (!border_next || !rows_next)))
        return fail(MD_EINVAL, "border lists: NULL argument or negative length");
    if (int rc = md_slab_kick_drift(sys, frame, pos, vel, force, id, dt, mass, flag, stop, stream)) return rc;
    if (k_prev + k_next == 0) return MD_OK;
    DeviceScope scope_(sys->device);
    if (scope_.rc) return scope_.rc;
    k_slab_pack2<<<blocks_for(k_prev + k_next), 256, 0, (cudaStream_t)stream>>>(*frame, (const float4 *)pos, border_prev, k_prev,
                                                                               (float4 *)rows_prev, border_next, k_next,
                                                                               (float4 *)rows_next);
    LAUNCH_OK();
    return MD_OK;
}

int md_slab_step_close(md_system *sys, const md_slab_frame *frame, const md_potential *pot, const void *rows_prev,
                       const int32_t *halo_prev, int h_prev, const void *rows_next, const int32_t *halo_next,
                       int h_next, void *pos, const int32_t *nbr_idx, const int32_t *nbr_count, void *force,
                       void *vel, float dt, float mass, const int32_t *flag, int32_t *stop, int32_t *done,
                       void *stream) {
    if (int rc = check_frame(frame)) return rc;
    if (!sys || !pos) return fail(MD_EINVAL, "NULL argument");
    if (h_prev < 0 || h_next < 0 || (h_prev > 0 && (!halo_prev || !rows_prev)) || (h_next > 0 && (!halo_next || !rows_next)))
        return fail(MD_EINVAL, "halo lists: NULL argument or negative length");
    if (h_prev + h_next > 0) {
        DeviceScope scope_(sys->device);
        if (scope_.rc) return scope_.rc;
        k_slab_unpack2<<<blocks_for(h_prev + h_next), 256, 0, (cudaStream_t)stream>>>(*frame, (const float4 *)rows_prev, halo_prev,
                                                                                   h_prev, (const float4 *)rows_next, halo_next,
                                                                                   h_next, (float4 *)pos);
        LAUNCH_OK();
    }
    return md_slab_force_half_kick(sys, pot, pos, nbr_idx, nbr_count, force, vel, dt, mass, flag, stop, done, stream);
}

int md_slab_split(const md_slab_frame *frame, float lo, float hi, const void *pos, const void *vel,
                  const int32_t *id, int n, void *own_pos, void *own_vel, int32_t *own_id, void *prev_rows,
                  int32_t *prev_ids, void *next_rows, int32_t *next_ids, int cap_rows, int32_t *counts,
                  void *stream) {
    if (int rc = check_frame(frame)) return rc;
    if (n < 0 || cap_rows < 0 || !counts) return fail(MD_EINVAL, "n, cap_rows >= 0 and counts != NULL");
    if (n > 0 && (!pos || !vel || !id || !own_pos || !own_vel || !own_id)) return fail(MD_EINVAL, "NULL argument");
    if (cap_rows > 0 && (!prev_rows || !prev_ids || !next_rows || !next_ids)) return fail(MD_EINVAL, "NULL argument");
    if (!(lo < hi)) return fail(MD_EINVAL, "slab [%g, %g) is empty", lo, hi);
    cudaStream_t st = (cudaStream_t)stream;
    CU(cudaMemsetAsync(counts, 0, 4 * sizeof(int), st));
    if (n == 0) return MD_OK;
    k_slab_split<<<blocks_for(n), 256, 0, st>>>(*frame, lo, hi, (const float4 *)pos, (const float4 *)vel, id, n,
                                                (float4 *)own_pos, (float4 *)own_vel, own_id, (float4 *)prev_rows,
                                                prev_ids, (float4 *)next_rows, next_ids, cap_rows, counts);
    LAUNCH_OK();
    return MD_OK;
}

int md_slab_append(const void *rows, const int32_t *ids, int m, float lo, float hi, void *own_pos, void *own_vel,
                   int32_t *own_id, int offset, int32_t *errors, void *stream) {
    if (m < 0 || offset < 0 || !errors) return fail(MD_EINVAL, "m, offset >= 0 and errors != NULL");
    if (m == 0) return MD_OK;
    if (!rows || !ids || !own_pos || !own_vel || !own_id) return fail(MD_EINVAL, "NULL argument");
    k_slab_append<<<blocks_for(m), 256, 0, (cudaStream_t)stream>>>((const float4 *)rows, ids, m, lo, hi, (float4 *)own_pos,
                                                                   (float4 *)own_vel, own_id, offset, errors);
    LAUNCH_OK();
    return MD_OK;
}

int md_slab_border(float lo_edge, float hi_edge, const void *own_pos, const int32_t *own_id, int n_own,
                   void *prev_rows, int32_t *prev_ids, void *next_rows, int32_t *next_ids, int cap_rows,
                   int32_t *map_prev, int32_t *map_next, int32_t *counts, void *stream) {
    if (n_own < 0 || cap_rows < 0 || !counts) return fail(MD_EINVAL, "n_own, cap_rows >= 0 and counts != NULL");
    cudaStream_t st = (cudaStream_t)stream;
    CU(cudaMemsetAsync(counts, 0, 3 * sizeof(int), st));
    if (n_own == 0) return MD_OK;
    if (!own_pos || !own_id || !prev_rows || !prev_ids || !next_rows || !next_ids || !map_prev || !map_next)
        return fail(MD_EINVAL, "NULL argument");
    k_slab_border<<<blocks_for(n_own), 256, 0, st>>>(lo_edge, hi_edge, (const float4 *)own_pos, own_id, n_own,
                                                     (float4 *)prev_rows, prev_ids, (float4 *)next_rows, next_ids,
                                                     cap_rows, map_prev, map_next, counts);
    LAUNCH_OK();
    return MD_OK;
}

int md_slab_load(const md_slab_frame *frame, const void *own_pos, const void *own_vel, const int32_t *own_id,
                 int n_own, const void *halo_prev_rows, const int32_t *halo_prev_ids, int h_prev,
                 const void *halo_next_rows, const int32_t *halo_next_ids, int h_next, void *pos, void *vel,
                 int32_t *id, int32_t *map_halo, void *stream) {
    if (int rc = check_frame(frame)) return rc;
    if (n_own < 0 || h_prev < 0 || h_next < 0) return fail(MD_EINVAL, "negative count");
    const int n = n_own + h_prev + h_next;
    if (n == 0) return MD_OK;
    if (!pos || !vel || !id || !map_halo || (n_own > 0 && (!own_pos || !own_vel || !own_id)) ||
        (h_prev > 0 && (!halo_prev_rows || !halo_prev_ids)) || (h_next > 0 && (!halo_next_rows || !halo_next_ids)))
        return fail(MD_EINVAL, "NULL argument");
    k_slab_load<<<blocks_for(n), 256, 0, (cudaStream_t)stream>>>(*frame, (const float4 *)own_pos, (const float4 *)own_vel,
                                                                 own_id, n_own, (const float4 *)halo_prev_rows,
                                                                 halo_prev_ids, h_prev, (const float4 *)halo_next_rows,
                                                                 halo_next_ids, h_next, (float4 *)pos, (float4 *)vel,
                                                                 id, map_halo);
    LAUNCH_OK();
    return MD_OK;
}

int md_slab_plan(const int32_t *id, int n, int32_t *nbr_count, int32_t *map_prev, int32_t *map_next,
                 int32_t *map_halo, int32_t *border_prev, int32_t *border_next, int32_t *halo_slots, void *stream) {
    if (n < 0) return fail(MD_EINVAL, "n >= 0");
    if (n == 0) return MD_OK;
    if (!id || !nbr_count || !map_prev || !map_next || !map_halo || !border_prev || !border_next || !halo_slots)
        return fail(MD_EINVAL, "NULL argument");
    k_slab_plan<<<blocks_for(n), 256, 0, (cudaStream_t)stream>>>(id, n, nbr_count, map_prev, map_next, map_halo,
                                                                 border_prev, border_next, halo_slots);
    LAUNCH_OK();
    return MD_OK;
}

int md_half_kick(md_system *sys, void *vel, const void *force, float dt, float mass, void *stream) {
    if (!sys || !vel || !force) return fail(MD_EINVAL, "NULL argument");
    if (!aligned16(vel) || !aligned16(force)) return fail(MD_EINVAL, "vel/force must be 16-byte aligned");
    if (!(dt > 0.0f) || !(mass > 0.0f)) return fail(MD_EINVAL, "dt and mass must be positive");
    DeviceScope scope_(sys->device);
    if (scope_.rc) return scope_.rc;
    const int m = sys->r1 - sys->r0;
    const size_t o = (size_t)sys->r0;
    k_half_kick<<<blocks_for(m), 256, 0, (cudaStream_t)stream>>>(m, sys->g.dim, (float4 *)vel + o, (const float4 *)force + o, dt / (2.0f * mass));
    LAUNCH_OK();
    return MD_OK;
}

int md_set_species_bks(md_system *sys, int nspecies, const float *A, const float *B, const float *C,
                       const float *charge, float coulomb_alpha, float k_e) {
    if (!sys || !A || !B || !C || !charge) return fail(MD_EINVAL, "NULL argument");
    if (nspecies < 1 || nspecies > 4) return fail(MD_EINVAL, "nspecies = %d must be in 1..4", nspecies);
    if (!(coulomb_alpha >= 0.0f) || !(k_e >= 0.0f)) return fail(MD_EINVAL, "coulomb_alpha and k_e must be >= 0");
    for (int t = 0; t < nspecies * nspecies; ++t)
        if (!(A[t] >= 0.0f) || !(B[t] > 0.0f) || !(C[t] >= 0.0f))
            return fail(MD_EINVAL, "species pair %d: need A >= 0, B > 0, C >= 0", t);
    sys->bks_ns = nspecies; sys->bks_alpha = coulomb_alpha; sys->bks_ke = k_e;
    for (int t = 0; t < nspecies * nspecies; ++t) { sys->bks_A[t] = A[t]; sys->bks_B[t] = B[t]; sys->bks_C[t] = C[t]; }
    for (int t = 0; t < nspecies; ++t) sys->bks_q[t] = charge[t];
    drop_graphs(sys);
    return MD_OK;
}

int md_flock_obstacles(md_system *sys, int nobs, const float *centre, const float *radius, float J) {
    if (!sys) return fail(MD_EINVAL, "NULL argument");
    if (nobs < 0 || nobs > MD_MAX_OBSTACLES) return fail(MD_EINVAL, "nobs = %d must be in 0..%d", nobs, MD_MAX_OBSTACLES);
    if (nobs > 0 && (!centre || !radius)) return fail(MD_EINVAL, "NULL argument");
    if (!(J >= 0.0f)) return fail(MD_EINVAL, "J_obstacle must be >= 0");
    for (int o = 0; o < nobs; ++o) {
        if (!(radius[o] > 0.0f) || !(2.0f * radius[o] < std::min(sys->g.L[0], sys->g.L[1])))
            return fail(MD_EINVAL, "obstacle %d: radius %g must be positive and below half the box", o, radius[o]);
        if (!(centre[2 * o] >= 0.0f && centre[2 * o] < sys->g.L[0] && centre[2 * o + 1] >= 0.0f && centre[2 * o + 1] < sys->g.L[1]))
            return fail(MD_EINVAL, "obstacle %d: centre outside the box", o);
    }
    sys->nobs = nobs; sys->J_obs = J;
    memset(sys->obs, 0, sizeof(sys->obs));
    for (int o = 0; o < nobs; ++o) {
        sys->obs[3 * o] = centre[2 * o]; sys->obs[3 * o + 1] = centre[2 * o + 1]; sys->obs[3 * o + 2] = radius[o];
    }
    return MD_OK;
}

int md_flock_predators(md_system *sys, int npred, void *pred, const md_predator_params *par) {
    if (!sys) return fail(MD_EINVAL, "NULL argument");
    if (npred < 0 || npred > MD_MAX_PREDATORS) return fail(MD_EINVAL, "npred = %d must be in 0..%d", npred, MD_MAX_PREDATORS);
    if (npred == 0) { sys->npred = 0; sys->pred = nullptr; memset(&sys->ppar, 0, sizeof(sys->ppar)); return MD_OK; }
    if (!pred || !par) return fail(MD_EINVAL, "NULL argument");
    if (!aligned16(pred)) return fail(MD_EINVAL, "pred must be 16-byte aligned");
    if (!(par->J_flee >= 0.0f) || !(par->R_flee > 0.0f) || !(par->J_chase >= 0.0f) || !(par->R_chase > 0.0f) ||
        !(par->speed >= 0.0f))
        return fail(MD_EINVAL, "predator parameters out of range");
    if (2.0f * std::max(par->R_flee, par->R_chase) >= std::min(sys->g.L[0], sys->g.L[1]))
        return fail(MD_EINVAL, "R_flee and R_chase must be below half the box");
    sys->npred = npred; sys->pred = pred; sys->ppar = *par;
    return MD_OK;
}

int md_flock_step(md_system *sys, const md_flock_params *par, void *pos, int32_t *id, int32_t *nbr_idx,
                  int32_t *nbr_count, float dt, int nsteps, int32_t *stats, void *stream) {
    if (!sys || !par || !pos || !nbr_idx || !nbr_count || !stats) return fail(MD_EINVAL, "NULL argument");
    if (!aligned16(pos)) return fail(MD_EINVAL, "pos must be 16-byte aligned");
    if (sys->g.dim != 2) return fail(MD_EINVAL, "flocking is 2-D (dim = %d)", sys->g.dim);
    if (!(dt > 0.0f) || nsteps < 0 || !(par->alpha >= 1.0f) || !(par->R_align > 0.0f) || !(par->R_avoid > 0.0f) ||
        !(par->R_cohesion > 0.0f) || !(par->J_align >= 0.0f) || !(par->J_avoid >= 0.0f) || !(par->J_cohesion >= 0.0f))
        return fail(MD_EINVAL, "flocking parameters out of range");
    const float rmax = std::max(par->R_align, std::max(par->R_avoid, par->R_cohesion));
    if (rmax > sys->cfg.r_cut) return fail(MD_EINVAL, "interaction range %g exceeds the list r_cut %g", rmax, sys->cfg.r_cut);
    DeviceScope scope_(sys->device);
    if (scope_.rc) return scope_.rc;
    Pair pp;
    memset(&pp, 0, sizeof(pp));
    RuleArgs A;
    memset(&A, 0, sizeof(A));
    A.rule = RULE_FLOCK; A.pos = pos; A.id = id; A.nbr_idx = nbr_idx; A.nbr_count = nbr_count; A.stats = stats;
    A.dt = dt; A.mass = 1.0f; A.flock = *par;
    A.nobs = sys->nobs; A.J_obs = sys->J_obs;
    memcpy(A.obs, sys->obs, sizeof(float) * 3 * (size_t)sys->nobs);
    A.npred = sys->npred; A.pred = sys->pred; A.ppar = sys->ppar;
    if (sys->npred > 0 && std::max(sys->ppar.R_flee, 0.0f) * 2.0f >= std::min(sys->g.L[0], sys->g.L[1]))
        return fail(MD_EINVAL, "R_flee %g must be below half the box", sys->ppar.R_flee);
    return run_rule(sys, pp, A, nsteps, (cudaStream_t)stream);
}

int md_fire_minimize(md_system *sys, const md_potential *pot, const md_fire_params *par, void *pos,
                     void *vel, void *force, int32_t *id, int32_t *nbr_idx, int32_t *nbr_count,
                     float *fire_state, int nsteps, int32_t *stats, void *stream) {
    if (!sys || !par || !pos || !vel || !force || !nbr_idx || !nbr_count || !fire_state || !stats)
        return fail(MD_EINVAL, "NULL argument");
    if (!aligned16(pos) || !aligned16(vel) || !aligned16(force)) return fail(MD_EINVAL, "pos/vel/force must be 16-byte aligned");
    if (!(par->dt_start > 0.0f) || !(par->dt_max >= par->dt_start) || par->n_min < 0 || !(par->f_inc >= 1.0f) ||
        !(par->f_dec > 0.0f && par->f_dec < 1.0f) || !(par->alpha_start >= 0.0f && par->alpha_start < 1.0f) ||
        !(par->f_alpha > 0.0f && par->f_alpha <= 1.0f) || nsteps < 0)
        return fail(MD_EINVAL, "FIRE parameters out of range");
    Pair pp;
    int rc = make_pair(sys, pot, &pp);
    if (rc) return rc;
    DeviceScope scope_(sys->device);
    if (scope_.rc) return scope_.rc;
    cudaStream_t st = (cudaStream_t)stream;
    const FirePar fp = {par->dt_start, par->dt_max, par->n_min, par->f_inc, par->f_dec, par->alpha_start, par->f_alpha};
    k_fire_init<<<1, 1, 0, st>>>(fp, fire_state, reinterpret_cast<float *>(sys->fire_tmp + (size_t)blocks_for(sys->g.n, FIRE_BLOCK) * 3));
    LAUNCH_OK();
    RuleArgs A;
    memset(&A, 0, sizeof(A));
    A.rule = RULE_FIRE; A.pos = pos; A.vel = vel; A.force = force; A.state = fire_state; A.id = id; A.nbr_idx = nbr_idx;
    A.nbr_count = nbr_count; A.stats = stats; A.pot = *pot; A.mass = 1.0f; A.fire = *par;
    return run_rule(sys, pp, A, nsteps, st);
}

// md_nve_run_host keeps ONE context (device allocation, system, stream, and through the system the
// captured step graphs) for the last (cfg, n, device) it was called with, so that a caller who
// streams states through it does not pay cudaMalloc / md_create / graph instantiation per call.
struct HostCtx {
    bool valid;
    md_config cfg;
    int n, device;
    char *d;
    size_t o_pos, o_vel, o_force, o_pos2, o_vel2, o_force2, o_id, o_cnt, o_list, o_small, o_ws;
    md_system *sys;
    cudaStream_t st;
};
static HostCtx g_host = {};
static std::mutex g_host_mutex;

static void host_ctx_drop() {
    if (!g_host.valid) return;
    int cur = -1;
    cudaGetDevice(&cur);
    if (cur != g_host.device) cudaSetDevice(g_host.device);
    if (g_host.sys) md_destroy(g_host.sys);
    if (g_host.st) cudaStreamDestroy(g_host.st);
    if (g_host.d) cudaFree(g_host.d);
    if (cur >= 0 && cur != g_host.device) cudaSetDevice(cur);
    memset(&g_host, 0, sizeof(g_host));
}

int md_nve_run_host_release(void) {
    std::lock_guard<std::mutex> lock(g_host_mutex);
    host_ctx_drop();
    return MD_OK;
}

int md_nve_run_host(const md_config *cfg, const md_potential *pot, int n, void *pos_host,
                    void *vel_host, void *force_host, double *energy_host, float dt, float mass,
                    int nsteps, int32_t *stats_host) {
    if (!pos_host || !vel_host) return fail(MD_EINVAL, "NULL host buffer");
    size_t wsb = 0;
    int rc = md_workspace_bytes(cfg, n, &wsb);
    if (rc) return rc;
    std::lock_guard<std::mutex> lock(g_host_mutex);
    int dev = 0;
    CU(cudaGetDevice(&dev));
    HostCtx &h = g_host;
    const size_t vec = (size_t)n * sizeof(float4);
    if (!(h.valid && h.n == n && h.device == dev && memcmp(&h.cfg, cfg, sizeof(*cfg)) == 0)) {
        host_ctx_drop();
        const size_t list = (size_t)((n + TILE - 1) / TILE) * TILE * cfg->capacity * sizeof(int);
        // one allocation: pos, vel, force, out x3, id, count, list, small words, workspace
        size_t o = 0;
        auto take = [&](size_t b) { size_t at = o; o += up(b); return at; };
        h.o_pos = take(vec); h.o_vel = take(vec); h.o_force = take(vec); h.o_pos2 = take(vec);
        h.o_vel2 = take(vec); h.o_force2 = take(vec); h.o_id = take((size_t)n * 4);
        h.o_cnt = take((size_t)n * 4); h.o_list = take(list); h.o_small = take(256);
        h.o_ws = take(wsb);
        CU(cudaMalloc(&h.d, o));
        h.valid = true; h.cfg = *cfg; h.n = n; h.device = dev;      // from here host_ctx_drop frees it
        rc = md_create(cfg, n, h.d + h.o_ws, wsb, &h.sys);
        if (rc) { host_ctx_drop(); return rc; }
        cudaError_t e0 = cudaStreamCreateWithFlags(&h.st, cudaStreamNonBlocking);
        if (e0 != cudaSuccess) { host_ctx_drop(); return fail(MD_ECUDA, "cudaStreamCreate: %s", cudaGetErrorString(e0)); }
    }
    char *d = h.d;
    md_system *sys = h.sys;
    cudaStream_t st = h.st;
    cudaError_t e;
    auto done = [&](int code) { if (code != MD_OK) host_ctx_drop(); return code; };
    float4 *pos = (float4 *)(d + h.o_pos), *vel = (float4 *)(d + h.o_vel), *force = (float4 *)(d + h.o_force);
    int *id = (int *)(d + h.o_id), *cnt = (int *)(d + h.o_cnt), *nbr = (int *)(d + h.o_list);
    int *small = (int *)(d + h.o_small);        // [0..1] status, [4..7] stats, [8..9] energy (double)
    double *etot = (double *)(small + 8);
#define RUN(x) do { e = (x); if (e != cudaSuccess) return done(fail(MD_ECUDA, "%s: %s", #x, cudaGetErrorString(e))); } while (0)
#define STEP(x) do { rc = (x); if (rc) return done(rc); } while (0)
    RUN(cudaMemcpyAsync(pos, pos_host, vec, cudaMemcpyHostToDevice, st));
    RUN(cudaMemcpyAsync(vel, vel_host, vec, cudaMemcpyHostToDevice, st));
    k_iota<<<blocks_for(n), 256, 0, st>>>(n, id);
    STEP(md_cell_list_build(sys, pos, vel, id, sys->cell_start_i, sys->perm_i, st));
    STEP(md_neighbor_list_build(sys, pos, sys->cell_start_i, sys->perm_i, nbr, cnt, small, st));
    STEP(md_pair_energy_force(sys, pot, pos, nbr, cnt, force, nullptr, st));
    STEP(md_nve_step(sys, pot, pos, vel, force, id, nbr, cnt, dt, mass, nsteps, small + 4, st));
    if (energy_host) STEP(md_pair_energy_force(sys, pot, pos, nbr, cnt, force, etot, st));
    k_unpermute<<<blocks_for(n), 256, 0, st>>>(n, id, pos, vel, force, (float4 *)(d + h.o_pos2),
                                               (float4 *)(d + h.o_vel2), (float4 *)(d + h.o_force2));
    RUN(cudaGetLastError());
    RUN(cudaMemcpyAsync(pos_host, d + h.o_pos2, vec, cudaMemcpyDeviceToHost, st));
    RUN(cudaMemcpyAsync(vel_host, d + h.o_vel2, vec, cudaMemcpyDeviceToHost, st));
    if (force_host) RUN(cudaMemcpyAsync(force_host, d + h.o_force2, vec, cudaMemcpyDeviceToHost, st));
    if (energy_host) RUN(cudaMemcpyAsync(energy_host, etot, sizeof(double), cudaMemcpyDeviceToHost, st));
    if (stats_host) RUN(cudaMemcpyAsync(stats_host, small + 4, 4 * sizeof(int), cudaMemcpyDeviceToHost, st));
    RUN(cudaStreamSynchronize(st));
#undef RUN
#undef STEP
    return MD_OK;
}

} // extern "C"
