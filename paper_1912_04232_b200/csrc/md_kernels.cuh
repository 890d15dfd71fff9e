// md_kernels.cuh -- device code of libmd_b200 (sm_100a).  CUDA cores only: nothing on this
// path is a dense contraction.  Citations: /root/reference/PAPER.md line + section; readings
// of open points: SURVEY.md §8c A1..A18 / DESIGN.md §3.  Shares nothing with oracle/.
#pragma once
#include <cuda_runtime.h>
#include <cooperative_groups.h>
#include <stdint.h>

// -DMD_CHECKED: device-side asserts on every index the hot path reads or writes through (list entries,
// gather indices, cell ids, sorted slots).  The pool's compute-sanitizer is closed, so this build is
// what the memory-safety workout of the tests runs against (profiles/r2_sanitizer.md).
#ifdef MD_CHECKED
#include <assert.h>
#define MD_CHECK(c) assert(c)
#else
#define MD_CHECK(c) ((void)0)
#endif

namespace mdk {

constexpr unsigned FULL = 0xffffffffu;

// Everything a kernel needs to know about the space and the partition (by value).
struct Geom {
    int   dim, n, capacity, cells;
    int   ntot;             // particles of the whole system (n is a context's range end under md_set_range)
    int   nc[3];            // cells per side n_k = floor(L_k / R)
    float L[3];             // box sides
    float h[3];             // fl(L/2)
    float inv_cell[3];      // fl32(n_k / L_k)
    float inv_L[3];         // fl32(1 / L_k) (wrap only)
    float R2;               // fl(R*R), R = fl(r_cut + skin)
    float half_skin2;       // fl((skin/2)^2)
    float face;             // R + skin: beyond this distance from every face no list pair wraps
};

struct Pair {
    int    kind;
    double deps, drc2;
    double dsig6x2;         // LJ: 2 sigma^6
    double du_cut4;         // LJ: shift * u(r_cut) / (4 eps) = shift * ((s/rc)^12 - (s/rc)^6)
    double dalpha, dr0;     // MORSE: alpha, r0
    double du_cutm;         // MORSE: shift * u(r_cut) / eps;  BUCKINGHAM: shift * u(r_cut)
    double dA, dC;          // BUCKINGHAM: A, C (B is dalpha)
    // LJ_SPECIES: per species pair t = a * ns + b (species = (int)pos.w)
    int ns;
    double sp_sig6x2[16];   // 2 sigma_ab^6
    double sp_fs[16];       // 24 eps_ab sigma_ab^6
    double sp_es[16];       // 2 eps_ab  (1/2 * 4 eps_ab)
    double sp_rc2[16];      // rc_ab^2
    double sp_ucut4[16];    // shift * ((s/rc)^12 - (s/rc)^6)
    // BKS (kind 5) reuses the five tables as A_ab, B_ab, C_ab, k q_a q_b, shift * u_exp6(r_cut) and adds
    // the damped shifted-force Coulomb constants: a, 2a/sqrt(pi), erfc(a rc)/rc, its force shift, rc
    double bks_a, bks_tsp, bks_ec, bks_fc, bks_rc;
};

__device__ __forceinline__ int ld_volatile(const int *p) { return *(const volatile int *)p; }

// Device words md_nve_step keeps between kernels.
struct Book {
    int *flag;      // rebuild needed (set by drift, cleared by the force kernel)
    int *status;    // {overflow, max count} of the last build
    int *stats;     // {steps, rebuilds, first overflow step | -1, max count}
    // slab steps enqueued ahead of the host (md_slab_force_half_kick): while *skip != 0 the kernel does
    // nothing but raise *stop, which the drift kernels of the steps behind it read; *done counts the
    // force evaluations that did run
    const int *skip;
    int *stop;
    int *done;
    // the two force launches of a forked step (md.cu run_fused_direct): the one on the main branch has
    // skip = the step's flag, the one behind the rebuild on the side branch only_if = that flag, so exactly one
    // of them runs; neither clears the flag the other may still have to read: they clear `clear`, the flag
    // word of the step before, instead
    const int *only_if;
    int *clear;
};
// true: this launch must not touch the state (a rank's list is stale and the host has not rebuilt yet; or
// the other force launch of a forked step is the one that runs)
__device__ __forceinline__ bool book_skips(const Book &book, int gid) {
    if (book.only_if && !ld_volatile(book.only_if)) return true;
    if (!book.skip || !ld_volatile(book.skip)) return false;
    if (gid == 0 && book.stop) *book.stop = 1;
    return true;
}


// What a drift kernel does when one of its particles has moved beyond skin/2: raise the device
// flag and, when the step runs inside a CUDA graph, the condition of the rebuild's IF node.
struct Raise {
    int *flag;
    cudaGraphConditionalHandle cond;
    int has_cond;
};
__device__ __forceinline__ void raise_rebuild(const Raise &r) {
    *r.flag = 1;
    if (r.has_cond) cudaGraphSetConditional(r.cond, 1);
}

// ---------------------------------------------------------------- space (L72 §3.2.1) ----

// Canonical cell coordinate c_k = min(n_k-1, (int)(x_k * inv_k)).
__device__ __forceinline__ int cell_coord(float x, float inv, int nk) {
    int c = (int)__fmul_rn(x, inv);
    return min(max(c, 0), nk - 1);
}

// Shift function mu(r, dr): wrap into [0, L).
__device__ __forceinline__ float wrap(float x, float L, float invL) {
    x = fmaf(-L, floorf(x * invL), x);
    if (x >= L) x = 0.0f;
    if (x < 0.0f) x = 0.0f;
    return x;
}

// Nearest-image displacement a - b with the box side taken off the larger coordinate
// first, so the result carries one rounding.
__device__ __forceinline__ float min_image(float a, float b, float L, float h) {
    float d = __fsub_rn(a, b);
    if (d > h) d = __fsub_rn(__fsub_rn(a, L), b);
    else if (d < -h) d = __fsub_rn(a, __fsub_rn(b, L));
    return d;
}

// Exact fp64 nearest-image displacement of two fp32 coordinates.
__device__ __forceinline__ double min_image64(float a, float b, double L, double h) {
    double d = (double)a - (double)b;
    if (d > h) d -= L;
    else if (d < -h) d += L;
    return d;
}

// ------------------------------------------------------ cell list (L84 §3.2.3) ----------
// histogram -> exclusive scan -> scatter -> in-cell ordering + payload gather [-> copy back]
// `cond` (may be NULL) is a device word: every kernel of a conditional rebuild returns at
// once when *cond == 0, so the decision never leaves the device.

__global__ void __launch_bounds__(256)
k_cell_assign(Geom g, const float4 *__restrict__ pos, int *__restrict__ cell_of,
              int *__restrict__ rank_tmp, int *__restrict__ cell_count, const int *cond) {
    if (cond && ld_volatile(cond) == 0) return;
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= g.n) return;
    float4 p = pos[i];
    int cx = cell_coord(p.x, g.inv_cell[0], g.nc[0]);
    int cy = cell_coord(p.y, g.inv_cell[1], g.nc[1]);
    int cz = g.dim == 3 ? cell_coord(p.z, g.inv_cell[2], g.nc[2]) : 0;
    int c = (cz * g.nc[1] + cy) * g.nc[0] + cx;
    MD_CHECK(c >= 0 && c < g.cells);
    cell_of[i] = c;
    rank_tmp[i] = atomicAdd(&cell_count[c], 1);   // arrival order; made canonical later
}

// One block: exclusive scan of cell_count[0..cells) into cell_start[0..cells]; zeroes
// cell_count for the next build and resets the build status words.  Every thread owns a run of
// consecutive cells (its loads are independent, so their latency overlaps), sums it, the 1024
// partial sums are scanned once through shared memory, and the run is written back.
__global__ void __launch_bounds__(1024)
k_cell_scan(int cells, int *__restrict__ cell_count, int *__restrict__ cell_start,
            int *status, const int *cond) {
    if (cond && ld_volatile(cond) == 0) return;
    __shared__ int warp_sum[32];
    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    if (tid == 0 && status) { status[0] = 0; status[1] = 0; }
    const int per = (cells + 1023) / 1024;
    const int c0 = min(tid * per, cells), c1 = min(c0 + per, cells);
    int sum = 0;
#pragma unroll 8
    for (int c = c0; c < c1; ++c) sum += cell_count[c];          // independent loads
    int x = sum;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        int y = __shfl_up_sync(FULL, x, o);
        if (lane >= o) x += y;
    }
    if (lane == 31) warp_sum[wid] = x;
    __syncthreads();
    if (wid == 0) {
        int w = warp_sum[lane];
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            int y = __shfl_up_sync(FULL, w, o);
            if (lane >= o) w += y;
        }
        warp_sum[lane] = w;
    }
    __syncthreads();
    int run = x - sum + (wid ? warp_sum[wid - 1] : 0);           // exclusive prefix of my run
#pragma unroll 4
    for (int c = c0; c < c1; ++c) {
        const int v = cell_count[c];
        cell_count[c] = 0;
        cell_start[c] = run;
        run += v;
    }
    if (tid == 1023) cell_start[cells] = warp_sum[31];
}

// Large grids (more than SCAN_ONE_BLOCK cells): the scan in two launches.  k_cell_sum: every block
// sums SCAN_CHUNK consecutive counters; the last block to finish turns the block sums into
// exclusive offsets.  k_cell_scan2: every block scans its chunk again, adds its offset, writes
// cell_start and zeroes the counters.
constexpr int SCAN_CHUNK = 4096;           // counters per block: 1024 threads x 4
#ifndef MD_SCAN_ONE_BLOCK
#define MD_SCAN_ONE_BLOCK 16384
#endif
constexpr int SCAN_ONE_BLOCK = MD_SCAN_ONE_BLOCK;      // up to this many cells k_cell_scan (one block) is used

__device__ __forceinline__ int4 load4_counts(const int *cell_count, int c, int cells) {
    int4 v = make_int4(0, 0, 0, 0);
    if (c + 3 < cells) v = *reinterpret_cast<const int4 *>(cell_count + c);
    else {
        if (c < cells) v.x = cell_count[c];
        if (c + 1 < cells) v.y = cell_count[c + 1];
        if (c + 2 < cells) v.z = cell_count[c + 2];
    }
    return v;
}

// inclusive scan of one value per thread over a block of 1024 threads; returns the inclusive
// prefix, *total receives the block total (valid in every thread after the call)
__device__ __forceinline__ int block_scan_1024(int x, int *warp_sum, int *total) {
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        int y = __shfl_up_sync(FULL, x, o);
        if (lane >= o) x += y;
    }
    __syncthreads();                        // warp_sum may still be read from a previous call
    if (lane == 31) warp_sum[wid] = x;
    __syncthreads();
    if (wid == 0) {
        int w = warp_sum[lane];
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            int y = __shfl_up_sync(FULL, w, o);
            if (lane >= o) w += y;
        }
        warp_sum[lane] = w;
    }
    __syncthreads();
    *total = warp_sum[31];
    return x + (wid ? warp_sum[wid - 1] : 0);
}

__global__ void __launch_bounds__(1024)
k_cell_sum(int cells, const int *__restrict__ cell_count, int *__restrict__ block_sum, int *ticket,
           int *status, const int *cond) {
    if (cond && ld_volatile(cond) == 0) return;
    __shared__ int warp_sum[32];
    __shared__ int is_last;
    const int tid = threadIdx.x;
    const int4 v = load4_counts(cell_count, blockIdx.x * SCAN_CHUNK + tid * 4, cells);
    int total;
    block_scan_1024(v.x + v.y + v.z + v.w, warp_sum, &total);
    if (tid == 0) {
        block_sum[blockIdx.x] = total;
        __threadfence();
        is_last = atomicAdd(ticket, 1) == (int)gridDim.x - 1;
    }
    __syncthreads();
    if (!is_last) return;
    __threadfence();
    if (tid == 0) { *ticket = 0; if (status) { status[0] = 0; status[1] = 0; } }
    int carry = 0;                           // exclusive scan of the block sums, 1024 at a time
    for (int b0 = 0; b0 < (int)gridDim.x; b0 += 1024) {
        const int b = b0 + tid;
        const int x = b < (int)gridDim.x ? ld_volatile(block_sum + b) : 0;
        int tot;
        const int incl = block_scan_1024(x, warp_sum, &tot);
        if (b < (int)gridDim.x) block_sum[b] = carry + incl - x;
        carry += tot;
    }
    if (tid == 0) block_sum[gridDim.x] = carry;
}

__global__ void __launch_bounds__(1024)
k_cell_scan2(int cells, int *__restrict__ cell_count, int *__restrict__ cell_start,
             const int *__restrict__ block_sum, const int *cond) {
    if (cond && ld_volatile(cond) == 0) return;
    __shared__ int warp_sum[32];
    const int tid = threadIdx.x;
    const int c = blockIdx.x * SCAN_CHUNK + tid * 4;
    const int4 v = load4_counts(cell_count, c, cells);
    const int mine = v.x + v.y + v.z + v.w;
    int total;
    const int incl = block_scan_1024(mine, warp_sum, &total);
    int run = block_sum[blockIdx.x] + incl - mine;
    if (c < cells) { cell_start[c] = run; cell_count[c] = 0; run += v.x; }
    if (c + 1 < cells) { cell_start[c + 1] = run; cell_count[c + 1] = 0; run += v.y; }
    if (c + 2 < cells) { cell_start[c + 2] = run; cell_count[c + 2] = 0; run += v.z; }
    if (c + 3 < cells) { cell_start[c + 3] = run; cell_count[c + 3] = 0; }
    if (blockIdx.x == gridDim.x - 1 && tid == 0) cell_start[cells] = block_sum[gridDim.x];
}

__global__ void __launch_bounds__(256)
k_cell_scatter(int n, const int *__restrict__ cell_of, const int *__restrict__ rank_tmp,
               const int *__restrict__ cell_start, int *__restrict__ perm_tmp, const int *cond) {
    if (cond && ld_volatile(cond) == 0) return;
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    MD_CHECK(cell_start[cell_of[i]] + rank_tmp[i] >= 0 && cell_start[cell_of[i]] + rank_tmp[i] < n);
    perm_tmp[cell_start[cell_of[i]] + rank_tmp[i]] = i;
}

// Canonical order inside a cell by counting: ascending x, ties by id (or index when id == NULL),
// so the sorted state does not depend on atomic arrival order and every x-row of cells is one
// run of slots sorted by x (cells are x-bins), which lets the neighbor-list builder cut its scan
// to the x-range of a tile.  Gathers the payload into the sorted scratch arrays.  One thread per slot.
__global__ void __launch_bounds__(256)
k_cell_order_gather(int n, const int *__restrict__ cell_of, const int *__restrict__ cell_start,
                    const int *__restrict__ perm_tmp, const int *__restrict__ id,
                    const float4 *__restrict__ pos, const float4 *__restrict__ vel,
                    int *__restrict__ perm, float4 *__restrict__ pos_s,
                    float4 *__restrict__ vel_s, int *__restrict__ id_s, const int *cond) {
    if (cond && ld_volatile(cond) == 0) return;
    int s = blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= n) return;
    int i = perm_tmp[s];
    int c = cell_of[i];
    int t0 = cell_start[c], t1 = cell_start[c + 1];
    const float4 pi = pos[i];
    int key = id ? id[i] : i;
    int rank = 0;
    for (int t = t0; t < t1; ++t) {
        int j = perm_tmp[t];
        int kj = id ? id[j] : j;
        float xj = pos[j].x;
        rank += (xj < pi.x) || (xj == pi.x && kj < key);
    }
    int dst = t0 + rank;
    MD_CHECK(i >= 0 && i < n && rank < t1 - t0 && dst >= 0 && dst < n);
    perm[dst] = i;
    pos_s[dst] = pi;
    if (vel_s) vel_s[dst] = vel[i];
    if (id_s) id_s[dst] = id[i];
}

__global__ void __launch_bounds__(256)
k_copy_back(int n, const float4 *__restrict__ pos_s, const float4 *__restrict__ vel_s,
            const int *__restrict__ id_s, float4 *__restrict__ pos, float4 *__restrict__ vel,
            int *__restrict__ id, const int *cond) {
    if (cond && ld_volatile(cond) == 0) return;
    int s = blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= n) return;
    pos[s] = pos_s[s];
    if (vel) vel[s] = vel_s[s];
    if (id) id[s] = id_s[s];
}

// The whole cell list in ONE cooperative launch (grid-wide barriers between the phases instead of
// kernel boundaries).  Pays for small systems, whose five launches are launch- and latency-bound
// (config 1, 16,384 disks: 29 us against 41 us); at 256,000 particles and above the phases are bound by
// their own gathers and the one resident wave of a cooperative grid is slower than full grids
// (52 against 55 us at 256k, 101 against 77 us at 1M), so md_create selects it up to 65,536 particles.  Phases: assign -> scan (every block scans its own run of cells, then adds the
// sum of the runs before it) -> scatter -> in-cell order + payload gather -> copy back (re-sort).
// Same arithmetic and the same results as the five kernels above.  block_sum: gridDim.x + 1 ints.
__global__ void __launch_bounds__(256)
k_cell_all(Geom g, float4 *__restrict__ pos, float4 *__restrict__ vel, int *__restrict__ id,
           int *__restrict__ cell_of, int *__restrict__ rank_tmp, int *__restrict__ cell_count,
           int *__restrict__ cell_start, int *__restrict__ perm_tmp, int *__restrict__ perm,
           float4 *__restrict__ pos_s, float4 *__restrict__ vel_s, int *__restrict__ id_s,
           int *__restrict__ block_sum, int *status, const int *cond, int resort) {
    if (cond && ld_volatile(cond) == 0) return;          // grid-uniform: nobody reaches a barrier
    namespace cg = cooperative_groups;
    cg::grid_group grid = cg::this_grid();
    __shared__ int sh[256];
    const int tid = threadIdx.x, nthr = gridDim.x * blockDim.x, gtid = blockIdx.x * blockDim.x + tid;
    const int n = g.n, cells = g.cells;
    // ---- assign
    for (int i = gtid; i < n; i += nthr) {
        const float4 p = pos[i];
        const int cx = cell_coord(p.x, g.inv_cell[0], g.nc[0]);
        const int cy = cell_coord(p.y, g.inv_cell[1], g.nc[1]);
        const int cz = g.dim == 3 ? cell_coord(p.z, g.inv_cell[2], g.nc[2]) : 0;
        const int c = (cz * g.nc[1] + cy) * g.nc[0] + cx;
        MD_CHECK(c >= 0 && c < cells);
        cell_of[i] = c;
        rank_tmp[i] = atomicAdd(&cell_count[c], 1);
    }
    grid.sync();
    // ---- scan, part 1: block b owns cells [b * per, (b + 1) * per), thread t the run [c0, c1) inside it
    const int per = (cells + gridDim.x - 1) / gridDim.x;
    const int b0 = min(blockIdx.x * per, cells), b1 = min(b0 + per, cells);
    const int tper = (per + blockDim.x - 1) / blockDim.x;
    const int c0 = min(b0 + tid * tper, b1), c1 = min(c0 + tper, b1);
    int sum = 0;
    for (int c = c0; c < c1; ++c) sum += cell_count[c];
    sh[tid] = sum;
    __syncthreads();
    for (int o = 1; o < 256; o <<= 1) {                  // inclusive scan of the 256 run sums
        const int v = tid >= o ? sh[tid - o] : 0;
        __syncthreads();
        sh[tid] += v;
        __syncthreads();
    }
    const int excl = sh[tid] - sum;                       // exclusive prefix of my run inside the block
    if (tid == 255) block_sum[blockIdx.x] = sh[255];
    if (gtid == 0 && status) { status[0] = 0; status[1] = 0; }
    grid.sync();
    // ---- scan, part 2: the sum of the blocks before mine
    int before = 0;
    for (int b = tid; b < (int)blockIdx.x; b += blockDim.x) before += block_sum[b];
    __syncthreads();                                      // sh is read above by every thread
    sh[tid] = before;
    __syncthreads();
    for (int o = 128; o > 0; o >>= 1) { if (tid < o) sh[tid] += sh[tid + o]; __syncthreads(); }
    int run = sh[0] + excl;
    for (int c = c0; c < c1; ++c) {
        const int v = cell_count[c];
        cell_count[c] = 0;
        cell_start[c] = run;
        run += v;
    }
    if (gtid == 0) cell_start[cells] = n;
    grid.sync();
    // ---- scatter
    for (int i = gtid; i < n; i += nthr) {
        const int dst = cell_start[cell_of[i]] + rank_tmp[i];
        MD_CHECK(dst >= 0 && dst < n);
        perm_tmp[dst] = i;
    }
    grid.sync();
    // ---- canonical order inside a cell (ascending x, ties by id) and payload gather
    for (int s = gtid; s < n; s += nthr) {
        const int i = perm_tmp[s];
        const int c = cell_of[i];
        const int t0 = cell_start[c], t1 = cell_start[c + 1];
        const float4 pi = pos[i];
        const int key = id ? id[i] : i;
        int rank = 0;
        for (int t = t0; t < t1; ++t) {
            const int j = perm_tmp[t];
            const int kj = id ? id[j] : j;
            const float xj = pos[j].x;
            rank += (xj < pi.x) || (xj == pi.x && kj < key);
        }
        const int dst = t0 + rank;
        MD_CHECK(rank < t1 - t0 && dst < n);
        perm[dst] = i;
        pos_s[dst] = pi;
        if (vel_s) vel_s[dst] = vel[i];
        if (id_s) id_s[dst] = id[i];
    }
    if (!resort) return;
    grid.sync();
    // ---- copy back: the caller's arrays in cell order
    for (int s = gtid; s < n; s += nthr) {
        pos[s] = pos_s[s];
        if (vel) vel[s] = vel_s[s];
        if (id) id[s] = id_s[s];
    }
}

__global__ void __launch_bounds__(256)
k_gather_pos(int n, const int *__restrict__ perm, const float4 *__restrict__ pos,
             float4 *__restrict__ pos_s) {
    int s = blockIdx.x * blockDim.x + threadIdx.x;
    if (s < n) pos_s[s] = pos[perm[s]];
}

// --------------------------------------------------- neighbor list (L84-L88, L74) ---------
// List layout (md_nbr_layout): tiles of TILE = 32 consecutive particles, slot-major inside a
// tile: entry (i, k) lives at  (i / 32) * 32 * capacity + k * 32 + (i % 32).  A warp that owns
// one tile reads or writes slot k of its 32 particles as one coalesced 128-byte row, which is
// what both the thread-per-particle force kernel and the builder below want.
//
// Builder: one warp per tile, one lane per particle, candidates broadcast from shared memory.
// The 32 sorted slots of a tile span a few consecutive cells; lanes that share an x-row of
// cells (same cy, cz) form a segment and scan the union of their stencils: for each of the
// 3^(D-1) adjacent rows one contiguous run of slots covering x-cells [cx_lo-1, cx_hi+1], plus
// the two periodic wrap pieces when that range leaves the row.  Every piece carries ONE image
// shift (-L on the candidates when the piece is the high-side cell, -L on the lane's own
// coordinate when the piece is the low-side cell), which reproduces the canonical predicate
// bit for bit for every true neighbor (SURVEY A3 "equivalence with a per-cell shift"); lanes
// for which the piece is not adjacent see a separation of at least one cell side >= R and
// reject it, so a union scan adds tests but never hits.  Pieces are staged in chunks of
// NB_CHUNK candidates: the next chunk's global loads are in flight while the current one is
// tested.  Hits are appended to a per-lane shared-memory column (bank = lane, conflict
// free) and the tile is written out row by row, pads (= N, A5) included.

constexpr int TILE = 32;
constexpr int NB_WARPS = 4;        // tiles per block (upper bound; fewer when capacity is large)
constexpr int NB_CHUNK = 128;      // candidates staged per round (4 per lane)

// dynamic shared memory per builder warp: (capacity + 1) rows of 32 ints + one SoA chunk
__host__ __device__ __forceinline__ size_t nb_smem_per_warp(int cap) {
    return (size_t)(cap + 1) * TILE * sizeof(int) + 3 * NB_CHUNK * sizeof(float);
}
__host__ __device__ __forceinline__ size_t nbr_tile_base(int i, int cap) {
    return (size_t)(i >> 5) * (size_t)(TILE * cap);
}
__host__ __device__ __forceinline__ size_t nbr_addr(int i, int k, int cap) {
    return nbr_tile_base(i, cap) + (size_t)k * TILE + (size_t)(i & 31);
}

__device__ __forceinline__ unsigned smem_u32(const void *p) {
    return (unsigned)__cvta_generic_to_shared(p);
}
__device__ __forceinline__ void st_shared(unsigned addr, int v) {
    asm volatile("st.shared.b32 [%0], %1;" ::"r"(addr), "r"(v) : "memory");
}
__device__ __forceinline__ int warp_min(int v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v = min(v, __shfl_xor_sync(FULL, v, o));
    return v;
}
__device__ __forceinline__ int warp_max(int v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v = max(v, __shfl_xor_sync(FULL, v, o));
    return v;
}

// MAPPED = false: particles are physically sorted (resort = 1): slot == particle index.
// MAPPED = true : spos is the sorted copy, map[slot] = particle index (resort = 0).
template <int DIM, bool MAPPED>
__global__ void __launch_bounds__(NB_WARPS * 32)
k_nbr_build(Geom g, const float4 *__restrict__ spos, const int *__restrict__ cell_start,
            const int *__restrict__ map, int *__restrict__ nbr_idx, int *__restrict__ nbr_count,
            int *status, float4 *__restrict__ ref_pos, const int *cond) {
    extern __shared__ __align__(16) unsigned char nb_smem[];
    if (cond && ld_volatile(cond) == 0) return;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int cap = g.capacity;
    const int rows = cap + 1;                          // my own slot is appended too, dropped on write-out
    const size_t per_warp = nb_smem_per_warp(cap);
    int *col = reinterpret_cast<int *>(nb_smem + warp * per_warp) + lane;      // my column
    float *sx = reinterpret_cast<float *>(nb_smem + warp * per_warp + (size_t)rows * TILE * sizeof(int));
    float *sy = sx + NB_CHUNK, *sz = sy + NB_CHUNK;     // staged candidates, negated, SoA
    const int ncx = g.nc[0], ncy = g.nc[1], ncz = g.nc[2];
    const float Lx = g.L[0], Ly = g.L[1], Lz = g.L[2];
    constexpr int ROWS = DIM == 3 ? 9 : 3;
    const int ntiles = (g.n + TILE - 1) / TILE;

    for (int tile = blockIdx.x * (blockDim.x >> 5) + warp; tile < ntiles; tile += gridDim.x * (blockDim.x >> 5)) {
        const int s = tile * TILE + lane;
        const bool act = s < g.n;
        const float4 pi = spos[act ? s : g.n - 1];
        const int cx = cell_coord(pi.x, g.inv_cell[0], ncx);
        const int cy = cell_coord(pi.y, g.inv_cell[1], ncy);
        const int cz = DIM == 3 ? cell_coord(pi.z, g.inv_cell[2], ncz) : 0;
        const int row = act ? cz * ncy + cy : 0x7fffffff;
        const unsigned w0 = smem_u32(col);             // my column (shared-window byte address)
        const unsigned wend = w0 + (unsigned)rows * TILE * sizeof(int);
        unsigned w = w0;                               // next free row
        constexpr unsigned ROWB = TILE * sizeof(int);
        unsigned todo = __ballot_sync(FULL, act);
        while (todo) {
            // ---- next segment: the lanes that share the x-row of the first remaining lane
            const int leader = __ffs(todo) - 1;
            const int r = __shfl_sync(FULL, row, leader);
            const bool inseg = act && row == r;
            todo &= ~__ballot_sync(FULL, inseg);
            const int rcy = __shfl_sync(FULL, cy, leader), rcz = __shfl_sync(FULL, cz, leader);
            const int a = warp_min(inseg ? cx : 0x7fffffff) - 1;
            const int b = warp_max(inseg ? cx : -1) + 1;
            // ---- piece table: lane p < 3*ROWS describes piece p = kind * ROWS + rr
            //      kind 0: x-cells [max(a,0), min(b,ncx-1)]   no x shift
            //      kind 1: x-cell  ncx-1 (a < 0)              candidates shifted by -Lx
            //      kind 2: x-cell  0     (b > ncx-1)          my own x shifted by -Lx
            int t0 = 0, t1 = 0;
            if (lane < 3 * ROWS) {
                const int kind = lane / ROWS, rr = lane % ROWS;
                const int dy = rr % 3 - 1, dz = DIM == 3 ? rr / 3 - 1 : 0;
                int yc = rcy + dy, zc = rcz + dz;
                yc += yc < 0 ? ncy : (yc >= ncy ? -ncy : 0);
                if (DIM == 3) zc += zc < 0 ? ncz : (zc >= ncz ? -ncz : 0);
                const int rowbase = (zc * ncy + yc) * ncx;
                int ca = 0, cb = -1;
                if (kind == 0) { ca = max(a, 0); cb = min(b, ncx - 1); }
                else if (kind == 1) { if (a < 0) { ca = ncx - 1; cb = ncx - 1; } }
                else { if (b > ncx - 1) { ca = 0; cb = 0; } }
                if (cb >= ca) { t0 = cell_start[rowbase + ca]; t1 = cell_start[rowbase + cb + 1]; }
            }
            // ---- walk the pieces; the next chunk is loaded while the current one is tested
            int p = 0, base = 0, pt1 = 0;
            auto seek = [&](int &pp, int &bb, int &tt1) {       // first non-empty piece >= pp
                while (pp < 3 * ROWS) {
                    bb = __shfl_sync(FULL, t0, pp); tt1 = __shfl_sync(FULL, t1, pp);
                    if (bb < tt1) return;
                    ++pp;
                }
            };
            seek(p, base, pt1);
            float4 q[NB_CHUNK / 32];
            auto fetch = [&](int bb, int tt1) {
#pragma unroll
                for (int u = 0; u < NB_CHUNK / 32; ++u) {
                    const int t = bb + u * 32 + lane;
                    if (t < tt1) q[u] = spos[t];
                }
            };
            if (p < 3 * ROWS) fetch(base, pt1);
            while (p < 3 * ROWS) {
                const int kind = p / ROWS, rr = p % ROWS;
                const int dy = rr % 3 - 1, dz = DIM == 3 ? rr / 3 - 1 : 0;
                // image shifts of this piece: candidates by -L when the piece is the
                // high-side row/cell, my own coordinate by -L when it is the low-side one
                const float sjx = kind == 1 ? Lx : 0.0f;
                const float sjy = rcy + dy < 0 ? Ly : 0.0f;
                const float sjz = (DIM == 3 && rcz + dz < 0) ? Lz : 0.0f;
                const float pix = kind == 2 ? __fsub_rn(pi.x, Lx) : pi.x;
                const float piy = rcy + dy >= ncy ? __fsub_rn(pi.y, Ly) : pi.y;
                const float piz = (DIM == 3 && rcz + dz >= ncz) ? __fsub_rn(pi.z, Lz) : pi.z;
                const int m = min(NB_CHUNK, pt1 - base);
                // stage -(candidate - shift), structure of arrays; the tail of the last group of
                // four is filled with a far-away point so the test loop needs no remainder
#pragma unroll
                for (int u = 0; u < NB_CHUNK / 32; ++u) {
                    const int c = u * 32 + lane;
                    if (c < m) {
                        sx[c] = __fsub_rn(sjx, q[u].x);
                        sy[c] = __fsub_rn(sjy, q[u].y);
                        if (DIM == 3) sz[c] = __fsub_rn(sjz, q[u].z);
                    } else if (c < ((m + 3) & ~3)) {
                        sx[c] = 1e18f; sy[c] = 0.0f;
                        if (DIM == 3) sz[c] = 0.0f;
                    }
                }
                __syncwarp();
                // next chunk
                int np = p, nbase = base + NB_CHUNK, npt1 = pt1;
                if (nbase >= pt1) { ++np; seek(np, nbase, npt1); }
                if (np < 3 * ROWS) fetch(nbase, npt1);
                // test the staged chunk, two candidates per packed fp32x2 instruction
                // (sm_100 FADD2 / FMUL2 / FFMA2, round-to-nearest: the bits of the scalar form)
                if (inseg) {
                    const float2 px2 = make_float2(pix, pix), py2 = make_float2(piy, piy);
                    const float2 pz2 = make_float2(piz, piz);
                    for (int c = 0; c < m; c += 4) {
                        const float4 X = *reinterpret_cast<const float4 *>(sx + c);
                        const float4 Y = *reinterpret_cast<const float4 *>(sy + c);
                        const float2 dxa = __fadd2_rn(px2, make_float2(X.x, X.y));
                        const float2 dxb = __fadd2_rn(px2, make_float2(X.z, X.w));
                        const float2 dya = __fadd2_rn(py2, make_float2(Y.x, Y.y));
                        const float2 dyb = __fadd2_rn(py2, make_float2(Y.z, Y.w));
                        float2 ra = __ffma2_rn(dya, dya, __fmul2_rn(dxa, dxa));
                        float2 rb = __ffma2_rn(dyb, dyb, __fmul2_rn(dxb, dxb));
                        if (DIM == 3) {
                            const float4 Z = *reinterpret_cast<const float4 *>(sz + c);
                            const float2 dza = __fadd2_rn(pz2, make_float2(Z.x, Z.y));
                            const float2 dzb = __fadd2_rn(pz2, make_float2(Z.z, Z.w));
                            ra = __ffma2_rn(dza, dza, ra);
                            rb = __ffma2_rn(dzb, dzb, rb);
                        }
                        const int t = base + c;
                        const bool h0 = ra.x < g.R2, h1 = ra.y < g.R2, h2 = rb.x < g.R2, h3 = rb.y < g.R2;
                        if (w + 4u * ROWB <= wend) {          // room for all four
                            if (h0) st_shared(w, t);
                            w += h0 ? ROWB : 0u;
                            if (h1) st_shared(w, t + 1);
                            w += h1 ? ROWB : 0u;
                            if (h2) st_shared(w, t + 2);
                            w += h2 ? ROWB : 0u;
                            if (h3) st_shared(w, t + 3);
                            w += h3 ? ROWB : 0u;
                        } else {                                           // overflowing row: count only
                            if (h0 && w < wend) st_shared(w, t);
                            w += h0 ? ROWB : 0u;
                            if (h1 && w < wend) st_shared(w, t + 1);
                            w += h1 ? ROWB : 0u;
                            if (h2 && w < wend) st_shared(w, t + 2);
                            w += h2 ? ROWB : 0u;
                            if (h3 && w < wend) st_shared(w, t + 3);
                            w += h3 ? ROWB : 0u;
                        }
                    }
                }
                __syncwarp();
                p = np; base = nbase; pt1 = npt1;
            }
        }
        // ---- write the tile out (rows of 32 consecutive ints; scattered when MAPPED), dropping
        //      my own slot, which the scan appended like any other point at distance 0
        const int appended = (int)((w - w0) / ROWB);
        const int cnt = act ? appended - 1 : 0;        // true count
        const int stored = min(appended, rows);
        int *out = nullptr;
        if (!MAPPED) out = nbr_idx + nbr_tile_base(s, cap) + lane;
        else if (act) { const int i = map[s]; out = nbr_idx + nbr_tile_base(i, cap) + (i & 31); }
        if (out) {
            int ko = 0;
            for (int k = 0; k < stored; ++k) {
                const int v = col[k * TILE];
                if (v != s && ko < cap) { out[ko * TILE] = MAPPED ? map[v] : v; ++ko; }
            }
            for (; ko < cap; ++ko) out[ko * TILE] = g.n;                  // pad = N (A5)
        }
        if (act) {
            const int i = MAPPED ? map[s] : s;
            nbr_count[i] = cnt; ref_pos[i] = pi;
        }
        const int mx = warp_max(act ? cnt : 0);
        if (lane == 0) {
            if (mx > ld_volatile(status + 1)) atomicMax(status + 1, mx);
            if (mx > cap) status[0] = 1;
        }
        __syncwarp();
    }
}

// ----------------------------------------------------- rebuild test (L49 §3.1) -----------

template <int DIM>
__device__ __forceinline__ float disp2_from_ref(const Geom &g, float4 p, float4 r) {
    float dx = min_image(p.x, r.x, g.L[0], g.h[0]);
    float dy = min_image(p.y, r.y, g.L[1], g.h[1]);
    float d2 = fmaf(dy, dy, dx * dx);
    if (DIM == 3) {
        float dz = min_image(p.z, r.z, g.L[2], g.h[2]);
        d2 = fmaf(dz, dz, d2);
    }
    return d2;
}

template <int DIM>
__global__ void __launch_bounds__(256)
k_needs_rebuild(Geom g, const float4 *__restrict__ pos, const float4 *__restrict__ ref,
                int *flag) {
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    bool moved = false;
    if (i < g.n) moved = disp2_from_ref<DIM>(g, pos[i], ref[i]) > g.half_skin2;
    if (__any_sync(FULL, moved) && (threadIdx.x & 31) == 0) *flag = 1;
}

// ------------------------------------------- velocity Verlet, first half (L100 §3.3.1) ----
// v += dt/(2m) F;  r = mu(r, dt v);  rebuild test against the reference positions.
// HAS_COND: the step runs inside a CUDA graph whose rebuild kernels sit in an IF node; the warp
// that sees a particle beyond skin/2 also raises the node's condition (default 0 per launch).
// v += a F on m particles (the closing half-kick as a kernel of its own: md_half_kick; inside
// md_nve_step it is the force kernel's epilogue, same fma on the same rounded force)
__global__ void __launch_bounds__(256)
k_half_kick(int m, int dim, float4 *__restrict__ vel, const float4 *__restrict__ force, float a) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= m) return;
    float4 v = vel[i];
    const float4 f = force[i];
    v.x = fmaf(a, f.x, v.x); v.y = fmaf(a, f.y, v.y);
    if (dim == 3) v.z = fmaf(a, f.z, v.z);
    vel[i] = v;
}

template <int DIM, bool HAS_COND>
__global__ void __launch_bounds__(256)
k_kick_drift(Geom g, float4 *__restrict__ pos, float4 *__restrict__ vel,
             const float4 *__restrict__ force, const float4 *__restrict__ ref, float a, float dt,
             int *flag, cudaGraphConditionalHandle cond) {
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    bool moved = false;
    if (i < g.n) {
        float4 p = pos[i], v = vel[i], f = force[i];
        v.x = fmaf(a, f.x, v.x);
        v.y = fmaf(a, f.y, v.y);
        p.x = wrap(fmaf(dt, v.x, p.x), g.L[0], g.inv_L[0]);
        p.y = wrap(fmaf(dt, v.y, p.y), g.L[1], g.inv_L[1]);
        if (DIM == 3) {
            v.z = fmaf(a, f.z, v.z);
            p.z = wrap(fmaf(dt, v.z, p.z), g.L[2], g.inv_L[2]);
        }
        pos[i] = p; vel[i] = v;
        moved = disp2_from_ref<DIM>(g, p, ref[i]) > g.half_skin2;
    }
    if (__any_sync(FULL, moved) && (threadIdx.x & 31) == 0) {
        *flag = 1;
        if (HAS_COND) cudaGraphSetConditional(cond, 1);
    }
}

// ------------------------------------- pair energy / force over the list (L78, L80, L104) --
// TPP lanes per particle (1, 2 or 4); with TPP = 1 a warp is exactly one list tile and slot k of
// its 32 particles is one coalesced 128-byte row.  Neighbor positions are gathered as float4
// through L1 (particles are cell-sorted, so the 32 lanes walk nearby lines).
//
// Precision: displacements are exact -- away from the box faces
// the fp32 difference of two coordinates >= 2 that are < 4 apart is exact, near a face the
// difference and the image shift are taken in fp64 -- and the pair chain r2 -> 1/r2 -> force
// coefficient and all accumulation run in fp64 (reciprocal: hardware seed + Newton steps on
// the FP64 pipe).  Results round to fp32 once, on store.  Pure fp32 pair arithmetic cannot hold
// the 1e-5 force tolerance: its typical error is already 3e-6 of |F| because the first shell
// sits where the LJ force changes sign.  The in/out decision at r_cut is taken on the fp64 r2.

struct Acc64 { double fx, fy, fz, e; };

// 1/x to ~1e-12: hardware seed (MUFU.RCP64H, measured 9.4e-7 on B200) + one Newton step.
__device__ __forceinline__ double rcp64(double x) {
    double y;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
    return fma(y, fma(-x, y, 1.0), y);
}

// One pair, LJ.  With y = 1/r2 and s6 = sig^6 y^3 the force coefficient is
// 24 eps s6 (2 s6 - 1) y = 24 eps sig^6 * y^4 (2 sig^6 y^3 - 1); the constant 24 eps sig^6 is
// applied once per particle.  Energy term: s6 (s6 - 1) - u_cut / (4 eps), times 4 eps / 2 later.
template <bool ENERGY>
__device__ __forceinline__ void lj_pair64(const Pair &pp, double dx, double dy, double dz,
                                          bool valid, Acc64 &a) {
    const double r2 = fma(dz, dz, fma(dy, dy, dx * dx));
    const bool in = valid && r2 < pp.drc2;
    const double y = rcp64(in ? r2 : 1.0);
    const double y2 = y * y;
    const double y3 = y2 * y;
    const double t = fma(pp.dsig6x2, y3, -1.0);           // 2 s6 - 1
    double c = (y2 * y2) * t;
    c = in ? c : 0.0;
    a.fx = fma(c, dx, a.fx); a.fy = fma(c, dy, a.fy); a.fz = fma(c, dz, a.fz);
    if (ENERGY) {
        const double s6 = 0.5 * pp.dsig6x2 * y3;
        a.e += in ? fma(s6, s6, -s6) - pp.du_cut4 : 0.0;
    }
}

// One pair, harmonic soft sphere: u = eps/2 (1 - r/d)^2, F = eps/d (1 - r/d) dvec/r for r < d.
template <bool ENERGY>
__device__ __forceinline__ void soft_pair64(const Pair &pp, double dx, double dy, double dz,
                                            double dsum, bool valid, Acc64 &a) {
    const double r2 = fma(dz, dz, fma(dy, dy, dx * dx));
    const double dij = 0.5 * dsum;
    const double r = sqrt(r2);
    const bool in = valid && r < dij;
    const double x = 1.0 - r / dij;
    const double c = (in && r > 0.0) ? x / (dij * r) : 0.0;
    a.fx = fma(c, dx, a.fx); a.fy = fma(c, dy, a.fy); a.fz = fma(c, dz, a.fz);
    if (ENERGY) a.e += in ? x * x : 0.0;
}

// One pair, Morse [75] (L104): u = D (1 - x)^2 - D, x = exp(-alpha (r - r0)); the force
// coefficient -u'(r)/r = -2 D alpha x (1 - x) / r; D is applied once per particle.
// 1/sqrt(x), x > 0 of ordinary magnitude: the fp32 reciprocal square root refined by one Newton
// step in fp64 (relative error ~1e-13), in place of an fp64 square root and an fp64 division.
__device__ __forceinline__ double rsqrt64(double x) {
    const double y = (double)rsqrtf((float)x);
    return y * fma(-0.5 * x, y * y, 1.5);
}

template <bool ENERGY>
__device__ __forceinline__ void morse_pair64(const Pair &pp, double dx, double dy, double dz,
                                             bool valid, Acc64 &a) {
    const double r2 = fma(dz, dz, fma(dy, dy, dx * dx));
    const bool in = valid && r2 < pp.drc2;
    const double r2v = in ? r2 : 1.0, r2s = r2v > 0.0 ? r2v : 1.0;
    const double ir = rsqrt64(r2s), r = r2v * ir;                   // r = 0 for coincident particles
    const double x = exp(-pp.dalpha * (r - pp.dr0));
    double c = (in && r2 > 0.0) ? -2.0 * pp.dalpha * x * (1.0 - x) * ir : 0.0;
    a.fx = fma(c, dx, a.fx); a.fy = fma(c, dy, a.fy); a.fz = fma(c, dz, a.fz);
    if (ENERGY) a.e += in ? (1.0 - x) * (1.0 - x) - 1.0 - pp.du_cutm : 0.0;
}

// One pair, Buckingham-type exp-6 [71-73] (L104): u = A exp(-B r) - C / r^6; the force coefficient
// -u'(r)/r = (A B exp(-B r) - 6 C / r^7) / r.  Nothing is factored out (fs = 1).
template <bool ENERGY>
__device__ __forceinline__ void buck_pair64(const Pair &pp, double dx, double dy, double dz,
                                            bool valid, Acc64 &a) {
    const double r2 = fma(dz, dz, fma(dy, dy, dx * dx));
    const bool in = valid && r2 < pp.drc2 && r2 > 0.0;
    const double r2s = in ? r2 : 1.0;
    const double r = sqrt(r2s), x = pp.dA * exp(-pp.dalpha * r);
    const double y = rcp64(r2s), y3 = y * y * y;                    // 1/r^6
    const double c = in ? (pp.dalpha * x * r - 6.0 * pp.dC * y3) * y : 0.0;   // (B x r - 6C/r^6)/r^2
    a.fx = fma(c, dx, a.fx); a.fy = fma(c, dy, a.fy); a.fz = fma(c, dz, a.fz);
    if (ENERGY) a.e += in ? x - pp.dC * y3 - pp.du_cutm : 0.0;
}

// One pair, species x species LJ (L104; the sigma matrix of L298-L305): as lj_pair64 with the
// constants of the pair's species; nothing is factored out (fs = es = 1).
// The species tables as one block of shared memory (a per-pair index into kernel parameters is a
// divergent constant load, replayed once per distinct species pair in the warp):
// sp[0..15] = 2 sigma^6, [16..31] = 24 eps sigma^6, [32..47] = 2 eps, [48..63] = rc^2, [64..79] = shift term.
constexpr int SP_TAB = 80;
__device__ __forceinline__ void species_tables_to_shared(const Pair &pp, double *sp) {
    for (int t = threadIdx.x; t < 16; t += blockDim.x) {
        sp[t] = pp.sp_sig6x2[t]; sp[16 + t] = pp.sp_fs[t]; sp[32 + t] = pp.sp_es[t];
        sp[48 + t] = pp.sp_rc2[t]; sp[64 + t] = pp.sp_ucut4[t];
    }
    __syncthreads();
}

template <bool ENERGY>
__device__ __forceinline__ void ljs_pair64(const Pair &pp, const double *sp, double dx, double dy, double dz,
                                           float wi, float wj, bool valid, Acc64 &a) {
    const int sa = min(max((int)wi, 0), pp.ns - 1), sb = min(max((int)wj, 0), pp.ns - 1);
    const int t = sa * pp.ns + sb;
    const double sig6x2 = sp[t];
    const double r2 = fma(dz, dz, fma(dy, dy, dx * dx));
    const bool in = valid && r2 < sp[48 + t];
    const double y = rcp64(in ? r2 : 1.0);
    const double y2 = y * y, y3 = y2 * y;
    const double tt = fma(sig6x2, y3, -1.0);
    const double c = in ? sp[16 + t] * (y2 * y2) * tt : 0.0;
    a.fx = fma(c, dx, a.fx); a.fy = fma(c, dy, a.fy); a.fz = fma(c, dz, a.fz);
    if (ENERGY) {
        const double s6 = 0.5 * sig6x2 * y3;
        a.e += in ? sp[32 + t] * (fma(s6, s6, -s6) - sp[64 + t]) : 0.0;
    }
}

// erfc(z) / exp(-z^2) for z in [0, 8] as a polynomial in u = (1 - 0.75 z) / (1 + 0.5 z), which maps [0, 8] onto
// [1, -1]: degree-18 fit of the scaled complementary error function at Chebyshev nodes, relative error 1.4e-14
// as an fp64 Horner sum (checked against scipy.special.erfcx on 400,001 points).  bks_pair64 has exp(-z^2)
// already, so this replaces a library erfc (which computes its own exponential) by 18 fused multiply-adds.
__device__ __forceinline__ double erfcx_poly64(double u) {
    double p = -1.24573901670517321e-09;
    p = fma(p, u, 1.89464270519370702e-09); p = fma(p, u, 9.34182355916646586e-09);
    p = fma(p, u, -3.17681098022790105e-08); p = fma(p, u, 7.15041583811810360e-09);
    p = fma(p, u, 2.07737375250764355e-07); p = fma(p, u, -5.96731148973458073e-07);
    p = fma(p, u, -1.91245751497578349e-07); p = fma(p, u, 5.68144898215161673e-06);
    p = fma(p, u, -1.11144478235017232e-05); p = fma(p, u, -3.27761796276374571e-05);
    p = fma(p, u, 1.75746287383741513e-04); p = fma(p, u, 1.23661544233961182e-04);
    p = fma(p, u, -2.35992473798610517e-03); p = fma(p, u, -1.43343007865939266e-03);
    p = fma(p, u, 4.04916498055216470e-02); p = fma(p, u, 1.85195333821254582e-01);
    p = fma(p, u, 4.26711073374306360e-01); p = fma(p, u, 3.51134694028905514e-01);
    return p;
}

// One pair, BKS-type (L104 [71-73]; A27): exp-6 with A, B, C of the species pair plus the
// damped shifted-force Coulomb term between the species' charges; one cutoff; nothing factored out.
//   -u'/r = (A B e^{-B r} - 6 C / r^7)/r + k q q' (erfc(a r)/r^2 + (2a/sqrt(pi)) e^{-a^2 r^2}/r - f_c)/r
template <bool ENERGY>
__device__ __forceinline__ void bks_pair64(const Pair &pp, const double *sp, double dx, double dy, double dz,
                                           float wi, float wj, bool valid, Acc64 &a) {
    const int sa = min(max((int)wi, 0), pp.ns - 1), sb = min(max((int)wj, 0), pp.ns - 1);
    const int t = sa * pp.ns + sb;
    const double r2 = fma(dz, dz, fma(dy, dy, dx * dx));
    const bool in = valid && r2 < pp.drc2 && r2 > 0.0;
    const double r2s = in ? r2 : 1.0;
    const double ir = rsqrt64(r2s), r = r2s * ir, y = ir * ir, y3 = y * y * y;
    const double x = sp[t] * exp(-sp[16 + t] * r), C6 = sp[32 + t] * y3, qq = sp[48 + t];
    const double z = pp.bks_a * r, e2 = exp(-pp.bks_a * pp.bks_a * r2s);
    const double er = z < 8.0 ? e2 * erfcx_poly64((1.0 - 0.75 * z) * rcp64(1.0 + 0.5 * z)) : 0.0;   // erfc(8) = 1e-29
    const double ex = pp.bks_tsp * e2;
    const double c = in ? (sp[16 + t] * x * r - 6.0 * C6) * y + qq * (er * y + ex * ir - pp.bks_fc) * ir : 0.0;
    a.fx = fma(c, dx, a.fx); a.fy = fma(c, dy, a.fy); a.fz = fma(c, dz, a.fz);
    if (ENERGY) a.e += in ? x - C6 - sp[64 + t] + qq * (er * ir - pp.bks_ec + pp.bks_fc * (r - pp.bks_rc)) : 0.0;
}

// Per-thread view of the space for the pair loop.
template <int DIM>
struct Me {
    float4 pi;
    double xi, yi, zi, Lx, Ly, Lz;
    float hx, hy, hz;
};

// Displacement r_i - r_j (nearest image) in fp64.  WRAP = false: the warp is away from every
// face, no pair crosses the boundary; the fp32 difference is exact for every pair that
// matters (coordinates >= r_cut + 2 skin, separations < 4) and at worst 1 rounding (6e-8 of a
// distance > 2, where the force is tiny) otherwise.  WRAP = true: difference and image shift
// in fp64; the image is picked on the fp32 difference (|d| < L/2 - or > L/2 + by a wide margin).
template <int DIM, bool WRAP>
__device__ __forceinline__ void displacement(const Me<DIM> &me, const float4 &q, double &dx,
                                             double &dy, double &dz) {
    const float fx = me.pi.x - q.x, fy = me.pi.y - q.y, fz = me.pi.z - q.z;
    if (!WRAP) {
        dx = (double)fx; dy = (double)fy; dz = DIM == 3 ? (double)fz : 0.0;
    } else {
        dx = me.xi - (double)q.x; dy = me.yi - (double)q.y;
        dx -= fx > me.hx ? me.Lx : (fx < -me.hx ? -me.Lx : 0.0);
        dy -= fy > me.hy ? me.Ly : (fy < -me.hy ? -me.Ly : 0.0);
        dz = 0.0;
        if (DIM == 3) {
            dz = me.zi - (double)q.z;
            dz -= fz > me.hz ? me.Lz : (fz < -me.hz ? -me.Lz : 0.0);
        }
    }
}

template <int KIND, int DIM, bool ENERGY, bool WRAP>
__device__ __forceinline__ void pair_any(const Pair &pp, const Me<DIM> &me, const float4 &q,
                                         bool valid, Acc64 &acc, const double *sp = nullptr) {
    double dx, dy, dz;
    displacement<DIM, WRAP>(me, q, dx, dy, dz);
    if (KIND == 0) lj_pair64<ENERGY>(pp, dx, dy, dz, valid, acc);
    else if (KIND == 2) morse_pair64<ENERGY>(pp, dx, dy, dz, valid, acc);
    else if (KIND == 3) buck_pair64<ENERGY>(pp, dx, dy, dz, valid, acc);
    else if (KIND == 4) ljs_pair64<ENERGY>(pp, sp, dx, dy, dz, me.pi.w, q.w, valid, acc);
    else if (KIND == 5) bks_pair64<ENERGY>(pp, sp, dx, dy, dz, me.pi.w, q.w, valid, acc);
    else soft_pair64<ENERGY>(pp, dx, dy, dz, (double)me.pi.w + (double)q.w, valid, acc);
}

template <int DIM>
__device__ __forceinline__ bool near_face(const Geom &g, const float4 &p) {
    bool near = p.x < g.face || p.x > g.L[0] - g.face || p.y < g.face || p.y > g.L[1] - g.face;
    if (DIM == 3) near = near || p.z < g.face || p.z > g.L[2] - g.face;
    return near;
}

template <int DIM>
__device__ __forceinline__ Me<DIM> make_me(const Geom &g, const float4 &pi) {
    Me<DIM> me;
    me.pi = pi; me.xi = pi.x; me.yi = pi.y; me.zi = pi.z;
    me.Lx = g.L[0]; me.Ly = g.L[1]; me.Lz = g.L[2];
    me.hx = g.h[0]; me.hy = g.h[1]; me.hz = g.h[2];
    return me;
}

// Epilogue shared by both force kernels: scale, round once, store, optional half-kick, energy
// reduction and step bookkeeping.
template <int KIND, int DIM, bool ENERGY>
__device__ __forceinline__ void force_epilogue(const Pair &pp, const Acc64 &acc, bool owner, int i,
                                               float4 *__restrict__ force, float4 *__restrict__ vel,
                                               float a, double *energy_total, const Book &book,
                                               int gid) {
    const double fs = KIND == 0 ? 12.0 * pp.deps * pp.dsig6x2 : (KIND == 3 || KIND == 4 || KIND == 5 ? 1.0 : pp.deps);   // 24 eps sig^6 | eps | D | 1
    const double es = KIND == 0 ? 2.0 * pp.deps
                    : (KIND == 2 ? 0.5 * pp.deps : (KIND == 3 || KIND == 5 ? 0.5 : (KIND == 4 ? 1.0 : 0.25 * pp.deps)));   // 1/2 * (4 eps | D | 1 | eps/2)
    const float fx = (float)(fs * acc.fx), fy = (float)(fs * acc.fy), fz = (float)(fs * acc.fz);
    const double e64 = ENERGY ? es * acc.e : 0.0;
    if (owner) {
        force[i] = make_float4(fx, fy, DIM == 3 ? fz : 0.0f, (float)e64);
        if (vel) {
            float4 v = vel[i];
            v.x = fmaf(a, fx, v.x); v.y = fmaf(a, fy, v.y);
            if (DIM == 3) v.z = fmaf(a, fz, v.z);
            vel[i] = v;
        }
    }
    if (ENERGY && energy_total) {
        __shared__ double red[4];
        double x = owner ? e64 : 0.0;
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) x += __shfl_xor_sync(FULL, x, o);
        if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = x;
        __syncthreads();
        if (threadIdx.x == 0) {
            double t = 0.0;
            for (int w = 0; w < (int)(blockDim.x >> 5); ++w) t += red[w];
            atomicAdd(energy_total, t);
        }
    }
    if (book.done && gid == 0) *book.done += 1;
    if (book.stats && gid == 0) {
        if (ld_volatile(book.flag)) {
            book.stats[1] += 1;
            int mc = ld_volatile(book.status + 1);
            if (mc > book.stats[3]) book.stats[3] = mc;
            if (ld_volatile(book.status) && book.stats[2] < 0) book.stats[2] = book.stats[0];
            if (!book.clear) *book.flag = 0;
        }
        if (book.clear) *book.clear = 0;
        book.stats[0] += 1;
    }
}

// ---- generic kernel: TPP lanes per particle (small systems: more warps, shorter chains) ----
// vel != NULL: also the second half-kick v += a F (L100).  energy_total != NULL (ENERGY only):
// adds sum_i e_i in fp64 (one atomic per block).  book.stats != NULL: per-step bookkeeping.
template <int KIND, int DIM, int TPP, bool ENERGY>
__global__ void __launch_bounds__(128)
k_force(Geom g, Pair pp, const float4 *__restrict__ pos, const int *__restrict__ nbr_idx,
        const int *__restrict__ nbr_count, float4 *__restrict__ force, float4 *__restrict__ vel,
        float a, double *energy_total, Book book, int i0) {
    __shared__ double sp[KIND == 4 || KIND == 5 ? SP_TAB : 1];
    if (KIND == 4 || KIND == 5) species_tables_to_shared(pp, sp);
    const int gid = i0 * TPP + blockIdx.x * blockDim.x + threadIdx.x;     // i0: first particle of the range
    if (book_skips(book, gid)) return;
    const int i = gid / TPP, sub = gid % TPP;
    const bool active = i < g.n;
    const int ii = active ? i : g.n - 1;
    const Me<DIM> me = make_me<DIM>(g, pos[ii]);
    const int cnt = active ? min(nbr_count[ii], g.capacity) : 0;
    const int *col = nbr_idx + nbr_tile_base(ii, g.capacity) + (ii & 31);
    const bool wrap_path = __any_sync(FULL, active && near_face<DIM>(g, me.pi));
    Acc64 acc = {0.0, 0.0, 0.0, 0.0};
    constexpr int U = 4;
    for (int k = sub; k < cnt; k += U * TPP) {
        int j[U]; float4 q[U];
#pragma unroll
        for (int u = 0; u < U; ++u) { const int kk = k + u * TPP; j[u] = kk < cnt ? col[kk * TILE] : ii; }
#pragma unroll
        for (int u = 0; u < U; ++u) { MD_CHECK(j[u] >= 0 && j[u] < g.ntot); q[u] = pos[j[u]]; }
        if (!wrap_path) {
#pragma unroll
            for (int u = 0; u < U; ++u) pair_any<KIND, DIM, ENERGY, false>(pp, me, q[u], k + u * TPP < cnt, acc, sp);
        } else {
#pragma unroll
            for (int u = 0; u < U; ++u) pair_any<KIND, DIM, ENERGY, true>(pp, me, q[u], k + u * TPP < cnt, acc, sp);
        }
    }
#pragma unroll
    for (int o = TPP / 2; o > 0; o >>= 1) {
        acc.fx += __shfl_xor_sync(FULL, acc.fx, o);
        acc.fy += __shfl_xor_sync(FULL, acc.fy, o);
        acc.fz += __shfl_xor_sync(FULL, acc.fz, o);
        if (ENERGY) acc.e += __shfl_xor_sync(FULL, acc.e, o);
    }
    force_epilogue<KIND, DIM, ENERGY>(pp, acc, active && sub == 0, i, force, vel, a, energy_total, book, gid);
}

// ---- streaming kernel: one warp = one list tile, one lane per particle.  The tile's index
// block (rows of 128 bytes, contiguous in HBM) is streamed into shared memory by the TMA engine
// (cp.async.bulk + mbarrier) FS_STAGES chunks of FS_ROWS rows ahead of the arithmetic, so the
// only long-latency loads a lane waits for are its position gathers (L1 / L2 hits).
constexpr int FS_ROWS = 16;       // rows per chunk (2 KiB)
constexpr int FS_STAGES = 3;      // chunks in flight per warp
constexpr int FS_WARPS = 4;

__device__ __forceinline__ void mbar_init(unsigned bar, int count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(unsigned bar, unsigned bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void bulk_g2s(unsigned dst, const void *src, unsigned bytes, unsigned bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(dst), "l"(src), "r"(bytes), "r"(bar) : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned bar, unsigned parity) {
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "WAIT_LOOP:\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n\t"
        "@p bra WAIT_DONE;\n\t"
        "bra WAIT_LOOP;\n\t"
        "WAIT_DONE:\n\t}" ::"r"(bar), "r"(parity) : "memory");
}

template <int KIND, int DIM, bool ENERGY>
__global__ void __launch_bounds__(FS_WARPS * 32)
k_force_stream(Geom g, Pair pp, const float4 *__restrict__ pos, const int *__restrict__ nbr_idx,
               const int *__restrict__ nbr_count, float4 *__restrict__ force,
               float4 *__restrict__ vel, float a, double *energy_total, Book book, int i0) {
    __shared__ __align__(128) int s_idx[FS_WARPS][FS_STAGES][FS_ROWS * TILE];
    __shared__ __align__(8) unsigned long long s_bar[FS_WARPS][FS_STAGES];
    __shared__ double sp[KIND == 4 || KIND == 5 ? SP_TAB : 1];
    if (KIND == 4 || KIND == 5) species_tables_to_shared(pp, sp);
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int gid = i0 + blockIdx.x * blockDim.x + threadIdx.x;
    if (book_skips(book, gid)) return;
    const int i = gid;
    const bool active = i < g.n;
    const int ii = active ? i : g.n - 1;
    if (lane == 0) {
#pragma unroll
        for (int s = 0; s < FS_STAGES; ++s) mbar_init(smem_u32(&s_bar[warp][s]), 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    }
    const int cnt = active ? min(nbr_count[ii], g.capacity) : 0;
    const int maxcnt = warp_max(cnt);                  // also orders the barrier init (shuffles sync)
    const int nch = (maxcnt + FS_ROWS - 1) / FS_ROWS;
    const int *tile_src = nbr_idx + nbr_tile_base(gid, g.capacity);     // gid: valid for the whole tile
    auto issue = [&](int c) {
        const int st = c % FS_STAGES;
        const unsigned bytes = (unsigned)min(FS_ROWS, maxcnt - c * FS_ROWS) * TILE * sizeof(int);
        const unsigned bar = smem_u32(&s_bar[warp][st]);
        mbar_expect_tx(bar, bytes);
        bulk_g2s(smem_u32(&s_idx[warp][st][0]), tile_src + (size_t)c * FS_ROWS * TILE, bytes, bar);
    };
    __syncwarp();
    if (lane == 0)
        for (int c = 0; c < min(FS_STAGES, nch); ++c) issue(c);
    const Me<DIM> me = make_me<DIM>(g, pos[ii]);
    const bool wrap_path = __any_sync(FULL, active && near_face<DIM>(g, me.pi));
    Acc64 acc = {0.0, 0.0, 0.0, 0.0};
    constexpr int U = 4;
    for (int c = 0; c < nch; ++c) {
        const int st = c % FS_STAGES;
        mbar_wait(smem_u32(&s_bar[warp][st]), (unsigned)(c / FS_STAGES) & 1u);
        const int *sm = &s_idx[warp][st][lane];
        const int k0 = c * FS_ROWS;
        const int rows = min(FS_ROWS, maxcnt - k0);
        for (int r = 0; r < rows; r += U) {
            int j[U]; float4 q[U];
#pragma unroll
            for (int u = 0; u < U; ++u) j[u] = k0 + r + u < cnt ? sm[(r + u) * TILE] : ii;
#pragma unroll
            for (int u = 0; u < U; ++u) { MD_CHECK(j[u] >= 0 && j[u] < g.ntot); q[u] = pos[j[u]]; }
            if (!wrap_path) {
#pragma unroll
                for (int u = 0; u < U; ++u) pair_any<KIND, DIM, ENERGY, false>(pp, me, q[u], k0 + r + u < cnt, acc, sp);
            } else {
#pragma unroll
                for (int u = 0; u < U; ++u) pair_any<KIND, DIM, ENERGY, true>(pp, me, q[u], k0 + r + u < cnt, acc, sp);
            }
        }
        __syncwarp();                                  // every lane is done reading this stage
        if (lane == 0 && c + FS_STAGES < nch) issue(c + FS_STAGES);
    }
    force_epilogue<KIND, DIM, ENERGY>(pp, acc, active, i, force, vel, a, energy_total, book, gid);
}

} // namespace mdk
