// md_nbr2.cuh -- neighbor-list builder, second design (L84-L88, L74).
//
// Same decomposition as k_nbr_build (md_kernels.cuh): one warp per list tile, one lane per
// particle, the lanes that share an x-row of cells scan the union of their stencils piece by
// piece, every piece carrying ONE image shift, candidates staged negated in shared memory and
// tested two at a time with packed fp32x2 arithmetic (bit-identical to the scalar canonical
// predicate).  What changed is how a hit is recorded.  k_nbr_build appended every hit to a
// per-lane column of capacity + 1 rows in shared memory (16.5 KB per warp at capacity 128:
// 12 warps per SM) through a chain of predicated store / pointer bumps, 12.5 instructions per
// candidate.  Here the sign bit of fl(r2 - R2) -- set exactly when r2 < R2 -- is shifted into a
// per-lane bit mask, one funnel shift per candidate and no branch, 32 candidates per word; the
// masks of up to NB2_WORDS words (4 KB per warp) are expanded afterwards, every lane pulling
// its next set bit per iteration, so row k of the tile leaves as one coalesced 128-byte store.
#pragma once
#include "md_kernels.cuh"

namespace mdk {

constexpr int NB2_WARPS = 8;          // tiles per block
constexpr int NB2_WORDS = 32;         // mask words per lane per batch (1024 candidates)
constexpr int NB2_CHUNK = 128;        // candidates staged per round (4 words)

struct Nb2Warp {                      // shared memory of one builder warp
    unsigned mask[NB2_WORDS][TILE];   // [word][lane]
    int wbase[NB2_WORDS];             // slot of bit 31 of each word
    float sx[NB2_CHUNK], sy[NB2_CHUNK], sz[NB2_CHUNK];
};

// Sign bits of four fl(r2 - R2) into the mask, oldest candidate in the highest bit.
__device__ __forceinline__ unsigned push4(unsigned m, float2 a, float2 b) {
    m = __funnelshift_l(__float_as_uint(a.x), m, 1);
    m = __funnelshift_l(__float_as_uint(a.y), m, 1);
    m = __funnelshift_l(__float_as_uint(b.x), m, 1);
    m = __funnelshift_l(__float_as_uint(b.y), m, 1);
    return m;
}

// MAPPED as in k_nbr_build.  incremental != 0 (a rebuild inside md_nve_step): every column
// already holds the pad value beyond its previous count, so only rows [count, previous count)
// are re-padded; 0: rows [count, capacity) are written.
template <int DIM, bool MAPPED>
__global__ void __launch_bounds__(NB2_WARPS * 32)
k_nbr_build2(Geom g, const float4 *__restrict__ spos, const int *__restrict__ cell_start,
             const int *__restrict__ map, int *__restrict__ nbr_idx, int *__restrict__ nbr_count,
             int *status, float4 *__restrict__ ref_pos, const int *cond, int incremental) {
    extern __shared__ __align__(16) unsigned char nb2_smem[];
    if (cond && ld_volatile(cond) == 0) return;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    Nb2Warp &W = reinterpret_cast<Nb2Warp *>(nb2_smem)[warp];
    const int cap = g.capacity;
    const int ncx = g.nc[0], ncy = g.nc[1], ncz = g.nc[2];
    const float Lx = g.L[0], Ly = g.L[1], Lz = g.L[2];
    const float2 nR2 = make_float2(-g.R2, -g.R2);
    constexpr int ROWS = DIM == 3 ? 9 : 3;
    const int ntiles = (g.n + TILE - 1) / TILE;

    for (int tile = blockIdx.x * NB2_WARPS + warp; tile < ntiles; tile += gridDim.x * NB2_WARPS) {
        const int s = tile * TILE + lane;
        const bool act = s < g.n;
        const float4 pi = spos[act ? s : g.n - 1];
        const int cx = cell_coord(pi.x, g.inv_cell[0], ncx);
        const int cy = cell_coord(pi.y, g.inv_cell[1], ncy);
        const int cz = DIM == 3 ? cell_coord(pi.z, g.inv_cell[2], ncz) : 0;
        const int row = act ? cz * ncy + cy : 0x7fffffff;
        const int me = act ? (MAPPED ? map[s] : s) : 0;           // the particle this lane owns
        int *outp = nullptr;                                     // its column of the list
        if (!MAPPED) outp = nbr_idx + nbr_tile_base(s, cap) + lane;
        else if (act) outp = nbr_idx + nbr_tile_base(me, cap) + (me & 31);
        const int prev = incremental ? (act ? min(nbr_count[me], cap) : 0) : cap;
        int cnt = 0;                                             // hits so far, self excluded
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
            // ---- piece table (as k_nbr_build): lane p < 3*ROWS describes piece p = kind*ROWS + rr
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
            int nw = 0;                      // mask words of the current batch (warp-uniform)
            unsigned nz = 0;                 // which of them are non-zero for this lane

            // every lane pulls its next hit per iteration: row k leaves as one 128-byte store
            auto expand = [&]() {
                __syncwarp();
                unsigned pend = inseg ? nz : 0u, word = 0u;
                int w = 0;
                while (true) {
                    if (word == 0u && pend) { w = __ffs(pend) - 1; pend &= pend - 1; word = W.mask[w][lane]; }
                    if (!__any_sync(FULL, word != 0u)) break;
                    if (word) {
                        const int bit = __clz(word);
                        word &= ~(0x80000000u >> bit);
                        const int slot = W.wbase[w] + bit;
                        if (slot != s) {
                            if (cnt < cap) outp[cnt * TILE] = MAPPED ? map[slot] : slot;
                            ++cnt;
                        }
                    }
                }
                __syncwarp();
                nw = 0; nz = 0u;
            };
