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
// per-lane bit mask, one funnel shift per candidate and no branch, 32 candidates per word; every
// lane keeps its NON-ZERO words (and the slot each starts at) densely in its own shared-memory column,
// up to NB2_WORDS of them (6 KB per warp), and they are expanded afterwards, every lane pulling
// its next set bit per iteration, so row k of the tile leaves as one coalesced 128-byte store.
#pragma once
#include "md_kernels.cuh"
#include <cstddef>

namespace mdk {

#ifndef MD_NB2_WARPS
#define MD_NB2_WARPS 4
#endif
constexpr int NB2_WARPS = MD_NB2_WARPS;   // tiles per block
constexpr int NB2_WORDS = 24;         // NON-ZERO mask words a lane can hold per batch
constexpr int NB2_CHUNK = 128;        // candidates staged per round (4 words)

struct Nb2Warp {                      // shared memory of one builder warp
    unsigned mask[NB2_WORDS][TILE];   // [k][lane]: the k-th non-zero mask word of the lane
    int wb[NB2_WORDS][TILE];          // slot of bit 31 of that word (directly behind mask: expand() relies on it)
    float sx[NB2_CHUNK], sy[NB2_CHUNK], sz[NB2_CHUNK];
};
static_assert(offsetof(Nb2Warp, wb) == sizeof(unsigned) * NB2_WORDS * TILE, "wb directly behind mask");

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
#ifndef MD_NB2_MINBLOCKS
#define MD_NB2_MINBLOCKS (32 / MD_NB2_WARPS)
#endif
// PARTS = 1, 2 or 4 warps share one tile: they build the same piece table, scan every PARTS-th
// piece each, exchange their per-lane hit counts through shared memory (a named barrier per tile)
// and expand their masks into disjoint row ranges of the tile.  The list is the same set of rows;
// a tile's critical path is 1/PARTS as long, which is what small systems (a few tiles per SM) and
// the last wave of large ones wait for, at the price of PARTS copies of the per-tile prologue.
__device__ __forceinline__ void bar_group(int id, int nthreads) {
    asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(nthreads) : "memory");
}
__device__ __forceinline__ int warp_sum_i(int v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(FULL, v, o);
    return v;
}

template <int DIM, bool MAPPED, int PARTS>
__global__ void __launch_bounds__(NB2_WARPS * 32, MD_NB2_MINBLOCKS)
k_nbr_build2(Geom g, const float4 *__restrict__ spos, const int *__restrict__ cell_start,
             const int *__restrict__ map, int *__restrict__ nbr_idx, int *__restrict__ nbr_count,
             int *status, float4 *__restrict__ ref_pos, const int *cond, int incremental,
             int tile0, int tile1) {
    extern __shared__ __align__(16) unsigned char nb2_smem[];
    if (cond && ld_volatile(cond) == 0) return;
    __shared__ int coop[NB2_WARPS][TILE];                  // per-lane hit counts of the parts of a tile
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    constexpr int TPB = NB2_WARPS / PARTS;                  // tiles per block
    const int tl = warp / PARTS, part = warp % PARTS;
    Nb2Warp &W = reinterpret_cast<Nb2Warp *>(nb2_smem)[warp];
    const int cap = g.capacity;
    const int ncx = g.nc[0], ncy = g.nc[1], ncz = g.nc[2];
    const float Lx = g.L[0], Ly = g.L[1], Lz = g.L[2];
    const float2 nR2 = make_float2(-g.R2, -g.R2);
    const float Rm = sqrtf(g.R2) * 1.0001f + 1e-4f * g.L[0];    // R plus a margin for the fp32 roundings
    constexpr int ROWS = DIM == 3 ? 9 : 3;
    const int ntiles = min(tile1, (g.n + TILE - 1) / TILE);     // this context's tiles: [tile0, tile1)

    for (int tile = tile0 + blockIdx.x * TPB + tl; tile < ntiles; tile += gridDim.x * TPB) {
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
        const int prev = incremental ? ((act && part == 0) ? min(nbr_count[me], cap) : 0) : cap;
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
            float seg_xlo = inseg ? pi.x : 3.0e38f, seg_xhi = inseg ? pi.x : -3.0e38f;
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) {
                seg_xlo = fminf(seg_xlo, __shfl_xor_sync(FULL, seg_xlo, o));
                seg_xhi = fmaxf(seg_xhi, __shfl_xor_sync(FULL, seg_xhi, o));
            }
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
                // md_cell_list_build leaves every x-row of cells sorted by x: cut the piece to the
                // candidates whose x lies within R (plus a rounding margin) of the segment's lanes
                const float lo = kind == 1 ? seg_xlo - Rm + Lx : seg_xlo - Rm;
                const float hi = kind == 2 ? seg_xhi + Rm - Lx : seg_xhi + Rm;
                if (kind != 2) {                                 // first slot with x >= lo
                    int a0 = t0, a1 = t1;
                    while (a0 < a1) { const int mid = (a0 + a1) >> 1; if (spos[mid].x < lo) a0 = mid + 1; else a1 = mid; }
                    t0 = a0;
                }
                if (kind != 1) {                                 // first slot with x > hi
                    int a0 = t0, a1 = t1;
                    while (a0 < a1) { const int mid = (a0 + a1) >> 1; if (spos[mid].x <= hi) a0 = mid + 1; else a1 = mid; }
                    t1 = a0;
                }
            }
            // a part whose pieces would not fit one batch of masks cannot flush on its own (its rows
            // start after the other parts' hits): part 0 then scans the whole segment alone
            bool solo = false;
            if (PARTS > 1) {
                const int words = lane < 3 * ROWS ? (t1 - t0 + 31) >> 5 : 0;     // chunks split a piece at multiples of 128
#pragma unroll
                for (int q = 0; q < PARTS; ++q)
                    solo = solo || warp_sum_i(lane % PARTS == q ? words : 0) > NB2_WORDS;
            }
            int myw = 0;                     // non-zero mask words this lane holds in the current batch
            int nhit = 0;                    // hits of this lane in the current batch (self excluded)
            // every lane pulls its next hit per iteration (taking its next stored word when the current one
            // is used up): row k of the tile leaves as one 128-byte store.  The trip count is the largest
            // number of hits any lane holds, so the loop needs no vote.
            auto expand = [&]() {
                __syncwarp();
                const int nit = warp_max(nhit);
                // a lane's hits are its first nhit iterations (its stored words are non-zero and taken in
                // order), of which the first `room` fit its column
                const int keep = min(nhit, max(cap - cnt, 0));
                const unsigned *pm = &W.mask[0][lane];               // my current word; its slot base sits
                constexpr int WB = (int)(sizeof(W.mask) / sizeof(unsigned));     // WB entries further on
                const unsigned *pend = &W.mask[NB2_WORDS - 1][lane];
                unsigned word = pm[0];
                int wbv = (int)pm[WB];
                int *optr = outp + (size_t)min(cnt, cap) * TILE;
                for (int it = 0; it < nit; ++it) {
                    const int bit = __clz(word) & 31;
                    const int slot = wbv + bit;
                    word &= 0x7fffffffu >> bit;                    // drop that bit (all above it are 0)
                    MD_CHECK(!(it < nhit) || (slot >= 0 && slot < g.n && slot != s));
                    MD_CHECK(!(it < keep) || (optr >= outp && optr < outp + (size_t)cap * TILE));
                    if (it < keep) *optr = MAPPED ? map[slot] : slot;
                    optr += TILE;
                    if (word == 0u) {                              // my next word (beyond my last one: anything)
                        pm = pm < pend ? pm + TILE : pm;
                        word = pm[0];
                        wbv = (int)pm[WB];
                    }
                }
                cnt += nhit;
                __syncwarp();
                myw = 0; nhit = 0;
            };

            // ---- walk the pieces; the next chunk is loaded while the current one is tested
            int p = 0, base = 0, pt1 = 0;
            auto seek = [&](int &pp, int &bb, int &tt1) {       // first non-empty piece >= pp
                while (pp < 3 * ROWS) {
                    bb = __shfl_sync(FULL, t0, pp); tt1 = __shfl_sync(FULL, t1, pp);
                    if (bb < tt1 && (PARTS == 1 || (solo ? part == 0 : pp % PARTS == part))) return;
                    ++pp;
                }
            };
            seek(p, base, pt1);
            float4 q[NB2_CHUNK / 32];
            auto fetch = [&](int bb, int tt1) {
#pragma unroll
                for (int u = 0; u < NB2_CHUNK / 32; ++u) {
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
                const int m = min(NB2_CHUNK, pt1 - base);
                // a lane's column could overflow if every word of this chunk came out non-zero: flush first
                if (__any_sync(FULL, myw + ((m + 31) >> 5) > NB2_WORDS)) expand();
                MD_CHECK(m > 0 && base >= 0 && pt1 <= g.n && myw + ((m + 31) >> 5) <= NB2_WORDS);
                // stage -(candidate - shift), structure of arrays; the tail of the last group of
                // four is a far-away point
#pragma unroll
                for (int u = 0; u < NB2_CHUNK / 32; ++u) {
                    const int c = u * 32 + lane;
                    if (c < m) {
                        W.sx[c] = __fsub_rn(sjx, q[u].x);
                        W.sy[c] = __fsub_rn(sjy, q[u].y);
                        if (DIM == 3) W.sz[c] = __fsub_rn(sjz, q[u].z);
                    } else if (c < ((m + 3) & ~3)) {
                        W.sx[c] = 1e18f; W.sy[c] = 0.0f;
                        if (DIM == 3) W.sz[c] = 0.0f;
                    }
                }
                __syncwarp();
                // next chunk
                int np = p, nbase = base + NB2_CHUNK, npt1 = pt1;
                if (nbase >= pt1) { ++np; seek(np, nbase, npt1); }
                if (np < 3 * ROWS) fetch(nbase, npt1);
                // test the staged chunk: 32 candidates per mask word, two per packed instruction
                // (FADD2 / FMUL2 / FFMA2, round-to-nearest: the bits of the scalar canonical form)
                const float2 px2 = make_float2(pix, pix), py2 = make_float2(piy, piy);
                const float2 pz2 = make_float2(piz, piz);
                auto four = [&](int c, unsigned acc) {
                    const float4 X = *reinterpret_cast<const float4 *>(W.sx + c);
                    const float4 Y = *reinterpret_cast<const float4 *>(W.sy + c);
                    const float2 dxa = __fadd2_rn(px2, make_float2(X.x, X.y));
                    const float2 dxb = __fadd2_rn(px2, make_float2(X.z, X.w));
                    const float2 dya = __fadd2_rn(py2, make_float2(Y.x, Y.y));
                    const float2 dyb = __fadd2_rn(py2, make_float2(Y.z, Y.w));
                    float2 ra = __ffma2_rn(dya, dya, __fmul2_rn(dxa, dxa));
                    float2 rb = __ffma2_rn(dyb, dyb, __fmul2_rn(dxb, dxb));
                    if (DIM == 3) {
                        const float4 Z = *reinterpret_cast<const float4 *>(W.sz + c);
                        const float2 dza = __fadd2_rn(pz2, make_float2(Z.x, Z.y));
                        const float2 dzb = __fadd2_rn(pz2, make_float2(Z.z, Z.w));
                        ra = __ffma2_rn(dza, dza, ra);
                        rb = __ffma2_rn(dzb, dzb, rb);
                    }
                    // sign(fl(r2 - R2)) is set exactly when r2 < R2 (a non-zero difference of two
                    // floats never rounds to zero, and x - x = +0)
                    return push4(acc, __fadd2_rn(ra, nR2), __fadd2_rn(rb, nR2));
                };
                for (int c0 = 0; c0 < m; c0 += 32) {
                    const int ng = min(8, (m - c0 + 3) >> 2);
                    unsigned hi = 0u, lo = 0u;
                    if (ng == 8) {
#pragma unroll
                        for (int gq = 0; gq < 4; ++gq) hi = four(c0 + 4 * gq, hi);
#pragma unroll
                        for (int gq = 4; gq < 8; ++gq) lo = four(c0 + 4 * gq, lo);
                        hi = (hi << 16) | lo;
                    } else {
                        for (int gq = 0; gq < ng; ++gq) hi = four(c0 + 4 * gq, hi);
                        hi <<= 32 - 4 * ng;
                    }
                    {   // my own slot passes the test at distance 0: drop its bit here
                        const unsigned self = (unsigned)(s - (base + c0));
                        if (self < 32u) hi &= ~(0x80000000u >> self);
                    }
                    if (!inseg) hi = 0u;                           // other segments' lanes record nothing
                    nhit += __popc(hi);
                    if (hi != 0u) {
                        W.mask[myw][lane] = hi;
                        W.wb[myw][lane] = base + c0;
                        ++myw;
                    }
                }
                __syncwarp();
                p = np; base = nbase; pt1 = npt1;
            }
            if (PARTS == 1) {
                expand();
            } else {
                // rows of this tile: part 0's hits, then part 1's, ...; every part learns the total
                coop[warp][lane] = inseg ? nhit : 0;
                bar_group(1 + tl, 32 * PARTS);
                int offset = 0, total = 0;
#pragma unroll
                for (int q = 0; q < PARTS; ++q) {
                    const int v = coop[tl * PARTS + q][lane];
                    offset += q < part ? v : 0;
                    total += v;
                }
                const int base_cnt = cnt;       // hits flushed earlier (solo part 0) or of an earlier segment
                cnt = base_cnt + offset;
                expand();
                cnt = base_cnt + total;
                bar_group(1 + tl, 32 * PARTS);  // coop is rewritten by the next segment
            }
        }
        // ---- pads (= N, A5), counts, rebuild reference, status (one part does it)
        if (PARTS > 1 && part != 0) continue;
        if (outp) {
            const int upto = incremental ? prev : cap;
            for (int k = min(cnt, cap); k < upto; ++k) outp[k * TILE] = g.n;
        }
        if (act) { nbr_count[me] = cnt; ref_pos[me] = pi; }
        const int mx = warp_max(act ? cnt : 0);
        if (lane == 0) {
            if (mx > ld_volatile(status + 1)) atomicMax(status + 1, mx);
            if (mx > cap) status[0] = 1;
        }
        __syncwarp();
    }
}

} // namespace mdk
