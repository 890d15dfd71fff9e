// md_force32.cuh -- Lennard-Jones force / energy over the neighbor list (L78, L80, L104), 3-D:
// fp32 fast path with an error estimate, fp64 re-evaluation where the estimate requires it.
//
// One warp = one list tile, one lane per particle (slot k of the 32 particles is one
// coalesced 128-byte row; neighbor positions are float4 gathers through L1).
//
// Precision.  The fp64 chain of md_kernels.cuh holds the 1e-5 force tolerance
// everywhere but is bound by the conversion / reciprocal unit (3 F2F + 1 RCP64H per pair).
// Here every pair is evaluated in fp32 first -- displacement by the canonical nearest-image
// form (one rounding), r2 = fma(dz,dz,fma(dy,dy,dx*dx)), y = 1/r2 (MUFU), force
// coefficient c = 24 eps sig^6 y^4 t, t = 2 sig^6 y^3 - 1 -- together with S_i^2 = sum_j (c r)^2 where t^2 is
// replaced by t^2 + 0.2^2: the coefficient vanishes at r = 2^(1/6) sigma while its rounding error
// (~3e-7 * 24 eps sig^6 y^4 there) does not, and the floor keeps the error-to-estimate ratio of
// such a pair in line with that of every other pair.
// The fp32 error of F_i is a random sum of per-pair errors of relative size ~1e-7 * (7..13), so it
// goes with the root-sum-square S_i: measured against the fp64 chain and the oracle (32k, 256k and
// 1M particles, lattice and liquid states, thirteen states in all) it stays below
// 7.0e-6 * max(|F_i|, 1e-3) whenever S_i <= 3.5 * max(|F_i|, 1e-3).  A particle that fails this
// test (its pair forces nearly cancel; 2-3 % of a liquid, 7 % of the jittered lattice), or that has a pair within 1e-5 of
// r_cut^2 (the truncated force jumps by 0.039 there, so the in/out decision must be the exact
// one), is re-evaluated in fp64 from exact displacements inside its own warp: groups of 32, 16 or
// 8 lanes stride over the particle's row (1, 2 or up to 4 flagged particles at a time) and reduce
// by shuffles.  Both results are rounded to fp32 once, on store.  (A separate queue + second kernel
// for the re-evaluation was measured slower.)
#pragma once
#include "md_kernels.cuh"

namespace mdk {

struct Pair32 {
    float rc2;          // fl32(r_cut^2)
    float sig6x2;       // 2 sigma^6
    float ucut4;        // shift * ((s/rc)^12 - (s/rc)^6)
    float fscale;       // 24 eps sigma^6
    float escale;       // 2 eps   (= 1/2 * 4 eps)
    float near_band;    // |r2 - rc2| <= near_band -> exact re-evaluation
    float est_thr;      // re-evaluate when fscale * S_i > est_thr * max(|F_i|, 1e-3), S_i^2 the accumulated sum
    // the other kinds of the fast path (the estimate term of each is scaled so that one est_thr serves all)
    float k_hi, k_lo;                 // MORSE: -alpha log2(e), BUCKINGHAM: -B log2(e), as a float and what it drops
    float s_unit;                     // scale of the estimate term against Lennard-Jones's
    float m_r0, m_2a, m_a;            // MORSE: r0, 2 alpha, alpha;  ucut4 = shift * u(r_cut) / D
    float b_A, b_B, b_C;              // BUCKINGHAM: A, B, C;        ucut4 = shift * u(r_cut)
};

struct Acc32 { float fx, fy, fz, s, e, near; };

// Canonical nearest-image displacement, fp32, one rounding; aL = a - L (exact).
__device__ __forceinline__ float min_image_pre(float a, float aL, float b, float L, float h) {
    float d = a - b;
    if (d > h) d = aL - b;
    else if (d < -h) d = a - (b - L);
    return d;
}

// 1/x by the reciprocal unit (MUFU.RCP, 1 ulp).
__device__ __forceinline__ float rcp32(float x) {
    float y;
    asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}


// Two list entries of one particle at once with packed fp32x2 arithmetic (FADD2 / FMUL2 / FFMA2:
// one instruction, two lanes of data), the same operations in the same order as lj_pair32 -- so the
// bits of every pair term are those of the scalar form.  Outside the cutoff (and for the far-away
// point that stands in for a missing slot) 1/r2 is multiplied by 0: every power and the coefficient
// vanish with it, no later select.
struct Acc2s { float2 fx, fy, fz, s, e; float near; };

template <bool ENERGY>
__device__ __forceinline__ void lj_pair32x2(const Pair32 &pp, float2 dx, float2 dy, float2 dz, Acc2s &a) {
    const float2 r2 = __ffma2_rn(dz, dz, __ffma2_rn(dy, dy, __fmul2_rn(dx, dx)));
    const float2 w = __fadd2_rn(r2, make_float2(-pp.rc2, -pp.rc2));
    a.near = fminf(a.near, fminf(fabsf(w.x), fabsf(w.y)));
    const float2 m = make_float2(w.x < 0.0f ? 1.0f : 0.0f, w.y < 0.0f ? 1.0f : 0.0f);
    const float2 y = __fmul2_rn(make_float2(rcp32(r2.x), rcp32(r2.y)), m);
    const float2 y2 = __fmul2_rn(y, y);
    const float2 y3 = __fmul2_rn(y2, y);
    const float2 t = __ffma2_rn(make_float2(pp.sig6x2, pp.sig6x2), y3, make_float2(-1.0f, -1.0f));
    const float2 y4 = __fmul2_rn(y2, y2);
    const float2 c = __fmul2_rn(y4, t);
    a.fx = __ffma2_rn(c, dx, a.fx); a.fy = __ffma2_rn(c, dy, a.fy); a.fz = __ffma2_rn(c, dz, a.fz);
    // S: (|coefficient| r)^2 with the coefficient floored near its zero, y4^2 r2 (t^2 + 0.2^2) = y^7 (t^2 + 0.04)
    a.s = __ffma2_rn(__fmul2_rn(y3, y4), __ffma2_rn(t, t, make_float2(0.04f, 0.04f)), a.s);
    if (ENERGY) {
        const float hs = 0.5f * pp.sig6x2;
        const float2 s6 = __fmul2_rn(make_float2(hs, hs), y3);
        float2 e = __ffma2_rn(s6, s6, make_float2(-s6.x, -s6.y));
        e = __ffma2_rn(m, make_float2(-pp.ucut4, -pp.ucut4), e);
        a.e = __fadd2_rn(a.e, e);
    }
}

__device__ __forceinline__ float ex2_32(float x) {
    float y;
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}
__device__ __forceinline__ float rsq32(float x) {
    float y;
    asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}

// The same for the other kinds of the fast path.  Each accumulates the force coefficient c (force = c d),
// the energy term and S, the scale of the coefficient's fp32 error: |c| times the factor by which the pair's
// functional form amplifies a relative error of r (normalised to Lennard-Jones, where it is ~10), with the
// floor that keeps S honest where c changes sign.
template <int KIND, bool ENERGY>
__device__ __forceinline__ void pair32x2(const Pair32 &pp, float2 dx, float2 dy, float2 dz, Acc2s &a) {
    if (KIND == 0) { lj_pair32x2<ENERGY>(pp, dx, dy, dz, a); return; }
    const float2 r2 = __ffma2_rn(dz, dz, __ffma2_rn(dy, dy, __fmul2_rn(dx, dx)));
    const float2 w = __fadd2_rn(r2, make_float2(-pp.rc2, -pp.rc2));
    a.near = fminf(a.near, fminf(fabsf(w.x), fabsf(w.y)));
    const float2 m = make_float2(w.x < 0.0f ? 1.0f : 0.0f, w.y < 0.0f ? 1.0f : 0.0f);
    // r and 1/r to an ulp from the 2-ulp hardware rsqrt (one Newton step), and the part of r that fp32
    // drops: an exponential amplifies the relative error of r by alpha r ~ 5..15
    const float2 ir0 = make_float2(rsq32(r2.x), rsq32(r2.y));
    const float2 h = __fmul2_rn(r2, ir0);
    const float2 nr = __ffma2_rn(make_float2(-h.x, -h.y), ir0, make_float2(1.0f, 1.0f));        // 1 - r2 ir0^2
    const float2 r = __ffma2_rn(__fmul2_rn(h, make_float2(0.5f, 0.5f)), nr, h);
    const float2 hir = __ffma2_rn(__fmul2_rn(ir0, make_float2(0.25f, 0.25f)), nr, __fmul2_rn(ir0, make_float2(0.5f, 0.5f)));   // 1 / (2 r)
    const float2 ir = __fadd2_rn(hir, hir);
    const float2 r_lo = __fmul2_rn(__ffma2_rn(make_float2(-r.x, -r.y), r, r2), hir);            // (r2 - r^2) / (2 r)
    if (KIND == 2) {
        // u / D = (1 - x)^2 - 1, x = exp(-alpha (r - r0));  c = -u'(r) / r / D = -2 alpha x (1 - x) / r
        // the exponent k (r - r0), k = -alpha log2(e) = k_hi + k_lo, as a rounded product plus its remainder
        const float2 d = __fadd2_rn(r, make_float2(-pp.m_r0, -pp.m_r0));
        const float2 khi = make_float2(pp.k_hi, pp.k_hi);
        const float2 a_hi = __fmul2_rn(d, khi);
        float2 a_lo = __ffma2_rn(d, khi, make_float2(-a_hi.x, -a_hi.y));
        a_lo = __ffma2_rn(d, make_float2(pp.k_lo, pp.k_lo), a_lo);
        a_lo = __ffma2_rn(r_lo, khi, a_lo);
        float2 x = make_float2(ex2_32(a_hi.x), ex2_32(a_hi.y));
        x = __ffma2_rn(__fmul2_rn(x, make_float2(0.69314718f, 0.69314718f)), a_lo, x);
        x = __fmul2_rn(x, m);
        const float2 om = __fadd2_rn(make_float2(1.0f, 1.0f), make_float2(-x.x, -x.y));
        const float2 x2a = __fmul2_rn(x, make_float2(pp.m_2a, pp.m_2a));
        const float2 g2 = __fmul2_rn(x2a, ir);                                                // 2 alpha x / r
        const float2 c = __fmul2_rn(g2, make_float2(-om.x, -om.y));
        a.fx = __ffma2_rn(c, dx, a.fx); a.fy = __ffma2_rn(c, dy, a.fy); a.fz = __ffma2_rn(c, dz, a.fz);
        // error of c: x and 1 - x both carry x alpha r eps_r, 1/r carries eps_r
        const float2 aom = make_float2(pp.s_unit * fabsf(om.x), pp.s_unit * fabsf(om.y));
        const float2 amp = __ffma2_rn(__ffma2_rn(x, make_float2(pp.s_unit, pp.s_unit), aom),
                                      __fmul2_rn(r, make_float2(pp.m_a, pp.m_a)), aom);
        const float2 er = __fmul2_rn(x2a, amp);                                               // (g2 amp) r
        a.s = __ffma2_rn(er, er, a.s);
        if (ENERGY) {
            float2 e = __ffma2_rn(om, om, make_float2(-1.0f - pp.ucut4, -1.0f - pp.ucut4));
            a.e = __ffma2_rn(e, m, a.e);
        }
    } else {
        // u = A exp(-B r) - C / r^6;  c = (A B exp(-B r) r - 6 C / r^6) / r^2
        const float2 y = __fmul2_rn(__fmul2_rn(ir, ir), m);
        const float2 y3 = __fmul2_rn(__fmul2_rn(y, y), y);
        const float2 khi = make_float2(pp.k_hi, pp.k_hi);                                     // -B log2(e)
        const float2 a_hi = __fmul2_rn(r, khi);
        float2 a_lo = __ffma2_rn(r, khi, make_float2(-a_hi.x, -a_hi.y));
        a_lo = __ffma2_rn(r, make_float2(pp.k_lo, pp.k_lo), a_lo);
        a_lo = __ffma2_rn(r_lo, khi, a_lo);
        float2 x = make_float2(ex2_32(a_hi.x), ex2_32(a_hi.y));
        x = __ffma2_rn(__fmul2_rn(x, make_float2(0.69314718f, 0.69314718f)), a_lo, x);
        x = __fmul2_rn(x, make_float2(pp.b_A, pp.b_A));
        const float2 t1 = __fmul2_rn(__fmul2_rn(x, r), make_float2(pp.b_B, pp.b_B));
        const float2 t2 = __fmul2_rn(y3, make_float2(6.0f * pp.b_C, 6.0f * pp.b_C));
        const float2 c = __fmul2_rn(__fadd2_rn(t1, make_float2(-t2.x, -t2.y)), y);
        a.fx = __ffma2_rn(c, dx, a.fx); a.fy = __ffma2_rn(c, dy, a.fy); a.fz = __ffma2_rn(c, dz, a.fz);
        // error of c: the exponential amplifies by B r + 3, the power law by 8
        const float2 k1 = __ffma2_rn(r, make_float2(pp.s_unit * pp.b_B, pp.s_unit * pp.b_B), make_float2(3.0f * pp.s_unit, 3.0f * pp.s_unit));
        const float2 amp = __ffma2_rn(t1, k1, __fmul2_rn(t2, make_float2(8.0f * pp.s_unit, 8.0f * pp.s_unit)));
        a.s = __ffma2_rn(__fmul2_rn(amp, amp), y, a.s);                                       // (amp y r)^2 = amp^2 y
        if (ENERGY) {
            float2 e = __ffma2_rn(y3, make_float2(-pp.b_C, -pp.b_C), __fadd2_rn(x, make_float2(-pp.ucut4, -pp.ucut4)));
            a.e = __ffma2_rn(e, m, a.e);
        }
    }
}

// Exact re-evaluation of one particle by a group of G = 8, 16 or 32 lanes striding over its row
// (32 / G particles per warp at a time); the sum is returned in every lane of the group.
template <int KIND, bool ENERGY, bool WRAP>
__device__ __forceinline__ Acc64 lj_row64(const Geom &g, const Pair &pp,
                                          const float4 *__restrict__ pos, const int *col, int cnt,
                                          const float4 &pb, int sub, int G) {
    const Me<3> me = make_me<3>(g, pb);
    Acc64 acc = {0.0, 0.0, 0.0, 0.0};
    for (int k = sub; k < cnt; k += 2 * G) {
        const bool v2 = k + G < cnt;
        const int j1 = col[k * TILE];
        const int j2 = v2 ? col[(k + G) * TILE] : j1;
        MD_CHECK(j1 >= 0 && j1 < g.ntot && j2 >= 0 && j2 < g.ntot);
        const float4 q1 = pos[j1], q2 = pos[j2];
        pair_any<KIND, 3, ENERGY, WRAP>(pp, me, q1, true, acc);
        pair_any<KIND, 3, ENERGY, WRAP>(pp, me, q2, v2, acc);
    }
    for (int o = G >> 1; o > 0; o >>= 1) {              // G is warp-uniform
        acc.fx += __shfl_xor_sync(FULL, acc.fx, o);
        acc.fy += __shfl_xor_sync(FULL, acc.fy, o);
        acc.fz += __shfl_xor_sync(FULL, acc.fz, o);
        if (ENERGY) acc.e += __shfl_xor_sync(FULL, acc.e, o);
    }
    return acc;
}

#ifndef MD_F32_WARPS
#define MD_F32_WARPS 2
#endif
#ifndef MD_F32_MINBLOCKS
#define MD_F32_MINBLOCKS 14
#endif
constexpr int F32_WARPS = MD_F32_WARPS;
#ifndef MD_F32_U
#define MD_F32_U 4
#endif
constexpr int F32_U = MD_F32_U;

// The pair loop of one lane over its column of the tile: rows [0, kmin) are owned by every lane
// of the warp (no validity test), rows [kmin, kmax) are the ragged tail.  WX / WY / WZ: the warp
// is near a box face in that direction and takes the nearest image there (warp-uniform).
template <int KIND, bool ENERGY, bool WX, bool WY, bool WZ>
__device__ __forceinline__ void lj_rows32(const Geom &g, const Pair32 &p32,
                                          const float4 *__restrict__ pos, const int *col,
                                          const float4 &pi, int ii, int cnt, int kmin, int kmax,
                                          bool active, Acc32 &acc) {
    // an idle lane of a ragged last tile owns no column: it loads no index (its column may hold
    // anything) and gathers its stand-in particle ii
    // List rows are prefetched one iteration ahead with ONE warp-uniform guard, k + U < kmax: some lane then
    // needs row k + U, and since capacity is a multiple of 4 (md_create) and so is k, rows k + U .. k + 2U - 1
    // all exist.  What a row holds beyond a lane's count is never used as an index (the tail selects).
    // A lane without a particle reads lane 0's column of the tile (valid entries of a valid particle) instead of
    // its own, which nobody wrote.
    static_assert(F32_U == 2 || F32_U == 4, "the row prefetch relies on capacity % F32_U == 0");
    const int *cs = active ? col : col - (threadIdx.x & 31);
    const float Lx = g.L[0], Ly = g.L[1], Lz = g.L[2];
    const float hx = g.h[0], hy = g.h[1], hz = g.h[2];
    const float pxL = pi.x - Lx, pyL = pi.y - Ly, pzL = pi.z - Lz;
    auto disp = [&](const float4 &q, float &dx, float &dy, float &dz) {
        dx = WX ? min_image_pre(pi.x, pxL, q.x, Lx, hx) : pi.x - q.x;
        dy = WY ? min_image_pre(pi.y, pyL, q.y, Ly, hy) : pi.y - q.y;
        dz = WZ ? min_image_pre(pi.z, pzL, q.z, Lz, hz) : pi.z - q.z;
    };
    static_assert(F32_U % 2 == 0, "the pair loop takes two slots per packed evaluation");
    Acc2s a2;
    a2.fx = a2.fy = a2.fz = a2.s = a2.e = make_float2(0.0f, 0.0f);
    a2.near = acc.near;
    auto two = [&](const float4 &qa, const float4 &qb) {
        float ax, ay, az, bx, by, bz;
        disp(qa, ax, ay, az);
        disp(qb, bx, by, bz);
        pair32x2<KIND, ENERGY>(p32, make_float2(ax, bx), make_float2(ay, by), make_float2(az, bz), a2);
    };
    int k = 0;
    int jn[F32_U];
#pragma unroll
    for (int u = 0; u < F32_U; ++u) jn[u] = kmax > 0 ? cs[u * TILE] : ii;
    for (; k < kmin; k += F32_U) {
        int j[F32_U]; float4 q[F32_U];
#pragma unroll
        for (int u = 0; u < F32_U; ++u) j[u] = jn[u];
#pragma unroll
        for (int u = 0; u < F32_U; ++u) { MD_CHECK(j[u] >= 0 && j[u] < g.ntot); q[u] = pos[j[u]]; }
        if (k + F32_U < kmax) {
#pragma unroll
            for (int u = 0; u < F32_U; ++u) jn[u] = cs[(k + F32_U + u) * TILE];
        }
#pragma unroll
        for (int u = 0; u < F32_U; u += 2) two(q[u], q[u + 1]);
    }
    // ragged tail: a slot this lane does not own reads the lane's own position (a valid address)
    // and is then moved 1e18 away, where it contributes exactly zero
    for (; k < kmax; k += F32_U) {
        int j[F32_U]; float4 q[F32_U];
#pragma unroll
        for (int u = 0; u < F32_U; ++u) j[u] = k + u < cnt ? jn[u] : ii;
#pragma unroll
        for (int u = 0; u < F32_U; ++u) { MD_CHECK(j[u] >= 0 && j[u] < g.ntot); q[u] = pos[j[u]]; }
        if (k + F32_U < kmax) {
#pragma unroll
            for (int u = 0; u < F32_U; ++u) jn[u] = cs[(k + F32_U + u) * TILE];
        }
#pragma unroll
        for (int u = 0; u < F32_U; ++u) if (!(k + u < cnt)) q[u].x = 1e18f;
#pragma unroll
        for (int u = 0; u < F32_U; u += 2) two(q[u], q[u + 1]);
    }
    acc.fx += a2.fx.x + a2.fx.y; acc.fy += a2.fy.x + a2.fy.y; acc.fz += a2.fz.x + a2.fz.y;
    acc.s += a2.s.x + a2.s.y; acc.e += a2.e.x + a2.e.y; acc.near = a2.near;
}

// vel != NULL: also the second half-kick v += a F.  energy_total != NULL (ENERGY only): adds
// sum_i e_i in fp64.  book.stats != NULL: per-step bookkeeping.  nfix (may be NULL): counts
// re-evaluated particles (diagnostics).
// Fused step (nx.pos_out != NULL, inside md_nve_step's graph): the epilogue also opens the NEXT
// step -- v += a F again (its first half-kick), r = mu(r, dt v) written to the other position
// buffer (other warps still gather from this one), half-skin test against the reference
// positions, raising nx.flag and the graph condition of the next step's rebuild node.  The
// arithmetic and its order are those of k_kick_drift, so fused and unfused runs agree bit for bit.
struct NextStep {
    float4 *pos_out;            // NULL: plain force kernel
    const float4 *ref;          // positions at the last list build
    float dt;
    int *flag;                  // rebuild-needed word of the next step
    cudaGraphConditionalHandle cond;
    int has_cond;
};
template <int KIND, bool ENERGY>
__global__ void __launch_bounds__(F32_WARPS * 32, MD_F32_MINBLOCKS)
k_force32(Geom g, Pair pp, Pair32 p32, const float4 *__restrict__ pos,
             const int *__restrict__ nbr_idx, const int *__restrict__ nbr_count,
             float4 *__restrict__ force, float4 *__restrict__ vel, float a, double *energy_total,
             Book book, int *nfix, NextStep nx, int remap_p, int nblocks, int i0) {
    const int lane = threadIdx.x & 31;
    // remap_p > 0: the grid has remap_p * Q blocks and block i works on tile block
    // (i % remap_p) * Q + i / remap_p, so that the blocks the hardware deals round-robin to one SM
    // are neighbors in space and share their gathers in L1
    int bid = blockIdx.x;
    if (remap_p > 0) {
        const int Q = gridDim.x / remap_p;
        bid = (bid % remap_p) * Q + bid / remap_p;
        if (bid >= nblocks) return;
    }
    const int gid = i0 + bid * blockDim.x + threadIdx.x;      // i0: first particle of this context's range
    if (book_skips(book, gid)) return;
    const int i = gid;
    const bool active = i < g.n;
    const int ii = active ? i : g.n - 1;
    const float4 pi = pos[ii];
    const int cnt = active ? min(nbr_count[ii], g.capacity) : 0;
    const int *col = nbr_idx + nbr_tile_base(gid, g.capacity) + lane;    // gid: valid for the whole tile
    const int kmax = warp_max(cnt);
    const int kmin = min(warp_min(active ? cnt : 0x7fffffff), kmax) & ~(F32_U - 1);  // rows every lane owns
    const bool wx = __any_sync(FULL, active && (pi.x < g.face || pi.x > g.L[0] - g.face));
    const bool wy = __any_sync(FULL, active && (pi.y < g.face || pi.y > g.L[1] - g.face));
    const bool wz = __any_sync(FULL, active && (pi.z < g.face || pi.z > g.L[2] - g.face));
    Acc32 acc = {0.0f, 0.0f, 0.0f, 0.0f, 0.0f, 1e30f};

    if (!(wx || wy || wz)) lj_rows32<KIND, ENERGY, false, false, false>(g, p32, pos, col, pi, ii, cnt, kmin, kmax, active, acc);
    else if (wx && !wy && !wz) lj_rows32<KIND, ENERGY, true, false, false>(g, p32, pos, col, pi, ii, cnt, kmin, kmax, active, acc);
    else if (!wx && wy && !wz) lj_rows32<KIND, ENERGY, false, true, false>(g, p32, pos, col, pi, ii, cnt, kmin, kmax, active, acc);
    else if (!wx && !wy && wz) lj_rows32<KIND, ENERGY, false, false, true>(g, p32, pos, col, pi, ii, cnt, kmin, kmax, active, acc);
    else lj_rows32<KIND, ENERGY, true, true, true>(g, p32, pos, col, pi, ii, cnt, kmin, kmax, active, acc);

    // ---- fp32 result, error estimate, exact re-evaluation of the lanes that need it
    float fx = p32.fscale * acc.fx, fy = p32.fscale * acc.fy, fz = p32.fscale * acc.fz;
    double e64 = ENERGY ? (double)(p32.escale * acc.e) : 0.0;
    const float fn = fmaxf(sqrtf(fmaf(fz, fz, fmaf(fy, fy, fx * fx))), 1e-3f);
    const float sf = p32.fscale * p32.fscale * acc.s, tf = p32.est_thr * fn;
    const bool redo = active && (sf > tf * tf || acc.near <= p32.near_band ||
                                 !(fn < 3.0e38f));
    unsigned todo = __ballot_sync(FULL, redo);
    if (nfix && lane == 0 && todo) atomicAdd(nfix, __popc(todo));
    const int *tile0 = col - lane;
    while (todo) {
        // 1 flagged lane left: the whole warp takes it; 2: half a warp each; else 8 lanes each
        const int nf = __popc(todo);
        const int G = nf == 1 ? 32 : (nf == 2 ? 16 : 8);
        const int ng = 32 / G;
        const int grp = lane / G, sub = lane % G;
        unsigned t = todo;
        int b = -1;
#pragma unroll
        for (int q = 0; q < 4; ++q) {
            const int f = (t && q < ng) ? __ffs(t) - 1 : -1;
            if (q == grp) b = f;
            if (q < ng) t &= t - 1;                       // 0 & anything stays 0
        }
        const int bb = b < 0 ? 0 : b;
        float4 pb;
        pb.x = __shfl_sync(FULL, pi.x, bb); pb.y = __shfl_sync(FULL, pi.y, bb);
        pb.z = __shfl_sync(FULL, pi.z, bb); pb.w = 0.0f;
        int cb = __shfl_sync(FULL, cnt, bb);              // every lane takes part in the shuffle
        if (b < 0) cb = 0;
        // away from every face the fp32 difference is exact for every pair inside the cutoff
        const Acc64 r = (wx || wy || wz) ? lj_row64<KIND, ENERGY, true>(g, pp, pos, tile0 + bb, cb, pb, sub, G)
                                         : lj_row64<KIND, ENERGY, false>(g, pp, pos, tile0 + bb, cb, pb, sub, G);
        // deliver: the lane whose rank among the flagged lanes is q < ng reads group q
        const int rank = __popc(todo & ((1u << lane) - 1u));
        const bool mine = ((todo >> lane) & 1u) && rank < ng;
        const int src = mine ? rank * G : lane;
        const double rx = __shfl_sync(FULL, r.fx, src), ry = __shfl_sync(FULL, r.fy, src);
        const double rz = __shfl_sync(FULL, r.fz, src);
        const double re = ENERGY ? __shfl_sync(FULL, r.e, src) : 0.0;
        if (mine) {
            // as force_epilogue: 24 eps sigma^6 | D | 1 and half of 4 eps | D | 1
            const double fs = KIND == 0 ? 12.0 * pp.deps * pp.dsig6x2 : (KIND == 2 ? pp.deps : 1.0);
            const double es = KIND == 0 ? 2.0 * pp.deps : (KIND == 2 ? 0.5 * pp.deps : 0.5);
            fx = (float)(fs * rx); fy = (float)(fs * ry); fz = (float)(fs * rz);
            if (ENERGY) e64 = es * re;
        }
        todo = t;
    }

    // ---- store, second half-kick, energy reduction, bookkeeping
    bool moved = false;
    if (active) {
        force[i] = make_float4(fx, fy, fz, (float)e64);
        if (vel) {
            float4 v = vel[i];
            v.x = fmaf(a, fx, v.x); v.y = fmaf(a, fy, v.y); v.z = fmaf(a, fz, v.z);
            if (nx.pos_out) {
                v.x = fmaf(a, fx, v.x); v.y = fmaf(a, fy, v.y); v.z = fmaf(a, fz, v.z);
                float4 p = pi;
                p.x = wrap(fmaf(nx.dt, v.x, p.x), g.L[0], g.inv_L[0]);
                p.y = wrap(fmaf(nx.dt, v.y, p.y), g.L[1], g.inv_L[1]);
                p.z = wrap(fmaf(nx.dt, v.z, p.z), g.L[2], g.inv_L[2]);
                nx.pos_out[i] = p;
                moved = disp2_from_ref<3>(g, p, nx.ref[i]) > g.half_skin2;
            }
            vel[i] = v;
        }
    }
    if (nx.pos_out && __any_sync(FULL, moved) && lane == 0) {
        *nx.flag = 1;
        if (nx.has_cond) cudaGraphSetConditional(nx.cond, 1);
    }
    if (ENERGY && energy_total) {
        __shared__ double red[F32_WARPS];
        double x = active ? e64 : 0.0;
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) x += __shfl_xor_sync(FULL, x, o);
        if (lane == 0) red[threadIdx.x >> 5] = x;
        __syncthreads();
        if (threadIdx.x == 0) {
            double t = 0.0;
            for (int w = 0; w < F32_WARPS; ++w) t += red[w];
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

} // namespace mdk
