// md_kernels.cuh -- device code of libmd_b200 (sm_100a).  CUDA cores only: nothing on this
// path is a dense contraction.  Citations: /root/reference/PAPER.md line + section; readings
// of open points: SURVEY.md §8c A1..A18 / DESIGN.md §3.  Shares nothing with oracle/.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace mdk {

constexpr unsigned FULL = 0xffffffffu;

// Everything a kernel needs to know about the space and the partition (by value).
struct Geom {
    int   dim, n, capacity, cells;
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
    float  eps, sig2, rc2, u_cut, thr;     // fp32 chain
    double deps, dsig2, drc2, du_cut;      // fp64 chain
};

// Device words md_nve_step keeps between kernels.
struct Book {
    int *flag;      // rebuild needed (set by drift, cleared by the force kernel)
    int *status;    // {overflow, max count} of the last build
    int *stats;     // {steps, rebuilds, first overflow step | -1, max count}
};

__device__ __forceinline__ int ld_volatile(const int *p) { return *(const volatile int *)p; }

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
    cell_of[i] = c;
    rank_tmp[i] = atomicAdd(&cell_count[c], 1);   // arrival order; made canonical later
}

// One block: exclusive scan of cell_count[0..cells) into cell_start[0..cells]; zeroes
// cell_count for the next build and resets the build status words.
__global__ void __launch_bounds__(1024)
k_cell_scan(int cells, int *__restrict__ cell_count, int *__restrict__ cell_start,
            int *status, const int *cond) {
    if (cond && ld_volatile(cond) == 0) return;
    __shared__ int warp_sum[32];
    __shared__ int carry;
    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    if (tid == 0) { carry = 0; if (status) { status[0] = 0; status[1] = 0; } }
    __syncthreads();
    for (int base = 0; base < cells; base += 1024) {
        int c = base + tid;
        int v = c < cells ? cell_count[c] : 0;
        if (c < cells) cell_count[c] = 0;
        int x = v;
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
        int incl = x + (wid ? warp_sum[wid - 1] : 0) + carry;
        if (c < cells) cell_start[c] = incl - v;
        __syncthreads();
        if (tid == 1023) carry = incl;
        __syncthreads();
    }
    if (tid == 0) cell_start[cells] = carry;
}

__global__ void __launch_bounds__(256)
k_cell_scatter(int n, const int *__restrict__ cell_of, const int *__restrict__ rank_tmp,
               const int *__restrict__ cell_start, int *__restrict__ perm_tmp, const int *cond) {
    if (cond && ld_volatile(cond) == 0) return;
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    perm_tmp[cell_start[cell_of[i]] + rank_tmp[i]] = i;
}

// Canonical order inside a cell (ascending id, or index when id == NULL) by counting, so the
// sorted state does not depend on atomic arrival order; gathers the payload into the sorted
// scratch arrays.  One thread per slot.
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
    int key = id ? id[i] : i;
    int rank = 0;
    for (int t = t0; t < t1; ++t) {
        int j = perm_tmp[t];
        int kj = id ? id[j] : j;
        rank += kj < key;
    }
    int dst = t0 + rank;
    perm[dst] = i;
    pos_s[dst] = pos[i];
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

__global__ void __launch_bounds__(256)
k_gather_pos(int n, const int *__restrict__ perm, const float4 *__restrict__ pos,
             float4 *__restrict__ pos_s) {
    int s = blockIdx.x * blockDim.x + threadIdx.x;
    if (s < n) pos_s[s] = pos[perm[s]];
}

// --------------------------------------------------- neighbor list (L84-L88, L74) ---------
// One warp per sorted slot.  The 3^D stencil is walked as runs of contiguous slots (the three
// x-cells of one (y,z) row are contiguous; a periodic wrap in x splits the run).  A whole run
// shares its image shift: the particle is moved by -L when it sits in the high-side cell, the
// run by -L when the run is the high-side cell, which reproduces the canonical predicate bit
// for bit (SURVEY A3 "equivalence with a per-cell shift").  Lanes test 32 candidates at a
// time; hits are compacted with ballot/popc so the row is written coalesced.

struct RowWriter {
    int *row; const int *map; int cap; int count; int self; unsigned lt;
};

template <int DIM>
__device__ __forceinline__ void scan_run(RowWriter &w, const float4 *__restrict__ spos,
                                         int t0, int t1, float pix, float piy, float piz,
                                         float sjx, float sjy, float sjz, float R2, int lane) {
    for (int base = t0; base < t1; base += 32) {
        int t = base + lane;
        bool in = t < t1;
        float4 pj = spos[in ? t : t0];
        float dx = __fsub_rn(pix, __fsub_rn(pj.x, sjx));
        float dy = __fsub_rn(piy, __fsub_rn(pj.y, sjy));
        float r2 = __fmaf_rn(dy, dy, __fmul_rn(dx, dx));
        if (DIM == 3) {
            float dz = __fsub_rn(piz, __fsub_rn(pj.z, sjz));
            r2 = __fmaf_rn(dz, dz, r2);
        }
        bool hit = in && (r2 < R2) && (t != w.self);
        unsigned m = __ballot_sync(FULL, hit);
        if (hit) {
            int k = w.count + __popc(m & w.lt);
            if (k < w.cap) w.row[k] = w.map ? w.map[t] : t;
        }
        w.count += __popc(m);
    }
}

template <int DIM>
__global__ void __launch_bounds__(256)
k_nbr_build(Geom g, const float4 *__restrict__ spos, const int *__restrict__ cell_start,
            const int *__restrict__ map, int *__restrict__ nbr_idx, int *__restrict__ nbr_count,
            int *status, float4 *__restrict__ ref_pos, const int *cond) {
    if (cond && ld_volatile(cond) == 0) return;
    const int lane = threadIdx.x & 31;
    const int s = (blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    if (s >= g.n) return;
    const float4 pi = spos[s];
    const int i = map ? map[s] : s;
    const int cx = cell_coord(pi.x, g.inv_cell[0], g.nc[0]);
    const int cy = cell_coord(pi.y, g.inv_cell[1], g.nc[1]);
    const int cz = DIM == 3 ? cell_coord(pi.z, g.inv_cell[2], g.nc[2]) : 0;
    RowWriter w;
    w.row = nbr_idx + (size_t)i * g.capacity;
    w.map = map; w.cap = g.capacity; w.count = 0; w.self = s;
    w.lt = (1u << lane) - 1u;
    const int ncx = g.nc[0], ncy = g.nc[1], ncz = g.nc[2];
    const float Lx = g.L[0], Ly = g.L[1], Lz = g.L[2];
    for (int dz = (DIM == 3 ? -1 : 0); dz <= (DIM == 3 ? 1 : 0); ++dz) {
        int zc = cz + dz; float piz = pi.z, sjz = 0.0f;
        if (DIM == 3) {
            if (zc < 0) { zc += ncz; sjz = Lz; }
            else if (zc >= ncz) { zc -= ncz; piz = __fsub_rn(pi.z, Lz); }
        }
        for (int dy = -1; dy <= 1; ++dy) {
            int yc = cy + dy; float piy = pi.y, sjy = 0.0f;
            if (yc < 0) { yc += ncy; sjy = Ly; }
            else if (yc >= ncy) { yc -= ncy; piy = __fsub_rn(pi.y, Ly); }
            const int rowbase = (zc * ncy + yc) * ncx;
            const int xa = max(cx - 1, 0), xb = min(cx + 1, ncx - 1);
            scan_run<DIM>(w, spos, cell_start[rowbase + xa], cell_start[rowbase + xb + 1],
                          pi.x, piy, piz, 0.0f, sjy, sjz, g.R2, lane);
            if (cx == 0)
                scan_run<DIM>(w, spos, cell_start[rowbase + ncx - 1], cell_start[rowbase + ncx],
                              pi.x, piy, piz, Lx, sjy, sjz, g.R2, lane);
            else if (cx == ncx - 1)
                scan_run<DIM>(w, spos, cell_start[rowbase], cell_start[rowbase + 1],
                              __fsub_rn(pi.x, Lx), piy, piz, 0.0f, sjy, sjz, g.R2, lane);
        }
    }
    for (int k = min(w.count, w.cap) + lane; k < w.cap; k += 32) w.row[k] = g.n;   // pad = N (A5)
    if (lane == 0) {
        nbr_count[i] = w.count;
        ref_pos[i] = pi;
        if (w.count > ld_volatile(status + 1)) atomicMax(status + 1, w.count);
        if (w.count > w.cap) status[0] = 1;
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
template <int DIM>
__global__ void __launch_bounds__(256)
k_kick_drift(Geom g, float4 *__restrict__ pos, float4 *__restrict__ vel,
             const float4 *__restrict__ force, const float4 *__restrict__ ref, float a, float dt,
             int *flag) {
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
    if (__any_sync(FULL, moved) && (threadIdx.x & 31) == 0) *flag = 1;
}

// ------------------------------------- pair energy / force over the list (L78, L80, L104) --
// TPP lanes share one particle; each lane walks every TPP-th entry of the row (a group reads
// TPP consecutive int32 = whole 32-byte sectors when TPP = 8).  Pass 1 evaluates every pair in
// fp32 and also sums S = sum_j (|f_rep| + |f_att|)|d|_1, a bound on what rounding can have
// been amplified by.  A particle whose S exceeds thr * max(|F|, 1e-3) is re-evaluated in fp64
// from exact displacements (pass 2), so the fp32 result is only kept where its error estimate
// is far inside the 1e-5 tolerance.  Pairs whose fp32 r2 falls in a
// 2e-6 relative band around the LJ cutoff take their in/out decision from the exact fp64 r2,
// because the truncated force is discontinuous there.

struct Acc32 { float fx, fy, fz, e, s; };
struct Acc64 { double fx, fy, fz, e; };

template <int KIND>
__device__ __forceinline__ void pair32(const Pair &pp, float dx, float dy, float dz, float r2,
                                       float dsum, bool in, Acc32 &a) {
    if (KIND == 0) {
        float y = __frcp_rn(r2);
        float s2 = pp.sig2 * y;
        float s6 = s2 * s2 * s2;
        float c24 = 24.0f * pp.eps * y * s6;
        float coef = in ? c24 * fmaf(2.0f, s6, -1.0f) : 0.0f;
        float mag = in ? c24 * fmaf(2.0f, s6, 1.0f) : 0.0f;
        float u = in ? fmaf(4.0f * pp.eps * s6, s6 - 1.0f, -pp.u_cut) : 0.0f;
        a.fx = fmaf(coef, dx, a.fx); a.fy = fmaf(coef, dy, a.fy); a.fz = fmaf(coef, dz, a.fz);
        a.e = fmaf(0.5f, u, a.e);
        a.s = fmaf(mag, fabsf(dx) + fabsf(dy) + fabsf(dz), a.s);
    } else {
        float dij = 0.5f * dsum;
        float idij = __frcp_rn(dij);
        float y = rsqrtf(r2);                   // r2 = 0 -> inf, handled below
        float r = r2 * y;
        bool ok = in && (r2 > 0.0f) && (r < dij);
        float x = 1.0f - r * idij;
        float k = pp.eps * idij * y;
        float coef = ok ? k * x : 0.0f;
        float mag = ok ? k * (1.0f + r * idij) : 0.0f;
        float u = ok ? 0.5f * pp.eps * x * x : ((in && r2 == 0.0f && dij > 0.0f) ? 0.5f * pp.eps : 0.0f);
        a.fx = fmaf(coef, dx, a.fx); a.fy = fmaf(coef, dy, a.fy); a.fz = fmaf(coef, dz, a.fz);
        a.e = fmaf(0.5f, u, a.e);
        a.s = fmaf(mag, fabsf(dx) + fabsf(dy) + fabsf(dz), a.s);
    }
}

template <int KIND>
__device__ __forceinline__ void pair64(const Pair &pp, double dx, double dy, double dz,
                                       double dsum, Acc64 &a) {
    double r2 = dx * dx + dy * dy + dz * dz;
    if (KIND == 0) {
        if (r2 < pp.drc2) {
            double y = (double)__frcp_rn((float)r2);
            y = y * (2.0 - r2 * y);               // Newton: fp32 seed -> ~1e-14
            y = y * (2.0 - r2 * y);
            double s2 = pp.dsig2 * y;
            double s6 = s2 * s2 * s2;
            double coef = 24.0 * pp.deps * y * s6 * (2.0 * s6 - 1.0);
            a.fx += coef * dx; a.fy += coef * dy; a.fz += coef * dz;
            a.e += 0.5 * (4.0 * pp.deps * s6 * (s6 - 1.0) - pp.du_cut);
        }
    } else {
        double dij = 0.5 * dsum;
        double r = sqrt(r2);
        if (r < dij) {
            double x = 1.0 - r / dij;
            a.e += 0.25 * pp.deps * x * x;
            if (r > 0.0) {
                double coef = pp.deps / dij * x / r;
                a.fx += coef * dx; a.fy += coef * dy; a.fz += coef * dz;
            }
        }
    }
}

template <int KIND, int DIM, int TPP, bool WRAP>
__device__ __forceinline__ void row_pass32(const Geom &g, const Pair &pp,
                                           const float4 *__restrict__ pos,
                                           const int *__restrict__ row, int cnt, int sub,
                                           float4 pi, Acc32 &a) {
    const float band_lo = pp.rc2 * (1.0f - 2e-6f), band_hi = pp.rc2 * (1.0f + 2e-6f);
    for (int k = sub; k < cnt; k += 2 * TPP) {
        const int k1 = k + TPP;
        const bool v1 = k1 < cnt;
        const int j0 = row[k];
        const int j1 = row[v1 ? k1 : k];
        const float4 q[2] = {pos[j0], pos[j1]};
#pragma unroll
        for (int u = 0; u < 2; ++u) {
            float dx, dy, dz = 0.0f;
            if (WRAP) {
                dx = min_image(pi.x, q[u].x, g.L[0], g.h[0]);
                dy = min_image(pi.y, q[u].y, g.L[1], g.h[1]);
                if (DIM == 3) dz = min_image(pi.z, q[u].z, g.L[2], g.h[2]);
            } else {
                dx = pi.x - q[u].x; dy = pi.y - q[u].y;
                if (DIM == 3) dz = pi.z - q[u].z;
            }
            float r2 = fmaf(dz, dz, fmaf(dy, dy, dx * dx));
            bool in = (u == 0) || v1;
            if (KIND == 0) {
                bool inr = r2 < pp.rc2;
                if (r2 > band_lo && r2 < band_hi) {       // rare: decide on the exact r2
                    double ex = min_image64(pi.x, q[u].x, (double)g.L[0], (double)g.h[0]);
                    double ey = min_image64(pi.y, q[u].y, (double)g.L[1], (double)g.h[1]);
                    double ez = DIM == 3 ? min_image64(pi.z, q[u].z, (double)g.L[2], (double)g.h[2]) : 0.0;
                    inr = (ex * ex + ey * ey + ez * ez) < pp.drc2;
                }
                in = in && inr;
            }
            pair32<KIND>(pp, dx, dy, dz, r2, pi.w + q[u].w, in, a);
        }
    }
}

template <int KIND, int DIM, int TPP>
__device__ __forceinline__ void row_pass64(const Geom &g, const Pair &pp,
                                           const float4 *__restrict__ pos,
                                           const int *__restrict__ row, int cnt, int sub,
                                           float4 pi, Acc64 &a) {
    for (int k = sub; k < cnt; k += TPP) {
        const float4 q = pos[row[k]];
        double dx = min_image64(pi.x, q.x, (double)g.L[0], (double)g.h[0]);
        double dy = min_image64(pi.y, q.y, (double)g.L[1], (double)g.h[1]);
        double dz = DIM == 3 ? min_image64(pi.z, q.z, (double)g.L[2], (double)g.h[2]) : 0.0;
        pair64<KIND>(pp, dx, dy, dz, (double)pi.w + (double)q.w, a);
    }
}

template <int TPP, typename T>
__device__ __forceinline__ T group_sum(T v) {
#pragma unroll
    for (int o = TPP / 2; o > 0; o >>= 1) v += __shfl_xor_sync(FULL, v, o);
    return v;
}

// vel != NULL: also the second half-kick v += a F (L100).  energy_total != NULL: adds
// sum_i e_i in fp64 (one atomic per block).  book.stats != NULL: per-step bookkeeping.
template <int KIND, int DIM, int TPP>
__global__ void __launch_bounds__(256)
k_force(Geom g, Pair pp, const float4 *__restrict__ pos, const int *__restrict__ nbr_idx,
        const int *__restrict__ nbr_count, float4 *__restrict__ force, float4 *__restrict__ vel,
        float a, double *energy_total, Book book) {
    const int gid = blockIdx.x * blockDim.x + threadIdx.x;
    const int i = gid / TPP, sub = gid % TPP;
    const bool active = i < g.n;
    const int ii = active ? i : g.n - 1;
    const float4 pi = pos[ii];
    const int cnt = active ? min(nbr_count[ii], g.capacity) : 0;
    const int *row = nbr_idx + (size_t)ii * g.capacity;

    bool near = pi.x < g.face || pi.x > g.L[0] - g.face || pi.y < g.face || pi.y > g.L[1] - g.face;
    if (DIM == 3) near = near || pi.z < g.face || pi.z > g.L[2] - g.face;
    Acc32 a32 = {0.f, 0.f, 0.f, 0.f, 0.f};
    if (__any_sync(FULL, near && active))
        row_pass32<KIND, DIM, TPP, true>(g, pp, pos, row, cnt, sub, pi, a32);
    else
        row_pass32<KIND, DIM, TPP, false>(g, pp, pos, row, cnt, sub, pi, a32);
    float fx = group_sum<TPP>(a32.fx), fy = group_sum<TPP>(a32.fy), fz = group_sum<TPP>(a32.fz);
    float e = group_sum<TPP>(a32.e), s = group_sum<TPP>(a32.s);

    // pass 2: fp64 re-evaluation where rounding may matter
    float fn = sqrtf(fmaf(fz, fz, fmaf(fy, fy, fx * fx)));
    const bool keep32 = (s <= pp.thr * fmaxf(fn, 1e-3f)) && (s < 1e30f);   // NaN/inf -> fp64
    if (!keep32) {                                // uniform within the TPP group
        Acc64 a64 = {0.0, 0.0, 0.0, 0.0};
        row_pass64<KIND, DIM, TPP>(g, pp, pos, row, cnt, sub, pi, a64);
        // reduce inside the group only: lanes of other groups are not here
        unsigned gm = (TPP == 32) ? FULL : (((1u << TPP) - 1u) << ((threadIdx.x & 31) / TPP * TPP));
#pragma unroll
        for (int o = TPP / 2; o > 0; o >>= 1) {
            a64.fx += __shfl_xor_sync(gm, a64.fx, o);
            a64.fy += __shfl_xor_sync(gm, a64.fy, o);
            a64.fz += __shfl_xor_sync(gm, a64.fz, o);
            a64.e += __shfl_xor_sync(gm, a64.e, o);
        }
        fx = (float)a64.fx; fy = (float)a64.fy; fz = (float)a64.fz; e = (float)a64.e;
    }
    if (active && sub == 0) {
        force[i] = make_float4(fx, fy, DIM == 3 ? fz : 0.0f, e);
        if (vel) {
            float4 v = vel[i];
            v.x = fmaf(a, fx, v.x); v.y = fmaf(a, fy, v.y);
            if (DIM == 3) v.z = fmaf(a, fz, v.z);
            vel[i] = v;
        }
    }
    if (energy_total) {
        __shared__ double red[8];
        double x = (active && sub == 0) ? (double)e : 0.0;
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
    if (book.stats && gid == 0) {
        if (ld_volatile(book.flag)) {
            book.stats[1] += 1;
            int mc = ld_volatile(book.status + 1);
            if (mc > book.stats[3]) book.stats[3] = mc;
            if (ld_volatile(book.status) && book.stats[2] < 0) book.stats[2] = book.stats[0];
            *book.flag = 0;
        }
        book.stats[0] += 1;
    }
}

} // namespace mdk
