// md_flock.cuh -- flocking as an energy model on the same cell / neighbor list (
// PAPER.md App. B: eqs. 3-10 and the forward-Euler dynamics of eqs. 4-5; what the text
// leaves open is DESIGN.md reading A25).  2-D; the heading theta_i travels in pos.w, so a neighbor's
// heading arrives with its position in one gather and follows the re-sort.
//   rho(r; Rc) = (1/alpha)(1 - r/Rc)^alpha, r < Rc
//   E_align = 1/2 sum_{i!=j} J_al rho(r; R_al)(1 - N_i.N_j)^2   (stop-gradient: no R gradient)
//   E_avoid = 1/2 sum_{i!=j} J_av rho(r; R_av)
//   E_coh   = sum_i 1/2 J_co (1 - Dhat_i.N_i)^2,  D_i = sum_{j: r < R_co} (R_j - R_i)
//   R_i' = mu(R_i, dt (v N_i - grad_{R_i} E)),  theta_i' = theta_i - dt grad_{theta_i} E
// grad_{R_k} E_coh = -|N_k| g_k + sum_{i: r_ki < R_co} g_i with g_i = dE_coh,i/dD_i, hence two passes
// over the list (g first, then its gather) before the update.  fp64 accumulation, fp32 state.
#pragma once
#include "md_kernels.cuh"

namespace mdk {

constexpr int FLOCK_U = 4;

struct FlockPar {
    double Jal, Ral, Jav, Rav, Jco, Rco, alpha, speed;
    int nobs;                                   // obstacles (App. B.3.1): centres, radii, J
    double Job;
    float ox[MD_MAX_OBSTACLES], oy[MD_MAX_OBSTACLES], oD[MD_MAX_OBSTACLES];
    int npred;                                  // predators (App. B.3.2): device state (x, y, 0, theta)
    const float4 *pred;
    double Jfl, Rfl, Jch, Rch, vpred;
};

__device__ __forceinline__ void flock_disp(const Geom &g, const float4 &pi, const float4 &q, double &dx, double &dy) {
    dx = (double)pi.x - (double)q.x; dy = (double)pi.y - (double)q.y;
    const double hx = 0.5 * (double)g.L[0], hy = 0.5 * (double)g.L[1];
    dx -= dx > hx ? (double)g.L[0] : (dx < -hx ? -(double)g.L[0] : 0.0);
    dy -= dy > hy ? (double)g.L[1] : (dy < -hy ? -(double)g.L[1] : 0.0);
}

// x^a for x in (0, 1].  AI > 0: a = AI is a small integer known at compile time (the usual alpha = 3)
// and the power is AI - 1 multiplications; AI = 0: any real a by pow.  NEG1: the exponent is a - 1.
template <int AI, bool NEG1>
__device__ __forceinline__ double flock_pow(double x, double a) {
    if (AI == 0) return pow(x, NEG1 ? a - 1.0 : a);
    constexpr int n = NEG1 ? AI - 1 : AI;
    double y = 1.0;
#pragma unroll
    for (int k = 0; k < n; ++k) y *= x;
    return y;
}

// The disk term of eq. 11 for one boid (or predator) at pi heading (ci, si) and one disk (centre, radius D):
// e = J rho(r; D)(1 + N.u)^2, u = (C - R)/r, inside the disk only; adds its gradients.
template <int AI>
__device__ __forceinline__ void flock_disk_term(const Geom &g, const FlockPar &fp, const float4 &pi, double ci,
                                                double si, float cx, float cy, double D, double J,
                                                double &gx, double &gy, double &gt) {
    double dx, dy;
    flock_disp(g, pi, make_float4(cx, cy, 0.0f, 0.0f), dx, dy);                      // R - C
    const double r2 = dx * dx + dy * dy;
    if (r2 < D * D && r2 > 0.0) {                     // most boids are outside most disks: no root for them
        const double r = sqrt(r2);
        const double ux = -dx / r, uy = -dy / r, c = ci * ux + si * uy, x = fmax(1.0 - r / D, 0.0);
        const double rho = flock_pow<AI, false>(x, fp.alpha) / fp.alpha;
        const double drho = -flock_pow<AI, true>(x, fp.alpha) / D;
        gt += 2.0 * J * rho * (1.0 + c) * (-si * ux + ci * uy);
        gx += -J * (drho * (1.0 + c) * (1.0 + c) * ux + 2.0 * rho * (1.0 + c) * (ci - c * ux) / r);
        gy += -J * (drho * (1.0 + c) * (1.0 + c) * uy + 2.0 * rho * (1.0 + c) * (si - c * uy) / r);
    }
}

// (cos theta_i, sin theta_i) in fp64, once per boid and step: pass 1 forms the sine and cosine of
// theta_i - theta_j from these by the angle-difference identities instead of one fp64 sincos per pair.
__global__ void __launch_bounds__(256)
k_flock_trig(int n, const float4 *__restrict__ pos, double2 *__restrict__ cs) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    double si, ci;
    sincos((double)pos[i].w, &si, &ci);
    cs[i] = make_double2(ci, si);
}

// pass 1: acc[i] = (grad_R without the gathered cohesion part, grad_theta, |N_i|), gco[i] = g_i
template <int AI>
__global__ void __launch_bounds__(128)
k_flock_pass1(Geom g, FlockPar fp, const float4 *__restrict__ pos, const double2 *__restrict__ cs,
              const int *__restrict__ nbr_idx, const int *__restrict__ nbr_count,
              float4 *__restrict__ acc, float4 *__restrict__ gco) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= g.n) return;
    const float4 pi = pos[i];
    const int cnt = min(nbr_count[i], g.capacity);
    const int *col = nbr_idx + nbr_tile_base(i, g.capacity) + (i & 31);
    const double2 ti = cs[i];
    const double ci = ti.x, si = ti.y;
    const double iRal = 1.0 / fp.Ral, iRav = 1.0 / fp.Rav;
    const double cal = 2.0 * fp.Jal / fp.alpha, cav = -fp.Jav * iRav;
    double gx = 0.0, gy = 0.0, gt = 0.0, Dx = 0.0, Dy = 0.0;
    int m = 0;
    for (int k = 0; k < cnt; k += FLOCK_U) {            // FLOCK_U independent gathers in flight
        int j[FLOCK_U]; float4 q[FLOCK_U]; double2 tj[FLOCK_U];
#pragma unroll
        for (int u = 0; u < FLOCK_U; ++u) j[u] = k + u < cnt ? col[(k + u) * TILE] : i;
#pragma unroll
        for (int u = 0; u < FLOCK_U; ++u) { q[u] = pos[j[u]]; tj[u] = cs[j[u]]; }
#pragma unroll
        for (int u = 0; u < FLOCK_U; ++u) {
            double dx, dy;
            flock_disp(g, pi, q[u], dx, dy);
            // r and 1/r: fp32 rsqrt refined by one Newton step in fp64 (relative error ~1e-13)
            // instead of an fp64 square root and an fp64 division per pair
            const double r2 = dx * dx + dy * dy;
            double ir = (double)rsqrtf((float)r2);
            ir = r2 > 0.0 ? ir * (1.5 - 0.5 * r2 * ir * ir) : 0.0;
            const double r = r2 * ir;
            const bool valid = k + u < cnt;
            if (valid && r < fp.Ral) {
                const double sd = si * tj[u].x - ci * tj[u].y, cd = ci * tj[u].x + si * tj[u].y;
                gt += cal * flock_pow<AI, false>(1.0 - r * iRal, fp.alpha) * (1.0 - cd) * sd;
            }
            if (valid && r < fp.Rav && r > 0.0) {
                const double dr = cav * flock_pow<AI, true>(1.0 - r * iRav, fp.alpha) * ir;
                gx += dr * dx; gy += dr * dy;
            }
            if (valid && r < fp.Rco) { Dx -= dx; Dy -= dy; ++m; }
        }
    }
    double Gx = 0.0, Gy = 0.0;
    const double Dn = sqrt(Dx * Dx + Dy * Dy);
    if (m > 0 && Dn > 0.0) {
        const double hx = Dx / Dn, hy = Dy / Dn, c = hx * ci + hy * si;
        Gx = -fp.Jco * (1.0 - c) * (ci - c * hx) / Dn;
        Gy = -fp.Jco * (1.0 - c) * (si - c * hy) / Dn;
        gt += -fp.Jco * (1.0 - c) * (-hx * si + hy * ci);
        gx -= m * Gx; gy -= m * Gy;
    }
    // obstacles (eq. 11), then the predators as moving disks of radius R_flee (eq. 12)
    for (int o = 0; o < fp.nobs; ++o)
        flock_disk_term<AI>(g, fp, pi, ci, si, fp.ox[o], fp.oy[o], (double)fp.oD[o], fp.Job, gx, gy, gt);
    for (int p = 0; p < fp.npred; ++p) {
        const float4 q = fp.pred[p];
        flock_disk_term<AI>(g, fp, pi, ci, si, q.x, q.y, fp.Rfl, fp.Jfl, gx, gy, gt);
    }
    acc[i] = make_float4((float)gx, (float)gy, (float)gt, (float)m);
    gco[i] = make_float4((float)Gx, (float)Gy, 0.0f, 0.0f);
}

// pass 2: acc[i].xy += sum over the neighbors within R_co of their g
__global__ void __launch_bounds__(128)
k_flock_pass2(Geom g, FlockPar fp, const float4 *__restrict__ pos, const int *__restrict__ nbr_idx,
              const int *__restrict__ nbr_count, float4 *__restrict__ acc, const float4 *__restrict__ gco) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= g.n) return;
    const float4 pi = pos[i];
    const int cnt = min(nbr_count[i], g.capacity);
    const int *col = nbr_idx + nbr_tile_base(i, g.capacity) + (i & 31);
    const double Rco2 = fp.Rco * fp.Rco;
    double gx = 0.0, gy = 0.0;
    for (int k = 0; k < cnt; k += FLOCK_U) {
        int j[FLOCK_U]; float4 q[FLOCK_U], G[FLOCK_U];
#pragma unroll
        for (int u = 0; u < FLOCK_U; ++u) j[u] = k + u < cnt ? col[(k + u) * TILE] : i;
#pragma unroll
        for (int u = 0; u < FLOCK_U; ++u) { q[u] = pos[j[u]]; G[u] = gco[j[u]]; }
#pragma unroll
        for (int u = 0; u < FLOCK_U; ++u) {
            double dx, dy;
            flock_disp(g, pi, q[u], dx, dy);
            if (k + u < cnt && dx * dx + dy * dy < Rco2) { gx += (double)G[u].x; gy += (double)G[u].y; }
        }
    }
    float4 a = acc[i];
    a.x = (float)((double)a.x + gx); a.y = (float)((double)a.y + gy);
    acc[i] = a;
}

// Predators (eq. 13), two stages so that the sum over all boids uses the whole GPU and still has a fixed
// order: block (c, p) sums its chunk of boids within R_chase of predator p into part[(p * nchunk + c) * 3],
// then one warp per predator adds the chunks in order, takes the chase gradient, adds the obstacles and
// moves the predator by forward Euler.  Both run after the boids' passes (which read the old predator
// state) and before the boids' update (they read the old boid positions).
constexpr int FLOCK_PRED_CHUNKS = 64;

__global__ void __launch_bounds__(256)
k_flock_pred_partial(Geom g, FlockPar fp, const float4 *__restrict__ pos, const float4 *__restrict__ pred,
                     double *__restrict__ part) {
    __shared__ double sx[8], sy[8], sm[8];
    const int p = blockIdx.y, lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const float4 q = pred[p];
    const double R2 = fp.Rch * fp.Rch;
    const int per = (g.n + gridDim.x - 1) / gridDim.x;
    const int i1 = min(g.n, (int)(blockIdx.x + 1) * per);
    double Dx = 0.0, Dy = 0.0, m = 0.0;
    for (int i = blockIdx.x * per + threadIdx.x; i < i1; i += 256) {
        double dx, dy;
        flock_disp(g, pos[i], q, dx, dy);                                            // R_i - R_p
        if (dx * dx + dy * dy < R2) { Dx += dx; Dy += dy; m += 1.0; }
    }
    for (int o = 16; o > 0; o >>= 1) {
        Dx += __shfl_xor_sync(FULL, Dx, o); Dy += __shfl_xor_sync(FULL, Dy, o); m += __shfl_xor_sync(FULL, m, o);
    }
    if (lane == 0) { sx[warp] = Dx; sy[warp] = Dy; sm[warp] = m; }
    __syncthreads();
    if (threadIdx.x == 0) {
        Dx = Dy = m = 0.0;
        for (int w = 0; w < 8; ++w) { Dx += sx[w]; Dy += sy[w]; m += sm[w]; }
        double *out = part + ((size_t)p * gridDim.x + blockIdx.x) * 3;
        out[0] = Dx; out[1] = Dy; out[2] = m;
    }
}

template <int AI>
__global__ void __launch_bounds__(32)
k_flock_predators(Geom g, FlockPar fp, float4 *pred, const double *__restrict__ part, int nchunk, float dt) {
    const int p = blockIdx.x;
    if (threadIdx.x != 0) return;
    const float4 q = pred[p];
    double Dx = 0.0, Dy = 0.0, md = 0.0;
    for (int c = 0; c < nchunk; ++c) {
        const double *in = part + ((size_t)p * nchunk + c) * 3;
        Dx += in[0]; Dy += in[1]; md += in[2];
    }
    const int m = (int)md;
    double sn, cp;
    sincos((double)q.w, &sn, &cp);
    double gx = 0.0, gy = 0.0, gt = 0.0;
    const double Dn = sqrt(Dx * Dx + Dy * Dy);
    if (m > 0 && Dn > 0.0) {
        const double hx = Dx / Dn, hy = Dy / Dn, c = hx * cp + hy * sn;
        gt = -fp.Jch * (1.0 - c) * (-hx * sn + hy * cp);
        gx = m * fp.Jch * (1.0 - c) * (cp - c * hx) / Dn;
        gy = m * fp.Jch * (1.0 - c) * (sn - c * hy) / Dn;
    }
    for (int o = 0; o < fp.nobs; ++o)
        flock_disk_term<AI>(g, fp, q, cp, sn, fp.ox[o], fp.oy[o], (double)fp.oD[o], fp.Job, gx, gy, gt);
    float4 out = q;
    const float v = (float)fp.vpred, ax = (float)gx, ay = (float)gy, at = (float)gt;
    float snf, csf;
    sincosf(q.w, &snf, &csf);
    out.x = wrap(fmaf(dt, fmaf(v, csf, -ax), q.x), g.L[0], g.inv_L[0]);
    out.y = wrap(fmaf(dt, fmaf(v, snf, -ay), q.y), g.L[1], g.inv_L[1]);
    out.w = fmaf(-dt, at, q.w);
    pred[p] = out;
}

// forward Euler (eqs. 4-5), half-skin test
__global__ void __launch_bounds__(256)
k_flock_update(Geom g, FlockPar fp, float4 *__restrict__ pos, const float4 *__restrict__ acc,
               const float4 *__restrict__ ref, float dt, Raise rs) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    bool moved = false;
    if (i < g.n) {
        float4 p = pos[i];
        const float4 a = acc[i];
        float sn, cs;
        sincosf(p.w, &sn, &cs);
        const float v = (float)fp.speed;
        p.x = wrap(fmaf(dt, fmaf(v, cs, -a.x), p.x), g.L[0], g.inv_L[0]);
        p.y = wrap(fmaf(dt, fmaf(v, sn, -a.y), p.y), g.L[1], g.inv_L[1]);
        p.w = fmaf(-dt, a.z, p.w);
        pos[i] = p;
        moved = disp2_from_ref<2>(g, p, ref[i]) > g.half_skin2;
    }
    if (__any_sync(FULL, moved) && (threadIdx.x & 31) == 0) raise_rebuild(rs);
}

// step bookkeeping (what the force kernel does for the other rules)
__global__ void k_flock_book(Book book) {
    if (ld_volatile(book.flag)) {
        book.stats[1] += 1;
        const int mc = ld_volatile(book.status + 1);
        if (mc > book.stats[3]) book.stats[3] = mc;
        if (ld_volatile(book.status) && book.stats[2] < 0) book.stats[2] = book.stats[0];
        *book.flag = 0;
    }
    book.stats[0] += 1;
}

} // namespace mdk
