// md_nh.cuh -- NVT by a Nose-Hoover thermostat (a chain of 1..8, below) around the velocity-Verlet step (
// PAPER.md:L100 "Nose-Hoover [67]"; no formulas in the paper: the explicit reversible splitting of
// Martyna, Tuckerman, Tobias and Klein, reading A23).  dof = dim n, Q = dof kT tau^2.
// Thermostat half step: K2 = sum m v^2; G = (K2 - dof kT)/Q; vxi += dt/4 G; s = exp(-dt/2 vxi);
// v *= s; xi += dt/2 vxi; K2 *= s^2; G = (K2 - dof kT)/Q; vxi += dt/4 G.  (xi, vxi) live in a
// device double[2]; the velocity sum is reduced in two deterministic stages.
#pragma once
#include "md_kernels.cuh"

namespace mdk {

constexpr int NH_BLOCK = 256;

__global__ void __launch_bounds__(NH_BLOCK)
k_nh_ke(int n, int dim, const float4 *__restrict__ vel, double *__restrict__ partial,
        const float *__restrict__ pending) {
    __shared__ double red[NH_BLOCK / 32];
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    double s = 0.0;
    const float sp = *pending;        // a scale the stored velocities have still to take (1: none)
    if (i < n) {
        float4 v = vel[i];
        v.x *= sp; v.y *= sp; v.z *= sp;
        s = (double)v.x * v.x + (double)v.y * v.y + (dim == 3 ? (double)v.z * v.z : 0.0);
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(FULL, s, o);
    if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = s;
    __syncthreads();
    if (threadIdx.x == 0) {
        double t = 0.0;
        for (int k = 0; k < NH_BLOCK / 32; ++k) t += red[k];                 // fixed order
        partial[blockIdx.x] = t;
    }
}

// Chain of M thermostats ([67] Martyna, Klein, Tuckerman): Q_1 = dof kT tau^2, Q_j = kT tau^2; state =
// {xi_1..xi_M, v_1..v_M}.  Half step, d = dt/2: v_M += d/2 G_M; for j = M-1..1: a = exp(-d/4 v_{j+1}),
// v_j = (v_j a + d/2 G_j) a; s = exp(-d v_1); K2 *= s^2; xi_j += d v_j; then the same updates for
// j = 1..M-1 and v_M last, with G_1 = (K2 - dof kT)/Q_1, G_j = (Q_{j-1} v_{j-1}^2 - kT)/Q_j.
constexpr int NH_MAX_CHAIN = 8;

__device__ __forceinline__ double nh_G(int j, double K2, double dofkT, double kT, const double *Q, const double *v) {
    return j == 0 ? (K2 - dofkT) / Q[0] : (Q[j - 1] * v[j - 1] * v[j - 1] - kT) / Q[j];
}

__global__ void __launch_bounds__(256)
k_nh_finalize(int nblocks, const double *__restrict__ partial, double mass, double dofkT, double kT, double tau2,
              int M, double dt, double *state, float *scale) {
    __shared__ double red[256];
    double s = 0.0;
    for (int b = threadIdx.x; b < nblocks; b += 256) s += partial[b];
    red[threadIdx.x] = s;
    __syncthreads();
    for (int o = 128; o > 0; o >>= 1) {
        if ((int)threadIdx.x < o) red[threadIdx.x] += red[threadIdx.x + o];
        __syncthreads();
    }
    if (threadIdx.x == 0) {
        double Q[NH_MAX_CHAIN], xi[NH_MAX_CHAIN], v[NH_MAX_CHAIN];
        for (int j = 0; j < M; ++j) { Q[j] = (j == 0 ? dofkT : kT) * tau2; xi[j] = state[j]; v[j] = state[M + j]; }
        double K2 = mass * red[0];
        v[M - 1] += 0.25 * dt * nh_G(M - 1, K2, dofkT, kT, Q, v);
        for (int j = M - 2; j >= 0; --j) {
            const double a = exp(-0.125 * dt * v[j + 1]);
            v[j] = (v[j] * a + 0.25 * dt * nh_G(j, K2, dofkT, kT, Q, v)) * a;
        }
        const double sc = exp(-0.5 * dt * v[0]);
        for (int j = 0; j < M; ++j) xi[j] += 0.5 * dt * v[j];
        K2 *= sc * sc;
        for (int j = 0; j < M - 1; ++j) {
            const double a = exp(-0.125 * dt * v[j + 1]);
            v[j] = (v[j] * a + 0.25 * dt * nh_G(j, K2, dofkT, kT, Q, v)) * a;
        }
        v[M - 1] += 0.25 * dt * nh_G(M - 1, K2, dofkT, kT, Q, v);
        for (int j = 0; j < M; ++j) { state[j] = xi[j]; state[M + j] = v[j]; }
        *scale = (float)sc;
    }
}

// first half: v *= s, then the opening of the velocity-Verlet step exactly as k_kick_drift
template <int DIM>
__global__ void __launch_bounds__(256)
k_nh_kick_drift(Geom g, float4 *__restrict__ pos, float4 *__restrict__ vel,
                const float4 *__restrict__ force, const float4 *__restrict__ ref, float a, float dt,
                const float *__restrict__ scale, const float *__restrict__ pending, Raise rs) {
    const float sc = *scale, sp = *pending;
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    bool moved = false;
    if (i < g.n) {
        float4 p = pos[i], v = vel[i], f = force[i];
        v.x *= sp; v.y *= sp; v.z *= sp;     // the closing thermostat half step of the previous MD step (k_nh_scale)
        v.x = fmaf(a, f.x, sc * v.x);
        v.y = fmaf(a, f.y, sc * v.y);
        p.x = wrap(fmaf(dt, v.x, p.x), g.L[0], g.inv_L[0]);
        p.y = wrap(fmaf(dt, v.y, p.y), g.L[1], g.inv_L[1]);
        if (DIM == 3) {
            v.z = fmaf(a, f.z, sc * v.z);
            p.z = wrap(fmaf(dt, v.z, p.z), g.L[2], g.inv_L[2]);
        }
        pos[i] = p; vel[i] = v;
        moved = disp2_from_ref<DIM>(g, p, ref[i]) > g.half_skin2;
    }
    if (__any_sync(FULL, moved) && (threadIdx.x & 31) == 0) raise_rebuild(rs);
}

// scale = {this half step's factor, the factor the stored velocities have still to take, 1}
__global__ void k_nh_begin(float *scale) { scale[1] = 1.0f; scale[2] = 1.0f; }

// the pending factor into the stored velocities (when a call ends)
__global__ void __launch_bounds__(256)
k_nh_scale(int n, float4 *__restrict__ vel, const float *__restrict__ scale) {
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const float sc = *scale;
    float4 v = vel[i];
    v.x *= sc; v.y *= sc; v.z *= sc;
    vel[i] = v;
}

} // namespace mdk
