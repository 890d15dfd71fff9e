// md_nh.cuh -- NVT by one Nose-Hoover thermostat around the velocity-Verlet step (
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
k_nh_ke(int n, int dim, const float4 *__restrict__ vel, double *__restrict__ partial) {
    __shared__ double red[NH_BLOCK / 32];
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    double s = 0.0;
    if (i < n) {
        const float4 v = vel[i];
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

__global__ void __launch_bounds__(256)
k_nh_finalize(int nblocks, const double *__restrict__ partial, double mass, double dofkT, double Q,
              double dt, double *state, float *scale) {
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
        double K2 = mass * red[0], xi = state[0], vxi = state[1];
        double G = (K2 - dofkT) / Q;
        vxi += 0.25 * dt * G;
        const double sc = exp(-0.5 * dt * vxi);
        xi += 0.5 * dt * vxi;
        K2 *= sc * sc;
        G = (K2 - dofkT) / Q;
        vxi += 0.25 * dt * G;
        state[0] = xi; state[1] = vxi;
        *scale = (float)sc;
    }
}

// first half: v *= s, then the opening of the velocity-Verlet step exactly as k_kick_drift
template <int DIM>
__global__ void __launch_bounds__(256)
k_nh_kick_drift(Geom g, float4 *__restrict__ pos, float4 *__restrict__ vel,
                const float4 *__restrict__ force, const float4 *__restrict__ ref, float a, float dt,
                const float *__restrict__ scale, Raise rs) {
    const float sc = *scale;
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    bool moved = false;
    if (i < g.n) {
        float4 p = pos[i], v = vel[i], f = force[i];
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
