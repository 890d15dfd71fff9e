// md_fire.cuh -- FIRE minimisation around the same drift / rebuild / force sequence as the NVE
// step ("FIRE Descent", used to relax packings in §4.2; the
// paper gives no formulas: algorithm of Bitzek et al. 2006, reading A20).  Unit mass.
//   1. v += dt/2 F;  r = mu(r, dt v);  [rebuild];  F = F(r);  v += dt/2 F
//   2. P = sum F.v, FF = sum F.F, VV = sum v.v                 (fp64 sums of fp32 products)
//   3. (applied at the start of the next step's kernel 1, or by k_fire_mix when the call ends)
//      P > 0: v = (1 - alpha) v + alpha sqrt(VV / FF) F; n_pos += 1;
//             n_pos > n_min: dt = min(dt f_inc, dt_max), alpha *= f_alpha
//      else:  v = 0; n_pos = 0; dt *= f_dec; alpha = alpha_start
// dt, alpha, n_pos live in a device float[4] (`state`), so the step size never leaves the device.
#pragma once
#include "md_kernels.cuh"

namespace mdk {

struct FirePar { float dt_start, dt_max; int n_min; float f_inc, f_dec, alpha_start, f_alpha; };

// state = {dt, alpha, n_pos, last P (sign only)}; a non-positive dt on entry means "start".
// coef: the mixing coefficients {c1, c2} the velocities have still to take; none at the start of a call
__global__ void k_fire_init(FirePar p, float *state, float *coef) {
    if (!(state[0] > 0.0f)) { state[0] = p.dt_start; state[1] = p.alpha_start; state[2] = 0.0f; state[3] = 0.0f; }
    coef[0] = 1.0f; coef[1] = 0.0f;
}

template <int DIM>
__global__ void __launch_bounds__(256)
k_fire_kick_drift(Geom g, float4 *__restrict__ pos, float4 *__restrict__ vel,
                  const float4 *__restrict__ force, const float4 *__restrict__ ref,
                  const float *__restrict__ state, const float *__restrict__ coef, Raise rs) {
    const float dt = state[0], a = 0.5f * dt;
    const float c1 = coef[0], c2 = coef[1];
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    bool moved = false;
    if (i < g.n) {
        float4 p = pos[i], v = vel[i], f = force[i];
        // the mixing step 3 of the previous MD step (k_fire_mix's arithmetic; {1, 0} leaves v as it is)
        v.x = fmaf(c2, f.x, c1 * v.x); v.y = fmaf(c2, f.y, c1 * v.y); v.z = fmaf(c2, f.z, c1 * v.z);
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
    if (__any_sync(FULL, moved) && (threadIdx.x & 31) == 0) raise_rebuild(rs);
}

// second half-kick and the three sums; block b writes its partial sums to partial[3 b ..]
constexpr int FIRE_BLOCK = 256;
__global__ void __launch_bounds__(FIRE_BLOCK)
k_fire_kick_reduce(int n, int dim, float4 *__restrict__ vel, const float4 *__restrict__ force,
                   const float *__restrict__ state, double *__restrict__ partial) {
    __shared__ double red[3][FIRE_BLOCK / 32];
    const float a = 0.5f * state[0];
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    double P = 0.0, FF = 0.0, VV = 0.0;
    if (i < n) {
        float4 v = vel[i];
        const float4 f = force[i];
        v.x = fmaf(a, f.x, v.x); v.y = fmaf(a, f.y, v.y);
        if (dim == 3) v.z = fmaf(a, f.z, v.z);
        vel[i] = v;
        P = (double)f.x * v.x + (double)f.y * v.y + (dim == 3 ? (double)f.z * v.z : 0.0);
        FF = (double)f.x * f.x + (double)f.y * f.y + (dim == 3 ? (double)f.z * f.z : 0.0);
        VV = (double)v.x * v.x + (double)v.y * v.y + (dim == 3 ? (double)v.z * v.z : 0.0);
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        P += __shfl_xor_sync(FULL, P, o); FF += __shfl_xor_sync(FULL, FF, o); VV += __shfl_xor_sync(FULL, VV, o);
    }
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    if (lane == 0) { red[0][w] = P; red[1][w] = FF; red[2][w] = VV; }
    __syncthreads();
    if (threadIdx.x < 3) {
        double t = 0.0;
        for (int k = 0; k < FIRE_BLOCK / 32; ++k) t += red[threadIdx.x][k];      // fixed order
        partial[3 * blockIdx.x + threadIdx.x] = t;
    }
}

// one block: sums the partials in a fixed order, takes the FIRE decision, writes the new state
// and the mixing coefficients coef = {c1, c2}: v = c1 v + c2 F
__global__ void __launch_bounds__(256)
k_fire_finalize(int nblocks, const double *__restrict__ partial, FirePar p, float *state, float *coef) {
    __shared__ double red[3][256];
    double s[3] = {0.0, 0.0, 0.0};
    for (int b = threadIdx.x; b < nblocks; b += 256) {
        s[0] += partial[3 * b]; s[1] += partial[3 * b + 1]; s[2] += partial[3 * b + 2];
    }
    for (int q = 0; q < 3; ++q) red[q][threadIdx.x] = s[q];
    __syncthreads();
    for (int o = 128; o > 0; o >>= 1) {
        if ((int)threadIdx.x < o) for (int q = 0; q < 3; ++q) red[q][threadIdx.x] += red[q][threadIdx.x + o];
        __syncthreads();
    }
    if (threadIdx.x == 0) {
        const double P = red[0][0], FF = red[1][0], VV = red[2][0];
        float dt = state[0], alpha = state[1];
        int n_pos = (int)state[2];
        float c1, c2;
        if (P > 0.0) {
            c1 = 1.0f - alpha;
            c2 = FF > 0.0 ? (float)((double)alpha * sqrt(VV / FF)) : 0.0f;
            n_pos += 1;
            if (n_pos > p.n_min) { dt = fminf(dt * p.f_inc, p.dt_max); alpha = alpha * p.f_alpha; }
        } else {
            c1 = 0.0f; c2 = 0.0f; n_pos = 0; dt = dt * p.f_dec; alpha = p.alpha_start;
        }
        state[0] = dt; state[1] = alpha; state[2] = (float)n_pos; state[3] = (float)(P > 0.0 ? 1.0 : -1.0);
        coef[0] = c1; coef[1] = c2;
    }
}

__global__ void __launch_bounds__(256)
k_fire_mix(int n, float4 *__restrict__ vel, const float4 *__restrict__ force, const float *__restrict__ coef) {
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const float c1 = coef[0], c2 = coef[1];
    float4 v = vel[i];
    const float4 f = force[i];
    v.x = fmaf(c2, f.x, c1 * v.x); v.y = fmaf(c2, f.y, c1 * v.y); v.z = fmaf(c2, f.z, c1 * v.z);
    vel[i] = v;
}

} // namespace mdk
