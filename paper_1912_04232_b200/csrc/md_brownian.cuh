// md_brownian.cuh -- overdamped (Brownian) dynamics and, at kT = 0, gradient descent around the same
// device-side rebuild / force sequence ("Brownian simulations at
// constant temperature", "Gradient Descent"; no formulas in the paper: Euler-Maruyama, DESIGN.md
// reading A21):   r_i = mu(r_i, (dt/gamma) F_i + sqrt(2 kT dt / gamma) xi_i).
// xi comes from a counter-based generator keyed by (seed, step, ORIGINAL particle id, pair index),
// so the noise does not depend on the particle order the re-sort leaves: splitmix64 finaliser ->
// two 24-bit uniforms -> Box-Muller (the CPU oracle implements the same generator on its own).
#pragma once
#include "md_kernels.cuh"

namespace mdk {

__device__ __forceinline__ void normal_pair(unsigned seed, unsigned step, unsigned id, unsigned c,
                                            float &g0, float &g1) {
    unsigned long long z = (unsigned long long)seed * 0x9E3779B97F4A7C15ull
                         + (unsigned long long)step * 0xBF58476D1CE4E5B9ull
                         + (unsigned long long)id * 0x94D049BB133111EBull + (unsigned long long)c;
    z ^= z >> 30; z *= 0xBF58476D1CE4E5B9ull;
    z ^= z >> 27; z *= 0x94D049BB133111EBull;
    z ^= z >> 31;
    const float u1 = (float)((unsigned)(z >> 40) + 1u) * (1.0f / 16777216.0f);        // (0, 1]
    const float u2 = (float)((unsigned)(z >> 8) & 0xFFFFFFu) * (1.0f / 16777216.0f);  // [0, 1)
    const float r = sqrtf(-2.0f * logf(u1));
    float sn, cs;
    sincospif(2.0f * u2, &sn, &cs);
    g0 = r * cs; g1 = r * sn;
}

template <int DIM>
__global__ void __launch_bounds__(256)
k_brownian_drift(Geom g, float4 *__restrict__ pos, const float4 *__restrict__ force,
                 const int *__restrict__ id, const float4 *__restrict__ ref, float mu, float amp,
                 const unsigned *__restrict__ seed_step0, const int *__restrict__ steps_done, Raise rs) {
    // {seed, step0} live in device words (written before every call), so that a caller who continues a
    // noise stream with a new step0 re-uses the captured graphs
    const unsigned seed = seed_step0[0];
    const unsigned step = seed_step0[1] + (unsigned)*steps_done;      // stats[0]: steps finished in this call
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    bool moved = false;
    if (i < g.n) {
        float4 p = pos[i];
        const float4 f = force[i];
        float gx = 0.0f, gy = 0.0f, gz = 0.0f, unused;
        if (amp != 0.0f) {
            const unsigned key = (unsigned)(id ? id[i] : i);
            normal_pair(seed, step, key, 0u, gx, gy);
            if (DIM == 3) normal_pair(seed, step, key, 1u, gz, unused);
        }
        p.x = wrap(fmaf(amp, gx, fmaf(mu, f.x, p.x)), g.L[0], g.inv_L[0]);
        p.y = wrap(fmaf(amp, gy, fmaf(mu, f.y, p.y)), g.L[1], g.inv_L[1]);
        if (DIM == 3) p.z = wrap(fmaf(amp, gz, fmaf(mu, f.z, p.z)), g.L[2], g.inv_L[2]);
        pos[i] = p;
        moved = disp2_from_ref<DIM>(g, p, ref[i]) > g.half_skin2;
    }
    if (__any_sync(FULL, moved) && (threadIdx.x & 31) == 0) raise_rebuild(rs);
}

// Langevin dynamics, BAOAB (reading A22), first four letters:
//   B: v += a F;  A: r += dt/2 v;  O: v = c1 v + c2 xi;  A: r = mu(r, dt/2 v);  half-skin test.
// The force kernel that follows applies the closing B (its second half-kick).
template <int DIM>
__global__ void __launch_bounds__(256)
k_langevin_baoa(Geom g, float4 *__restrict__ pos, float4 *__restrict__ vel,
                const float4 *__restrict__ force, const int *__restrict__ id,
                const float4 *__restrict__ ref, float a, float dt, float c1, float c2,
                const unsigned *__restrict__ seed_step0, const int *__restrict__ steps_done, Raise rs) {
    const unsigned seed = seed_step0[0];
    const unsigned step = seed_step0[1] + (unsigned)*steps_done;      // stats[0]: steps finished in this call
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    bool moved = false;
    if (i < g.n) {
        float4 p = pos[i], v = vel[i];
        const float4 f = force[i];
        float gx = 0.0f, gy = 0.0f, gz = 0.0f, unused;
        if (c2 != 0.0f) {
            const unsigned key = (unsigned)(id ? id[i] : i);
            normal_pair(seed, step, key, 0u, gx, gy);
            if (DIM == 3) normal_pair(seed, step, key, 1u, gz, unused);
        }
        const float hdt = 0.5f * dt;
        v.x = fmaf(a, f.x, v.x); v.y = fmaf(a, f.y, v.y);
        float rx = fmaf(hdt, v.x, p.x), ry = fmaf(hdt, v.y, p.y);
        v.x = fmaf(c2, gx, c1 * v.x); v.y = fmaf(c2, gy, c1 * v.y);
        p.x = wrap(fmaf(hdt, v.x, rx), g.L[0], g.inv_L[0]);
        p.y = wrap(fmaf(hdt, v.y, ry), g.L[1], g.inv_L[1]);
        if (DIM == 3) {
            v.z = fmaf(a, f.z, v.z);
            const float rz = fmaf(hdt, v.z, p.z);
            v.z = fmaf(c2, gz, c1 * v.z);
            p.z = wrap(fmaf(hdt, v.z, rz), g.L[2], g.inv_L[2]);
        }
        pos[i] = p; vel[i] = v;
        moved = disp2_from_ref<DIM>(g, p, ref[i]) > g.half_skin2;
    }
    if (__any_sync(FULL, moved) && (threadIdx.x & 31) == 0) raise_rebuild(rs);
}

} // namespace mdk
