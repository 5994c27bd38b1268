// Kick-drift-kick leapfrog on the device store (paper section 7.3,
// once the lists are resident, the per-step transfers of particles and forces and the host
// integration (P:177 step 5) are what remains, so they move to the device too).
//
// HBM-bound, one thread per particle, 16-B vector accesses, grid-stride over a grid sized to the SM count:
//   k_kick_drift  reads accp, vel, store (48 B), writes vel, store (32 B)  -> 80 B / particle
//   k_kick        reads accp, vel (32 B), writes vel (16 B)                -> 48 B / particle
// The updates are single fp32 FMAs: v' = fma(a, dt/2, v), x' = fma(v', dt, x); mass and pot untouched.
#include "mwf_internal.h"

namespace mwf {

__global__ void __launch_bounds__(256) k_kick_drift(float4* __restrict__ store, float4* __restrict__ vel,
                                                    const float4* __restrict__ accp, int64_t n, float dt) {
    const float h = 0.5f * dt;
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) {
        const float4 a = __ldcs(accp + i);  // streamed: not needed again before the next force kernel rewrites it
        float4 v = vel[i];
        float4 x = store[i];
        v.x = fmaf(a.x, h, v.x);
        v.y = fmaf(a.y, h, v.y);
        v.z = fmaf(a.z, h, v.z);
        x.x = fmaf(v.x, dt, x.x);
        x.y = fmaf(v.y, dt, x.y);
        x.z = fmaf(v.z, dt, x.z);
        vel[i] = v;
        store[i] = x;
    }
}

__global__ void __launch_bounds__(256) k_kick(float4* __restrict__ vel, const float4* __restrict__ accp, int64_t n, float dt) {
    const float h = 0.5f * dt;
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) {
        const float4 a = accp[i];
        float4 v = vel[i];
        v.x = fmaf(a.x, h, v.x);
        v.y = fmaf(a.y, h, v.y);
        v.z = fmaf(a.z, h, v.z);
        vel[i] = v;
    }
}

static int grid_for(int64_t n) {
    const int64_t want = (n + 255) / 256;
    const int64_t cap = 148 * 8;  // 8 CTAs of 256 threads per SM keep HBM saturated
    return (int)(want < cap ? want : cap);
}

cudaError_t launch_kick_drift(float4* store, float4* vel, const float4* accp, int64_t n, float dt, cudaStream_t s) {
    if (n <= 0) return cudaSuccess;
    k_kick_drift<<<grid_for(n), 256, 0, s>>>(store, vel, accp, n, dt);
    return cudaGetLastError();
}

cudaError_t launch_kick(float4* vel, const float4* accp, int64_t n, float dt, cudaStream_t s) {
    if (n <= 0) return cudaSuccess;
    k_kick<<<grid_for(n), 256, 0, s>>>(vel, accp, n, dt);
    return cudaGetLastError();
}

}  // namespace mwf
