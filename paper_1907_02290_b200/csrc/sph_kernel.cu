// Short-range workload through the same index lists (paper P:79 "short-range
// interaction such as SPH ... treewalk but with cell-opening criterion different from the standard opening angle",
// P:109-111 particle records "much larger in the case of SPH", P:117 list reuse under a stability-limited step).
// Reading S23 of DESIGN.md: cubic-spline kernel with support 2h,
//     W(r,h) = 1/(4 pi h^3) [ (2-q)+^3 - 4 (1-q)+^3 ],   dW/dr = -3/(4 pi h^4) [ (2-q)+^2 - 4 (1-q)+^2 ],   q = r/h
//   k_sph_density:  rho_i = sum_k m_k W(|x_i - x_k|, h_i)   (gather, self term included);  P_i/rho_i^2 = (gamma-1) u_i / rho_i
//   k_sph_hydro:    a_i = - sum_k m_k (P_i/rho_i^2 + P_k/rho_k^2) 1/2 [gradW(r_ik,h_i) + gradW(r_ik,h_k)]
//
// Same mapping as the gravity kernel (force_kernel.cu): a warp owns a work item (2W i-particles of one group, two per
// lane, 32/W j-slices combined by shuffles), streams the group's index list in 64-entry tiles, gathers the j records
// into a warp-private shared-memory tile in pair layout and sweeps it with packed FP32.  The hydro kernel gathers TWO
// records per j (position/mass and the SPH record) and stages per j the values that do not depend on i
// (1/h_k and m_k/(pi h_k^4)), so the sweep pays for them once per tile instead of once per pair.
// Entries beyond 2h contribute exactly 0 through the clamps; padded list entries have m = 0.
#include "mwf_internal.h"

namespace mwf {

namespace {

constexpr float INV_PI = 0.318309886183790671538f;

__device__ __forceinline__ float rsqrt_approx(float x) {
    float r;
    asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x));
    return r;
}
__device__ __forceinline__ float sqrt_approx(float x) {
    float r;
    asm("sqrt.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x));
    return r;
}
__device__ __forceinline__ int2 ld_stream_int2(const int2* p) {
    int2 v;
    asm volatile("ld.global.nc.L1::no_allocate.v2.s32 {%0, %1}, [%2];" : "=r"(v.x), "=r"(v.y) : "l"(p));
    return v;
}
__device__ __forceinline__ float2 f2(float a) { return make_float2(a, a); }
// (c - s q)+ for both halves
__device__ __forceinline__ float2 clamp_lin(float c, float s, float2 q) {
    const float2 t = __ffma2_rn(q, f2(-s), f2(c));
    return make_float2(fmaxf(t.x, 0.f), fmaxf(t.y, 0.f));
}
// Both branches of the cubic spline in one branch-free polynomial of t2 = (2 - q)+ and a scaled (1 - q)+, arranged so that
// the last operation has only two distinct register operands (a three-operand FFMA2 costs 3 pipe cycles):
//   P = 2:  (2-q)+^2 - 4 (1-q)+^2 = t2^2 - u^2,      u = (2 - 2q)+            (exactly 2 (1-q)+)
//   P = 3:  (2-q)+^3 - 4 (1-q)+^3 = t2^3 - u^3,      u = (k - k q)+, k = 4^(1/3)
template <int P>
__device__ __forceinline__ float2 spline_poly(float2 q) {
    const float2 t2 = clamp_lin(2.f, 1.f, q);
    float2 a = __fmul2_rn(t2, t2);
    if constexpr (P == 2) {
        const float2 u = clamp_lin(2.f, 2.f, q);
        return __ffma2_rn(make_float2(-u.x, -u.y), u, a);
    } else {
        constexpr float K = 1.58740105196819947475f;
        const float2 u = clamp_lin(K, K, q);
        a = __fmul2_rn(a, t2);
        const float2 c = __fmul2_rn(u, u);
        return __ffma2_rn(make_float2(-c.x, -c.y), u, a);
    }
}

struct ItemSetup {
    int sl, il;
    int64_t l0;
    int n_tiles;
};

template <int W>
__device__ __forceinline__ ItemSetup setup(const SphArgs& a, const WorkItem& it, int lane) {
    ItemSetup s;
    s.sl = lane / W;
    s.il = lane % W;
    s.l0 = a.list_off[it.group];
    s.n_tiles = (int)((a.list_off[it.group + 1] - s.l0) / TILE_J);
    return s;
}

// ---------------------------------------------------------------- density
template <int W>
__device__ __forceinline__ void density_item(const SphArgs& a, const WorkItem it, float4* __restrict__ sbuf, int lane) {
    constexpr int S = 32 / W;
    const ItemSetup st = setup<W>(a, it, lane);
    const float4* __restrict__ J = a.store;
    float nx[2], ny[2], nz[2], hinv[2], ui[2];
    bool valid[2];
#pragma unroll
    for (int k = 0; k < 2; ++k) {
        const int off = st.il + W * k;
        valid[k] = off < it.n_i;
        const int64_t i = it.i_first + (valid[k] ? off : 0);
        const float4 p = __ldg(J + i);
        const float4 s = a.sph[i];
        nx[k] = -p.x; ny[k] = -p.y; nz[k] = -p.z;
        hinv[k] = 1.f / s.x;
        ui[k] = s.y;
    }
    float2 acc[2] = {f2(0.f), f2(0.f)}, part[2] = {f2(0.f), f2(0.f)};
    const int2* __restrict__ lst = reinterpret_cast<const int2*>(a.list + st.l0);
    int2 idn = make_int2(0, 0);
    float4 j0 = make_float4(0.f, 0.f, 0.f, 0.f), j1 = j0;
    if (st.n_tiles > 0) {
        const int2 id = ld_stream_int2(lst + lane);
        j0 = __ldg(J + id.x);
        j1 = __ldg(J + id.y);
        if (st.n_tiles > 1) idn = ld_stream_int2(lst + 32 + lane);
    }
    for (int t = 0; t < st.n_tiles; ++t) {
        float4* sA = sbuf + (t & 1) * TILE_J;
        float4* sB = sA + TILE_J / 2;
        sA[lane] = make_float4(j0.x, j1.x, j0.y, j1.y);
        sB[lane] = make_float4(j0.z, j1.z, j0.w, j1.w);
        __syncwarp();
        if (t + 1 < st.n_tiles) {
            j0 = __ldg(J + idn.x);
            j1 = __ldg(J + idn.y);
            if (t + 2 < st.n_tiles) idn = ld_stream_int2(lst + (int64_t)(t + 2) * 32 + lane);
        }
#pragma unroll 8
        for (int pp = 0; pp < W; ++pp) {
            const int p = pp * S + st.sl;
            const float4 A = sA[p];
            const float4 B = sB[p];
            const float2 jx = make_float2(A.x, A.y), jy = make_float2(A.z, A.w);
            const float2 jz = make_float2(B.x, B.y), jm = make_float2(B.z, B.w);
#pragma unroll
            for (int k = 0; k < 2; ++k) {
                const float2 dx = __fadd2_rn(jx, f2(nx[k]));
                const float2 dy = __fadd2_rn(jy, f2(ny[k]));
                const float2 dz = __fadd2_rn(jz, f2(nz[k]));
                float2 r2 = __fmul2_rn(dx, dx);
                r2 = __ffma2_rn(dy, dy, r2);
                r2 = __ffma2_rn(dz, dz, r2);
                const float2 r = make_float2(sqrt_approx(r2.x), sqrt_approx(r2.y));
                const float2 q = __fmul2_rn(r, f2(hinv[k]));
                part[k] = __ffma2_rn(jm, spline_poly<3>(q), part[k]);
            }
        }
        constexpr int FLUSH = S > 2 ? S : 2;
        if ((t & (FLUSH - 1)) == FLUSH - 1) {
#pragma unroll
            for (int k = 0; k < 2; ++k) { acc[k] = __fadd2_rn(acc[k], part[k]); part[k] = f2(0.f); }
        }
    }
#pragma unroll
    for (int k = 0; k < 2; ++k) {
        acc[k] = __fadd2_rn(acc[k], part[k]);
        float r = acc[k].x + acc[k].y;
#pragma unroll
        for (int m = W; m < 32; m <<= 1) r += __shfl_xor_sync(0xffffffffu, r, m);
        if (valid[k] && st.sl == 0) {
            const float rho = r * (0.25f * INV_PI) * hinv[k] * hinv[k] * hinv[k];
            float2* out = reinterpret_cast<float2*>(a.sph + it.i_first + st.il + W * k) + 1;  // fields (rho, P/rho^2)
            *out = make_float2(rho, a.gamma_m1 * ui[k] / rho);
        }
    }
    __syncwarp();
}

// ---------------------------------------------------------------- pressure-gradient acceleration
constexpr int HYDRO_TILE_F4 = 2 * TILE_J;  // per buffer: 32 pairs x (A, B, C, D) float4; D holds only 2 floats per pair

template <int W>
__device__ __forceinline__ void hydro_item(const SphArgs& a, const WorkItem it, float4* __restrict__ sbuf, int lane) {
    constexpr int S = 32 / W;
    const ItemSetup st = setup<W>(a, it, lane);
    const float4* __restrict__ J = a.store;
    const float4* __restrict__ Q = a.sph;
    const int32_t n_ptcl = (int32_t)a.n_ptcl;
    float nx[2], ny[2], nz[2], hinv[2], ki[2], pi[2];
    bool valid[2];
#pragma unroll
    for (int k = 0; k < 2; ++k) {
        const int off = st.il + W * k;
        valid[k] = off < it.n_i;
        const int64_t i = it.i_first + (valid[k] ? off : 0);
        const float4 p = __ldg(J + i);
        const float4 s = __ldg(Q + i);
        nx[k] = -p.x; ny[k] = -p.y; nz[k] = -p.z;
        hinv[k] = 1.f / s.x;
        const float h2 = hinv[k] * hinv[k];
        ki[k] = INV_PI * h2 * h2;   // 1 / (pi h_i^4)
        pi[k] = s.w;
    }
    float2 ax[2], ay[2], az[2], px[2], py[2], pz[2];
#pragma unroll
    for (int k = 0; k < 2; ++k) ax[k] = ay[k] = az[k] = px[k] = py[k] = pz[k] = f2(0.f);
    const int2* __restrict__ lst = reinterpret_cast<const int2*>(a.list + st.l0);
    int2 idn = make_int2(0, 0);
    const float4 none = make_float4(1.f, 0.f, 0.f, 0.f);
    float4 j0 = make_float4(0.f, 0.f, 0.f, 0.f), j1 = j0, s0 = none, s1 = none;
    if (st.n_tiles > 0) {
        const int2 id = ld_stream_int2(lst + lane);
        j0 = __ldg(J + id.x);
        j1 = __ldg(J + id.y);
        s0 = id.x < n_ptcl ? __ldg(Q + id.x) : none;   // padding entries point at the zero-mass dummy behind the SPJ
        s1 = id.y < n_ptcl ? __ldg(Q + id.y) : none;
        if (st.n_tiles > 1) idn = ld_stream_int2(lst + 32 + lane);
    }
    for (int t = 0; t < st.n_tiles; ++t) {
        float4* sA = sbuf + (t & 1) * HYDRO_TILE_F4;
        float4* sB = sA + TILE_J / 2;
        float4* sC = sB + TILE_J / 2;
        float2* sD = reinterpret_cast<float2*>(sC + TILE_J / 2);
        {
            const float g0 = 1.f / s0.x, g1 = 1.f / s1.x;
            const float g02 = g0 * g0, g12 = g1 * g1;
            sA[lane] = make_float4(j0.x, j1.x, j0.y, j1.y);
            sB[lane] = make_float4(j0.z, j1.z, j0.w, j1.w);
            sC[lane] = make_float4(g0, g1, j0.w * INV_PI * g02 * g02, j1.w * INV_PI * g12 * g12);  // 1/h_k, m_k/(pi h_k^4)
            sD[lane] = make_float2(s0.w, s1.w);                                                   // P_k/rho_k^2
        }
        __syncwarp();
        if (t + 1 < st.n_tiles) {
            j0 = __ldg(J + idn.x);
            j1 = __ldg(J + idn.y);
            s0 = idn.x < n_ptcl ? __ldg(Q + idn.x) : none;
            s1 = idn.y < n_ptcl ? __ldg(Q + idn.y) : none;
            if (t + 2 < st.n_tiles) idn = ld_stream_int2(lst + (int64_t)(t + 2) * 32 + lane);
        }
#pragma unroll 4
        for (int pp = 0; pp < W; ++pp) {
            const int p = pp * S + st.sl;
            const float4 A = sA[p];
            const float4 B = sB[p];
            const float4 C = sC[p];
            const float2 jp = sD[p];
            const float2 jx = make_float2(A.x, A.y), jy = make_float2(A.z, A.w);
            const float2 jz = make_float2(B.x, B.y), jm = make_float2(B.z, B.w);
            const float2 jh = make_float2(C.x, C.y), jk = make_float2(C.z, C.w);
#pragma unroll
            for (int k = 0; k < 2; ++k) {
                const float2 dx = __fadd2_rn(jx, f2(nx[k]));   // x_k - x_i
                const float2 dy = __fadd2_rn(jy, f2(ny[k]));
                const float2 dz = __fadd2_rn(jz, f2(nz[k]));
                float2 r2 = __ffma2_rn(dx, dx, f2(1e-30f));    // keeps 1/r finite at r = 0, where the polynomial is exactly 0
                r2 = __ffma2_rn(dy, dy, r2);
                r2 = __ffma2_rn(dz, dz, r2);
                const float2 ri = make_float2(rsqrt_approx(r2.x), rsqrt_approx(r2.y));
                const float2 r = __fmul2_rn(r2, ri);
                const float2 gi = spline_poly<2>(__fmul2_rn(r, f2(hinv[k])));
                const float2 gk = spline_poly<2>(__fmul2_rn(r, jh));
                float2 s = __fmul2_rn(__fmul2_rn(jm, f2(ki[k])), gi);   // m_k/(pi h_i^4) g(q_i)
                s = __ffma2_rn(jk, gk, s);                              //  + m_k/(pi h_k^4) g(q_k)
                const float2 f = __fmul2_rn(__fmul2_rn(s, __fadd2_rn(jp, f2(pi[k]))), ri);
                px[k] = __ffma2_rn(f, dx, px[k]);
                py[k] = __ffma2_rn(f, dy, py[k]);
                pz[k] = __ffma2_rn(f, dz, pz[k]);
            }
        }
        constexpr int FLUSH = S > 2 ? S : 2;
        if ((t & (FLUSH - 1)) == FLUSH - 1) {
#pragma unroll
            for (int k = 0; k < 2; ++k) {
                ax[k] = __fadd2_rn(ax[k], px[k]); ay[k] = __fadd2_rn(ay[k], py[k]); az[k] = __fadd2_rn(az[k], pz[k]);
                px[k] = py[k] = pz[k] = f2(0.f);
            }
        }
    }
#pragma unroll
    for (int k = 0; k < 2; ++k) {
        ax[k] = __fadd2_rn(ax[k], px[k]); ay[k] = __fadd2_rn(ay[k], py[k]); az[k] = __fadd2_rn(az[k], pz[k]);
        float rx = ax[k].x + ax[k].y, ry = ay[k].x + ay[k].y, rz = az[k].x + az[k].y;
#pragma unroll
        for (int m = W; m < 32; m <<= 1) {
            rx += __shfl_xor_sync(0xffffffffu, rx, m);
            ry += __shfl_xor_sync(0xffffffffu, ry, m);
            rz += __shfl_xor_sync(0xffffffffu, rz, m);
        }
        // a_i = -sum m_k (..) 1/2 dW/dr (x_i - x_k)/r with dW/dr = -3/(4 pi h^4) g(q):  = -3/8 sum [..] g (x_k - x_i)/r
        if (valid[k] && st.sl == 0) a.accp[it.i_first + st.il + W * k] = make_float4(-0.375f * rx, -0.375f * ry, -0.375f * rz, 0.f);
    }
    __syncwarp();
}

template <bool HYDRO>
__device__ __forceinline__ void sph_body(const SphArgs& a, float4* sbuf) {
    const int lane = threadIdx.x & 31;
    const int warp = threadIdx.x >> 5;
    int64_t w = (int64_t)blockIdx.x * WARPS_PER_CTA + warp;
    const int64_t n_warps = (int64_t)gridDim.x * WARPS_PER_CTA;
    while (w < a.n_items) {
        const int64_t pos = a.item_begin + w;
        const WorkItem it = a.items[a.order ? a.order[pos] : pos];
        if constexpr (HYDRO) {
            switch (it.width) {
                case 32: hydro_item<32>(a, it, sbuf, lane); break;
                case 16: hydro_item<16>(a, it, sbuf, lane); break;
                case 8: hydro_item<8>(a, it, sbuf, lane); break;
                case 4: hydro_item<4>(a, it, sbuf, lane); break;
                default: hydro_item<2>(a, it, sbuf, lane); break;
            }
        } else {
            switch (it.width) {
                case 32: density_item<32>(a, it, sbuf, lane); break;
                case 16: density_item<16>(a, it, sbuf, lane); break;
                case 8: density_item<8>(a, it, sbuf, lane); break;
                case 4: density_item<4>(a, it, sbuf, lane); break;
                default: density_item<2>(a, it, sbuf, lane); break;
            }
        }
        if (a.counter) {
            unsigned int nxt = 0;
            if (lane == 0) nxt = atomicAdd(a.counter, 1u);
            w = n_warps + (int64_t)__shfl_sync(0xffffffffu, nxt, 0);
        } else {
            w += n_warps;
        }
    }
}

}  // namespace

__global__ void __launch_bounds__(WARPS_PER_CTA * 32, 2) k_sph_density(const SphArgs a) {
    __shared__ float4 s_tiles[WARPS_PER_CTA][2 * TILE_J];
    sph_body<false>(a, s_tiles[threadIdx.x >> 5]);
}

__global__ void __launch_bounds__(WARPS_PER_CTA * 32, 2) k_sph_hydro(const SphArgs a) {
    __shared__ float4 s_tiles[WARPS_PER_CTA][2 * HYDRO_TILE_F4];
    sph_body<true>(a, s_tiles[threadIdx.x >> 5]);
}

cudaError_t launch_sph(const SphArgs& a, bool hydro, int grid, cudaStream_t s) {
    if (a.n_items <= 0 || grid <= 0) return cudaSuccess;
    if (hydro)
        k_sph_hydro<<<grid, WARPS_PER_CTA * 32, 0, s>>>(a);
    else
        k_sph_density<<<grid, WARPS_PER_CTA * 32, 0, s>>>(a);
    return cudaGetLastError();
}

int sph_max_ctas_per_sm(bool hydro) {
    int n = 0;
    const cudaError_t e = hydro ? cudaOccupancyMaxActiveBlocksPerMultiprocessor(&n, k_sph_hydro, WARPS_PER_CTA * 32, 0)
                                : cudaOccupancyMaxActiveBlocksPerMultiprocessor(&n, k_sph_density, WARPS_PER_CTA * 32, 0);
    return e == cudaSuccess ? n : 0;
}

}  // namespace mwf
