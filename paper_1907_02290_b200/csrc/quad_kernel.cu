// Quadrupole correction of the SPJ entries (the paper speaks of "multipole moments",
// P:160, and measures the monopole case).  Reading S22 of DESIGN.md: an SPJ entry acts through the
// second-order Taylor expansion of the softened kernel about the cell's centre of mass X, with
// Q = sum m (x - X)(x - X)^T, R = X - x_i, s^2 = |R|^2 + eps^2:
//     pot_i -= G [ M/s - tr(Q)/(2 s^3) + 3 (R.Q.R)/(2 s^5) ]
//     acc_i += G [ M R/s^3 - 3 tr(Q) R/(2 s^5) - 3 (Q R)/s^5 + 15 (R.Q.R) R/(2 s^7) ]
// The monopole terms are what k_force already evaluates for every list entry; this kernel runs behind it on the same
// stream and ADDS the Q terms for the SPJ part of every group's list (entries n_epj .. n_epj + n_spj of the merged
// list), so the monopole kernel and its lists stay exactly as they are.
//
// Mapping: the same work items, schedule and warp layout as k_force (one warp per item, two i-particles per lane held
// negated in registers, 32 / W j-slices combined by shuffles).  Per 64-entry tile every lane gathers two cells: the
// float4 (X, M) record of the store and the two float4 of the cell's quadrupole record (Qxx Qyy Qzz Qxy | Qxz Qyz
// tr(Q)/2 0), and writes them to a warp-private shared-memory tile in pair layout (five float4 per j-pair), so the
// sweep is packed FP32 (two j per instruction): 36 packed operations + 2 MUFU.RSQ per i per j-pair = 60 flop per
// correction with the paper's counting (FMA = 2, rsqrt = 4).
#include "mwf_internal.h"

namespace mwf {

namespace {

__device__ __forceinline__ float rsqrt_approx_q(float x) {
    float r;
    asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x));
    return r;
}

constexpr int QT = 5;  // float4 per j-pair in the tile

struct QAcc {
    float2 x[2], y[2], z[2], p[2];
};

template <int W>
__device__ __forceinline__ void quad_sweep(const float4* __restrict__ tile, int sl, const float (&nx)[2], const float (&ny)[2],
                                           const float (&nz)[2], float eps2, QAcc& t) {
    constexpr int S = 32 / W;
    const float2 e2 = make_float2(eps2, eps2);
    const float2 m15 = make_float2(-1.5f, -1.5f), p75 = make_float2(7.5f, 7.5f), m3 = make_float2(-3.f, -3.f);
    constexpr int UNROLL = W < 4 ? W : 4;
#pragma unroll UNROLL
    for (int pp = 0; pp < W; ++pp) {
        const int p = pp * S + sl;
        const float4 A = tile[p], B = tile[32 + p], C = tile[64 + p], D = tile[96 + p], E = tile[128 + p];
        const float2 jx = make_float2(A.x, A.y), jy = make_float2(A.z, A.w), jz = make_float2(B.x, B.y), h = make_float2(B.z, B.w);
        const float2 qxx = make_float2(C.x, C.y), qyy = make_float2(C.z, C.w), qzz = make_float2(D.x, D.y), qxy = make_float2(D.z, D.w);
        const float2 qxz = make_float2(E.x, E.y), qyz = make_float2(E.z, E.w);
#pragma unroll
        for (int k = 0; k < 2; ++k) {
            const float2 dx = __fadd2_rn(jx, make_float2(nx[k], nx[k]));
            const float2 dy = __fadd2_rn(jy, make_float2(ny[k], ny[k]));
            const float2 dz = __fadd2_rn(jz, make_float2(nz[k], nz[k]));
            float2 r2 = __ffma2_rn(dx, dx, e2);
            r2 = __ffma2_rn(dy, dy, r2);
            r2 = __ffma2_rn(dz, dz, r2);
            float2 ri;
            ri.x = rsqrt_approx_q(r2.x);
            ri.y = rsqrt_approx_q(r2.y);
            const float2 ri2 = __fmul2_rn(ri, ri);
            const float2 ri3 = __fmul2_rn(ri2, ri);
            const float2 ri5 = __fmul2_rn(ri3, ri2);
            const float2 ri7 = __fmul2_rn(ri5, ri2);
            float2 Qx = __fmul2_rn(qxx, dx);
            Qx = __ffma2_rn(qxy, dy, Qx);
            Qx = __ffma2_rn(qxz, dz, Qx);
            float2 Qy = __fmul2_rn(qxy, dx);
            Qy = __ffma2_rn(qyy, dy, Qy);
            Qy = __ffma2_rn(qyz, dz, Qy);
            float2 Qz = __fmul2_rn(qxz, dx);
            Qz = __ffma2_rn(qyz, dy, Qz);
            Qz = __ffma2_rn(qzz, dz, Qz);
            float2 dQd = __fmul2_rn(dx, Qx);
            dQd = __ffma2_rn(dy, Qy, dQd);
            dQd = __ffma2_rn(dz, Qz, dQd);
            // potential sum: tr(Q)/(2 s^3) - 3 dQd/(2 s^5)
            t.p[k] = __ffma2_rn(h, ri3, t.p[k]);
            const float2 u = __fmul2_rn(dQd, ri5);
            t.p[k] = __ffma2_rn(m15, u, t.p[k]);
            // acceleration: c1 d + c2 Qd, c1 = -3 tr/(2 s^5) + 15 dQd/(2 s^7), c2 = -3/s^5
            const float2 v = __fmul2_rn(h, ri5);
            const float2 w = __fmul2_rn(dQd, ri7);
            float2 c1 = __fmul2_rn(m3, v);
            c1 = __ffma2_rn(p75, w, c1);
            const float2 c2 = __fmul2_rn(m3, ri5);
            t.x[k] = __ffma2_rn(c1, dx, t.x[k]);
            t.y[k] = __ffma2_rn(c1, dy, t.y[k]);
            t.z[k] = __ffma2_rn(c1, dz, t.z[k]);
            t.x[k] = __ffma2_rn(c2, Qx, t.x[k]);
            t.y[k] = __ffma2_rn(c2, Qy, t.y[k]);
            t.z[k] = __ffma2_rn(c2, Qz, t.z[k]);
        }
    }
}

struct CellRec {
    float4 xm, q0, q1;
};

// SPJ entry e of a group: the first n_far of them sit behind the EPJ entries in run 1 (lst_far), the others in run 2 (lst_near)
__device__ __forceinline__ CellRec ld_cell(const QuadArgs& a, const int32_t* __restrict__ lst_far, const int32_t* __restrict__ lst_near, int64_t n_far,
                                           int64_t e, int64_t n_spj) {
    CellRec r;
    r.xm = r.q0 = r.q1 = make_float4(0.f, 0.f, 0.f, 0.f);  // past the end: a cell without moments
    if (e < n_spj) {
        const int32_t id = __ldg(e < n_far ? lst_far + e : lst_near + (e - n_far));  // index into the store: n_ptcl + cell
        r.xm = __ldg(a.store + id);
        const float4* q = a.quad + 2 * (int64_t)(id - a.n_ptcl);
        r.q0 = __ldg(q);
        r.q1 = __ldg(q + 1);
    }
    return r;
}

template <int W>
__device__ __forceinline__ void quad_item(const QuadArgs& a, const WorkItem it, float4* __restrict__ sbuf, int lane) {
    const int sl = lane / W;
    const int il = lane % W;
    const int64_t n_spj = a.spj_off[it.group + 1] - a.spj_off[it.group];
    if (n_spj == 0) return;
    const int64_t n_epj = a.epj_off[it.group + 1] - a.epj_off[it.group], n_far = a.n_far[it.group];
    const int32_t* __restrict__ lst_far = a.list + a.list_off[it.group] + n_epj;
    const int32_t* __restrict__ lst_near = a.list + a.list_off[it.group] + (n_epj + n_far + TILE_J - 1) / TILE_J * TILE_J;
    float nx[2], ny[2], nz[2];
    bool valid[2];
#pragma unroll
    for (int k = 0; k < 2; ++k) {
        const int off = il + W * k;
        valid[k] = off < it.n_i;
        const float4 p = __ldg(a.store + it.i_first + (valid[k] ? off : 0));
        nx[k] = -p.x; ny[k] = -p.y; nz[k] = -p.z;
    }
    QAcc acc;
#pragma unroll
    for (int k = 0; k < 2; ++k) acc.x[k] = acc.y[k] = acc.z[k] = acc.p[k] = make_float2(0.f, 0.f);
    const int n_tiles = (int)((n_spj + TILE_J - 1) / TILE_J);
    CellRec c0 = ld_cell(a, lst_far, lst_near, n_far, 2 * lane, n_spj), c1 = ld_cell(a, lst_far, lst_near, n_far, 2 * lane + 1, n_spj);
    for (int t = 0; t < n_tiles; ++t) {
        float4* tile = sbuf + (t & 1) * (QT * 32);
        tile[lane] = make_float4(c0.xm.x, c1.xm.x, c0.xm.y, c1.xm.y);
        tile[32 + lane] = make_float4(c0.xm.z, c1.xm.z, c0.q1.z, c1.q1.z);
        tile[64 + lane] = make_float4(c0.q0.x, c1.q0.x, c0.q0.y, c1.q0.y);
        tile[96 + lane] = make_float4(c0.q0.z, c1.q0.z, c0.q0.w, c1.q0.w);
        tile[128 + lane] = make_float4(c0.q1.x, c1.q1.x, c0.q1.y, c1.q1.y);
        __syncwarp();
        if (t + 1 < n_tiles) {
            const int64_t e = (int64_t)(t + 1) * TILE_J + 2 * lane;
            c0 = ld_cell(a, lst_far, lst_near, n_far, e, n_spj);
            c1 = ld_cell(a, lst_far, lst_near, n_far, e + 1, n_spj);
        }
        quad_sweep<W>(tile, sl, nx, ny, nz, a.eps2, acc);
    }
#pragma unroll
    for (int k = 0; k < 2; ++k) {
        float rx = acc.x[k].x + acc.x[k].y, ry = acc.y[k].x + acc.y[k].y, rz = acc.z[k].x + acc.z[k].y, rp = acc.p[k].x + acc.p[k].y;
#pragma unroll
        for (int m = W; m < 32; m <<= 1) {
            rx += __shfl_xor_sync(0xffffffffu, rx, m);
            ry += __shfl_xor_sync(0xffffffffu, ry, m);
            rz += __shfl_xor_sync(0xffffffffu, rz, m);
            rp += __shfl_xor_sync(0xffffffffu, rp, m);
        }
        if (valid[k] && sl == 0) {
            float4* dst = a.accp + it.i_first + il + W * k;
            float4 f = *dst;  // written by k_force earlier on this stream
            f.x += a.G * rx; f.y += a.G * ry; f.z += a.G * rz; f.w += a.G * rp;
            *dst = f;
        }
    }
    __syncwarp();  // the next item reuses the warp's tile buffers
}

}  // namespace

__global__ void __launch_bounds__(WARPS_PER_CTA * 32, 2) k_quad(const QuadArgs a) {
    __shared__ float4 s_tiles[WARPS_PER_CTA][2 * QT * 32];
    const int lane = threadIdx.x & 31;
    const int warp = threadIdx.x >> 5;
    float4* sbuf = s_tiles[warp];
    int64_t w = (int64_t)blockIdx.x * WARPS_PER_CTA + warp;
    const int64_t n_warps = (int64_t)gridDim.x * WARPS_PER_CTA;
    while (w < a.n_items) {
        const int64_t pos = a.item_begin + w;
        const WorkItem it = a.items[a.order ? a.order[pos] : pos];
        switch (it.width) {
            case 32: quad_item<32>(a, it, sbuf, lane); break;
            case 16: quad_item<16>(a, it, sbuf, lane); break;
            case 8: quad_item<8>(a, it, sbuf, lane); break;
            case 4: quad_item<4>(a, it, sbuf, lane); break;
            default: quad_item<2>(a, it, sbuf, lane); break;
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

cudaError_t launch_quad(const QuadArgs& a, int grid, cudaStream_t s) {
    if (a.n_items <= 0 || grid <= 0) return cudaSuccess;
    k_quad<<<grid, WARPS_PER_CTA * 32, 0, s>>>(a);
    return cudaGetLastError();
}

int quad_max_ctas_per_sm() {
    int n = 0;
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&n, k_quad, WARPS_PER_CTA * 32, 0) != cudaSuccess) return 0;
    return n;
}

}  // namespace mwf
