// Index-based multi-walk force kernel for sm_100a (paper: ForceKernelIndex,
// P:557-569; multiwalk P:89; indirect addressing P:107).
//
// Mapping:
//   * work item = 2W consecutive i-particles of one group (W = 32, 16, 8, 4 or 2) x the group's whole merged
//     list; one WARP owns an item from start to end, so there is no block-level barrier and no atomics on
//     the results.  Every lane holds TWO i-particles in registers (i = il and il + W, il = lane % W); the
//     warp is split into S = 32 / W j-slices that share those i-particles and take every S-th j-pair
//     (the north_star's "warp shuffles for splitting"); the slices' partial sums are combined by
//     __shfl_xor at the end.  A group of n_i particles is cut on the host into 64-particle items plus
//     power-of-two pieces, so that lanes are never padded by more than a few particles per group.
//   * the warp streams the list in tiles of 64 entries: each lane reads two 4-byte indices (one coalesced
//     256-B request per warp), gathers the two float4 (x,y,z,m) records through them and writes them to a
//     warp-private shared-memory tile in PAIR layout [x0 x1 y0 y1][z0 z1 m0 m1]; the gathers of tile t+1
//     and the indices of tile t+2 are in flight while tile t is swept.
//   * every lane sweeps its slice of the tile with broadcast LDS.128 and packed FP32 math (FADD2 / FMUL2 /
//     FFMA2 of sm_100: two j per instruction): 13 packed FP32 ops + 2 MUFU.RSQ per i per j-pair, which is
//     exactly the paper's 23-flop interaction (3 sub, 3 fma, rsqrt, 3 mul, 3 fma, 1 add).
//   * accumulation is two-level: partial sums over 32 j-pairs are added into running totals (two
//     independent sums per component from the j-pairing), which keeps the fp32 summation error far inside
//     the tolerance.
//   * two coordinate conventions (reading S11b of DESIGN.md).  The tiles of a list's run 1 -- every EPJ entry and every
//     FAR SPJ entry -- are swept in the caller's coordinates: particle positions are exact fp32 inputs and
//     d = fl(x_j - x_i) is good to half an ulp of the DIFFERENCE however small it is; a cell at least 1/32 of its
//     own coordinates away from the group (SPJ_FAR_KAPPA) is placed well enough by its fp32 record.  The tiles of run 2,
//     the NEAR SPJ entries, are swept in item-centred coordinates, c = the item's first i-particle: a centre of mass is
//     not an fp32 input -- on the fp32 grid it is up to 2^-25 |X| off, which for a cell 1e-3 away at coordinates of
//     order 1 is the north_star's whole error budget -- so the refresh keeps its rounding remainder (spj_lo) and the
//     staged position (hi - c) + lo carries 24 bits of the DISTANCE to the item; the i-side switches by adding c to -x_i.
//     The two runs of a group's list are padded to whole tiles separately and swept by a tile loop each (run_item).
//   * order 2 (k_force_quad, reading S22): from a list's first SPJ entry on the tiles also carry the cells' quadrupoles, and the
//     sweep evaluates the Q terms from the monopole interaction's own distances and rsqrt.
//   * the self term (an i-particle meets itself in its own EPJ list) contributes exactly 0 to acc and
//     m_i * rsqrt(eps^2) to the potential sum; the same value is subtracted up front (reading S2).
#include "mwf_internal.h"

namespace mwf {

__device__ __forceinline__ float rsqrt_approx(float x) {
    float r;
    asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x));
    return r;
}

__device__ __forceinline__ int2 ld_stream_int2(const int2* p) {
    int2 v;
    asm volatile("ld.global.nc.L1::no_allocate.v2.s32 {%0, %1}, [%2];" : "=r"(v.x), "=r"(v.y) : "l"(p));
    return v;
}

// 16-byte asynchronous copy global -> shared (LDGSTS), through L1 like the plain gathers
__device__ __forceinline__ void cp_async16(float4* smem, const float4* gmem) {
    asm volatile("cp.async.ca.shared.global [%0], [%1], 16;" ::"r"((unsigned)__cvta_generic_to_shared(smem)), "l"(gmem) : "memory");
}
// the same with src_bytes (0 or 16) read and the rest of the 16 bytes zero-filled
__device__ __forceinline__ void cp_async16_zfill(float4* smem, const float4* gmem, int src_bytes) {
    asm volatile("cp.async.ca.shared.global [%0], [%1], 16, %2;" ::"r"((unsigned)__cvta_generic_to_shared(smem)), "l"(gmem), "r"(src_bytes) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_all;" ::: "memory"); }

struct Acc2 {  // sums for the two i-particles of a lane; .x / .y halves are the two j of a pair
    float2 x[2], y[2], z[2], p[2];
};

__device__ __forceinline__ void zero(Acc2& a) {
#pragma unroll
    for (int k = 0; k < 2; ++k) a.x[k] = a.y[k] = a.z[k] = a.p[k] = make_float2(0.f, 0.f);
}

__device__ __forceinline__ void add_into(Acc2& a, const Acc2& t) {
#pragma unroll
    for (int k = 0; k < 2; ++k) {
        a.x[k] = __fadd2_rn(a.x[k], t.x[k]);
        a.y[k] = __fadd2_rn(a.y[k], t.y[k]);
        a.z[k] = __fadd2_rn(a.z[k], t.z[k]);
        a.p[k] = __fadd2_rn(a.p[k], t.p[k]);
    }
}

// Sweep one staged tile: the lane belongs to slice `sl` of S and takes pairs sl, sl + S, ... (W = 32 / S of them).
template <int W, int UNROLL_CAP = MWF_UNROLL_WIDE>
__device__ __forceinline__ void sweep_tile(const float4* __restrict__ sA, const float4* __restrict__ sB, int sl,
                                           const float (&nx)[2], const float (&ny)[2], const float (&nz)[2], float eps2, Acc2& t) {
    constexpr int S = 32 / W;
    const float2 e2 = make_float2(eps2, eps2);
    constexpr int UNROLL = W < UNROLL_CAP ? W : UNROLL_CAP;
#pragma unroll UNROLL
    for (int pp = 0; pp < W; ++pp) {
        const int p = pp * S + sl;
        const float4 A = sA[p];
        const float4 B = sB[p];
        const float2 jx = make_float2(A.x, A.y), jy = make_float2(A.z, A.w);
        const float2 jz = make_float2(B.x, B.y), jm = make_float2(B.z, B.w);
#pragma unroll
        for (int k = 0; k < 2; ++k) {
            const float2 dx = __fadd2_rn(jx, make_float2(nx[k], nx[k]));
            const float2 dy = __fadd2_rn(jy, make_float2(ny[k], ny[k]));
            const float2 dz = __fadd2_rn(jz, make_float2(nz[k], nz[k]));
            float2 r2 = __ffma2_rn(dx, dx, e2);
            r2 = __ffma2_rn(dy, dy, r2);
            r2 = __ffma2_rn(dz, dz, r2);
            float2 ri;
            ri.x = rsqrt_approx(r2.x);
            ri.y = rsqrt_approx(r2.y);
            const float2 mr = __fmul2_rn(jm, ri);
            t.p[k] = __fadd2_rn(t.p[k], mr);
            const float2 ri2 = __fmul2_rn(ri, ri);
            const float2 mr3 = __fmul2_rn(mr, ri2);
            t.x[k] = __ffma2_rn(mr3, dx, t.x[k]);
            t.y[k] = __ffma2_rn(mr3, dy, t.y[k]);
            t.z[k] = __ffma2_rn(mr3, dz, t.z[k]);
        }
    }
}

// Entries (2 * lane, 2 * lane + 1) of tile t of a DATA list (method G1: the list carries the records themselves);
// entries past the end of the list read as a zero-mass record at the origin.
__device__ __forceinline__ void ld_data_pair(const float4* __restrict__ jd, int64_t n_list, int t, int lane, float4& j0, float4& j1) {
    const int64_t e = (int64_t)t * TILE_J + 2 * lane;
    const float4 zero = make_float4(0.f, 0.f, 0.f, 0.f);
    j0 = e < n_list ? __ldg(jd + e) : zero;
    j1 = e + 1 < n_list ? __ldg(jd + e + 1) : zero;
}

// per warp: two tiles in pair layout, the remainders of the near tile in flight
constexpr int FORCE_SMEM_FLOAT4_PER_WARP = 2 * TILE_J + TILE_J;

#ifndef MWF_NEAR_UNROLL
#define MWF_NEAR_UNROLL 4
#endif
#ifndef MWF_QUAD_UNROLL
#define MWF_QUAD_UNROLL 4
#endif

// The lane's two i-particles (negated positions), the running totals started at minus the self term (slice 0 only:
// the slices are added later).
template <int W>
__device__ __forceinline__ void item_begin(const ForceArgs& a, const WorkItem& it, int lane, float (&nx)[2], float (&ny)[2], float (&nz)[2],
                                           bool (&valid)[2], Acc2& acc) {
    const int sl = lane / W, il = lane % W;
    const float self_rinv = rsqrt_approx(a.eps2);  // what the sweep computes for d = 0
    const bool self_in = a.grp_self[it.group] != 0;
    zero(acc);
#pragma unroll
    for (int k = 0; k < 2; ++k) {
        const int off = il + W * k;
        valid[k] = off < it.n_i;
        const float4 p = __ldg(a.store + it.i_first + (valid[k] ? off : 0));
        nx[k] = -p.x; ny[k] = -p.y; nz[k] = -p.z;
        acc.p[k].x = (self_in && sl == 0) ? -p.w * self_rinv : 0.f;
    }
}

// Slices combined by shuffles; slice 0 writes (ax, ay, az, pot) and, in the device-resident step, the closing kick.
template <int W>
__device__ __forceinline__ void item_end(const ForceArgs& a, const WorkItem& it, int lane, const bool (&valid)[2], const Acc2& acc) {
    const int sl = lane / W, il = lane % W;
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
            const int64_t i = it.i_first + il + W * k;
            const float4 r = make_float4(a.G * rx, a.G * ry, a.G * rz, -a.G * rp);
            a.accp[i] = r;
            if (a.vel) {  // device-resident step: the closing kick of the leapfrog, the arithmetic of k_kick bit for bit
                float4 v = a.vel[i];
                v.x = fmaf(r.x, a.kick_h, v.x); v.y = fmaf(r.y, a.kick_h, v.y); v.z = fmaf(r.z, a.kick_h, v.z);
                a.vel[i] = v;
            }
        }
    }
    __syncwarp();  // the next item reuses the warp's tile buffers
}

// every partial sum covers 32 j-pairs per lane whatever the slice count (MWF_FLUSH_MIN tiles at least)
template <int W>
__device__ __forceinline__ void flush_partial(int t, Acc2& acc, Acc2& part) {
    constexpr int S = 32 / W;
    constexpr int FLUSH = S > MWF_FLUSH_MIN ? S : MWF_FLUSH_MIN;
    if ((t & (FLUSH - 1)) == FLUSH - 1) {
        add_into(acc, part);
        zero(part);
    }
}

// Index lists (method G2, the hot path), one tile loop per run.  Loop 1 (run 1: EPJ and far SPJ entries, caller's
// coordinates) knows nothing of run 2: its staging is a plain transpose of the two gathered records.  The remainders of the
// FIRST tile of run 2 are requested (cp.async) in the item's prologue, so that they arrive behind loop 1; between the
// loops the i-side moves to item-centred coordinates; loop 2 stages (x - c) + q with the remainders of tile t + 1 under
// way during the sweep of tile t.  One loop with both stagings costs 5 % on the tiles of run 1, whether a list has a run 2
// or not (profiles/r02_kforce_variants.md); the sweep of loop 2 is unrolled less (MWF_NEAR_UNROLL) to keep the kernel small.
template <int W>
__device__ __forceinline__ void run_item(const ForceArgs& a, const WorkItem it, float4* __restrict__ sbuf, int lane) {
    const int sl = lane / W;
    const float4* __restrict__ J = a.store;
    float4* lo_raw = sbuf + 2 * TILE_J;
    const float4* __restrict__ LO = a.spj_lo - a.n_ptcl;  // SPJ entries are cell index + N

    const int64_t l0 = a.list_off[it.group];
    const int n_tiles = (int)((a.list_off[it.group + 1] - l0) / TILE_J);
    // tiles [0, te): run 1 (EPJ and far SPJ entries), [te, n_tiles): run 2 (near SPJ entries)
    const int te = (a.run1_len[it.group] + TILE_J - 1) / TILE_J;
    const int2* __restrict__ lst = reinterpret_cast<const int2*>(a.list + l0);

    int2 idn = make_int2(0, 0);
    float4 j0 = make_float4(0.f, 0.f, 0.f, 0.f), j1 = j0;
    if (n_tiles > 0) {
        const int2 id = ld_stream_int2(lst + lane);
        if (te < n_tiles) {  // remainders of the first near tile: under way while run 1 is swept
            const int2 ide = te == 0 ? id : ld_stream_int2(lst + (int64_t)te * 32 + lane);
            cp_async16(lo_raw + lane, LO + ide.x);
            cp_async16(lo_raw + 32 + lane, LO + ide.y);
            cp_async_commit();
        }
        j0 = __ldg(J + id.x);
        j1 = __ldg(J + id.y);
        if (n_tiles > 1) idn = ld_stream_int2(lst + 32 + lane);
    }

    float nx[2], ny[2], nz[2];
    bool valid[2];
    Acc2 acc, part;
    item_begin<W>(a, it, lane, nx, ny, nz, valid, acc);
    zero(part);

    int t = 0;
    for (; t < te; ++t) {
        float4* sA = sbuf + (t & 1) * TILE_J;
        float4* sB = sA + TILE_J / 2;
        sA[lane] = make_float4(j0.x, j1.x, j0.y, j1.y);
        sB[lane] = make_float4(j0.z, j1.z, j0.w, j1.w);
        __syncwarp();
        if (t + 1 < n_tiles) {
            j0 = __ldg(J + idn.x);
            j1 = __ldg(J + idn.y);
            if (t + 2 < n_tiles) idn = ld_stream_int2(lst + (int64_t)(t + 2) * 32 + lane);
        }
        sweep_tile<W>(sA, sB, sl, nx, ny, nz, a.eps2, part);
        flush_partial<W>(t, acc, part);
    }
    if (t < n_tiles) {
        const float4 c = __ldg(J + it.i_first);  // from here on: item-centred
#pragma unroll
        for (int k = 0; k < 2; ++k) { nx[k] += c.x; ny[k] += c.y; nz[k] += c.z; }
        for (; t < n_tiles; ++t) {
            float4* sA = sbuf + (t & 1) * TILE_J;
            float4* sB = sA + TILE_J / 2;
            cp_async_wait_all();  // the lane's own two remainders
            const float4 q0 = lo_raw[lane], q1 = lo_raw[32 + lane];
            sA[lane] = make_float4((j0.x - c.x) + q0.x, (j1.x - c.x) + q1.x, (j0.y - c.y) + q0.y, (j1.y - c.y) + q1.y);
            sB[lane] = make_float4((j0.z - c.z) + q0.z, (j1.z - c.z) + q1.z, j0.w, j1.w);
            __syncwarp();
            if (t + 1 < n_tiles) {
                j0 = __ldg(J + idn.x);
                j1 = __ldg(J + idn.y);
                cp_async16(lo_raw + lane, LO + idn.x);
                cp_async16(lo_raw + 32 + lane, LO + idn.y);
                cp_async_commit();
                if (t + 2 < n_tiles) idn = ld_stream_int2(lst + (int64_t)(t + 2) * 32 + lane);
            }
            sweep_tile<W, MWF_NEAR_UNROLL>(sA, sB, sl, nx, ny, nz, a.eps2, part);
            flush_partial<W>(t, acc, part);
        }
    }
    add_into(acc, part);
    item_end<W>(a, it, lane, valid, acc);
}

// Data lists (method G1 of the paper, A/B variant): the group's list is a contiguous run of j RECORDS sent with the
// dispatch; same items, same sweep, one coordinate convention (the records are all fp32).
template <int W>
__device__ __forceinline__ void run_item_data(const ForceArgs& a, const WorkItem it, float4* __restrict__ sbuf, int lane) {
    const int sl = lane / W;
    const int64_t l0 = a.joff[it.group - a.g_base];
    const int64_t n_list = a.joff[it.group - a.g_base + 1] - l0;
    const int n_tiles = (int)((n_list + TILE_J - 1) / TILE_J);
    const float4* __restrict__ jd = a.jdata + l0;
    float4 j0 = make_float4(0.f, 0.f, 0.f, 0.f), j1 = j0;
    if (n_tiles > 0) ld_data_pair(jd, n_list, 0, lane, j0, j1);

    float nx[2], ny[2], nz[2];
    bool valid[2];
    Acc2 acc, part;
    item_begin<W>(a, it, lane, nx, ny, nz, valid, acc);
    zero(part);
    for (int t = 0; t < n_tiles; ++t) {
        float4* sA = sbuf + (t & 1) * TILE_J;
        float4* sB = sA + TILE_J / 2;
        sA[lane] = make_float4(j0.x, j1.x, j0.y, j1.y);
        sB[lane] = make_float4(j0.z, j1.z, j0.w, j1.w);
        __syncwarp();
        if (t + 1 < n_tiles) ld_data_pair(jd, n_list, t + 1, lane, j0, j1);
        sweep_tile<W>(sA, sB, sl, nx, ny, nz, a.eps2, part);
        flush_partial<W>(t, acc, part);
    }
    add_into(acc, part);
    item_end<W>(a, it, lane, valid, acc);
}

// ---- order 2 (NEXT-3, reading S22): the quadrupole terms of the SPJ entries in the same sweep ---------------------------
// A quad tile carries, per j-pair, the two tile rows of the monopole sweep and Q of the two cells: [qxx qyy] [qzz qxy]
// [qxz qyz] and -tr(Q)/2 (zero for particles and padding).  With R = X - x_i, s^2 = |R|^2 + eps^2 (include/mwf.h):
//     potential sum  += m/s - (tr/2)/s^3 + (3/2) (R.Q.R)/s^5
//     acceleration   += [ m/s^3 - 3 (tr/2)/s^5 + (15/2) (R.Q.R)/s^7 ] R - 3 (Q R)/s^5
// 40 packed FP32 operations + 2 MUFU per i per j-pair; distances, r^2, rsqrt and the gathers are those of the monopole
// interaction and are not done twice (a separate correction kernel behind k_force cost 36 + 13 operations and a second
// pass over the lists).
constexpr int QUAD_TILE_FLOAT4 = 5 * 32 + 16;                                    // five rows of 32 pairs + 32 float2
#ifndef MWF_QUAD_ASYNC
#define MWF_QUAD_ASYNC 1
#endif
// + remainders of the near tile in flight + (MWF_QUAD_ASYNC) the Q records of the tile in flight, as gathered
constexpr int QUAD_SMEM_FLOAT4_PER_WARP = 2 * QUAD_TILE_FLOAT4 + TILE_J + (MWF_QUAD_ASYNC ? 2 * TILE_J : 0);

template <int W>
__device__ __forceinline__ void sweep_tile_quad(const float4* __restrict__ T, int sl, const float (&nx)[2], const float (&ny)[2],
                                                const float (&nz)[2], float eps2, Acc2& t) {
    constexpr int S = 32 / W;
    const float2 e2 = make_float2(eps2, eps2);
    const float2 p15 = make_float2(1.5f, 1.5f), p75 = make_float2(7.5f, 7.5f), p3 = make_float2(3.f, 3.f), m3 = make_float2(-3.f, -3.f);
    const float2* __restrict__ H = reinterpret_cast<const float2*>(T + 160);
    constexpr int UNROLL = W < MWF_QUAD_UNROLL ? W : MWF_QUAD_UNROLL;
#pragma unroll UNROLL
    for (int pp = 0; pp < W; ++pp) {
        const int p = pp * S + sl;
        const float4 A = T[p], B = T[32 + p], C = T[64 + p], D = T[96 + p], E = T[128 + p];
        const float2 nh = H[p];
        const float2 jx = make_float2(A.x, A.y), jy = make_float2(A.z, A.w), jz = make_float2(B.x, B.y), jm = make_float2(B.z, B.w);
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
            ri.x = rsqrt_approx(r2.x);
            ri.y = rsqrt_approx(r2.y);
            const float2 mr = __fmul2_rn(jm, ri);
            const float2 ri2 = __fmul2_rn(ri, ri);
            const float2 mr3 = __fmul2_rn(mr, ri2);
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
            t.p[k] = __fadd2_rn(t.p[k], mr);
            t.p[k] = __ffma2_rn(nh, ri3, t.p[k]);
            const float2 u = __fmul2_rn(dQd, ri5);
            t.p[k] = __ffma2_rn(p15, u, t.p[k]);
            const float2 v = __fmul2_rn(nh, ri5);
            float2 c1 = __ffma2_rn(p3, v, mr3);
            const float2 w = __fmul2_rn(dQd, ri7);
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

struct QuadRec {
    float4 a, b;  // (Qxx Qyy Qzz Qxy) (Qxz Qyz tr/2 0)
};

template <int W>
__device__ __forceinline__ void run_item_quad(const ForceArgs& a, const WorkItem it, float4* __restrict__ sbuf, int lane) {
    const int sl = lane / W;
    const float4* __restrict__ J = a.store;
    float4* lo_raw = sbuf + 2 * QUAD_TILE_FLOAT4;
    float4* q_raw = lo_raw + TILE_J;
    const float4* __restrict__ LO = a.spj_lo - a.n_ptcl;

    const int64_t l0 = a.list_off[it.group];
    const int n_tiles = (int)((a.list_off[it.group + 1] - l0) / TILE_J);
    const int run1 = a.run1_len[it.group];
    const int te = (run1 + TILE_J - 1) / TILE_J;                  // first tile of run 2
    const int ts = (run1 - a.n_far[it.group]) / TILE_J;           // first tile with an SPJ entry (whole EPJ tiles before it)
    const int2* __restrict__ lst = reinterpret_cast<const int2*>(a.list + l0);

    int2 idn = make_int2(0, 0);
    float4 j0 = make_float4(0.f, 0.f, 0.f, 0.f), j1 = j0;
    QuadRec q0, q1;
    q0.a = q0.b = q1.a = q1.b = j0;
    // records of the lane's two entries of tile t; from tile ts on with Q (zero for particles and the padding), from te on
    // also the remainders of the centres of mass (cp.async into lo_raw)
    auto gather = [&](int t, const int2 id) {
        j0 = __ldg(J + id.x);
        j1 = __ldg(J + id.y);
        if (t >= ts) {
            const unsigned c0 = (unsigned)(id.x - a.n_ptcl), c1 = (unsigned)(id.y - a.n_ptcl);
            const bool v0 = c0 < (unsigned)a.n_cell, v1 = c1 < (unsigned)a.n_cell;
#if MWF_QUAD_ASYNC
            const float4* g0 = a.quad + (v0 ? 2 * (size_t)c0 : 0), *g1 = a.quad + (v1 ? 2 * (size_t)c1 : 0);
            cp_async16_zfill(q_raw + lane, g0, v0 ? 16 : 0);
            cp_async16_zfill(q_raw + 32 + lane, g0 + 1, v0 ? 16 : 0);
            cp_async16_zfill(q_raw + 64 + lane, g1, v1 ? 16 : 0);
            cp_async16_zfill(q_raw + 96 + lane, g1 + 1, v1 ? 16 : 0);
#else
            const float4 z = make_float4(0.f, 0.f, 0.f, 0.f);
            q0.a = v0 ? __ldg(a.quad + 2 * (size_t)c0) : z;
            q0.b = v0 ? __ldg(a.quad + 2 * (size_t)c0 + 1) : z;
            q1.a = v1 ? __ldg(a.quad + 2 * (size_t)c1) : z;
            q1.b = v1 ? __ldg(a.quad + 2 * (size_t)c1 + 1) : z;
#endif
        }
        if (t >= te) {
            cp_async16(lo_raw + lane, LO + id.x);
            cp_async16(lo_raw + 32 + lane, LO + id.y);
        }
        if (t >= ts) cp_async_commit();
    };
    if (n_tiles > 0) {
        gather(0, ld_stream_int2(lst + lane));
        if (n_tiles > 1) idn = ld_stream_int2(lst + 32 + lane);
    }

    float nx[2], ny[2], nz[2];
    bool valid[2];
    Acc2 acc, part;
    item_begin<W>(a, it, lane, nx, ny, nz, valid, acc);
    zero(part);
    const float4 c = __ldg(J + it.i_first);  // origin of the tiles of run 2

    for (int t = 0; t < n_tiles; ++t) {
        float4* T = sbuf + (t & 1) * QUAD_TILE_FLOAT4;
        if (t < te) {
            T[lane] = make_float4(j0.x, j1.x, j0.y, j1.y);
            T[32 + lane] = make_float4(j0.z, j1.z, j0.w, j1.w);
        } else {
            if (t == te) {  // from here on: item-centred
#pragma unroll
                for (int k = 0; k < 2; ++k) { nx[k] += c.x; ny[k] += c.y; nz[k] += c.z; }
            }
            cp_async_wait_all();  // the lane's own remainders (and Q records)
            const float4 r0 = lo_raw[lane], r1 = lo_raw[32 + lane];
            T[lane] = make_float4((j0.x - c.x) + r0.x, (j1.x - c.x) + r1.x, (j0.y - c.y) + r0.y, (j1.y - c.y) + r1.y);
            T[32 + lane] = make_float4((j0.z - c.z) + r0.z, (j1.z - c.z) + r1.z, j0.w, j1.w);
        }
        if (t >= ts) {
#if MWF_QUAD_ASYNC
            cp_async_wait_all();
            q0.a = q_raw[lane]; q0.b = q_raw[32 + lane]; q1.a = q_raw[64 + lane]; q1.b = q_raw[96 + lane];
#endif
            T[64 + lane] = make_float4(q0.a.x, q1.a.x, q0.a.y, q1.a.y);
            T[96 + lane] = make_float4(q0.a.z, q1.a.z, q0.a.w, q1.a.w);
            T[128 + lane] = make_float4(q0.b.x, q1.b.x, q0.b.y, q1.b.y);
            reinterpret_cast<float2*>(T + 160)[lane] = make_float2(-q0.b.z, -q1.b.z);
        }
        __syncwarp();
        if (t + 1 < n_tiles) {
            gather(t + 1, idn);
            if (t + 2 < n_tiles) idn = ld_stream_int2(lst + (int64_t)(t + 2) * 32 + lane);
        }
        if (t < ts) sweep_tile<W, MWF_NEAR_UNROLL>(T, T + 32, sl, nx, ny, nz, a.eps2, part);
        else sweep_tile_quad<W>(T, sl, nx, ny, nz, a.eps2, part);
        flush_partial<W>(t, acc, part);
    }
    add_into(acc, part);
    item_end<W>(a, it, lane, valid, acc);
}

template <int W, bool INDEXED>
__device__ __forceinline__ void run_item_any(const ForceArgs& a, const WorkItem it, float4* __restrict__ sbuf, int lane) {
    if constexpr (INDEXED) run_item<W>(a, it, sbuf, lane);
    else run_item_data<W>(a, it, sbuf, lane);
}

// work index -> position in the class-sorted permutation (ForceArgs::n_seg)
__device__ __forceinline__ int64_t seg_position(const ForceArgs& a, int64_t w) {
    int k = 0;
#pragma unroll
    for (int q = 1; q < N_WIDTH_CLASS; ++q) k += w >= a.seg_cum[q] ? 1 : 0;
    return a.seg_begin[k] + (w - a.seg_cum[k]);
}

// The block has blockDim.x / 32 warps (WARPS_PER_CTA for a whole-machine dispatch, fewer for a sub-wave one, see
// launch_force); s_tiles is dynamic shared memory, two tiles per warp.
template <bool INDEXED>
__device__ __forceinline__ void force_body(const ForceArgs& a, float4* s_tiles) {
    const int lane = threadIdx.x & 31;
    const int warp = threadIdx.x >> 5;
    const int warps_per_cta = blockDim.x >> 5;
    float4* sbuf = s_tiles + warp * FORCE_SMEM_FLOAT4_PER_WARP;
    int64_t w = (int64_t)blockIdx.x * warps_per_cta + warp;  // first item: static
    const int64_t n_warps = (int64_t)gridDim.x * warps_per_cta;
    while (w < a.n_items) {
        const int64_t pos = a.n_seg ? seg_position(a, w) : a.item_begin + w;
        const WorkItem it = a.items[a.order ? a.order[pos] : pos];
        switch (it.width) {
            case 32: run_item_any<32, INDEXED>(a, it, sbuf, lane); break;
            case 16: run_item_any<16, INDEXED>(a, it, sbuf, lane); break;
            case 8: run_item_any<8, INDEXED>(a, it, sbuf, lane); break;
            case 4: run_item_any<4, INDEXED>(a, it, sbuf, lane); break;
            default: run_item_any<2, INDEXED>(a, it, sbuf, lane); break;
        }
        if (a.counter) {  // dynamic: next unclaimed item
            unsigned int nxt = 0;
            if (lane == 0) nxt = atomicAdd(a.counter, 1u);
            w = n_warps + (int64_t)__shfl_sync(0xffffffffu, nxt, 0);
        } else {
            w += n_warps;
        }
    }
}

extern __shared__ float4 s_force_tiles[];

__global__ void __launch_bounds__(WARPS_PER_CTA * 32, MWF_MIN_CTAS) k_force(const ForceArgs a) {
    force_body<true>(a, s_force_tiles);
}

// Method G1 of the paper (multiwalk without indirect addressing, Fig. 2): same items, same sweep, but
// every group's list is a contiguous run of j RECORDS sent with the dispatch.  A/B variant.
__global__ void __launch_bounds__(WARPS_PER_CTA * 32, MWF_MIN_CTAS) k_force_data(const ForceArgs a) {
    force_body<false>(a, s_force_tiles);
}

// Order 2: the same items and schedule, quadrupole terms of the SPJ entries in the sweep (NEXT-3).
__global__ void __launch_bounds__(WARPS_PER_CTA * 32, MWF_MIN_CTAS) k_force_quad(const ForceArgs a) {
    const int lane = threadIdx.x & 31;
    const int warp = threadIdx.x >> 5;
    const int warps_per_cta = blockDim.x >> 5;
    float4* sbuf = s_force_tiles + warp * QUAD_SMEM_FLOAT4_PER_WARP;
    int64_t w = (int64_t)blockIdx.x * warps_per_cta + warp;
    const int64_t n_warps = (int64_t)gridDim.x * warps_per_cta;
    while (w < a.n_items) {
        const int64_t pos = a.n_seg ? seg_position(a, w) : a.item_begin + w;
        const WorkItem it = a.items[a.order ? a.order[pos] : pos];
        switch (it.width) {
            case 32: run_item_quad<32>(a, it, sbuf, lane); break;
            case 16: run_item_quad<16>(a, it, sbuf, lane); break;
            case 8: run_item_quad<8>(a, it, sbuf, lane); break;
            case 4: run_item_quad<4>(a, it, sbuf, lane); break;
            default: run_item_quad<2>(a, it, sbuf, lane); break;
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

constexpr size_t FORCE_SMEM_PER_WARP = FORCE_SMEM_FLOAT4_PER_WARP * sizeof(float4);
constexpr size_t QUAD_SMEM_PER_WARP = QUAD_SMEM_FLOAT4_PER_WARP * sizeof(float4);

// warps = warps per block: WARPS_PER_CTA for a dispatch that fills the machine (persistent grid, items claimed dynamically);
// a sub-wave dispatch (a batch of the multiwalk pipeline) is launched with small blocks, one item per warp, so
// that a block gives its registers back as soon as its own items are done and the batches of the other tags' streams
// pack beside it.
cudaError_t launch_force(const ForceArgs& a, int grid, int warps, cudaStream_t s) {
    if (a.n_items <= 0 || grid <= 0) return cudaSuccess;
    if (warps < 1 || warps > WARPS_PER_CTA) return cudaErrorInvalidValue;
    if (a.quad) {
        if (a.jdata) return cudaErrorInvalidValue;
        // 8 warps x 544 float4 = 68 KB of dynamic shared memory per block: above the default limit, so the kernel needs the opt-in of
        // force_quad_max_ctas_per_sm().  Function attributes are per device; mwf_set_spj_order(2) makes that call for every ctx on
        // the ctx's own device before it hands out a quad pointer, so no process-wide flag is kept here.
        k_force_quad<<<grid, warps * 32, warps * QUAD_SMEM_PER_WARP, s>>>(a);
    } else if (a.jdata)
        k_force_data<<<grid, warps * 32, warps * FORCE_SMEM_PER_WARP, s>>>(a);
    else
        k_force<<<grid, warps * 32, warps * FORCE_SMEM_PER_WARP, s>>>(a);
    return cudaGetLastError();
}

int force_quad_max_ctas_per_sm() {
    int n = 0;
    if (cudaFuncSetAttribute(k_force_quad, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)(WARPS_PER_CTA * QUAD_SMEM_PER_WARP)) != cudaSuccess) return 0;
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&n, k_force_quad, WARPS_PER_CTA * 32, WARPS_PER_CTA * QUAD_SMEM_PER_WARP) != cudaSuccess) return 0;
    return n;
}

int force_max_ctas_per_sm() {
    int n = 0;
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&n, k_force, WARPS_PER_CTA * 32, WARPS_PER_CTA * FORCE_SMEM_PER_WARP) != cudaSuccess) return 0;
    return n;
}

}  // namespace mwf
