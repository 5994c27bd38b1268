// Construction-step re-encoding of the uploaded CSR index lists.
// The two lists of a group (EPJ particle indices, SPJ cell indices) become ONE list of indices into the
// combined store -- EPJ ids, then SPJ ids + N -- the paper's layout ("id_epj ... id_spj + n_epj_tot"),
// cut into two RUNS, each padded to a whole number of 64-entry tiles with the index of a zero-mass dummy record
// (the paper pads with a sentinel walk whose list is empty):
//   run 1  entries the force kernel sweeps in the caller's coordinates with 16-byte records: every EPJ entry, and
//          every FAR SPJ entry -- a cell whose coordinates are no larger than SPJ_FAR_KAPPA times its distance from
//          the group, so that the fp32 rounding of its centre of mass (2^-24 of the coordinate) stays within
//          2e-6 of the separation;
//   run 2  the NEAR SPJ entries, swept in item-centred coordinates with the rounding remainder of the centre
//          (reading S11b of DESIGN.md).
// Indices are validated here, once; the force kernel then runs check-free on every reuse step.
#include "mwf_internal.h"

namespace mwf {

namespace {

constexpr unsigned FAR_BIT = 0x40000000u;  // marks a far SPJ entry in the staging ids between the two passes

// Pass 0: the tight bounding box of every cell's particles, bottom-up over the fixed tree like the climb variant of the
// monopole refresh: a leaf takes min / max over its particle range, the last child to arrive at a cell (self-resetting
// arrival counter) combines the children's boxes and carries on.  box[2c] = (lo, -), box[2c + 1] = (hi, -).  An uploaded
// tree carries no geometry, and min / max of fp32 values are exact, so these boxes are the one bound that holds for any
// tree and any list: the cell's centre of mass lies inside its box (convex hull of the particles).
__global__ void __launch_bounds__(128) k_cell_boxes(const mwf_cell* __restrict__ cells, const int32_t* __restrict__ parent, int64_t n_cell,
                                                    const float4* __restrict__ store, float4* __restrict__ box, int32_t* __restrict__ counter) {
    const int64_t c0 = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (c0 >= n_cell) return;
    const mwf_cell leaf = cells[c0];
    if (leaf.n_child != 0) return;
    float lo[3] = {INFINITY, INFINITY, INFINITY}, hi[3] = {-INFINITY, -INFINITY, -INFINITY};
    const float4* __restrict__ p = store + leaf.first_ptcl;
    for (int k = 0; k < leaf.n_ptcl; ++k) {
        const float4 q = p[k];
        lo[0] = fminf(lo[0], q.x); hi[0] = fmaxf(hi[0], q.x);
        lo[1] = fminf(lo[1], q.y); hi[1] = fmaxf(hi[1], q.y);
        lo[2] = fminf(lo[2], q.z); hi[2] = fmaxf(hi[2], q.z);
    }
    box[2 * c0] = make_float4(lo[0], lo[1], lo[2], 0.f);
    box[2 * c0 + 1] = make_float4(hi[0], hi[1], hi[2], 0.f);
    int64_t c = c0;
    for (;;) {
        const int32_t par = parent[c];
        if (par < 0) break;
        const mwf_cell pc = cells[par];
        __threadfence();  // publish this cell's box before announcing arrival
        if (atomicAdd(&counter[par], 1) != pc.n_child - 1) break;
        counter[par] = 0;
        __threadfence();
        for (int a = 0; a < 3; ++a) { lo[a] = INFINITY; hi[a] = -INFINITY; }
        for (int k = 0; k < pc.n_child; ++k) {
            const float4 l = __ldcg(&box[2 * (int64_t)(pc.first_child + k)]), h = __ldcg(&box[2 * (int64_t)(pc.first_child + k) + 1]);
            lo[0] = fminf(lo[0], l.x); hi[0] = fmaxf(hi[0], h.x);
            lo[1] = fminf(lo[1], l.y); hi[1] = fmaxf(hi[1], h.y);
            lo[2] = fminf(lo[2], l.z); hi[2] = fmaxf(hi[2], h.z);
        }
        box[2 * (int64_t)par] = make_float4(lo[0], lo[1], lo[2], 0.f);
        box[2 * (int64_t)par + 1] = make_float4(hi[0], hi[1], hi[2], 0.f);
        c = par;
    }
}

// Pass 1: classifies every SPJ entry of every group as far or near and counts the far ones.  There are no moments yet at
// this point of the construction step, so the cell is located by the tight box of its particles (pass 0) and the group by
// the tight box of its own: the gap between the two boxes is a lower bound of the distance from any i-particle to the
// cell's centre of mass, and the largest |coordinate| of the cell's box an upper bound of the centre's -- so "far" is a
// bound, for any list, not an estimate.  have_ptcl = 0 (the particles of this step are not in the store yet): everything is near.
__global__ void __launch_bounds__(256) k_classify_spj(int64_t n_group, const int32_t* __restrict__ grp_first, const int32_t* __restrict__ grp_n,
                                                      const int64_t* __restrict__ spj_off, int32_t* __restrict__ spj_id, const float4* __restrict__ box,
                                                      const float4* __restrict__ store, int64_t n_ptcl, int64_t n_cell, int have_ptcl,
                                                      int32_t* __restrict__ n_far) {
    __shared__ float s_box[6][8];
    __shared__ int s_cnt;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    for (int64_t g = blockIdx.x; g < n_group; g += gridDim.x) {
        if (threadIdx.x == 0) s_cnt = 0;
        const int32_t gf = grp_first[g], gn = grp_n[g];
        const bool ok = have_ptcl && gf >= 0 && gn > 0 && (int64_t)gf + gn <= n_ptcl;
        float lo[3] = {INFINITY, INFINITY, INFINITY}, hi[3] = {-INFINITY, -INFINITY, -INFINITY};
        if (ok)
            for (int i = threadIdx.x; i < gn; i += blockDim.x) {
                const float4 p = store[gf + i];
                lo[0] = fminf(lo[0], p.x); hi[0] = fmaxf(hi[0], p.x);
                lo[1] = fminf(lo[1], p.y); hi[1] = fmaxf(hi[1], p.y);
                lo[2] = fminf(lo[2], p.z); hi[2] = fmaxf(hi[2], p.z);
            }
#pragma unroll
        for (int a = 0; a < 3; ++a) {
#pragma unroll
            for (int d = 16; d > 0; d >>= 1) {
                lo[a] = fminf(lo[a], __shfl_xor_sync(0xffffffffu, lo[a], d));
                hi[a] = fmaxf(hi[a], __shfl_xor_sync(0xffffffffu, hi[a], d));
            }
            if (lane == 0) { s_box[a][warp] = lo[a]; s_box[3 + a][warp] = hi[a]; }
        }
        __syncthreads();
#pragma unroll
        for (int a = 0; a < 3; ++a)
            for (int w = 0; w < 8; ++w) { lo[a] = fminf(lo[a], s_box[a][w]); hi[a] = fmaxf(hi[a], s_box[3 + a][w]); }
        const int64_t s0 = spj_off[g], ns = spj_off[g + 1] - s0;
        int far = 0;
        for (int64_t k = threadIdx.x; k < ns; k += blockDim.x) {
            const int32_t id = spj_id[s0 + k];
            // A bad index is reported by the merge pass.  It is overwritten here, before any far mark is set, so that an uploaded
            // id that happens to carry FAR_BIT over valid low bits cannot pass for a marked entry (n_cell < 2^30: params_ok).
            if (id < 0 || id >= n_cell) { spj_id[s0 + k] = -1; continue; }
            if (!ok) continue;
            const float4 a = box[2 * (int64_t)id], b = box[2 * (int64_t)id + 1];
            const float pa[3] = {a.x, a.y, a.z}, pb[3] = {b.x, b.y, b.z};
            float d2 = 0.f, amax = 0.f;
#pragma unroll
            for (int q = 0; q < 3; ++q) {
                const float clo = pa[q], chi = pb[q];
                const float gap = fmaxf(0.f, fmaxf(lo[q] - chi, clo - hi[q]));
                d2 += gap * gap;
                amax = fmaxf(amax, fmaxf(fabsf(clo), fabsf(chi)));
            }
            if (amax <= SPJ_FAR_KAPPA * sqrtf(d2)) {
                spj_id[s0 + k] = id | (int32_t)FAR_BIT;
                ++far;
            }
        }
        if (far) atomicAdd(&s_cnt, far);
        __syncthreads();
        if (threadIdx.x == 0) n_far[g] = s_cnt;
        __syncthreads();
    }
}

// Ordered compaction of one chunk of a block: returns the number of flagged threads before this one, *total = all of them.
__device__ __forceinline__ int block_rank(bool flag, int* s_warp, int* total) {
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const unsigned m = __ballot_sync(0xffffffffu, flag);
    if (lane == 0) s_warp[warp] = __popc(m);
    __syncthreads();
    int before = 0, tot = 0;
    for (int w = 0; w < 8; ++w) {
        if (w == warp) before = tot;
        tot += s_warp[w];
    }
    *total = tot;
    __syncthreads();
    return before + __popc(m & ((1u << lane) - 1u));
}

// Pass 2: writes the merged list.  list_off[g] = start of group g's list, run1_len[g] = EPJ + far SPJ entries.
__global__ void __launch_bounds__(256) k_merge_lists(int64_t n_group, const int32_t* __restrict__ grp_first,
                                                     const int32_t* __restrict__ grp_n, const int64_t* __restrict__ epj_off,
                                                     const int32_t* __restrict__ epj_id, const int64_t* __restrict__ spj_off,
                                                     const int32_t* __restrict__ spj_id, const int64_t* __restrict__ list_off,
                                                     const int32_t* __restrict__ n_far, int32_t* __restrict__ run1_len,
                                                     int64_t n_ptcl, int64_t n_cell, int32_t* __restrict__ list,
                                                     uint8_t* __restrict__ grp_self, unsigned int* __restrict__ err) {
    __shared__ int s_self;
    __shared__ int s_warp[8];
    const int32_t dummy = (int32_t)(n_ptcl + n_cell);
    for (int64_t g = blockIdx.x; g < n_group; g += gridDim.x) {
        if (threadIdx.x == 0) s_self = 0;
        __syncthreads();
        const int64_t e0 = epj_off[g], ne = epj_off[g + 1] - e0;
        const int64_t s0 = spj_off[g], ns = spj_off[g + 1] - s0;
        const int64_t o0 = list_off[g], padded = list_off[g + 1] - o0;
        const int64_t n1 = ne + n_far[g];
        const int64_t n1_pad = (n1 + TILE_J - 1) / TILE_J * TILE_J;  // run 2 starts on a tile boundary
        const int32_t gf = grp_first[g], gn = grp_n[g];
        unsigned int e = 0;
        int self = 0;
        if (gf < 0 || gn <= 0 || (int64_t)gf + gn > n_ptcl) e |= ERR_GROUP_RANGE;
        for (int64_t k = threadIdx.x; k < ne; k += blockDim.x) {
            int32_t id = epj_id[e0 + k];
            if (id < 0 || id >= n_ptcl) { e |= ERR_EPJ_INDEX; id = dummy; }
            if (id >= gf && id < gf + gn) ++self;
            list[o0 + k] = id;
        }
        // SPJ entries in their order, far ones behind the EPJ entries, near ones into run 2
        int64_t at_far = o0 + ne, at_near = o0 + n1_pad;
        for (int64_t k0 = 0; k0 < ns; k0 += blockDim.x) {
            const int64_t k = k0 + threadIdx.x;
            const bool in = k < ns;
            int32_t raw = in ? spj_id[s0 + k] : 0;
            const bool far = in && (raw & (int32_t)FAR_BIT) != 0 && raw >= 0;
            if (far) raw &= ~(int32_t)FAR_BIT;
            int64_t v = n_ptcl + raw;
            if (in && (raw < 0 || raw >= n_cell)) { e |= ERR_SPJ_INDEX; v = dummy; }
            int n_f, n_n;
            const int r_f = block_rank(far, s_warp, &n_f);
            const int r_n = block_rank(in && !far, s_warp, &n_n);
            if (far) list[at_far + r_f] = (int32_t)v;
            else if (in) list[at_near + r_n] = (int32_t)v;
            at_far += n_f;
            at_near += n_n;
        }
        for (int64_t k = n1 + threadIdx.x; k < n1_pad; k += blockDim.x) list[o0 + k] = dummy;
        for (int64_t k = n1_pad + (ns - n_far[g]) + threadIdx.x; k < padded; k += blockDim.x) list[o0 + k] = dummy;
        if (self) atomicAdd(&s_self, self);
        __syncthreads();
        if (threadIdx.x == 0) {
            run1_len[g] = (int32_t)n1;
            if (s_self == gn) grp_self[g] = 1;
            else if (s_self == 0) grp_self[g] = 0;
            else { grp_self[g] = 0; e |= ERR_SELF_MIXED; }
        }
        if (e) atomicOr(err, e);
        __syncthreads();
    }
}

}  // namespace

// box: scratch for 2 float4 per cell; parent / counter: those of the validated tree (counter all zero, left all zero).
cudaError_t launch_classify_spj(int64_t n_group, const int32_t* grp_first, const int32_t* grp_n, const int64_t* spj_off, int32_t* spj_id,
                                const mwf_cell* cells, const int32_t* parent, int32_t* counter, float4* box, const float4* store, int64_t n_ptcl,
                                int64_t n_cell, bool have_ptcl, int32_t* n_far, cudaStream_t s) {
    if (n_group <= 0) return cudaSuccess;
    if (have_ptcl) {
        k_cell_boxes<<<(unsigned)((n_cell + 127) / 128), 128, 0, s>>>(cells, parent, n_cell, store, box, counter);
        const cudaError_t e = cudaGetLastError();
        if (e != cudaSuccess) return e;
    }
    const int64_t grid = n_group < 148 * 16 ? n_group : 148 * 16;
    k_classify_spj<<<(unsigned)grid, 256, 0, s>>>(n_group, grp_first, grp_n, spj_off, spj_id, box, store, n_ptcl, n_cell, have_ptcl ? 1 : 0, n_far);
    return cudaGetLastError();
}

cudaError_t launch_merge_lists(int64_t n_group, const int32_t* grp_first, const int32_t* grp_n, const int64_t* epj_off,
                               const int32_t* epj_id, const int64_t* spj_off, const int32_t* spj_id, const int64_t* list_off,
                               const int32_t* n_far, int32_t* run1_len, int64_t n_ptcl, int64_t n_cell, int32_t* list, uint8_t* grp_self,
                               unsigned int* err, cudaStream_t s) {
    if (n_group <= 0) return cudaSuccess;
    const int64_t grid = n_group < 148 * 16 ? n_group : 148 * 16;
    k_merge_lists<<<(unsigned)grid, 256, 0, s>>>(n_group, grp_first, grp_n, epj_off, epj_id, spj_off, spj_id, list_off, n_far, run1_len, n_ptcl,
                                                 n_cell, list, grp_self, err);
    return cudaGetLastError();
}

}  // namespace mwf
