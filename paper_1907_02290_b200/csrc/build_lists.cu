// Device-side construction step, part 2: one tree walk per i-group emitting its interaction list as indices
// (paper: Barnes' vectorisation, one traversal per group of particles and one
// shared list; for the index method the list holds indices).
//
// Reading O4 / S6-S7 of DESIGN.md, identical to the host builder: for a cell of side l and geometric centre s,
// d = distance from s to the group's tight particle bounding box (0 inside); OPEN iff l > theta * d, evaluated
// as l*l > theta^2 * d^2 in fp64 with explicitly rounded operations.  Opened internal cell -> its children are
// visited; opened leaf -> its particles join the EPJ list; cell not opened -> it joins the SPJ list.
//
// One WARP per group, groups claimed from an atomic counter.  The warp keeps a LIFO stack of cell indices in
// global memory (L2-resident scratch, one slab per warp), pops up to 32 cells per round, tests one per lane and
// compacts the three outcomes with ballots / warp prefix sums.  At most 256 cells of any one level are ever on
// the stack, so 22 levels x 256 entries bound it.  The walk runs twice: a counting pass (n_epj, n_spj per group)
// and, after the offsets have been scanned, a fill pass that writes the merged, padded list the force kernel
// reads: EPJ ids, then SPJ ids + N (P:441-477 layout), each run padded with the dummy index to a multiple of 64.
#include "mwf_internal.h"
#include "scan_sort.cuh"

namespace mwf {

namespace {

template <bool FILL, bool NEIGH>
__global__ void __launch_bounds__(256) k_walk(const mwf_cell* __restrict__ cells, const double4* __restrict__ geom, const float* __restrict__ grp_box,
                                              int64_t n_group, double th2, double reach, const float* __restrict__ cell_h, const float* __restrict__ grp_h,
                                              int32_t* __restrict__ stacks, unsigned int* __restrict__ counter,
                                              int32_t* __restrict__ n_epj, int32_t* __restrict__ n_spj, int32_t* __restrict__ n_far,
                                              const int64_t* __restrict__ list_off, int32_t* __restrict__ list, int32_t n_ptcl, int32_t dummy) {
    const int lane = threadIdx.x & 31;
    const unsigned lt = (1u << lane) - 1u;
    const int64_t warp_global = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    int32_t* __restrict__ stack = stacks + warp_global * WALK_STACK;
    for (;;) {
        unsigned int gi = 0;
        if (lane == 0) gi = atomicAdd(counter, 1u);
        const int64_t g = __shfl_sync(0xffffffffu, gi, 0);
        if (g >= n_group) break;
        double lo[3], hi[3];
#pragma unroll
        for (int a = 0; a < 3; ++a) {
            lo[a] = (double)grp_box[g * 6 + a];
            hi[a] = (double)grp_box[g * 6 + 3 + a];
        }
        double rg = 0.0;
        if constexpr (NEIGH) rg = __dmul_rn(reach, (double)grp_h[g]);
        int64_t off_e = 0, off_f = 0, off_s = 0;  // where the group's EPJ, far SPJ and near SPJ entries go
        if (FILL) {
            off_e = list_off[g];
            off_f = off_e + n_epj[g];                                                    // run 1: EPJ, then far SPJ
            off_s = off_e + (n_epj[g] + n_far[g] + TILE_J - 1) / TILE_J * TILE_J;        // run 2 starts on a tile boundary
        }
        int ne = 0, ns = 0, nf = 0, sp = 1;  // ns: near SPJ, nf: far SPJ
        if (lane == 0) stack[0] = 0;
        __syncwarp();
        while (sp > 0) {
            const int take = sp < 32 ? sp : 32;
            sp -= take;
            const int c = lane < take ? stack[sp + lane] : -1;
            __syncwarp();
            int kind = 0;  // 1: SPJ, 2: opened internal cell, 3: opened leaf
            bool far = false;
            mwf_cell cc = {0, 0, 0, 0};
            if (c >= 0) {
                cc = cells[c];
                const double4 gm = geom[c];
                const double s3[3] = {gm.x, gm.y, gm.z};
                double d2 = 0.0;
                if constexpr (NEIGH) {  // gap between the cell's cube and the group's box against the search radius
                    const double half = __dmul_rn(0.5, gm.w);
#pragma unroll
                    for (int a = 0; a < 3; ++a) {
                        const double top = __dadd_rn(s3[a], half), bot = __dsub_rn(s3[a], half);
                        double d = 0.0;
                        if (top < lo[a]) d = __dsub_rn(lo[a], top);
                        else if (bot > hi[a]) d = __dsub_rn(bot, hi[a]);
                        d2 = __dadd_rn(d2, __dmul_rn(d, d));
                    }
                    const double rc = __dmul_rn(reach, (double)cell_h[c]);
                    const double r = rg > rc ? rg : rc;
                    kind = !(d2 <= __dmul_rn(r, r)) ? 0 : (cc.n_child == 0 ? 3 : 2);  // out of reach: dropped, there are no SPJ
                } else {
#pragma unroll
                    for (int a = 0; a < 3; ++a) {
                        double d = 0.0;
                        if (s3[a] < lo[a]) d = __dsub_rn(lo[a], s3[a]);
                        else if (s3[a] > hi[a]) d = __dsub_rn(s3[a], hi[a]);
                        d2 = __dadd_rn(d2, __dmul_rn(d, d));
                    }
                    const bool open = __dmul_rn(gm.w, gm.w) > __dmul_rn(th2, d2);
                    kind = !open ? 1 : (cc.n_child == 0 ? 3 : 2);
                    if (!open) {  // far or near (SPJ_FAR_KAPPA): the centre of mass lies within the cell's cube
                        const double half = 0.5 * gm.w;
                        const double amax = fmax(fmax(fabs(s3[0]), fabs(s3[1])), fabs(s3[2])) + half;
                        far = amax <= (double)SPJ_FAR_KAPPA * fmax(0.0, sqrt(d2) - 1.7320508075688772 * half);
                    }
                }
            }
            // SPJ entries: far ones behind the EPJ entries of run 1, near ones in run 2
            const unsigned m_f = __ballot_sync(0xffffffffu, kind == 1 && far);
            const unsigned m_s = __ballot_sync(0xffffffffu, kind == 1 && !far);
            if (FILL && kind == 1) {
                if (far) list[off_f + nf + __popc(m_f & lt)] = n_ptcl + c;
                else list[off_s + ns + __popc(m_s & lt)] = n_ptcl + c;
            }
            nf += __popc(m_f);
            ns += __popc(m_s);
            // opened leaves: their particles
            const unsigned m_l = __ballot_sync(0xffffffffu, kind == 3);
            if (m_l) {
                int cnt = kind == 3 ? cc.n_ptcl : 0, incl = cnt;
#pragma unroll
                for (int d = 1; d < 32; d <<= 1) {
                    const int up = __shfl_up_sync(0xffffffffu, incl, d);
                    if (lane >= d) incl += up;
                }
                const int total = __shfl_sync(0xffffffffu, incl, 31);
                if (FILL) {
                    const int excl = incl - cnt;
                    unsigned m = m_l;
                    while (m) {
                        const int src = __ffs(m) - 1;
                        m &= m - 1;
                        const int first = __shfl_sync(0xffffffffu, cc.first_ptcl, src);
                        const int n_in = __shfl_sync(0xffffffffu, cnt, src);
                        const int base = __shfl_sync(0xffffffffu, excl, src);
                        for (int k = lane; k < n_in; k += 32) list[off_e + ne + base + k] = first + k;
                    }
                }
                ne += total;
            }
            // opened internal cells: push their children
            const unsigned m_o = __ballot_sync(0xffffffffu, kind == 2);
            if (m_o) {
                int cnt = kind == 2 ? cc.n_child : 0, incl = cnt;
#pragma unroll
                for (int d = 1; d < 32; d <<= 1) {
                    const int up = __shfl_up_sync(0xffffffffu, incl, d);
                    if (lane >= d) incl += up;
                }
                const int total = __shfl_sync(0xffffffffu, incl, 31);
                const int excl = incl - cnt;
                for (int k = 0; k < cnt; ++k) stack[sp + excl + k] = cc.first_child + k;
                sp += total;
            }
            __syncwarp();
        }
        if (FILL) {  // pad both runs to whole tiles with the zero-mass dummy record
            const int64_t end = list_off[g + 1];
            for (int64_t k = off_f + nf + lane; k < off_s; k += 32) list[k] = dummy;
            for (int64_t k = off_s + ns + lane; k < end; k += 32) list[k] = dummy;
        } else if (lane == 0) {
            n_epj[g] = ne;
            n_spj[g] = ns + nf;
            n_far[g] = nf;
        }
    }
}

// Largest smoothing length among the particles of every cell (bits of a positive float order like ints): each leaf
// takes the maximum over its particles and raises its ancestors with atomicMax until one is already as large.
__global__ void __launch_bounds__(256) k_cell_hmax(const mwf_cell* __restrict__ cells, const int32_t* __restrict__ parent, const float4* __restrict__ sph,
                                                   int64_t n_cell, int* __restrict__ cell_h) {
    const int64_t c0 = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (c0 >= n_cell) return;
    const mwf_cell cc = cells[c0];
    if (cc.n_child != 0) return;
    float m = 0.f;
    for (int k = 0; k < cc.n_ptcl; ++k) m = fmaxf(m, sph[cc.first_ptcl + k].x);
    const int bits = __float_as_int(m);
    int32_t c = (int32_t)c0;
    while (c >= 0) {
        if (atomicMax(&cell_h[c], bits) >= bits && c != (int32_t)c0) break;
        c = parent[c];
    }
}

__global__ void __launch_bounds__(256) k_group_hmax(const float4* __restrict__ sph, const int32_t* __restrict__ grp_first, const int32_t* __restrict__ grp_n,
                                                    int64_t n_group, float* __restrict__ grp_h) {
    const int lane = threadIdx.x & 31;
    const int64_t g = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    if (g >= n_group) return;
    const int f = grp_first[g], cnt = grp_n[g];
    float m = 0.f;
    for (int i = lane; i < cnt; i += 32) m = fmaxf(m, sph[f + i].x);
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) m = fmaxf(m, __shfl_xor_sync(0xffffffffu, m, d));
    if (lane == 0) grp_h[g] = m;
}

// list_off[g] (to be scanned) = padded length of group g's merged list
__global__ void __launch_bounds__(256) k_padded_len(const int32_t* __restrict__ n_epj, const int32_t* __restrict__ n_spj, const int32_t* __restrict__ n_far,
                                                    int64_t n_group, int32_t* __restrict__ run1_len, int64_t* __restrict__ list_off,
                                                    int64_t* __restrict__ epj_off, int64_t* __restrict__ spj_off) {
    const int64_t g = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (g > n_group) return;
    if (g == n_group) { list_off[g] = 0; epj_off[g] = 0; spj_off[g] = 0; return; }
    const int64_t n1 = (int64_t)n_epj[g] + n_far[g], n2 = (int64_t)n_spj[g] - n_far[g];  // run 1: EPJ + far SPJ, run 2: near SPJ
    run1_len[g] = (int32_t)n1;
    list_off[g] = (n1 + TILE_J - 1) / TILE_J * TILE_J + (n2 + TILE_J - 1) / TILE_J * TILE_J;
    epj_off[g] = n_epj[g];
    spj_off[g] = n_spj[g];
}

// merged list -> the two CSR id arrays of the upload interface (read-back hook)
__global__ void __launch_bounds__(256) k_unmerge(const int32_t* __restrict__ list, const int64_t* __restrict__ list_off, const int64_t* __restrict__ epj_off,
                                                 const int64_t* __restrict__ spj_off, const int32_t* __restrict__ n_far, int64_t n_group, int32_t n_ptcl,
                                                 int32_t* __restrict__ epj_id, int32_t* __restrict__ spj_id) {
    for (int64_t g = blockIdx.x; g < n_group; g += gridDim.x) {
        const int64_t l0 = list_off[g], e0 = epj_off[g], ne = epj_off[g + 1] - e0, s0 = spj_off[g], ns = spj_off[g + 1] - s0;
        const int64_t nf = n_far[g], n1_pad = (ne + nf + TILE_J - 1) / TILE_J * TILE_J;  // far SPJ behind the EPJ, near SPJ in run 2
        for (int64_t k = threadIdx.x; k < ne; k += blockDim.x) epj_id[e0 + k] = list[l0 + k];
        for (int64_t k = threadIdx.x; k < ns; k += blockDim.x) spj_id[s0 + k] = list[k < nf ? l0 + ne + k : l0 + n1_pad + (k - nf)] - n_ptcl;
    }
}

}  // namespace

#define BL(call)                                \
    do {                                        \
        cudaError_t e__ = (call);               \
        if (e__ != cudaSuccess) return e__;     \
    } while (0)

int64_t walk_warps(int64_t max_group) {
    const int64_t cap = 148 * 32;
    return max_group < cap ? (max_group < 8 ? 8 : (max_group + 7) / 8 * 8) : cap;
}

// Counting pass + offsets.  Leaves list_off / epj_off / spj_off scanned (n_group + 1 entries each); the totals go to pinned
// host memory on the stream (no synchronisation here).
cudaError_t build_smoothing_reach(const BuildBuffers& b, const float4* sph, int64_t n_cell, int64_t n_group, float* cell_h, float* grp_h, cudaStream_t s) {
    BL(cudaMemsetAsync(cell_h, 0, (size_t)n_cell * 4, s));
    k_cell_hmax<<<(unsigned)((n_cell + 255) / 256), 256, 0, s>>>(b.cells, b.parent, sph, n_cell, reinterpret_cast<int*>(cell_h));
    BL(cudaGetLastError());
    k_group_hmax<<<(unsigned)((n_group * 32 + 255) / 256), 256, 0, s>>>(sph, b.grp_first, b.grp_n, n_group, grp_h);
    return cudaGetLastError();
}

cudaError_t build_lists_count(const BuildBuffers& b, int64_t n_group, const WalkRule& rule, int64_t n_warps, int64_t* totals_pinned, cudaStream_t s) {
    const double th2 = rule.theta * rule.theta;
    BL(cudaMemsetAsync(b.walk_counter, 0, 4, s));
    if (rule.neighbours)
        k_walk<false, true><<<(unsigned)(n_warps / 8), 256, 0, s>>>(b.cells, b.geom, b.grp_box, n_group, th2, rule.reach, rule.cell_h, rule.grp_h, b.walk_stacks,
                                                                    b.walk_counter, b.n_epj, b.n_spj, b.n_far, nullptr, nullptr, 0, 0);
    else
        k_walk<false, false><<<(unsigned)(n_warps / 8), 256, 0, s>>>(b.cells, b.geom, b.grp_box, n_group, th2, 0.0, nullptr, nullptr, b.walk_stacks,
                                                                     b.walk_counter, b.n_epj, b.n_spj, b.n_far, nullptr, nullptr, 0, 0);
    BL(cudaGetLastError());
    k_padded_len<<<(unsigned)((n_group + 1 + 255) / 256), 256, 0, s>>>(b.n_epj, b.n_spj, b.n_far, n_group, b.run1_len, b.list_off, b.epj_off, b.spj_off);
    BL(cudaGetLastError());
    BL(scan_exclusive<int64_t>(b.list_off, n_group + 1, b.scan_scratch64, s));
    BL(scan_exclusive<int64_t>(b.epj_off, n_group + 1, b.scan_scratch64, s));
    BL(scan_exclusive<int64_t>(b.spj_off, n_group + 1, b.scan_scratch64, s));
    BL(cudaMemcpyAsync(totals_pinned + 0, b.list_off + n_group, 8, cudaMemcpyDeviceToHost, s));
    BL(cudaMemcpyAsync(totals_pinned + 1, b.epj_off + n_group, 8, cudaMemcpyDeviceToHost, s));
    BL(cudaMemcpyAsync(totals_pinned + 2, b.spj_off + n_group, 8, cudaMemcpyDeviceToHost, s));
    return cudaSuccess;
}

cudaError_t build_lists_fill(const BuildBuffers& b, int64_t n_group, const WalkRule& rule, int64_t n_warps, int64_t n_ptcl, int64_t n_cell, cudaStream_t s) {
    const double th2 = rule.theta * rule.theta;
    BL(cudaMemsetAsync(b.walk_counter, 0, 4, s));
    if (rule.neighbours)
        k_walk<true, true><<<(unsigned)(n_warps / 8), 256, 0, s>>>(b.cells, b.geom, b.grp_box, n_group, th2, rule.reach, rule.cell_h, rule.grp_h, b.walk_stacks,
                                                                   b.walk_counter, b.n_epj, b.n_spj, b.n_far, b.list_off, b.list, (int32_t)n_ptcl, (int32_t)(n_ptcl + n_cell));
    else
        k_walk<true, false><<<(unsigned)(n_warps / 8), 256, 0, s>>>(b.cells, b.geom, b.grp_box, n_group, th2, 0.0, nullptr, nullptr, b.walk_stacks,
                                                                    b.walk_counter, b.n_epj, b.n_spj, b.n_far, b.list_off, b.list, (int32_t)n_ptcl, (int32_t)(n_ptcl + n_cell));
    return cudaGetLastError();
}

cudaError_t unmerge_lists(const BuildBuffers& b, int64_t n_group, int64_t n_ptcl, int32_t* epj_id, int32_t* spj_id, cudaStream_t s) {
    if (n_group <= 0) return cudaSuccess;
    const int64_t grid = n_group < 148 * 16 ? n_group : 148 * 16;
    k_unmerge<<<(unsigned)grid, 256, 0, s>>>(b.list, b.list_off, b.epj_off, b.spj_off, b.n_far, n_group, (int32_t)n_ptcl, epj_id, spj_id);
    return cudaGetLastError();
}

}  // namespace mwf
