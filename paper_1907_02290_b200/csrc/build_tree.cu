// Device-side construction step, part 1: root cell, Morton keys, sort, reorder, octree cells level by level,
// i-groups (paper P:149 root cell, "Morton keys -> radix sort ->
// reorder -> link cells level by level, top to bottom", P:77 / P:401 groups of <= n_grp particles).
//
// Readings O1-O3 / S8-S9 of DESIGN.md, identical to the host builder and to the plain restatement the tests
// compare against: cube root cell centred on the bounding box with side = extent x (1 + 2^-10); 21 bits per
// axis; a cell with <= n_leaf particles (or at depth 21) is a leaf; empty octants get no cell; children are
// contiguous, after their parent, in level (BFS) order; a group is the first cell on a root path with
// <= n_grp particles (or a leaf).  All geometry is fp64 with explicitly rounded operations (no FMA
// contraction), so that grid coordinates and cell centres are bit-identical to the host's.
#include "mwf_internal.h"
#include "scan_sort.cuh"

namespace mwf {

namespace {

constexpr int KEY_BITS = 21;

// ---- root cell -------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) k_bbox_partial(const float4* __restrict__ p, int64_t n, float* __restrict__ part) {
    float lo[3] = {INFINITY, INFINITY, INFINITY}, hi[3] = {-INFINITY, -INFINITY, -INFINITY};
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) {
        const float4 q = p[i];
        lo[0] = fminf(lo[0], q.x); hi[0] = fmaxf(hi[0], q.x);
        lo[1] = fminf(lo[1], q.y); hi[1] = fmaxf(hi[1], q.y);
        lo[2] = fminf(lo[2], q.z); hi[2] = fmaxf(hi[2], q.z);
    }
    __shared__ float s[6][8];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
#pragma unroll
    for (int a = 0; a < 3; ++a) {
#pragma unroll
        for (int d = 16; d > 0; d >>= 1) {
            lo[a] = fminf(lo[a], __shfl_xor_sync(0xffffffffu, lo[a], d));
            hi[a] = fmaxf(hi[a], __shfl_xor_sync(0xffffffffu, hi[a], d));
        }
        if (lane == 0) { s[a][warp] = lo[a]; s[3 + a][warp] = hi[a]; }
    }
    __syncthreads();
    if (threadIdx.x < 6) {
        float v = s[threadIdx.x][0];
        for (int w = 1; w < 8; ++w) v = threadIdx.x < 3 ? fminf(v, s[threadIdx.x][w]) : fmaxf(v, s[threadIdx.x][w]);
        part[(int64_t)blockIdx.x * 6 + threadIdx.x] = v;
    }
}

// root[0..2] = centre, root[3] = side, root[4..6] = lower corner (all fp64, rounded like the host's)
__global__ void k_root(const float* __restrict__ part, int n_part, double* __restrict__ root) {
    // one warp: min / max are exact, so the order in which the partial boxes are combined does not matter
    if (blockIdx.x != 0 || threadIdx.x >= 32) return;
    double lo[3] = {INFINITY, INFINITY, INFINITY}, hi[3] = {-INFINITY, -INFINITY, -INFINITY};
    for (int b = threadIdx.x; b < n_part; b += 32)
        for (int a = 0; a < 3; ++a) {
            lo[a] = fmin(lo[a], (double)part[6 * b + a]);
            hi[a] = fmax(hi[a], (double)part[6 * b + 3 + a]);
        }
    for (int a = 0; a < 3; ++a)
        for (int d = 16; d > 0; d >>= 1) {
            lo[a] = fmin(lo[a], __shfl_xor_sync(0xffffffffu, lo[a], d));
            hi[a] = fmax(hi[a], __shfl_xor_sync(0xffffffffu, hi[a], d));
        }
    if (threadIdx.x != 0) return;
    double ext = 0.0;
    for (int a = 0; a < 3; ++a) {
        root[a] = __dmul_rn(0.5, __dadd_rn(lo[a], hi[a]));
        ext = fmax(ext, __dsub_rn(hi[a], lo[a]));
    }
    if (!(ext > 0.0)) ext = 1.0;
    const double side = __dmul_rn(ext, 1.0 + 1.0 / 1024.0);
    root[3] = side;
    for (int a = 0; a < 3; ++a) root[4 + a] = __dsub_rn(root[a], __dmul_rn(0.5, side));
}

// ---- keys ------------------------------------------------------------------------------------------
__device__ __forceinline__ uint64_t spread3(uint64_t v) {  // 21 bits -> every third bit
    v &= 0x1fffffULL;
    v = (v | v << 32) & 0x1f00000000ffffULL;
    v = (v | v << 16) & 0x1f0000ff0000ffULL;
    v = (v | v << 8) & 0x100f00f00f00f00fULL;
    v = (v | v << 4) & 0x10c30c30c30c30c3ULL;
    v = (v | v << 2) & 0x1249249249249249ULL;
    return v;
}

__device__ __forceinline__ uint64_t grid_coord(double x, double lo, double side) {
    const double t = __dmul_rn(__ddiv_rn(__dsub_rn(x, lo), side), (double)(1 << KEY_BITS));
    long long i = (long long)floor(t);
    if (i < 0) i = 0;
    if (i > (1 << KEY_BITS) - 1) i = (1 << KEY_BITS) - 1;
    return (uint64_t)i;
}

__global__ void __launch_bounds__(256) k_keys(const float4* __restrict__ p, int64_t n, const double* __restrict__ root,
                                              uint64_t* __restrict__ key, int32_t* __restrict__ idx) {
    const double side = root[3], lx = root[4], ly = root[5], lz = root[6];
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) {
        const float4 q = p[i];
        const uint64_t ix = grid_coord((double)q.x, lx, side), iy = grid_coord((double)q.y, ly, side), iz = grid_coord((double)q.z, lz, side);
        key[i] = (spread3(ix) << 2) | (spread3(iy) << 1) | spread3(iz);
        idx[i] = (int32_t)i;
    }
}

__global__ void __launch_bounds__(256) k_gather16(const float4* __restrict__ src, const int32_t* __restrict__ idx, int64_t n, float4* __restrict__ dst) {
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) dst[i] = src[idx[i]];
}

// ---- cells, one level at a time ----------------------------------------------------------------------
// Eight lanes per cell: lane o finds, by binary search in the cell's sorted key range, the first position whose
// digit at this level exceeds o (the end of octant o); the eight boundaries are kept for k_level_emit.
__global__ void __launch_bounds__(128) k_level_count(const mwf_cell* __restrict__ cells, int64_t lev_begin, int64_t lev_end,
                                                     const uint64_t* __restrict__ key, int shift, int n_leaf, int32_t* __restrict__ n_child,
                                                     int32_t* __restrict__ bounds) {
    const int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    const int64_t c = lev_begin + (t >> 3);
    const int oct = (int)(t & 7);
    const bool live = c < lev_end;
    mwf_cell cc = {0, 0, 0, 0};
    if (live) cc = cells[c];
    int end = 0;
    const bool split = live && cc.n_ptcl > n_leaf;
    if (split) {
        const uint64_t* kb = key + cc.first_ptcl;
        int lo = 0, hi = cc.n_ptcl;
        while (lo < hi) {
            const int mid = (lo + hi) >> 1;
            if ((int)((kb[mid] >> shift) & 7) <= oct) lo = mid + 1; else hi = mid;
        }
        end = lo;
    }
    const int prev = __shfl_up_sync(0xffffffffu, end, 1);
    const int begin = oct == 0 ? 0 : prev;
    const unsigned nonempty = __ballot_sync(0xffffffffu, split && end > begin);
    if (live) {
        bounds[(c - lev_begin) * 8 + oct] = end;
        if (oct == 0) n_child[c - lev_begin] = __popc((nonempty >> (threadIdx.x & 24)) & 0xffu);
    }
}

// Writes the children of every cell of the level behind the level (child offsets = exclusive scan of n_child).
__global__ void __launch_bounds__(128) k_level_emit(mwf_cell* __restrict__ cells, double4* __restrict__ geom, int32_t* __restrict__ parent,
                                                    int64_t lev_begin, int64_t lev_end, const int32_t* __restrict__ bounds,
                                                    const int32_t* __restrict__ child_off, int64_t max_cell, unsigned int* __restrict__ err) {
    const int64_t c = lev_begin + (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (c >= lev_end) return;
    mwf_cell cc = cells[c];
    const int nc = child_off[c - lev_begin + 1] - child_off[c - lev_begin];
    cc.first_child = 0;
    cc.n_child = 0;
    if (nc > 0) {
        const int64_t first_child = lev_end + child_off[c - lev_begin];
        if (first_child + nc > max_cell) {
            atomicOr(err, ERR_BUILD_CAPACITY);
        } else {
            cc.first_child = (int32_t)first_child;
            cc.n_child = nc;
            const double4 g = geom[c];
            const double hs = __dmul_rn(0.5, g.w), qs = __dmul_rn(0.25, g.w);
            const int4 b0 = *reinterpret_cast<const int4*>(bounds + (c - lev_begin) * 8);
            const int4 b1 = *reinterpret_cast<const int4*>(bounds + (c - lev_begin) * 8 + 4);
            const int be[8] = {b0.x, b0.y, b0.z, b0.w, b1.x, b1.y, b1.z, b1.w};
            int p = 0, k = 0;
#pragma unroll
            for (int oct = 0; oct < 8; ++oct) {
                const int lo = be[oct];
                if (lo > p) {
                    mwf_cell ch;
                    ch.first_ptcl = cc.first_ptcl + p;
                    ch.n_ptcl = lo - p;
                    ch.first_child = 0;
                    ch.n_child = 0;
                    cells[first_child + k] = ch;
                    geom[first_child + k] = make_double4((oct & 4) ? __dadd_rn(g.x, qs) : __dsub_rn(g.x, qs), (oct & 2) ? __dadd_rn(g.y, qs) : __dsub_rn(g.y, qs),
                                                         (oct & 1) ? __dadd_rn(g.z, qs) : __dsub_rn(g.z, qs), hs);
                    parent[first_child + k] = (int32_t)c;
                    ++k;
                }
                p = lo;
            }
        }
    }
    cells[c] = cc;
}

__global__ void k_root_cell(mwf_cell* cells, double4* geom, int32_t* parent, const double* root, int32_t n) {
    if (threadIdx.x != 0 || blockIdx.x != 0) return;
    mwf_cell r;
    r.first_ptcl = 0; r.n_ptcl = n; r.first_child = 0; r.n_child = 0;
    cells[0] = r;
    geom[0] = make_double4(root[0], root[1], root[2], root[3]);
    parent[0] = -1;
}

// ---- groups ----------------------------------------------------------------------------------------
// mark[first_ptcl] = 1 for every group cell: the first cell on its root path with <= n_grp particles or no children.
__global__ void __launch_bounds__(256) k_group_mark(const mwf_cell* __restrict__ cells, const int32_t* __restrict__ parent, int64_t n_cell, int n_grp,
                                                    int32_t* __restrict__ mark) {
    const int64_t c = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (c >= n_cell) return;
    const mwf_cell cc = cells[c];
    const bool ok = cc.n_ptcl <= n_grp || cc.n_child == 0;
    bool par_ok = false;
    if (parent[c] >= 0) {
        const mwf_cell pc = cells[parent[c]];
        par_ok = pc.n_ptcl <= n_grp || pc.n_child == 0;  // then the parent (or one of its ancestors) is the group
    }
    if (ok && !par_ok) mark[cc.first_ptcl] = 1;
}

// rank[] = exclusive scan of mark[]: group index in Morton order
__global__ void __launch_bounds__(256) k_group_emit(const mwf_cell* __restrict__ cells, const int32_t* __restrict__ parent, int64_t n_cell, int n_grp,
                                                    const int32_t* __restrict__ rank, int64_t max_group, int32_t* __restrict__ grp_cell,
                                                    int32_t* __restrict__ grp_first, int32_t* __restrict__ grp_n) {
    const int64_t c = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (c >= n_cell) return;
    const mwf_cell cc = cells[c];
    const bool ok = cc.n_ptcl <= n_grp || cc.n_child == 0;
    bool par_ok = false;
    if (parent[c] >= 0) {
        const mwf_cell pc = cells[parent[c]];
        par_ok = pc.n_ptcl <= n_grp || pc.n_child == 0;
    }
    if (ok && !par_ok) {
        const int32_t g = rank[cc.first_ptcl];
        if (g < max_group) {
            grp_cell[g] = (int32_t)c;
            grp_first[g] = cc.first_ptcl;
            grp_n[g] = cc.n_ptcl;
        }
    }
}

// Tight bounding box of every group's particles (reading S8): one warp per group.  box[g] = lo xyz, hi xyz (fp32 values are exact).
__global__ void __launch_bounds__(256) k_group_box(const float4* __restrict__ store, const int32_t* __restrict__ grp_first, const int32_t* __restrict__ grp_n,
                                                   int64_t n_group, float* __restrict__ box) {
    const int lane = threadIdx.x & 31;
    const int64_t g = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    if (g >= n_group) return;
    const int f = grp_first[g], cnt = grp_n[g];
    float lo[3] = {INFINITY, INFINITY, INFINITY}, hi[3] = {-INFINITY, -INFINITY, -INFINITY};
    for (int i = lane; i < cnt; i += 32) {
        const float4 q = store[f + i];
        lo[0] = fminf(lo[0], q.x); hi[0] = fmaxf(hi[0], q.x);
        lo[1] = fminf(lo[1], q.y); hi[1] = fmaxf(hi[1], q.y);
        lo[2] = fminf(lo[2], q.z); hi[2] = fmaxf(hi[2], q.z);
    }
#pragma unroll
    for (int a = 0; a < 3; ++a)
#pragma unroll
        for (int d = 16; d > 0; d >>= 1) {
            lo[a] = fminf(lo[a], __shfl_xor_sync(0xffffffffu, lo[a], d));
            hi[a] = fmaxf(hi[a], __shfl_xor_sync(0xffffffffu, hi[a], d));
        }
    if (lane < 3) box[g * 6 + lane] = lane == 0 ? lo[0] : lane == 1 ? lo[1] : lo[2];
    else if (lane < 6) box[g * 6 + lane] = lane == 3 ? hi[0] : lane == 4 ? hi[1] : hi[2];
}

inline unsigned grid_for(int64_t n, int block, int cap) {
    const int64_t want = (n + block - 1) / block;
    return (unsigned)(want < cap ? (want < 1 ? 1 : want) : cap);
}

}  // namespace

#define BT(call)                                \
    do {                                        \
        cudaError_t e__ = (call);               \
        if (e__ != cudaSuccess) return e__;     \
    } while (0)

// Sorts the particles of store[0, n) into Morton order (and vel[] with them when vel != nullptr), builds the
// cells, their geometry, parents and the groups.  Synchronises the stream once per tree level to learn the
// level's size.  Outputs the counts through *n_cell / *n_group; ERR_BUILD_CAPACITY in *err when max_cell /
// max_group are too small.
cudaError_t build_tree_device(const BuildBuffers& b, int64_t n, int n_leaf, int n_grp, int64_t max_cell, int64_t max_group, bool with_vel, float4* sph,
                              int64_t* n_cell_out, int64_t* n_group_out, int* n_level_out, cudaStream_t s) {
    const int n_part = 148 * 4;
    k_bbox_partial<<<n_part, 256, 0, s>>>(b.store, n, b.bbox_part);
    BT(cudaGetLastError());
    k_root<<<1, 32, 0, s>>>(b.bbox_part, n_part, b.root);
    BT(cudaGetLastError());
    k_keys<<<grid_for(n, 256, 148 * 8), 256, 0, s>>>(b.store, n, b.root, b.key_a, b.idx_a);
    BT(cudaGetLastError());
    BT(radix_sort_pairs(b.key_a, b.idx_a, b.key_b, b.idx_b, n, 3 * KEY_BITS, b.hist, b.scan_scratch, s));
    // reorder: particles, and velocities when the caller integrates on the device
    k_gather16<<<grid_for(n, 256, 148 * 8), 256, 0, s>>>(b.store, b.idx_a, n, b.tmp16);
    BT(cudaGetLastError());
    BT(cudaMemcpyAsync(b.store, b.tmp16, (size_t)n * 16, cudaMemcpyDeviceToDevice, s));
    if (with_vel) {
        k_gather16<<<grid_for(n, 256, 148 * 8), 256, 0, s>>>(b.vel, b.idx_a, n, b.tmp16);
        BT(cudaGetLastError());
        BT(cudaMemcpyAsync(b.vel, b.tmp16, (size_t)n * 16, cudaMemcpyDeviceToDevice, s));
    }
    if (sph) {  // short-range workload: the per-particle SPH records travel with their particles
        k_gather16<<<grid_for(n, 256, 148 * 8), 256, 0, s>>>(sph, b.idx_a, n, b.tmp16);
        BT(cudaGetLastError());
        BT(cudaMemcpyAsync(sph, b.tmp16, (size_t)n * 16, cudaMemcpyDeviceToDevice, s));
    }
    // cells level by level
    k_root_cell<<<1, 32, 0, s>>>(b.cells, b.geom, b.parent, b.root, (int32_t)n);
    BT(cudaGetLastError());
    int64_t lev_begin = 0, lev_end = 1;
    int n_level = 1;
    for (int lev = 0; lev < KEY_BITS; ++lev) {
        const int64_t m = lev_end - lev_begin;
        if (m + 1 > b.level_cap) return cudaErrorInvalidValue;
        const int shift = 3 * (KEY_BITS - 1 - lev);
        k_level_count<<<(unsigned)((m * 8 + 127) / 128), 128, 0, s>>>(b.cells, lev_begin, lev_end, b.key_a, shift, n_leaf, b.level_cnt, b.level_bounds);
        BT(cudaGetLastError());
        BT(cudaMemsetAsync(b.level_cnt + m, 0, 4, s));
        BT(scan_exclusive<int32_t>(b.level_cnt, m + 1, b.scan_scratch, s));
        k_level_emit<<<(unsigned)((m + 127) / 128), 128, 0, s>>>(b.cells, b.geom, b.parent, lev_begin, lev_end, b.level_bounds, b.level_cnt, max_cell, b.err);
        BT(cudaGetLastError());
        BT(cudaMemcpyAsync(b.h_i32, b.level_cnt + m, 4, cudaMemcpyDeviceToHost, s));
        BT(cudaStreamSynchronize(s));
        const int32_t n_new = b.h_i32[0];
        if (n_new == 0) break;
        if (lev_end + n_new > max_cell) { *n_cell_out = lev_end + n_new; *n_group_out = 0; *n_level_out = n_level; return cudaSuccess; }  // err word is set
        lev_begin = lev_end;
        lev_end += n_new;
        ++n_level;
    }
    const int64_t n_cell = lev_end;
    *n_cell_out = n_cell;
    *n_level_out = n_level;
    // groups in Morton order
    BT(cudaMemsetAsync(b.mark, 0, (size_t)(n + 1) * 4, s));
    k_group_mark<<<(unsigned)((n_cell + 255) / 256), 256, 0, s>>>(b.cells, b.parent, n_cell, n_grp, b.mark);
    BT(cudaGetLastError());
    BT(scan_exclusive<int32_t>(b.mark, n + 1, b.scan_scratch, s));
    BT(cudaMemcpyAsync(b.h_i32 + 1, b.mark + n, 4, cudaMemcpyDeviceToHost, s));
    BT(cudaStreamSynchronize(s));
    const int32_t n_group = b.h_i32[1];
    *n_group_out = n_group;
    if (n_group > max_group) return cudaSuccess;  // caller reports the capacity error
    k_group_emit<<<(unsigned)((n_cell + 255) / 256), 256, 0, s>>>(b.cells, b.parent, n_cell, n_grp, b.mark, max_group, b.grp_cell, b.grp_first, b.grp_n);
    BT(cudaGetLastError());
    k_group_box<<<(unsigned)(((int64_t)n_group * 32 + 255) / 256), 256, 0, s>>>(b.store, b.grp_first, b.grp_n, n_group, b.grp_box);
    return cudaGetLastError();
}

}  // namespace mwf
