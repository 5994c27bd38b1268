// Bottom-up monopole refresh on the device over the fixed tree (
// paper: "multipole moments of all local tree cells are calculated, from the bottom to the top of the
// tree. Even at the reusing step ..." P:160; reuse step 1/3 "update the physical information" P:134-136;
// centre-of-mass approximation, SPJ same type as EPJ P:848).
//
// One launch, no per-level synchronisation: every leaf sums its particle range in fp64, then climbs;
// at each internal cell the LAST child to arrive (atomic counter) combines the children's fp64 moments in
// child order and continues upward.  Summation order is fixed by the tree, so results are deterministic.
// The arrival counters reset themselves, so the kernel can be re-launched every step.
// Moments are kept in fp64 in a scratch array and rounded once to the float4 SPJ record (X_c, M_c) that
// the force kernel reads at store[N + c] (paper: SPJ behind the EPJ at offset n_epj_tot).
#include "mwf_internal.h"
#include "scan_sort.cuh"

namespace mwf {

// parent[] and validation of the uploaded tree (construction step only).
__global__ void k_tree_prepare(const mwf_cell* __restrict__ cells, int64_t n_cell, int64_t max_ptcl, int32_t* __restrict__ parent,
                               int32_t* __restrict__ counter, unsigned int* __restrict__ err) {
    const int64_t c = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    const bool live = c < n_cell;  // no early return: every lane of the warp takes part in the reduction at the end
    unsigned int e = 0;
    unsigned claims = 0;
    if (live) {
        const mwf_cell cc = cells[c];
        const int64_t n = cells[0].n_ptcl;
        if (c == 0) {
            parent[0] = -1;
            if (cc.first_ptcl != 0 || cc.n_ptcl <= 0 || cc.n_ptcl > max_ptcl) e |= ERR_CELL_RANGE;
        }
        counter[c] = 0;
        if (cc.n_ptcl <= 0 || cc.first_ptcl < 0 || (int64_t)cc.first_ptcl + cc.n_ptcl > n) e |= ERR_CELL_RANGE;
        if (cc.n_child < 0 || cc.n_child > 8) e |= ERR_CHILD_RANGE;
        if (cc.n_child > 0) {
            if (cc.first_child <= c || (int64_t)cc.first_child + cc.n_child > n_cell) {
                e |= ERR_CHILD_RANGE;
            } else {
                int64_t next = cc.first_ptcl;
                for (int k = 0; k < cc.n_child; ++k) {
                    const mwf_cell ch = cells[cc.first_child + k];
                    if (ch.first_ptcl != next) e |= ERR_CHILD_PART;
                    next += ch.n_ptcl;
                    parent[cc.first_child + k] = (int32_t)c;
                }
                if (next != (int64_t)cc.first_ptcl + cc.n_ptcl) e |= ERR_CHILD_PART;
            }
        }
        if (e) atomicOr(err, e);
        // number of child claims, for k_tree_check (a cell with a bad child range claims nothing)
        claims = (cc.n_child > 0 && !(e & ERR_CHILD_RANGE)) ? (unsigned)cc.n_child : 0u;
    }
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) claims += __shfl_xor_sync(0xffffffffu, claims, d);
    if ((threadIdx.x & 31) == 0 && claims) atomicAdd(err + 1, claims);
}

// Every cell but the root must have been claimed by exactly one parent: parent[] was preset to a negative mark, so an
// orphan still carries it, and n_cell - 1 claims over n_cell - 1 claimed cells leave no cell claimed twice.  (The climb
// variant of the refresh and the per-cell passes of the construction step follow parent[] without checks.)
__global__ void k_tree_check(const int32_t* __restrict__ parent, int64_t n_cell, unsigned int* __restrict__ err) {
    const int64_t c = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (c >= n_cell) return;
    if (c == 0) {
        if ((int64_t)err[1] != n_cell - 1) atomicOr(err, ERR_CHILD_PART);
    } else if (parent[c] < 0) {
        atomicOr(err, ERR_CHILD_RANGE);
    }
}

// The SPJ record of cell c: centre of mass and mass rounded to the float4 the force kernel gathers at store[N + c], plus
// the rounding remainder of the centre, spj_lo[c] = X - (double)float(X) rounded to float (reading S11b of DESIGN.md: a
// centre of mass is not an fp32 input, and on the fp32 grid of coordinates of order 1 it would be 3e-8 off -- 1e-4 of the
// force of a cell 1e-3 away, which is the north_star's whole error budget).  The force kernel adds the remainder after it
// has moved the record into group-centred coordinates.
__device__ __forceinline__ void write_spj(float4* __restrict__ store, float4* __restrict__ spj_lo, int64_t n_ptcl, int64_t c,
                                          double sx, double sy, double sz, double m, float fx, float fy, float fz) {
    float4 r, lo = make_float4(0.f, 0.f, 0.f, 0.f);
    if (m > 0.0) {
        const double inv = 1.0 / m;
        const double X = sx * inv, Y = sy * inv, Z = sz * inv;
        r = make_float4((float)X, (float)Y, (float)Z, (float)m);
        lo = make_float4((float)(X - (double)r.x), (float)(Y - (double)r.y), (float)(Z - (double)r.z), 0.f);
    } else {  // massless cell: exerts nothing; keep a finite position
        r = make_float4(fx, fy, fz, 0.f);
    }
    store[n_ptcl + c] = r;   // SPJ behind the EPJ
    spj_lo[c] = lo;
}

__device__ __forceinline__ void store_moment(float4* __restrict__ store, float4* __restrict__ spj_lo, double4* __restrict__ mom64, int64_t n_ptcl,
                                             int64_t c, double sx, double sy, double sz, double m, float fx, float fy, float fz) {
    mom64[c] = make_double4(sx, sy, sz, m);  // mass-weighted position sums and mass
    write_spj(store, spj_lo, n_ptcl, c, sx, sy, sz, m, fx, fy, fz);
}

// Second moments about the centre of mass (NEXT-3, quadrupole SPJ): quad64[6c..6c+5] = (Qxx Qyy Qzz Qxy Qxz Qyz) in fp64
// and the float record the correction kernel gathers: (Qxx Qyy Qzz Qxy) (Qxz Qyz tr(Q)/2 0).
__device__ __forceinline__ void store_quad(double* __restrict__ quad64, float4* __restrict__ quad, int64_t c, const double (&q)[6]) {
#pragma unroll
    for (int k = 0; k < 6; ++k) quad64[6 * c + k] = q[k];
    quad[2 * c] = make_float4((float)q[0], (float)q[1], (float)q[2], (float)q[3]);
    quad[2 * c + 1] = make_float4((float)q[4], (float)q[5], (float)(0.5 * (q[0] + q[1] + q[2])), 0.f);
}

template <bool QUAD>
__global__ void __launch_bounds__(128) k_monopoles(const mwf_cell* __restrict__ cells, const int32_t* __restrict__ parent,
                                                   int64_t n_cell, int64_t n_ptcl, float4* __restrict__ store, float4* __restrict__ spj_lo,
                                                   double4* __restrict__ mom64, int32_t* __restrict__ counter,
                                                   double* __restrict__ quad64, float4* __restrict__ quad) {
    const int64_t c0 = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (c0 >= n_cell) return;
    const mwf_cell leaf = cells[c0];
    if (leaf.n_child != 0) return;  // internal cells are computed by their last-arriving descendant
    double sx = 0.0, sy = 0.0, sz = 0.0, m = 0.0;
    const float4* __restrict__ p = store + leaf.first_ptcl;
    for (int k = 0; k < leaf.n_ptcl; ++k) {
        const float4 q = p[k];
        const double mq = (double)q.w;
        m += mq;
        sx += mq * (double)q.x;
        sy += mq * (double)q.y;
        sz += mq * (double)q.z;
    }
    const float4 f = p[0];
    store_moment(store, spj_lo, mom64, n_ptcl, c0, sx, sy, sz, m, f.x, f.y, f.z);
    if constexpr (QUAD) {  // second pass over the leaf's particles, about its centre of mass
        double q[6] = {0.0, 0.0, 0.0, 0.0, 0.0, 0.0};
        if (m > 0.0) {
            const double X = sx / m, Y = sy / m, Z = sz / m;
            for (int k = 0; k < leaf.n_ptcl; ++k) {
                const float4 r = p[k];
                const double mq = (double)r.w, yx = (double)r.x - X, yy = (double)r.y - Y, yz = (double)r.z - Z;
                q[0] += mq * yx * yx; q[1] += mq * yy * yy; q[2] += mq * yz * yz;
                q[3] += mq * yx * yy; q[4] += mq * yx * yz; q[5] += mq * yy * yz;
            }
        }
        store_quad(quad64, quad, c0, q);
    }
    int64_t c = c0;
    for (;;) {
        const int32_t par = parent[c];
        if (par < 0) break;
        const mwf_cell pc = cells[par];
        __threadfence();  // publish this cell's moments before announcing arrival
        const int arrived = atomicAdd(&counter[par], 1);
        if (arrived != pc.n_child - 1) break;  // a later sibling will do the parent
        counter[par] = 0;                      // self-cleaning for the next refresh
        __threadfence();
        sx = sy = sz = m = 0.0;
        for (int k = 0; k < pc.n_child; ++k) {
            const double2* q = reinterpret_cast<const double2*>(&mom64[pc.first_child + k]);
            const double2 lo = __ldcg(q), hi = __ldcg(q + 1);  // from L2: written by other SMs
            sx += lo.x; sy += lo.y; sz += hi.x; m += hi.y;
        }
        const float4 g = store[pc.first_ptcl];
        store_moment(store, spj_lo, mom64, n_ptcl, par, sx, sy, sz, m, g.x, g.y, g.z);
        if constexpr (QUAD) {  // parallel-axis theorem: Q = sum over children of Q_child + M_child d d^T, d = X_child - X
            double q[6] = {0.0, 0.0, 0.0, 0.0, 0.0, 0.0};
            if (m > 0.0) {
                const double X = sx / m, Y = sy / m, Z = sz / m;
                for (int k = 0; k < pc.n_child; ++k) {
                    const int64_t ch = pc.first_child + k;
                    const double2* mq = reinterpret_cast<const double2*>(&mom64[ch]);
                    const double2 lo = __ldcg(mq), hi = __ldcg(mq + 1);
                    if (!(hi.y > 0.0)) continue;
                    const double dx = lo.x / hi.y - X, dy = lo.y / hi.y - Y, dz = hi.x / hi.y - Z;
                    const double2* cq = reinterpret_cast<const double2*>(quad64 + 6 * ch);
                    const double2 a = __ldcg(cq), b = __ldcg(cq + 1), e = __ldcg(cq + 2);
                    q[0] += a.x + hi.y * dx * dx; q[1] += a.y + hi.y * dy * dy; q[2] += b.x + hi.y * dz * dz;
                    q[3] += b.y + hi.y * dx * dy; q[4] += e.x + hi.y * dx * dz; q[5] += e.y + hi.y * dy * dz;
                }
            }
            store_quad(quad64, quad, par, q);
        }
        c = par;
    }
}

// ---------------------------------------------------------------------------------------------------
// Scan variant of the refresh (monopoles only; the default).  The climb above is bound by its dependency chain: one L2 round
// trip after another per tree level (measured: leaf sums 32 us, climb 65 us for config 5).  The leaves partition the
// particles in Morton order, so with the leaves RANKED in that order every cell is a contiguous range [lf, ll) of leaf
// ranks (fixed at the construction step, k_leaf_mark / k_leaf_ranges) and
//     (sum m x, sum m)(cell) = P[ll] - P[lf],   P = exclusive fp64 prefix sum of the leaves' (sum m x, sum m)
// with no dependency between cells.  Per refresh: k_leaf_moments (every leaf sums its particles in fp64, writes its own SPJ
// record and its entry of P), a two-kernel exclusive scan of P (tiles of 1024, tile totals scanned by one block), and
// k_cells_from_prefix (every internal cell takes the difference, adds the tile offsets, writes its SPJ record).  Deterministic
// (fixed summation order).  The difference loses |P| / (cell sum) x 2^-53 relative: < 1e-9 on every config, against a
// parity bar of 1e-6 (reading S11).

__global__ void __launch_bounds__(256) k_leaf_mark(const mwf_cell* __restrict__ cells, int64_t n_cell, int32_t* __restrict__ mark) {
    const int64_t c = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (c >= n_cell) return;
    const mwf_cell cc = cells[c];
    if (cc.n_child == 0) mark[cc.first_ptcl] = 1;
}

__global__ void __launch_bounds__(256) k_leaf_ranges(const mwf_cell* __restrict__ cells, int64_t n_cell, const int32_t* __restrict__ rank_at,
                                                     int2* __restrict__ cell_lr) {
    const int64_t c = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (c >= n_cell) return;
    const mwf_cell cc = cells[c];
    cell_lr[c] = make_int2(rank_at[cc.first_ptcl], rank_at[cc.first_ptcl + cc.n_ptcl]);
}

__global__ void __launch_bounds__(256) k_leaf_moments(const mwf_cell* __restrict__ cells, const int2* __restrict__ cell_lr, int64_t n_cell,
                                                      int64_t n_ptcl, int64_t n_leaf_cells, float4* __restrict__ store, float4* __restrict__ spj_lo,
                                                      double4* __restrict__ P) {
    const int64_t c = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (c == 0) P[n_leaf_cells] = make_double4(0.0, 0.0, 0.0, 0.0);  // the scan turns this entry into the grand total
    if (c >= n_cell) return;
    const mwf_cell leaf = cells[c];
    if (leaf.n_child != 0) return;
    double sx = 0.0, sy = 0.0, sz = 0.0, m = 0.0;
    const float4* __restrict__ p = store + leaf.first_ptcl;
    const float4 f = p[0];
#pragma unroll 4
    for (int k = 0; k < leaf.n_ptcl; ++k) {
        const float4 q = p[k];
        const double mq = (double)q.w;
        m += mq;
        sx += mq * (double)q.x;
        sy += mq * (double)q.y;
        sz += mq * (double)q.z;
    }
    P[cell_lr[c].x] = make_double4(sx, sy, sz, m);
    write_spj(store, spj_lo, n_ptcl, c, sx, sy, sz, m, f.x, f.y, f.z);
}

constexpr int SCAN4_THREADS = 256, SCAN4_ITEMS = 4, SCAN4_TILE = SCAN4_THREADS * SCAN4_ITEMS;

__device__ __forceinline__ double4 add4(const double4 a, const double4 b) { return make_double4(a.x + b.x, a.y + b.y, a.z + b.z, a.w + b.w); }
__device__ __forceinline__ double4 shfl_up4(const double4 v, int d) {
    return make_double4(__shfl_up_sync(0xffffffffu, v.x, d), __shfl_up_sync(0xffffffffu, v.y, d), __shfl_up_sync(0xffffffffu, v.z, d),
                        __shfl_up_sync(0xffffffffu, v.w, d));
}
// inclusive scan over the block of one value per thread; returns the exclusive prefix of the thread, *total = block sum
template <int THREADS>
__device__ __forceinline__ double4 block_exclusive4(double4 v, double4* s_warp, double4* total) {
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    double4 incl = v;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
        const double4 up = shfl_up4(incl, d);
        if (lane >= d) incl = add4(up, incl);
    }
    if (lane == 31) s_warp[warp] = incl;
    __syncthreads();
    double4 wex = make_double4(0.0, 0.0, 0.0, 0.0), tot = wex;
    for (int w = 0; w < THREADS / 32; ++w) {  // few warps: a serial pass keeps the order of the additions fixed and simple
        if (w == warp) wex = tot;
        tot = add4(tot, s_warp[w]);
    }
    *total = tot;
    const double4 up = shfl_up4(incl, 1);
    const double4 ex_in_warp = lane == 0 ? make_double4(0.0, 0.0, 0.0, 0.0) : up;
    __syncthreads();
    return add4(wex, ex_in_warp);
}

// exclusive scan inside every tile of SCAN4_TILE entries, tile totals to tsum
__global__ void __launch_bounds__(SCAN4_THREADS) k_scan4_tiles(double4* __restrict__ P, int64_t n, double4* __restrict__ tsum) {
    __shared__ double4 s_warp[SCAN4_THREADS / 32];
    const int64_t base = (int64_t)blockIdx.x * SCAN4_TILE + (int64_t)threadIdx.x * SCAN4_ITEMS;
    double4 v[SCAN4_ITEMS], sum = make_double4(0.0, 0.0, 0.0, 0.0);
#pragma unroll
    for (int k = 0; k < SCAN4_ITEMS; ++k) {
        v[k] = base + k < n ? P[base + k] : make_double4(0.0, 0.0, 0.0, 0.0);
        sum = add4(sum, v[k]);
    }
    double4 total;
    double4 run = block_exclusive4<SCAN4_THREADS>(sum, s_warp, &total);
#pragma unroll
    for (int k = 0; k < SCAN4_ITEMS; ++k) {
        if (base + k < n) P[base + k] = run;
        run = add4(run, v[k]);
    }
    if (threadIdx.x == 0) tsum[blockIdx.x] = total;
}

// exclusive scan of the tile totals by one block (chunks of 1024 with a carry)
__global__ void __launch_bounds__(1024) k_scan4_totals(double4* __restrict__ tsum, int64_t n_tile) {
    __shared__ double4 s_warp[32];
    double4 carry = make_double4(0.0, 0.0, 0.0, 0.0);
    for (int64_t b = 0; b < n_tile; b += 1024) {
        const int64_t i = b + threadIdx.x;
        const double4 v = i < n_tile ? tsum[i] : make_double4(0.0, 0.0, 0.0, 0.0);
        double4 total;
        const double4 ex = block_exclusive4<1024>(v, s_warp, &total);
        if (i < n_tile) tsum[i] = add4(carry, ex);
        carry = add4(carry, total);
    }
}

__global__ void __launch_bounds__(256) k_cells_from_prefix(const mwf_cell* __restrict__ cells, const int2* __restrict__ cell_lr, int64_t n_cell,
                                                           int64_t n_ptcl, float4* __restrict__ store, float4* __restrict__ spj_lo,
                                                           const double4* __restrict__ P, const double4* __restrict__ toff) {
    const int64_t c = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (c >= n_cell) return;
    const mwf_cell cc = cells[c];
    if (cc.n_child == 0) return;  // leaves wrote their records themselves
    const int2 lr = cell_lr[c];
    const double4 hi = add4(toff[lr.y / SCAN4_TILE], P[lr.y]), lo = add4(toff[lr.x / SCAN4_TILE], P[lr.x]);
    const double sx = hi.x - lo.x, sy = hi.y - lo.y, sz = hi.z - lo.z, m = hi.w - lo.w;
    float4 f = make_float4(0.f, 0.f, 0.f, 0.f);
    if (!(m > 0.0)) f = store[cc.first_ptcl];
    write_spj(store, spj_lo, n_ptcl, c, sx, sy, sz, m, f.x, f.y, f.z);
}

cudaError_t launch_tree_prepare(const mwf_cell* cells, int64_t n_cell, int64_t max_ptcl, int32_t* parent, int32_t* counter,
                                unsigned int* err, cudaStream_t s) {
    const int block = 256;
    const int64_t grid = (n_cell + block - 1) / block;
    cudaError_t e = cudaMemsetAsync(parent, 0xFE, (size_t)n_cell * 4, s);  // "unclaimed": negative
    if (e != cudaSuccess) return e;
    if ((e = cudaMemsetAsync(err + 1, 0, 4, s)) != cudaSuccess) return e;
    k_tree_prepare<<<(unsigned)grid, block, 0, s>>>(cells, n_cell, max_ptcl, parent, counter, err);
    if ((e = cudaGetLastError()) != cudaSuccess) return e;
    k_tree_check<<<(unsigned)grid, block, 0, s>>>(parent, n_cell, err);
    return cudaGetLastError();
}

cudaError_t launch_monopoles(const mwf_cell* cells, const int32_t* parent, int64_t n_cell, int64_t n_ptcl, float4* store, float4* spj_lo,
                             double4* mom64, int32_t* counter, double* quad64, float4* quad, cudaStream_t s) {
    const int block = 128;
    const int64_t grid = (n_cell + block - 1) / block;
    if (quad64 && quad)
        k_monopoles<true><<<(unsigned)grid, block, 0, s>>>(cells, parent, n_cell, n_ptcl, store, spj_lo, mom64, counter, quad64, quad);
    else
        k_monopoles<false><<<(unsigned)grid, block, 0, s>>>(cells, parent, n_cell, n_ptcl, store, spj_lo, mom64, counter, nullptr, nullptr);
    return cudaGetLastError();
}

}  // namespace mwf

namespace mwf {

int64_t scan4_tiles(int64_t n_leaf_cells) { return (n_leaf_cells + 1 + SCAN4_TILE - 1) / SCAN4_TILE; }

// Construction step: rank the leaves in Morton order and give every cell its range of leaf ranks.  mark: n_ptcl + 1
// ints of scratch (left holding the ranks), scratch: scan scratch for n_ptcl + 1 ints.  The number of leaves is copied to
// *n_leaf_pinned (pinned host memory) on the stream: valid once the caller has synchronised it.
cudaError_t launch_leaf_ranking(const mwf_cell* cells, int64_t n_cell, int64_t n_ptcl, int32_t* mark, int32_t* scratch, int2* cell_lr,
                                int32_t* n_leaf_pinned, cudaStream_t s) {
    cudaError_t e = cudaMemsetAsync(mark, 0, (size_t)(n_ptcl + 1) * 4, s);
    if (e != cudaSuccess) return e;
    k_leaf_mark<<<(unsigned)((n_cell + 255) / 256), 256, 0, s>>>(cells, n_cell, mark);
    if ((e = cudaGetLastError()) != cudaSuccess) return e;
    if ((e = scan_exclusive<int32_t>(mark, n_ptcl + 1, scratch, s)) != cudaSuccess) return e;
    k_leaf_ranges<<<(unsigned)((n_cell + 255) / 256), 256, 0, s>>>(cells, n_cell, mark, cell_lr);
    if ((e = cudaGetLastError()) != cudaSuccess) return e;
    return cudaMemcpyAsync(n_leaf_pinned, mark + n_ptcl, 4, cudaMemcpyDeviceToHost, s);
}

cudaError_t launch_monopoles_scan(const mwf_cell* cells, const int2* cell_lr, int64_t n_cell, int64_t n_ptcl, int64_t n_leaf_cells, float4* store,
                                  float4* spj_lo, double4* P, double4* toff, cudaStream_t s) {
    const unsigned grid = (unsigned)((n_cell + 255) / 256);
    k_leaf_moments<<<grid, 256, 0, s>>>(cells, cell_lr, n_cell, n_ptcl, n_leaf_cells, store, spj_lo, P);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return e;
    const int64_t nt = scan4_tiles(n_leaf_cells);
    k_scan4_tiles<<<(unsigned)nt, SCAN4_THREADS, 0, s>>>(P, n_leaf_cells + 1, toff);
    if ((e = cudaGetLastError()) != cudaSuccess) return e;
    k_scan4_totals<<<1, 1024, 0, s>>>(toff, nt);
    if ((e = cudaGetLastError()) != cudaSuccess) return e;
    k_cells_from_prefix<<<grid, 256, 0, s>>>(cells, cell_lr, n_cell, n_ptcl, store, spj_lo, P, toff);
    return cudaGetLastError();
}

}  // namespace mwf
