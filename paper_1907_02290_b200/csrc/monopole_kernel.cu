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

namespace mwf {

// parent[] and validation of the uploaded tree (construction step only).
__global__ void k_tree_prepare(const mwf_cell* __restrict__ cells, int64_t n_cell, int64_t max_ptcl, int32_t* __restrict__ parent,
                               int32_t* __restrict__ counter, unsigned int* __restrict__ err) {
    const int64_t c = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (c >= n_cell) return;
    const mwf_cell cc = cells[c];
    const int64_t n = cells[0].n_ptcl;
    unsigned int e = 0;
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
}

__device__ __forceinline__ void store_moment(float4* __restrict__ store, double4* __restrict__ mom64, int64_t n_ptcl, int64_t c,
                                             double sx, double sy, double sz, double m, double fx, double fy, double fz) {
    mom64[c] = make_double4(sx, sy, sz, m);  // mass-weighted position sums and mass
    float4 r;
    if (m > 0.0) {
        const double inv = 1.0 / m;
        r = make_float4((float)(sx * inv), (float)(sy * inv), (float)(sz * inv), (float)m);
    } else {  // massless cell: exerts nothing; keep a finite position
        r = make_float4((float)fx, (float)fy, (float)fz, 0.f);
    }
    store[n_ptcl + c] = r;
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
                                                   int64_t n_cell, int64_t n_ptcl, float4* __restrict__ store,
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
    store_moment(store, mom64, n_ptcl, c0, sx, sy, sz, m, f.x, f.y, f.z);
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
        store_moment(store, mom64, n_ptcl, par, sx, sy, sz, m, g.x, g.y, g.z);
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

cudaError_t launch_tree_prepare(const mwf_cell* cells, int64_t n_cell, int64_t max_ptcl, int32_t* parent, int32_t* counter,
                                unsigned int* err, cudaStream_t s) {
    const int block = 256;
    const int64_t grid = (n_cell + block - 1) / block;
    k_tree_prepare<<<(unsigned)grid, block, 0, s>>>(cells, n_cell, max_ptcl, parent, counter, err);
    return cudaGetLastError();
}

cudaError_t launch_monopoles(const mwf_cell* cells, const int32_t* parent, int64_t n_cell, int64_t n_ptcl, float4* store,
                             double4* mom64, int32_t* counter, double* quad64, float4* quad, cudaStream_t s) {
    const int block = 128;
    const int64_t grid = (n_cell + block - 1) / block;
    if (quad64 && quad)
        k_monopoles<true><<<(unsigned)grid, block, 0, s>>>(cells, parent, n_cell, n_ptcl, store, mom64, counter, quad64, quad);
    else
        k_monopoles<false><<<(unsigned)grid, block, 0, s>>>(cells, parent, n_cell, n_ptcl, store, mom64, counter, nullptr, nullptr);
    return cudaGetLastError();
}

}  // namespace mwf
