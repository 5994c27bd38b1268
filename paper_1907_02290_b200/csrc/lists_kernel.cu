// Construction-step re-encoding of the uploaded CSR index lists.
// The two lists of a group (EPJ particle indices, SPJ cell indices) become ONE list of indices into the
// combined store -- EPJ ids, then SPJ ids + N -- the paper's layout ("id_epj ... id_spj + n_epj_tot"),
// with EACH of the two runs padded to a whole number of 64-entry tiles with the index of a zero-mass dummy record
// (the paper pads with a sentinel walk whose list is empty): the force kernel sweeps EPJ tiles
// and SPJ tiles in different coordinate conventions (reading S11b), so no tile may hold both kinds.  Indices are validated
// here, once; the force kernel then runs check-free on every reuse step.
#include "mwf_internal.h"

namespace mwf {

__global__ void __launch_bounds__(256) k_merge_lists(int64_t n_group, const int32_t* __restrict__ grp_first,
                                                     const int32_t* __restrict__ grp_n, const int64_t* __restrict__ epj_off,
                                                     const int32_t* __restrict__ epj_id, const int64_t* __restrict__ spj_off,
                                                     const int32_t* __restrict__ spj_id, const int64_t* __restrict__ list_off,
                                                     int64_t n_ptcl, int64_t n_cell, int32_t* __restrict__ list,
                                                     uint8_t* __restrict__ grp_self, unsigned int* __restrict__ err) {
    __shared__ int s_self;
    for (int64_t g = blockIdx.x; g < n_group; g += gridDim.x) {
        if (threadIdx.x == 0) s_self = 0;
        __syncthreads();
        const int64_t e0 = epj_off[g], ne = epj_off[g + 1] - e0;
        const int64_t s0 = spj_off[g], ns = spj_off[g + 1] - s0;
        const int64_t o0 = list_off[g], padded = list_off[g + 1] - o0;
        const int64_t ne_pad = (ne + TILE_J - 1) / TILE_J * TILE_J;  // the SPJ run starts on a tile boundary
        const int32_t gf = grp_first[g], gn = grp_n[g];
        unsigned int e = 0;
        int self = 0;
        if (gf < 0 || gn <= 0 || (int64_t)gf + gn > n_ptcl) e |= ERR_GROUP_RANGE;
        for (int64_t k = threadIdx.x; k < ne; k += blockDim.x) {
            int32_t id = epj_id[e0 + k];
            if (id < 0 || id >= n_ptcl) { e |= ERR_EPJ_INDEX; id = (int32_t)(n_ptcl + n_cell); }
            if (id >= gf && id < gf + gn) ++self;
            list[o0 + k] = id;
        }
        for (int64_t k = threadIdx.x; k < ns; k += blockDim.x) {
            const int32_t id = spj_id[s0 + k];
            int64_t v = n_ptcl + id;
            if (id < 0 || id >= n_cell) { e |= ERR_SPJ_INDEX; v = n_ptcl + n_cell; }
            list[o0 + ne_pad + k] = (int32_t)v;
        }
        for (int64_t k = ne + threadIdx.x; k < ne_pad; k += blockDim.x) list[o0 + k] = (int32_t)(n_ptcl + n_cell);
        for (int64_t k = ne_pad + ns + threadIdx.x; k < padded; k += blockDim.x) list[o0 + k] = (int32_t)(n_ptcl + n_cell);
        if (self) atomicAdd(&s_self, self);
        __syncthreads();
        if (threadIdx.x == 0) {
            if (s_self == gn) grp_self[g] = 1;
            else if (s_self == 0) grp_self[g] = 0;
            else { grp_self[g] = 0; e |= ERR_SELF_MIXED; }
        }
        if (e) atomicOr(err, e);
        __syncthreads();
    }
}

cudaError_t launch_merge_lists(int64_t n_group, const int32_t* grp_first, const int32_t* grp_n, const int64_t* epj_off,
                               const int32_t* epj_id, const int64_t* spj_off, const int32_t* spj_id, const int64_t* list_off,
                               int64_t n_ptcl, int64_t n_cell, int32_t* list, uint8_t* grp_self, unsigned int* err, cudaStream_t s) {
    if (n_group <= 0) return cudaSuccess;
    const int64_t grid = n_group < 148 * 16 ? n_group : 148 * 16;
    k_merge_lists<<<(unsigned)grid, 256, 0, s>>>(n_group, grp_first, grp_n, epj_off, epj_id, spj_off, spj_id, list_off, n_ptcl, n_cell,
                                                 list, grp_self, err);
    return cudaGetLastError();
}

}  // namespace mwf
