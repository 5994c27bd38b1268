// The work schedule of the force kernels, made on the device: the order in which the persistent
// warps claim the work items.  Inside every WINDOW of consecutive items: longest first (so that the tail of a launch is
// made of short items), except that the NARROW items (width <= 8: few j-pairs per staged tile, so they wait on the
// gathers rather than on the FP32 pipe) are spread evenly over the first 7/8 of the wide ones, which keep the pipe busy
// meanwhile.  Windows: one over everything; or SCHED_WINDOWS of equal modelled cost when the store exceeds the L2 (the
// gathers of the items in flight then touch one stretch of the store at a time); or one per tag, for the dispatches
// that mwf_calc_force_all splits over the tags.
//
// One stable radix sort of the keys (window, narrow, cost descending) followed by a closed-form placement: the two sorted
// runs of a window are merged by rank, narrow item i going in front of the first wide item w with i * span <= w * n_narrow.
#include "mwf_internal.h"
#include "scan_sort.cuh"

namespace mwf {

namespace {

constexpr int COST_BITS = 26;  // a cost is tiles x (40 + 33 W), at most 1096 per tile: lists of up to 3.9e6 entries sort exactly, longer ones tie
constexpr uint64_t COST_MAX = (1ULL << COST_BITS) - 1;

// Modelled cost of every item (issue cycles of its warp: tiles x (staging + width j-pairs x 2 i)), plus a zero behind the last.
__global__ void __launch_bounds__(256) k_item_cost(const WorkItem* __restrict__ items, int64_t n_items, const int64_t* __restrict__ list_off,
                                                   int64_t* __restrict__ cost) {
    const int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (k > n_items) return;
    if (k == n_items) { cost[k] = 0; return; }
    const WorkItem it = items[k];
    const int64_t n_tiles = (list_off[it.group + 1] - list_off[it.group]) / TILE_J;
    cost[k] = n_tiles * (COST_STAGE + COST_PAIR * it.width);
}

// cum = exclusive scan of the costs (entry n_items: the total), kept when the windows are cut by cost
__global__ void __launch_bounds__(256) k_item_keys(const WorkItem* __restrict__ items, int64_t n_items, const int64_t* __restrict__ cost,
                                                   const int64_t* __restrict__ cum, int n_win, SchedTags tags, uint64_t* __restrict__ key,
                                                   int32_t* __restrict__ idx) {
    const int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= n_items) return;
    const WorkItem it = items[k];
    uint64_t win = 0;
    if (tags.n_tag > 0) {  // window = the tag whose group range holds the item's group
        for (int t = 1; t < tags.n_tag; ++t) win += it.group >= tags.bound[t];
    } else if (n_win > 1) {  // window w takes the items whose cost prefix lies in [w, w + 1) x total / n_win
        const int64_t step = cum[n_items] / n_win, c = cum[k];
        for (int j = 1; j < n_win; ++j) win += c >= step * j;
    }
    const uint64_t narrow = it.width > 8 ? 0 : 1;
    const uint64_t c = (uint64_t)cost[k] > COST_MAX ? COST_MAX : (uint64_t)cost[k];
    key[k] = (win << (COST_BITS + 1)) | (narrow << COST_BITS) | (COST_MAX - c);
    idx[k] = (int32_t)k;
}

// seg[s] = first sorted position of segment s = 2 x window + narrow (n_items for a segment nobody is in, fixed up below)
__global__ void __launch_bounds__(256) k_seg_mark(const uint64_t* __restrict__ key, int64_t n_items, int32_t* __restrict__ seg) {
    const int64_t r = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (r >= n_items) return;
    const int s = (int)(key[r] >> COST_BITS);
    if (r == 0 || (int)(key[r - 1] >> COST_BITS) != s) seg[s] = (int32_t)r;
}
__global__ void k_seg_fix(int32_t* seg, int n_seg, int32_t n_items) {
    if (threadIdx.x != 0 || blockIdx.x != 0) return;
    seg[n_seg] = n_items;
    for (int s = n_seg - 1; s >= 0; --s)
        if (seg[s] < 0) seg[s] = seg[s + 1];
}

__global__ void __launch_bounds__(256) k_place(const uint64_t* __restrict__ key, const int32_t* __restrict__ idx, int64_t n_items,
                                               const int32_t* __restrict__ seg, int32_t* __restrict__ order) {
    const int64_t r = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (r >= n_items) return;
    const int s = (int)(key[r] >> COST_BITS), w = s >> 1;
    const int64_t base = seg[2 * w], nw = seg[2 * w + 1] - base, nn = seg[2 * w + 2] - seg[2 * w + 1];
    const int64_t span = nw - nw / 8;  // the narrow items go between the first `span` wide ones
    int64_t pos;
    if ((s & 1) == 0) {  // wide item of rank iw: behind the narrow items i with i * span <= iw * nn
        const int64_t iw = r - base;
        const int64_t before = iw >= span ? nn : (nn == 0 ? 0 : (iw * nn / span + 1 < nn ? iw * nn / span + 1 : nn));
        pos = iw + before;
    } else {  // narrow item of rank i: behind the wide items w with w * nn < i * span
        const int64_t i = r - seg[2 * w + 1];
        const int64_t before = span == 0 ? 0 : ((i * span + nn - 1) / nn < span ? (i * span + nn - 1) / nn : span);
        pos = i + before;
    }
    order[base + pos] = idx[r];
}

}  // namespace

#define SC(call)                                \
    do {                                        \
        cudaError_t e__ = (call);               \
        if (e__ != cudaSuccess) return e__;     \
    } while (0)

// order[0, n_items) = the schedule of items[0, n_items).  n_win windows of equal cost, or one window per tag (tags.n_tag > 0).
cudaError_t launch_schedule(const SchedBuffers& b, const WorkItem* items, int64_t n_items, const int64_t* list_off, int n_win, const SchedTags& tags,
                            int32_t* order, cudaStream_t s) {
    if (n_items <= 0) return cudaSuccess;
    const unsigned grid = (unsigned)((n_items + 1 + 255) / 256);
    k_item_cost<<<grid, 256, 0, s>>>(items, n_items, list_off, b.cost);
    SC(cudaGetLastError());
    const bool by_cost = tags.n_tag == 0 && n_win > 1;
    if (by_cost) {
        SC(cudaMemcpyAsync(b.cum, b.cost, (size_t)(n_items + 1) * 8, cudaMemcpyDeviceToDevice, s));
        SC(scan_exclusive<int64_t>(b.cum, n_items + 1, b.scan_scratch64, s));
    }
    k_item_keys<<<grid, 256, 0, s>>>(items, n_items, b.cost, b.cum, by_cost ? n_win : 1, tags, b.key_a, b.idx_a);
    SC(cudaGetLastError());
    const int n_windows = tags.n_tag > 0 ? tags.n_tag : (by_cost ? n_win : 1);
    int bits = COST_BITS + 1;
    while ((1 << (bits - COST_BITS - 1)) < n_windows) ++bits;
    SC(radix_sort_pairs(b.key_a, b.idx_a, b.key_b, b.idx_b, n_items, bits, b.hist, b.scan_scratch, s));
    const int n_seg = 2 * n_windows;
    SC(cudaMemsetAsync(b.seg, 0xFF, (size_t)(n_seg + 1) * 4, s));
    k_seg_mark<<<grid, 256, 0, s>>>(b.key_a, n_items, b.seg);
    SC(cudaGetLastError());
    k_seg_fix<<<1, 32, 0, s>>>(b.seg, n_seg, (int32_t)n_items);
    SC(cudaGetLastError());
    k_place<<<grid, 256, 0, s>>>(b.key_a, b.idx_a, n_items, b.seg, order);
    return cudaGetLastError();
}

}  // namespace mwf
